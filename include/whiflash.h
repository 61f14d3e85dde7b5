/* whiflash.h — C ABI of the B200-native (sm_100a) verify-and-switch hot path of WhiFlash
 * (arxiv/paper_2606_07710).  Citations are lines of /root/reference/PAPER.md and readings
 * C1..C25 of DESIGN.md.
 *
 * Conventions
 *  - Every call returns int: WF_OK (0) or a negative wf_status.  Nothing throws or aborts.
 *    wf_last_error(ctx) returns a static/ctx-owned message for the last failing call.
 *  - Pointers are DEVICE pointers unless the name ends in _host.  Tensor bases and row strides are
 *    16-byte aligned.  bf16 tensors are passed as void* (raw bf16 bits, little endian).
 *  - Hot calls are asynchronous on the caller's CUDA stream (a cudaStream_t passed as void*; NULL =
 *    the legacy default stream) and never synchronise the host.  Conditions only the device can
 *    see (page exhaustion, backlog overflow, a length beyond the host bound that sized a launch)
 *    set a sticky device status word read by wf_poll_status; the first error of a poll interval
 *    wins.
 *  - Calls that share a wf_ctx, a wf_paged_kv or a wf_drafter must be stream-ordered with respect to
 *    one another (one stream, or events between streams): the handles own per-call scratch
 *    (completion counters, row plans, operand packs).  Distinct contexts may run concurrently.
 *  - Ownership: the caller allocates and owns every tensor (pools, block tables, lengths, weights,
 *    backlog, workspaces).  Handles (wf_ctx, wf_paged_kv, wf_drafter) are opaque, created and
 *    destroyed here; they borrow the caller's pointers and own only small bookkeeping buffers
 *    (free-page ring, pages-held counters, RoPE table, tensor maps, row plans).
 *  - Every step of every call runs in this library's own CUDA kernels; there is no CPU path.
 */
#ifndef WHIFLASH_H_
#define WHIFLASH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  WF_OK = 0,
  WF_ERR_INVALID_ARG = -1,
  WF_ERR_UNSUPPORTED_SHAPE = -2,
  WF_ERR_OUT_OF_PAGES = -3,     /* device status: a reserve could not be served; nothing was allocated */
  WF_ERR_QUEUE_OVERFLOW = -4,   /* device status: one round's rows alone exceed backlog_cap */
  WF_ERR_CUDA = -5
} wf_status;

#define WF_ROUTE_DIFFUSION 0
#define WF_ROUTE_AR 1

typedef struct wf_ctx wf_ctx;
typedef struct wf_paged_kv wf_paged_kv;
typedef struct wf_drafter wf_drafter;

/* ---- lifecycle ------------------------------------------------------------------------------ */
int wf_ctx_create(wf_ctx** out, int device_ordinal);
int wf_ctx_destroy(wf_ctx* ctx);
const char* wf_last_error(const wf_ctx* ctx);
/* Copies the sticky device status word to *status_host (synchronises `stream`) and clears it. */
int wf_poll_status(wf_ctx* ctx, void* stream, int* status_host);
/* Number of kernels this library has launched through ctx since creation (host counter). */
int64_t wf_launch_count(const wf_ctx* ctx);

/* ---- paged KV cache + block table (BASELINE.json north_star "plus a paged-KV block table";
 *      the paper itself uses the HF cache).  The target cache and every drafter
 *      cache are instances.
 * Pools: bf16 [n_layers][num_pages][n_kv_heads][page_size][head_dim], K and V separate.
 * block_table int32 [max_seqs][max_pages_per_seq] (-1 = no page); seq_len int32 [max_seqs] =
 * tokens that are final in the cache.  Both are caller-owned and may be written by the caller
 * between calls (e.g. to set the initial context after a reserve).
 * Allocation order (reading C24): the free list is an explicit ordered ring initialised from
 * free_pages_host; one reserve call serves sequences in ascending index, each taking consecutive
 * ring entries from the head; released pages go to the tail in block-table order. */
typedef struct {
  int n_layers, n_kv_heads, head_dim, page_size, num_pages, max_seqs, max_pages_per_seq;
} wf_kv_shape;

int wf_kv_create(wf_ctx* ctx, const wf_kv_shape* shape, void* k_pool, void* v_pool,
                 int32_t* block_table, int32_t* seq_len,
                 const int32_t* free_pages_host, int n_free, wf_paged_kv** out);
int wf_kv_destroy(wf_paged_kv* kv);
/* Grow block tables so that sequence b in [0,B) can hold seq_len[b] + add_tokens[b] tokens.
 * If the ring cannot serve the whole call, nothing is allocated and the device status becomes
 * WF_ERR_OUT_OF_PAGES.  seq_len is not changed. */
int wf_kv_reserve(wf_paged_kv* kv, const int32_t* add_tokens, int B, void* stream);
/* Return all pages of sequence `seq` to the ring tail; seq_len[seq] = 0. */
int wf_kv_release_seq(wf_paged_kv* kv, int seq, void* stream);
/* Device pointer to the int32 [max_seqs] pages-held counters (library-owned; for inspection). */
const int32_t* wf_kv_pages_held(const wf_paged_kv* kv);

/* ---- (a) verification attention for ONE target layer -------------------------------------------
 * PAPER.md:65 (§3.2 "returned to the target model for parallel verification"); north_star (a).
 * For sequence b with ctx_b = target_kv.seq_len[b], rows i in [0, q_b), q_b = q_indptr[b+1] -
 * q_indptr[b] <= max_q_len, query head h, kv head g = h / (n_q_heads / n_kv_heads) (C11):
 *     s_j = <Q[i,h,:], K[b,j,g,:]> * sm_scale, j = 0 .. ctx_b + i      (causal within block, C10)
 *     O[i,h,:] = sum_j softmax(s)_j V[b,j,g,:]                          (fp32 accumulate, C13)
 * The block's own K/V must already be in the cache at positions ctx_b .. ctx_b+q_b-1 (C10).
 * q, out: bf16 [sum_q][n_q_heads][head_dim].  workspace: >= wf_verify_attn_workspace_bytes.
 * Supported: head_dim 64 or 128; page_size 16; max_q_len <= 64 and group = n_q_heads/n_kv_heads <= 64 (rows of a block
 * beyond max_q_len are not computed and the sticky status becomes WF_ERR_INVALID_ARG).  Blocks of up to 64 rows per kv head
 * (max_q_len * group <= 64: every config of BASELINE.json) run on the chain kernel; longer ones (e.g. gamma = 15 at a group of
 * 8) are run as degenerate trees on the tree kernel's 128-row tiles (one extra tiny launch writes their masks into the
 * workspace), subject to wf_verify_attn_tree's limit B * ceil(max_q_len * group / 128) <= 1024. */
int wf_verify_attn(wf_ctx* ctx, const wf_paged_kv* target_kv, int layer,
                   const void* q, const int32_t* q_indptr, int B, int n_q_heads, int max_q_len,
                   float sm_scale, void* out, void* workspace, size_t workspace_bytes, void* stream);
size_t wf_verify_attn_workspace_bytes(const wf_kv_shape* shape, int B, int n_q_heads, int max_q_len);
/* Launch shape of wf_verify_attn (a tuning / test hook; results are within tolerance of one another, not bit-equal).
 * -1 (default): automatic: with few (sequence, kv head) pairs (batch 1-2 at 8 kv heads) one thread-block cluster per pair,
 * partials folded through distributed shared memory in a fixed order (bit-reproducible); otherwise, and whenever the
 * last launch over the same cache was long enough to be HBM-paced, persistent stream-K ranges over all SMs.
 * 0: never use clusters.  1..16: force that many CTAs per pair whenever the pairs fit (else stream-K); 1 = one CTA per pair,
 * no merge at all (what the automatic mode picks for an HBM-paced launch whose pairs cover at least 80 % of the SMs). */
int wf_ctx_set_attn_cluster(wf_ctx* ctx, int cluster_size);
/* Early K/V (off by default).  Every kernel of this library is launched with programmatic dependent launch and waits for
 * the previous kernel of the stream before it touches anything that kernel may have written.  With on = 1 the caller
 * PROMISES, for every later wf_verify_attn / wf_verify_attn_tree / wf_final_token_full through this context, that the
 * kernel launched immediately before it on the same stream writes none of: q_indptr, the cache's seq_len, its block-table
 * entries for pages below seq_len[b], and its K/V rows at positions below seq_len[b] (in a decoding loop these are the
 * previous rounds' data: the preceding kernel is the layer's QKV projection, which writes Q and the block's own rows at
 * positions >= seq_len[b], or wf_kv_reserve, which only appends block-table entries), and that this preceding kernel, if
 * it uses programmatic launch completion itself, signals it only after its own dependency wait (this library's kernels do).
 * The attention launch then reads lengths and page ids and streams the K/V tiles that lie wholly below seq_len[b] while
 * the previous kernel is still running; only Q, the tree masks and the tiles holding the block's own rows wait for it.
 * Results are identical; a broken promise is a data race.  PAPER.md:133 (batch 1: the round is a chain of short launches). */
int wf_ctx_set_attn_early_kv(wf_ctx* ctx, int on);
/* Reproducible attention bits.  A (sequence, kv head) pair whose keys are split over several CTAs is merged from partial
 * (max, sum, O) triples.  on = 0 (default): in the stream-K shape the CTA that arrives last folds the others' partials into
 * its own, so the order of the floating-point merges (not the tolerance) depends on timing.  on = 1: every merge folds
 * the partials of a pair in key-range order, whoever arrives last: repeated calls on the same inputs give identical
 * bits (costs one extra round trip of the last arriver's partial through L2).  The cluster shape and every other call of
 * this library are order-fixed regardless.  Applies to wf_verify_attn and wf_verify_attn_tree. */
int wf_ctx_set_deterministic(wf_ctx* ctx, int on);

/* ---- (b) accept + bonus + entropy + route -------------------------------------------------------
 * PAPER.md:65, 75-81 (§3.3.1), 135; readings C1-C9.  Per sequence b (block rows r0..r0+gamma):
 *     g_i = argmax_v logits[r0+i][v] (lowest id on ties);  a = longest prefix with
 *     draft_tokens[r0+j] == g_{j-1}, j = 1..a;  bonus = g_a;  n_commit = a+1;
 *     H = Shannon entropy (nats) of softmax(logits[r0+a]);  route = AR(1) if H > tau else 0.
 * If target_kv != NULL, target_kv.seq_len[b] += n_commit[b].
 * tau: device fp32 [B], or [1] if tau_is_scalar.  logits rows must be finite or -inf (C23).
 * max_q_len: host upper bound on q_b (<= 64) that sizes the grid; a longer block is verified up to the bound and
 * raises WF_ERR_INVALID_ARG in the sticky status.
 * workspace: >= wf_accept_workspace_bytes(B * max_q_len, V); contents need no initialisation. */
int wf_accept_entropy_route(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens,
                            const int32_t* q_indptr, int B, int max_q_len, const float* tau,
                            int tau_is_scalar, int32_t* accept_len, int32_t* bonus_token,
                            float* entropy, int32_t* route, int32_t* n_commit,
                            wf_paged_kv* target_kv, void* workspace, size_t workspace_bytes,
                            void* stream);
size_t wf_accept_workspace_bytes(int sum_q, int V);
/* The same operation for callers that cannot allocate and do not want to carry a workspace (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the slice partials and completion counters live in one file-scope
 * device array inside the library (516 KB, held by every GPU that loads the library until the process exits).  The call makes
 * no cudaMalloc / cudaFree and calls no allocating routine; inputs and outputs are the caller's, exactly as above, and the
 * results are those of wf_accept_entropy_route bit for bit (same kernel).
 * Limits: B <= 1024 and B * max(max_q_len, 1) * ceil(V / 8192) <= 32768 (e.g. 64 sequences x 16 rows at V = 151936 use
 * 19456); anything larger returns WF_ERR_UNSUPPORTED_SHAPE with a message and launches nothing.
 * Every call on a device shares the array, which keeps the last call's contents: the call clears its counters itself (a
 * memset node in stream order); two calls that overlap on the GPU (different streams, or two contexts on one device) RACE on
 * it: keep them stream-ordered.  The first call on each device resolves the array's address (cudaGetSymbolAddress; no
 * allocation) and needs the context's device to be current: make that call before starting a stream capture. */
int wf_accept_entropy_route_static(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens,
                                   const int32_t* q_indptr, int B, int max_q_len, const float* tau,
                                   int tau_is_scalar, int32_t* accept_len, int32_t* bonus_token,
                                   float* entropy, int32_t* route, int32_t* n_commit,
                                   wf_paged_kv* target_kv, void* stream);

/* ---- drafter descriptor -------------------------------------------------------------------------
 * PAPER.md:119; readings C14-C18: every layer l projects the same hidden rows X with its own
 * W_K[l], W_V[l]: bf16 [hidden][n_kv_heads*head_dim] (K = X W; column c -> head c / D, lane c % D).
 * w_k_host_ptrs / w_v_host_ptrs: HOST arrays of n_layers DEVICE pointers.
 * backlog: bf16 [max_seqs][backlog_cap][hidden]; backlog_len: int32 [max_seqs] (caller-owned,
 * zero-initialised by the caller).  RoPE: rotate-half pairs (r, r + D/2), angle pos * theta^(-2r/D),
 * cos/sin table [max_pos][D/2] built in fp64 on the host at creation (C17). */
typedef struct {
  int n_layers, hidden, n_kv_heads, head_dim;
  float rope_theta;
  int max_pos;
  int backlog_cap;
} wf_drafter_shape;

int wf_drafter_create(wf_ctx* ctx, const wf_drafter_shape* shape,
                      const void* const* w_k_host_ptrs, const void* const* w_v_host_ptrs,
                      wf_paged_kv* drafter_kv, void* backlog, int32_t* backlog_len,
                      wf_drafter** out);
int wf_drafter_destroy(wf_drafter* d);

/* ---- (c) KV-only prefill (eager) ----------------------------------------------------------------
 * PAPER.md:119 (§3.4 "KV-only Prefill"), :206.  For each b in [0,B): rows t = 0..n_rows[b]-1 of the
 * block (hidden[q_indptr[b]+t]) are projected by every layer's W_K (+RoPE at position
 * p0+t, p0 = drafter_kv.seq_len[seq_ids[b]]) and W_V, rounded to bf16 (RNE) and written at logical
 * positions p0+t through the drafter's block table (pages reserved first, C24);
 * drafter_kv.seq_len[seq] += n_rows[b].  No attention, MLP or LM head runs.
 * seq_ids may be NULL (= identity).  n_rows[b] <= max_rows (host upper bound that sizes grids; a larger
 * n_rows[b] is clamped and raises WF_ERR_INVALID_ARG in the sticky status).  B <= 1024.
 * Every call of sections (c)/(d) is two launches: plan + operand pack, then the projection (which also
 * carries the enqueue copies and commits the backlog lengths). */
int wf_kv_only_prefill(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                       const int32_t* n_rows, const int32_t* seq_ids, int B, int max_rows,
                       void* stream);

/* ---- (d) Lazy Catch-up --------------------------------------------------------------------------
 * PAPER.md:117 (§3.4 "Lazy Catch-up"), :204.  enqueue: for each b with idle_mask[b] != 0 append rows
 * 0..n_rows[b]-1 of the block to the FIFO backlog of sequence seq_ids[b]; no projection work is
 * done.  If the rows would not fit (len + n > backlog_cap) that sequence's backlog is flushed first
 * (one batched prefill for all such sequences of the call), then the rows are enqueued: rows are
 * never dropped or reordered (C20).  n > backlog_cap sets WF_ERR_QUEUE_OVERFLOW and skips the rows.
 * If the forced flush cannot get its pages the sticky status becomes WF_ERR_OUT_OF_PAGES and the call
 * changes nothing (no row is written, no length moves).
 * flush: one batched KV-only prefill (same device code as (c)) over the whole backlog of every
 * sequence b in [0,B) with flush_mask[b] != 0 (NULL = all); backlog_len <- 0 for those.
 * Postcondition: the drafter cache is bit-identical to eager per-round appends. */
int wf_lazy_catchup_enqueue(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                            const int32_t* n_rows, const int32_t* seq_ids, const int32_t* idle_mask,
                            int B, int max_rows, void* stream);
int wf_lazy_catchup_flush(wf_ctx* ctx, wf_drafter* d, const int32_t* flush_mask, int B, void* stream);

/* ---- (c) + (d) fused: everything one round asks of a drafter, in ONE projection ---------------------
 * PAPER.md:117-119.  Per sequence b in [0,B), with idle = idle_mask && idle_mask[b], flush = flush_mask && flush_mask[b]:
 *   not idle          : the drafter is active for b: its backlog (normally empty) and then rows 0..n_rows[b]-1 of the
 *                       block are projected and appended (= wf_kv_only_prefill);
 *   idle and flush    : b switches to this drafter: its backlog and then this round's rows are projected and appended,
 *                       backlog_len <- 0 (= wf_lazy_catchup_enqueue followed by wf_lazy_catchup_flush, reading C21);
 *   idle, no flush    : the rows are enqueued (a backlog that would overflow is projected first, C20)
 *                       (= wf_lazy_catchup_enqueue).
 * All projected rows of the call share one plan, one operand pack and one projection: a drafter's weights are streamed
 * once per round instead of up to three times.  If the pages do not fit (WF_ERR_OUT_OF_PAGES) the call changes nothing.  A row's K/V bits are those of the separate calls (same device code,
 * per-row results do not depend on the call that carries them).  idle_mask / flush_mask may be NULL (none idle / none
 * flushed).  B <= 1024, max_rows <= 64 (and <= backlog_cap when idle_mask is given). */
int wf_lazy_catchup_round(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                          const int32_t* n_rows, const int32_t* seq_ids, const int32_t* idle_mask,
                          const int32_t* flush_mask, int B, int max_rows, void* stream);

/* ---- the switch, driven on the device by the router's output --------------------------------------------
 * PAPER.md:117 ("Upon preparing for a switch, the incoming drafter prefills its KV cache over all tokens accepted during
 * its inactivity as a single batched operation"), :65 (the chosen drafter drafts the next round); reading C21.
 * cur_drafter: device int32 [B], in/out: the drafter that drafted THIS round's block (WF_ROUTE_AR / WF_ROUTE_DIFFUSION).
 * route: device int32 [B]: this round's output of wf_accept_entropy_route (or wf_neural_route).  For drafter X with
 * route code c_X (drafter_ar: WF_ROUTE_AR, drafter_diffusion: WF_ROUTE_DIFFUSION) the call derives
 *     idle_X[b] = cur_drafter[b] != c_X,      flush_X[b] = idle_X[b] && route[b] == c_X
 * and does for BOTH drafters what wf_lazy_catchup_round(idle_X, flush_X) does for one, in the same two launches (the
 * tiles of both projections share one grid).  Afterwards cur_drafter[b] <- route[b] and, if next_q_len != NULL,
 * next_q_len[b] <- (route[b] == WF_ROUTE_AR ? q_len_ar : q_len_diffusion): the block length the chosen drafter will
 * bring next round; if switched != NULL, switched[b] <- route[b] where the sequence switched drafters this round
 * (route[b] != the old cur_drafter[b]), else -1: the selection wf_final_token_full takes.  No mask and no length crosses
 * the host.  Both drafters need the same hidden size and head_dim and distinct caches; other limits as
 * wf_lazy_catchup_round. */
int wf_switch_round(wf_ctx* ctx, wf_drafter* drafter_ar, wf_drafter* drafter_diffusion, const void* hidden,
                    const int32_t* q_indptr, const int32_t* n_rows, const int32_t* seq_ids, const int32_t* route,
                    int32_t* cur_drafter, int32_t* next_q_len, int32_t* switched, int q_len_ar, int q_len_diffusion,
                    int B, int max_rows, void* stream);

/* ---- (f3) the final backlog token in full -----------------------------------------------------------
 * PAPER.md:119 (§3.4: "we compute only the attention layer on tokens accepted by another drafter, processing only the
 * final token in full, so that its post-MLP hidden state can feed the next draft round"), :206; SURVEY.md §8(f) f3;
 * DESIGN.md readings F1-F6.
 *
 * wf_drafter_set_full_layer: gives the drafter the weights KV-only prefill skips, per layer l (HOST arrays of
 * n_layers DEVICE pointers, bf16, row vector times matrix as C18): W_Q [hidden][n_q_heads*head_dim],
 * W_O [n_q_heads*head_dim][hidden], W_up [hidden][ffn], W_down [ffn][hidden].  The library keeps its own repacked
 * copy (the caller's matrices are not read again) and activation scratch for max_tokens (<= 256) tokens per call.
 * hidden, n_q_heads*head_dim and ffn must be multiples of 128.  Synchronous; once per drafter.
 *
 * wf_final_token_full: for every b in [0,B) with (select == NULL || select[b] == select_code), n_rows[b] > 0 and a
 * non-empty cache: x = hidden[q_indptr[b] + n_rows[b] - 1] (the last row this round's catch-up prefill appended),
 * p = drafter_kv.seq_len[b] - 1 (its position; its K/V are in the cache already: call this AFTER the switch / flush
 * of the round), and for every drafter layer l (independent branches over the same x, reading C14 / F3)
 *     q = RoPE(x W_Q[l], p);  att = softmax(q K_l^T / sqrt(head_dim)) V_l over cache positions 0..p (GQA map C11);
 *     y = x + att W_O[l];     h_out[b][l] = y + GELU(y W_up[l]) W_down[l]     (tanh-form GELU, no norms, no biases).
 * h_out: bf16 [B][n_layers][hidden]; rows of unselected sequences are not written.  bf16 operands, fp32 accumulation,
 * bf16 RNE at q, att, the operand copies of y and GELU(.), and h_out; split-K sums in a fixed order (deterministic).
 * More selected sequences than max_tokens: the surplus (highest b) is skipped and the sticky status becomes
 * WF_ERR_INVALID_ARG.  Sequence b uses block-table row b (no seq_ids).  select is typically the `switched` output of
 * wf_switch_round with select_code = this drafter's route code, or a 0/1 mask with select_code = 1.
 * workspace: >= wf_final_token_workspace_bytes(d, B).  5 + n_layers launches, asynchronous on `stream`. */
int wf_drafter_set_full_layer(wf_ctx* ctx, wf_drafter* d, int n_q_heads, int ffn, int max_tokens,
                              const void* const* w_q_host_ptrs, const void* const* w_o_host_ptrs,
                              const void* const* w_up_host_ptrs, const void* const* w_down_host_ptrs);
size_t wf_final_token_workspace_bytes(const wf_drafter* d, int B);
int wf_final_token_full(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr, const int32_t* n_rows,
                        const int32_t* select, int select_code, int B, void* h_out, void* workspace,
                        size_t workspace_bytes, void* stream);

/* ---- (f1) WhiFlash-Neural routing policy --------------------------------------------------------
 * PAPER.md:87 (§3.3.2), :103-107 (decision rule), :325 (App. A architecture); readings N1-N6.
 * For each sequence b with a non-empty block: h = hidden_final[q_indptr[b] + accept_len[b]] (the target's
 * final hidden row of the last accepted position), dAL = <w2, GELU(W1 h + b1)> + b2 with the exact (erf)
 * GELU, route = WF_ROUTE_AR if dAL > tau else WF_ROUTE_DIFFUSION (ties -> diffusion).  An empty block
 * yields (0, WF_ROUTE_DIFFUSION).
 * hidden_final: bf16 [sum_q][d]; q_indptr int32 [B+1]; accept_len int32 [B] (device; the output of
 * wf_accept_entropy_route; NULL = row 0 of every block); w1: bf16 [m][d] (one row per hidden unit,
 * nn.Linear layout), b1: fp32 [m], w2: bf16 [m], b2: fp32 [1]; tau: fp32 [B] or [1]; delta_al: fp32 [B];
 * route: int32 [B].  All device pointers, 16-byte aligned; d % 8 == 0, m <= 8192, B <= 1024.
 * workspace: wf_neural_route_workspace_bytes(B, m) bytes.  bf16 inputs, fp32 accumulation in a fixed order
 * (deterministic).  Asynchronous on `stream`. */
size_t wf_neural_route_workspace_bytes(int B, int m);
int wf_neural_route(wf_ctx* ctx, const void* hidden_final, const int32_t* q_indptr, const int32_t* accept_len,
                    int B, int d, int m, const void* w1, const float* b1, const void* w2, const float* b2,
                    const float* tau, int tau_is_scalar, float* delta_al, int32_t* route,
                    void* workspace, size_t workspace_bytes, void* stream);

/* ---- (f2) tree verification: ancestor masks, tree attention, acceptance walk, path compaction -------
 * PAPER.md:65 ("an autoregressive drafter which produces a tree of candidate tokens ... returned to the
 * target model for parallel verification"), :39, :317/:327 (depth 8, top-k 10, 60 draft tokens);
 * DESIGN.md readings T1-T5; SURVEY.md §8(f) f2.
 * Block layout (T1): row 0 of sequence b's block is the committed root, rows 1..n_b-1 are tree nodes in
 * topological order: parent[r0_b + i] in [0, i) (an index INSIDE the block), parent[r0_b] = -1, n_b <= 64.
 * Node i's K/V sit at cache position seq_len[b] + i.  A chain block is parent[i] = i - 1, so one call
 * serves batches that mix trees and chains.  All pointers are device pointers; every call is asynchronous
 * on `stream`.
 *
 * wf_tree_masks: parent int32 [sum_q] -> tree_mask uint64 [sum_q], bit j of row i set iff node j is i or
 * an ancestor of i (T2).  Once per round: every layer uses the same masks.  A pointer that breaks T1
 * raises WF_ERR_INVALID_ARG in the sticky device status (wf_poll_status) and leaves that row its own bit.
 *
 * wf_verify_attn_tree: as wf_verify_attn, but row i of sequence b sees keys 0..seq_len[b]-1 and
 * seq_len[b] + j for the set bits j of tree_mask[r0_b + i].  max_nodes <= 64;
 * B * ceil(max_nodes * group / 128) <= 1024.  workspace: wf_verify_attn_workspace_bytes(.., max_nodes).
 *
 * wf_accept_tree_entropy_route: as wf_accept_entropy_route with the greedy tree walk (T3): from the root,
 * step to the lowest-index child whose token equals the argmax of the current node's logits, until none
 * does.  accept_len = steps, bonus_token = argmax at the last node, entropy / route from that node's
 * logits (T4), n_commit = accept_len + 1, path[b][0..accept_len] = the nodes visited, -1 beyond
 * (path: int32 [B][path_stride], path_stride >= max_nodes).  The target cache length is NOT advanced:
 *
 * wf_kv_compact_path: for every layer of `kv` move the K/V rows of path[b][k] from position
 * seq_len[b] + path[b][k] to seq_len[b] + k (k = 1..n_commit[b]-1), then seq_len[b] += n_commit[b] (T5).
 * Rows are moved as if every source were read before any destination is written.  A path entry outside
 * [k, 64) raises WF_ERR_INVALID_ARG in the sticky device status and moves nothing for that step. */
int wf_tree_masks(wf_ctx* ctx, const int32_t* parent, const int32_t* q_indptr, int B, int max_nodes,
                  uint64_t* tree_mask, void* stream);
int wf_verify_attn_tree(wf_ctx* ctx, const wf_paged_kv* kv, int layer, const void* q, const int32_t* q_indptr,
                        const uint64_t* tree_mask, int B, int n_q_heads, int max_nodes, float sm_scale,
                        void* out, void* workspace, size_t workspace_bytes, void* stream);
int wf_accept_tree_entropy_route(wf_ctx* ctx, const float* logits, int V, const int32_t* node_tokens,
                                 const int32_t* parent, const int32_t* q_indptr, int B, int max_nodes,
                                 const float* tau, int tau_is_scalar, int32_t* accept_len,
                                 int32_t* bonus_token, float* entropy, int32_t* route, int32_t* n_commit,
                                 int32_t* path, int path_stride, void* workspace, size_t workspace_bytes,
                                 void* stream);
int wf_kv_compact_path(wf_paged_kv* kv, const int32_t* path, int path_stride, const int32_t* n_commit, int B,
                       void* stream);

/* ---- (f4) stochastic acceptance: speculative sampling with temperature ----------------------------
 * PAPER.md:19 (the speculative-decoding rule of the papers cited there), :79-81 (under sampling the
 * softmax already exists and the router reads its entropy); readings S1-S5; SURVEY.md §8(f) f4.
 * Chain block layout as wf_accept_entropy_route.  p_i = softmax(logits[r0+i] / temperature).
 * draft_q: fp32 [sum_q][V], row r0+i = the drafter's distribution for the token after row i, or NULL for a
 * deterministic drafter (one-hot at the proposed token).  u_accept: fp32 [sum_q], u_sample: fp32 [B],
 * uniforms in [0, 1) drawn by the caller (row r0 of u_accept is unused).
 *     draft j (j = 1..gamma) is accepted iff u_accept[r0+j] < min(1, p_{j-1}(x_j) / q_{j-1}(x_j)) (q = 0: ratio 1);
 *     accept_len = a = drafts accepted before the first rejection; n_commit = a + 1;
 *     token = inverse CDF at u_sample[b], in vocabulary order, of max(0, p_a - q_a) if a < gamma (of p_a if
 *     that is empty), of p_a if a = gamma: the smallest v whose cumulative mass exceeds u * total;
 *     entropy = H(p_a) in nats, route = AR iff entropy > tau.
 * If target_kv != NULL, target_kv.seq_len[b] += n_commit[b].  Probabilities are evaluated in fp32 and accumulated
 * in fp64; workspace as wf_accept_workspace_bytes(B * max_q_len, V).  Asynchronous on `stream`. */
int wf_accept_sample_entropy_route(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens,
                                   const int32_t* q_indptr, int B, int max_q_len, float temperature,
                                   const float* draft_q, const float* u_accept, const float* u_sample,
                                   const float* tau, int tau_is_scalar, int32_t* accept_len, int32_t* token,
                                   float* entropy, int32_t* route, int32_t* n_commit, wf_paged_kv* target_kv,
                                   void* workspace, size_t workspace_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* WHIFLASH_H_ */

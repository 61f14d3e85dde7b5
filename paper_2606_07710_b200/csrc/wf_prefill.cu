// (c) KV-only Prefill and (d) Lazy Catch-up.
// PAPER.md:117-119 (§3.4), :204-206; readings C14-C22.
//
// One device path serves eager prefill, flush and the forced flush inside enqueue (bit-identity of
// lazy vs eager):
//   plan kernel (1 CTA)  : which rows go where.  Compacts the rows of the call into a row table
//                          (source pointer, RoPE position, physical page*16+slot), reserves pages in
//                          the drafter's block table (C24) and advances seq_len / backlog_len.
//   pack kernel          : the call's rows -> the shared-memory image of the X operand, k-block by k-block
//                          (K-major, 128-byte swizzle), so that a projection CTA fetches a stage's X with one
//                          bulk copy instead of gathering rows with its own threads.
//   projection kernel    : one CTA per (layer, K|V, kv head): out^T[D, tokens] = W^T[D, hidden] . X^T on tcgen05
//                          (UMMA 128 x tokens x 16, bf16 in, fp32 accumulators in TMEM; swapped operands, so an
//                          MMA costs tokens/2 cycles).  W was repacked once at wf_drafter_create into stage
//                          images (MN-major, 128-byte swizzle): a stage is one cp.async.bulk for W and one per X
//                          k-block, completing on an mbarrier ring.  Epilogue: tcgen05.ld, transpose through
//                          shared memory, RoPE (fp32, host-built fp64 table) on K tiles, bf16 RNE, 16-byte
//                          stores straight into the paged pool.
// A row's bits do not depend on M, on its position in the call or on the call that carries it: one code
// path, a fixed K order, a split-K factor fixed per drafter (partials summed in split order by the last CTA to
// arrive); an accumulator column depends only on its own X row.
#include <cuda.h>
#include <math.h>

#include <new>
#include <type_traits>
#include <vector>

#include "wf_internal.cuh"
#include "wf_sm100.cuh"

namespace {

constexpr int PF_BLOCK_M = 128;         // UMMA M
constexpr int PF_BLOCK_K = 64;          // one 128-byte swizzle row of bf16
constexpr int PF_KSUB = 2;              // 64-wide k-blocks per pipeline stage: halves the per-stage hand-offs of the one-thread loops
constexpr int PF_MAX_MT = 2;            // m-tiles per pass (TMEM columns = PF_MAX_MT * D)
constexpr int PF_THREADS = 192;         // warp 0: bulk-copy producer, warp 1: MMA, warps 2-5: epilogue (+ enqueue, commit)
constexpr int PF_SMEM_BUDGET = 200 * 1024;
constexpr int PF_SMEM_LAUNCH = PF_SMEM_BUDGET + 1024;   // UMMA reads n_pad (multiple of 16) rows of an X stage that holds a
                                                        // multiple of 8: the last stage's surplus rows lie behind the ring
constexpr int PF_W_PRE_BYTES = 128 * 1024;   // weight stages that are prefetched ahead of the dependency wait
constexpr int PP_THREADS = 256;         // plan + pack kernel
constexpr int PP_MAX_B = KV_RESERVE_SMEM;   // sequences per call (the per-sequence plan lives in shared memory)
constexpr int PP_MAX_PACK_CTAS = 296;   // pack CTAs per drafter: two per SM
using RowEntry = wf_row_entry;

// ---- kernel 1 of 2: plan + pack ------------------------------------------------------------------
// What one call asks of a drafter, per sequence b (seq = seq_ids ? seq_ids[b] : b, len = its backlog length, add = n_rows[b]):
//   EAGER   : the block rows are projected (wf_kv_only_prefill).
//   FLUSH   : the backlog of every flagged sequence is projected (wf_lazy_catchup_flush).
//   ENQUEUE : the block rows of idle sequences are enqueued; a backlog they would overflow is projected first (C20).
//   ROUND   : everything a round asks of the drafter in ONE projection: active sequences (not idle) and sequences that
//             switch to it (idle and flush) get backlog + block rows projected; the others are enqueued as in ENQUEUE.
//             idle / flush come from host-planned masks (wf_lazy_catchup_round) or, device-driven, from the router's
//             output: idle = cur[b] != code, flush = idle && route[b] == code (wf_switch_round, reading C21).
// Every CTA of the launch derives the same per-sequence plan in shared memory from the device-resident inputs (they are
// read-only in this kernel: lengths that the call changes are committed by kernel 2).  CTA 0 of a drafter is its PLANNER:
// reserves pages (C24), writes the row table (RoPE position, physical page*16+slot), the enqueue offsets and the new
// backlog lengths, and advances the cache length.  The other CTAs PACK: row r of the call -> the shared-memory image
// of the X operand, k-block by k-block (xpack[hidden/64][m_pad][128 B], K-major, 16-byte chunks XOR-swizzled with r & 7),
// so that a projection CTA fetches a stage's X with one bulk copy.  Two drafters share one launch (blockIdx picks).
enum PlanMode { PLAN_EAGER = 0, PLAN_FLUSH = 1, PLAN_ENQUEUE = 2, PLAN_ROUND = 3 };

struct PlanJob {
  int mode, B, hidden, cap, max_pos, row_cap, max_rows;
  int code;                             // ROUND, device-driven: this drafter's route code (WF_ROUTE_AR / WF_ROUTE_DIFFUSION)
  const __nv_bfloat16* hidden_rows;     // block hidden states [sum_q][hidden]
  const int32_t* q_indptr;
  const int32_t* n_rows;
  const int32_t* seq_ids;               // NULL = identity
  const int32_t* idle_mask;             // ENQUEUE / ROUND (host masks; NULL = none idle)
  const int32_t* flush_mask;            // FLUSH (NULL = all) / ROUND (host masks; NULL = none)
  const int32_t* route;                 // ROUND, device-driven (route != NULL): the router's output this round
  const int32_t* cur;                   //                       the drafter that drafted this round's block
  const __nv_bfloat16* backlog;         // [max_seqs][cap][hidden]
  const int32_t* backlog_len;
  KvView kv;
  RowEntry* rows;
  int32_t* m_total;
  int32_t* enq_base;                    // [B] backlog offset at which kernel 2 enqueues the block rows, -1 = none
  int32_t* new_blen;                    // [B] backlog length kernel 2 commits, -1 = unchanged
  uint8_t* xpack;
  int* status;
};

struct PlanPackParams {
  PlanJob job[2];
  int n_jobs, ctas_job0;                // CTAs [0, ctas_job0) serve job 0, the rest job 1
};

__global__ void __launch_bounds__(PP_THREADS) wf_plan_pack_kernel(const __grid_constant__ PlanPackParams pp) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  __shared__ int s_n[PP_MAX_B], s_nb[PP_MAX_B], s_off[PP_MAX_B + 1], s_eb[PP_MAX_B], s_nl[PP_MAX_B];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = PP_THREADS >> 5;
  wf_pdl_wait();
  wf_pdl_trigger();
  const int jb = (int)blockIdx.x >= pp.ctas_job0 ? 1 : 0;
  const PlanJob& p = pp.job[jb];
  const int c = (int)blockIdx.x - (jb ? pp.ctas_job0 : 0);
  const int n_pack = (jb ? (int)gridDim.x - pp.ctas_job0 : pp.ctas_job0) - 1;
  const bool planner = c == 0;
  auto seq_of = [&](int b) { return p.seq_ids ? p.seq_ids[b] : b; };
  // ---- the per-sequence plan (every CTA, identical) ----
  for (int b = tid; b < p.B; b += PP_THREADS) {
    const int sq = seq_of(b);
    const int len = p.cap > 0 ? p.backlog_len[sq] : 0;
    int add = p.mode == PLAN_FLUSH ? 0 : p.n_rows[b];
    if (add > p.max_rows || add < 0) {                         // the host bound sizes the launch: clamp, never overrun
      if (planner) wf_raise(p.status, (int)WF_ERR_INVALID_ARG);
      add = min(max(add, 0), p.max_rows);
    }
    bool idle = false, fl = false;
    if (p.mode == PLAN_ROUND) {
      if (p.route) { idle = p.cur[b] != p.code; fl = idle && p.route[b] == p.code; }
      else { idle = p.idle_mask && p.idle_mask[b]; fl = p.flush_mask && p.flush_mask[b]; }
    } else if (p.mode == PLAN_ENQUEUE) {
      idle = p.idle_mask[b] != 0;
    } else if (p.mode == PLAN_FLUSH) {
      fl = !p.flush_mask || p.flush_mask[b];
    }
    int n_back = 0, n_blk = 0, n_enq = 0;
    if (p.mode == PLAN_EAGER) n_blk = add;
    else if (p.mode == PLAN_FLUSH) n_back = fl ? len : 0;
    else {
      const bool project_block = p.mode == PLAN_ROUND && (!idle || fl);
      n_enq = (idle && !project_block) ? add : 0;
      if (n_enq > p.cap) {                                     // one round's rows alone exceed the cap: skipped (R1)
        if (planner) wf_raise(p.status, (int)WF_ERR_QUEUE_OVERFLOW);
        n_enq = 0;
      }
      // the backlog goes first whenever anything of this sequence is projected (FIFO), or when the enqueue would overflow
      n_back = (project_block || (n_enq > 0 && len + n_enq > p.cap)) ? len : 0;
      n_blk = project_block ? add : 0;
    }
    s_nb[b] = n_back;
    s_n[b] = n_back + n_blk;
    s_eb[b] = n_enq > 0 ? (n_back > 0 ? 0 : len) : -1;
    s_nl[b] = (p.mode == PLAN_EAGER || p.cap == 0) ? -1 : (n_back > 0 ? 0 : len) + n_enq;
  }
  if (tid == 0) s_carry = 0;
  __syncthreads();
  auto nothing = [&]() {                                       // planner: the call projects and enqueues nothing
    if (tid == 0) *p.m_total = 0;
    for (int b = tid; b < p.B; b += PP_THREADS) { p.enq_base[b] = -1; p.new_blen[b] = -1; }
  };
  // pages first (C24: ascending b, consecutive ring entries); nothing is written if they do not fit
  if (planner) {
    const bool ok = kv_reserve_block(p.kv, p.B, [&](int b) { return s_n[b]; }, seq_of, p.status);
    if (!ok) { nothing(); return; }
  }
  // exclusive scan of the row counts -> first compact row of each sequence
  for (int base = 0; base < p.B; base += PP_THREADS) {
    const int b = base + tid;
    const int n = b < p.B ? s_n[b] : 0;
    int x = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) s_warp[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int w = lane < nw ? s_warp[lane] : 0;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, w, d);
        if (lane >= d) w += y;
      }
      s_warp[lane] = w;
    }
    __syncthreads();
    if (b < p.B) s_off[b] = s_carry + (wid ? s_warp[wid - 1] : 0) + x - n;
    __syncthreads();
    if (tid == 0) s_carry += s_warp[nw - 1];
    __syncthreads();
  }
  const int total = s_carry;
  if (total > p.row_cap) {                                     // host bounds make this unreachable
    if (planner) { if (tid == 0) wf_raise(p.status, (int)WF_ERR_INVALID_ARG); nothing(); }
    return;
  }
  if (planner) {
    // row table: one warp per sequence
    for (int b = wid; b < p.B; b += nw) {
      const int sq = seq_of(b);
      const int n = s_n[b], off = s_off[b];
      const int p0 = p.kv.seq_len[sq];
      for (int t = lane; t < n; t += 32) {
        const int pos = p0 + t;
        if (pos >= p.max_pos) wf_raise(p.status, (int)WF_ERR_INVALID_ARG);
        const int page = p.kv.block_table[(size_t)sq * p.kv.max_pages_per_seq + (pos >> 4)];
        RowEntry e;
        e.pos = min(pos, p.max_pos - 1);
        e.page_slot = page * 16 + (pos & 15);
        p.rows[off + t] = e;
      }
      __syncwarp();
      if (lane == 0) {
        p.enq_base[b] = s_eb[b];
        p.new_blen[b] = s_nl[b];
        if (n > 0) p.kv.seq_len[sq] = p0 + n;
      }
    }
    if (tid == 0) *p.m_total = total;
    return;
  }
  // ---- pack: rows c-1, c-1+n_pack, ... of the call ----
  const int m_pad = (total + 7) & ~7;
  const size_t kb_stride = (size_t)m_pad * 128;
  for (int r = c - 1; r < total; r += n_pack) {
    int lo = 0, hi = p.B;                                      // the sequence whose rows hold r: largest b with off[b] <= r
    while (hi - lo > 1) {                                      // and n[b] > 0 (empty sequences share their successor's offset)
      const int mid = (lo + hi) >> 1;
      if (s_off[mid] <= r) lo = mid; else hi = mid;
    }
    const int b = lo, t = r - s_off[b];
    const int sq = seq_of(b);
    const __nv_bfloat16* srow = t < s_nb[b] ? p.backlog + ((size_t)sq * p.cap + t) * p.hidden
                                            : p.hidden_rows + (size_t)(p.q_indptr[b] + t - s_nb[b]) * p.hidden;
    const uint4* src = reinterpret_cast<const uint4*>(srow);
    uint8_t* dst = p.xpack + (size_t)r * 128;
    for (int q = tid; q < p.hidden / 8; q += PP_THREADS) {   // 16-byte chunk q of the row -> k-block q/8, chunk q%8
      const uint4 v = __ldg(src + q);
      *reinterpret_cast<uint4*>(dst + (size_t)(q >> 3) * kb_stride + (((q & 7) ^ (r & 7)) << 4)) = v;
    }
  }
}

// ---- the projection kernel ------------------------------------------------------------------
constexpr int PF_MAX_STAGES = 12;

// One-time repack of a drafter's weights (wf_drafter_create) into the exact shared-memory image of a W stage:
// tile (layer, K|V, head) x k-block of 64 rows -> D/64 column halves x [64 k][128 B], 16-byte chunks XOR-swizzled
// with (k & 7) (the 128-byte swizzle the MN-major UMMA descriptor expects).  A stage is then ONE contiguous
// cp.async.bulk of 64*D*2 bytes instead of 64*D/64 strided 128-byte TMA rows out of a [hidden][Hkv*D] matrix.
__global__ void wf_pack_w_kernel(const __nv_bfloat16* __restrict__ w, uint8_t* __restrict__ dst, int hidden, int n_cols, int D) {
  // grid (hidden/64, n_cols/D); dst points at this (layer, K|V) block: [head][kb][D/64][64][128 B]
  const int kb = blockIdx.x, head = blockIdx.y, n_kb = hidden / 64;
  uint8_t* out = dst + ((size_t)head * n_kb + kb) * (64 * D * 2);
  for (int i = threadIdx.x; i < 64 * D / 8; i += blockDim.x) {       // one 16-byte chunk per step
    const int k = i / (D / 8), c16 = i % (D / 8);                       // row of the k-block, chunk of the D columns
    const int j = c16 >> 3, cc = c16 & 7;                               // column half, chunk inside the 128-byte row
    const uint4 v = *reinterpret_cast<const uint4*>(w + (size_t)(kb * 64 + k) * n_cols + head * D + c16 * 8);
    *reinterpret_cast<uint4*>(out + j * 8192 + k * 128 + ((cc ^ (k & 7)) << 4)) = v;
  }
}

// ---- kernel 2 of 2: projection + enqueue + commit ----------------------------------------------------
struct GemmJob {
  const uint8_t* wpack;                 // [n_layers][2][Hkv][hidden/64][64 * D * 2 B] pre-swizzled W stages
  const uint8_t* xpack;                 // [hidden/64][m_pad][128 B] pre-swizzled X k-blocks of this call (kernel 1)
  const RowEntry* rows;
  const int32_t* m_total;
  const float2* rope;                   // [max_pos][D/2] (cos, sin)
  __nv_bfloat16* k_pool;
  __nv_bfloat16* v_pool;
  int hidden, n_kv_heads, num_pages;
  // split-K (fixed per drafter, so the summation order never depends on the call): CTA = (tile, split), partials
  // [tile][split][row_cap][D] fp32, one self-resetting counter per (tile, pass)
  int n_split, row_cap, max_pass;
  float* ws_part;
  unsigned int* split_cnt;
  // enqueue (ENQUEUE / ROUND): block row t of sequence b -> backlog[seq][enq_base[b] + t]; commit: backlog lengths
  const __nv_bfloat16* hidden_rows;
  const int32_t* q_indptr;
  const int32_t* n_rows;
  const int32_t* seq_ids;
  const int32_t* enq_base;              // NULL: the call enqueues nothing
  const int32_t* new_blen;              // NULL: the call changes no backlog length
  __nv_bfloat16* backlog;
  int32_t* backlog_len;
  int B, cap, max_rows;
  // device-driven switch (wf_switch_round; job 0 commits): cur <- route, next block length per sequence
  const int32_t* route;
  int32_t* cur;
  int32_t* next_q_len;                  // nullable
  int32_t* switched;                    // nullable: route[b] where it differs from cur[b] (a switch), else -1
  int q_len_ar, q_len_diffusion;
};

struct GemmParams {
  GemmJob job[2];
  int n_jobs, ctas_job0;
};

template <int D>
__global__ void __launch_bounds__(PF_THREADS, 1) wf_prefill_gemm_kernel(const __grid_constant__ GemmParams gp) {
  // Swapped operands: out^T[D x tokens] = W^T[D x hidden] . X^T[hidden x tokens].  The head's D output columns are the
  // UMMA M dimension (always issued as M = 128; for D = 64 the upper 64 lanes compute on whatever follows in the
  // ring and are never read), the call's tokens are the UMMA N dimension (padded to 16).  An MMA then costs
  // max(128, M) * N / 256 = tokens / 2 cycles instead of 64: small calls stop being tensor-issue bound, and there
  // is still ONE code path for every token count (lazy == eager bit for bit).
  constexpr int W_SUB = PF_BLOCK_K * D * 2;               // one 64-row k-block of the W tile: D/64 x [64 k][128 B]
  constexpr int W_BYTES = PF_KSUB * W_SUB;                // W stage, contiguous in wpack
  constexpr int N_MAX = PF_MAX_MT * PF_BLOCK_M;           // tokens per pass (TMEM columns)
  constexpr uint32_t TMEM_COLS = N_MAX;                   // 256: a power of two >= 32
  extern __shared__ __align__(1024) uint8_t smem[];
  // Two rings: W stages (32 KB at D = 128, contiguous in the packed image) and X stages (the call's rows, size known only
  // after the dependency wait).  The W ring sits at offset 0 with a depth that is fixed for its first PF_W_PRE slots
  // whatever the call's row count turns out to be, so those slots are filled BEFORE griddepcontrol.wait: the weights are
  // constants, and under programmatic dependent launch this kernel's CTAs are resident while the plan + pack kernel (a few
  // small CTAs) still runs: the head of the weight stream (all of it for a 1-layer drafter) overlaps the predecessor.
  __shared__ __align__(8) uint64_t w_full[PF_MAX_STAGES], w_empty[PF_MAX_STAGES], x_full[PF_MAX_STAGES], x_empty[PF_MAX_STAGES],
      s_acc_full, s_acc_empty;
  __shared__ uint32_t s_tmem;
  __shared__ int s_last;
  constexpr int W_PRE = PF_W_PRE_BYTES / W_BYTES;          // W slots valid under every layout

  const int jb = (int)blockIdx.x >= gp.ctas_job0 ? 1 : 0;
  const GemmJob& p = gp.job[jb];
  const int cta = (int)blockIdx.x - (jb ? gp.ctas_job0 : 0);
  const int n_ctas = jb ? (int)gridDim.x - gp.ctas_job0 : gp.ctas_job0;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int tile = cta / p.n_split;                    // (layer, K|V, kv head)
  const int split = cta % p.n_split;                   // this CTA's share of the k-blocks
  const int layer = tile / (2 * p.n_kv_heads);
  const int is_v = (tile / p.n_kv_heads) & 1;
  const int head = tile % p.n_kv_heads;
  const int n_kb_tile = p.hidden / (PF_KSUB * PF_BLOCK_K);   // pipeline stages of a whole tile
  const int n_kb = n_kb_tile / p.n_split;                    // stages this CTA runs per pass (n_split divides them)
  const int kb0 = split * n_kb;
  const int n_pre = min(n_kb, W_PRE);
  if (tid == 0) {
    for (int i = 0; i < PF_MAX_STAGES; ++i) {
      mbar_init(smem_u32(&w_full[i]), 1); mbar_init(smem_u32(&w_empty[i]), 1);
      mbar_init(smem_u32(&x_full[i]), 1); mbar_init(smem_u32(&x_empty[i]), 1);
    }
    mbar_init(smem_u32(&s_acc_full), 1);
    mbar_init(smem_u32(&s_acc_empty), 128);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(smem_u32(&s_tmem), TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = s_tmem;
  const uint8_t* w_tile = p.wpack + ((size_t)tile * n_kb_tile + kb0) * W_BYTES;   // tile = (layer, K|V, head), packed in that order
  if (warp == 0 && elect_one()) {
    for (int s2 = 0; s2 < n_pre; ++s2) {
      mbar_arrive_expect_tx(smem_u32(&w_full[s2]), W_BYTES);
      bulk_load(smem_u32(smem) + s2 * W_BYTES, w_tile + (size_t)s2 * W_BYTES, W_BYTES, smem_u32(&w_full[s2]));
    }
  }
  __syncwarp();
  wf_pdl_wait();
  wf_pdl_trigger();
  const int M = *p.m_total;

  // Enqueue and commit ride on this kernel (kernel 1 has packed the projection's operand, backlog rows included, so
  // the backlog may be overwritten; nobody in this kernel reads a length).  The (sequence, row) pairs are dealt
  // round-robin to the drafter's CTAs; its CTA 0 commits the backlog lengths the planner decided, and job 0's CTA 0
  // the switch itself (cur <- route, the next block's length).  The epilogue warps do it while the operands stream.
  auto enqueue_commit = [&](int t0, int nt) {
    if (p.enq_base) {
      for (int pair = cta; pair < p.B * p.max_rows; pair += n_ctas) {
        const int b = pair / p.max_rows, t = pair % p.max_rows;
        const int base = p.enq_base[b];
        if (base < 0 || t >= p.n_rows[b]) continue;
        const int sq = p.seq_ids ? p.seq_ids[b] : b;
        const uint4* src = reinterpret_cast<const uint4*>(p.hidden_rows + (size_t)(p.q_indptr[b] + t) * p.hidden);
        uint4* dst = reinterpret_cast<uint4*>(p.backlog + ((size_t)sq * p.cap + base + t) * p.hidden);
        for (int i = t0; i < p.hidden / 8; i += nt) dst[i] = __ldg(src + i);
      }
    }
    if (cta == 0) {
      if (p.new_blen)
        for (int b = t0; b < p.B; b += nt) {
          const int nl = p.new_blen[b];
          if (nl >= 0) p.backlog_len[p.seq_ids ? p.seq_ids[b] : b] = nl;
        }
      if (p.route && jb == 0)
        for (int b = t0; b < p.B; b += nt) {
          const int r = p.route[b];
          if (p.switched) p.switched[b] = r != p.cur[b] ? r : -1;
          p.cur[b] = r;
          if (p.next_q_len) p.next_q_len[b] = r == WF_ROUTE_AR ? p.q_len_ar : p.q_len_diffusion;
        }
    }
  };
  const int n_pass = (M + N_MAX - 1) / N_MAX;
  if (M == 0) {
    // nothing to project for this drafter: let the prefetched weight stages land (the CTA's shared memory must outlive the
    // copies), give the TMEM columns back, do the enqueue / commit work and leave
    if (warp == 0) for (int s2 = 0; s2 < n_pre; ++s2) mbar_wait(smem_u32(&w_full[s2]), 0);
    if (warp == 1) tmem_dealloc(tmem_base, TMEM_COLS);
    enqueue_commit(tid, PF_THREADS);
    return;
  }

  // An X stage holds only the rows that exist (8-row swizzle atoms); UMMA reads n_pad (multiple of 16) rows from
  // its start, the few surplus rows feed accumulator columns nobody reads.  Layout: W ring (n_sw stages) | X ring (n_sx).
  const int m_first = min(M, N_MAX);
  const int x_sub = ((m_first + 7) / 8) * 1024;          // one 64-wide k-block of the X operand
  // The X ring is cut into single 64-wide k-blocks (a W stage spans PF_KSUB of them): at 256 rows a k-block is 32 KB and the
  // 72 KB beside the four prefetched W stages hold two of them, so the load of one overlaps the MMAs of the other (with
  // whole stages as ring units a call of >= 128 rows had ONE X stage: load and MMA took turns, 0.23 us per row).
  // Small calls keep whole stages as ring units (xg = PF_KSUB k-blocks per slot): every hand-off costs the one-thread loops a
  // barrier round trip, and there is room for many slots anyway.
  const int n_sw = (PF_SMEM_BUDGET - PF_W_PRE_BYTES - W_BYTES) >= 2 * PF_KSUB * x_sub ? W_PRE + 1 : W_PRE;
  const int xg = (PF_SMEM_BUDGET - n_sw * W_BYTES) >= 2 * PF_KSUB * x_sub ? PF_KSUB : 1;   // k-blocks per X ring slot
  const int x_slot = xg * x_sub;
  const int n_sx = max(PF_KSUB / xg, min(PF_MAX_STAGES, (PF_SMEM_BUDGET - n_sw * W_BYTES) / x_slot));
  uint8_t* w_base = smem;
  uint8_t* x_base = smem + (size_t)n_sw * W_BYTES;         // 1024-aligned: W_BYTES is a multiple of 1024

  if (warp == 0) {
    // ===== bulk-copy producer: per stage ONE contiguous copy of the pre-swizzled W k-blocks and one per packed X
    //       k-block (wf_plan_pack_kernel): no thread touches operand bytes.  Stage indices, phases and addresses advance
    //       incrementally: a runtime division per stage in a one-thread loop costs more than the MMAs it feeds.
    //       The whole warp runs the loop (warp-uniform control flow) and one elected lane issues: ptxas then emits
    //       straight-line UBLKCP / UTCHMMA instead of a divergence loop around every instruction. =====
    {
      const size_t x_kb_stride = (size_t)((M + 7) & ~7) * 128;
      const uint32_t wf0 = smem_u32(&w_full[0]), we0 = smem_u32(&w_empty[0]), xf0 = smem_u32(&x_full[0]), xe0 = smem_u32(&x_empty[0]);
      const uint32_t x0 = smem_u32(x_base), w0 = smem_u32(w_base);
      int sw = 0, sx = 0, kw = 0;                        // W slot, X slot, W stages issued so far (the first n_pre are in flight)
      uint32_t phw = 1, phx = 1;                         // parities to wait for on the empty barriers: the rings start empty
      auto produce = [&](auto xg_c) {
      constexpr int XG = decltype(xg_c)::value;              // compile-time copy of xg: the one-thread loop stays straight-line
      for (int pass = 0; pass < n_pass; ++pass) {
        const int rows_here = min(M - pass * N_MAX, N_MAX);
        const uint32_t x_bytes = (uint32_t)((rows_here + 7) / 8) * 1024;
        const uint8_t* x_src = p.xpack + (size_t)pass * N_MAX * 128 + (size_t)kb0 * PF_KSUB * x_kb_stride;
        const uint8_t* w_kb = w_tile;
        // the epilogue of the previous pass transposes through the rings: do not refill them before it is done
        if (pass > 0) mbar_wait(smem_u32(&s_acc_empty), (pass - 1) & 1);
        for (int kb = 0; kb < n_kb; ++kb, ++kw) {
          if (kw >= n_pre) {
            mbar_wait(we0 + 8 * sw, phw);
            if (elect_one()) {
              mbar_arrive_expect_tx(wf0 + 8 * sw, W_BYTES);
              bulk_load(w0 + sw * W_BYTES, w_kb, W_BYTES, wf0 + 8 * sw);
            }
          }
#pragma unroll
          for (int u = 0; u < PF_KSUB; u += XG) {
            mbar_wait(xe0 + 8 * sx, phx);
            if (elect_one()) {
              mbar_arrive_expect_tx(xf0 + 8 * sx, XG * x_bytes);
#pragma unroll
              for (int uu = 0; uu < XG; ++uu)
                bulk_load(x0 + sx * x_slot + uu * x_sub, x_src + (u + uu) * x_kb_stride, x_bytes, xf0 + 8 * sx);
            }
            __syncwarp();
            if (++sx == n_sx) { sx = 0; phx ^= 1; }
          }
          w_kb += W_BYTES;
          x_src += PF_KSUB * x_kb_stride;
          if (++sw == n_sw) { sw = 0; phw ^= 1; }
        }
      }
      };
      if (xg == 1) produce(std::integral_constant<int, 1>{}); else produce(std::integral_constant<int, PF_KSUB>{});
    }
  } else if (warp == 1) {
    // ===== MMA issuer: one thread drives the tensor core for the CTA.  Descriptors are built once and advanced by
    //       constant offsets.  A = W tile (MN-major, 128-byte swizzle), B = X rows (K-major, 128-byte swizzle). =====
    {
      const uint64_t dw0 = umma_desc(smem_u32(w_base), 8192, 1024);        // MN-major: 64-column halves 8 KB apart
      const uint64_t dx0 = umma_desc(smem_u32(x_base), 16, 1024);          // K-major
      const uint32_t wf0 = smem_u32(&w_full[0]), we0 = smem_u32(&w_empty[0]), xf0 = smem_u32(&x_full[0]), xe0 = smem_u32(&x_empty[0]);
      const uint64_t dw_step = (uint64_t)(W_BYTES >> 4), dx_step = (uint64_t)(x_slot >> 4);
      int sw = 0, sx = 0;
      uint32_t phw = 0, phx = 0;
      uint64_t dw = dw0, dx = dx0;
      auto issue = [&](auto xg_c) {
      constexpr int XG = decltype(xg_c)::value;
      for (int pass = 0; pass < n_pass; ++pass) {
        const int rows_here = min(M - pass * N_MAX, N_MAX);
        const uint32_t idesc = umma_idesc_mn_k(128, (rows_here + 15) & ~15);
        if (pass > 0) { mbar_wait(smem_u32(&s_acc_empty), (pass - 1) & 1); tc_fence_after(); }
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(wf0 + 8 * sw, phw);
          // k-block u of the stage: W k-block u (W_SUB apart), its own X ring slot; k16 step j: 16 k-rows = 2 KB of W,
          // 32 bytes of X
#pragma unroll
          for (int u = 0; u < PF_KSUB; u += XG) {
            mbar_wait(xf0 + 8 * sx, phx);
            tc_fence_after();
            if (elect_one()) {
#pragma unroll
              for (int uu = 0; uu < XG; ++uu) {
#pragma unroll
                for (int k16 = 0; k16 < PF_BLOCK_K / 16; ++k16)
                  umma_bf16(tmem_base, dw + (uint64_t)(((u + uu) * W_SUB + k16 * 2048) >> 4),
                            dx + (uint64_t)((uu * x_sub + k16 * 32) >> 4), idesc, (kb | u | uu | k16) != 0);
              }
              umma_commit(xe0 + 8 * sx);                 // frees the X slot when these MMAs retire
              if (u + XG == PF_KSUB) umma_commit(we0 + 8 * sw);
            }
            __syncwarp();
            dx += dx_step;
            if (++sx == n_sx) { sx = 0; phx ^= 1; dx = dx0; }
          }
          dw += dw_step;
          if (++sw == n_sw) { sw = 0; phw ^= 1; dw = dw0; }
        }
        if (elect_one()) umma_commit(smem_u32(&s_acc_full));
        __syncwarp();
      }
      };
      if (xg == 1) issue(std::integral_constant<int, 1>{}); else issue(std::integral_constant<int, PF_KSUB>{});
    }
  } else {
    // ===== warps 2-5: epilogue.  TMEM lane = output column d of the head, TMEM column = token.  The accumulator is
    //       transposed through shared memory (the operand ring is idle: every MMA of the pass has retired and the
    //       producer waits for s_acc_empty), then each thread finishes 8 + 8 columns (r.., r + D/2..) of one token:
    //       RoPE in fp32 on K tiles, bf16 RNE, two 16-byte stores straight into the paged pool. =====
    const int quarter = warp & 3;                        // TMEM lane quarter this warp may read
    const int et = quarter * 32 + lane;                  // 0..127
    float* tr = reinterpret_cast<float*>(smem);          // [tokens][D] fp32
    enqueue_commit(et, 128);                             // while the first stages stream
    constexpr int PC = D / 16;                           // column-pair chunks per token
    for (int pass = 0; pass < n_pass; ++pass) {
      const int m_base = pass * N_MAX;
      const int rows_here = min(M - m_base, N_MAX);
      const int n_pad = (rows_here + 15) & ~15;
      mbar_wait(smem_u32(&s_acc_full), pass & 1);
      tc_fence_after();
      bool finish = true;                                // this CTA writes the pass's rows (always, without split-K)
      if (p.n_split == 1) {
        for (int col0 = 0; col0 < n_pad; col0 += 32) {   // a load past n_pad stays inside the 256 allocated columns
          uint32_t v[32];
          tmem_ld32(tmem_base + ((uint32_t)(quarter * 32) << 16) + col0, v);
          tmem_ld_wait();
          if (et < D) {
#pragma unroll
            for (int j = 0; j < 32; ++j)
              if (col0 + j < rows_here) tr[(col0 + j) * D + et] = __uint_as_float(v[j]);
          }
        }
        tc_fence_before();
        named_bar_sync(1, 128);
      } else {
        // split-K: publish this CTA's partial [token][D] (coalesced: lane = column); the last CTA of the tile to
        // arrive sums the n_split partials in split order 0, 1, ... (its own included, re-read from L2), so the
        // bits never depend on which CTA finishes last.
        float* mine = p.ws_part + (((size_t)tile * p.n_split + split) * p.row_cap + m_base) * D;
        for (int col0 = 0; col0 < n_pad; col0 += 32) {
          uint32_t v[32];
          tmem_ld32(tmem_base + ((uint32_t)(quarter * 32) << 16) + col0, v);
          tmem_ld_wait();
          if (et < D) {
#pragma unroll
            for (int j = 0; j < 32; ++j)
              if (col0 + j < rows_here) mine[(size_t)(col0 + j) * D + et] = __uint_as_float(v[j]);
          }
        }
        tc_fence_before();
        __threadfence();
        named_bar_sync(1, 128);
        if (et == 0) {
          unsigned int* cnt = p.split_cnt + tile * p.max_pass + pass;
          const unsigned int old = atomicAdd(cnt, 1u);
          s_last = (old == (unsigned int)p.n_split - 1);
          if (s_last) *cnt = 0;                          // self-resetting for the next call
        }
        named_bar_sync(1, 128);
        finish = s_last != 0;
        if (finish) {
          __threadfence();
          const float* part0 = p.ws_part + ((size_t)tile * p.n_split * p.row_cap + m_base) * D;
          const size_t split_stride = (size_t)p.row_cap * D;
          // every load of a step is issued before the first is consumed (8 splits x 4 positions in flight per thread);
          // the additions run in split order
          constexpr int UI = 4, MAXS = 8;
          const int n_pos = rows_here * (D / 4);               // float4 positions: idx = token * D/4 + chunk
          for (int base = et; base < n_pos; base += 128 * UI) {
            float4 x[UI][MAXS];
#pragma unroll
            for (int u = 0; u < UI; ++u)
#pragma unroll
              for (int sp = 0; sp < MAXS; ++sp)
                if (sp < p.n_split && base + u * 128 < n_pos)
                  x[u][sp] = __ldcg(reinterpret_cast<const float4*>(part0 + sp * split_stride) + base + u * 128);
#pragma unroll
            for (int u = 0; u < UI; ++u) {
              if (base + u * 128 >= n_pos) continue;
              float4 acc = x[u][0];
#pragma unroll
              for (int sp = 1; sp < MAXS; ++sp)
                if (sp < p.n_split) { acc.x += x[u][sp].x; acc.y += x[u][sp].y; acc.z += x[u][sp].z; acc.w += x[u][sp].w; }
              reinterpret_cast<float4*>(tr)[base + u * 128] = acc;
            }
          }
          named_bar_sync(1, 128);
        }
      }
      // (read-only loads and an unroll of 4: the row entry -> RoPE entry -> store chains of four iterations overlap; one at a
      // time they cost about 1.5k cycles each, 16 of them per 256-row pass)
#pragma unroll 4
      for (int idx = et; finish && idx < rows_here * PC; idx += 128) {
        const int t = idx / PC, pc = idx % PC;
        const int2 e2 = __ldg(reinterpret_cast<const int2*>(p.rows + m_base + t));
        RowEntry e;
        e.pos = e2.x; e.page_slot = e2.y;
        const float* lo = tr + t * D + pc * 8;
        const float4 a0 = *reinterpret_cast<const float4*>(lo), a1 = *reinterpret_cast<const float4*>(lo + 4);
        const float4 b0 = *reinterpret_cast<const float4*>(lo + D / 2), b1 = *reinterpret_cast<const float4*>(lo + D / 2 + 4);
        const float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
        const float b[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
        float olo[8], ohi[8];
        if (!is_v) {
          const float4* cs = reinterpret_cast<const float4*>(p.rope + (size_t)e.pos * (D / 2) + pc * 8);   // (cos, sin) x 2
#pragma unroll
          for (int i = 0; i < 8; i += 2) {
            const float4 c2 = __ldg(cs + i / 2);
            olo[i] = a[i] * c2.x - b[i] * c2.y;
            ohi[i] = b[i] * c2.x + a[i] * c2.y;
            olo[i + 1] = a[i + 1] * c2.z - b[i + 1] * c2.w;
            ohi[i + 1] = b[i + 1] * c2.z + a[i + 1] * c2.w;
          }
        } else {
#pragma unroll
          for (int i = 0; i < 8; ++i) { olo[i] = a[i]; ohi[i] = b[i]; }
        }
        __nv_bfloat16* dst = (is_v ? p.v_pool : p.k_pool) +
            ((((size_t)layer * p.num_pages + (e.page_slot >> 4)) * p.n_kv_heads + head) * 16 + (e.page_slot & 15)) * D + pc * 8;
        *reinterpret_cast<uint4*>(dst) = make_uint4(pack_bf16(olo[0], olo[1]), pack_bf16(olo[2], olo[3]),
                                                    pack_bf16(olo[4], olo[5]), pack_bf16(olo[6], olo[7]));
        *reinterpret_cast<uint4*>(dst + D / 2) = make_uint4(pack_bf16(ohi[0], ohi[1]), pack_bf16(ohi[2], ohi[3]),
                                                            pack_bf16(ohi[4], ohi[5]), pack_bf16(ohi[6], ohi[7]));
      }
      fence_proxy_async();                               // generic reads of the ring before the next async-proxy writes
      named_bar_sync(1, 128);                            // the transpose buffer is read: the ring may be refilled
      mbar_arrive(smem_u32(&s_acc_empty));               // TMEM and the ring may be overwritten by the next pass
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, TMEM_COLS);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------

namespace {

// One call = ONE launch of each of the two kernels, for one drafter or for both drafters of a round.  This is the only
// device path behind eager prefill, flush, enqueue (with its forced flush) and the fused round calls.
struct CallJob {
  wf_drafter* d;
  PlanJob plan;                         // mode, B, inputs and masks filled by the caller
  int rows_upper;                       // host upper bound of the rows the call projects (sizes the pack grid)
  bool enqueues;                        // ENQUEUE / ROUND with idle sequences
};

int run_jobs(wf_ctx* ctx, CallJob* jobs, int n_jobs, const int32_t* route, int32_t* cur, int32_t* next_q_len,
             int32_t* switched, int q_len_ar, int q_len_diffusion, cudaStream_t st) {
  PlanPackParams pp{};
  GemmParams gp{};
  pp.n_jobs = gp.n_jobs = n_jobs;
  int pack_grid = 0, gemm_grid = 0;
  const int D = jobs[0].d->s.head_dim;
  for (int j = 0; j < n_jobs; ++j) {
    wf_drafter* d = jobs[j].d;
    PlanJob& pj = jobs[j].plan;
    const int S = d->kv->s.max_seqs;
    pj.hidden = d->s.hidden; pj.cap = d->s.backlog_cap; pj.max_pos = d->s.max_pos; pj.row_cap = d->row_cap;
    pj.backlog = d->backlog; pj.backlog_len = d->backlog_len;
    pj.kv = kv_view(d->kv);
    pj.rows = d->d_rows; pj.m_total = d->d_m_total;
    pj.enq_base = d->d_plan; pj.new_blen = d->d_plan + S;
    pj.xpack = d->d_xpack;
    pj.status = ctx->d_status;
    pp.job[j] = pj;
    int rows_upper = jobs[j].rows_upper < d->row_cap ? jobs[j].rows_upper : d->row_cap;
    const int n_pack = rows_upper < 1 ? 1 : (rows_upper > PP_MAX_PACK_CTAS ? PP_MAX_PACK_CTAS : rows_upper);
    pack_grid += 1 + n_pack;
    if (j == 0) pp.ctas_job0 = 1 + n_pack;
    GemmJob& g = gp.job[j];
    g.wpack = d->d_wpack; g.xpack = d->d_xpack; g.rows = d->d_rows; g.m_total = d->d_m_total; g.rope = d->d_rope;
    g.k_pool = d->kv->k_pool; g.v_pool = d->kv->v_pool;
    g.hidden = d->s.hidden; g.n_kv_heads = d->s.n_kv_heads; g.num_pages = d->kv->s.num_pages;
    g.n_split = d->n_split; g.row_cap = d->row_cap; g.max_pass = d->max_pass; g.ws_part = d->d_ws_part; g.split_cnt = d->d_split_cnt;
    g.hidden_rows = pj.hidden_rows; g.q_indptr = pj.q_indptr; g.n_rows = pj.n_rows; g.seq_ids = pj.seq_ids;
    g.enq_base = jobs[j].enqueues ? pj.enq_base : nullptr;
    g.new_blen = (pj.mode == PLAN_EAGER || pj.cap == 0) ? nullptr : pj.new_blen;
    g.backlog = const_cast<__nv_bfloat16*>(d->backlog); g.backlog_len = d->backlog_len;
    g.B = pj.B; g.cap = pj.cap; g.max_rows = pj.max_rows;
    g.route = route; g.cur = cur; g.next_q_len = next_q_len; g.switched = switched; g.q_len_ar = q_len_ar; g.q_len_diffusion = q_len_diffusion;
    const int ctas = d->s.n_layers * 2 * d->s.n_kv_heads * d->n_split;
    gemm_grid += ctas;
    if (j == 0) gp.ctas_job0 = ctas;
  }
  if (n_jobs == 1) { pp.ctas_job0 = pack_grid; gp.ctas_job0 = gemm_grid; }
  wf_launch(wf_plan_pack_kernel, dim3(pack_grid), dim3(PP_THREADS), 0, st, pp);
  int rc = wf_check_launch(ctx, "wf_plan_pack_kernel");
  if (rc != WF_OK) return rc;
  if (D == 128) {
    WF_CONFIGURE_ONCE(ctx, WF_FUNC_GEMM_128, wf_prefill_gemm_kernel<128>, PF_SMEM_LAUNCH);
    wf_launch(wf_prefill_gemm_kernel<128>, dim3(gemm_grid), dim3(PF_THREADS), PF_SMEM_LAUNCH, st, gp);
  } else {
    WF_CONFIGURE_ONCE(ctx, WF_FUNC_GEMM_64, wf_prefill_gemm_kernel<64>, PF_SMEM_LAUNCH);
    wf_launch(wf_prefill_gemm_kernel<64>, dim3(gemm_grid), dim3(PF_THREADS), PF_SMEM_LAUNCH, st, gp);
  }
  return wf_check_launch(ctx, "wf_prefill_gemm_kernel");
}

int run_one(wf_ctx* ctx, wf_drafter* d, const PlanJob& pj, int rows_upper, bool enqueues, cudaStream_t st) {
  CallJob job{d, pj, rows_upper, enqueues};
  return run_jobs(ctx, &job, 1, nullptr, nullptr, nullptr, nullptr, 0, 0, st);
}

}  // namespace

extern "C" int wf_drafter_create(wf_ctx* ctx, const wf_drafter_shape* s, const void* const* w_k_host_ptrs,
                                 const void* const* w_v_host_ptrs, wf_paged_kv* kv, void* backlog,
                                 int32_t* backlog_len, wf_drafter** out) {
  if (!ctx || !out) return WF_ERR_INVALID_ARG;
  *out = nullptr;
  WF_REQUIRE(ctx, s && w_k_host_ptrs && w_v_host_ptrs && kv, WF_ERR_INVALID_ARG, "wf_drafter_create: null argument");
  WF_REQUIRE(ctx, s->n_layers == kv->s.n_layers && s->n_kv_heads == kv->s.n_kv_heads && s->head_dim == kv->s.head_dim,
             WF_ERR_INVALID_ARG, "wf_drafter_create: drafter shape does not match its KV cache");
  WF_REQUIRE(ctx, s->head_dim == 64 || s->head_dim == 128, WF_ERR_UNSUPPORTED_SHAPE, "wf_drafter_create: head_dim must be 64 or 128");
  WF_REQUIRE(ctx, s->hidden > 0 && s->hidden % (PF_KSUB * PF_BLOCK_K) == 0, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_drafter_create: hidden must be a positive multiple of %d", PF_KSUB * PF_BLOCK_K);
  WF_REQUIRE(ctx, s->max_pos > 0 && s->rope_theta > 0.f && s->backlog_cap >= 0, WF_ERR_INVALID_ARG, "wf_drafter_create: bad max_pos/theta/cap");
  WF_REQUIRE(ctx, s->backlog_cap == 0 || (backlog && backlog_len), WF_ERR_INVALID_ARG, "wf_drafter_create: backlog buffers missing");
  const int L = s->n_layers, D = s->head_dim, N = s->n_kv_heads * D;
  for (int l = 0; l < L; ++l)
    for (int v = 0; v < 2; ++v) {
      const void* w = v ? w_v_host_ptrs[l] : w_k_host_ptrs[l];
      WF_REQUIRE(ctx, w && (uintptr_t)w % 16 == 0, WF_ERR_INVALID_ARG, "wf_drafter_create: weight pointer null or unaligned");
    }
  // RoPE table in fp64 on the host (C17): angle = pos * theta^(-2r/D)
  const int half = D / 2;
  std::vector<float2> rope((size_t)s->max_pos * half);
  std::vector<double> inv_freq(half);
  for (int r = 0; r < half; ++r) inv_freq[r] = pow((double)s->rope_theta, -2.0 * r / D);
  for (int pos = 0; pos < s->max_pos; ++pos)
    for (int r = 0; r < half; ++r) {
      const double a = (double)pos * inv_freq[r];
      rope[(size_t)pos * half + r] = make_float2((float)cos(a), (float)sin(a));
    }

  wf_drafter* d = new (std::nothrow) wf_drafter();
  if (!d) return wf_set_error(ctx, WF_ERR_INVALID_ARG, "wf_drafter_create: host allocation failed");
  d->ctx = ctx; d->s = *s; d->kv = kv;
  d->backlog = (const __nv_bfloat16*)backlog; d->backlog_len = backlog_len;
  d->d_wpack = nullptr; d->d_xpack = nullptr; d->d_rope = nullptr; d->d_ws_part = nullptr; d->d_split_cnt = nullptr; d->d_rows = nullptr; d->d_m_total = nullptr; d->d_plan = nullptr; d->full = nullptr;
  // rows one call can carry: a whole backlog plus a block (64 rows at most) per sequence (wf_lazy_catchup_round)
  d->row_cap = kv->s.max_seqs * ((s->backlog_cap > 64 ? s->backlog_cap : 64) + 64);
  // Split-K: a call with few tiles (a 1-layer drafter has 16) cannot pull HBM bandwidth through 16 SMs; spread each
  // tile's k-blocks over the largest power of two of CTAs that still fits one CTA per SM.  The factor depends on the
  // drafter's shape only, never on the call, so a row's bits do not depend on M (lazy == eager).
  {
    const int tiles = L * 2 * s->n_kv_heads, stages = s->hidden / (PF_KSUB * PF_BLOCK_K);
    int ns = 1;
    while (ns * 2 <= 8 && tiles * ns * 2 <= ctx->sm_count && stages % (ns * 2) == 0) ns *= 2;
    d->n_split = ns;
    d->max_pass = (d->row_cap + PF_MAX_MT * PF_BLOCK_M - 1) / (PF_MAX_MT * PF_BLOCK_M);
  }
  const size_t w_bytes = (size_t)s->hidden * N * 2;                    // one [hidden][Hkv*D] matrix
  cudaError_t e = cudaMalloc(&d->d_wpack, w_bytes * 2 * L);
  if (e == cudaSuccess) e = cudaMalloc(&d->d_xpack, (size_t)s->hidden * 2 * d->row_cap);
  if (e == cudaSuccess && d->n_split > 1) {
    const size_t tiles = (size_t)L * 2 * s->n_kv_heads;
    e = cudaMalloc(&d->d_ws_part, tiles * d->n_split * d->row_cap * D * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&d->d_split_cnt, tiles * d->max_pass * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(d->d_split_cnt, 0, tiles * d->max_pass * sizeof(unsigned int));
  }
  if (e == cudaSuccess) e = cudaMalloc(&d->d_rope, sizeof(float2) * rope.size());
  if (e == cudaSuccess) e = cudaMalloc(&d->d_rows, sizeof(RowEntry) * d->row_cap);
  if (e == cudaSuccess) e = cudaMalloc(&d->d_m_total, sizeof(int32_t));
  if (e == cudaSuccess) e = cudaMalloc(&d->d_plan, sizeof(int32_t) * 3 * kv->s.max_seqs);
  if (e == cudaSuccess) {
    for (int l = 0; l < L; ++l)
      for (int v = 0; v < 2; ++v)
        wf_pack_w_kernel<<<dim3(s->hidden / PF_BLOCK_K, s->n_kv_heads), 256>>>(
            (const __nv_bfloat16*)(v ? w_v_host_ptrs[l] : w_k_host_ptrs[l]), d->d_wpack + (size_t)(l * 2 + v) * w_bytes, s->hidden, N, D);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();   // creation is synchronous: the caller may free or rewrite W afterwards
  }
  if (e == cudaSuccess) e = cudaMemcpy(d->d_rope, rope.data(), sizeof(float2) * rope.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemset(d->d_m_total, 0, sizeof(int32_t));
  if (e != cudaSuccess) {
    wf_drafter_destroy(d);
    return wf_set_error(ctx, WF_ERR_CUDA, "wf_drafter_create: %s", cudaGetErrorString(e));
  }
  *out = d;
  return WF_OK;
}

extern "C" int wf_drafter_destroy(wf_drafter* d) {
  if (!d) return WF_ERR_INVALID_ARG;
  cudaFree(d->d_wpack); cudaFree(d->d_xpack); cudaFree(d->d_ws_part); cudaFree(d->d_split_cnt); cudaFree(d->d_rope); cudaFree(d->d_rows); cudaFree(d->d_m_total); cudaFree(d->d_plan);
  if (d->full) wf_full_layer_destroy(d->full);
  delete d;
  return WF_OK;
}

extern "C" int wf_kv_only_prefill(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                  const int32_t* n_rows, const int32_t* seq_ids, int B, int max_rows, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows, WF_ERR_INVALID_ARG, "wf_kv_only_prefill: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && B <= PP_MAX_B && max_rows >= 0 && (long long)B * max_rows <= d->row_cap,
             WF_ERR_INVALID_ARG, "wf_kv_only_prefill: need B <= %d and B * max_rows <= the row table (%d)", PP_MAX_B, d->row_cap);
  WF_REQUIRE(ctx, (uintptr_t)hidden % 16 == 0, WF_ERR_INVALID_ARG, "wf_kv_only_prefill: hidden must be 16-byte aligned");
  if (B == 0 || max_rows == 0) return WF_OK;
  PlanJob pj{};
  pj.mode = PLAN_EAGER; pj.B = B; pj.max_rows = max_rows;
  pj.hidden_rows = (const __nv_bfloat16*)hidden; pj.q_indptr = q_indptr; pj.n_rows = n_rows; pj.seq_ids = seq_ids;
  return run_one(ctx, d, pj, B * max_rows, false, (cudaStream_t)stream);
}

extern "C" int wf_lazy_catchup_flush(wf_ctx* ctx, wf_drafter* d, const int32_t* flush_mask, int B, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && B <= PP_MAX_B, WF_ERR_INVALID_ARG, "wf_lazy_catchup_flush: bad B (max %d)", PP_MAX_B);
  WF_REQUIRE(ctx, d->s.backlog_cap > 0, WF_ERR_INVALID_ARG, "wf_lazy_catchup_flush: drafter has no backlog");
  if (B == 0) return WF_OK;
  PlanJob pj{};
  pj.mode = PLAN_FLUSH; pj.B = B; pj.flush_mask = flush_mask; pj.max_rows = 0;
  return run_one(ctx, d, pj, B * d->s.backlog_cap, false, (cudaStream_t)stream);
}

extern "C" int wf_lazy_catchup_enqueue(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                       const int32_t* n_rows, const int32_t* seq_ids, const int32_t* idle_mask,
                                       int B, int max_rows, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows && idle_mask, WF_ERR_INVALID_ARG, "wf_lazy_catchup_enqueue: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && B <= PP_MAX_B && max_rows >= 0, WF_ERR_INVALID_ARG,
             "wf_lazy_catchup_enqueue: bad B (max %d)", PP_MAX_B);
  WF_REQUIRE(ctx, d->s.backlog_cap > 0 && max_rows <= d->s.backlog_cap, WF_ERR_INVALID_ARG,
             "wf_lazy_catchup_enqueue: max_rows exceeds backlog_cap");
  WF_REQUIRE(ctx, (uintptr_t)hidden % 16 == 0, WF_ERR_INVALID_ARG, "wf_lazy_catchup_enqueue: hidden must be 16-byte aligned");
  if (B == 0 || max_rows == 0) return WF_OK;
  // the forced flush of the sequences whose backlog would overflow (C20) and the append are one call: the planner
  // decides the offsets (-1 where nothing may be written, e.g. when the forced flush found no pages)
  PlanJob pj{};
  pj.mode = PLAN_ENQUEUE; pj.B = B; pj.max_rows = max_rows;
  pj.hidden_rows = (const __nv_bfloat16*)hidden; pj.q_indptr = q_indptr; pj.n_rows = n_rows; pj.seq_ids = seq_ids;
  pj.idle_mask = idle_mask;
  return run_one(ctx, d, pj, B * d->s.backlog_cap, true, (cudaStream_t)stream);
}

namespace {
int check_round_args(wf_ctx* ctx, wf_drafter* d, const char* who, const void* hidden, const int32_t* q_indptr,
                     const int32_t* n_rows, int B, int max_rows, bool may_idle) {
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows, WF_ERR_INVALID_ARG, "%s: null argument", who);
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && B <= PP_MAX_B && max_rows >= 0 && max_rows <= 64, WF_ERR_INVALID_ARG,
             "%s: need B <= min(max_seqs, %d) and max_rows <= 64", who, PP_MAX_B);
  WF_REQUIRE(ctx, !may_idle || (d->s.backlog_cap > 0 && max_rows <= d->s.backlog_cap), WF_ERR_INVALID_ARG,
             "%s: idle sequences need a backlog with max_rows <= backlog_cap", who);
  WF_REQUIRE(ctx, (long long)B * (d->s.backlog_cap + max_rows) <= d->row_cap, WF_ERR_INVALID_ARG,
             "%s: B * (backlog_cap + max_rows) exceeds the row table (%d)", who, d->row_cap);
  WF_REQUIRE(ctx, (uintptr_t)hidden % 16 == 0, WF_ERR_INVALID_ARG, "%s: hidden must be 16-byte aligned", who);
  return WF_OK;
}
}  // namespace

extern "C" int wf_lazy_catchup_round(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                     const int32_t* n_rows, const int32_t* seq_ids, const int32_t* idle_mask,
                                     const int32_t* flush_mask, int B, int max_rows, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  int rc = check_round_args(ctx, d, "wf_lazy_catchup_round", hidden, q_indptr, n_rows, B, max_rows, idle_mask != nullptr);
  if (rc != WF_OK) return rc;
  if (B == 0 || max_rows == 0) return WF_OK;
  PlanJob pj{};
  pj.mode = PLAN_ROUND; pj.B = B; pj.max_rows = max_rows;
  pj.hidden_rows = (const __nv_bfloat16*)hidden; pj.q_indptr = q_indptr; pj.n_rows = n_rows; pj.seq_ids = seq_ids;
  pj.idle_mask = idle_mask; pj.flush_mask = flush_mask;
  return run_one(ctx, d, pj, B * (d->s.backlog_cap + max_rows), idle_mask != nullptr, (cudaStream_t)stream);
}

extern "C" int wf_switch_round(wf_ctx* ctx, wf_drafter* drafter_ar, wf_drafter* drafter_diffusion, const void* hidden,
                               const int32_t* q_indptr, const int32_t* n_rows, const int32_t* seq_ids,
                               const int32_t* route, int32_t* cur_drafter, int32_t* next_q_len, int32_t* switched,
                               int q_len_ar, int q_len_diffusion, int B, int max_rows, void* stream) {
  if (!ctx || !drafter_ar || !drafter_diffusion) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, route && cur_drafter, WF_ERR_INVALID_ARG, "wf_switch_round: null route / cur_drafter");
  WF_REQUIRE(ctx, drafter_ar != drafter_diffusion && drafter_ar->kv != drafter_diffusion->kv, WF_ERR_INVALID_ARG,
             "wf_switch_round: the two drafters must be distinct and own distinct caches");
  WF_REQUIRE(ctx, drafter_ar->s.head_dim == drafter_diffusion->s.head_dim && drafter_ar->s.hidden == drafter_diffusion->s.hidden,
             WF_ERR_UNSUPPORTED_SHAPE, "wf_switch_round: the drafters must share hidden size and head_dim");
  wf_drafter* ds[2] = {drafter_diffusion, drafter_ar};     // the 5-layer stream first: its CTAs are the long ones
  const int codes[2] = {WF_ROUTE_DIFFUSION, WF_ROUTE_AR};
  CallJob jobs[2];
  for (int j = 0; j < 2; ++j) {
    int rc = check_round_args(ctx, ds[j], "wf_switch_round", hidden, q_indptr, n_rows, B, max_rows, true);
    if (rc != WF_OK) return rc;
    PlanJob pj{};
    pj.mode = PLAN_ROUND; pj.B = B; pj.max_rows = max_rows; pj.code = codes[j];
    pj.hidden_rows = (const __nv_bfloat16*)hidden; pj.q_indptr = q_indptr; pj.n_rows = n_rows; pj.seq_ids = seq_ids;
    pj.route = route; pj.cur = cur_drafter;
    jobs[j] = CallJob{ds[j], pj, B * (ds[j]->s.backlog_cap + max_rows), true};
  }
  if (B == 0 || max_rows == 0) return WF_OK;
  return run_jobs(ctx, jobs, 2, route, cur_drafter, next_q_len, switched, q_len_ar, q_len_diffusion, (cudaStream_t)stream);
}

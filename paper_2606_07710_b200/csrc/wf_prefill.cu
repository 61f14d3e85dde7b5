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
// path, a fixed K order, no split-K; an accumulator column depends only on its own X row.
#include <cuda.h>
#include <math.h>

#include <new>
#include <vector>

#include "wf_internal.cuh"
#include "wf_sm100.cuh"

namespace {

constexpr int PF_BLOCK_M = 128;         // UMMA M
constexpr int PF_BLOCK_K = 64;          // one 128-byte swizzle row of bf16
constexpr int PF_KSUB = 2;              // 64-wide k-blocks per pipeline stage: halves the per-stage hand-offs of the one-thread loops
constexpr int PF_MAX_MT = 2;            // m-tiles per pass (TMEM columns = PF_MAX_MT * D)
constexpr int PF_THREADS = 192;         // warp 0: bulk-copy producer, warp 1: MMA, warps 2-5: epilogue
constexpr int PF_SMEM_BUDGET = 200 * 1024;
struct RowEntry {
  const __nv_bfloat16* src;             // hidden row
  int32_t pos;                          // absolute position (RoPE)
  int32_t page_slot;                    // physical page * 16 + slot in the drafter cache
};

// ---- the plan kernel -------------------------------------------------------------------------
// PLAN_ROUND fuses what one round asks of a drafter into ONE projection: block rows of the sequences it is active for,
// backlog + block rows of the sequences that switch to it (flush), a forced flush where an enqueue would overflow;
// the rows of idle sequences are enqueued afterwards (wf_enqueue_round_kernel) at the offsets this plan decides.
enum PlanMode { PLAN_EAGER = 0, PLAN_FLUSH = 1, PLAN_FORCED = 2, PLAN_ROUND = 3 };

struct PlanParams {
  int mode, B, hidden, cap, max_pos, row_cap;
  const __nv_bfloat16* hidden_rows;     // EAGER: block hidden states [sum_q][hidden]
  const int32_t* q_indptr;              // EAGER / FORCED
  const int32_t* n_rows;                // EAGER / FORCED
  const int32_t* seq_ids;               // EAGER / FORCED (NULL = identity)
  const int32_t* mask;                  // FLUSH: flush_mask (NULL = all); FORCED / ROUND: idle_mask (ROUND: NULL = none idle)
  const int32_t* mask2;                 // ROUND: flush_mask (NULL = none)
  int32_t* enq_base;                    // ROUND: [B] backlog offset at which the block rows are enqueued afterwards, -1 = none
  const __nv_bfloat16* backlog;         // [max_seqs][cap][hidden]
  int32_t* backlog_len;
  KvView kv;
  RowEntry* rows;
  int32_t* m_total;
  int32_t* plan_n;                      // [max_seqs] rows of sequence b in this call
  int32_t* plan_off;                    // [max_seqs] first compact row of sequence b
  int* status;
};

__global__ void __launch_bounds__(1024) wf_prefill_plan_kernel(const PlanParams p) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  // rows / first compact row per sequence: shared memory for the first 1024 sequences, global scratch beyond
  __shared__ int s_pn[KV_RESERVE_SMEM], s_po[KV_RESERVE_SMEM];
  // ROUND (B <= 1024): backlog rows at the front of b's rows, backlog length after the call, enqueue offset (-1 = none)
  __shared__ int s_nb[KV_RESERVE_SMEM], s_nl[KV_RESERVE_SMEM], s_eb[KV_RESERVE_SMEM];
  auto plan_n = [&](int b) -> int& { return b < KV_RESERVE_SMEM ? s_pn[b] : p.plan_n[b]; };
  auto plan_off = [&](int b) -> int& { return b < KV_RESERVE_SMEM ? s_po[b] : p.plan_off[b]; };
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
  wf_pdl_trigger();
  wf_pdl_wait();
  auto seq_of = [&](int b) { return (p.mode != PLAN_FLUSH && p.seq_ids) ? p.seq_ids[b] : b; };
  // rows each sequence contributes to this call
  for (int b = tid; b < p.B; b += blockDim.x) {
    const int sq = seq_of(b);
    int n;
    if (p.mode == PLAN_ROUND) {
      const int add = p.n_rows[b], len = p.cap > 0 ? p.backlog_len[sq] : 0;
      const bool idle = p.mask && p.mask[b], fl = p.mask2 && p.mask2[b];
      const bool project_block = !idle || fl;
      int n_enq = project_block ? 0 : add;
      if (n_enq > p.cap) { *p.status = WF_ERR_QUEUE_OVERFLOW; n_enq = 0; }     // rows skipped, as in enqueue
      // the backlog goes first whenever anything of this sequence is projected (FIFO), or when the enqueue would overflow
      const int n_back = (project_block || len + n_enq > p.cap) ? len : 0;
      s_nb[b] = n_back;
      n = n_back + (project_block ? add : 0);
      s_eb[b] = n_enq > 0 ? (n_back > 0 ? 0 : len) : -1;
      s_nl[b] = (n_back > 0 ? 0 : len) + n_enq;
    } else if (p.mode == PLAN_EAGER) {
      n = p.n_rows[b];
    } else if (p.mode == PLAN_FLUSH) {
      n = (!p.mask || p.mask[b]) ? p.backlog_len[sq] : 0;
    } else {                                                   // forced flush before an enqueue (C20)
      const int add = p.n_rows[b];
      if (p.mask[b] && add > p.cap) *p.status = WF_ERR_QUEUE_OVERFLOW;
      n = (p.mask[b] && add <= p.cap && p.backlog_len[sq] + add > p.cap) ? p.backlog_len[sq] : 0;
    }
    plan_n(b) = n;
  }
  if (tid == 0) s_carry = 0;
  __syncthreads();
  // pages first (C24: ascending b, consecutive ring entries); nothing is written if they do not fit
  const bool ok = kv_reserve_block(p.kv, p.B, [&](int b) { return plan_n(b); }, seq_of, p.status);
  if (!ok) {                                                   // nothing is projected, nothing is enqueued, no length moves
    if (tid == 0) *p.m_total = 0;
    if (p.mode == PLAN_ROUND)
      for (int b = tid; b < p.B; b += blockDim.x) p.enq_base[b] = -1;
    return;
  }
  // exclusive scan of plan_n -> plan_off
  for (int base = 0; base < p.B; base += blockDim.x) {
    const int b = base + tid;
    const int n = b < p.B ? plan_n(b) : 0;
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
    if (b < p.B) plan_off(b) = s_carry + (wid ? s_warp[wid - 1] : 0) + x - n;
    __syncthreads();
    if (tid == 0) s_carry += s_warp[nw - 1];
    __syncthreads();
  }
  const int total = s_carry;
  if (total > p.row_cap) {                                     // host bounds make this unreachable
    if (tid == 0) { *p.status = WF_ERR_INVALID_ARG; *p.m_total = 0; }
    return;
  }
  // row table: one warp per sequence
  for (int b = wid; b < p.B; b += nw) {
    const int sq = seq_of(b);
    const int n = plan_n(b), off = plan_off(b);
    const int p0 = p.kv.seq_len[sq];
    const bool from_block = p.mode == PLAN_EAGER || p.mode == PLAN_ROUND;
    const int n_back = p.mode == PLAN_ROUND ? s_nb[b] : (from_block ? 0 : n);
    const __nv_bfloat16* blk = from_block ? p.hidden_rows + (size_t)p.q_indptr[b] * p.hidden : nullptr;
    const __nv_bfloat16* bkl = p.backlog + (size_t)sq * p.cap * p.hidden;
    for (int t = lane; t < n; t += 32) {
      const int pos = p0 + t;
      if (pos >= p.max_pos) *p.status = WF_ERR_INVALID_ARG;
      const int page = p.kv.block_table[(size_t)sq * p.kv.max_pages_per_seq + (pos >> 4)];
      RowEntry e;
      e.src = t < n_back ? bkl + (size_t)t * p.hidden : blk + (size_t)(t - n_back) * p.hidden;
      e.pos = min(pos, p.max_pos - 1);
      e.page_slot = page * 16 + (pos & 15);
      p.rows[off + t] = e;
    }
    __syncwarp();
    if (lane == 0 && p.mode == PLAN_ROUND) {
      p.enq_base[b] = s_eb[b];
      if (p.cap > 0) p.backlog_len[sq] = s_nl[b];
    }
    if (lane == 0 && n > 0) {
      p.kv.seq_len[sq] = p0 + n;
      if (p.mode == PLAN_FLUSH || p.mode == PLAN_FORCED) p.backlog_len[sq] = 0;
    }
  }
  if (tid == 0) *p.m_total = total;
}

// ---- the projection kernel ------------------------------------------------------------------
constexpr int PF_MAX_STAGES = 12;

// Per call: the rows of the plan's row table -> the shared-memory image of the A operand, k-block by k-block:
// xpack[kb][m_pad][128 B], row m of k-block kb = X[m][64 kb .. 64 kb + 63], 16-byte chunks XOR-swizzled with (m & 7)
// (K-major, 128-byte swizzle).  One block per row; every projection CTA then fetches a stage's A operand with
// one bulk copy instead of gathering it with 128 threads.
__global__ void __launch_bounds__(256) wf_pack_x_kernel(const RowEntry* __restrict__ rows, const int32_t* __restrict__ m_total,
                                                        uint8_t* __restrict__ xpack, int hidden) {
  wf_pdl_trigger();
  wf_pdl_wait();
  const int M = *m_total;
  const int r = blockIdx.x;                              // one row per block: every load of the block is independent
  if (r >= M) return;
  const int m_pad = (M + 7) & ~7;
  const uint4* src = reinterpret_cast<const uint4*>(rows[r].src);
  uint8_t* dst = xpack + (size_t)r * 128;
  const size_t kb_stride = (size_t)m_pad * 128;
  for (int q = threadIdx.x; q < hidden / 8; q += 256) {  // 16-byte chunk q of the row -> k-block q/8, chunk q%8
    const uint4 v = __ldg(src + q);
    *reinterpret_cast<uint4*>(dst + (size_t)(q >> 3) * kb_stride + (((q & 7) ^ (r & 7)) << 4)) = v;
  }
}

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

struct GemmParams {
  const uint8_t* wpack;                 // [n_layers][2][Hkv][hidden/64][64 * D * 2 B] pre-swizzled W stages
  const uint8_t* xpack;                 // [hidden/64][m_pad][128 B] pre-swizzled X k-blocks of this call (wf_pack_x_kernel)
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
};

template <int D>
__global__ void __launch_bounds__(PF_THREADS, 1) wf_prefill_gemm_kernel(const GemmParams p) {
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
  __shared__ __align__(8) uint64_t s_full[PF_MAX_STAGES], s_empty[PF_MAX_STAGES], s_acc_full, s_acc_empty;
  __shared__ uint32_t s_tmem;
  __shared__ int s_last;

  wf_pdl_trigger();
  wf_pdl_wait();
  const int M = *p.m_total;
  if (M == 0) return;                                  // nothing queued for this call
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int tile = blockIdx.x / p.n_split;             // (layer, K|V, kv head)
  const int split = blockIdx.x % p.n_split;            // this CTA's share of the k-blocks
  const int layer = tile / (2 * p.n_kv_heads);
  const int is_v = (tile / p.n_kv_heads) & 1;
  const int head = tile % p.n_kv_heads;
  const int n_kb_tile = p.hidden / (PF_KSUB * PF_BLOCK_K);   // pipeline stages of a whole tile
  const int n_kb = n_kb_tile / p.n_split;                    // stages this CTA runs per pass (n_split divides them)
  const int kb0 = split * n_kb;
  const int n_pass = (M + N_MAX - 1) / N_MAX;

  // An X stage holds only the rows that exist (8-row swizzle atoms); UMMA reads n_pad (multiple of 16) rows from
  // its start, the few surplus rows feed accumulator columns nobody reads.
  const int m_first = min(M, N_MAX);
  const int x_sub = ((m_first + 7) / 8) * 1024;          // one 64-wide k-block of the X operand
  const int x_stage = PF_KSUB * x_sub;
  const int n_stages = min(PF_MAX_STAGES, PF_SMEM_BUDGET / (x_stage + W_BYTES));
  uint8_t* x_base = smem;
  uint8_t* w_base = smem + (size_t)n_stages * x_stage;     // 1024-aligned: x_stage is a multiple of 1024

  if (tid == 0) {
    for (int i = 0; i < n_stages; ++i) { mbar_init(smem_u32(&s_full[i]), 1); mbar_init(smem_u32(&s_empty[i]), 1); }
    mbar_init(smem_u32(&s_acc_full), 1);
    mbar_init(smem_u32(&s_acc_empty), 128);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(smem_u32(&s_tmem), TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = s_tmem;

  if (warp == 0) {
    // ===== bulk-copy producer: per stage ONE contiguous copy of the pre-swizzled W k-blocks and one per packed X
    //       k-block (wf_pack_x_kernel): no thread touches operand bytes.  Stage index, phase and addresses advance
    //       incrementally: a runtime division per stage in a one-thread loop costs more than the MMAs it feeds.
    //       The whole warp runs the loop (warp-uniform control flow) and one elected lane issues: ptxas then emits
    //       straight-line UBLKCP / UTCHMMA instead of a divergence loop around every instruction. =====
    {
      const uint8_t* w_src = p.wpack + ((size_t)tile * n_kb_tile + kb0) * W_BYTES;   // tile = (layer, K|V, head), packed in that order
      const size_t x_kb_stride = (size_t)((M + 7) & ~7) * 128;
      const uint32_t full0 = smem_u32(&s_full[0]), empty0 = smem_u32(&s_empty[0]);
      const uint32_t x0 = smem_u32(x_base), w0 = smem_u32(w_base);
      int s = 0;
      uint32_t ph = 1;                                   // parity to wait for on s_empty: the ring starts empty
      for (int pass = 0; pass < n_pass; ++pass) {
        const int rows_here = min(M - pass * N_MAX, N_MAX);
        const uint32_t x_bytes = (uint32_t)((rows_here + 7) / 8) * 1024;
        const uint8_t* x_src = p.xpack + (size_t)pass * N_MAX * 128 + (size_t)kb0 * PF_KSUB * x_kb_stride;
        const uint8_t* w_kb = w_src;
        // the epilogue of the previous pass transposes through the ring: do not refill it before it is done
        if (pass > 0) mbar_wait(smem_u32(&s_acc_empty), (pass - 1) & 1);
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(empty0 + 8 * s, ph);
          if (elect_one()) {
            const uint32_t bar = full0 + 8 * s;
            mbar_arrive_expect_tx(bar, W_BYTES + PF_KSUB * x_bytes);
            bulk_load(w0 + s * W_BYTES, w_kb, W_BYTES, bar);
#pragma unroll
            for (int u = 0; u < PF_KSUB; ++u) bulk_load(x0 + s * x_stage + u * x_sub, x_src + u * x_kb_stride, x_bytes, bar);
          }
          __syncwarp();
          w_kb += W_BYTES;
          x_src += PF_KSUB * x_kb_stride;
          if (++s == n_stages) { s = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: one thread drives the tensor core for the CTA.  Descriptors are built once and advanced by
    //       constant offsets.  A = W tile (MN-major, 128-byte swizzle), B = X rows (K-major, 128-byte swizzle). =====
    {
      const uint64_t dw0 = umma_desc(smem_u32(w_base), 8192, 1024);        // MN-major: 64-column halves 8 KB apart
      const uint64_t dx0 = umma_desc(smem_u32(x_base), 16, 1024);          // K-major
      const uint32_t full0 = smem_u32(&s_full[0]), empty0 = smem_u32(&s_empty[0]);
      const uint64_t dw_step = (uint64_t)(W_BYTES >> 4), dx_step = (uint64_t)(x_stage >> 4);
      int s = 0;
      uint32_t ph = 0;
      uint64_t dw = dw0, dx = dx0;
      for (int pass = 0; pass < n_pass; ++pass) {
        const int rows_here = min(M - pass * N_MAX, N_MAX);
        const uint32_t idesc = umma_idesc_mn_k(128, (rows_here + 15) & ~15);
        if (pass > 0) { mbar_wait(smem_u32(&s_acc_empty), (pass - 1) & 1); tc_fence_after(); }
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(full0 + 8 * s, ph);
          tc_fence_after();
          if (elect_one()) {
          // k16 step j of the stage: W k-block j/4 (W_SUB apart), 16 k-rows = 2 KB per step; X k-block j/4 (x_sub apart),
          // 32 bytes per step
#pragma unroll
          for (int k16 = 0; k16 < PF_KSUB * PF_BLOCK_K / 16; ++k16)
            umma_bf16(tmem_base, dw + (uint64_t)(((k16 >> 2) * W_SUB + (k16 & 3) * 2048) >> 4),
                      dx + (uint64_t)(((k16 >> 2) * x_sub + (k16 & 3) * 32) >> 4), idesc, (kb | k16) != 0);
          umma_commit(empty0 + 8 * s);                   // frees the stage when these MMAs retire
          }
          __syncwarp();
          dw += dw_step; dx += dx_step;
          if (++s == n_stages) { s = 0; ph ^= 1; dw = dw0; dx = dx0; }
        }
        if (elect_one()) umma_commit(smem_u32(&s_acc_full));
        __syncwarp();
      }
    }
  } else {
    // ===== warps 2-5: epilogue.  TMEM lane = output column d of the head, TMEM column = token.  The accumulator is
    //       transposed through shared memory (the operand ring is idle: every MMA of the pass has retired and the
    //       producer waits for s_acc_empty), then each thread finishes 8 + 8 columns (r.., r + D/2..) of one token:
    //       RoPE in fp32 on K tiles, bf16 RNE, two 16-byte stores straight into the paged pool. =====
    const int quarter = warp & 3;                        // TMEM lane quarter this warp may read
    const int et = quarter * 32 + lane;                  // 0..127
    float* tr = reinterpret_cast<float*>(smem);          // [tokens][D] fp32
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
      for (int idx = et; finish && idx < rows_here * PC; idx += 128) {
        const int t = idx / PC, pc = idx % PC;
        const RowEntry e = p.rows[m_base + t];
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
struct wf_drafter {
  wf_ctx* ctx;
  wf_drafter_shape s;
  wf_paged_kv* kv;
  const __nv_bfloat16* backlog;
  int32_t* backlog_len;
  uint8_t* d_wpack;            // library-owned pre-swizzled copy of the weights (see wf_pack_w_kernel)
  uint8_t* d_xpack;            // library-owned [hidden/64][row_cap][128 B] scratch (see wf_pack_x_kernel)
  int n_split;                 // split-K factor of the projection, fixed at creation (a power of two)
  int max_pass;
  float* d_ws_part;            // [tiles][n_split][row_cap][D] fp32 partials (n_split > 1)
  unsigned int* d_split_cnt;   // [tiles][max_pass]
  float2* d_rope;              // [max_pos][D/2]
  RowEntry* d_rows;
  int row_cap;
  int32_t* d_m_total;
  int32_t* d_plan;             // [3 * max_seqs]: plan_n, plan_off, enq_base
};

namespace {

template <int D>
int launch_gemm(wf_drafter* d, cudaStream_t st) {
  wf_ctx* ctx = d->ctx;
  static bool configured = false;
  if (!configured) {
    WF_CUDA(ctx, cudaFuncSetAttribute(wf_prefill_gemm_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, PF_SMEM_BUDGET));
    configured = true;
  }
  GemmParams g;
  g.wpack = d->d_wpack; g.xpack = d->d_xpack; g.rows = d->d_rows; g.m_total = d->d_m_total; g.rope = d->d_rope;
  g.k_pool = d->kv->k_pool; g.v_pool = d->kv->v_pool;
  g.hidden = d->s.hidden; g.n_kv_heads = d->s.n_kv_heads; g.num_pages = d->kv->s.num_pages;
  g.n_split = d->n_split; g.row_cap = d->row_cap; g.max_pass = d->max_pass; g.ws_part = d->d_ws_part; g.split_cnt = d->d_split_cnt;
  const int grid = d->s.n_layers * 2 * d->s.n_kv_heads * d->n_split;
  wf_launch(wf_prefill_gemm_kernel<D>, dim3(grid), dim3(PF_THREADS), PF_SMEM_BUDGET, st, g);
  return wf_check_launch(ctx, "wf_prefill_gemm_kernel");
}

// plan + projection: the one device path behind eager prefill, flush and forced flush
int run_prefill(wf_drafter* d, PlanParams& pp, int rows_upper, cudaStream_t st) {
  wf_ctx* ctx = d->ctx;
  pp.hidden = d->s.hidden; pp.cap = d->s.backlog_cap; pp.max_pos = d->s.max_pos; pp.row_cap = d->row_cap;
  pp.backlog = d->backlog; pp.backlog_len = d->backlog_len;
  pp.kv = kv_view(d->kv);
  pp.rows = d->d_rows; pp.m_total = d->d_m_total;
  pp.plan_n = d->d_plan; pp.plan_off = d->d_plan + d->kv->s.max_seqs; pp.enq_base = d->d_plan + 2 * d->kv->s.max_seqs;
  pp.status = ctx->d_status;
  wf_launch(wf_prefill_plan_kernel, dim3(1), dim3(1024), 0, st, pp);
  int rc = wf_check_launch(ctx, "wf_prefill_plan_kernel");
  if (rc != WF_OK) return rc;
  rows_upper = rows_upper < d->row_cap ? rows_upper : d->row_cap;
  wf_launch(wf_pack_x_kernel, dim3(rows_upper > 0 ? rows_upper : 1), dim3(256), 0, st, (const RowEntry*)d->d_rows, (const int32_t*)d->d_m_total, d->d_xpack, d->s.hidden);
  rc = wf_check_launch(ctx, "wf_pack_x_kernel");
  if (rc != WF_OK) return rc;
  return d->s.head_dim == 128 ? launch_gemm<128>(d, st) : launch_gemm<64>(d, st);
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
  d->d_wpack = nullptr; d->d_xpack = nullptr; d->d_rope = nullptr; d->d_ws_part = nullptr; d->d_split_cnt = nullptr; d->d_rows = nullptr; d->d_m_total = nullptr; d->d_plan = nullptr;
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
  delete d;
  return WF_OK;
}

extern "C" int wf_kv_only_prefill(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                  const int32_t* n_rows, const int32_t* seq_ids, int B, int max_rows, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows, WF_ERR_INVALID_ARG, "wf_kv_only_prefill: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && max_rows >= 0 && (long long)B * max_rows <= d->row_cap,
             WF_ERR_INVALID_ARG, "wf_kv_only_prefill: B * max_rows exceeds the row table (%d)", d->row_cap);
  WF_REQUIRE(ctx, (uintptr_t)hidden % 16 == 0, WF_ERR_INVALID_ARG, "wf_kv_only_prefill: hidden must be 16-byte aligned");
  if (B == 0 || max_rows == 0) return WF_OK;
  PlanParams pp{};
  pp.mode = PLAN_EAGER; pp.B = B;
  pp.hidden_rows = (const __nv_bfloat16*)hidden; pp.q_indptr = q_indptr; pp.n_rows = n_rows; pp.seq_ids = seq_ids;
  pp.mask = nullptr;
  return run_prefill(d, pp, B * max_rows, (cudaStream_t)stream);
}

extern "C" int wf_lazy_catchup_flush(wf_ctx* ctx, wf_drafter* d, const int32_t* flush_mask, int B, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs, WF_ERR_INVALID_ARG, "wf_lazy_catchup_flush: bad B");
  WF_REQUIRE(ctx, d->s.backlog_cap > 0, WF_ERR_INVALID_ARG, "wf_lazy_catchup_flush: drafter has no backlog");
  if (B == 0) return WF_OK;
  PlanParams pp{};
  pp.mode = PLAN_FLUSH; pp.B = B; pp.mask = flush_mask;
  return run_prefill(d, pp, B * d->s.backlog_cap, (cudaStream_t)stream);
}

namespace {
// copy rows 0..n_rows[b]-1 of each idle sequence's block to the tail of its backlog (FIFO)
__global__ void wf_enqueue_kernel(const __nv_bfloat16* __restrict__ hidden, const int32_t* __restrict__ q_indptr,
                                  const int32_t* __restrict__ n_rows, const int32_t* __restrict__ seq_ids,
                                  const int32_t* __restrict__ idle_mask, __nv_bfloat16* __restrict__ backlog,
                                  const int32_t* __restrict__ backlog_len, int hidden_dim, int cap) {
  wf_pdl_trigger();
  wf_pdl_wait();
  const int b = blockIdx.y, t = blockIdx.x;
  if (!idle_mask[b]) return;
  const int n = n_rows[b];
  if (t >= n || n > cap) return;
  const int sq = seq_ids ? seq_ids[b] : b;
  const uint4* src = reinterpret_cast<const uint4*>(hidden + (size_t)(q_indptr[b] + t) * hidden_dim);
  uint4* dst = reinterpret_cast<uint4*>(backlog + ((size_t)sq * cap + backlog_len[sq] + t) * hidden_dim);
  for (int i = threadIdx.x; i < hidden_dim / 8; i += blockDim.x) dst[i] = src[i];
}
// ROUND: rows 0..n_rows[b]-1 of each block go to backlog[seq][enq_base[b] + t] (enq_base < 0: nothing to enqueue);
// the lengths were already advanced by the plan
__global__ void wf_enqueue_round_kernel(const __nv_bfloat16* __restrict__ hidden, const int32_t* __restrict__ q_indptr,
                                        const int32_t* __restrict__ n_rows, const int32_t* __restrict__ seq_ids,
                                        const int32_t* __restrict__ enq_base, __nv_bfloat16* __restrict__ backlog,
                                        int hidden_dim, int cap) {
  wf_pdl_trigger();
  wf_pdl_wait();
  const int b = blockIdx.y, t = blockIdx.x;
  const int base = enq_base[b];
  if (base < 0 || t >= n_rows[b]) return;
  const int sq = seq_ids ? seq_ids[b] : b;
  const uint4* src = reinterpret_cast<const uint4*>(hidden + (size_t)(q_indptr[b] + t) * hidden_dim);
  uint4* dst = reinterpret_cast<uint4*>(backlog + ((size_t)sq * cap + base + t) * hidden_dim);
  for (int i = threadIdx.x; i < hidden_dim / 8; i += blockDim.x) dst[i] = src[i];
}
__global__ void wf_enqueue_len_kernel(const int32_t* __restrict__ n_rows, const int32_t* __restrict__ seq_ids,
                                      const int32_t* __restrict__ idle_mask, int32_t* __restrict__ backlog_len, int B, int cap) {
  wf_pdl_trigger();
  wf_pdl_wait();
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < B && idle_mask[b] && n_rows[b] <= cap) backlog_len[seq_ids ? seq_ids[b] : b] += n_rows[b];
}
}  // namespace

extern "C" int wf_lazy_catchup_enqueue(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                       const int32_t* n_rows, const int32_t* seq_ids, const int32_t* idle_mask,
                                       int B, int max_rows, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows && idle_mask, WF_ERR_INVALID_ARG, "wf_lazy_catchup_enqueue: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && max_rows >= 0, WF_ERR_INVALID_ARG, "wf_lazy_catchup_enqueue: bad B");
  WF_REQUIRE(ctx, d->s.backlog_cap > 0 && max_rows <= d->s.backlog_cap, WF_ERR_INVALID_ARG,
             "wf_lazy_catchup_enqueue: max_rows exceeds backlog_cap");
  if (B == 0 || max_rows == 0) return WF_OK;
  cudaStream_t st = (cudaStream_t)stream;
  // (1) forced flush of the sequences whose backlog would overflow (C20): same device path as flush
  PlanParams pp{};
  pp.mode = PLAN_FORCED; pp.B = B;
  pp.q_indptr = q_indptr; pp.n_rows = n_rows; pp.seq_ids = seq_ids; pp.mask = idle_mask;
  int rc = run_prefill(d, pp, B * d->s.backlog_cap, st);
  if (rc != WF_OK) return rc;
  // (2) append the rows, (3) advance the lengths
  wf_launch(wf_enqueue_kernel, dim3(max_rows, B), dim3(128), 0, st, (const __nv_bfloat16*)hidden, q_indptr, n_rows, seq_ids, idle_mask,
            const_cast<__nv_bfloat16*>(d->backlog), (const int32_t*)d->backlog_len, d->s.hidden, d->s.backlog_cap);
  rc = wf_check_launch(ctx, "wf_enqueue_kernel");
  if (rc != WF_OK) return rc;
  wf_launch(wf_enqueue_len_kernel, dim3((B + 255) / 256), dim3(256), 0, st, n_rows, seq_ids, idle_mask, d->backlog_len, B, d->s.backlog_cap);
  return wf_check_launch(ctx, "wf_enqueue_len_kernel");
}

extern "C" int wf_lazy_catchup_round(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                     const int32_t* n_rows, const int32_t* seq_ids, const int32_t* idle_mask,
                                     const int32_t* flush_mask, int B, int max_rows, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows, WF_ERR_INVALID_ARG, "wf_lazy_catchup_round: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && B <= KV_RESERVE_SMEM && max_rows >= 0 && max_rows <= 64, WF_ERR_INVALID_ARG,
             "wf_lazy_catchup_round: need B <= min(max_seqs, %d) and max_rows <= 64", KV_RESERVE_SMEM);
  WF_REQUIRE(ctx, !idle_mask || (d->s.backlog_cap > 0 && max_rows <= d->s.backlog_cap), WF_ERR_INVALID_ARG,
             "wf_lazy_catchup_round: idle sequences need a backlog with max_rows <= backlog_cap");
  WF_REQUIRE(ctx, (long long)B * (d->s.backlog_cap + max_rows) <= d->row_cap, WF_ERR_INVALID_ARG,
             "wf_lazy_catchup_round: B * (backlog_cap + max_rows) exceeds the row table (%d)", d->row_cap);
  WF_REQUIRE(ctx, (uintptr_t)hidden % 16 == 0, WF_ERR_INVALID_ARG, "wf_lazy_catchup_round: hidden must be 16-byte aligned");
  if (B == 0 || max_rows == 0) return WF_OK;
  cudaStream_t st = (cudaStream_t)stream;
  PlanParams pp{};
  pp.mode = PLAN_ROUND; pp.B = B;
  pp.hidden_rows = (const __nv_bfloat16*)hidden; pp.q_indptr = q_indptr; pp.n_rows = n_rows; pp.seq_ids = seq_ids;
  pp.mask = idle_mask; pp.mask2 = flush_mask;
  int rc = run_prefill(d, pp, B * (d->s.backlog_cap + max_rows), st);
  if (rc != WF_OK || !idle_mask) return rc;
  // the projection's operand was packed from the backlog by wf_pack_x_kernel (stream order): the backlog may be overwritten
  wf_launch(wf_enqueue_round_kernel, dim3(max_rows, B), dim3(128), 0, st, (const __nv_bfloat16*)hidden, q_indptr, n_rows, seq_ids,
            (const int32_t*)(d->d_plan + 2 * d->kv->s.max_seqs), const_cast<__nv_bfloat16*>(d->backlog), d->s.hidden, d->s.backlog_cap);
  return wf_check_launch(ctx, "wf_enqueue_round_kernel");
}

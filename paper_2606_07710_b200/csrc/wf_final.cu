// (f3) The final backlog token through the drafter layer in full.
// PAPER.md:119 (§3.4: "processing only the final token in full, so that its post-MLP hidden state can feed the next
// draft round"), :206; readings F1-F6.
//
// Per selected sequence b (it switched to this drafter this round) the token is the last row the catch-up prefill
// appended: hidden row n_rows[b]-1 of the block, position p = seq_len[b] - 1, K/V already in the drafter's cache (F1).
// Per layer l (independent branches over the same row x, C14 / F3):
//     q = RoPE(x W_Q, p);  att = softmax(q K^T / sqrt(D)) V over positions 0..p;  y = x + att W_O;
//     h = y + GELU_tanh(y W_up) W_down.
// Launches (all asynchronous, programmatic dependent launch, nothing crosses the host):
//   plan     : compacts the selected sequences (ascending b) into token slots m, gathers their rows, writes the
//              per-sequence query offsets the attention kernel walks (one row for a selected sequence, none otherwise);
//   GEMM x4  : Q, O, up, down.  At the token counts of a switch (<= the batch) these are weight streams: one CTA per
//              (128 output columns, K split), operands swapped as in the KV-only projection (the 128 output columns
//              are the UMMA M dimension, the tokens the N dimension), W repacked once into contiguous pre-swizzled
//              stage images (one cp.async.bulk per stage), X fetched by TMA from the row-major activation the previous
//              step wrote (128-byte swizzle = the K-major UMMA layout), fp32 accumulators in TMEM, fixed-order split-K,
//              and the step's own epilogue: RoPE (Q), residual (O, down), GELU (up);
//   attention: the chain kernel of wf_attn.cu, one launch per drafter layer, one query row per selected sequence over the
//              drafter's paged cache with seq_len - 1 as the context (the token is the last CACHED one).
#include <math.h>

#include <new>

#include "wf_internal.cuh"
#include "wf_sm100.cuh"

namespace {

constexpr int FT_THREADS = 192;          // warp 0: producer, warp 1: MMA issuer, warps 2-5: epilogue
constexpr int FT_BK = 64;                // one 128-byte swizzle row of bf16
constexpr int FT_KSUB = 2;               // 64-wide k-blocks per pipeline stage
constexpr int FT_TILE = 128;             // output columns per CTA tile = UMMA M
constexpr int FT_MAX_TOK = 256;          // tokens per call = UMMA N (one pass)
constexpr int FT_BOX = 32;               // token rows per TMA box of the X operand
constexpr int FT_SMEM = 200 * 1024;
constexpr int FT_MAX_STAGES = 12;
constexpr int FT_W_PRE = 4;               // weight stages prefetched ahead of the dependency wait (128 KB)
constexpr int FT_W_SUB = FT_BK * FT_TILE * 2;        // one k-block of a W tile: 2 column halves x [64 k][128 B] = 16 KB
constexpr int FT_W_BYTES = FT_KSUB * FT_W_SUB;       // one W stage, contiguous in the packed image
constexpr int FT_PLAN_THREADS = 256;
constexpr int FT_MAX_B = 1024;

enum { EPI_Q = 0, EPI_O = 1, EPI_UP = 2, EPI_DOWN = 3 };

struct FtTok {
  int32_t b;                             // sequence (row of h_out, block-table row)
  int32_t pos;                           // position of the token = seq_len[b] - 1 (F1)
};

// ---- plan: who is selected, token slots, gathered rows -------------------------------------------
struct FtPlanParams {
  const __nv_bfloat16* hidden;           // [sum_q][hid]
  const int32_t* q_indptr;
  const int32_t* n_rows;
  const int32_t* select;                 // [B]; b is selected iff select[b] == select_code (NULL: every b)
  const int32_t* seq_len;                // the drafter cache's lengths (after this round's catch-up prefill)
  int select_code, B, hid, m_cap;
  FtTok* tok;
  int32_t* attn_indptr;                  // [B + 1]
  int32_t* m_total;
  __nv_bfloat16* x_last;                 // [m_cap][hid]
  int* status;
};

__global__ void __launch_bounds__(FT_PLAN_THREADS) wf_final_plan_kernel(const FtPlanParams p) {
  __shared__ int s_b[FT_MAX_TOK];
  __shared__ int s_total;
  const int tid = threadIdx.x, lane = tid & 31;
  wf_pdl_wait();
  wf_pdl_trigger();
  if (tid < 32) {                                             // every CTA derives the same compaction (ascending b)
    int run = 0;
    for (int base = 0; base < p.B; base += 32) {
      const int b = base + lane;
      bool on = false;
      if (b < p.B) {
        const int n = p.n_rows[b], q_b = p.q_indptr[b + 1] - p.q_indptr[b];
        on = (!p.select || p.select[b] == p.select_code) && n > 0 && p.seq_len[b] > 0;
        if (on && n > q_b) {                                  // the row would lie outside the block
          if (blockIdx.x == 0) wf_raise(p.status, (int)WF_ERR_INVALID_ARG);
          on = false;
        }
      }
      const unsigned int bal = __ballot_sync(0xffffffffu, on);
      int idx = run + __popc(bal & ((1u << lane) - 1u));
      if (on && idx >= p.m_cap) {                             // more switches than token slots: dropped, reported
        if (blockIdx.x == 0) wf_raise(p.status, (int)WF_ERR_INVALID_ARG);
        on = false;
      }
      if (b < p.B) {
        if (on) s_b[idx] = b;
        if (blockIdx.x == 0) {
          p.attn_indptr[b] = min(idx, p.m_cap);
          if (on) p.tok[idx] = FtTok{b, p.seq_len[b] - 1};
        }
      }
      run = min(run + __popc(bal), p.m_cap);
    }
    if (lane == 0) {
      s_total = run;
      if (blockIdx.x == 0) { p.attn_indptr[p.B] = run; *p.m_total = run; }
    }
  }
  __syncthreads();
  const int total = s_total;
  for (int m = blockIdx.x; m < total; m += gridDim.x) {
    const int b = s_b[m];
    const uint4* src = reinterpret_cast<const uint4*>(p.hidden + (size_t)(p.q_indptr[b] + p.n_rows[b] - 1) * p.hid);
    uint4* dst = reinterpret_cast<uint4*>(p.x_last + (size_t)m * p.hid);
    for (int i = tid; i < p.hid / 8; i += FT_PLAN_THREADS) dst[i] = __ldg(src + i);
  }
}

// ---- one-time repack of a weight matrix [K][N] into stage images -----------------------------------
// tile (128 output columns) x k-block (64 rows) -> 2 column halves x [64 k][128 B], 16-byte chunks XOR-swizzled with
// k & 7: the 128-byte-swizzled MN-major image the UMMA A descriptor reads; a stage is one contiguous bulk copy.
__global__ void wf_final_pack_w_kernel(const __nv_bfloat16* __restrict__ w, uint8_t* __restrict__ dst, int K, int N) {
  const int kb = blockIdx.x, tile = blockIdx.y, n_kb = K / FT_BK;
  uint8_t* out = dst + ((size_t)tile * n_kb + kb) * FT_W_SUB;
  for (int i = threadIdx.x; i < FT_BK * FT_TILE / 8; i += blockDim.x) {
    const int k = i / (FT_TILE / 8), c16 = i % (FT_TILE / 8);
    const int j = c16 >> 3, cc = c16 & 7;
    const uint4 v = *reinterpret_cast<const uint4*>(w + (size_t)(kb * FT_BK + k) * N + tile * FT_TILE + c16 * 8);
    *reinterpret_cast<uint4*>(out + j * 8192 + k * 128 + ((cc ^ (k & 7)) << 4)) = v;
  }
}

// ---- the weight-streaming GEMM -----------------------------------------------------------------
struct FtGemmParams {
  const uint8_t* wpack;                  // [L][N/128][K/64][16 KB]
  const CUtensorMap* xmap;               // X as bf16 [rows][K], box {64 columns, 32 rows}, 128-byte swizzle
  int K, N, L, m_cap;
  int x_per_layer;                       // 1: layer l reads rows [l * m_cap, ...) of X; 0: every layer reads rows [0, ...)
  int n_split;                           // CTAs per tile along K (fixed per matrix shape: the summation order never varies)
  float* ws_part;                        // [tiles][n_split][m_cap][128] fp32 (n_split > 1)
  unsigned int* cnt;                     // [tiles], self-resetting
  const int32_t* m_total;
  const FtTok* tok;
  // epilogues
  const float2* rope;                    // EPI_Q: [max_pos][D/2] (cos, sin)
  int D, hidden, max_pos;
  __nv_bfloat16* q_out;                  // EPI_Q   : [L][m_cap][N]
  const __nv_bfloat16* x_res;            // EPI_O   : [m_cap][hidden], the residual
  float* y32;                            // EPI_O out / EPI_DOWN in: [L][m_cap][hidden]
  __nv_bfloat16* y16;                    // EPI_O out: the operand copy of y
  __nv_bfloat16* g16;                    // EPI_UP out: [L][m_cap][N]
  __nv_bfloat16* h_out;                  // EPI_DOWN out: [B][L][hidden]
};

__device__ __forceinline__ float gelu_tanh(float u) {
  return 0.5f * u * (1.f + tanhf(0.7978845608028654f * (u + 0.044715f * u * u * u)));
}

template <int EPI>
__global__ void __launch_bounds__(FT_THREADS, 1) wf_final_gemm_kernel(const __grid_constant__ FtGemmParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  // Two rings, as in the KV-only projection (wf_prefill.cu): W stages at offset 0, the first FT_W_PRE of them filled BEFORE
  // the dependency wait (the weights are constants; under programmatic dependent launch the head of this kernel's weight
  // stream overlaps the tail of the kernel that produces its activations), then the X ring, sized by the call's tokens.
  __shared__ __align__(8) uint64_t w_full[FT_MAX_STAGES], w_empty[FT_MAX_STAGES], x_full[FT_MAX_STAGES], x_empty[FT_MAX_STAGES], s_acc_full;
  __shared__ uint32_t s_tmem;
  __shared__ int s_last;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if constexpr (EPI != EPI_Q) {
    // O / up / down: the token count was written by the plan kernel, at least two launches back, and every kernel in
    // between triggered its successor only after its own dependency wait: the count is final when this CTA starts.  A call
    // in which nobody switched leaves before it has prefetched a byte of weights or allocated TMEM.
    if (*reinterpret_cast<const volatile int32_t*>(p.m_total) == 0) {
      wf_pdl_wait();
      wf_pdl_trigger();
      return;
    }
  }
  const int tile = (int)blockIdx.x / p.n_split, split = (int)blockIdx.x % p.n_split;
  const int tiles_n = p.N / FT_TILE;
  const int layer = tile / tiles_n, nt = tile % tiles_n;
  const int n_kb_tile = p.K / (FT_KSUB * FT_BK);
  const int n_kb = n_kb_tile / p.n_split, kb0 = split * n_kb;
  const int n_pre = min(n_kb, FT_W_PRE);
  if (tid == 0) {
    for (int i = 0; i < FT_MAX_STAGES; ++i) {
      mbar_init(smem_u32(&w_full[i]), 1); mbar_init(smem_u32(&w_empty[i]), 1);
      mbar_init(smem_u32(&x_full[i]), 1); mbar_init(smem_u32(&x_empty[i]), 1);
    }
    mbar_init(smem_u32(&s_acc_full), 1);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(smem_u32(&s_tmem), FT_MAX_TOK);
  if (warp == 0 && lane == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(p.xmap)) : "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = s_tmem;
  const uint8_t* w_tile = p.wpack + ((size_t)tile * n_kb_tile + kb0) * FT_W_BYTES;
  if (warp == 0 && elect_one()) {
    for (int s2 = 0; s2 < n_pre; ++s2) {
      mbar_arrive_expect_tx(smem_u32(&w_full[s2]), FT_W_BYTES);
      bulk_load(smem_u32(smem) + s2 * FT_W_BYTES, w_tile + (size_t)s2 * FT_W_BYTES, FT_W_BYTES, smem_u32(&w_full[s2]));
    }
  }
  __syncwarp();
  wf_pdl_wait();
  wf_pdl_trigger();
  const int M = min(*p.m_total, p.m_cap);
  if (M == 0) {
    // nobody switched: let the prefetched stages land (shared memory must outlive the copies), return the TMEM columns
    if (warp == 0) for (int s2 = 0; s2 < n_pre; ++s2) mbar_wait(smem_u32(&w_full[s2]), 0);
    if (warp == 1) tmem_dealloc(tmem_base, FT_MAX_TOK);
    return;
  }
  const int n_box = (M + FT_BOX - 1) / FT_BOX;
  const int x_sub = n_box * FT_BOX * 128;                     // one 64-wide k-block of the X operand (whole boxes)
  const int x_stage = FT_KSUB * x_sub;
  const int n_sw = (FT_SMEM - (FT_W_PRE + 1) * FT_W_BYTES) >= 2 * x_stage ? FT_W_PRE + 1 : FT_W_PRE;
  const int n_sx = max(1, min(FT_MAX_STAGES, (FT_SMEM - n_sw * FT_W_BYTES) / x_stage));
  uint8_t* w_base = smem;
  uint8_t* x_base = smem + (size_t)n_sw * FT_W_BYTES;

  if (warp == 0) {
    // ===== producer: per stage one bulk copy of the W image and n_box TMA boxes per X k-block =====
    const uint8_t* w_kb = w_tile;
    const uint32_t wf0 = smem_u32(&w_full[0]), we0 = smem_u32(&w_empty[0]), xf0 = smem_u32(&x_full[0]), xe0 = smem_u32(&x_empty[0]);
    const uint32_t x0 = smem_u32(x_base), w0 = smem_u32(w_base);
    const int row0 = p.x_per_layer ? layer * p.m_cap : 0;
    int sw = 0, sx = 0;
    uint32_t phw = 1, phx = 1;
    for (int kb = 0; kb < n_kb; ++kb) {
      if (kb >= n_pre) {
        mbar_wait(we0 + 8 * sw, phw);
        if (elect_one()) {
          mbar_arrive_expect_tx(wf0 + 8 * sw, FT_W_BYTES);
          bulk_load(w0 + sw * FT_W_BYTES, w_kb, FT_W_BYTES, wf0 + 8 * sw);
        }
      }
      mbar_wait(xe0 + 8 * sx, phx);
      if (elect_one()) {
        const uint32_t bar = xf0 + 8 * sx;
        mbar_arrive_expect_tx(bar, FT_KSUB * x_sub);
        for (int u = 0; u < FT_KSUB; ++u)
          for (int bx = 0; bx < n_box; ++bx)
            tma_load_2d(x0 + sx * x_stage + u * x_sub + bx * (FT_BOX * 128), p.xmap, ((kb0 + kb) * FT_KSUB + u) * FT_BK,
                        row0 + bx * FT_BOX, bar);
      }
      __syncwarp();
      w_kb += FT_W_BYTES;
      if (++sw == n_sw) { sw = 0; phw ^= 1; }
      if (++sx == n_sx) { sx = 0; phx ^= 1; }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: A = W tile (MN-major), B = X rows (K-major), D[128 columns x tokens] in TMEM =====
    const uint64_t dw0 = umma_desc(smem_u32(w_base), 8192, 1024);
    const uint64_t dx0 = umma_desc(smem_u32(x_base), 16, 1024);
    const uint32_t wf0 = smem_u32(&w_full[0]), we0 = smem_u32(&w_empty[0]), xf0 = smem_u32(&x_full[0]), xe0 = smem_u32(&x_empty[0]);
    const uint64_t dw_step = (uint64_t)(FT_W_BYTES >> 4), dx_step = (uint64_t)(x_stage >> 4);
    const uint32_t idesc = umma_idesc_mn_k(128, (M + 15) & ~15);
    int sw = 0, sx = 0;
    uint32_t phw = 0, phx = 0;
    uint64_t dw = dw0, dx = dx0;
    for (int kb = 0; kb < n_kb; ++kb) {
      mbar_wait(wf0 + 8 * sw, phw);
      mbar_wait(xf0 + 8 * sx, phx);
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int k16 = 0; k16 < FT_KSUB * FT_BK / 16; ++k16)
          umma_bf16(tmem_base, dw + (uint64_t)(((k16 >> 2) * FT_W_SUB + (k16 & 3) * 2048) >> 4),
                    dx + (uint64_t)(((k16 >> 2) * x_sub + (k16 & 3) * 32) >> 4), idesc, (kb | k16) != 0);
        umma_commit(we0 + 8 * sw);
        umma_commit(xe0 + 8 * sx);
      }
      __syncwarp();
      dw += dw_step; dx += dx_step;
      if (++sw == n_sw) { sw = 0; phw ^= 1; dw = dw0; }
      if (++sx == n_sx) { sx = 0; phx ^= 1; dx = dx0; }
    }
    if (elect_one()) umma_commit(smem_u32(&s_acc_full));
    __syncwarp();
  } else {
    // ===== warps 2-5: epilogue.  TMEM lane = output column of the tile, TMEM column = token. =====
    const int quarter = warp & 3;
    const int et = quarter * 32 + lane;                       // 0..127 = column of the tile
    float* tr = reinterpret_cast<float*>(smem);               // [token][128] fp32 (the ring is idle by then)
    const int n_pad = (M + 15) & ~15;
    mbar_wait(smem_u32(&s_acc_full), 0);
    tc_fence_after();
    bool finish = true;
    float* mine = p.n_split > 1 ? p.ws_part + ((size_t)(tile * p.n_split + split) * p.m_cap) * FT_TILE : tr;
    for (int col0 = 0; col0 < n_pad; col0 += 32) {
      uint32_t v[32];
      tmem_ld32(tmem_base + ((uint32_t)(quarter * 32) << 16) + col0, v);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 32; ++j)
        if (col0 + j < M) mine[(size_t)(col0 + j) * FT_TILE + et] = __uint_as_float(v[j]);
    }
    tc_fence_before();
    if (p.n_split > 1) {
      // split-K: the last CTA of the tile to arrive sums the partials in split order 0, 1, ... (its own re-read from
      // L2), so the bits do not depend on which CTA finishes last
      __threadfence();
      named_bar_sync(1, 128);
      if (et == 0) {
        const unsigned int old = atomicAdd(&p.cnt[tile], 1u);
        s_last = old == (unsigned int)p.n_split - 1;
        if (s_last) p.cnt[tile] = 0;
      }
      named_bar_sync(1, 128);
      finish = s_last != 0;
      if (finish) {
        __threadfence();
        const float4* part0 = reinterpret_cast<const float4*>(p.ws_part + (size_t)tile * p.n_split * p.m_cap * FT_TILE);
        const size_t stride4 = (size_t)p.m_cap * FT_TILE / 4;
        for (int i = et; i < M * (FT_TILE / 4); i += 128) {
          float4 acc = __ldcg(part0 + i);
          for (int sp = 1; sp < p.n_split; ++sp) {
            const float4 x = __ldcg(part0 + sp * stride4 + i);
            acc.x += x.x; acc.y += x.y; acc.z += x.z; acc.w += x.w;
          }
          reinterpret_cast<float4*>(tr)[i] = acc;
        }
      }
    }
    named_bar_sync(1, 128);
    if (finish) {
      const int c0 = nt * FT_TILE;                            // first output column of the tile
      if constexpr (EPI == EPI_Q) {
        // RoPE on the (r, r + D/2) pairs of each head inside the tile (D = 128: one head; D = 64: two), bf16 RNE
        const int half = p.D / 2, pph = half / 8, n_pc = FT_TILE / 16;   // 8-column pair chunks per head / per tile
        for (int idx = et; idx < M * n_pc; idx += 128) {
          const int t = idx / n_pc, pc = idx % n_pc;
          const int lo = (pc / pph) * p.D + (pc % pph) * 8, hi = lo + half, r0 = (pc % pph) * 8;
          const float* a = tr + t * FT_TILE + lo;
          const float* b = tr + t * FT_TILE + hi;
          const float4* cs = reinterpret_cast<const float4*>(p.rope + (size_t)min(p.tok[t].pos, p.max_pos - 1) * half + r0);
          uint32_t olo[4], ohi[4];
#pragma unroll
          for (int i = 0; i < 8; i += 2) {
            const float4 c2 = __ldg(cs + i / 2);              // (cos, sin) of r0 + i and r0 + i + 1
            olo[i / 2] = pack_bf16(a[i] * c2.x - b[i] * c2.y, a[i + 1] * c2.z - b[i + 1] * c2.w);
            ohi[i / 2] = pack_bf16(b[i] * c2.x + a[i] * c2.y, b[i + 1] * c2.z + a[i + 1] * c2.w);
          }
          __nv_bfloat16* dst = p.q_out + ((size_t)layer * p.m_cap + t) * p.N + c0;
          *reinterpret_cast<uint4*>(dst + lo) = make_uint4(olo[0], olo[1], olo[2], olo[3]);
          *reinterpret_cast<uint4*>(dst + hi) = make_uint4(ohi[0], ohi[1], ohi[2], ohi[3]);
        }
      } else {
        for (int idx = et; idx < M * (FT_TILE / 8); idx += 128) {
          const int t = idx / (FT_TILE / 8), c = (idx % (FT_TILE / 8)) * 8;
          const float4 a0 = *reinterpret_cast<const float4*>(tr + t * FT_TILE + c);
          const float4 a1 = *reinterpret_cast<const float4*>(tr + t * FT_TILE + c + 4);
          float v[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
          const size_t row = (size_t)layer * p.m_cap + t;
          if constexpr (EPI == EPI_O) {
            const uint4 xr = __ldg(reinterpret_cast<const uint4*>(p.x_res + (size_t)t * p.hidden + c0 + c));
            const uint32_t xw[4] = {xr.x, xr.y, xr.z, xr.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              v[2 * i] += __uint_as_float(xw[i] << 16);
              v[2 * i + 1] += __uint_as_float(xw[i] & 0xffff0000u);
            }
            float4* y = reinterpret_cast<float4*>(p.y32 + row * p.hidden + c0 + c);
            y[0] = make_float4(v[0], v[1], v[2], v[3]);
            y[1] = make_float4(v[4], v[5], v[6], v[7]);
            *reinterpret_cast<uint4*>(p.y16 + row * p.hidden + c0 + c) =
                make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
          } else if constexpr (EPI == EPI_UP) {
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = gelu_tanh(v[i]);
            *reinterpret_cast<uint4*>(p.g16 + row * p.N + c0 + c) =
                make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
          } else {
            const float4* y = reinterpret_cast<const float4*>(p.y32 + row * p.hidden + c0 + c);
            const float4 y0 = y[0], y1 = y[1];
            v[0] += y0.x; v[1] += y0.y; v[2] += y0.z; v[3] += y0.w;
            v[4] += y1.x; v[5] += y1.y; v[6] += y1.z; v[7] += y1.w;
            *reinterpret_cast<uint4*>(p.h_out + ((size_t)p.tok[t].b * p.L + layer) * p.hidden + c0 + c) =
                make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, FT_MAX_TOK);
}

int pick_split(int tiles, int stages, int sm_count) {
  int ns = 1;
  while (ns * 2 <= 8 && tiles * ns * 2 <= sm_count && stages % (ns * 2) == 0) ns *= 2;
  return ns;
}

}  // namespace

struct wf_full_layer {
  int n_q_heads, ffn, m_cap;
  uint8_t* w[4];                         // packed W_Q, W_O, W_up, W_down of every layer
  __nv_bfloat16 *x_last, *q_buf, *att, *y16, *g16;
  float* y32;
  FtTok* tok;
  int32_t* attn_indptr;
  int32_t* m_total;
  float* ws_part;
  unsigned int* cnt;                     // [4][tiles_max]
  int tiles_max;
  CUtensorMap* d_maps;                   // [4]: x_last, att, y16, g16
  int ns[4];
};

void wf_full_layer_destroy(wf_full_layer* f) {
  if (!f) return;
  for (int i = 0; i < 4; ++i) cudaFree(f->w[i]);
  cudaFree(f->x_last); cudaFree(f->q_buf); cudaFree(f->att); cudaFree(f->y16); cudaFree(f->g16); cudaFree(f->y32);
  cudaFree(f->tok); cudaFree(f->attn_indptr); cudaFree(f->m_total); cudaFree(f->ws_part); cudaFree(f->cnt); cudaFree(f->d_maps);
  delete f;
}

extern "C" int wf_drafter_set_full_layer(wf_ctx* ctx, wf_drafter* d, int n_q_heads, int ffn, int max_tokens,
                                         const void* const* w_q_host_ptrs, const void* const* w_o_host_ptrs,
                                         const void* const* w_up_host_ptrs, const void* const* w_down_host_ptrs) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, w_q_host_ptrs && w_o_host_ptrs && w_up_host_ptrs && w_down_host_ptrs, WF_ERR_INVALID_ARG,
             "wf_drafter_set_full_layer: null argument");
  WF_REQUIRE(ctx, !d->full, WF_ERR_INVALID_ARG, "wf_drafter_set_full_layer: already set");
  const int L = d->s.n_layers, D = d->s.head_dim, hid = d->s.hidden, Hkv = d->s.n_kv_heads;
  WF_REQUIRE(ctx, n_q_heads > 0 && n_q_heads % Hkv == 0 && n_q_heads / Hkv <= 64, WF_ERR_INVALID_ARG,
             "wf_drafter_set_full_layer: n_q_heads must be a multiple of n_kv_heads (group <= 64)");
  const int qd = n_q_heads * D;
  WF_REQUIRE(ctx, hid % 128 == 0 && qd % 128 == 0 && ffn > 0 && ffn % 128 == 0, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_drafter_set_full_layer: hidden, n_q_heads * head_dim and ffn must be multiples of 128");
  WF_REQUIRE(ctx, max_tokens >= 1 && max_tokens <= FT_MAX_TOK, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_drafter_set_full_layer: max_tokens must be in [1, %d]", FT_MAX_TOK);
  for (int l = 0; l < L; ++l) {
    const void* ws[4] = {w_q_host_ptrs[l], w_o_host_ptrs[l], w_up_host_ptrs[l], w_down_host_ptrs[l]};
    for (int i = 0; i < 4; ++i)
      WF_REQUIRE(ctx, ws[i] && (uintptr_t)ws[i] % 16 == 0, WF_ERR_INVALID_ARG, "wf_drafter_set_full_layer: weight pointer null or unaligned");
  }
  wf_full_layer* f = new (std::nothrow) wf_full_layer();
  if (!f) return wf_set_error(ctx, WF_ERR_INVALID_ARG, "wf_drafter_set_full_layer: host allocation failed");
  *f = wf_full_layer{};
  f->n_q_heads = n_q_heads; f->ffn = ffn;
  f->m_cap = (max_tokens + FT_BOX - 1) / FT_BOX * FT_BOX;
  const int m_cap = f->m_cap;
  // K and N of the four matrices: Q [hid][qd], O [qd][hid], up [hid][ffn], down [ffn][hid]
  const int Ks[4] = {hid, qd, hid, ffn}, Ns[4] = {qd, hid, ffn, hid};
  size_t part_elems = 0;
  f->tiles_max = 0;
  for (int i = 0; i < 4; ++i) {
    const int tiles = L * (Ns[i] / FT_TILE);
    f->ns[i] = pick_split(tiles, Ks[i] / (FT_KSUB * FT_BK), ctx->sm_count);
    if (f->ns[i] > 1 && (size_t)tiles * f->ns[i] * m_cap * FT_TILE > part_elems) part_elems = (size_t)tiles * f->ns[i] * m_cap * FT_TILE;
    if (tiles > f->tiles_max) f->tiles_max = tiles;
  }
  cudaError_t e = cudaSuccess;
  for (int i = 0; i < 4 && e == cudaSuccess; ++i) e = cudaMalloc(&f->w[i], (size_t)L * Ks[i] * Ns[i] * 2);
  if (e == cudaSuccess) e = cudaMalloc(&f->x_last, (size_t)m_cap * hid * 2);
  if (e == cudaSuccess) e = cudaMalloc(&f->q_buf, (size_t)L * m_cap * qd * 2);
  if (e == cudaSuccess) e = cudaMalloc(&f->att, (size_t)L * m_cap * qd * 2);
  if (e == cudaSuccess) e = cudaMalloc(&f->y16, (size_t)L * m_cap * hid * 2);
  if (e == cudaSuccess) e = cudaMalloc(&f->y32, (size_t)L * m_cap * hid * 4);
  if (e == cudaSuccess) e = cudaMalloc(&f->g16, (size_t)L * m_cap * ffn * 2);
  if (e == cudaSuccess) e = cudaMalloc(&f->tok, sizeof(FtTok) * m_cap);
  if (e == cudaSuccess) e = cudaMalloc(&f->attn_indptr, sizeof(int32_t) * (d->kv->s.max_seqs + 1));
  if (e == cudaSuccess) e = cudaMalloc(&f->m_total, sizeof(int32_t));
  if (e == cudaSuccess && part_elems) e = cudaMalloc(&f->ws_part, part_elems * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&f->cnt, sizeof(unsigned int) * 4 * f->tiles_max);
  if (e == cudaSuccess) e = cudaMalloc(&f->d_maps, sizeof(CUtensorMap) * 4);
  if (e == cudaSuccess) e = cudaMemset(f->cnt, 0, sizeof(unsigned int) * 4 * f->tiles_max);
  if (e == cudaSuccess) e = cudaMemset(f->m_total, 0, sizeof(int32_t));
  // the activations start as zeros: a TMA box may cover token rows no call has written yet
  if (e == cudaSuccess) e = cudaMemset(f->x_last, 0, (size_t)m_cap * hid * 2);
  if (e == cudaSuccess) e = cudaMemset(f->att, 0, (size_t)L * m_cap * qd * 2);
  if (e == cudaSuccess) e = cudaMemset(f->y16, 0, (size_t)L * m_cap * hid * 2);
  if (e == cudaSuccess) e = cudaMemset(f->g16, 0, (size_t)L * m_cap * ffn * 2);
  if (e != cudaSuccess) {
    wf_full_layer_destroy(f);
    return wf_set_error(ctx, WF_ERR_CUDA, "wf_drafter_set_full_layer: %s", cudaGetErrorString(e));
  }
  const void* const* srcs[4] = {w_q_host_ptrs, w_o_host_ptrs, w_up_host_ptrs, w_down_host_ptrs};
  for (int i = 0; i < 4; ++i)
    for (int l = 0; l < L; ++l)
      wf_final_pack_w_kernel<<<dim3(Ks[i] / FT_BK, Ns[i] / FT_TILE), 256>>>((const __nv_bfloat16*)srcs[i][l],
                                                                          f->w[i] + (size_t)l * Ks[i] * Ns[i] * 2, Ks[i], Ns[i]);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaDeviceSynchronize();     // synchronous: the caller may free or rewrite the weights afterwards
  int rc = WF_OK;
  if (e == cudaSuccess) {
    CUtensorMap maps[4];
    const void* bases[4] = {f->x_last, f->att, f->y16, f->g16};
    const uint64_t rows[4] = {(uint64_t)m_cap, (uint64_t)L * m_cap, (uint64_t)L * m_cap, (uint64_t)L * m_cap};
    for (int i = 0; i < 4 && rc == WF_OK; ++i) rc = wf_make_tmap_2d(ctx, &maps[i], bases[i], rows[i], (uint64_t)Ks[i], FT_BK, FT_BOX);
    if (rc == WF_OK) e = cudaMemcpy(f->d_maps, maps, sizeof(maps), cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess || rc != WF_OK) {
    wf_full_layer_destroy(f);
    return rc != WF_OK ? rc : wf_set_error(ctx, WF_ERR_CUDA, "wf_drafter_set_full_layer: %s", cudaGetErrorString(e));
  }
  d->full = f;
  return WF_OK;
}

extern "C" size_t wf_final_token_workspace_bytes(const wf_drafter* d, int B) {
  if (!d || !d->full) return 16;
  return wf_verify_attn_workspace_bytes(&d->kv->s, B, d->full->n_q_heads, 1);
}

namespace {
template <int EPI>
int launch_gemm(wf_ctx* ctx, const FtGemmParams& gp, int grid, cudaStream_t st) {
  WF_CONFIGURE_ONCE(ctx, WF_FUNC_FINAL_TOKEN + EPI, wf_final_gemm_kernel<EPI>, FT_SMEM);
  wf_launch(wf_final_gemm_kernel<EPI>, dim3(grid), dim3(FT_THREADS), FT_SMEM, st, gp);
  return wf_check_launch(ctx, "wf_final_gemm_kernel");
}
}  // namespace

extern "C" int wf_final_token_full(wf_ctx* ctx, wf_drafter* d, const void* hidden, const int32_t* q_indptr,
                                   const int32_t* n_rows, const int32_t* select, int select_code, int B, void* h_out,
                                   void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx || !d) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, d->full, WF_ERR_INVALID_ARG, "wf_final_token_full: wf_drafter_set_full_layer was not called");
  WF_REQUIRE(ctx, hidden && q_indptr && n_rows && h_out && workspace, WF_ERR_INVALID_ARG, "wf_final_token_full: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= d->kv->s.max_seqs && B <= FT_MAX_B, WF_ERR_INVALID_ARG, "wf_final_token_full: bad B (max %d)", FT_MAX_B);
  WF_REQUIRE(ctx, (uintptr_t)hidden % 16 == 0 && (uintptr_t)h_out % 16 == 0, WF_ERR_INVALID_ARG,
             "wf_final_token_full: hidden / h_out must be 16-byte aligned");
  if (B == 0) return WF_OK;
  wf_full_layer* f = d->full;
  cudaStream_t st = (cudaStream_t)stream;
  const int L = d->s.n_layers, D = d->s.head_dim, hid = d->s.hidden, qd = f->n_q_heads * D, m_cap = f->m_cap;
  FtPlanParams pp;
  pp.hidden = (const __nv_bfloat16*)hidden; pp.q_indptr = q_indptr; pp.n_rows = n_rows; pp.select = select;
  pp.seq_len = d->kv->seq_len; pp.select_code = select_code; pp.B = B; pp.hid = hid; pp.m_cap = m_cap;
  pp.tok = f->tok; pp.attn_indptr = f->attn_indptr; pp.m_total = f->m_total; pp.x_last = f->x_last; pp.status = ctx->d_status;
  const int plan_grid = B < m_cap ? (B < 64 ? B : 64) : (m_cap < 64 ? m_cap : 64);
  wf_launch(wf_final_plan_kernel, dim3(plan_grid), dim3(FT_PLAN_THREADS), 0, st, pp);
  int rc = wf_check_launch(ctx, "wf_final_plan_kernel");
  if (rc != WF_OK) return rc;

  FtGemmParams gp{};
  gp.L = L; gp.m_cap = m_cap; gp.ws_part = f->ws_part; gp.m_total = f->m_total; gp.tok = f->tok;
  gp.rope = d->d_rope; gp.D = D; gp.hidden = hid; gp.max_pos = d->s.max_pos;
  gp.q_out = f->q_buf; gp.x_res = f->x_last; gp.y32 = f->y32; gp.y16 = f->y16; gp.g16 = f->g16; gp.h_out = (__nv_bfloat16*)h_out;
  auto set = [&](int i, int K, int N, int x_per_layer) {
    gp.wpack = f->w[i]; gp.xmap = f->d_maps + i; gp.K = K; gp.N = N; gp.x_per_layer = x_per_layer;
    gp.n_split = f->ns[i]; gp.cnt = f->cnt + (size_t)i * f->tiles_max;
    return L * (N / FT_TILE) * f->ns[i];
  };
  int grid = set(0, hid, qd, 0);
  rc = launch_gemm<EPI_Q>(ctx, gp, grid, st);
  if (rc != WF_OK) return rc;
  const float sm_scale = 1.0f / sqrtf((float)D);
  for (int l = 0; l < L; ++l) {
    rc = wf_attn_launch_chain(ctx, d->kv, l, f->q_buf + (size_t)l * m_cap * qd, f->attn_indptr, B, f->n_q_heads, 1, sm_scale,
                              -1, f->att + (size_t)l * m_cap * qd, workspace, workspace_bytes, stream, "wf_final_token_full");
    if (rc != WF_OK) return rc;
  }
  grid = set(1, qd, hid, 1);
  rc = launch_gemm<EPI_O>(ctx, gp, grid, st);
  if (rc != WF_OK) return rc;
  grid = set(2, hid, f->ffn, 1);
  rc = launch_gemm<EPI_UP>(ctx, gp, grid, st);
  if (rc != WF_OK) return rc;
  grid = set(3, f->ffn, hid, 1);
  return launch_gemm<EPI_DOWN>(ctx, gp, grid, st);
}

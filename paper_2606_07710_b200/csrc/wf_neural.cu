// (f1) WhiFlash-Neural routing policy: dAL = <w2, GELU(W1 h + b1)> + b2, route = AR iff dAL > tau.
// PAPER.md:87 (§3.3.2), :103-107 (decision rule), :325 (App. A: d -> d/8 -> GELU -> dropout -> 1);
// DESIGN.md readings N1-N6.
//
// The policy is a batched GEMV against 2.1 M weights (4.2 MB of bf16 at d = 4096): HBM/latency-bound, no
// tensor cores.  One warp owns one hidden unit j: it streams row j of W1 exactly once per tile of 16
// sequences (16-byte coalesced loads; the tiles are spread over blockIdx.y) against the 16 hidden rows staged in shared memory, reduces with a
// fixed shuffle tree, applies bias and the exact (erf) GELU and scales by w2[j].  A CTA (8 warps = 8 units)
// adds its 8 terms in unit order and publishes one partial per sequence; the last CTA to finish (self-
// resetting counter) adds the partials in CTA order, adds b2 and thresholds.  Every sum has a fixed order:
// the decision is deterministic.
#include "wf_internal.cuh"

namespace {

constexpr int NR_WARPS = 8;            // hidden units per CTA (4 per CTA doubles the CTAs that each stage the 16 rows: 34 us against 24 at B = 16)
constexpr int NR_TILE_B = 16;          // sequences staged per pass
constexpr int NR_THREADS = NR_WARPS * 32;

struct NeuralParams {
  const __nv_bfloat16* hidden;         // [sum_q][d]
  const int32_t* q_indptr;
  const int32_t* accept_len;           // nullable
  const __nv_bfloat16* w1;             // [m][d]
  const float* b1;                     // [m]
  const __nv_bfloat16* w2;             // [m]
  const float* b2;                     // [1]
  const float* tau;
  float* delta_al;
  int32_t* route;
  float* ws;                           // [gridDim.x][B] partial sums
  unsigned int* counter;
  int B, d, m, tau_is_scalar;
};

__device__ __forceinline__ float bf16_lo(uint32_t x) { return __uint_as_float(x << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t x) { return __uint_as_float(x & 0xffff0000u); }

__device__ __forceinline__ float dot8(const uint4& a, const uint4& b, float acc) {
  acc = fmaf(bf16_lo(a.x), bf16_lo(b.x), acc); acc = fmaf(bf16_hi(a.x), bf16_hi(b.x), acc);
  acc = fmaf(bf16_lo(a.y), bf16_lo(b.y), acc); acc = fmaf(bf16_hi(a.y), bf16_hi(b.y), acc);
  acc = fmaf(bf16_lo(a.z), bf16_lo(b.z), acc); acc = fmaf(bf16_hi(a.z), bf16_hi(b.z), acc);
  acc = fmaf(bf16_lo(a.w), bf16_lo(b.w), acc); acc = fmaf(bf16_hi(a.w), bf16_hi(b.w), acc);
  return acc;
}

__global__ void __launch_bounds__(NR_THREADS) wf_neural_route_kernel(const NeuralParams p) {
  extern __shared__ __align__(16) uint8_t smem[];          // [NR_TILE_B][d] bf16
  __shared__ float s_term[NR_WARPS][NR_TILE_B];
  __shared__ int s_last;
  wf_pdl_wait();
  wf_pdl_trigger();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int chunks = p.d / 8;                               // 16-byte chunks per row
  const int j = blockIdx.x * NR_WARPS + warp;               // this warp's hidden unit
  const uint4* wrow = reinterpret_cast<const uint4*>(p.w1 + (size_t)min(j, p.m - 1) * p.d);
  uint4* hs = reinterpret_cast<uint4*>(smem);

  // blockIdx.y = tile of 16 sequences (the tiles run side by side: at B = 64 one CTA per unit group walking four tiles in turn
  // took 108 us on 64 SMs)
  for (int b0 = blockIdx.y * NR_TILE_B; b0 < p.B; b0 += gridDim.y * NR_TILE_B) {
    const int nb = min(NR_TILE_B, p.B - b0);
    // stage row a_b of each block (reading N4); an empty block stages zeros
    for (int i = tid; i < nb * chunks; i += NR_THREADS) {
      const int s = i / chunks, c = i % chunks, b = b0 + s;
      const int r0 = p.q_indptr[b], q_b = p.q_indptr[b + 1] - r0;
      uint4 v = make_uint4(0, 0, 0, 0);
      if (q_b > 0) {
        const int a = p.accept_len ? min(max(p.accept_len[b], 0), q_b - 1) : 0;
        v = __ldg(reinterpret_cast<const uint4*>(p.hidden + (size_t)(r0 + a) * p.d) + c);
      }
      hs[s * chunks + c] = v;
    }
    __syncthreads();
    float acc[NR_TILE_B];
#pragma unroll
    for (int s = 0; s < NR_TILE_B; ++s) acc[s] = 0.f;
    if (j < p.m) {
      // 8 chunks of the W1 row are in flight per lane before the first is used: the row costs two round trips at
      // d = 4096 instead of sixteen
      constexpr int WU = 8;
      for (int c0 = lane; c0 < chunks; c0 += 32 * WU) {
        uint4 wv[WU];
#pragma unroll
        for (int u = 0; u < WU; ++u)
          if (c0 + 32 * u < chunks) wv[u] = __ldg(wrow + c0 + 32 * u);
#pragma unroll
        for (int u = 0; u < WU; ++u) {
          const int c = c0 + 32 * u;
          if (c < chunks) {
#pragma unroll
            for (int s = 0; s < NR_TILE_B; ++s) acc[s] = dot8(wv[u], hs[s * chunks + c], acc[s]);   // rows >= nb: stale, unused
          }
        }
      }
    }
#pragma unroll
    for (int s = 0; s < NR_TILE_B; ++s) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[s] += __shfl_xor_sync(0xffffffffu, acc[s], o);
    }
    if (lane == 0) {
      const float bias = j < p.m ? p.b1[j] : 0.f;
      const float w2j = j < p.m ? __bfloat162float(p.w2[j]) : 0.f;
#pragma unroll
      for (int s = 0; s < NR_TILE_B; ++s) {
        const float z = acc[s] + bias;
        const float u = 0.5f * z * (1.f + erff(z * 0.70710678118654752f));     // exact GELU (N2)
        s_term[warp][s] = j < p.m ? w2j * u : 0.f;
      }
    }
    __syncthreads();
    if (tid < nb) {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < NR_WARPS; ++w) t += s_term[w][tid];                   // unit order
      p.ws[(size_t)blockIdx.x * p.B + b0 + tid] = t;
    }
    __syncthreads();                                                            // s_term and the staged rows are reused
  }

  // ---- the last CTA adds the partials in CTA order, adds b2, thresholds ----
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    const unsigned int old = atomicAdd(p.counter, 1u);
    s_last = (old == gridDim.x * gridDim.y - 1);
    if (s_last) *p.counter = 0;                                                 // self-resetting
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  const float b2 = p.b2[0];
  for (int b = tid; b < p.B; b += NR_THREADS) {
    float t = 0.f;
    for (unsigned int c = 0; c < gridDim.x; ++c) t += __ldcg(&p.ws[(size_t)c * p.B + b]);
    const bool empty = p.q_indptr[b + 1] == p.q_indptr[b];
    const float dal = empty ? 0.f : t + b2;
    const float thr = p.tau_is_scalar ? p.tau[0] : p.tau[b];
    p.delta_al[b] = dal;
    p.route[b] = (!empty && dal > thr) ? WF_ROUTE_AR : WF_ROUTE_DIFFUSION;      // N5: ties -> diffusion
  }
}

}  // namespace

extern "C" size_t wf_neural_route_workspace_bytes(int B, int m) {
  if (B <= 0 || m <= 0) return 16;
  return (size_t)((m + NR_WARPS - 1) / NR_WARPS) * (size_t)B * sizeof(float);
}

extern "C" int wf_neural_route(wf_ctx* ctx, const void* hidden_final, const int32_t* q_indptr, const int32_t* accept_len,
                               int B, int d, int m, const void* w1, const float* b1, const void* w2, const float* b2,
                               const float* tau, int tau_is_scalar, float* delta_al, int32_t* route,
                               void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, hidden_final && q_indptr && w1 && b1 && w2 && b2 && tau && delta_al && route && workspace,
             WF_ERR_INVALID_ARG, "wf_neural_route: null argument");
  WF_REQUIRE(ctx, B >= 0 && B <= 1024, WF_ERR_INVALID_ARG, "wf_neural_route: B must be in [0, 1024]");
  WF_REQUIRE(ctx, d > 0 && d % 8 == 0 && m > 0 && m <= 8192, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_neural_route: need d %% 8 == 0 and 0 < m <= 8192");
  WF_REQUIRE(ctx, (size_t)NR_TILE_B * d * 2 <= 200 * 1024, WF_ERR_UNSUPPORTED_SHAPE, "wf_neural_route: d too large (max 6400)");
  WF_REQUIRE(ctx, ((uintptr_t)hidden_final % 16 == 0) && ((uintptr_t)w1 % 16 == 0), WF_ERR_INVALID_ARG,
             "wf_neural_route: hidden_final and w1 must be 16-byte aligned");
  WF_REQUIRE(ctx, workspace_bytes >= wf_neural_route_workspace_bytes(B, m), WF_ERR_INVALID_ARG, "wf_neural_route: workspace too small");
  if (B == 0) return WF_OK;
  const size_t smem = (size_t)NR_TILE_B * d * 2;
  WF_CONFIGURE_ONCE(ctx, WF_FUNC_NEURAL, wf_neural_route_kernel, 200 * 1024);
  NeuralParams p;
  p.hidden = (const __nv_bfloat16*)hidden_final; p.q_indptr = q_indptr; p.accept_len = accept_len;
  p.w1 = (const __nv_bfloat16*)w1; p.b1 = b1; p.w2 = (const __nv_bfloat16*)w2; p.b2 = b2; p.tau = tau;
  p.delta_al = delta_al; p.route = route; p.ws = (float*)workspace;
  p.counter = ctx->d_counters + (ctx->n_counters - 1);     // the accept sweep uses [0, B) with B <= 65535
  p.B = B; p.d = d; p.m = m; p.tau_is_scalar = tau_is_scalar;
  const int grid = (m + NR_WARPS - 1) / NR_WARPS;
  const int tiles = (B + NR_TILE_B - 1) / NR_TILE_B;
  wf_launch(wf_neural_route_kernel, dim3(grid, tiles < 8 ? tiles : 8), dim3(NR_THREADS), smem, (cudaStream_t)stream, p);
  return wf_check_launch(ctx, "wf_neural_route_kernel");
}

// (b) accept + bonus + entropy + route: ONE vectorised sweep over the block's target logits.
// PAPER.md:65, 75-81 (§3.3.1), 135; readings C1-C9, C23.
//
// Grid (n_chunks, max_q_len, B).  A CTA owns one ACC_CHUNK-float slice of one logits row: it loads
// the slice with 16-byte loads into registers, block-reduces (max, lowest argmax), then, relative
// to the slice max, Z_c = sum e^{z-m_c} and S_c = sum e^{z-m_c}(z-m_c), and writes a 16-byte
// partial.  The last CTA of a sequence (self-resetting counter) combines the partials per row
// (argmax g_i), walks the draft tokens for the accepted prefix a, combines row a's (m_c,Z_c,S_c)
// in fp64 into H = ln Z - S/Z, thresholds it, and advances the target cache length.
#include "wf_internal.cuh"

namespace {

constexpr int ACC_THREADS = 256;
constexpr int ACC_VEC_PER_THREAD = 8;                              // 8 x float4 in flight per thread
constexpr int ACC_CHUNK = ACC_THREADS * ACC_VEC_PER_THREAD * 4;    // 8192 floats = 32 KB per CTA
constexpr int ACC_MAX_Q = 64;

struct __align__(16) AccPartial {
  float m;      // slice max (-inf if the slice carries no mass)
  int idx;      // lowest index attaining m
  float Z;      // sum e^{z-m}
  float S;      // sum e^{z-m} (z-m)
};

__device__ __forceinline__ float4 ld_stream(const float4* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
  return r;
}

__device__ __forceinline__ void argmax_merge(float& m, int& i, float om, int oi) {
  if (om > m || (om == m && oi < i)) { m = om; i = oi; }
}

__device__ __forceinline__ int thi_of(int t, int lo, int hi, int piece) { return min(hi, min(hi, lo + t * piece) + piece); }

// Stochastic acceptance (readings S1-S5): u_accept != nullptr switches the finalise step from the greedy prefix to
// speculative sampling at temperature 1 / inv_t.
struct AccSample {
  const float* u_accept;     // [sum_q] uniforms, one per draft row (row 0 of a block unused)
  const float* u_sample;     // [B] uniform of the residual / bonus draw
  const float* draft_q;      // nullptr (deterministic drafter: one-hot at the proposed token) or [sum_q][V]
  float inv_t;               // 1 / temperature; 1.0f in the greedy modes (z * 1.0f is exact)
};

template <bool VEC>
// 5 CTAs per SM: the sweep keeps a CTA's 32 KB slice in registers, so the bytes in flight per SM are what the register file
// holds: at the compiler's own 80 registers 3 CTAs fit and the sweep ran at 4.46 TB/s (cfg5), capped at 48 registers 5 CTAs
// fit: 6.10 TB/s; the rarely executed finalise spills 80 bytes.  (4 CTAs: 5.54 TB/s; 6 CTAs spill inside the sweep: 5.44.)
__global__ void __launch_bounds__(ACC_THREADS, 5)
wf_accept_kernel(const float* __restrict__ logits, int V, int n_chunks, const int32_t* __restrict__ draft_tokens,
                 const int32_t* __restrict__ q_indptr, const float* __restrict__ tau, int tau_is_scalar,
                 int32_t* __restrict__ accept_len, int32_t* __restrict__ bonus_token, float* __restrict__ entropy,
                 int32_t* __restrict__ route, int32_t* __restrict__ n_commit, int32_t* __restrict__ kv_seq_len,
                 AccPartial* __restrict__ partials, unsigned int* __restrict__ counters,
                 const int32_t* __restrict__ parent, int32_t* __restrict__ path, int path_stride, const AccSample smp,
                 int* __restrict__ status) {
  // parent == nullptr: chain block (C6).  Else tree block (T1-T4): greedy walk over parent pointers, the accepted
  // node indices go to path[b][0..a] (-1 beyond), and the cache length is left to wf_kv_compact_path.
  wf_pdl_wait();
  wf_pdl_trigger();
  const int b = blockIdx.z, i = blockIdx.y, chunk = blockIdx.x;
  const int r0 = q_indptr[b];
  const size_t prow0 = (size_t)b * gridDim.y;             // partials are indexed by (sequence, row): in bounds whatever q_indptr says
  int q_b = q_indptr[b + 1] - r0;
  if (q_b > (int)gridDim.y) {
    // the host bound max_q_len sizes the grid: a longer block is verified up to the bound (its counter still reaches
    // its total and resets) and the sticky status says so
    if (i == 0 && blockIdx.x == 0 && threadIdx.x == 0) wf_raise(status, (int)WF_ERR_INVALID_ARG);
    q_b = (int)gridDim.y;
  }
  if (q_b == 0 && i == 0 && blockIdx.x == 0 && threadIdx.x == 0) {
    // empty block: nothing verified, nothing committed
    accept_len[b] = 0; bonus_token[b] = 0; entropy[b] = 0.f; route[b] = 0; n_commit[b] = 0;
    if (path) for (int k = 0; k < path_stride; ++k) path[(size_t)b * path_stride + k] = -1;
  }
  if (i >= q_b) return;                                   // whole CTA exits together
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const float* row = logits + (size_t)(r0 + i) * V;
  const int c0 = chunk * ACC_CHUNK;
  const int n_here = min(ACC_CHUNK, V - c0);

  float v[ACC_VEC_PER_THREAD * 4];
  if (VEC) {
    const float4* p = reinterpret_cast<const float4*>(row + c0);
#pragma unroll
    for (int k = 0; k < ACC_VEC_PER_THREAD; ++k) {
      const int e = (k * ACC_THREADS + tid) * 4;
      float4 x = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
      if (e < n_here) x = ld_stream(p + k * ACC_THREADS + tid);     // V % 4 == 0: all or nothing
      v[4 * k + 0] = x.x * smp.inv_t; v[4 * k + 1] = x.y * smp.inv_t; v[4 * k + 2] = x.z * smp.inv_t; v[4 * k + 3] = x.w * smp.inv_t;
    }
  } else {
#pragma unroll
    for (int k = 0; k < ACC_VEC_PER_THREAD; ++k)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int e = (k * ACC_THREADS + tid) * 4 + j;
        v[4 * k + j] = e < n_here ? __ldg(row + c0 + e) * smp.inv_t : -INFINITY;
      }
  }

  // The sweep is issue-bound if every element pays for index tracking and special cases (ncu: 66 % issue
  // utilisation at 3.1 TB/s), so: max by FMNMX only; the index is recovered afterwards by the few threads that
  // hold the slice maximum; exp through MUFU.EX2 with d clamped instead of a -inf test (7 instructions per element).
  float m = -INFINITY;
#pragma unroll
  for (int k = 0; k < ACC_VEC_PER_THREAD * 4; ++k) m = fmaxf(m, v[k]);
  const float tm = m;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
  __shared__ float s_m[ACC_THREADS / 32];
  __shared__ int s_i[ACC_THREADS / 32];
  __shared__ float s_z[ACC_THREADS / 32], s_s[ACC_THREADS / 32];
  if (lane == 0) { s_m[wid] = m; s_i[wid] = 0x7fffffff; }
  __syncthreads();
  m = s_m[0];
#pragma unroll
  for (int w = 1; w < ACC_THREADS / 32; ++w) m = fmaxf(m, s_m[w]);
  // lowest index attaining the slice max (C7): indices ascend with (k, j) inside a thread; across threads atomicMin
  if (tm == m && m > -INFINITY) {
    int mi = 0x7fffffff;
#pragma unroll
    for (int k = ACC_VEC_PER_THREAD - 1; k >= 0; --k)
#pragma unroll
      for (int j = 3; j >= 0; --j)
        if (v[4 * k + j] == m) mi = c0 + (k * ACC_THREADS + tid) * 4 + j;
    atomicMin(&s_i[0], mi);
  }

  // Z_c, S_c relative to the slice max; -inf entries contribute 0 (0 * ln 0 := 0, C23): d is clamped to a finite
  // floor, e = 2^(d log2 e) underflows to +0 there and e * d = -0
  float Z = 0.f, S = 0.f;
  if (m > -INFINITY) {
    constexpr float LOG2E = 1.4426950408889634f;
#pragma unroll
    for (int k = 0; k < ACC_VEC_PER_THREAD * 4; ++k) {
      const float d = fmaxf(v[k] - m, -1.0e30f);
      float e;
      asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(d * LOG2E));
      Z += e;
      S = fmaf(e, d, S);
    }
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    Z += __shfl_xor_sync(0xffffffffu, Z, d);
    S += __shfl_xor_sync(0xffffffffu, S, d);
  }
  if (lane == 0) { s_z[wid] = Z; s_s[wid] = S; }
  __syncthreads();
  const int mi = s_i[0];

  __shared__ bool s_last;
  if (tid == 0) {
    float Zt = 0.f, St = 0.f;
#pragma unroll
    for (int w = 0; w < ACC_THREADS / 32; ++w) { Zt += s_z[w]; St += s_s[w]; }
    AccPartial p; p.m = m; p.idx = mi; p.Z = Zt; p.S = St;
    partials[(prow0 + i) * n_chunks + chunk] = p;
    __threadfence();
    const unsigned int total = (unsigned int)(q_b * n_chunks);
    const unsigned int old = atomicAdd(&counters[b], 1u);
    s_last = (old == total - 1);
    if (s_last) counters[b] = 0;                          // self-reset for the next call
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();

  // ---- finalise sequence b (one CTA) ----
  __shared__ int s_g[ACC_MAX_Q];
  __shared__ int s_a;
  __shared__ float s_M[ACC_MAX_Q];                         // per row: max over the slices, and relative to it ...
  __shared__ double s_Z[ACC_MAX_Q], s_S[ACC_MAX_Q];        // ... Z = sum e^{z-M} and S = sum e^{z-M}(z-M), combined in fp64
  __shared__ int s_ok[ACC_MAX_Q];
  __shared__ int s_row;                                    // the row whose logits give the bonus token and the entropy
  __shared__ int s_par[ACC_MAX_Q], s_tok[ACC_MAX_Q];
  if (tid < q_b) { s_par[tid] = parent ? parent[r0 + tid] : tid - 1; s_tok[tid] = draft_tokens[r0 + tid]; }   // one round trip for all
  // One pass over the slice partials (16 bytes each, one load), one warp per row and TWO rows of a warp in flight: per row
  // the argmax g_i AND (M, Z, S), so that neither the acceptance test of the sampling mode nor the entropy of the last
  // accepted row (whichever row that turns out to be) needs another round trip to L2.  (The finalise used to make three
  // dependent ones: argmax, then max, then Z and S of row a.)
  for (int rb = wid; rb < q_b; rb += 2 * (ACC_THREADS / 32)) {
    const int rows[2] = {rb, rb + ACC_THREADS / 32};
    float4 first[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      first[u] = make_float4(-INFINITY, __int_as_float(0x7fffffff), 0.f, 0.f);
      if (rows[u] < q_b && lane < n_chunks)
        first[u] = __ldcg(reinterpret_cast<const float4*>(&partials[(prow0 + rows[u]) * n_chunks + lane]));
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int r = rows[u];
      if (r >= q_b) continue;                              // whole warp together
      const AccPartial* pr = &partials[(prow0 + r) * n_chunks];
      float rm = first[u].x;
      int ri = __float_as_int(first[u].y);
      for (int c = lane + 32; c < n_chunks; c += 32) {      // vocabularies of more than 32 slices
        const float4 x = __ldcg(reinterpret_cast<const float4*>(&pr[c]));
        argmax_merge(rm, ri, x.x, __float_as_int(x.y));
      }
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        float om = __shfl_xor_sync(0xffffffffu, rm, d);
        int oi = __shfl_xor_sync(0xffffffffu, ri, d);
        argmax_merge(rm, ri, om, oi);
      }
      const float gm = rm;                                 // the row maximum (every lane)
      double Zd = 0.0, Sd = 0.0;
      for (int c = lane; c < n_chunks; c += 32) {
        const float4 x = c == lane ? first[u] : __ldcg(reinterpret_cast<const float4*>(&pr[c]));
        if (x.x > -INFINITY) {
          const double dm = (double)x.x - (double)gm;
          const double w = exp(dm);
          Zd += (double)x.z * w;
          Sd += w * ((double)x.w + dm * (double)x.z);
        }
      }
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        Zd += __shfl_xor_sync(0xffffffffu, Zd, d);
        Sd += __shfl_xor_sync(0xffffffffu, Sd, d);
      }
      if (lane == 0) { s_g[r] = ri; s_M[r] = gm; s_Z[r] = Zd; s_S[r] = Sd; }
    }
  }
  __syncthreads();
  if (smp.u_accept) {
    // ---- speculative sampling (S3): p_{j-1}(x_j) from row j-1's (M, Z) (the pass above) and one gathered logit ----
    if (tid >= 1 && tid < q_b) {                           // draft j = tid against row j - 1
      const int x = draft_tokens[r0 + tid];
      if (x < 0 || x >= V) {                               // not a token: rejected, never gathered
        wf_raise(status, (int)WF_ERR_INVALID_ARG);
        s_ok[tid] = 0;
      } else {
        const size_t at = (size_t)(r0 + tid - 1) * V + x;
        const double px = exp((double)(logits[at] * smp.inv_t) - (double)s_M[tid - 1]) / s_Z[tid - 1];
        const double qx = smp.draft_q ? (double)smp.draft_q[at] : 1.0;
        const double ratio = qx <= 0.0 ? 1.0 : fmin(1.0, px / qx);
        s_ok[tid] = (double)smp.u_accept[r0 + tid] < ratio;
      }
    }
    __syncthreads();
    if (tid == 0) {
      int a = 0;
      while (a < q_b - 1 && s_ok[a + 1]) ++a;
      s_a = a;
      s_row = a;
    }
  } else if (!parent) {
    if (tid == 0) {                                        // longest accepted prefix (C6)
      const int gamma = q_b - 1;
      int a = 0;
      while (a < gamma && s_tok[a + 1] == s_g[a]) ++a;
      s_a = a;
      s_row = a;
    }
  } else if (wid == 0) {                                   // greedy walk from the root (T3), one warp
    int cur = 0, a = 0;
    int32_t* pb = path ? path + (size_t)b * path_stride : nullptr;
    if (pb) for (int k = lane; k < path_stride; k += 32) pb[k] = k == 0 ? 0 : -1;
    __syncwarp();
    for (;;) {
      const int g = s_g[cur];
      int nxt = -1;
      for (int base = cur + 1; base < q_b && nxt < 0; base += 32) {   // children sit above their parent (T1)
        const int c = base + lane;
        const bool hit = c < q_b && s_par[c] == cur && s_tok[c] == g;
        const unsigned int bal = __ballot_sync(0xffffffffu, hit);
        if (bal) nxt = base + __ffs(bal) - 1;              // the lowest-index matching child
      }
      if (nxt < 0) break;
      cur = nxt;
      ++a;
      if (pb && lane == 0 && a < path_stride) pb[a] = cur;
    }
    if (lane == 0) { s_a = a; s_row = cur; }
  }
  __syncthreads();
  if (tid == 0) {                                          // entropy of the last accepted row from its fp64 (Z, S) (C3, C4, T4)
    const int a = s_a, row_a = s_row;
    {
      const double Zd = s_Z[row_a], Sd = s_S[row_a];
      const float H = (float)(log(Zd) - Sd / Zd);
      const float t = tau_is_scalar ? tau[0] : tau[b];
      accept_len[b] = a;
      if (!smp.u_accept) bonus_token[b] = s_g[row_a];
      n_commit[b] = a + 1;
      entropy[b] = H;
      route[b] = (H > t) ? WF_ROUTE_AR : WF_ROUTE_DIFFUSION;     // C1, C2
      if (kv_seq_len) kv_seq_len[b] += a + 1;
    }
  }
  if (!smp.u_accept) return;

  // ---- the token after the accepted prefix (S4): inverse CDF, in vocabulary order, of the residual max(0, p - q)
  //      of row a (of p itself for the bonus token, or if the residual is empty).  Masses are evaluated in fp32 and
  //      accumulated in fp64. ----
  __shared__ double s_seg[ACC_THREADS];
  __shared__ double s_target;
  __shared__ int s_pick, s_resid, s_tok_out;
  const int a = s_a, gamma = q_b - 1;
  const float* zr = logits + (size_t)(r0 + a) * V;
  const float* qr = smp.draft_q ? smp.draft_q + (size_t)(r0 + a) * V : nullptr;
  int xrej = a < gamma ? draft_tokens[r0 + a + 1] : -1;
  if (xrej >= V || xrej < 0) xrej = -1;                                 // an out-of-range draft (flagged above) removes no mass
  const float Mr = s_M[a];
  const double Zinv = 1.0 / s_Z[a];
  const float Zinv_f = (float)Zinv;
  auto mass = [&](int v, bool resid) -> double {           // fp32 per token (MUFU exp: a -inf logit gives exactly 0)
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"((zr[v] * smp.inv_t - Mr) * 1.4426950408889634f));
    float pv = e * Zinv_f;
    if (resid) pv = fmaxf(0.f, pv - (qr ? qr[v] : (v == xrej ? 1.f : 0.f)));
    return (double)pv;
  };
  // Search from coarse to fine, every level parallel over the CTA.  Level 0 costs no memory pass when the drafter is
  // deterministic (or for the bonus token): the sweep's slice partials already hold each 8192-token slice's share of
  // the mass (minus the rejected token's in its slice).  Then the range is cut into 8 contiguous parts, warp w sums
  // part w with its lanes striding through it, and thread 0 picks the part that holds the target (twice when level 0
  // had to be skipped because the residual needs the drafter's full row); the last ~1k tokens are cut into one short
  // piece per thread and the owner of the piece that holds the target walks it.
  constexpr int NW = ACC_THREADS / 32;
  if (tid == 0) { s_resid = a < gamma; s_tok_out = -1; }
  __syncthreads();
  int lo = 0, hi = V;
  double base = 0.0;                                       // mass below lo
  int levels = 2;
  if (!qr && n_chunks <= ACC_THREADS) {
    const AccPartial* pr = &partials[(prow0 + a) * n_chunks];
    for (int attempt = 0; attempt < 2; ++attempt) {
      double mc = 0.0;
      if (tid < n_chunks) {
        const float pm = __ldcg(&pr[tid].m);
        if (pm > -INFINITY) mc = (double)__ldcg(&pr[tid].Z) * exp((double)pm - (double)Mr) * Zinv;
        if (s_resid && xrej >= 0 && xrej / ACC_CHUNK == tid)
          mc = fmax(0.0, mc - exp((double)(zr[xrej] * smp.inv_t) - (double)Mr) * Zinv);
      }
      s_seg[tid] = mc;
      __syncthreads();
      if (tid == 0) {
        double run = 0.0;
        for (int t = 0; t < n_chunks; ++t) { const double x = s_seg[t]; s_seg[t] = run; run += x; }
        if (!(run > 0.0) && s_resid) { s_resid = 0; s_pick = -1; }      // the rejected token held all the mass: draw from p
        else {
          s_target = (double)smp.u_sample[b] * run;
          int pick = 0;
          for (int t = 1; t < n_chunks; ++t)
            if (s_seg[t] <= s_target) pick = t;
          s_pick = pick;
        }
      }
      __syncthreads();
      if (s_pick >= 0) break;
      __syncthreads();
    }
    base = s_seg[s_pick];
    lo = s_pick * ACC_CHUNK;
    hi = min(V, lo + ACC_CHUNK);
    levels = 1;
    __syncthreads();
  }
  for (int level = 0; level < levels; ++level) {
    const bool first = levels == 2 && level == 0;          // this level also fixes the total and the target
    const int part = (((hi - lo + NW - 1) / NW) + 127) & ~127;             // whole 128-token strips: 16-byte loads stay aligned
    const bool resid = s_resid != 0;
    const int plo = min(hi, lo + wid * part), phi = min(hi, plo + part);
    double acc = 0.0;
    if (VEC) {
      // V % 4 == 0 and 16-byte aligned rows: 8 x 16-byte loads of z (and of q) in flight per lane; the pass is one CTA
      // streaming up to 2 x 600 KB, i.e. bound by the bytes it keeps in flight
      for (int v0 = plo + 4 * lane; v0 < phi; v0 += 128 * 8) {
        float4 zz[8], qq[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int v = v0 + 128 * k;
          zz[k] = v < phi ? *reinterpret_cast<const float4*>(zr + v) : make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
          qq[k] = (resid && qr && v < phi) ? *reinterpret_cast<const float4*>(qr + v) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const float z4[4] = {zz[k].x, zz[k].y, zz[k].z, zz[k].w}, q4[4] = {qq[k].x, qq[k].y, qq[k].z, qq[k].w};
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int v = v0 + 128 * k + j;
            float e;
            asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"((z4[j] * smp.inv_t - Mr) * 1.4426950408889634f));
            float pv = e * Zinv_f;
            if (resid) pv = fmaxf(0.f, pv - (qr ? q4[j] : (v == xrej ? 1.f : 0.f)));
            acc += (double)pv;
          }
        }
      }
    } else
    for (int v0 = plo + lane; v0 < phi; v0 += 32 * 8) {    // 8 loads in flight per lane
      float zz[8], qq[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const int v = v0 + 32 * k;
        zz[k] = v < phi ? zr[v] : -INFINITY;
        qq[k] = (resid && qr && v < phi) ? qr[v] : 0.f;
      }
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const int v = v0 + 32 * k;
        float e;
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"((zz[k] * smp.inv_t - Mr) * 1.4426950408889634f));
        float pv = e * Zinv_f;
        if (resid) pv = fmaxf(0.f, pv - (qr ? qq[k] : (v == xrej ? 1.f : 0.f)));
        acc += (double)pv;
      }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (lane == 0) s_seg[wid] = acc;
    __syncthreads();
    if (tid == 0) {
      double run = base;
      for (int t = 0; t < NW; ++t) { const double x = s_seg[t]; s_seg[t] = run; run += x; }     // mass below part t
      s_pick = 0;
      if (first) {
        if (!(run > 0.0) && s_resid) { s_resid = 0; s_pick = -1; }    // empty residual (p <= q everywhere): draw from p
        else s_target = (double)smp.u_sample[b] * run;
      }
      if (s_pick >= 0) {
        int pick = 0;
        for (int t = 1; t < NW; ++t)
          if (s_seg[t] <= s_target) pick = t;              // the last part that starts at or below the target
        s_pick = pick;
      }
    }
    __syncthreads();
    if (s_pick < 0) { level = -1; __syncthreads(); continue; }        // block-uniform: start over without the residual
    base = s_seg[s_pick];
    lo = min(hi, lo + s_pick * part);
    hi = min(hi, lo + part);
    __syncthreads();
  }
  const bool resid = s_resid != 0;
  const int piece = (hi - lo + ACC_THREADS - 1) / ACC_THREADS;
  const int tlo = min(hi, lo + tid * piece), thi = min(hi, tlo + piece);
  {
    double acc = 0.0;
    for (int v = tlo; v < thi; ++v) acc += mass(v, resid);
    s_seg[tid] = acc;
  }
  __syncthreads();
  if (tid == 0) {
    double run = base;
    int pick = 0;
    for (int t = 0; t < ACC_THREADS; ++t) {
      const double x = s_seg[t];
      s_seg[t] = run;
      if (run <= s_target) pick = t;
      run += x;
    }
    s_pick = pick;
  }
  __syncthreads();
  if (tid == s_pick) {
    double run = s_seg[tid];
    int tok = -1;
    for (int v = tlo; v < thi; ++v) {
      const double mv = mass(v, resid);
      run += mv;
      if (run > s_target && mv > 0.0) { tok = v; break; }
    }
    s_tok_out = tok;
  }
  __syncthreads();
  if (tid == 0) {
    int tok = s_tok_out;
    if (tok < 0) {
      // rounding put the target at or past the end of the picked piece: the next token with mass, else the last one
      for (int v = min(V, thi_of(s_pick, lo, hi, piece)); v < V && tok < 0; ++v)
        if (mass(v, resid) > 0.0) tok = v;
      for (int v = V - 1; v >= 0 && tok < 0; --v)
        if (mass(v, resid) > 0.0) tok = v;
      if (tok < 0) tok = 0;
    }
    bonus_token[b] = tok;
  }
}

}  // namespace

extern "C" size_t wf_accept_workspace_bytes(int sum_q, int V) {
  if (sum_q <= 0 || V <= 0) return 16;
  const size_t n_chunks = ((size_t)V + ACC_CHUNK - 1) / ACC_CHUNK;
  return (size_t)sum_q * n_chunks * sizeof(AccPartial);
}

namespace {
int accept_launch(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens, const int32_t* q_indptr, int B,
                  int max_q_len, const float* tau, int tau_is_scalar, int32_t* accept_len, int32_t* bonus_token,
                  float* entropy, int32_t* route, int32_t* n_commit, wf_paged_kv* target_kv, void* workspace,
                  size_t workspace_bytes, void* stream, const int32_t* parent, int32_t* path, int path_stride,
                  const AccSample& smp);
const AccSample kGreedy = {nullptr, nullptr, nullptr, 1.0f};
}

extern "C" int wf_accept_entropy_route(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens,
                                       const int32_t* q_indptr, int B, int max_q_len, const float* tau,
                                       int tau_is_scalar, int32_t* accept_len, int32_t* bonus_token,
                                       float* entropy, int32_t* route, int32_t* n_commit,
                                       wf_paged_kv* target_kv, void* workspace, size_t workspace_bytes,
                                       void* stream) {
  return accept_launch(ctx, logits, V, draft_tokens, q_indptr, B, max_q_len, tau, tau_is_scalar, accept_len,
                       bonus_token, entropy, route, n_commit, target_kv, workspace, workspace_bytes, stream, nullptr,
                       nullptr, 0, kGreedy);
}

extern "C" int wf_accept_sample_entropy_route(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens,
                                              const int32_t* q_indptr, int B, int max_q_len, float temperature,
                                              const float* draft_q, const float* u_accept, const float* u_sample,
                                              const float* tau, int tau_is_scalar, int32_t* accept_len, int32_t* token,
                                              float* entropy, int32_t* route, int32_t* n_commit, wf_paged_kv* target_kv,
                                              void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, u_accept && u_sample, WF_ERR_INVALID_ARG, "wf_accept_sample_entropy_route: the uniforms are inputs");
  WF_REQUIRE(ctx, temperature > 0.f && temperature < INFINITY, WF_ERR_INVALID_ARG,
             "wf_accept_sample_entropy_route: temperature must be positive and finite");
  const AccSample smp = {u_accept, u_sample, draft_q, 1.0f / temperature};
  return accept_launch(ctx, logits, V, draft_tokens, q_indptr, B, max_q_len, tau, tau_is_scalar, accept_len, token,
                       entropy, route, n_commit, target_kv, workspace, workspace_bytes, stream, nullptr, nullptr, 0, smp);
}

extern "C" int wf_accept_tree_entropy_route(wf_ctx* ctx, const float* logits, int V, const int32_t* node_tokens,
                                            const int32_t* parent, const int32_t* q_indptr, int B, int max_nodes,
                                            const float* tau, int tau_is_scalar, int32_t* accept_len,
                                            int32_t* bonus_token, float* entropy, int32_t* route, int32_t* n_commit,
                                            int32_t* path, int path_stride, void* workspace, size_t workspace_bytes,
                                            void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, parent && path && path_stride >= 1 && path_stride >= max_nodes, WF_ERR_INVALID_ARG,
             "wf_accept_tree_entropy_route: parent / path missing or path_stride < max_nodes");
  return accept_launch(ctx, logits, V, node_tokens, q_indptr, B, max_nodes, tau, tau_is_scalar, accept_len,
                       bonus_token, entropy, route, n_commit, nullptr, workspace, workspace_bytes, stream, parent, path,
                       path_stride, kGreedy);
}

namespace {
int accept_launch(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens, const int32_t* q_indptr, int B,
                  int max_q_len, const float* tau, int tau_is_scalar, int32_t* accept_len, int32_t* bonus_token,
                  float* entropy, int32_t* route, int32_t* n_commit, wf_paged_kv* target_kv, void* workspace,
                  size_t workspace_bytes, void* stream, const int32_t* parent, int32_t* path, int path_stride,
                  const AccSample& smp) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, logits && draft_tokens && q_indptr && tau && accept_len && bonus_token && entropy && route &&
                 n_commit && workspace, WF_ERR_INVALID_ARG, "wf_accept_entropy_route: null argument");
  WF_REQUIRE(ctx, V > 0 && B >= 0 && B <= ctx->n_counters && B <= 65535, WF_ERR_INVALID_ARG,
             "wf_accept_entropy_route: bad V or B");
  WF_REQUIRE(ctx, max_q_len >= 0 && max_q_len <= ACC_MAX_Q, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_accept_entropy_route: max_q_len must be <= %d", ACC_MAX_Q);
  WF_REQUIRE(ctx, !target_kv || B <= target_kv->s.max_seqs, WF_ERR_INVALID_ARG,
             "wf_accept_entropy_route: B exceeds the cache's max_seqs");
  if (B == 0) return WF_OK;
  cudaStream_t st = (cudaStream_t)stream;
  if (max_q_len == 0) max_q_len = 1;                       // still launch: empty blocks get zeroed outputs
  const int n_chunks = (V + ACC_CHUNK - 1) / ACC_CHUNK;
  WF_REQUIRE(ctx, workspace_bytes >= wf_accept_workspace_bytes(B * max_q_len, V), WF_ERR_INVALID_ARG, "wf_accept_entropy_route: workspace too small");
  dim3 grid(n_chunks, max_q_len, B);
  int32_t* kv_len = target_kv ? target_kv->seq_len : nullptr;
  const bool vec = (V % 4 == 0) && ((uintptr_t)logits % 16 == 0) && (!smp.draft_q || (uintptr_t)smp.draft_q % 16 == 0);
  if (vec)
    wf_launch(wf_accept_kernel<true>, grid, dim3(ACC_THREADS), 0, st, logits, V, n_chunks, draft_tokens, q_indptr, tau,
        tau_is_scalar, accept_len, bonus_token, entropy, route, n_commit, kv_len, (AccPartial*)workspace, ctx->d_counters,
        parent, path, path_stride, smp, ctx->d_status);
  else
    wf_launch(wf_accept_kernel<false>, grid, dim3(ACC_THREADS), 0, st, logits, V, n_chunks, draft_tokens, q_indptr, tau,
        tau_is_scalar, accept_len, bonus_token, entropy, route, n_commit, kv_len, (AccPartial*)workspace, ctx->d_counters,
        parent, path, path_stride, smp, ctx->d_status);
  return wf_check_launch(ctx, "wf_accept_kernel");
}
}  // namespace

// ------------------------------------------------------------------------------------------------
// wf_accept_entropy_route_static: the same sweep for callers that cannot allocate (CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc) and do not want to carry a workspace: the slice partials and the completion
// counters live in ONE file-scope device array of a fixed size.  Every GPU that loads the library holds the array
// (516 KB) until the process exits.  Nothing here calls cudaMalloc, cudaFree or an allocating library routine.
// ------------------------------------------------------------------------------------------------
#include <mutex>

namespace {
constexpr int ACC_STATIC_MAX_B = 1024;                         // counters (one per sequence)
constexpr int ACC_STATIC_MAX_PARTIALS = 32768;                 // B * max_q_len * ceil(V / 8192) slice partials of 16 bytes
constexpr size_t ACC_STATIC_COUNTER_BYTES = ACC_STATIC_MAX_B * sizeof(unsigned int);
constexpr size_t ACC_STATIC_BYTES = ACC_STATIC_COUNTER_BYTES + (size_t)ACC_STATIC_MAX_PARTIALS * sizeof(AccPartial);
constexpr int ACC_STATIC_MAX_DEVICES = 64;
}  // namespace

// layout: [ACC_STATIC_MAX_B] unsigned int counters | [ACC_STATIC_MAX_PARTIALS] AccPartial.  In host code this NAME is a
// host-side stand-in, not a device address: the address a kernel may use comes from cudaGetSymbolAddress (below).
static __device__ __align__(256) unsigned char wf_accept_static_scratch[ACC_STATIC_BYTES];

namespace {
std::mutex g_static_mu;
void* g_static_ptr[ACC_STATIC_MAX_DEVICES];                    // per device: the array's device address, resolved once

// set-up, once per device, with that device current
int accept_static_setup(wf_ctx* ctx, void** out) {
  const int dev = ctx->device;
  WF_REQUIRE(ctx, dev >= 0 && dev < ACC_STATIC_MAX_DEVICES, WF_ERR_INVALID_ARG,
             "wf_accept_entropy_route_static: device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    int cur = -1;
    WF_CUDA(ctx, cudaGetDevice(&cur));
    WF_REQUIRE(ctx, cur == dev, WF_ERR_INVALID_ARG,
               "wf_accept_entropy_route_static: the context's device (%d) must be current (current: %d)", dev, cur);
    void* ptr = nullptr;
    WF_CUDA(ctx, cudaGetSymbolAddress((void**)&ptr, wf_accept_static_scratch));
    WF_REQUIRE(ctx, ptr != nullptr, WF_ERR_CUDA, "wf_accept_entropy_route_static: cudaGetSymbolAddress returned null");
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return WF_OK;
}
}  // namespace

extern "C" int wf_accept_entropy_route_static(wf_ctx* ctx, const float* logits, int V, const int32_t* draft_tokens,
                                              const int32_t* q_indptr, int B, int max_q_len, const float* tau,
                                              int tau_is_scalar, int32_t* accept_len, int32_t* bonus_token,
                                              float* entropy, int32_t* route, int32_t* n_commit,
                                              wf_paged_kv* target_kv, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, logits && draft_tokens && q_indptr && tau && accept_len && bonus_token && entropy && route && n_commit,
             WF_ERR_INVALID_ARG, "wf_accept_entropy_route_static: null argument");
  WF_REQUIRE(ctx, V > 0 && B >= 0 && B <= 65535, WF_ERR_INVALID_ARG, "wf_accept_entropy_route_static: bad V or B");
  WF_REQUIRE(ctx, max_q_len >= 0 && max_q_len <= ACC_MAX_Q, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_accept_entropy_route_static: max_q_len must be <= %d", ACC_MAX_Q);
  WF_REQUIRE(ctx, !target_kv || B <= target_kv->s.max_seqs, WF_ERR_INVALID_ARG,
             "wf_accept_entropy_route_static: B exceeds the cache's max_seqs");
  if (max_q_len == 0) max_q_len = 1;                       // still launch: empty blocks get zeroed outputs
  const int n_chunks = (V + ACC_CHUNK - 1) / ACC_CHUNK;
  const long long need = (long long)B * max_q_len * n_chunks;
  WF_REQUIRE(ctx, B <= ACC_STATIC_MAX_B && need <= ACC_STATIC_MAX_PARTIALS, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_accept_entropy_route_static: B = %d, B * max_q_len * ceil(V / %d) = %lld exceed the static scratch "
             "(at most %d sequences and %d slice partials); use wf_accept_entropy_route with a caller workspace",
             B, ACC_CHUNK, need, ACC_STATIC_MAX_B, ACC_STATIC_MAX_PARTIALS);
  if (B == 0) return WF_OK;
  void* base = nullptr;
  const int rc = accept_static_setup(ctx, &base);
  if (rc != WF_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned int* counters = reinterpret_cast<unsigned int*>(base);
  AccPartial* partials = reinterpret_cast<AccPartial*>(reinterpret_cast<unsigned char*>(base) + ACC_STATIC_COUNTER_BYTES);
  // The array keeps the last call's contents.  The counters must start at zero (they reset themselves when a call completes,
  // but a call that was cut short would leave them counting): cleared here, in stream order.  The partials need no clearing:
  // every one that is read was written by this call.
  WF_CUDA(ctx, cudaMemsetAsync(counters, 0, (size_t)B * sizeof(unsigned int), st));
  dim3 grid(n_chunks, max_q_len, B);
  int32_t* kv_len = target_kv ? target_kv->seq_len : nullptr;
  const bool vec = (V % 4 == 0) && ((uintptr_t)logits % 16 == 0);
  if (vec)
    wf_launch(wf_accept_kernel<true>, grid, dim3(ACC_THREADS), 0, st, logits, V, n_chunks, draft_tokens, q_indptr, tau,
        tau_is_scalar, accept_len, bonus_token, entropy, route, n_commit, kv_len, partials, counters,
        (const int32_t*)nullptr, (int32_t*)nullptr, 0, kGreedy, ctx->d_status);
  else
    wf_launch(wf_accept_kernel<false>, grid, dim3(ACC_THREADS), 0, st, logits, V, n_chunks, draft_tokens, q_indptr, tau,
        tau_is_scalar, accept_len, bonus_token, entropy, route, n_commit, kv_len, partials, counters,
        (const int32_t*)nullptr, (int32_t*)nullptr, 0, kGreedy, ctx->d_status);
  return wf_check_launch(ctx, "wf_accept_kernel<static scratch>");
}

// (a) Target-model verification attention over the paged bf16 GQA KV cache.
// PAPER.md:65 (§3.2 "parallel verification"); readings C10-C13.
//
// Split-KV, decode-style.  A work item is (sequence b, kv head g, key range [k0,k1)); its query
// tile is all q_b rows of all `group` query heads that share kv head g (<= 64 rows), so K and V are
// read from HBM once per kv head.  A persistent grid (2 CTAs per SM) strides over the item list,
// which every CTA derives from the device-resident lengths (no host sync).  K/V pages are staged
// through a 3-deep cp.async ring (16-byte coalesced copies, XOR-swizzled rows), QK^T and PV run on
// bf16 tensor-core MMA with fp32 accumulators, the online softmax lives in registers with
// warp-shuffle reductions, and the last CTA to finish a (b,g) pair merges the split partials.
#include "wf_internal.cuh"

namespace {

constexpr int AT_THREADS = 128;        // 4 warps: (row group rg = warp & 1) x (key part kp = warp >> 1)
constexpr int AT_BN = 64;              // keys per pipeline stage
constexpr int AT_STAGES = 3;
constexpr int AT_MIN_CHUNK = 256;      // never split below this many keys
constexpr int AT_ITEMS_PER_SM = 8;     // target number of work items per SM
constexpr int AT_MAX_B = 1024;
constexpr float LOG2E = 1.4426950408889634f;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  const int n = valid ? 16 : 0;        // src-size 0 -> 16 zero bytes
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

struct AttnParams {
  const __nv_bfloat16* q;
  __nv_bfloat16* out;
  const int32_t* q_indptr;
  KvView kv;
  int layer, B, n_q_heads, group;
  float scale_log2;                    // sm_scale * log2(e)
  int target_items;
  float* ws_o;                         // [items][R_PAD][D] fp32, unnormalised
  float2* ws_ml;                       // [items][R_PAD] (m in log2 units, l)
  unsigned int* counters;              // [B * Hkv], self-resetting
};

// swizzled byte offset of 16-byte chunk `ch` of row `row` (row pitch = D*2 bytes)
template <int D>
__device__ __forceinline__ uint32_t swz(int row, int ch) { return (uint32_t)(row * (D * 2) + ((ch ^ (row & 7)) << 4)); }

template <int D, int MT>
__global__ void __launch_bounds__(AT_THREADS, (D == 128 && MT == 2) ? 2 : 3)
wf_verify_attn_kernel(const AttnParams p) {
  constexpr int R_PAD = 32 * MT;                 // query rows per tile (2 row groups x MT x 16)
  constexpr int CPR = D / 8;                     // 16-byte chunks per row
  constexpr int TILE_BYTES = AT_BN * D * 2;      // one K (or V) stage
  constexpr int NT_O = D / 8;                    // output n-tiles per warp
  constexpr int LD_ITERS = AT_BN * CPR / AT_THREADS;

  extern __shared__ __align__(128) uint8_t smem[];
  uint8_t* q_s = smem;                                          // R_PAD x D bf16
  uint8_t* kv_s = smem + R_PAD * D * 2;                         // AT_STAGES x (K tile, V tile)
  __shared__ int s_red[AT_THREADS / 32];
  __shared__ int s_chunk;
  __shared__ bool s_last;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int rg = warp & 1, kp = warp >> 1;
  const KvView& kv = p.kv;
  const int Hkv = kv.n_kv_heads;

  // ---- split size from the device-resident lengths (identical in every CTA, no host sync) ----
  int part = 0;
  for (int b = tid; b < p.B; b += AT_THREADS) {
    const int qb = p.q_indptr[b + 1] - p.q_indptr[b];
    part += qb > 0 ? kv.seq_len[b] + qb : 0;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
  if (lane == 0) s_red[warp] = part;
  __syncthreads();
  if (tid == 0) {
    long long total = 0;
    for (int w = 0; w < AT_THREADS / 32; ++w) total += s_red[w];
    long long c = (total * Hkv + p.target_items - 1) / p.target_items;
    c = (c + AT_BN - 1) / AT_BN * AT_BN;
    s_chunk = (int)max((long long)AT_MIN_CHUNK, c);
  }
  __syncthreads();
  const int chunk_target = s_chunk;
  // n_split of a sequence of `len` keys: page-aligned equal parts of about chunk_target keys
  auto splits_of = [&](int len) {
    if (len <= 0) return 0;
    const int pages = (len + 15) >> 4;
    const int ns0 = (len + chunk_target - 1) / chunk_target;
    const int pps = (pages + ns0 - 1) / ns0;
    return (pages + pps - 1) / pps;
  };
  auto len_of = [&](int b) {
    const int qb = p.q_indptr[b + 1] - p.q_indptr[b];
    return qb > 0 ? kv.seq_len[b] + qb : 0;
  };
  // Items are numbered b-major: item = pref_b + split * Hkv + g.  A CTA visits its items in
  // ascending order, so it walks (b_cur, pref_cur) forward instead of keeping a table.
  int b_cur = 0, pref_cur = 0;
  int ns_cur = p.B > 0 ? splits_of(len_of(0)) : 0;

  float o[MT][NT_O][4];
  float s[MT][4][4];

  for (int item = blockIdx.x;; item += gridDim.x) {
    while (b_cur < p.B && item >= pref_cur + ns_cur * Hkv) {   // uniform across the CTA
      pref_cur += ns_cur * Hkv;
      ++b_cur;
      ns_cur = b_cur < p.B ? splits_of(len_of(b_cur)) : 0;
    }
    if (b_cur >= p.B) break;
    const int b = b_cur;
    const int n_split = ns_cur;
    const int local = item - pref_cur;
    const int split = local / Hkv, g = local % Hkv;
    const int r0 = p.q_indptr[b];
    const int q_b = p.q_indptr[b + 1] - r0;
    const int ctx = kv.seq_len[b];
    const int len = ctx + q_b;
    const int pages = (len + 15) >> 4;
    const int pps = (pages + n_split - 1) / n_split;
    const int k0 = split * pps * 16;
    const int k1 = min(len, k0 + pps * 16);
    const int n_tiles = (k1 - k0 + AT_BN - 1) / AT_BN;
    const int R = q_b * p.group;                               // valid query rows
    const int32_t* bt = kv.block_table + (size_t)b * kv.max_pages_per_seq;
    const size_t layer_off = (size_t)p.layer * kv.num_pages;

    __syncthreads();                                           // previous item's smem fully consumed

    // ---- Q tile -> smem (rows r = i*group + hg are contiguous in global memory per i) ----
    for (int c = tid; c < R_PAD * CPR; c += AT_THREADS) {
      const int r = c / CPR, ch = c % CPR;
      const int i = r / p.group, hg = r % p.group;
      const __nv_bfloat16* src = p.q + ((size_t)(r0 + i) * p.n_q_heads + g * p.group + hg) * D + ch * 8;
      cp_async16(smem_u32(q_s) + swz<D>(r, ch), r < R ? src : p.q, r < R);
    }
    auto load_tile = [&](int t) {
      if (t < n_tiles) {
        uint8_t* ks = kv_s + (t % AT_STAGES) * 2 * TILE_BYTES;
        uint8_t* vs = ks + TILE_BYTES;
        const int tk0 = k0 + t * AT_BN;
#pragma unroll
        for (int it = 0; it < LD_ITERS; ++it) {
          const int c = it * AT_THREADS + tid;
          const int key = c / CPR, ch = c % CPR;
          const int pos = tk0 + key;
          const bool valid = pos < k1;
          const int page = valid ? __ldg(bt + (pos >> 4)) : 0;
          const size_t off = (((layer_off + page) * Hkv + g) * 16 + (pos & 15)) * D + ch * 8;
          const uint32_t so = swz<D>(key, ch);
          cp_async16(smem_u32(ks) + so, kv.k_pool + (valid ? off : 0), valid);
          cp_async16(smem_u32(vs) + so, kv.v_pool + (valid ? off : 0), valid);
        }
      }
      cp_async_commit();
    };
#pragma unroll
    for (int t = 0; t < AT_STAGES - 1; ++t) load_tile(t);      // group 0 also carries the Q tile

    float m_run[MT][2], l_run[MT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
      m_run[mt][0] = m_run[mt][1] = -INFINITY;
      l_run[mt][0] = l_run[mt][1] = 0.f;
#pragma unroll
      for (int nt = 0; nt < NT_O; ++nt) o[mt][nt][0] = o[mt][nt][1] = o[mt][nt][2] = o[mt][nt][3] = 0.f;
    }
    const int row_base = rg * 16 * MT;                         // this warp's first query row

    for (int t = 0; t < n_tiles; ++t) {
      cp_async_wait<AT_STAGES - 2>();
      __syncthreads();
      load_tile(t + AT_STAGES - 1);
      const uint32_t ks = smem_u32(kv_s + (t % AT_STAGES) * 2 * TILE_BYTES);
      const uint32_t vs = ks + TILE_BYTES;
      const uint32_t qs = smem_u32(q_s);

      // ---- S = Q K^T for this warp's 16*MT rows x 32 keys ----
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) s[mt][nt][0] = s[mt][nt][1] = s[mt][nt][2] = s[mt][nt][3] = 0.f;
#pragma unroll
      for (int ks16 = 0; ks16 < D / 16; ++ks16) {
        uint32_t a[MT][4];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
          const int row = row_base + mt * 16 + (lane & 15);
          ldsm_x4(qs + swz<D>(row, ks16 * 2 + (lane >> 4)), a[mt][0], a[mt][1], a[mt][2], a[mt][3]);
        }
#pragma unroll
        for (int np = 0; np < 2; ++np) {
          uint32_t b0, b1, b2, b3;
          const int key = kp * 32 + np * 16 + (lane & 7) + ((lane >> 4) << 3);
          ldsm_x4(ks + swz<D>(key, ks16 * 2 + ((lane >> 3) & 1)), b0, b1, b2, b3);
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) {
            mma_bf16(s[mt][np * 2 + 0], a[mt], b0, b1);
            mma_bf16(s[mt][np * 2 + 1], a[mt], b2, b3);
          }
        }
      }

      // ---- causal / tail mask (only tiles that reach the block's own tokens or the item end) ----
      const int tk0 = k0 + t * AT_BN + kp * 32;                // first key of this warp's slice
      if (tk0 + 32 > min(ctx + 1, k1)) {
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int r = row_base + mt * 16 + (lane >> 2) + h * 8;
            const int lim = min(k1, ctx + r / p.group + 1);    // keys j < lim are visible to row r
#pragma unroll
            for (int nt = 0; nt < 4; ++nt)
#pragma unroll
              for (int e = 0; e < 2; ++e) {
                const int j = tk0 + nt * 8 + (lane & 3) * 2 + e;
                if (j >= lim) s[mt][nt][h * 2 + e] = -INFINITY;
              }
          }
      }

      // ---- online softmax (log2 domain), P -> bf16 A fragments ----
      uint32_t pa[MT][2][4];
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          float mx = -INFINITY;
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) mx = fmaxf(mx, fmaxf(s[mt][nt][h * 2], s[mt][nt][h * 2 + 1]));
          mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
          mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
          const float m_new = fmaxf(m_run[mt][h], mx * p.scale_log2);
          const float m_use = m_new == -INFINITY ? 0.f : m_new;
          const float alpha = exp2f(m_run[mt][h] - m_use);
          m_run[mt][h] = m_new;
          float rs = 0.f;
#pragma unroll
          for (int nt = 0; nt < 4; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const float pv = exp2f(fmaf(s[mt][nt][h * 2 + e], p.scale_log2, -m_use));
              s[mt][nt][h * 2 + e] = pv;
              rs += pv;
            }
          l_run[mt][h] = l_run[mt][h] * alpha + rs;
#pragma unroll
          for (int nt = 0; nt < NT_O; ++nt) { o[mt][nt][h * 2] *= alpha; o[mt][nt][h * 2 + 1] *= alpha; }
        }
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) {
          pa[mt][kk][0] = pack_bf16(s[mt][kk * 2][0], s[mt][kk * 2][1]);
          pa[mt][kk][1] = pack_bf16(s[mt][kk * 2][2], s[mt][kk * 2][3]);
          pa[mt][kk][2] = pack_bf16(s[mt][kk * 2 + 1][0], s[mt][kk * 2 + 1][1]);
          pa[mt][kk][3] = pack_bf16(s[mt][kk * 2 + 1][2], s[mt][kk * 2 + 1][3]);
        }

      // ---- O += P V ----
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
        const int key = kp * 32 + kk * 16 + (lane & 7) + (((lane >> 3) & 1) << 3);
#pragma unroll
        for (int dp = 0; dp < NT_O / 2; ++dp) {
          uint32_t b0, b1, b2, b3;
          ldsm_x4_t(vs + swz<D>(key, dp * 2 + (lane >> 4)), b0, b1, b2, b3);
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) {
            mma_bf16(o[mt][dp * 2 + 0], pa[mt][kk], b0, b1);
            mma_bf16(o[mt][dp * 2 + 1], pa[mt][kk], b2, b3);
          }
        }
      }
    }
    cp_async_wait<0>();
    __syncthreads();                                           // all stages idle: reuse them as scratch

    // ---- merge the two key parts of each row group through smem ----
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        float l = l_run[mt][h];
        l += __shfl_xor_sync(0xffffffffu, l, 1);
        l += __shfl_xor_sync(0xffffffffu, l, 2);
        l_run[mt][h] = l;
      }
    float* xo = reinterpret_cast<float*>(kv_s) + (size_t)rg * (16 * MT) * (D + 2);   // [16*MT rows][D+2]
    if (kp == 1) {
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          float* rowp = xo + (mt * 16 + (lane >> 2) + h * 8) * (D + 2);
#pragma unroll
          for (int nt = 0; nt < NT_O; ++nt)
            *reinterpret_cast<float2*>(rowp + nt * 8 + (lane & 3) * 2) = make_float2(o[mt][nt][h * 2], o[mt][nt][h * 2 + 1]);
          if ((lane & 3) == 0) { rowp[D] = m_run[mt][h]; rowp[D + 1] = l_run[mt][h]; }
        }
    }
    __syncthreads();
    if (kp == 0) {
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int rl = mt * 16 + (lane >> 2) + h * 8;
          const float* rowp = xo + rl * (D + 2);
          const float m1 = rowp[D], l1 = rowp[D + 1];
          const float m0 = m_run[mt][h];
          const float m = fmaxf(m0, m1);
          const float mu = m == -INFINITY ? 0.f : m;
          const float e0 = exp2f(m0 - mu), e1 = exp2f(m1 - mu);
          const float l = l_run[mt][h] * e0 + l1 * e1;
          const int r = row_base + rl;
          if (r < R) {
            const int i = r / p.group, hg = r % p.group;
            if (n_split == 1) {
              const float inv = 1.f / l;                       // row r always sees key 0: l > 0
              __nv_bfloat16* dst = p.out + ((size_t)(r0 + i) * p.n_q_heads + g * p.group + hg) * D;
#pragma unroll
              for (int nt = 0; nt < NT_O; ++nt) {
                const int col = nt * 8 + (lane & 3) * 2;
                const float2 x = *reinterpret_cast<const float2*>(rowp + col);
                *reinterpret_cast<uint32_t*>(dst + col) =
                    pack_bf16((o[mt][nt][h * 2] * e0 + x.x * e1) * inv, (o[mt][nt][h * 2 + 1] * e0 + x.y * e1) * inv);
              }
            } else {
              float* dst = p.ws_o + ((size_t)item * R_PAD + r) * D;
#pragma unroll
              for (int nt = 0; nt < NT_O; ++nt) {
                const int col = nt * 8 + (lane & 3) * 2;
                const float2 x = *reinterpret_cast<const float2*>(rowp + col);
                *reinterpret_cast<float2*>(dst + col) =
                    make_float2(o[mt][nt][h * 2] * e0 + x.x * e1, o[mt][nt][h * 2 + 1] * e0 + x.y * e1);
              }
              if ((lane & 3) == 0) p.ws_ml[(size_t)item * R_PAD + r] = make_float2(m, l);
            }
          }
        }
    }
    if (n_split == 1) continue;

    // ---- split-KV combine by the last CTA to finish (b, g) ----
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      const unsigned int old = atomicAdd(&p.counters[b * Hkv + g], 1u);
      s_last = (old == (unsigned int)n_split - 1);
      if (s_last) p.counters[b * Hkv + g] = 0;
    }
    __syncthreads();
    if (!s_last) continue;
    __threadfence();
    const int item0 = pref_cur + g;                            // split s of (b,g) is item0 + s*Hkv
    // (1) normalised weight of every (split, row): w = 2^(m_s - m) / sum_s l_s 2^(m_s - m)  -> smem
    float* wgt = reinterpret_cast<float*>(kv_s);               // [n_split][R_PAD]; stages are idle here
    for (int r = tid; r < R; r += AT_THREADS) {
      float m = -INFINITY;
      for (int sp = 0; sp < n_split; ++sp) m = fmaxf(m, __ldcg(&p.ws_ml[(size_t)(item0 + sp * Hkv) * R_PAD + r].x));
      float l = 0.f;
      for (int sp = 0; sp < n_split; ++sp) {
        const float2 ml = __ldcg(&p.ws_ml[(size_t)(item0 + sp * Hkv) * R_PAD + r]);
        const float w = exp2f(ml.x - m);                       // -inf partials get weight 0
        wgt[sp * R_PAD + r] = w;
        l += ml.y * w;
      }
      const float inv = 1.f / l;
      for (int sp = 0; sp < n_split; ++sp) wgt[sp * R_PAD + r] *= inv;
    }
    __syncthreads();
    // (2) out[r][:] = sum_s w[s][r] O_s[r][:]; one warp per row, 16-byte loads, 4 splits in flight
    constexpr int C4 = D / 4;                                  // float4 per row
    for (int r = warp; r < R; r += AT_THREADS / 32) {
      const int i = r / p.group, hg = r % p.group;
      __nv_bfloat16* dst = p.out + ((size_t)(r0 + i) * p.n_q_heads + g * p.group + hg) * D;
      for (int c = lane; c < C4; c += 32) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        int sp = 0;
        for (; sp + 4 <= n_split; sp += 4) {
          float4 x[4];
#pragma unroll
          for (int u = 0; u < 4; ++u)
            x[u] = __ldcg(reinterpret_cast<const float4*>(p.ws_o + ((size_t)(item0 + (sp + u) * Hkv) * R_PAD + r) * D) + c);
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const float w = wgt[(sp + u) * R_PAD + r];
            acc.x += w * x[u].x; acc.y += w * x[u].y; acc.z += w * x[u].z; acc.w += w * x[u].w;
          }
        }
        for (; sp < n_split; ++sp) {
          const float4 x = __ldcg(reinterpret_cast<const float4*>(p.ws_o + ((size_t)(item0 + sp * Hkv) * R_PAD + r) * D) + c);
          const float w = wgt[sp * R_PAD + r];
          acc.x += w * x.x; acc.y += w * x.y; acc.z += w * x.z; acc.w += w * x.w;
        }
        uint2 pk = make_uint2(pack_bf16(acc.x, acc.y), pack_bf16(acc.z, acc.w));
        *reinterpret_cast<uint2*>(dst + c * 4) = pk;
      }
    }
  }
}

template <int D, int MT>
size_t attn_smem_bytes() { return (size_t)(32 * MT) * D * 2 + (size_t)AT_STAGES * 2 * AT_BN * D * 2; }

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int AT_TARGET_ITEMS_MAX = 148 * 16;      // the workspace is sized for this many + B*Hkv

int attn_target_items() {
  static int v = [] {
    const char* e = getenv("WF_ATTN_TARGET_ITEMS");   // tuning knob; default 148 SMs x AT_ITEMS_PER_SM
    int x = e ? atoi(e) : 148 * AT_ITEMS_PER_SM;
    return x < 1 ? 1 : (x > AT_TARGET_ITEMS_MAX ? AT_TARGET_ITEMS_MAX : x);
  }();
  return v;
}

template <int D, int MT>
int launch_attn(wf_ctx* ctx, const AttnParams& p, cudaStream_t st) {
  static int grid = 0;
  const size_t smem = attn_smem_bytes<D, MT>();
  if (grid == 0) {
    WF_CUDA(ctx, cudaFuncSetAttribute(wf_verify_attn_kernel<D, MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    WF_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, wf_verify_attn_kernel<D, MT>, AT_THREADS, smem));
    WF_REQUIRE(ctx, occ > 0, WF_ERR_CUDA, "wf_verify_attn: kernel does not fit on an SM");
    grid = occ * ctx->sm_count;
  }
  wf_verify_attn_kernel<D, MT><<<grid, AT_THREADS, smem, st>>>(p);
  return wf_check_launch(ctx, "wf_verify_attn_kernel");
}

inline int attn_r_pad(int n_q_heads, int n_kv_heads, int max_q_len) {
  const int rows = max_q_len * (n_q_heads / n_kv_heads);
  return rows <= 32 ? 32 : 64;
}

}  // namespace

extern "C" size_t wf_verify_attn_workspace_bytes(const wf_kv_shape* s, int B, int n_q_heads, int max_q_len) {
  if (!s || B <= 0 || n_q_heads <= 0 || s->n_kv_heads <= 0) return 16;
  const size_t items = (size_t)AT_TARGET_ITEMS_MAX + (size_t)B * s->n_kv_heads;
  const size_t r_pad = attn_r_pad(n_q_heads, s->n_kv_heads, max_q_len);
  return items * r_pad * ((size_t)s->head_dim * sizeof(float) + sizeof(float2));
}

extern "C" int wf_verify_attn(wf_ctx* ctx, const wf_paged_kv* kv, int layer, const void* q,
                              const int32_t* q_indptr, int B, int n_q_heads, int max_q_len, float sm_scale,
                              void* out, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, kv && q && q_indptr && out && workspace, WF_ERR_INVALID_ARG, "wf_verify_attn: null argument");
  WF_REQUIRE(ctx, layer >= 0 && layer < kv->s.n_layers, WF_ERR_INVALID_ARG, "wf_verify_attn: bad layer");
  WF_REQUIRE(ctx, B >= 0 && B <= kv->s.max_seqs && B <= AT_MAX_B && B * kv->s.n_kv_heads <= ctx->n_counters,
             WF_ERR_INVALID_ARG, "wf_verify_attn: bad B (max %d)", AT_MAX_B);
  WF_REQUIRE(ctx, n_q_heads > 0 && n_q_heads % kv->s.n_kv_heads == 0, WF_ERR_INVALID_ARG,
             "wf_verify_attn: n_q_heads must be a multiple of n_kv_heads");
  const int group = n_q_heads / kv->s.n_kv_heads;
  WF_REQUIRE(ctx, max_q_len >= 1 && max_q_len * group <= 64, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_verify_attn: max_q_len * group must be in [1, 64]");
  WF_REQUIRE(ctx, workspace_bytes >= wf_verify_attn_workspace_bytes(&kv->s, B, n_q_heads, max_q_len),
             WF_ERR_INVALID_ARG, "wf_verify_attn: workspace too small");
  WF_REQUIRE(ctx, ((uintptr_t)q % 16 == 0) && ((uintptr_t)out % 16 == 0) && ((uintptr_t)workspace % 16 == 0),
             WF_ERR_INVALID_ARG, "wf_verify_attn: q/out/workspace must be 16-byte aligned");
  if (B == 0) return WF_OK;
  const int r_pad = attn_r_pad(n_q_heads, kv->s.n_kv_heads, max_q_len);
  const size_t items = (size_t)AT_TARGET_ITEMS_MAX + (size_t)B * kv->s.n_kv_heads;
  AttnParams p;
  p.q = (const __nv_bfloat16*)q;
  p.out = (__nv_bfloat16*)out;
  p.q_indptr = q_indptr;
  p.kv = kv_view(kv);
  p.layer = layer; p.B = B; p.n_q_heads = n_q_heads; p.group = group;
  p.scale_log2 = sm_scale * LOG2E;
  p.target_items = attn_target_items();
  p.ws_o = (float*)workspace;
  p.ws_ml = (float2*)((char*)workspace + items * r_pad * kv->s.head_dim * sizeof(float));
  p.counters = ctx->d_counters_attn;
  cudaStream_t st = (cudaStream_t)stream;
  const int D = kv->s.head_dim;
  if (D == 128 && r_pad == 64) return launch_attn<128, 2>(ctx, p, st);
  if (D == 128 && r_pad == 32) return launch_attn<128, 1>(ctx, p, st);
  if (D == 64 && r_pad == 64) return launch_attn<64, 2>(ctx, p, st);
  if (D == 64 && r_pad == 32) return launch_attn<64, 1>(ctx, p, st);
  return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "wf_verify_attn: head_dim %d unsupported", D);
}

// (a) Target-model verification attention over the paged bf16 GQA KV cache.
// PAPER.md:65 (§3.2 "parallel verification"); readings C10-C13.
//
// Split-KV, decode-style, tcgen05.  A work item is (sequence b, kv head g, key range [k0,k1)); its
// query tile is all q_b rows of the `group` query heads that share kv head g (<= 64 rows), so K and V
// are read from HBM once per kv head.  One persistent CTA per SM walks the item list, which every CTA
// derives from the device-resident lengths (no host sync).  Warp roles:
//   warp 2    : TMA producer.  Per 128-key tile, lane p issues the 16-key page p of K and of V
//               (cp.async.bulk.tensor.2d, 128-byte swizzle) into an mbarrier ring of stages.
//   warp 3    : MMA issuer (one thread).  S = Q K^T (UMMA 128 x 128 x 16, both K-major) into TMEM,
//               double buffered; O_t = P V (128 x D x 16, V MN-major) into TMEM, double buffered.
//   warps 0,1,4,5 : softmax.  Thread = (query row = TMEM lane, half of the tile's keys).  S comes out
//               of TMEM with tcgen05.ld, online softmax in the log2 domain, P goes to smem as the bf16
//               A operand of the PV MMA, and the per-tile O_t is folded into fp32 registers with the
//               running rescale.  QK^T of tile t+1 overlaps the softmax of tile t.
// Split partials (fp32 O, m, l) are merged by the last CTA to finish a (b, g) pair.
#include "wf_internal.cuh"
#include "wf_sm100.cuh"

namespace {

constexpr int AT_THREADS = 256;
constexpr int AT_BN = 128;             // keys per tile
constexpr int AT_ROWS = 64;            // query rows staged (UMMA M = 128; rows 64.. are never read back)
constexpr int AT_MIN_CHUNK = 256;      // never split below this many keys
constexpr int AT_ITEMS_PER_SM = 8;     // target number of work items per SM
constexpr int AT_MAX_B = 1024;
constexpr int AT_MAX_STAGES = 4;
constexpr float LOG2E = 1.4426950408889634f;

struct AttnParams {
  const __nv_bfloat16* q;
  __nv_bfloat16* out;
  const int32_t* q_indptr;
  KvView kv;
  int layer, B, n_q_heads, group;
  float scale_log2;                    // sm_scale * log2(e)
  int target_items;
  float* ws_o;                         // [items][64][D] fp32, unnormalised
  float2* ws_ml;                       // [items][64] (m in log2 units, l)
  unsigned int* counters;              // [B * Hkv], self-resetting
};

template <int D>
struct AttnCfg {
  static constexpr int NH = D / 64;                         // 64-element (128-byte) column halves of a K/V row
  static constexpr int Q_BYTES = AT_ROWS * D * 2;           // NH halves x 64 rows x 128 B
  static constexpr int P_BYTES = 2 * AT_ROWS * 128;         // 2 key halves x 64 rows x 128 B
  static constexpr int KV_HALF = AT_BN * 128;               // one column half of a K (or V) tile: 16 KB
  static constexpr int K_BYTES = NH * KV_HALF;
  static constexpr int STAGE_BYTES = 2 * K_BYTES;
  static constexpr int STAGES = D == 128 ? 3 : 4;
  static constexpr int SMEM = Q_BYTES + P_BYTES + STAGES * STAGE_BYTES;
  static constexpr uint32_t TM_S = 0, TM_O = 2 * AT_BN;     // TMEM columns: S0, S1, then O0, O1
};

struct ItemInfo {
  int b, g, split, n_split, r0, q_b, ctx, k0, k1, n_tiles, item0;
};

// shared state of one CTA (static smem)
struct AttnShared {
  uint64_t kv_full[AT_MAX_STAGES], kv_empty[AT_MAX_STAGES];
  uint64_t s_full[2], s_empty[2], o_empty[2], p_full, pv_done, q_ready;
  float xmax[2][2][AT_ROWS];
  float xl[2][AT_ROWS];
  int red[AT_THREADS / 32];
  int chunk;
  uint32_t tmem;
  int last;
};

// Walks the b-major item list (item = pref_b + split * Hkv + g); every role keeps its own walker.
struct ItemWalker {
  const AttnParams& p;
  int chunk_target;
  int b_cur = 0, pref_cur = 0, ns_cur = 0;
  __device__ ItemWalker(const AttnParams& p_, int chunk) : p(p_), chunk_target(chunk) {
    ns_cur = p.B > 0 ? splits_of(len_of(0)) : 0;
  }
  __device__ int len_of(int b) const {
    const int qb = p.q_indptr[b + 1] - p.q_indptr[b];
    return qb > 0 ? p.kv.seq_len[b] + qb : 0;
  }
  __device__ int splits_of(int len) const {     // page-aligned equal parts of about chunk_target keys
    if (len <= 0) return 0;
    const int pages = (len + 15) >> 4;
    const int ns0 = (len + chunk_target - 1) / chunk_target;
    const int pps = (pages + ns0 - 1) / ns0;
    return (pages + pps - 1) / pps;
  }
  __device__ bool next(int item, ItemInfo& it) {
    const int Hkv = p.kv.n_kv_heads;
    while (b_cur < p.B && item >= pref_cur + ns_cur * Hkv) {
      pref_cur += ns_cur * Hkv;
      ++b_cur;
      ns_cur = b_cur < p.B ? splits_of(len_of(b_cur)) : 0;
    }
    if (b_cur >= p.B) return false;
    it.b = b_cur; it.n_split = ns_cur;
    const int local = item - pref_cur;
    it.split = local / Hkv; it.g = local % Hkv;
    it.r0 = p.q_indptr[b_cur];
    it.q_b = p.q_indptr[b_cur + 1] - it.r0;
    it.ctx = p.kv.seq_len[b_cur];
    const int len = it.ctx + it.q_b;
    const int pages = (len + 15) >> 4;
    const int pps = (pages + ns_cur - 1) / ns_cur;
    it.k0 = it.split * pps * 16;
    it.k1 = min(len, it.k0 + pps * 16);
    it.n_tiles = (it.k1 - it.k0 + AT_BN - 1) / AT_BN;
    it.item0 = pref_cur + it.g;
    return true;
  }
};

// ================= warp 2: TMA producer =================
template <int D>
__device__ __forceinline__ void attn_loader(const AttnParams& p, AttnShared& sh, uint8_t* kv_s, int chunk, int lane) {
  using C = AttnCfg<D>;
  const KvView& kv = p.kv;
  ItemWalker walk(p, chunk);
  ItemInfo it;
  uint32_t gt = 0;
  for (int item = blockIdx.x; walk.next(item, it); item += gridDim.x) {
    const int32_t* bt = kv.block_table + (size_t)it.b * kv.max_pages_per_seq;
    for (int t = 0; t < it.n_tiles; ++t, ++gt) {
      const int st = gt % C::STAGES;
      mbar_wait(smem_u32(&sh.kv_empty[st]), ((gt / C::STAGES) & 1) ^ 1);
      const int tk0 = it.k0 + t * AT_BN;
      const int npages = min(AT_BN / 16, (it.k1 - tk0 + 15) >> 4);
      if (lane == 0) mbar_arrive_expect_tx(smem_u32(&sh.kv_full[st]), (uint32_t)npages * 2 * 16 * D * 2);
      __syncwarp();
      if (lane < npages) {
        const int page = __ldg(bt + (tk0 >> 4) + lane);
        const int row = (((p.layer * kv.num_pages + page) * kv.n_kv_heads) + it.g) * 16;
        const uint32_t ks = smem_u32(kv_s + (size_t)st * C::STAGE_BYTES) + lane * 2048;
        const uint32_t vs = ks + C::K_BYTES;
#pragma unroll
        for (int h = 0; h < C::NH; ++h) {
          tma_load_2d(ks + h * C::KV_HALF, kv.tmaps + 0, h * 64, row, smem_u32(&sh.kv_full[st]));
          tma_load_2d(vs + h * C::KV_HALF, kv.tmaps + 1, h * 64, row, smem_u32(&sh.kv_full[st]));
        }
      }
    }
  }
}

// ================= warp 3, one thread: MMA issuer =================
template <int D>
__device__ __forceinline__ void attn_mma(const AttnParams& p, AttnShared& sh, uint8_t* q_s, uint8_t* p_s, uint8_t* kv_s,
                                         int chunk, uint32_t tmem_base) {
  using C = AttnCfg<D>;
  const uint32_t idesc_qk = umma_idesc_kk(128, AT_BN);
  const uint32_t idesc_pv = umma_idesc(128, D);
  ItemWalker walk(p, chunk);
  ItemInfo it;
  uint32_t gt = 0, n_item = 0;
  auto issue_qk = [&](uint32_t g2) {
    const int st = g2 % C::STAGES;
    mbar_wait(smem_u32(&sh.kv_full[st]), (g2 / C::STAGES) & 1);
    mbar_wait(smem_u32(&sh.s_empty[g2 & 1]), ((g2 >> 1) & 1) ^ 1);
    tc_fence_after();
    const uint32_t ks = smem_u32(kv_s + (size_t)st * C::STAGE_BYTES);
    const uint32_t qs = smem_u32(q_s);
#pragma unroll
    for (int k16 = 0; k16 < D / 16; ++k16) {
      const uint64_t da = umma_desc(qs + (k16 >> 2) * (AT_ROWS * 128) + (k16 & 3) * 32, 16, 1024);
      const uint64_t db = umma_desc(ks + (k16 >> 2) * C::KV_HALF + (k16 & 3) * 32, 16, 1024);
      umma_bf16(tmem_base + C::TM_S + (g2 & 1) * AT_BN, da, db, idesc_qk, k16 != 0);
    }
    umma_commit(smem_u32(&sh.s_full[g2 & 1]));
  };
  for (int item = blockIdx.x; walk.next(item, it); item += gridDim.x, ++n_item) {
    mbar_wait(smem_u32(&sh.q_ready), n_item & 1);
    tc_fence_after();
    issue_qk(gt);
    for (int t = 0; t < it.n_tiles; ++t, ++gt) {
      if (t + 1 < it.n_tiles) issue_qk(gt + 1);
      const int st = gt % C::STAGES;
      mbar_wait(smem_u32(&sh.p_full), gt & 1);
      mbar_wait(smem_u32(&sh.o_empty[gt & 1]), ((gt >> 1) & 1) ^ 1);
      tc_fence_after();
      const uint32_t vs = smem_u32(kv_s + (size_t)st * C::STAGE_BYTES) + C::K_BYTES;
      const uint32_t ps = smem_u32(p_s);
#pragma unroll
      for (int k16 = 0; k16 < AT_BN / 16; ++k16) {
        const uint64_t da = umma_desc(ps + (k16 >> 2) * (AT_ROWS * 128) + (k16 & 3) * 32, 16, 1024);
        const uint64_t db = umma_desc(vs + k16 * 2048, C::KV_HALF, 1024);               // MN-major
        umma_bf16(tmem_base + C::TM_O + (gt & 1) * D, da, db, idesc_pv, k16 != 0);
      }
      umma_commit(smem_u32(&sh.pv_done));
      umma_commit(smem_u32(&sh.kv_empty[st]));
    }
  }
}

// ================= warps 0, 1, 4, 5: softmax, O accumulation, output, split combine =================
template <int D>
__device__ __forceinline__ void attn_softmax(const AttnParams& p, AttnShared& sh, uint8_t* q_s, uint8_t* p_s, uint8_t* kv_s,
                                             int chunk, uint32_t tmem_base, int warp, int lane) {
  using C = AttnCfg<D>;
  const int Hkv = p.kv.n_kv_heads;
  const int quarter = warp & 3, ch = warp >> 2;
  const int r = quarter * 32 + lane;                           // query row = TMEM lane
  const int stid = ch * 64 + r;                                // 0..127 among the softmax threads
  const uint32_t t_lane = tmem_base + ((uint32_t)(quarter * 32) << 16);
  ItemWalker walk(p, chunk);
  ItemInfo it;
  uint32_t gt = 0;
  for (int item = blockIdx.x; walk.next(item, it); item += gridDim.x) {
    const int R = it.q_b * p.group;
    const int qi = r / p.group, hg = r % p.group;
    // ---- Q tile -> smem (K-major, 128-byte swizzle); rows >= R are zero.  All MMAs of the previous
    //      item have retired: this thread waited for its last pv_done. ----
    for (int c = stid; c < AT_ROWS * (D / 8); c += 128) {
      const int rr = c / (D / 8), chn = c % (D / 8);
      uint4 v = make_uint4(0, 0, 0, 0);
      if (rr < R) {
        const int i2 = rr / p.group, h2 = rr % p.group;
        v = __ldg(reinterpret_cast<const uint4*>(p.q + ((size_t)(it.r0 + i2) * p.n_q_heads + it.g * p.group + h2) * D) + chn);
      }
      *reinterpret_cast<uint4*>(q_s + (chn >> 3) * (AT_ROWS * 128) + rr * 128 + (((chn & 7) ^ (rr & 7)) << 4)) = v;
    }
    fence_proxy_async();
    mbar_arrive(smem_u32(&sh.q_ready));

    float m_run = -INFINITY, l_run = 0.f, alpha_prev = 0.f;
    float o[D / 2];
#pragma unroll
    for (int c = 0; c < D / 2; ++c) o[c] = 0.f;
    const int lim_row = min(it.k1, it.ctx + qi + 1);           // keys j < lim_row are visible to this row

    auto fold_o = [&](uint32_t g2, float alpha) {              // o = o * alpha + O_tile(g2)
      const uint32_t ta = t_lane + C::TM_O + (g2 & 1) * D + ch * (D / 2);
#pragma unroll
      for (int c0 = 0; c0 < D / 2; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(ta + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int c = 0; c < 32; ++c) o[c0 + c] = fmaf(o[c0 + c], alpha, __uint_as_float(v[c]));
      }
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.o_empty[g2 & 1]));
    };

    for (int t = 0; t < it.n_tiles; ++t, ++gt) {
      const int tk0 = it.k0 + t * AT_BN;
      mbar_wait(smem_u32(&sh.s_full[gt & 1]), (gt >> 1) & 1);
      tc_fence_after();
      uint32_t sv[64];
      {
        uint32_t a0[32], a1[32];
        const uint32_t ta = t_lane + C::TM_S + (gt & 1) * AT_BN + ch * 64;
        tmem_ld32(ta, a0);
        tmem_ld32(ta + 32, a1);
        tmem_ld_wait();
#pragma unroll
        for (int c = 0; c < 32; ++c) { sv[c] = a0[c]; sv[32 + c] = a1[c]; }
      }
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.s_empty[gt & 1]));              // S buffer may be overwritten by QK(t+2)

      const bool tail = tk0 + AT_BN > min(it.ctx + 1, it.k1);
      float mx = -INFINITY;
      if (tail) {
        const int j0 = tk0 + ch * 64;
#pragma unroll
        for (int c = 0; c < 64; ++c) {
          const float x = (j0 + c < lim_row) ? __uint_as_float(sv[c]) : -INFINITY;
          sv[c] = __float_as_uint(x);
          mx = fmaxf(mx, x);
        }
      } else {
#pragma unroll
        for (int c = 0; c < 64; ++c) mx = fmaxf(mx, __uint_as_float(sv[c]));
      }
      sh.xmax[gt & 1][ch][r] = mx;
      named_bar_sync(1 + quarter, 64);
      mx = fmaxf(mx, sh.xmax[gt & 1][ch ^ 1][r]);
      const float m_new = fmaxf(m_run, mx * p.scale_log2);
      const float m_use = m_new == -INFINITY ? 0.f : m_new;
      const float alpha = exp2f(m_run - m_use);
      m_run = m_new;
      float rs = 0.f;
      uint32_t pk[32];
#pragma unroll
      for (int c = 0; c < 64; c += 2) {
        const float p0 = exp2f(fmaf(__uint_as_float(sv[c]), p.scale_log2, -m_use));
        const float p1 = exp2f(fmaf(__uint_as_float(sv[c + 1]), p.scale_log2, -m_use));
        rs += p0 + p1;
        pk[c >> 1] = pack_bf16(p0, p1);
      }
      l_run = l_run * alpha + rs;

      if (tk0 + AT_BN > it.k1) {
        // Last tile of the sequence: keys >= k1 hold stale or never-written V bits.  Zero them so that
        // 0 * garbage cannot produce NaN in the PV product (P is exactly 0 there).
        mbar_wait(smem_u32(&sh.kv_full[gt % C::STAGES]), (gt / C::STAGES) & 1);
        const int key = (it.k1 - tk0) + stid;
        if (key < AT_BN) {
          uint8_t* vrow = kv_s + (size_t)(gt % C::STAGES) * C::STAGE_BYTES + C::K_BYTES + key * 128;
#pragma unroll
          for (int h = 0; h < C::NH; ++h)
#pragma unroll
            for (int c = 0; c < 8; ++c) *reinterpret_cast<uint4*>(vrow + h * C::KV_HALF + c * 16) = make_uint4(0, 0, 0, 0);
        }
      }
      if (t > 0) mbar_wait(smem_u32(&sh.pv_done), (gt - 1) & 1);          // PV(t-1) retired: P is free, O(t-1) is ready
      {
        uint8_t* prow = p_s + ch * (AT_ROWS * 128) + r * 128;
#pragma unroll
        for (int c = 0; c < 8; ++c)
          *reinterpret_cast<uint4*>(prow + ((c ^ (r & 7)) << 4)) = make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
      }
      fence_proxy_async();
      mbar_arrive(smem_u32(&sh.p_full));
      if (t > 0) { tc_fence_after(); fold_o(gt - 1, alpha_prev); }
      alpha_prev = alpha;
    }
    mbar_wait(smem_u32(&sh.pv_done), (gt - 1) & 1);
    tc_fence_after();
    fold_o(gt - 1, alpha_prev);

    // ---- row sums of the two key halves; write the final rows or the split partial ----
    sh.xl[ch][r] = l_run;
    named_bar_sync(1 + quarter, 64);
    const float l_tot = l_run + sh.xl[ch ^ 1][r];
    if (r < R) {
      if (it.n_split == 1) {
        const float inv = 1.f / l_tot;                         // every row sees key 0: l > 0
        __nv_bfloat16* dst = p.out + ((size_t)(it.r0 + qi) * p.n_q_heads + it.g * p.group + hg) * D + ch * (D / 2);
#pragma unroll
        for (int c = 0; c < D / 2; c += 8)
          *reinterpret_cast<uint4*>(dst + c) = make_uint4(pack_bf16(o[c] * inv, o[c + 1] * inv), pack_bf16(o[c + 2] * inv, o[c + 3] * inv),
                                                          pack_bf16(o[c + 4] * inv, o[c + 5] * inv), pack_bf16(o[c + 6] * inv, o[c + 7] * inv));
      } else {
        float* dst = p.ws_o + ((size_t)item * AT_ROWS + r) * D + ch * (D / 2);
#pragma unroll
        for (int c = 0; c < D / 2; c += 4) *reinterpret_cast<float4*>(dst + c) = make_float4(o[c], o[c + 1], o[c + 2], o[c + 3]);
        if (ch == 0) p.ws_ml[(size_t)item * AT_ROWS + r] = make_float2(m_run, l_tot);
      }
    }
    if (it.n_split == 1) continue;

    // ---- split-KV combine by the last CTA to finish (b, g) ----
    __threadfence();
    named_bar_sync(3, 128);
    if (stid == 0) {
      const unsigned int old = atomicAdd(&p.counters[it.b * Hkv + it.g], 1u);
      sh.last = (old == (unsigned int)it.n_split - 1);
      if (sh.last) p.counters[it.b * Hkv + it.g] = 0;
    }
    named_bar_sync(3, 128);
    const bool last = sh.last != 0;
    named_bar_sync(3, 128);                                    // everyone has read the flag before it is reused
    if (!last) continue;
    __threadfence();
    const int cw = stid >> 5;                                  // 4 combine warps, one row at a time each
    for (int rr = cw; rr < R; rr += 4) {
      float m = -INFINITY;
      for (int sp = lane; sp < it.n_split; sp += 32)
        m = fmaxf(m, __ldcg(&p.ws_ml[(size_t)(it.item0 + sp * Hkv) * AT_ROWS + rr].x));
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      float l = 0.f;
      for (int base = 0; base < it.n_split; base += 32) {
        const int sp = base + lane;
        float w = 0.f, lw = 0.f;
        if (sp < it.n_split) {
          const float2 ml = __ldcg(&p.ws_ml[(size_t)(it.item0 + sp * Hkv) * AT_ROWS + rr]);
          w = exp2f(ml.x - m);                                 // -inf partials get weight 0
          lw = ml.y * w;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) lw += __shfl_xor_sync(0xffffffffu, lw, d);
        l += lw;
        const int cnt = min(32, it.n_split - base);
#pragma unroll 4
        for (int u = 0; u < cnt; ++u) {
          const float wu = __shfl_sync(0xffffffffu, w, u);
          if (lane < D / 4) {
            const float4 x = __ldcg(reinterpret_cast<const float4*>(p.ws_o + ((size_t)(it.item0 + (base + u) * Hkv) * AT_ROWS + rr) * D) + lane);
            acc.x = fmaf(wu, x.x, acc.x); acc.y = fmaf(wu, x.y, acc.y); acc.z = fmaf(wu, x.z, acc.z); acc.w = fmaf(wu, x.w, acc.w);
          }
        }
      }
      const float inv = 1.f / l;
      const int i2 = rr / p.group, h2 = rr % p.group;
      __nv_bfloat16* dst = p.out + ((size_t)(it.r0 + i2) * p.n_q_heads + it.g * p.group + h2) * D;
      if (lane < D / 4)
        *reinterpret_cast<uint2*>(dst + lane * 4) = make_uint2(pack_bf16(acc.x * inv, acc.y * inv), pack_bf16(acc.z * inv, acc.w * inv));
    }
  }
}

template <int D>
__global__ void __launch_bounds__(AT_THREADS, 1) wf_verify_attn_kernel(const AttnParams p) {
  using C = AttnCfg<D>;
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) AttnShared sh;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint8_t* q_s = smem;
  uint8_t* p_s = smem + C::Q_BYTES;
  uint8_t* kv_s = p_s + C::P_BYTES;

  // split size from the device-resident lengths (identical in every CTA, no host sync)
  int part = 0;
  for (int b = tid; b < p.B; b += AT_THREADS) {
    const int qb = p.q_indptr[b + 1] - p.q_indptr[b];
    part += qb > 0 ? p.kv.seq_len[b] + qb : 0;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
  if (lane == 0) sh.red[warp] = part;
  if (tid == 0) {
    for (int i = 0; i < C::STAGES; ++i) { mbar_init(smem_u32(&sh.kv_full[i]), 1); mbar_init(smem_u32(&sh.kv_empty[i]), 1); }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&sh.s_full[i]), 1);
      mbar_init(smem_u32(&sh.s_empty[i]), 128);
      mbar_init(smem_u32(&sh.o_empty[i]), 128);
    }
    mbar_init(smem_u32(&sh.p_full), 128);
    mbar_init(smem_u32(&sh.pv_done), 1);
    mbar_init(smem_u32(&sh.q_ready), 128);
    fence_barrier_init();
  }
  if (warp == 3) tmem_alloc(smem_u32(&sh.tmem), 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = sh.tmem;
  if (tid == 0) {
    long long total = 0;
    for (int w = 0; w < AT_THREADS / 32; ++w) total += sh.red[w];
    long long c = (total * p.kv.n_kv_heads + p.target_items - 1) / p.target_items;
    c = (c + AT_BN - 1) / AT_BN * AT_BN;
    sh.chunk = (int)max((long long)AT_MIN_CHUNK, c);
  }
  __syncthreads();
  const int chunk = sh.chunk;

  if (warp == 2) {
    attn_loader<D>(p, sh, kv_s, chunk, lane);
  } else if (warp == 3) {
    if (lane == 0) attn_mma<D>(p, sh, q_s, p_s, kv_s, chunk, tmem_base);
  } else if ((warp & 3) < 2) {
    attn_softmax<D>(p, sh, q_s, p_s, kv_s, chunk, tmem_base, warp, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 3) tmem_dealloc(tmem_base, 512);
}

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

template <int D>
int launch_attn(wf_ctx* ctx, const AttnParams& p, cudaStream_t st) {
  static bool configured = false;
  const size_t smem = AttnCfg<D>::SMEM;
  if (!configured) {
    WF_CUDA(ctx, cudaFuncSetAttribute(wf_verify_attn_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = true;
  }
  wf_verify_attn_kernel<D><<<ctx->sm_count, AT_THREADS, smem, st>>>(p);     // one persistent CTA per SM
  return wf_check_launch(ctx, "wf_verify_attn_kernel");
}

}  // namespace

extern "C" size_t wf_verify_attn_workspace_bytes(const wf_kv_shape* s, int B, int n_q_heads, int max_q_len) {
  if (!s || B <= 0 || n_q_heads <= 0 || s->n_kv_heads <= 0) return 16;
  const size_t items = (size_t)AT_TARGET_ITEMS_MAX + (size_t)B * s->n_kv_heads;
  const size_t r_pad = AT_ROWS;
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
  const int r_pad = AT_ROWS;
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
  if (D == 128) return launch_attn<128>(ctx, p, st);
  if (D == 64) return launch_attn<64>(ctx, p, st);
  return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "wf_verify_attn: head_dim %d unsupported", D);
}

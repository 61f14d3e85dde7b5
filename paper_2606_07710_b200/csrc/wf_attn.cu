// (a) Target-model verification attention over the paged bf16 GQA KV cache.
// PAPER.md:65 (§3.2 "parallel verification"); readings C10-C13.
//
// Split-KV, decode-style, tcgen05.  The query tile of a (sequence b, kv head g) pair is all q_b rows of
// the `group` query heads that share kv head g (<= 64 rows), so K and V are read from HBM once per kv
// head.  Work is the flattened list of 128-key tiles over all (b, g) pairs, each pair preceded by
// AT_SEG_COST positions that stand for the fixed cost of a segment; persistent CTA c (one per SM) owns the
// contiguous position range [c*T/G, (c+1)*T/G) (cost-weighted stream-K), which every CTA derives from the
// device-resident lengths through a per-sequence table in shared memory (no host sync, no global round
// trips in the walkers).  A range cuts at most two (b, g) pairs.  The last CTA to arrive at a shared pair
// keeps its partial in registers and folds in the partials the others published (fragment-order float4,
// coalesced; more than two are staged through the idle shared memory with cp.async); nobody re-reads
// its own partial.  Launched with programmatic dependent launch: barrier init and TMEM allocation run
// before griddepcontrol.wait; in the early-KV mode (wf_ctx_set_attn_early_kv) so do the length table, the page ids and the
// TMA loads of every tile below the cached length: only Q, the tree masks and the tiles that hold the block's own rows wait.
// Other launch shapes (launch_attn): one thread-block cluster per (b, g) pair with the merge through distributed shared memory
// (few pairs: batch 1-4), or one CTA per pair with no merge at all (HBM-paced launches whose pairs cover >= 80 % of the SMs).
// Warp roles:
//   warps 8,10: TMA producers (K ring, V ring).  One elected lane issues the 16 page boxes of a tile
//               (cp.async.bulk.tensor.2d, 128-byte swizzle) in straight-line code; the page ids of the
//               next tile are prefetched; a K tile is released when its QK^T retires.
//   warps 9,11: MMA issuers (one elected thread each).  Warp 9: S = Q K^T (UMMA 64 x 128 x 16, both K-major) into
//               TMEM, double buffered; warp 11: O_t = P V (64 x D x 16, V MN-major) into TMEM, double buffered.
//   warps 0-7 : softmax, two groups of 4 warps that ping-pong over the tiles.  UMMA M = 64 puts rows
//               16w..16w+15 on TMEM lanes 32w..32w+15, so warp w owns 16 rows; tcgen05.ld.16x256b hands
//               them out like an mma C fragment (a quad per row).  Online softmax in the log2 domain
//               with quad shuffles, P goes to smem as the bf16 A operand of the PV MMA, the per-tile
//               O_t is folded into fp32 registers with the running rescale.  The next segment's Q rows
//               are prefetched into L2; the Q tile is loaded with all loads ahead of the stores.
//
// Tree mode (wf_verify_attn_tree; template flag TREE, readings T1-T2): the draft tree of a
// sequence (<= 64 nodes, one 64-bit ancestor mask per row) is cut into blocks of 128 query rows = UMMA M = 128: two 64-row
// sub-blocks stacked on the TMEM lanes (A on lanes 32w..32w+15, B on 32w+16..32w+31 of quadrant w).  Softmax group g
// works on sub-block g of the same K/V tile (attn_softmax_tree); the blocks of a tree are listed level-major so that
// they stream the same K/V tiles from different CTAs at the same time: HBM is read once, the second reader hits L2.
#include "wf_internal.cuh"
#include "wf_sm100.cuh"

// Timeline probes (clock64 per CTA; compiled in only with -DWF_PROBE): slot k of CTA c.
#ifdef WF_PROBE
__device__ long long* wf_probe_buf = nullptr;
#define WF_PROBE_AT(k, cond) do { if (wf_probe_buf && (cond)) wf_probe_buf[blockIdx.x * 32 + (k)] = clock64(); } while (0)
extern "C" int wf_debug_set_attn_probe(long long* buf) { return (int)cudaMemcpyToSymbol(wf_probe_buf, &buf, sizeof(buf)); }
#else
#define WF_PROBE_AT(k, cond) do { } while (0)
#endif

namespace {

constexpr int AT_THREADS = 384;           // 12 warps: 0-3 / 4-7 softmax groups, 8 K loader, 9 QK^T issuer, 10 V loader, 11 PV issuer
constexpr int AT_BN = 128;             // keys per tile
constexpr int AT_ROWS = 64;            // query rows = UMMA M
constexpr int AT_MAX_B = 1024;
constexpr int AT_MAX_STAGES = 5;
constexpr int AT_MAX_CTAS = 160;       // workspace is sized for this many persistent CTAs
constexpr int AT_MAX_SEG = 32;         // partials merged per (b, g) pair
constexpr int AT_SEG_COST = 5;         // fixed cost of a segment (Q load, pipeline restart, merge, stores) in tiles; measured at cfg5
                                       // (us per launch): 2: 192.6, 3: 184.8, 4: 178.5, 5: 176.3-177.2, 6: 176.9-178.3, 7: 178.8-179.3,
                                       // 8: 179.4, 10: 184.8, 14: 190.7
constexpr int AT_SEG_COST_TREE = 8;    // the same for a 128-row tree block (Q tile of 32 KB, merges per sub-block); 60-node trees at cfg5
                                       // shapes (us per launch): 4: 388, 5: 369, 8: 352, 12: 354, 16: 362
template <bool TREE> constexpr int seg_cost() { return TREE ? AT_SEG_COST_TREE : AT_SEG_COST; }
constexpr float LOG2E = 1.4426950408889634f;

struct AttnParams {
  const __nv_bfloat16* q;
  __nv_bfloat16* out;
  const int32_t* q_indptr;
  const unsigned long long* tree_mask; // TREE only: [sum_q] ancestor mask of each row (bit j = node j of its sequence)
  KvView kv;
  int layer, B, n_q_heads, group;
  int cl;                              // > 0: cluster mode (launched with clusters of `cl` CTAs, one cluster per (b, g) pair)
  int deterministic;                   // stream-K merges fold the partials of a pair in range order, whoever arrives last
  int early;                           // wf_ctx_set_attn_early_kv: lengths, page ids and the K/V tiles below the cached length are
                                       // read AHEAD of the dependency wait (only Q, the tree masks and the tiles that hold the
                                       // block's own rows wait for the previous kernel of the stream)
  int ctx_adj;                         // added to seq_len: 0 for verification (the block sits behind the cache length, C10);
                                       // -1 for the final-token path (wf_final.cu: the token is the last cached one, F1)
  float scale_log2;                    // sm_scale * log2(e)
  float4* ws_o;                        // [2 * CTAs][D/8][128 threads] float4: unnormalised O in fragment order
  float4* ws_ml;                       // [2 * CTAs][128 threads] (m, l) of the thread's two rows (m in log2 units)
  int* tiles_hint;                     // mapped host memory: total tiles of this launch (read by the host before a later launch)
  unsigned int* counters;              // [B * Hkv] arrived | published << 16, self-resetting
  int* status;                         // sticky device status word
};

// TREE: the query tile has 128 rows (UMMA M = 128): two 64-row sub-blocks of a draft tree stacked on the TMEM lanes, rows
// of sub-block A on lanes 32w..32w+15 and of sub-block B on lanes 32w+16..32w+31 of every warp quadrant w, so that softmax
// group 0 works on A and group 1 on B of the SAME K/V tile with the chain kernel's fragment code (M = 64 puts its rows on
// lanes 32w..32w+15 as well).  S and O are double buffered over the tiles; P(t) is written with tcgen05.st over the head of
// the S buffer it was computed from (bf16, two keys per 32-bit column) and is the A operand of the PV product FROM TMEM.
template <int D, bool TREE>
struct AttnCfg {
  static constexpr int NH = D / 64;                         // 64-element (128-byte) column halves of a K/V row
  static constexpr int Q_ROWS = TREE ? 128 : AT_ROWS;
  static constexpr int Q_HALF = Q_ROWS * 128;               // rows x 128 B: one 64-column half of the Q (or P) tile
  static constexpr int Q_BYTES = NH * Q_HALF;
  static constexpr int P_BYTES = 2 * Q_HALF;                // 2 key halves x rows x 128 B
  static constexpr int KV_HALF = AT_BN * 128;               // one column half of a K (or V) tile: 16 KB
  static constexpr int K_BYTES = NH * KV_HALF;               // one K (or V) tile
  static constexpr int STAGES_K = D == 128 ? 3 : 4;                       // K ring (TREE: P lives in TMEM, its 32 KB went to a third K stage)
  static constexpr int STAGES_V = D == 128 ? 2 : 4;                       // V ring
  // smem map, chain: P0 | Q | P1 | K ring | V ring (Q + P1 double as the group-merge buffer); tree: Q | K ring | V ring
  static constexpr int SMEM = Q_BYTES + (TREE ? 0 : 2) * P_BYTES + (STAGES_K + STAGES_V) * K_BYTES;
  static constexpr uint32_t TM_S = 0, TM_O = 2 * AT_BN;     // TMEM columns: S0, S1, then O0, O1
};

struct Segment {
  int b, g, t_lo, t_hi, nt;            // tiles [t_lo, t_hi) of the pair's nt tiles; b = sequence (block table row)
  int pb;                              // table index of the pair (TREE: the sub-block; else b): merge counter
  int r0, q_b, ctx, k0, k1, n_tiles;   // r0 / q_b: first query row and rows/group of this tile (TREE: of the sub-block)
  int partial, slot;                   // partial: the pair is shared with other CTAs; slot = 2c + (0 head | 1 tail)
  int flat0;                           // weighted position of the pair (its tile t sits at flat0 + AT_SEG_COST + t)
};

// shared state of one CTA (static smem).  TREE: the table is indexed by SUB-BLOCK (a sequence's tree of up to 64
// nodes is cut into sub-blocks of 64 / group nodes = one 64-row query tile each), see the kernel prologue.
template <bool TREE>
struct AttnShared {
  uint64_t k_full[AT_MAX_STAGES], k_empty[AT_MAX_STAGES], v_full[AT_MAX_STAGES], v_empty[AT_MAX_STAGES];
  uint64_t s_full[2], s_empty[2], o_empty[2], p_full[2], pv_done[2], q_ready;
  float xm[2][128], xl[2][128];        // group-1 running max / row-sum partials for the group merge
  int pref[AT_MAX_B + 1];              // exclusive prefix over the sequences of (tiles per kv head + AT_SEG_COST)
  int r0[AT_MAX_B + 1];                // q_indptr
  int ctx[AT_MAX_B];                   // seq_len
  int meta[TREE ? AT_MAX_B : 1];       // TREE: nodes in the sub-block | nodes of the tree << 7 | first node << 14 | sequence << 21
  int total_tiles, g_eff, B;
  int cl;                              // cluster mode: CTAs per (b, g) pair (0 = stream-K ranges)
  int cl_b;                            // cluster mode: the sequence of this CTA's pair (its table entry is index 0)
  int n_stk, n_stv;                    // K / V ring depths
  uint64_t k_done;                     // cluster mode: this CTA's last QK^T has retired: its K ring is free to receive
  uint64_t cl_ready;                   // cluster mode: every CTA of the cluster can receive (cl arrivals)
  uint64_t cl_bar;                     // cluster mode: completes when every CTA of the pair has pushed its slice for this CTA's rows
  float2 cl_ml[AT_ROWS + 16];          // cluster mode: received (m, l), [sender][row of this CTA's slice]
  int cl_rb[17];                       // cluster mode: rank o owns rows [cl_rb[o], cl_rb[o + 1]) of the pair's live rows
  int cl_dst[AT_ROWS];                 // cluster mode: row -> owner rank | element offset of the row in `out` << 5
  uint32_t tmem;
  int last;
};


// Walks the range of one CTA over the flattened, WEIGHTED (b, g, tile) list; every role keeps its own walker.
// A pair of nt tiles occupies AT_SEG_COST + nt positions: the first AT_SEG_COST stand for the fixed cost of a
// segment, tile t sits at position AT_SEG_COST + t.  Equal shares of positions are then equal shares of time
// even when some CTAs get many short pairs (cfg5: 16 five-tile pairs in one range cost twice the average
// before).  The per-sequence table lives in shared memory (built once in the prologue), so a walk costs no
// global round trips.
template <bool TREE>
struct SegWalker {
  const AttnShared<TREE>& sh;
  int Hkv, c;
  int lo, hi, x, b;
  bool first = true;
  const Segment* lean = nullptr;                               // cluster mode: this CTA's one segment, held by every thread
  __device__ SegWalker(const AttnShared<TREE>& sh_, int Hkv_, int c_, const Segment* lean_) : sh(sh_), Hkv(Hkv_), c(c_), lean(lean_) {
    if (sh.cl > 0) { lo = hi = x = b = 0; return; }          // cluster mode: next() derives the one segment of this CTA
    const int T = sh.total_tiles, G = sh.g_eff;
    lo = (int)((long long)c * T / G);
    hi = (int)((long long)(c + 1) * T / G);
    x = lo;
    int l = 0, r = sh.B;                                       // largest b with Hkv * pref[b] <= lo
    while (r - l > 1) {
      const int mid = (l + r) >> 1;
      if (Hkv * sh.pref[mid] <= lo) l = mid; else r = mid;
    }
    b = l;
  }
  __device__ bool next(Segment& s) {
    if (sh.cl > 0) {
      // Cluster mode: the one segment of this CTA was derived in the prologue, by every thread for itself from one
      // global round trip (a walk costs 1.2k cycles of integer divisions, measured, on the critical path of a batch-1 launch)
      if (!first || lean->n_tiles <= 0) return false;
      first = false;
      s = *lean;
      return true;
    }
    while (x < hi) {
      while (x >= Hkv * sh.pref[b + 1]) ++b;                   // also skips empty sequences
      const int wlen = sh.pref[b + 1] - sh.pref[b], nt = wlen - seg_cost<TREE>();
      const int base = Hkv * sh.pref[b];
      const int g = (x - base) / wlen;
      const int wbase = base + g * wlen;
      const int t_lo = max(0, x - wbase - seg_cost<TREE>());
      const int t_hi = min(nt, hi - wbase - seg_cost<TREE>());
      x = t_hi >= nt ? wbase + wlen : hi;                      // the pair is finished, or the range is
      if (t_hi <= t_lo) continue;                              // the range ends inside the cost positions
      s.b = b; s.pb = b; s.nt = nt; s.g = g; s.t_lo = t_lo; s.t_hi = t_hi;
      s.flat0 = wbase;
      s.r0 = sh.r0[b];
      s.ctx = sh.ctx[b];
      int q_tot;
      if constexpr (TREE) {
        const int meta = sh.meta[b];
        s.q_b = meta & 127;
        q_tot = (meta >> 7) & 127;
        s.b = meta >> 21;
      } else {
        s.q_b = sh.r0[b + 1] - s.r0;
        q_tot = s.q_b;
      }
      s.k0 = t_lo * AT_BN;
      s.k1 = min(s.ctx + q_tot, t_hi * AT_BN);
      s.n_tiles = t_hi - t_lo;
      s.partial = !(t_lo == 0 && t_hi == nt);
      s.slot = 2 * c + (first ? 0 : 1);
      first = false;
      return true;
    }
    return false;
  }
};

__device__ __forceinline__ int cta_of_tile(int x, int T, int G) {      // largest c with c*T/G <= x
  int c = (int)(((long long)x * G) / T);
  while ((int)((long long)(c + 1) * T / G) <= x) ++c;
  while ((int)((long long)c * T / G) > x) --c;
  return c;
}

// ================= warps 8 (K) and 10 (V): TMA producers =================
// K and V have separate rings so that a K tile is released as soon as its QK^T retires: more bytes in flight.
template <int D, bool TREE>
__device__ __forceinline__ void attn_loader(const AttnParams& p, AttnShared<TREE>& sh, uint8_t* ring, uint8_t* k_ring, int which, int lane,
                                            const Segment* lean) {
  using C = AttnCfg<D, TREE>;
  const KvView& kv = p.kv;
  uint64_t* full = which ? sh.v_full : sh.k_full;
  uint64_t* empty = which ? sh.v_empty : sh.k_empty;
  SegWalker<TREE> walk(sh, p.kv.n_kv_heads, blockIdx.x, lean);
  Segment sg;
  uint32_t gt = 0;
  constexpr int PP = AT_BN / 16;                              // pages per tile
  const void* tmap = kv.tmaps + which;
  const uint32_t ring_s = smem_u32(ring);
  // Early mode: tiles that lie wholly below the cached length (rows and block-table entries of earlier rounds) are fetched
  // ahead of the dependency wait; the wait comes before the first page id of a tile that reaches the block's own rows
  // (page ids are fetched one tile ahead, hence the look-ahead of one tile).
  bool waited = !p.early;
  while (walk.next(sg)) {
    if (!waited && sg.k0 + AT_BN > sg.ctx) { wf_pdl_wait(); waited = true; }
    const int32_t* bt = kv.block_table + (size_t)sg.b * kv.max_pages_per_seq + (sg.k0 >> 4);
    const int pages_seg = (sg.k1 - sg.k0 + 15) >> 4;           // pages of this segment, tile t takes [8t, 8t+8)
    // The page ids of tile t+1 are fetched while tile t is issued: the block-table latency is off the ring's
    // critical path.  Lane q holds page q of the tile.  (L2 loads: in early mode a line fetched ahead of the wait may
    // hold entries the previous kernel writes later.)
    int page_next = lane < min(PP, pages_seg) ? __ldcg(bt + lane) : 0;
    for (int t = 0; t < sg.n_tiles; ++t, ++gt) {
      const int n_st = which ? sh.n_stv : sh.n_stk;
      const int st = gt % n_st;
      const int npages = min(PP, pages_seg - t * PP);
      const int row = (((p.layer * kv.num_pages + page_next) * kv.n_kv_heads) + sg.g) * 16;
      // early mode: when the NEXT tile reaches the block's own rows, its page ids are fetched behind the wait, after this
      // tile (still wholly below the cached length) has been issued
      const bool defer_next = !waited && sg.k0 + (t + 2) * AT_BN > sg.ctx;
      if (!defer_next && (t + 1) * PP + lane < pages_seg && lane < PP) page_next = __ldcg(bt + (t + 1) * PP + lane);
      int rows[PP];
#pragma unroll
      for (int q = 0; q < PP; ++q) rows[q] = __shfl_sync(0xffffffffu, row, q);
      mbar_wait(smem_u32(&empty[st]), ((gt / n_st) & 1) ^ 1);
      // Cluster mode (latency-bound): the very first K tile of the CTA is what the first QK^T waits for, and one thread issues
      // a box about every 70 cycles: the V loader issues the second half of that K tile (same page ids) before its own V tile.
      const bool split_first = !TREE && sh.cl > 0 && gt == 0;
      if (split_first && which == 1 && elect_one()) {
        const uint32_t kbar = smem_u32(&sh.k_full[0]);
        const uint32_t kdst = smem_u32(k_ring);
#pragma unroll
        for (int q = PP / 2; q < PP; ++q)
          if (q < npages) {
#pragma unroll
            for (int h = 0; h < C::NH; ++h) tma_load_2d(kdst + q * 2048 + h * C::KV_HALF, kv.tmaps, h * 64, rows[q], kbar);
          }
      }
      if (elect_one()) {                                       // one lane issues the whole tile: straight-line TMA issue
        const uint32_t bar = smem_u32(&full[st]);
        const uint32_t dst = ring_s + (uint32_t)st * C::K_BYTES;
        mbar_arrive_expect_tx(bar, (uint32_t)npages * 16 * D * 2);
        const int q_end = (split_first && which == 0) ? PP / 2 : PP;
#pragma unroll
        for (int q = 0; q < PP; ++q)
          if (q < npages && q < q_end) {
#pragma unroll
            for (int h = 0; h < C::NH; ++h) tma_load_2d(dst + q * 2048 + h * C::KV_HALF, tmap, h * 64, rows[q], bar);
          }
      }
      __syncwarp();
      if (defer_next) {
        wf_pdl_wait();
        waited = true;
        if ((t + 1) * PP + lane < pages_seg && lane < PP) page_next = __ldcg(bt + (t + 1) * PP + lane);
      }
    }
  }
}

// ================= warps 9 (S = Q K^T) and 11 (O_t = P V): MMA issuers =================
// Tile g2 (global tile counter) belongs to softmax group g2 & 1, which owns S[g2&1], P[g2&1], O[g2&1].
// The two products have their own issuing warp: a tcgen05.mma is accepted at the pace of the tensor pipe and every
// mbarrier poll costs the issuing thread about a hundred cycles, so ONE warp that polls five barriers per tile
// between its two batches left the pipe idle half of the time whenever the loop was compute-paced (L2-resident
// K/V: tree sub-blocks, small launches).  With two issuers one polls while the other's batch executes.  The whole
// warp runs the loop so that addresses and descriptors stay warp-uniform; one elected lane issues.  Descriptors
// are built once and advanced by constant offsets.  Hazards are carried by the barriers alone: QK^T(g2) needs
// K(g2) and S[g2&1] read out by the softmax of tile g2 - 2 (s_empty); PV(g2) needs V(g2), P(g2) (p_full) and
// O[g2&1] folded (o_empty).  tcgen05.commit covers the MMAs of the committing thread, i.e. exactly its batch.
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank);

template <int D, bool TREE>
__device__ __forceinline__ void attn_mma_qk(const AttnParams& p, AttnShared<TREE>& sh, uint8_t* q_s, uint8_t* k_s,
                                            uint32_t tmem_base, const Segment* lean) {
  using C = AttnCfg<D, TREE>;
  const uint32_t idesc_qk = umma_idesc_kk(C::Q_ROWS, AT_BN);
  const uint64_t dq0 = umma_desc(smem_u32(q_s), 16, 1024);                  // K-major
  const uint64_t dk0 = umma_desc(smem_u32(k_s), 16, 1024);                  // K-major
  SegWalker<TREE> walk(sh, p.kv.n_kv_heads, blockIdx.x, lean);
  Segment sg;
  uint32_t gt = 0, n_seg = 0;
  while (walk.next(sg)) {
    mbar_wait(smem_u32(&sh.q_ready), n_seg & 1);
    ++n_seg;
    for (int t = 0; t < sg.n_tiles; ++t, ++gt) {
      const int n_stk = sh.n_stk;
      const int st = gt % n_stk;
      mbar_wait(smem_u32(&sh.k_full[st]), (gt / n_stk) & 1);
      WF_PROBE_AT(12 + (gt < 3 ? (int)gt : 3), (threadIdx.x & 31) == 0 && gt < 3);
      mbar_wait(smem_u32(&sh.s_empty[gt & 1]), ((gt >> 1) & 1) ^ 1);
      // TREE: P(gt - 2) lives in the S buffer this product overwrites (tcgen05.st by the softmax warps, A operand of PV from
      // TMEM): the PV of tile gt - 2 must have retired (the two issuers' MMAs are not ordered with each other)
      if constexpr (TREE) { if (gt >= 2) mbar_wait(smem_u32(&sh.pv_done[gt & 1]), ((gt - 2) >> 1) & 1); }
      tc_fence_after();
      if (elect_one()) {
        const uint64_t dk = dk0 + (uint64_t)((st * C::K_BYTES) >> 4);
        const uint32_t td = tmem_base + C::TM_S + (gt & 1) * AT_BN;
#pragma unroll
        for (int k16 = 0; k16 < D / 16; ++k16)
          umma_bf16(td, dq0 + (uint64_t)(((k16 >> 2) * C::Q_HALF + (k16 & 3) * 32) >> 4),
                    dk + (uint64_t)(((k16 >> 2) * C::KV_HALF + (k16 & 3) * 32) >> 4), idesc_qk, k16 != 0);
        umma_commit(smem_u32(&sh.s_full[gt & 1]));
        umma_commit(smem_u32(&sh.k_empty[st]));                // the K tile is free once QK^T has retired
      }
      __syncwarp();
    }
  }
  if constexpr (!TREE) {
    if (sh.cl > 1) {
      // Cluster mode: once the last QK^T has retired this CTA's K ring is idle and becomes its receive buffer: tell every
      // CTA of the cluster (they push their slices only when all are ready; in practice long before anybody is done)
      if (gt > 0) {
        if (elect_one()) umma_commit(smem_u32(&sh.k_done));
        __syncwarp();
        mbar_wait(smem_u32(&sh.k_done), 0);
      }
      const int lane = threadIdx.x & 31;
      if (lane < sh.cl)
        asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(mapa_u32(smem_u32(&sh.cl_ready), (uint32_t)lane)) : "memory");
    }
  }
}

template <int D, bool TREE>
__device__ __forceinline__ void attn_mma_pv(const AttnParams& p, AttnShared<TREE>& sh, uint8_t* p0_s, uint8_t* p1_s,
                                            uint8_t* v_s, uint32_t tmem_base, const Segment* lean) {
  using C = AttnCfg<D, TREE>;
  const uint32_t idesc_pv = umma_idesc(C::Q_ROWS, D);
  const uint64_t dp0 = umma_desc(smem_u32(p0_s), 16, 1024);                 // K-major
  const uint64_t dp1 = umma_desc(smem_u32(p1_s), 16, 1024);
  const uint64_t dv0 = umma_desc(smem_u32(v_s), C::KV_HALF, 1024);          // MN-major
  SegWalker<TREE> walk(sh, p.kv.n_kv_heads, blockIdx.x, lean);
  Segment sg;
  uint32_t gt = 0;
  while (walk.next(sg)) {
    for (int t = 0; t < sg.n_tiles; ++t, ++gt) {
      const int st = gt % sh.n_stv, g = gt & 1;
      mbar_wait(smem_u32(&sh.v_full[st]), (gt / sh.n_stv) & 1);
      // one barrier per P buffer (TREE: P shares the S buffer of its tile).  With a single barrier a softmax thread that runs
      // one tile ahead of another would arrive twice in one phase: nothing holds it back between P(t) and P(t+1) any more
      // (two tiles ahead is impossible: S(t+2) needs PV(t), which needs every arrival of P(t)).
      mbar_wait(smem_u32(&sh.p_full[g]), (gt >> 1) & 1);
      mbar_wait(smem_u32(&sh.o_empty[g]), ((gt >> 1) & 1) ^ 1);
      tc_fence_after();
      if (elect_one()) {
        const uint64_t dv = dv0 + (uint64_t)((st * C::K_BYTES) >> 4);
        const uint64_t dp = (!TREE && g) ? dp1 : dp0;
        const uint32_t td = tmem_base + C::TM_O + g * D;
        if constexpr (TREE) {
          // A = P(gt) from TMEM: 128 rows on the lanes, 16 keys = 8 packed columns per step, at the head of S buffer g
          const uint32_t ta = tmem_base + C::TM_S + g * AT_BN;
#pragma unroll
          for (int k16 = 0; k16 < AT_BN / 16; ++k16)
            umma_bf16_ts(td, ta + k16 * 8, dv + (uint64_t)((k16 * 2048) >> 4), idesc_pv, k16 != 0);
        } else {
#pragma unroll
          for (int k16 = 0; k16 < AT_BN / 16; ++k16)
            umma_bf16(td, dp + (uint64_t)(((k16 >> 2) * C::Q_HALF + (k16 & 3) * 32) >> 4), dv + (uint64_t)((k16 * 2048) >> 4),
                      idesc_pv, k16 != 0);
        }
        umma_commit(smem_u32(&sh.pv_done[g]));
        umma_commit(smem_u32(&sh.v_empty[st]));
      }
      __syncwarp();
    }
  }
}

template <int N>
__device__ __forceinline__ void tmem_ld_frag(uint32_t taddr, uint32_t (&v)[N]) {
  static_assert(N == 64 || N == 32, "fragment of 128 or 64 columns");
  if constexpr (N == 64) tmem_ld_16x256b_x16(taddr, v); else tmem_ld_16x256b_x8(taddr, v);
}

// ---- thread-block cluster helpers (cluster mode) ----
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank) {   // my shared address -> the same offset in CTA `rank`
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
// the exit barrier of the cluster shape orders no data (it only keeps every CTA's shared memory alive until all pushes have
// landed, which the receivers have observed through their mbarriers): no release fence
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// bulk copy own shared memory -> a peer CTA's shared memory, completing (bytes) on the PEER's mbarrier
__device__ __forceinline__ void bulk_push_dsmem(uint32_t dst_cluster, uint32_t src_cta, uint32_t bytes, uint32_t bar_cluster) {
  asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst_cluster), "r"(src_cta), "r"(bytes), "r"(bar_cluster) : "memory");
}
// 8-byte store into a peer CTA's shared memory, completing (8 bytes) on the PEER's mbarrier
__device__ __forceinline__ void st_async_f2(uint32_t dst_cluster, float a, float b, uint32_t bar_cluster) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];"
               ::"r"(dst_cluster), "f"(a), "f"(b), "r"(bar_cluster) : "memory");
}

// Cluster mode: how the R live rows of a pair are dealt to the cl CTAs of its cluster (rank o owns rows [a_o, b_o)).
__device__ __forceinline__ int cl_row_begin(int o, int R, int cl) { return o * R / cl; }
__device__ __forceinline__ int cl_row_owner(int r, int R, int cl) { return ((r + 1) * cl - 1) / R; }   // largest o with a_o <= r

// Cluster mode, sender side (lane o of one warp serves owner o): the partial lies in this CTA's shared memory as
// [64 rows][D fp32], 16-byte chunks XOR-swizzled with (row & 7); every owner gets its rows with ONE bulk copy through
// distributed shared memory, into slot `rank` of its receive buffer, completing on ITS mbarrier.  Nothing crosses global
// memory and nobody waits for anybody here.  (Measured alternatives: one thread walking the owners, 240 cycles per owner;
// every thread storing its fragment straight into the owners' buffers with st.async, 4.0k cycles against 2.5k for this.)
template <int D>
__device__ __forceinline__ void attn_cluster_push(const AttnShared<false>& sh, uint8_t* part_s, uint8_t* recv_s, int lane) {
  const int cl = sh.cl, rank = (int)blockIdx.x % cl;
  if (lane < cl) {
    const int a = sh.cl_rb[lane], n = sh.cl_rb[lane + 1] - a;
    if (n > 0)
      bulk_push_dsmem(mapa_u32(smem_u32(recv_s) + (uint32_t)(rank * n) * (D * 4), (uint32_t)lane), smem_u32(part_s) + (uint32_t)a * (D * 4),
                      (uint32_t)n * (D * 4), mapa_u32(smem_u32(&sh.cl_bar), (uint32_t)lane));
  }
}
// (m, l) of row r (thread-held) to the owner of the row
__device__ __forceinline__ void attn_cluster_push_ml(const AttnShared<false>& sh, int r, float m, float l) {
  const int rank = (int)blockIdx.x % sh.cl;
  const int o = sh.cl_dst[r] & 31;
  const int a = sh.cl_rb[o], n = sh.cl_rb[o + 1] - a;
  st_async_f2(mapa_u32(smem_u32(&sh.cl_ml[rank * n + (r - a)]), (uint32_t)o), m, l, mapa_u32(smem_u32(&sh.cl_bar), (uint32_t)o));
}

// Cluster mode, receiver side (all 256 softmax threads, after cl_bar completed): fold this CTA's rows out of the cl received
// slices in sender order (the bits do not depend on timing), normalise, store.  Local shared memory only.
template <int D>
__device__ __forceinline__ void attn_cluster_reduce(const AttnParams& p, const AttnShared<false>& sh, const uint8_t* recv_s, int tid256) {
  constexpr int MAXCL = 16;
  const int cl = sh.cl, rank = (int)blockIdx.x % cl;
  const int row_a = sh.cl_rb[rank], n = sh.cl_rb[rank + 1] - row_a;
  for (int idx = tid256; idx < n * (D / 4); idx += 256) {
    const int i = idx / (D / 4), c4 = idx % (D / 4), row = row_a + i;
    const uint8_t* base = recv_s + (size_t)i * (D * 4) + ((c4 ^ (row & 7)) << 4);
    float2 ml[MAXCL];
    float4 ov[MAXCL];
#pragma unroll
    for (int s2 = 0; s2 < MAXCL; ++s2)
      if (s2 < cl) {
        ml[s2] = sh.cl_ml[s2 * n + i];
        ov[s2] = *reinterpret_cast<const float4*>(base + (size_t)s2 * n * (D * 4));
      }
    float m = -INFINITY;
#pragma unroll
    for (int s2 = 0; s2 < MAXCL; ++s2)
      if (s2 < cl) m = fmaxf(m, ml[s2].x);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    float l = 0.f;
#pragma unroll
    for (int s2 = 0; s2 < MAXCL; ++s2)
      if (s2 < cl && ml[s2].y > 0.f) {                         // a CTA without tiles (or without a visible key) sends l = 0
        const float w = fast_exp2(ml[s2].x - m);
        l = fmaf(w, ml[s2].y, l);
        acc.x = fmaf(w, ov[s2].x, acc.x); acc.y = fmaf(w, ov[s2].y, acc.y);
        acc.z = fmaf(w, ov[s2].z, acc.z); acc.w = fmaf(w, ov[s2].w, acc.w);
      }
    const float inv = 1.f / l;                                 // every row sees key 0: l > 0
    __nv_bfloat16* dst = p.out + ((size_t)(unsigned int)sh.cl_dst[row] >> 5) + c4 * 4;
    *reinterpret_cast<uint2*>(dst) = make_uint2(pack_bf16(acc.x * inv, acc.y * inv), pack_bf16(acc.z * inv, acc.w * inv));
  }
}

// ================= warps 0-3 (group 0) and 4-7 (group 1): softmax, O accumulation, output, merges =================
// The two groups ping-pong over the tiles: group g takes the tiles whose global counter has parity g and
// keeps its own running (m, l, O); at the end of a segment group 1 hands its state to group 0 through smem.
template <int D>
__device__ __forceinline__ void attn_softmax(const AttnParams& p, AttnShared<false>& sh, uint8_t* q_s, uint8_t* p0_s, uint8_t* p1_s,
                                             uint8_t* v_s, uint8_t* part_s, uint8_t* recv_s, uint32_t tmem_base, int warp, int lane,
                                             const Segment* lean) {
  using C = AttnCfg<D, false>;
  constexpr int NO = D / 2;                                    // O registers per thread (2 rows x D/4 columns)
  const int Hkv = p.kv.n_kv_heads;
  const int grp = warp >> 2, qw = warp & 3;                    // group, TMEM lane quarter
  const int stid = qw * 32 + lane;                             // 0..127 inside the group
  const int rw = lane >> 2, cq = (lane & 3) * 2;               // row within the 8-row group, first column of the pair
  const int row_lo = qw * 16 + rw;                             // this thread's rows: row_lo and row_lo + 8
  const uint32_t t_lane = tmem_base + ((uint32_t)(qw * 32) << 16);
  uint8_t* p_s = grp ? p1_s : p0_s;
  float* xch = reinterpret_cast<float*>(q_s);                  // [NO][128] group-merge buffer (Q + P1 regions)
  const int T = sh.total_tiles, G = sh.g_eff;
  SegWalker<false> walk(sh, p.kv.n_kv_heads, blockIdx.x, lean);
  Segment sg;
  uint32_t gt0 = 0;                                            // global tile counter at the start of the segment
  bool waited = !p.early;
  if (sh.cl > 1) {
    // cluster mode: the row-dealing tables of the merge, by threads that would otherwise idle through the Q load's
    // integer work: group 1 builds them, everybody reads them behind the named barriers of the group merge
    const int Rt = min(lean->q_b * p.group, AT_ROWS);
    if (grp == 1 && stid <= sh.cl) sh.cl_rb[stid] = cl_row_begin(stid, Rt, sh.cl);
    if (grp == 1 && stid >= 64 && stid - 64 < Rt) {
      const int r = stid - 64, qi = r / p.group, hg = r % p.group;
      const unsigned int off = (unsigned int)(((lean->r0 + qi) * p.n_q_heads + lean->g * p.group + hg) * D);
      sh.cl_dst[r] = (int)((off << 5) | (unsigned int)cl_row_owner(r, Rt, sh.cl));
    }
  }
  WF_PROBE_AT(16, warp == 0 && lane == 0);
  while (walk.next(sg)) {
    WF_PROBE_AT(17, warp == 0 && lane == 0);
    const int R = sg.q_b * p.group;
    bool has_next;                                             // this CTA has another segment after this one
    {
      // The NEXT segment's Q rows go to L2 now: under a saturated HBM a cold Q load took 6k cycles at every
      // segment start.  A token's `group` heads are contiguous: group * D * 2 bytes = D / 64 * group lines of 128 B.
      SegWalker<false> peek = walk;
      Segment nx;
      has_next = peek.next(nx);
      if (has_next) {
        const int lines_per_tok = p.group * D * 2 / 128;
        const int idx = grp * 128 + stid;
        if (idx < nx.q_b * lines_per_tok) {
          const char* a = reinterpret_cast<const char*>(p.q + ((size_t)(nx.r0 + idx / lines_per_tok) * p.n_q_heads + nx.g * p.group) * D) +
                          (idx % lines_per_tok) * 128;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
        }
      }
    }
    // ---- Q tile -> smem (K-major, 128-byte swizzle) by both groups; rows >= R are zero.  Every MMA of the
    //      previous segment has retired (both groups waited for their last pv_done). ----
    if (!waited) {                                             // early mode: Q is what the previous kernel produces
      wf_pdl_wait();
      if (grp == 0 && stid == 0) wf_pdl_trigger();
      waited = true;
      WF_PROBE_AT(15, warp == 0 && lane == 0);
    }
    {
      // all loads first, then the stores: one round trip instead of one per chunk
      constexpr int NQ = AT_ROWS * (D / 8) / 256;
      uint4 qv[NQ];
#pragma unroll
      for (int u = 0; u < NQ; ++u) {
        const int c = grp * 128 + stid + u * 256;
        const int rr = c / (D / 8), chn = c % (D / 8);
        qv[u] = make_uint4(0, 0, 0, 0);
        if (rr < R) {
          const int i2 = rr / p.group, h2 = rr % p.group;
          qv[u] = __ldg(reinterpret_cast<const uint4*>(p.q + ((size_t)(sg.r0 + i2) * p.n_q_heads + sg.g * p.group + h2) * D) + chn);
        }
      }
      WF_PROBE_AT(18, warp == 0 && lane == 0);
#pragma unroll
      for (int u = 0; u < NQ; ++u) {
        const int c = grp * 128 + stid + u * 256;
        const int rr = c / (D / 8), chn = c % (D / 8);
        *reinterpret_cast<uint4*>(q_s + (chn >> 3) * C::Q_HALF + rr * 128 + (((chn & 7) ^ (rr & 7)) << 4)) = qv[u];
      }
      WF_PROBE_AT(19, warp == 0 && lane == 0 && qv[0].x != 0x12345678u);
    }
    fence_proxy_async();
    mbar_arrive(smem_u32(&sh.q_ready));
    WF_PROBE_AT(3, warp == 0 && lane == 0);

    float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f}, alpha_prev[2] = {0.f, 0.f};
    float o[NO];
#pragma unroll
    for (int c = 0; c < NO; ++c) o[c] = 0.f;
    int lim[2];                                                // keys j < lim[h] are visible to row (row_lo + 8h)
    lim[0] = min(sg.k1, sg.ctx + row_lo / p.group + 1);
    lim[1] = min(sg.k1, sg.ctx + (row_lo + 8) / p.group + 1);

    auto fold_o = [&]() {                                      // o = o * alpha_prev + O_tile (this group's buffer)
      uint32_t v[NO];
      tmem_ld_frag<NO>(t_lane + C::TM_O + grp * D, v);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.o_empty[grp]));
#pragma unroll
      for (int c = 0; c < NO; c += 2) {
        const float a = alpha_prev[(c >> 1) & 1];
        const float2 r = ffma2(make_float2(o[c], o[c + 1]), make_float2(a, a), make_float2(__uint_as_float(v[c]), __uint_as_float(v[c + 1])));
        o[c] = r.x; o[c + 1] = r.y;
      }
    };

    bool pending = false;                                      // a PV of this group is in flight and not folded yet
    uint32_t g_prev = 0;
    const int t_first = ((gt0 & 1) == (uint32_t)grp) ? 0 : 1;
    // A warp whose 16 rows are all padding (rows >= R: a gamma = 7 block with 4 query heads per kv head fills 32 of the 64
    // rows) walks the tiles through the barrier protocol alone: it never reads S, its P rows keep whatever the buffer held
    // (a P row only feeds its own O row, which nobody reads) and its (m, l, O) stay (-inf, 0, 0).  A loop of its own,
    // so that the live warps' code is untouched.
    const bool live = qw * 16 < R;
    for (int t = t_first; !live && t < sg.n_tiles; t += 2) {
      const uint32_t g2 = gt0 + t;
      const int tk0 = sg.k0 + t * AT_BN;
      mbar_wait(smem_u32(&sh.s_full[grp]), (g2 >> 1) & 1);
      mbar_arrive(smem_u32(&sh.s_empty[grp]));
      if (tk0 + AT_BN > sg.k1) {                               // its share of the stale V rows of the last tile (see below)
        if (pending) mbar_wait(smem_u32(&sh.pv_done[grp]), (g_prev >> 1) & 1);
        mbar_wait(smem_u32(&sh.v_full[g2 % sh.n_stv]), (g2 / sh.n_stv) & 1);
        const int key = (sg.k1 - tk0) + stid;
        if (key < AT_BN) {
          uint8_t* vrow = v_s + (size_t)(g2 % sh.n_stv) * C::K_BYTES + key * 128;
#pragma unroll
          for (int h = 0; h < C::NH; ++h)
#pragma unroll
            for (int c = 0; c < 8; ++c) *reinterpret_cast<uint4*>(vrow + h * C::KV_HALF + c * 16) = make_uint4(0, 0, 0, 0);
        }
      }
      if (pending) mbar_wait(smem_u32(&sh.pv_done[grp]), (g_prev >> 1) & 1);
      fence_proxy_async();
      mbar_arrive(smem_u32(&sh.p_full[grp]));
      if (pending) mbar_arrive(smem_u32(&sh.o_empty[grp]));
      pending = true;
      g_prev = g2;
    }
    for (int t = t_first; live && t < sg.n_tiles; t += 2) {
      const uint32_t g2 = gt0 + t;
      const int tk0 = sg.k0 + t * AT_BN;
      mbar_wait(smem_u32(&sh.s_full[grp]), (g2 >> 1) & 1);
      const int pti = (t - t_first) >> 1;
      WF_PROBE_AT(20 + 6 * pti, warp == 4 && lane == 0 && pti < 2);
      WF_PROBE_AT(4, warp == 0 && lane == 0 && t == t_first);
      tc_fence_after();
      uint32_t sv[64];
      tmem_ld_16x256b_x16(t_lane + C::TM_S + grp * AT_BN, sv);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.s_empty[grp]));                 // S buffer may be overwritten by QK(g2 + 2)

      if (tk0 + AT_BN > min(sg.ctx + 1, sg.k1)) {              // causal / tail mask
#pragma unroll
        for (int c = 0; c < 64; ++c) {
          const int j = tk0 + (c >> 2) * 8 + cq + (c & 1);
          if (j >= lim[(c >> 1) & 1]) sv[c] = 0xff800000u;     // -inf
        }
      }
      float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
      for (int c = 0; c < 64; ++c) mx[(c >> 1) & 1] = fmaxf(mx[(c >> 1) & 1], __uint_as_float(sv[c]));
      float alpha[2], m_use[2], rs[2] = {0.f, 0.f};
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
        mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
        const float m_new = fmaxf(m_run[h], mx[h] * p.scale_log2);
        m_use[h] = m_new == -INFINITY ? 0.f : m_new;
        alpha[h] = fast_exp2(m_run[h] - m_use[h]);
        m_run[h] = m_new;
      }
      uint32_t pk[32];
#pragma unroll
      float2 rs2[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
      const float2 sc2 = make_float2(p.scale_log2, p.scale_log2);
#pragma unroll
      for (int c = 0; c < 64; c += 2) {
        const int h = (c >> 1) & 1;
        const float2 x = ffma2(make_float2(__uint_as_float(sv[c]), __uint_as_float(sv[c + 1])), sc2, make_float2(-m_use[h], -m_use[h]));
        const float p0 = fast_exp2(x.x), p1 = fast_exp2(x.y);
        rs2[h] = fadd2(rs2[h], make_float2(p0, p1));
        pk[c >> 1] = pack_bf16(p0, p1);
      }
      rs[0] = rs2[0].x + rs2[0].y;
      rs[1] = rs2[1].x + rs2[1].y;
      l_run[0] = l_run[0] * alpha[0] + rs[0];
      l_run[1] = l_run[1] * alpha[1] + rs[1];
      WF_PROBE_AT(21 + 6 * pti, warp == 4 && lane == 0 && pti < 2);

      if (tk0 + AT_BN > sg.k1) {
        // Last tile of the sequence: keys >= k1 hold stale or never-written V bits.  Zero them so that
        // 0 * garbage cannot produce NaN in the PV product (P is exactly 0 there).
        // The parity wait below is only unambiguous once the previous occupant of this V stage is consumed:
        // wait for this group's previous PV first (independent of the order the MMA warp issues in).
        if (pending) mbar_wait(smem_u32(&sh.pv_done[grp]), (g_prev >> 1) & 1);
        mbar_wait(smem_u32(&sh.v_full[g2 % sh.n_stv]), (g2 / sh.n_stv) & 1);
        const int key = (sg.k1 - tk0) + stid;
        if (key < AT_BN) {
          uint8_t* vrow = v_s + (size_t)(g2 % sh.n_stv) * C::K_BYTES + key * 128;
#pragma unroll
          for (int h = 0; h < C::NH; ++h)
#pragma unroll
            for (int c = 0; c < 8; ++c) *reinterpret_cast<uint4*>(vrow + h * C::KV_HALF + c * 16) = make_uint4(0, 0, 0, 0);
        }
      }
      if (pending) mbar_wait(smem_u32(&sh.pv_done[grp]), (g_prev >> 1) & 1);   // own PV retired: P is free, O is ready
      {
        // P -> smem, K-major 128-byte swizzle.  The fragment is four 8x8 matrices per pair of 16-byte chunks (rows 0-7 /
        // 8-15 of the warp's 16, chunks j / j+1): one stmatrix.x4 each instead of four 4-byte stores per thread.
        const int mi = lane >> 3, r8 = lane & 7;
        const uint32_t prow = smem_u32(p_s) + (uint32_t)(qw * 16 + (mi & 1) * 8 + r8) * 128;
#pragma unroll
        for (int j = 0; j < 16; j += 2)
          stmatrix_x4(prow + (j >> 3) * C::Q_HALF + ((((j & 7) + (mi >> 1)) ^ r8) << 4), pk[2 * j], pk[2 * j + 1], pk[2 * j + 2],
                      pk[2 * j + 3]);
      }
      fence_proxy_async();
      mbar_arrive(smem_u32(&sh.p_full[grp]));
      WF_PROBE_AT(22 + 6 * pti, warp == 4 && lane == 0 && pti < 2);
      if (pending) { tc_fence_after(); fold_o(); }
      WF_PROBE_AT(23 + 6 * pti, warp == 4 && lane == 0 && pti < 2);
      alpha_prev[0] = alpha[0];
      alpha_prev[1] = alpha[1];
      pending = true;
      g_prev = g2;
    }
    if (pending && !live) {
      mbar_wait(smem_u32(&sh.pv_done[grp]), (g_prev >> 1) & 1);
      mbar_arrive(smem_u32(&sh.o_empty[grp]));
    } else if (pending) {
      mbar_wait(smem_u32(&sh.pv_done[grp]), (g_prev >> 1) & 1);
      WF_PROBE_AT(24, warp == 4 && lane == 0);
      tc_fence_after();
      fold_o();
      WF_PROBE_AT(25, warp == 4 && lane == 0);
    } else {
      // one-tile segment owned by the other group: wait for its PV so that every MMA reading Q / P has retired
      mbar_wait(smem_u32(&sh.pv_done[grp ^ 1]), (gt0 >> 1) & 1);
    }
    gt0 += sg.n_tiles;
    WF_PROBE_AT(5, warp == 0 && lane == 0);

    // Shared pair: arrive NOW (one packed counter: arrived in the low half, published in the high half); the
    // round trip overlaps the group merge below.  Arriving only decides who merges, it publishes nothing.
    int c_first = 0, n_seg = 1;
    unsigned int arrive_old = 0;
    if (sg.partial && grp == 0 && sh.cl == 0) {
      c_first = cta_of_tile(sg.flat0 + seg_cost<false>(), T, G);
      n_seg = cta_of_tile(sg.flat0 + seg_cost<false>() + sg.nt - 1, T, G) - c_first + 1;
      if (stid == 0) arrive_old = atomicAdd(&p.counters[sg.pb * Hkv + sg.g], 1u);
    }

    // ---- group 1 hands (m, l, O) to group 0 through smem (Q and P1 must be idle: every MMA has to have retired) ----
    if (grp == 1) {
      // The buffer overlays the Q tile.  Group 1's own last PV has retired, but when the segment's LAST tile belongs to
      // group 0 its QK^T may still be waiting for a late K tile, i.e. still to read Q: wait for that S tile first.  (Found in
      // round 2: without this wait about one cfg5-sized launch in a thousand returned NaN for one (sequence, kv head) pair:
      // the late QK^T read fp32 O bits as bf16 Q rows.  The hazard needs a K tile that arrives a whole softmax + PV late.)
      const uint32_t g_last = gt0 - 1;                         // gt0 already counts this segment's tiles
      if ((g_last & 1) != (uint32_t)grp) mbar_wait(smem_u32(&sh.s_full[grp ^ 1]), (g_last >> 1) & 1);
#pragma unroll
      for (int c = 0; c < NO; ++c) xch[c * 128 + stid] = o[c];
      sh.xm[0][stid] = m_run[0]; sh.xm[1][stid] = m_run[1];
      sh.xl[0][stid] = l_run[0]; sh.xl[1][stid] = l_run[1];
      named_bar_sync(4, 256);
      named_bar_sync(5, 256);                                  // group 0 has read the buffer: Q may be rewritten
      continue;
    }
    named_bar_sync(4, 256);
    {
      float e0[2], e1[2];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const float m1 = sh.xm[h][stid], l1 = sh.xl[h][stid];
        const float m = fmaxf(m_run[h], m1);
        const float mu = m == -INFINITY ? 0.f : m;
        e0[h] = fast_exp2(m_run[h] - mu);
        e1[h] = fast_exp2(m1 - mu);
        l_run[h] = l_run[h] * e0[h] + l1 * e1[h];
        m_run[h] = m;
      }
#pragma unroll
      for (int c = 0; c < NO; ++c) o[c] = o[c] * e0[(c >> 1) & 1] + xch[c * 128 + stid] * e1[(c >> 1) & 1];
    }
    named_bar_sync(5, 256);
    WF_PROBE_AT(6, warp == 0 && lane == 0);

    // ---- finish the rows: quad-reduce the row sums, write final rows or the partial ----
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 1);
      l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 2);
    }
    if (sh.cl > 1) {
      // Cluster mode: the partial (m, l, unnormalised O) of this CTA goes to its OWN shared memory (the last K stage is idle: every
      // MMA has retired), then warp 0 pushes every owner its rows (attn_cluster_push).  Group 0 only.
      const int Rc = min(R, AT_ROWS);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int r = row_lo + 8 * h;
        uint8_t* prow = part_s + (size_t)r * (D * 4) + (cq & 3) * 4;
#pragma unroll
        for (int j = 0; j < D / 8; ++j)
          *reinterpret_cast<float2*>(prow + (((2 * j + (cq >> 2)) ^ (r & 7)) << 4)) = make_float2(o[4 * j + 2 * h], o[4 * j + 2 * h + 1]);
      }
      fence_proxy_async();
      named_bar_sync(3, 128);
      // (m, l) go to cl_ml of the owner, which is static shared memory nobody else uses: no readiness needed
#pragma unroll
      for (int h = 0; h < 2; ++h)
        if ((lane & 3) == 0 && row_lo + 8 * h < Rc) attn_cluster_push_ml(sh, row_lo + 8 * h, m_run[h], l_run[h]);
      if (warp == 0) {
        mbar_wait(smem_u32(&sh.cl_ready), 0);                  // every CTA of the cluster can receive (its K ring is idle)
        attn_cluster_push<D>(sh, part_s, recv_s, lane);
      }
      continue;
    }
    auto write_rows = [&]() {                                  // normalise and store this thread's two rows
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int r = row_lo + 8 * h;
        if (r >= R) continue;
        const float inv = 1.f / l_run[h];                      // every row sees key 0: l > 0
        const int qi = r / p.group, hg = r % p.group;
        __nv_bfloat16* dst = p.out + ((size_t)(sg.r0 + qi) * p.n_q_heads + sg.g * p.group + hg) * D + cq;
#pragma unroll
        for (int j = 0; j < D / 8; ++j)
          *reinterpret_cast<uint32_t*>(dst + 8 * j) = pack_bf16(o[4 * j + 2 * h] * inv, o[4 * j + 2 * h + 1] * inv);
      }
    };
    if (!sg.partial) { write_rows(); continue; }

    // ---- the pair is shared with other CTAs (group 0 only from here).  The LAST CTA to arrive keeps its
    //      partial in registers and folds the others' partials into it; every other CTA publishes its
    //      partial in fragment order (thread-major float4: coalesced for writer and reader alike).
    //      In steady state the last arriver is the CTA that holds the pair's head at the end of its range,
    //      and the others published long ago. ----
    unsigned int* cnt = p.counters + sg.pb * Hkv + sg.g;
    if (stid == 0) sh.last = (arrive_old & 0xffffu) == (unsigned int)n_seg - 1 ? 1 + (int)(arrive_old >> 16) : 0;
    named_bar_sync(3, 128);
    const int last = sh.last;                                  // 0: not last; else 1 + partials already published
    if (!last) {
      float4* dst = p.ws_o + (size_t)sg.slot * (NO / 4) * 128 + stid;
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) dst[k * 128] = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
      p.ws_ml[(size_t)sg.slot * 128 + stid] = make_float4(m_run[0], l_run[0], m_run[1], l_run[1]);
      __threadfence();
      named_bar_sync(3, 128);                                  // also: sh.last may be rewritten
      if (stid == 0) atomicAdd(cnt, 0x10000u);
      continue;
    }
    if (last - 1 < n_seg - 1) {                                // rare: somebody arrived but has not published yet
      if (stid == 0) {                                         // it has arrived, so it is running: bounded wait
        for (uint32_t spins = 0; (atomicAdd(cnt, 0u) >> 16) < (unsigned int)n_seg - 1; ++spins)
          if (spins > (1u << 24)) __trap();
      }
      named_bar_sync(3, 128);
    }
    if (stid == 0) *cnt = 0;                                   // self-resetting for the next launch
    __threadfence();
    // the head partial of every CTA is slot 2c; only the first CTA can hold the pair as its tail (slot 2c+1)
    const int first_slot = 2 * c_first + ((int)((long long)c_first * T / G) < sg.flat0 ? 1 : 0);
    const int s_own = (int)blockIdx.x - c_first;
    auto fold = [&](const float4 (&x)[NO / 4], const float4 ml) {    // (m, l, O) <- (m, l, O) (+) one published partial
      float e0[2], e1[2];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const float m1 = h ? ml.z : ml.x, l1 = h ? ml.w : ml.y;
        const float m = fmaxf(m_run[h], m1);
        const float mu = m == -INFINITY ? 0.f : m;
        e0[h] = fast_exp2(m_run[h] - mu);
        e1[h] = fast_exp2(m1 - mu);
        l_run[h] = l_run[h] * e0[h] + l1 * e1[h];
        m_run[h] = m;
      }
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) {
        const float xv[4] = {x[k].x, x[k].y, x[k].z, x[k].w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int c = 4 * k + u;
          o[c] = o[c] * e0[(c >> 1) & 1] + xv[u] * e1[(c >> 1) & 1];
        }
      }
    };
    auto slot_of = [&](int s2) { return s2 == 0 ? first_slot : 2 * (c_first + s2); };
    if (p.deterministic) {
      // Reproducible bits: the last arriver stores its own partial like everybody else (each thread reads back exactly
      // what it wrote), starts from the identity and folds ALL partials of the pair in range order 0, 1, ...: the chain of
      // merges no longer depends on which CTA happened to arrive last.  One more 34 KB round trip through L2.
      float4* own = p.ws_o + (size_t)sg.slot * (NO / 4) * 128 + stid;
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) own[k * 128] = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
      p.ws_ml[(size_t)sg.slot * 128 + stid] = make_float4(m_run[0], l_run[0], m_run[1], l_run[1]);
      m_run[0] = m_run[1] = -INFINITY; l_run[0] = l_run[1] = 0.f;
#pragma unroll
      for (int c = 0; c < NO; ++c) o[c] = 0.f;
      for (int s2 = 0; s2 < n_seg; ++s2) {
        const int slot = slot_of(s2);
        const float4* src = p.ws_o + (size_t)slot * (NO / 4) * 128 + stid;
        float4 x[NO / 4];
#pragma unroll
        for (int k = 0; k < NO / 4; ++k) x[k] = __ldcg(src + k * 128);
        fold(x, __ldcg(&p.ws_ml[(size_t)slot * 128 + stid]));
      }
    } else if (!has_next && n_seg > 2) {
      // Many partials (small launches cut a pair into up to 32 ranges): folding them one load round trip at a time
      // cost 2.2k cycles each.  This is the CTA's last segment, so its whole shared memory is idle: every thread
      // copies ITS OWN fragments of up to `cap` partials with cp.async (all in flight together), waits for its
      // own copies only, and folds them out of shared memory in slot order.
      constexpr int PART_BYTES = NO * 512 + 2048;              // O fragments + (m, l) of one partial
      constexpr int cap = C::SMEM / PART_BYTES;
      const uint32_t base_s = smem_u32(p0_s);
      for (int s0 = 0; s0 < n_seg; s0 += cap) {
        const int s1 = min(n_seg, s0 + cap);
        for (int s2 = s0; s2 < s1; ++s2) {
          if (s2 == s_own) continue;
          const int slot = slot_of(s2);
          const uint32_t dst = base_s + (uint32_t)(s2 - s0) * PART_BYTES + stid * 16;
          const float4* src = p.ws_o + (size_t)slot * (NO / 4) * 128 + stid;
#pragma unroll
          for (int k = 0; k < NO / 4; ++k) cp_async16(dst + k * 2048, src + k * 128);
          cp_async16(dst + NO * 512, p.ws_ml + (size_t)slot * 128 + stid);
        }
        cp_async_commit();
        cp_async_wait<0>();
        for (int s2 = s0; s2 < s1; ++s2) {
          if (s2 == s_own) continue;
          const float4* lp = reinterpret_cast<const float4*>(p0_s + (size_t)(s2 - s0) * PART_BYTES) + stid;
          float4 x[NO / 4];
#pragma unroll
          for (int k = 0; k < NO / 4; ++k) x[k] = lp[k * 128];
          fold(x, lp[(NO / 4) * 128]);
        }
      }
    } else {
      for (int s2 = 0; s2 < n_seg; ++s2) {
        if (s2 == s_own) continue;
        const int slot = slot_of(s2);
        const float4* src = p.ws_o + (size_t)slot * (NO / 4) * 128 + stid;
        float4 x[NO / 4];
#pragma unroll
        for (int k = 0; k < NO / 4; ++k) x[k] = __ldcg(src + k * 128);
        fold(x, __ldcg(&p.ws_ml[(size_t)slot * 128 + stid]));
      }
    }
    write_rows();
  }
  if (sh.cl > 1) {
    const int R = min(lean->q_b * p.group, AT_ROWS);
    if (gt0 == 0) {
      // a CTA without tiles still owes every owner a slice: l = 0 marks it empty (its O bits are never read)
      named_bar_sync(4, 256);                                  // the tables above
      if (grp == 0 && stid < R) attn_cluster_push_ml(sh, stid, -INFINITY, 0.f);
      if (warp == 0) {
        mbar_wait(smem_u32(&sh.cl_ready), 0);
        attn_cluster_push<D>(sh, part_s, recv_s, lane);
      }
    }
    WF_PROBE_AT(7, warp == 0 && lane == 0);
    mbar_wait(smem_u32(&sh.cl_bar), 0);                        // every slice of this CTA's rows has landed
    WF_PROBE_AT(8, warp == 0 && lane == 0);
    cluster_arrive_relaxed();                                  // "what was pushed to me has landed": see the kernel's epilogue
    attn_cluster_reduce<D>(p, sh, recv_s, grp * 128 + stid);
    WF_PROBE_AT(9, warp == 0 && lane == 0);
    cluster_wait();
    WF_PROBE_AT(10, warp == 0 && lane == 0);
  }
}

// ================= TREE: warps 0-3 (sub-block A) and 4-7 (sub-block B) on the same K/V tile =================
// Group g owns the 64 rows of sub-block g of the 128-row tile (TMEM lanes 32w + 16g .. +15 of quadrant w) for EVERY tile
// of the segment: running (m, l, O) per group, no hand-over between the groups; S and O alternate between two TMEM
// buffers from tile to tile, P(t) goes to TMEM over the head of S(t)'s buffer (nothing waits for PV(t-1)).  Fragment code, mask,
// partial publishing and the last-arriver fold are those of the chain kernel; a partial slot is (CTA slot, group).
template <int D>
__device__ __forceinline__ void attn_softmax_tree(const AttnParams& p, AttnShared<true>& sh, uint8_t* q_s, uint8_t* p_s,
                                                  uint8_t* v_s, uint32_t tmem_base, int warp, int lane) {
  using C = AttnCfg<D, true>;
  constexpr int NO = D / 2;                                    // O registers per thread (2 rows x D/4 columns)
  const int Hkv = p.kv.n_kv_heads;
  const int grp = warp >> 2, qw = warp & 3;                    // sub-block, TMEM lane quarter
  const int stid = qw * 32 + lane;                             // 0..127 inside the group
  const int rw = lane >> 2, cq = (lane & 3) * 2;               // row within the 8-row group, first column of the pair
  const int row_lo = qw * 16 + rw;                             // this thread's rows of the sub-block: row_lo and row_lo + 8
  const uint32_t t_lane = tmem_base + ((uint32_t)(qw * 32 + grp * 16) << 16);
  const int npt = AT_ROWS / p.group;                           // nodes per sub-block
  const int T = sh.total_tiles, G = sh.g_eff;
  SegWalker<true> walk(sh, p.kv.n_kv_heads, blockIdx.x, nullptr);
  Segment sg;
  uint32_t gt0 = 0;                                            // global tile counter at the start of the segment
  bool waited = !p.early;
  while (walk.next(sg)) {
    const int n_mine = max(0, min(sg.q_b - grp * npt, npt));   // nodes of this group's sub-block
    const int R = n_mine * p.group;                            // its live rows
    const int node0 = sg.r0 + grp * npt;                       // its first node's row in q / out / tree_mask
    {
      SegWalker<true> peek = walk;                             // next segment's Q rows -> L2 (see the chain kernel)
      Segment nx;
      if (peek.next(nx)) {
        const int lines_per_tok = p.group * D * 2 / 128;
        const int idx = grp * 128 + stid;
        if (idx < nx.q_b * lines_per_tok) {
          const char* a = reinterpret_cast<const char*>(p.q + ((size_t)(nx.r0 + idx / lines_per_tok) * p.n_q_heads + nx.g * p.group) * D) +
                          (idx % lines_per_tok) * 128;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
        }
      }
    }
    // ---- Q tile -> smem: 128 rows (K-major, 128-byte swizzle) by both groups; padding rows are zero.  Every MMA of the
    //      previous segment has retired (both groups waited for the last pv_done). ----
    if (!waited) {                                             // early mode: Q and the masks are the previous kernels' outputs
      wf_pdl_wait();
      if (grp == 0 && stid == 0) wf_pdl_trigger();
      waited = true;
    }
    {
      constexpr int NQ = 128 * (D / 8) / 256;
      uint4 qv[NQ];
#pragma unroll
      for (int u = 0; u < NQ; ++u) {
        const int c = grp * 128 + stid + u * 256;
        const int tr = c / (D / 8), chn = c % (D / 8);         // tile row -> (quadrant, sub-block, row in the 16)
        const int rr = (tr >> 5) * 16 + (tr & 15), sb = (tr >> 4) & 1;
        const int node = sb * npt + rr / p.group, h2 = rr % p.group;
        qv[u] = make_uint4(0, 0, 0, 0);
        if (node < sg.q_b)
          qv[u] = __ldg(reinterpret_cast<const uint4*>(p.q + ((size_t)(sg.r0 + node) * p.n_q_heads + sg.g * p.group + h2) * D) + chn);
      }
#pragma unroll
      for (int u = 0; u < NQ; ++u) {
        const int c = grp * 128 + stid + u * 256;
        const int tr = c / (D / 8), chn = c % (D / 8);
        *reinterpret_cast<uint4*>(q_s + (chn >> 3) * C::Q_HALF + tr * 128 + (((chn & 7) ^ (tr & 7)) << 4)) = qv[u];
      }
    }
    fence_proxy_async();
    mbar_arrive(smem_u32(&sh.q_ready));

    float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f}, alpha_prev[2] = {0.f, 0.f};
    float o[NO];
#pragma unroll
    for (int c = 0; c < NO; ++c) o[c] = 0.f;
    unsigned long long anc[2] = {0ull, 0ull};                  // ancestor masks of this thread's two rows (0: padding row)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int node = (row_lo + 8 * h) / p.group;
      if (node < n_mine) anc[h] = __ldg(p.tree_mask + node0 + node);
    }

    auto fold_o = [&](uint32_t gprev) {                        // o = o * alpha_prev + O_tile of tile gprev
      uint32_t v[NO];
      tmem_ld_frag<NO>(t_lane + C::TM_O + (gprev & 1) * D, v);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.o_empty[gprev & 1]));
#pragma unroll
      for (int c = 0; c < NO; c += 2) {
        const float a = alpha_prev[(c >> 1) & 1];
        const float2 r = ffma2(make_float2(o[c], o[c + 1]), make_float2(a, a), make_float2(__uint_as_float(v[c]), __uint_as_float(v[c + 1])));
        o[c] = r.x; o[c + 1] = r.y;
      }
    };

    for (int t = 0; t < sg.n_tiles; ++t) {
      const uint32_t g2 = gt0 + t;
      const int sb = g2 & 1;
      const int tk0 = sg.k0 + t * AT_BN;
      mbar_wait(smem_u32(&sh.s_full[sb]), (g2 >> 1) & 1);
      tc_fence_after();
      uint32_t sv[64];
      tmem_ld_16x256b_x16(t_lane + C::TM_S + sb * AT_BN, sv);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.s_empty[sb]));                  // S buffer may be overwritten by QK(g2 + 2)

      if (tk0 + AT_BN > sg.ctx) {                              // the tile holds tree keys (or the tail beyond them)
        const int rel0 = tk0 + cq - sg.ctx;
#pragma unroll
        for (int c = 0; c < 64; ++c) {
          const int rel = rel0 + (c >> 2) * 8 + (c & 1);
          const bool vis = rel < 0 || (rel < 64 && ((anc[(c >> 1) & 1] >> (rel & 63)) & 1ull));
          if (!vis) sv[c] = 0xff800000u;                       // -inf
        }
      }
      float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
      for (int c = 0; c < 64; ++c) mx[(c >> 1) & 1] = fmaxf(mx[(c >> 1) & 1], __uint_as_float(sv[c]));
      float alpha[2], m_use[2], rs[2] = {0.f, 0.f};
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
        mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
        const float m_new = fmaxf(m_run[h], mx[h] * p.scale_log2);
        m_use[h] = m_new == -INFINITY ? 0.f : m_new;
        alpha[h] = fast_exp2(m_run[h] - m_use[h]);
        m_run[h] = m_new;
      }
      uint32_t pk[32];
      float2 rs2[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
      const float2 sc2 = make_float2(p.scale_log2, p.scale_log2);
#pragma unroll
      for (int c = 0; c < 64; c += 2) {
        // Both groups run this phase at the same time and the four MUFUs of a sub-partition are its bottleneck (64 ex2
        // per thread and tile): every fourth pair is evaluated on the FMA pipe instead, which balances the two pipes.
        const int h = (c >> 1) & 1;
        const float2 x = ffma2(make_float2(__uint_as_float(sv[c]), __uint_as_float(sv[c + 1])), sc2, make_float2(-m_use[h], -m_use[h]));
        float2 e;
        if ((c & 6) == 0) e = poly_exp2_2(x);
        else e = make_float2(fast_exp2(x.x), fast_exp2(x.y));
        rs2[h] = fadd2(rs2[h], e);
        pk[c >> 1] = pack_bf16(e.x, e.y);
      }
      rs[0] = rs2[0].x + rs2[0].y;
      rs[1] = rs2[1].x + rs2[1].y;
      l_run[0] = l_run[0] * alpha[0] + rs[0];
      l_run[1] = l_run[1] * alpha[1] + rs[1];

      if (tk0 + AT_BN > sg.k1 && grp == 0) {
        // Last tile of the sequence: keys >= k1 hold stale or never-written V bits; zero them so that 0 * garbage cannot
        // produce NaN in the PV product (P is exactly 0 there).  Group 0 does it; PV waits for all 256 P arrivals.
        mbar_wait(smem_u32(&sh.v_full[g2 % sh.n_stv]), (g2 / sh.n_stv) & 1);
        const int key = (sg.k1 - tk0) + stid;
        if (key < AT_BN) {
          uint8_t* vrow = v_s + (size_t)(g2 % sh.n_stv) * C::K_BYTES + key * 128;
#pragma unroll
          for (int h = 0; h < C::NH; ++h)
#pragma unroll
            for (int c = 0; c < 8; ++c) *reinterpret_cast<uint4*>(vrow + h * C::KV_HALF + c * 16) = make_uint4(0, 0, 0, 0);
        }
      }
      // P(t) -> TMEM, over the first 64 columns of the S buffer it was computed from (this warp's 16 lanes; S(t) is in
      // registers): the packed fragment is the 16x128b store layout.  P is double buffered with S, so nothing waits for
      // PV(t-1) here; QK^T(t+2) waits for PV(t) before it overwrites the buffer (attn_mma_qk).
      tmem_st_16x128b_x16(t_lane + C::TM_S + sb * AT_BN, pk);
      tmem_st_wait();
      fence_proxy_async();                                     // the zeroed V rows above are generic-proxy writes the MMA reads
      tc_fence_before();
      mbar_arrive(smem_u32(&sh.p_full[sb]));
      if (t > 0) {                                             // O(t-1): its PV has had the whole softmax of tile t to retire
        mbar_wait(smem_u32(&sh.pv_done[(g2 - 1) & 1]), ((g2 - 1) >> 1) & 1);
        tc_fence_after();
        fold_o(g2 - 1);
      }
      alpha_prev[0] = alpha[0];
      alpha_prev[1] = alpha[1];
    }
    {
      const uint32_t gl = gt0 + sg.n_tiles - 1;
      mbar_wait(smem_u32(&sh.pv_done[gl & 1]), (gl >> 1) & 1);
      tc_fence_after();
      fold_o(gl);
    }
    gt0 += sg.n_tiles;

    // ---- finish the rows: quad-reduce the row sums, write final rows or the partial ----
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 1);
      l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 2);
    }
    auto write_rows = [&]() {                                  // normalise and store this thread's two rows
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int r = row_lo + 8 * h;
        if (r >= R) continue;
        const float inv = 1.f / l_run[h];                      // every live row sees itself: l > 0
        const int qi = r / p.group, hg = r % p.group;
        __nv_bfloat16* dst = p.out + ((size_t)(node0 + qi) * p.n_q_heads + sg.g * p.group + hg) * D + cq;
#pragma unroll
        for (int j = 0; j < D / 8; ++j)
          *reinterpret_cast<uint32_t*>(dst + 8 * j) = pack_bf16(o[4 * j + 2 * h] * inv, o[4 * j + 2 * h + 1] * inv);
      }
    };
    if (!sg.partial) { write_rows(); continue; }

    // ---- the pair is shared with other CTAs: last-arriver fold as in the chain kernel, both groups in step ----
    unsigned int* cnt = p.counters + sg.pb * Hkv + sg.g;
    const int c_first = cta_of_tile(sg.flat0 + seg_cost<true>(), T, G);
    const int n_seg = cta_of_tile(sg.flat0 + seg_cost<true>() + sg.nt - 1, T, G) - c_first + 1;
    if (grp == 0 && stid == 0) {
      const unsigned int arrive_old = atomicAdd(cnt, 1u);
      sh.last = (arrive_old & 0xffffu) == (unsigned int)n_seg - 1 ? 1 + (int)(arrive_old >> 16) : 0;
    }
    named_bar_sync(3, 256);
    const int last = sh.last;                                  // 0: not last; else 1 + partials already published
    if (!last) {
      float4* dst = p.ws_o + (size_t)(sg.slot * 2 + grp) * (NO / 4) * 128 + stid;
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) dst[k * 128] = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
      p.ws_ml[(size_t)(sg.slot * 2 + grp) * 128 + stid] = make_float4(m_run[0], l_run[0], m_run[1], l_run[1]);
      __threadfence();
      named_bar_sync(3, 256);                                  // also: sh.last may be rewritten
      if (grp == 0 && stid == 0) atomicAdd(cnt, 0x10000u);
      continue;
    }
    if (last - 1 < n_seg - 1) {                                // rare: somebody arrived but has not published yet
      if (grp == 0 && stid == 0) {
        for (uint32_t spins = 0; (atomicAdd(cnt, 0u) >> 16) < (unsigned int)n_seg - 1; ++spins)
          if (spins > (1u << 24)) __trap();
      }
    }
    named_bar_sync(3, 256);                                    // also: sh.last may be rewritten
    if (grp == 0 && stid == 0) *cnt = 0;                       // self-resetting for the next launch
    __threadfence();
    const int first_slot = 2 * c_first + ((int)((long long)c_first * T / G) < sg.flat0 ? 1 : 0);
    int s_own = (int)blockIdx.x - c_first;
    if (p.deterministic) {                                     // as in the chain kernel: identity, then every partial in range order
      float4* own = p.ws_o + (size_t)(sg.slot * 2 + grp) * (NO / 4) * 128 + stid;
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) own[k * 128] = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
      p.ws_ml[(size_t)(sg.slot * 2 + grp) * 128 + stid] = make_float4(m_run[0], l_run[0], m_run[1], l_run[1]);
      m_run[0] = m_run[1] = -INFINITY; l_run[0] = l_run[1] = 0.f;
#pragma unroll
      for (int c = 0; c < NO; ++c) o[c] = 0.f;
      s_own = -1;
    }
    for (int s2 = 0; s2 < n_seg; ++s2) {
      if (s2 == s_own) continue;
      const int slot = (s2 == 0 ? first_slot : 2 * (c_first + s2)) * 2 + grp;
      const float4* src = p.ws_o + (size_t)slot * (NO / 4) * 128 + stid;
      float4 x[NO / 4];
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) x[k] = __ldcg(src + k * 128);
      const float4 ml = __ldcg(&p.ws_ml[(size_t)slot * 128 + stid]);
      float e0[2], e1[2];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const float m1 = h ? ml.z : ml.x, l1 = h ? ml.w : ml.y;
        const float m = fmaxf(m_run[h], m1);
        const float mu = m == -INFINITY ? 0.f : m;
        e0[h] = fast_exp2(m_run[h] - mu);
        e1[h] = fast_exp2(m1 - mu);
        l_run[h] = l_run[h] * e0[h] + l1 * e1[h];
        m_run[h] = m;
      }
#pragma unroll
      for (int k = 0; k < NO / 4; ++k) {
        const float xv[4] = {x[k].x, x[k].y, x[k].z, x[k].w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int c = 4 * k + u;
          o[c] = o[c] * e0[(c >> 1) & 1] + xv[u] * e1[(c >> 1) & 1];
        }
      }
    }
    write_rows();
  }
}

template <int D, bool TREE>
__global__ void __launch_bounds__(AT_THREADS, 1) wf_verify_attn_kernel(const AttnParams p) {
  using C = AttnCfg<D, TREE>;
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) AttnShared<TREE> sh;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint8_t* p0_s = smem;                                        // smem map: P0 | Q | P1 | K ring | V ring
  uint8_t* q_s = p0_s + (TREE ? 0 : C::P_BYTES);               // TREE: no P buffer in shared memory (P goes to TMEM)
  uint8_t* p1_s = q_s + C::Q_BYTES;
  uint8_t* k_s = p1_s + (TREE ? 0 : C::P_BYTES);             // TREE: no P buffers
  uint8_t* v_s = k_s + C::STAGES_K * C::K_BYTES;

  // barrier init and TMEM allocation touch no global memory: they run before the dependency wait and overlap the
  // tail of the previous kernel of the stream (programmatic dependent launch)
  WF_PROBE_AT(0, tid == 0);
  if (tid == 0) {
    for (int i = 0; i < AT_MAX_STAGES; ++i) {
      mbar_init(smem_u32(&sh.k_full[i]), 1); mbar_init(smem_u32(&sh.k_empty[i]), 1);
      mbar_init(smem_u32(&sh.v_full[i]), 1); mbar_init(smem_u32(&sh.v_empty[i]), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&sh.s_full[i]), 1);
      mbar_init(smem_u32(&sh.s_empty[i]), TREE ? 256 : 128);   // TREE: both groups read every S, O and write every P
      mbar_init(smem_u32(&sh.o_empty[i]), TREE ? 256 : 128);
      mbar_init(smem_u32(&sh.p_full[i]), TREE ? 256 : 128);
      mbar_init(smem_u32(&sh.pv_done[i]), 1);
    }
    mbar_init(smem_u32(&sh.q_ready), 256);
    if constexpr (!TREE) {
      mbar_init(smem_u32(&sh.cl_bar), 1);
      mbar_init(smem_u32(&sh.k_done), 1);
      mbar_init(smem_u32(&sh.cl_ready), p.cl > 0 ? p.cl : 1);
    }
    sh.n_stk = C::STAGES_K;
    sh.n_stv = C::STAGES_V;
    if (!TREE && p.cl > 0) {                                   // cluster mode: what does not depend on device memory
      sh.cl = p.cl; sh.B = 1; sh.g_eff = (int)gridDim.x;
      sh.cl_b = ((int)blockIdx.x / p.cl) / p.kv.n_kv_heads;
    }
    fence_barrier_init();
  }
  if (warp == 9) tmem_alloc(smem_u32(&sh.tmem), 512);
  if constexpr (!TREE) {
    // cluster mode: peers push into this CTA's shared memory and arrive on its mbarrier: nobody may do so before the
    // barrier exists.  This cluster barrier sits ahead of the dependency wait: it overlaps the previous kernel's tail.
    if (p.cl > 0) { cluster_arrive(); cluster_wait(); }
  }
  if (tid == 32 * 8 || tid == 32 * 10)                         // the K / V tensor maps are constants: fetch them ahead of the wait
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(p.kv.tmaps + (tid == 32 * 10 ? 1 : 0))) : "memory");
  // The successor may be scheduled once this launch has passed ITS dependency wait (wf_internal.cuh).  Early mode: the roles
  // wait where they first need the previous kernel's output (loaders: the tiles with the block's own rows; softmax warps: Q).
  if (!p.early) { wf_pdl_wait(); wf_pdl_trigger(); }
  WF_PROBE_AT(1, tid == 0);
  // Cluster mode: a CTA serves ONE (b, g) pair.  Every thread loads that sequence's three lengths itself (one global round
  // trip, the same for all) and derives the CTA's one segment in registers: no table, no barrier behind the dependency wait
  // (the full table costs two barriers and a scan, 2.4k cycles; thread 0 + one barrier + a copy of the segment still cost
  // 1.1k + 0.6k before a loader could fetch its first page id: measured, on the critical path of a batch-1 launch).  The
  // cluster barrier ahead of the wait has already made the barriers, the TMEM address and the mode visible to everybody.
  const bool lean = !TREE && p.cl > 0;
  Segment lean_sg;
  lean_sg.n_tiles = 0;
  int lean_nt = 0;
  if (lean) {
    const int pair = (int)blockIdx.x / p.cl, rank = (int)blockIdx.x % p.cl, b = pair / p.kv.n_kv_heads;
    const int r0 = p.q_indptr[b], r1 = p.q_indptr[b + 1], ctx = p.kv.seq_len[b] + p.ctx_adj;
    const int nt = r1 > r0 ? (ctx + (r1 - r0) + AT_BN - 1) / AT_BN : 0;
    lean_nt = nt;
    // cluster `pair` = (b, g) over ALL sequences of the call (an empty one idles its cluster); CTA rank r of the cluster owns
    // tiles [r * nt / cl, (r + 1) * nt / cl) of the pair: pair-aligned, equal shares, one segment
    lean_sg.b = b; lean_sg.pb = 0; lean_sg.nt = nt; lean_sg.g = pair % p.kv.n_kv_heads;
    // The pair's LAST tile holds the block's own rows: it is never fetched ahead of the dependency wait, it is ragged (stale V
    // rows to clear, causal mask) and the rank that owns it was the cluster's straggler (profiles/r2_final.md: its push landed
    // 2.5k cycles after everybody else's).  It counts as two tiles in the split: the ranks share nt + 1 units.
    lean_sg.t_lo = min(rank * (nt + 1) / p.cl, nt); lean_sg.t_hi = min((rank + 1) * (nt + 1) / p.cl, nt);
    lean_sg.flat0 = 0; lean_sg.r0 = r0; lean_sg.ctx = ctx; lean_sg.q_b = r1 - r0;
    lean_sg.k0 = lean_sg.t_lo * AT_BN; lean_sg.k1 = min(ctx + lean_sg.q_b, lean_sg.t_hi * AT_BN);
    lean_sg.n_tiles = lean_sg.t_hi - lean_sg.t_lo; lean_sg.partial = p.cl > 1; lean_sg.slot = 0;   // one CTA per pair: no merge at all
    if (tid == 0) {
      if (rank == 0 && lean_sg.g == 0 && (r1 - r0) * p.group > AT_ROWS) wf_raise(p.status, (int)WF_ERR_INVALID_ARG);
      // what this CTA will receive: from each of the cl CTAs, its rows [row_a, row_b) of (m, l) and of O
      const int R = min((r1 - r0) * p.group, AT_ROWS);
      const int n_mine = cl_row_begin(rank + 1, R, p.cl) - cl_row_begin(rank, R, p.cl);
      if (nt > 0 && p.cl > 1) mbar_arrive_expect_tx(smem_u32(&sh.cl_bar), (uint32_t)(p.cl * n_mine * (D * 4 + 8)));
    }
  } else {
    // per-sequence table (tiles per kv head, q_indptr, context) from the device-resident lengths, identical in
    // every CTA; then total tiles and the longest pair
    // TREE: the per-sequence values go to the (still idle) dynamic shared memory first; warp 0 then expands them
    // into the sub-block table below.
    int* t_r0 = reinterpret_cast<int*>(smem);
    int* t_ctx = t_r0 + AT_MAX_B;
    int* t_q = t_ctx + AT_MAX_B;
    for (int b = tid; b < p.B; b += AT_THREADS) {
      const int r0 = p.q_indptr[b], r1 = p.q_indptr[b + 1], ctx = p.kv.seq_len[b] + p.ctx_adj;
      // the host bound max_q_len / max_nodes is a promise: a longer block has its rows beyond the query tile dropped
      if (blockIdx.x == 0 && (TREE ? r1 - r0 > 64 : (r1 - r0) * p.group > AT_ROWS)) wf_raise(p.status, (int)WF_ERR_INVALID_ARG);
      if constexpr (TREE) {
        t_r0[b] = r0;
        t_ctx[b] = ctx;
        t_q[b] = min(r1 - r0, 64);
      } else {
        sh.r0[b] = r0;
        sh.ctx[b] = ctx;
        sh.pref[b + 1] = r1 > r0 ? (ctx + (r1 - r0) + AT_BN - 1) / AT_BN + seg_cost<false>() : 0;
        if (b == p.B - 1) sh.r0[p.B] = r1;
      }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (warp == 0) {                                             // in-place scan of the tile counts, 32 sequences per step
      int n_tab = p.B;                                           // table entries
      if constexpr (TREE) {
        // Block s of sequence b = nodes [s * npt, (s+1) * npt), npt = 2 * 64 / group nodes = one 128-row query tile
        // (two sub-blocks).  Each block is a pair of its own that streams the sequence's whole KV; the table lists them
        // LEVEL-MAJOR (all first blocks, then all second ones, ...): with equal trees the level copies of a (b, g) pair
        // sit T / levels positions apart, i.e. in CTAs c, c + G / levels, ... at the same offset of their ranges,
        // which stream the same K/V tiles at the same time: HBM serves one of them, L2 the rest.
        const int npt = 2 * (AT_ROWS / p.group);                // nodes per 128-row tile (two sub-blocks)
        int cursor = 0;
        for (int s0 = 0; s0 < 64; s0 += npt) {
          const int before = cursor;
          for (int base = 0; base < p.B; base += 32) {
            const int b = base + lane;
            const int q = b < p.B ? t_q[b] : 0;
            const bool on = q > s0;
            const unsigned int bal = __ballot_sync(0xffffffffu, on);
            const int idx = cursor + __popc(bal & ((1u << lane) - 1u));
            if (on && idx < AT_MAX_B) {
              const int ctx = t_ctx[b];
              sh.r0[idx] = t_r0[b] + s0;
              sh.ctx[idx] = ctx;
              sh.meta[idx] = min(npt, q - s0) | (q << 7) | (s0 << 14) | (b << 21);
              sh.pref[idx + 1] = (ctx + q + AT_BN - 1) / AT_BN + seg_cost<true>();
            }
            cursor += __popc(bal);
          }
          if (cursor == before) break;                           // no tree is this large
        }
        n_tab = min(cursor, AT_MAX_B);
        __syncwarp();
      }
      int run = 0, lg = 0, live = 0;
      for (int base = 0; base < n_tab; base += 32) {
        const int n = base + lane < n_tab ? sh.pref[base + lane + 1] : 0;
        lg = max(lg, n);
        live += n > 0;
        int v = n;
  #pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const int y = __shfl_up_sync(0xffffffffu, v, d);
          if (lane >= d) v += y;
        }
        if (base + lane < n_tab) sh.pref[base + lane + 1] = run + v;
        run += __shfl_sync(0xffffffffu, v, 31);
      }
  #pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        lg = max(lg, __shfl_xor_sync(0xffffffffu, lg, d));
        live += __shfl_xor_sync(0xffffffffu, live, d);
      }
      if (lane == 0) {
        sh.pref[0] = 0;
        const int total = run * p.kv.n_kv_heads;
        // ranges of at least ceil(longest / 30) tiles keep the partials of one pair <= AT_MAX_SEG
        const int min_range = max(1, (lg + AT_MAX_SEG - 3) / (AT_MAX_SEG - 2));
        sh.total_tiles = total;
        // Small launches (under 24 tiles per SM) are latency-bound: every segment costs about 10k cycles of fixed
        // latency, a pair cut into n ranges streams (tiles/n) * 1.3k cycles and its last arriver folds n partials at
        // about 1k cycles each: least at n = sqrt(1.3 * tiles per pair).  G = n * pairs keeps the ranges aligned with
        // the pairs (one segment per CTA) when the contexts are equal.  Large launches use one CTA per SM.
        const int pairs = live * p.kv.n_kv_heads;
        int G = (int)gridDim.x;
        if (pairs > 0 && total < 24 * G) {
          int n = (int)(sqrtf(1.3f * (float)total / (float)pairs) + 0.5f);
          n = max(1, min(n, G / pairs));
          G = min(G, n * pairs);
        }
        sh.g_eff = p.cl > 0 ? (int)gridDim.x : max(1, min(G, total / min_range));
        sh.B = n_tab;
        sh.cl = TREE ? 0 : p.cl;
        if (blockIdx.x == 0 && p.tiles_hint) *p.tiles_hint = total;      // feedback for the host's next choice of launch shape
      }
    }
    __syncthreads();

  }
  const uint32_t tmem_base = sh.tmem;
  const bool run = lean ? lean_nt > 0 : (sh.total_tiles > 0 && (int)blockIdx.x < sh.g_eff);
  const Segment* lp = lean ? &lean_sg : nullptr;
  WF_PROBE_AT(2, tid == 0);
  if (p.early && !run && tid == 0) { wf_pdl_wait(); wf_pdl_trigger(); }   // an idle CTA must not hold back the successor's launch
  if (run) {
    if (warp < 8) {
      asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
      if constexpr (TREE) attn_softmax_tree<D>(p, sh, q_s, p0_s, v_s, tmem_base, warp, lane);
      else {
        // Cluster mode buffers inside the (then idle) K ring: the receive buffer at its start (cl slices of this CTA's rows: at
        // most (64 + cl - 1) rows of D fp32 = 40 KB at D = 128), this CTA's own staged partial in its LAST stage (64 rows of D
        // fp32 = exactly one stage).  They must not overlap: a peer's slice may land before this CTA has staged or pushed its
        // own partial.  (Until the end of round 2 the partial sat in stage 1 and the slices of an owner with 7 rows, 35 KB from
        // 10 senders, reached 3 KB into it: harmless only as long as the last rank was also the last to push, which stopped
        // being true when its ragged tile was weighted as two; the early / waiting bit-identity test caught it, 1 run in 6.)
        static_assert((AT_ROWS + 15) * D * 4 <= (C::STAGES_K - 1) * C::K_BYTES && AT_ROWS * D * 4 <= C::K_BYTES, "cluster buffers");
        attn_softmax<D>(p, sh, q_s, p0_s, p1_s, v_s, k_s + (C::STAGES_K - 1) * C::K_BYTES, k_s, tmem_base, warp, lane, lp);
      }
    } else {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
      if (warp == 8) attn_loader<D, TREE>(p, sh, k_s, k_s, 0, lane, lp);
      else if (warp == 10) attn_loader<D, TREE>(p, sh, v_s, k_s, 1, lane, lp);
      else if (warp == 9) attn_mma_qk<D, TREE>(p, sh, q_s, k_s, tmem_base, lp);
      else if (warp == 11) attn_mma_pv<D, TREE>(p, sh, p0_s, p1_s, v_s, tmem_base, lp);
    }
  }
  if constexpr (!TREE) {
    if (lean && blockIdx.x == 0 && tid == 32 * 8 && p.tiles_hint) {   // off the critical path: the loader warp is done
      int total = 0;
      for (int b = 0; b < p.B; ++b) {
        const int q = p.q_indptr[b + 1] - p.q_indptr[b];
        if (q > 0) total += (p.kv.seq_len[b] + p.ctx_adj + q + AT_BN - 1) / AT_BN;
      }
      *p.tiles_hint = total * p.kv.n_kv_heads;
    }
    // cluster mode: nobody leaves while a copy it pushed may still be reading its shared memory: a CTA arrives once
    // everything pushed TO it has landed (the softmax warps of a running CTA do so inside attn_softmax), and all wait
    if (sh.cl > 1 && !(run && warp < 8)) { cluster_arrive_relaxed(); cluster_wait(); }
  }
  tc_fence_before();
  __syncthreads();
  WF_PROBE_AT(11, tid == 0);
  if (warp == 9) tmem_dealloc(tmem_base, 512);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
namespace {

template <int D, bool TREE>
int launch_attn(wf_ctx* ctx, AttnParams& p, int* h_hint, cudaStream_t st) {
  const size_t smem = AttnCfg<D, TREE>::SMEM;
  WF_CONFIGURE_ONCE(ctx, (TREE ? WF_FUNC_ATTN_TREE_128 : WF_FUNC_ATTN_128) + (D == 64 ? 1 : 0), (wf_verify_attn_kernel<D, TREE>), smem);
  const int grid = ctx->sm_count < AT_MAX_CTAS ? ctx->sm_count : AT_MAX_CTAS;   // one persistent CTA per SM
  p.cl = 0;
  p.tiles_hint = nullptr;
  if (h_hint) WF_CUDA(ctx, cudaHostGetDevicePointer((void**)&p.tiles_hint, h_hint, 0));
  if constexpr (!TREE) {
    // Launch shape.  Few (b, g) pairs (batch 1-2): one thread-block CLUSTER per pair, the pair's tiles split evenly over
    // its CTAs, partials folded through distributed shared memory (no global round trip, fixed order).  The cluster size is
    // the largest that lets every pair's cluster be resident at once (GPC sizes allow 7 clusters of 12-16 CTAs, 11 of 10,
    // 15 of 8-9, 22 of 6, 33 of 4 with one CTA per SM).  Whether a launch is long enough for stream-K over all SMs to win
    // (HBM-paced: >= 24 tiles per SM) depends on the device-resident lengths: the kernel leaves the tile count of each
    // launch in mapped host memory, and the host reads the last value it can see (no synchronisation; either shape
    // is correct for any lengths, the hint only picks the faster one).
    const int pairs = p.B * p.kv.n_kv_heads;
    int* tab = ctx->attn_max_clusters[D == 64 ? 1 : 0];
    if (!tab[0]) {
      tab[0] = 1;
      cudaFuncSetAttribute(wf_verify_attn_kernel<D, TREE>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
      for (int cl = 2; cl <= 16; ++cl) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(cl); cfg.blockDim = dim3(AT_THREADS); cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, wf_verify_attn_kernel<D, TREE>, &cfg) != cudaSuccess) n = 0;
        tab[cl] = n;
      }
      cudaGetLastError();
    }
    int cl = 0;
    // (deterministic mode: the shape may not depend on when the host happens to see the feedback value, or repeated calls
    // would differ in their bits: the hint is ignored)
    const int hint = (h_hint && !ctx->deterministic) ? *(volatile int*)h_hint : -1;
    const bool hbm_paced = hint >= 24 * grid;
    tab[1] = grid;                                             // one CTA per pair needs no cluster
    if (ctx->attn_cluster_override > 0) cl = ctx->attn_cluster_override;
    else if (ctx->attn_cluster_override < 0 && pairs > 0) {
      for (int c2 = 16; c2 >= 1; --c2)
        if (tab[c2] >= pairs) { cl = c2; break; }
      // An HBM-paced launch wants (nearly) every SM streaming: pair-aligned CTAs only if they cover most of the machine.
      // Measured: batch 4, context 32768: 32 clusters of 4 = 128 CTAs stream 5.9-6.2 TB/s against 5.7 for stream-K ranges on
      // 148 (no global merge, no partial traffic); batch 16, context 8192: 128 CTAs, one whole pair each, no merge at all.
      if (hbm_paced && pairs * cl * 5 < grid * 4) cl = 0;
      // a latency-bound launch with one short pair per CTA gains nothing from this shape over stream-K's own small-launch path
      if (!hbm_paced && cl == 1) cl = 0;
    }
    if (cl >= 1 && cl <= 16 && tab[cl] >= pairs) {
      p.cl = cl;
      if (cl == 1) wf_launch(wf_verify_attn_kernel<D, TREE>, dim3(pairs), dim3(AT_THREADS), smem, st, p);
      else wf_launch_cluster(wf_verify_attn_kernel<D, TREE>, dim3(pairs * cl), dim3(AT_THREADS), smem, cl, st, p);
      return wf_check_launch(ctx, cl == 1 ? "wf_verify_attn_kernel<pair per CTA>" : "wf_verify_attn_kernel<cluster>");
    }
  }
  wf_launch(wf_verify_attn_kernel<D, TREE>, dim3(grid), dim3(AT_THREADS), smem, st, p);
  return wf_check_launch(ctx, TREE ? "wf_verify_attn_kernel<tree>" : "wf_verify_attn_kernel");
}

// One thread per tree node walks its parent pointers (staged in shared memory) up to the root and ORs the bits.
// A node whose pointers do not lead to the root through strictly decreasing indices (reading T1) raises
// WF_ERR_INVALID_ARG in the sticky status word and keeps only its own bit.
__global__ void __launch_bounds__(64) wf_tree_masks_kernel(const int32_t* parent, const int32_t* q_indptr,
                                                           unsigned long long* mask, int* status) {
  __shared__ int par[64];
  wf_pdl_wait();
  wf_pdl_trigger();
  const int b = blockIdx.x, i = threadIdx.x;
  const int r0 = q_indptr[b], n = min(q_indptr[b + 1] - r0, 64);
  if (i < n) par[i] = parent[r0 + i];
  __syncthreads();
  if (i >= n) return;
  unsigned long long m = 1ull << i;
  bool bad = i == 0 && par[0] != -1;
  for (int j = i; j > 0;) {
    const int pj = par[j];
    if (pj < 0 || pj >= j) { bad = true; m = 1ull << i; break; }
    j = pj;
    m |= 1ull << j;
  }
  if (bad) atomicCAS(status, 0, (int)WF_ERR_INVALID_ARG);
  mask[r0 + i] = m;
}

// ancestor masks of a CHAIN block (parent[i] = i - 1): row i sees block rows 0..i.  For blocks of more than 64 / group rows,
// which wf_verify_attn runs on the tree kernel's 128-row tiles.
__global__ void __launch_bounds__(64) wf_chain_masks_kernel(const int32_t* q_indptr, unsigned long long* mask) {
  wf_pdl_wait();
  wf_pdl_trigger();
  const int b = blockIdx.x, i = threadIdx.x;
  const int r0 = q_indptr[b], n = min(q_indptr[b + 1] - r0, 64);
  if (i < n) mask[r0 + i] = i == 63 ? ~0ull : (2ull << i) - 1ull;
}

}  // namespace

extern "C" size_t wf_verify_attn_workspace_bytes(const wf_kv_shape* s, int B, int n_q_heads, int max_q_len) {
  if (!s || B <= 0 || n_q_heads <= 0 || s->n_kv_heads <= 0) return 16;
  const size_t items = 4 * (size_t)AT_MAX_CTAS;            // a CTA writes at most a head and a tail partial (tree: per group)
  const size_t r_pad = AT_ROWS;
  const size_t base = items * (r_pad * (size_t)s->head_dim * sizeof(float) + 128 * sizeof(float4));
  // a chain block of more than 64 rows per kv head runs on the tree kernel: its chain masks live behind the partials
  const bool wide = max_q_len > 0 && (long long)max_q_len * (n_q_heads / s->n_kv_heads) > AT_ROWS;
  return base + (wide ? (((size_t)B * (size_t)max_q_len * sizeof(unsigned long long) + 15) & ~(size_t)15) : 0);
}

// shared by wf_verify_attn (ctx_adj = 0) and the final-token path of wf_final.cu (ctx_adj = -1, one query row per
// selected sequence over a drafter's cache)
int wf_attn_launch_chain(wf_ctx* ctx, const wf_paged_kv* kv, int layer, const void* q, const int32_t* q_indptr, int B,
                         int n_q_heads, int max_q_len, float sm_scale, int ctx_adj, void* out, void* workspace,
                         size_t workspace_bytes, void* stream, const char* who) {
  WF_REQUIRE(ctx, kv && q && q_indptr && out && workspace, WF_ERR_INVALID_ARG, "%s: null argument", who);
  WF_REQUIRE(ctx, layer >= 0 && layer < kv->s.n_layers, WF_ERR_INVALID_ARG, "%s: bad layer", who);
  WF_REQUIRE(ctx, B >= 0 && B <= kv->s.max_seqs && B <= AT_MAX_B && B * kv->s.n_kv_heads <= ctx->n_counters,
             WF_ERR_INVALID_ARG, "%s: bad B (max %d)", who, AT_MAX_B);
  WF_REQUIRE(ctx, n_q_heads > 0 && n_q_heads % kv->s.n_kv_heads == 0, WF_ERR_INVALID_ARG,
             "%s: n_q_heads must be a multiple of n_kv_heads", who);
  const int group = n_q_heads / kv->s.n_kv_heads;
  WF_REQUIRE(ctx, max_q_len >= 1 && max_q_len <= 64 && group <= 64, WF_ERR_UNSUPPORTED_SHAPE,
             "%s: max_q_len must be in [1, 64] and the GQA group <= 64", who);
  WF_REQUIRE(ctx, workspace_bytes >= wf_verify_attn_workspace_bytes(&kv->s, B, n_q_heads, max_q_len),
             WF_ERR_INVALID_ARG, "%s: workspace too small", who);
  WF_REQUIRE(ctx, ((uintptr_t)q % 16 == 0) && ((uintptr_t)out % 16 == 0) && ((uintptr_t)workspace % 16 == 0),
             WF_ERR_INVALID_ARG, "%s: q/out/workspace must be 16-byte aligned", who);
  if (B == 0) return WF_OK;
  if (max_q_len * group > AT_ROWS) {
    // More than 64 rows per kv head (e.g. gamma = 15 at a GQA group of 8): the block is a degenerate tree (parent[i] = i - 1)
    // and runs on the tree kernel's 128-row tiles; its masks are written into the tail of the workspace first.
    WF_REQUIRE(ctx, ctx_adj == 0, WF_ERR_UNSUPPORTED_SHAPE, "%s: more than 64 rows per kv head", who);
    const size_t base = wf_verify_attn_workspace_bytes(&kv->s, B, n_q_heads, 1);
    unsigned long long* masks = reinterpret_cast<unsigned long long*>((char*)workspace + base);
    wf_launch(wf_chain_masks_kernel, dim3(B), dim3(64), 0, (cudaStream_t)stream, q_indptr, masks);
    const int rc = wf_check_launch(ctx, "wf_chain_masks_kernel");
    if (rc != WF_OK) return rc;
    return wf_verify_attn_tree(ctx, kv, layer, q, q_indptr, (const uint64_t*)masks, B, n_q_heads, max_q_len, sm_scale, out,
                               workspace, workspace_bytes, stream);
  }
  const int r_pad = AT_ROWS;
  const size_t items = 4 * (size_t)AT_MAX_CTAS;
  AttnParams p;
  p.q = (const __nv_bfloat16*)q;
  p.out = (__nv_bfloat16*)out;
  p.q_indptr = q_indptr;
  p.kv = kv_view(kv);
  p.layer = layer; p.B = B; p.n_q_heads = n_q_heads; p.group = group;
  p.ctx_adj = ctx_adj;
  p.deterministic = ctx->deterministic;
  p.early = ctx->attn_early;
  p.scale_log2 = sm_scale * LOG2E;
  p.ws_o = (float4*)workspace;
  p.ws_ml = (float4*)((char*)workspace + items * r_pad * kv->s.head_dim * sizeof(float));
  p.counters = ctx->d_counters_attn;
  p.status = ctx->d_status;
  cudaStream_t st = (cudaStream_t)stream;
  const int D = kv->s.head_dim;
  p.tree_mask = nullptr;
  if (D == 128) return launch_attn<128, false>(ctx, p, kv->h_tiles_hint, st);
  if (D == 64) return launch_attn<64, false>(ctx, p, kv->h_tiles_hint, st);
  return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "%s: head_dim %d unsupported", who, D);
}

extern "C" int wf_verify_attn(wf_ctx* ctx, const wf_paged_kv* kv, int layer, const void* q,
                              const int32_t* q_indptr, int B, int n_q_heads, int max_q_len, float sm_scale,
                              void* out, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  return wf_attn_launch_chain(ctx, kv, layer, q, q_indptr, B, n_q_heads, max_q_len, sm_scale, 0, out, workspace,
                              workspace_bytes, stream, "wf_verify_attn");
}

extern "C" int wf_tree_masks(wf_ctx* ctx, const int32_t* parent, const int32_t* q_indptr, int B, int max_nodes,
                             uint64_t* tree_mask, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, parent && q_indptr && tree_mask && B >= 0, WF_ERR_INVALID_ARG, "wf_tree_masks: bad argument");
  WF_REQUIRE(ctx, max_nodes >= 1 && max_nodes <= 64, WF_ERR_UNSUPPORTED_SHAPE, "wf_tree_masks: max_nodes must be in [1, 64]");
  if (B == 0) return WF_OK;
  wf_launch(wf_tree_masks_kernel, dim3(B), dim3(64), 0, (cudaStream_t)stream, parent, q_indptr,
            (unsigned long long*)tree_mask, ctx->d_status);
  return wf_check_launch(ctx, "wf_tree_masks_kernel");
}

extern "C" int wf_verify_attn_tree(wf_ctx* ctx, const wf_paged_kv* kv, int layer, const void* q, const int32_t* q_indptr,
                                   const uint64_t* tree_mask, int B, int n_q_heads, int max_nodes, float sm_scale,
                                   void* out, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, kv && q && q_indptr && tree_mask && out && workspace, WF_ERR_INVALID_ARG, "wf_verify_attn_tree: null argument");
  WF_REQUIRE(ctx, layer >= 0 && layer < kv->s.n_layers, WF_ERR_INVALID_ARG, "wf_verify_attn_tree: bad layer");
  WF_REQUIRE(ctx, n_q_heads > 0 && n_q_heads % kv->s.n_kv_heads == 0, WF_ERR_INVALID_ARG,
             "wf_verify_attn_tree: n_q_heads must be a multiple of n_kv_heads");
  const int group = n_q_heads / kv->s.n_kv_heads;
  WF_REQUIRE(ctx, group <= 64 && max_nodes >= 1 && max_nodes <= 64, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_verify_attn_tree: max_nodes must be in [1, 64] and the GQA group <= 64");
  const int npt = 2 * (AT_ROWS / group);                     // nodes per 128-row query tile (two 64-row sub-blocks)
  const int levels = (max_nodes + npt - 1) / npt;            // tiles per tree
  WF_REQUIRE(ctx, B >= 0 && B <= kv->s.max_seqs && (long long)B * levels <= AT_MAX_B &&
                      (long long)B * levels * kv->s.n_kv_heads <= ctx->n_counters,
             WF_ERR_INVALID_ARG, "wf_verify_attn_tree: B * ceil(max_nodes * group / 128) must be <= %d", AT_MAX_B);
  WF_REQUIRE(ctx, workspace_bytes >= wf_verify_attn_workspace_bytes(&kv->s, B, n_q_heads, max_nodes),
             WF_ERR_INVALID_ARG, "wf_verify_attn_tree: workspace too small");
  WF_REQUIRE(ctx, ((uintptr_t)q % 16 == 0) && ((uintptr_t)out % 16 == 0) && ((uintptr_t)workspace % 16 == 0) &&
                      ((uintptr_t)tree_mask % 8 == 0),
             WF_ERR_INVALID_ARG, "wf_verify_attn_tree: q/out/workspace must be 16-byte aligned");
  if (B == 0) return WF_OK;
  const size_t items = 4 * (size_t)AT_MAX_CTAS;
  AttnParams p;
  p.q = (const __nv_bfloat16*)q;
  p.out = (__nv_bfloat16*)out;
  p.q_indptr = q_indptr;
  p.tree_mask = (const unsigned long long*)tree_mask;
  p.kv = kv_view(kv);
  p.layer = layer; p.B = B; p.n_q_heads = n_q_heads; p.group = group;
  p.ctx_adj = 0;
  p.deterministic = ctx->deterministic;
  p.early = ctx->attn_early;
  p.scale_log2 = sm_scale * LOG2E;
  p.ws_o = (float4*)workspace;
  p.ws_ml = (float4*)((char*)workspace + items * AT_ROWS * kv->s.head_dim * sizeof(float));
  p.counters = ctx->d_counters_attn;
  p.status = ctx->d_status;
  cudaStream_t st = (cudaStream_t)stream;
  const int D = kv->s.head_dim;
  if (D == 128) return launch_attn<128, true>(ctx, p, nullptr, st);
  if (D == 64) return launch_attn<64, true>(ctx, p, nullptr, st);
  return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "wf_verify_attn_tree: head_dim %d unsupported", D);
}

extern "C" int wf_ctx_set_attn_cluster(wf_ctx* ctx, int cluster_size) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  WF_REQUIRE(ctx, cluster_size >= -1 && cluster_size <= 16, WF_ERR_INVALID_ARG,
             "wf_ctx_set_attn_cluster: cluster_size must be -1 (automatic), 0 (never) or 1..16");
  ctx->attn_cluster_override = cluster_size;
  return WF_OK;
}

extern "C" int wf_ctx_set_attn_early_kv(wf_ctx* ctx, int on) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  ctx->attn_early = on ? 1 : 0;
  return WF_OK;
}

extern "C" int wf_ctx_set_deterministic(wf_ctx* ctx, int on) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  ctx->deterministic = on ? 1 : 0;
  return WF_OK;
}

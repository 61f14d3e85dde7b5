// Internal definitions shared by the CUDA translation units of libwhiflash (product path only;
// nothing under oracle/ includes or links this).
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "whiflash.h"

struct wf_ctx {
  int device;
  int sm_count;
  int* d_status;               // sticky device status word (0 = ok, else a negative wf_status)
  unsigned int* d_counters;    // self-resetting "blocks done" counters for the accept sweep
  unsigned int* d_counters_attn; // same, per (sequence, kv head), for the split-KV combine
  int n_counters;
  int64_t launches;            // kernels launched through this ctx (host counter)
  unsigned int func_configured; // bit k: kernel k's dynamic-smem opt-in was made on THIS ctx's device (WF_FUNC_*)
  int deterministic;           // wf_ctx_set_deterministic: fixed-order split merges
  int attn_max_clusters[2][17]; // [D == 64][cluster size]: co-resident clusters of the chain attention kernel (0 = not queried)
  int attn_cluster_override;   // test / tuning hook: -1 = automatic, 0 = never, n > 0 = force cluster size n
  int attn_early;              // wf_ctx_set_attn_early_kv
  char err[256];
};

// kernels that need cudaFuncSetAttribute(MaxDynamicSharedMemorySize): the attribute is per device, so the
// bookkeeping is per ctx (a ctx is bound to one device), never per process
enum {
  WF_FUNC_ATTN_128 = 0, WF_FUNC_ATTN_64, WF_FUNC_ATTN_TREE_128, WF_FUNC_ATTN_TREE_64, WF_FUNC_GEMM_128, WF_FUNC_GEMM_64,
  WF_FUNC_NEURAL, WF_FUNC_ACCEPT, WF_FUNC_FINAL_TOKEN /* + EPI 0..3 */, WF_FUNC_FINAL_TOKEN_LAST = WF_FUNC_FINAL_TOKEN + 3
};
#define WF_CONFIGURE_ONCE(ctx, bit, kernel, bytes)                                                          \
  do {                                                                                                      \
    if (!((ctx)->func_configured & (1u << (bit)))) {                                                        \
      WF_CUDA((ctx), cudaFuncSetAttribute((kernel), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes))); \
      (ctx)->func_configured |= 1u << (bit);                                                                \
    }                                                                                                       \
  } while (0)

struct wf_paged_kv {
  wf_ctx* ctx;
  wf_kv_shape s;
  __nv_bfloat16* k_pool;
  __nv_bfloat16* v_pool;
  int32_t* block_table;        // caller-owned [max_seqs][max_pages_per_seq]
  int32_t* seq_len;            // caller-owned [max_seqs]
  int32_t* pages_held;         // library-owned [max_seqs]
  int32_t* free_ring;          // library-owned [num_pages]
  int32_t* ring_state;         // library-owned [2]: head, count
  int32_t* scratch;            // library-owned [2*max_seqs]: need, offset
  CUtensorMap* d_tmaps;        // library-owned [2]: K pool, V pool as [rows][D], box {64, 16}, 128B swizzle
  int* h_tiles_hint;           // library-owned, pinned + mapped: total 128-key tiles of the last attention launch over this
                               // cache (written by the kernel, read without a sync by the host to pick the next launch shape)
};

// Device-side view of a paged KV cache passed by value to kernels.
struct KvView {
  __nv_bfloat16* k_pool;
  __nv_bfloat16* v_pool;
  int32_t* block_table;
  int32_t* seq_len;
  int32_t* pages_held;
  int32_t* free_ring;
  int32_t* ring_state;
  int32_t* scratch;
  const CUtensorMap* tmaps;    // [0] = K pool, [1] = V pool
  int n_layers, n_kv_heads, head_dim, page_size, num_pages, max_seqs, max_pages_per_seq;
};

static inline KvView kv_view(const wf_paged_kv* kv) {
  KvView v;
  v.k_pool = kv->k_pool; v.v_pool = kv->v_pool;
  v.block_table = kv->block_table; v.seq_len = kv->seq_len;
  v.pages_held = kv->pages_held; v.free_ring = kv->free_ring;
  v.ring_state = kv->ring_state; v.scratch = kv->scratch;
  v.tmaps = kv->d_tmaps;
  v.n_layers = kv->s.n_layers; v.n_kv_heads = kv->s.n_kv_heads; v.head_dim = kv->s.head_dim;
  v.page_size = kv->s.page_size; v.num_pages = kv->s.num_pages; v.max_seqs = kv->s.max_seqs;
  v.max_pages_per_seq = kv->s.max_pages_per_seq;
  return v;
}

struct wf_row_entry {
  int32_t pos;                 // absolute position (RoPE)
  int32_t page_slot;           // physical page * 16 + slot in the drafter cache
};
struct wf_full_layer;          // wf_final.cu: the weights and scratch of the final-token path (f3)

struct wf_drafter {
  wf_ctx* ctx;
  wf_drafter_shape s;
  wf_paged_kv* kv;
  const __nv_bfloat16* backlog;
  int32_t* backlog_len;
  uint8_t* d_wpack;            // library-owned pre-swizzled copy of the weights (see wf_pack_w_kernel)
  uint8_t* d_xpack;            // library-owned [hidden/64][row_cap][128 B] scratch (see wf_plan_pack_kernel)
  int n_split;                 // split-K factor of the projection, fixed at creation (a power of two)
  int max_pass;
  float* d_ws_part;            // [tiles][n_split][row_cap][D] fp32 partials (n_split > 1)
  unsigned int* d_split_cnt;   // [tiles][max_pass]
  float2* d_rope;              // [max_pos][D/2]
  wf_row_entry* d_rows;
  int row_cap;
  int32_t* d_m_total;
  int32_t* d_plan;             // [2 * max_seqs]: enq_base, new_blen (planner -> kernel 2)
  wf_full_layer* full;         // NULL until wf_drafter_set_full_layer
};
void wf_full_layer_destroy(wf_full_layer* f);
// wf_attn.cu: the chain attention kernel with seq_len + ctx_adj as the context (see AttnParams::ctx_adj)
int wf_attn_launch_chain(wf_ctx* ctx, const wf_paged_kv* kv, int layer, const void* q, const int32_t* q_indptr, int B,
                         int n_q_heads, int max_q_len, float sm_scale, int ctx_adj, void* out, void* workspace,
                         size_t workspace_bytes, void* stream, const char* who);

int wf_set_error(wf_ctx* ctx, int code, const char* fmt, ...);
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time libcuda dependency)
typedef CUresult (*wf_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                       const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                       CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
wf_encode_tiled_fn wf_get_encode_tiled();
// 2-D bf16 tensor map, row-major [rows][cols], box {box_cols, box_rows}, 128-byte swizzle
int wf_make_tmap_2d(wf_ctx* ctx, CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                    uint32_t box_rows);
int wf_check_launch(wf_ctx* ctx, const char* what);   // cudaGetLastError -> WF_ERR_CUDA; counts the launch

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch.  Every kernel of the library is launched with programmatic stream
// serialisation: it may be scheduled while the previous kernel of the stream is still running.  A
// kernel calls wf_pdl_wait() before its first access to global memory that another kernel may have
// written (blocks until the previous grid has completed and its writes are visible) and
// wf_pdl_trigger() right AFTER it (its successor may then be scheduled).  Order matters: a successor
// that starts only once this kernel has passed its wait knows that everything up to this kernel's
// PREDECESSOR is complete, so it may read, ahead of its own wait, whatever this kernel does not
// write (constants such as weights; in the attention kernel's early mode also the lengths, page ids
// and K/V rows of earlier rounds).  What runs before the wait (barrier init, TMEM allocation,
// prefetches, launch latency) overlaps the predecessor.
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void wf_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void wf_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
// sticky device status: the FIRST error of a poll interval wins (a later one never overwrites it)
__device__ __forceinline__ void wf_raise(int* status, int code) { atomicCAS(status, 0, code); }

// the same, as thread-block clusters of `cluster` CTAs (grid must be a multiple of it)
template <typename... KArgs, typename... Args>
inline cudaError_t wf_launch_cluster(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, int cluster, cudaStream_t st,
                                     Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = (unsigned)cluster; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

template <typename... KArgs, typename... Args>
inline cudaError_t wf_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

#define WF_REQUIRE(ctx, cond, code, ...)                         \
  do {                                                           \
    if (!(cond)) return wf_set_error((ctx), (code), __VA_ARGS__); \
  } while (0)

#define WF_CUDA(ctx, expr)                                                                   \
  do {                                                                                       \
    cudaError_t e__ = (expr);                                                                \
    if (e__ != cudaSuccess)                                                                  \
      return wf_set_error((ctx), WF_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e__));     \
  } while (0)

// ---------------------------------------------------------------------------------------------
// Block-wide page reservation (reading C24), callable from any kernel that runs as ONE block.
// add(b) gives the tokens sequence slot `seq(b)` must additionally hold, b in [0,B).
// Sequences are served in ascending b; each takes consecutive ring entries from the head.
// If the ring cannot serve the whole call (or a sequence would exceed max_pages_per_seq), nothing
// is allocated, *status becomes WF_ERR_OUT_OF_PAGES and false is returned (block-uniform).
// Requires blockDim.x a multiple of 32, <= 1024.
// ---------------------------------------------------------------------------------------------
constexpr int KV_RESERVE_SMEM = 1024;
template <typename AddFn, typename SeqFn>
__device__ inline bool kv_reserve_block(const KvView& kv, int B, AddFn add, SeqFn seq, int* status) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  __shared__ int s_bad;
  // need / offset per sequence: shared memory for the first KV_RESERVE_SMEM sequences (the usual case: no global
  // round trip between the scan and the ring copy), the library's global scratch beyond
  __shared__ int s_need[KV_RESERVE_SMEM], s_off[KV_RESERVE_SMEM];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
  const int head = kv.ring_state[0], count = kv.ring_state[1];     // issued early: off the critical path
  if (tid == 0) { s_carry = 0; s_bad = 0; }
  __syncthreads();
  int* g_need = kv.scratch;
  int* g_off = kv.scratch + kv.max_seqs;
  auto need = [&](int b) -> int& { return b < KV_RESERVE_SMEM ? s_need[b] : g_need[b]; };
  auto off = [&](int b) -> int& { return b < KV_RESERVE_SMEM ? s_off[b] : g_off[b]; };
  for (int base = 0; base < B; base += blockDim.x) {
    const int b = base + tid;
    int n = 0;
    if (b < B) {
      const int s = seq(b);
      const int want = (kv.seq_len[s] + add(b) + kv.page_size - 1) / kv.page_size;
      if (want > kv.max_pages_per_seq) s_bad = 1;
      n = max(0, want - kv.pages_held[s]);
    }
    int x = n;                                   // inclusive warp scan
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      int y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) s_warp[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int w = lane < nw ? s_warp[lane] : 0;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, w, d);
        if (lane >= d) w += y;
      }
      s_warp[lane] = w;                          // inclusive scan of warp totals
    }
    __syncthreads();
    const int warp_excl = wid == 0 ? 0 : s_warp[wid - 1];
    if (b < B) { need(b) = n; off(b) = s_carry + warp_excl + x - n; }
    __syncthreads();
    if (tid == 0) s_carry += s_warp[nw - 1];
    __syncthreads();
  }
  const int total = s_carry;
  if (s_bad || total > count) {
    if (tid == 0) wf_raise(status, (int)WF_ERR_OUT_OF_PAGES);
    return false;
  }
  for (int b = wid; b < B; b += nw) {            // one warp per sequence copies its ring entries
    const int s = seq(b);
    const int n = need(b), o = off(b), held = kv.pages_held[s];
    for (int i = lane; i < n; i += 32)
      kv.block_table[(size_t)s * kv.max_pages_per_seq + held + i] = kv.free_ring[(head + o + i) % kv.num_pages];
    __syncwarp();
    if (lane == 0 && n > 0) kv.pages_held[s] = held + n;
  }
  __syncthreads();
  if (tid == 0) {
    kv.ring_state[0] = (head + total) % kv.num_pages;
    kv.ring_state[1] = count - total;
  }
  __syncthreads();
  return true;
}

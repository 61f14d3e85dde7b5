// Context lifecycle, device status word, and the paged-KV block table (reading C24).
#include <stdarg.h>
#include <string.h>

#include <new>
#include <vector>

#include "wf_internal.cuh"

int wf_set_error(wf_ctx* ctx, int code, const char* fmt, ...) {
  if (ctx) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

int wf_check_launch(wf_ctx* ctx, const char* what) {
  ctx->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return wf_set_error(ctx, WF_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
  return WF_OK;
}

wf_encode_tiled_fn wf_get_encode_tiled() {
  static wf_encode_tiled_fn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return (wf_encode_tiled_fn)f;
  }();
  return fn;
}

int wf_make_tmap_2d(wf_ctx* ctx, CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                    uint32_t box_rows) {
  wf_encode_tiled_fn encode = wf_get_encode_tiled();
  WF_REQUIRE(ctx, encode, WF_ERR_CUDA, "cuTensorMapEncodeTiled unavailable");
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * 2};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  WF_REQUIRE(ctx, r == CUDA_SUCCESS, WF_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return WF_OK;
}

extern "C" int wf_ctx_create(wf_ctx** out, int device_ordinal) {
  if (!out) return WF_ERR_INVALID_ARG;
  *out = nullptr;
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || device_ordinal < 0 || device_ordinal >= n) return WF_ERR_CUDA;
  if (cudaSetDevice(device_ordinal) != cudaSuccess) return WF_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device_ordinal) != cudaSuccess) return WF_ERR_CUDA;
  if (prop.major != 10) return WF_ERR_UNSUPPORTED_SHAPE;   // sm_100a code only; no fallback path
  wf_ctx* c = new (std::nothrow) wf_ctx();
  if (!c) return WF_ERR_INVALID_ARG;
  c->device = device_ordinal;
  c->sm_count = prop.multiProcessorCount;
  c->launches = 0;
  c->func_configured = 0;
  c->deterministic = 0;
  c->attn_early = 0;
  memset(c->attn_max_clusters, 0, sizeof(c->attn_max_clusters));
  c->attn_cluster_override = -1;
  c->err[0] = 0;
  c->n_counters = 1 << 16;
  if (cudaMalloc(&c->d_status, sizeof(int)) != cudaSuccess ||
      cudaMalloc(&c->d_counters, sizeof(unsigned int) * c->n_counters) != cudaSuccess ||
      cudaMalloc(&c->d_counters_attn, sizeof(unsigned int) * c->n_counters) != cudaSuccess) {
    delete c;
    return WF_ERR_CUDA;
  }
  cudaMemset(c->d_status, 0, sizeof(int));
  cudaMemset(c->d_counters, 0, sizeof(unsigned int) * c->n_counters);
  cudaMemset(c->d_counters_attn, 0, sizeof(unsigned int) * c->n_counters);
  cudaDeviceSynchronize();
  *out = c;
  return WF_OK;
}

extern "C" int wf_ctx_destroy(wf_ctx* ctx) {
  if (!ctx) return WF_ERR_INVALID_ARG;
  cudaFree(ctx->d_status);
  cudaFree(ctx->d_counters);
  cudaFree(ctx->d_counters_attn);
  delete ctx;
  return WF_OK;
}

extern "C" const char* wf_last_error(const wf_ctx* ctx) { return ctx ? ctx->err : "null ctx"; }

extern "C" int64_t wf_launch_count(const wf_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int wf_poll_status(wf_ctx* ctx, void* stream, int* status_host) {
  if (!ctx || !status_host) return WF_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  WF_CUDA(ctx, cudaMemcpyAsync(status_host, ctx->d_status, sizeof(int), cudaMemcpyDeviceToHost, st));
  WF_CUDA(ctx, cudaMemsetAsync(ctx->d_status, 0, sizeof(int), st));
  WF_CUDA(ctx, cudaStreamSynchronize(st));
  return WF_OK;
}

// ------------------------------------------------------------------------------------------------
// paged KV
// ------------------------------------------------------------------------------------------------
extern "C" int wf_kv_create(wf_ctx* ctx, const wf_kv_shape* s, void* k_pool, void* v_pool,
                            int32_t* block_table, int32_t* seq_len, const int32_t* free_pages_host,
                            int n_free, wf_paged_kv** out) {
  if (!ctx || !out) return WF_ERR_INVALID_ARG;
  *out = nullptr;
  WF_REQUIRE(ctx, s && k_pool && v_pool && block_table && seq_len, WF_ERR_INVALID_ARG, "wf_kv_create: null argument");
  WF_REQUIRE(ctx, s->n_layers > 0 && s->n_kv_heads > 0 && s->num_pages > 0 && s->max_seqs > 0 &&
                 s->max_pages_per_seq > 0, WF_ERR_INVALID_ARG, "wf_kv_create: non-positive shape");
  WF_REQUIRE(ctx, s->page_size == 16, WF_ERR_UNSUPPORTED_SHAPE, "wf_kv_create: page_size must be 16");
  WF_REQUIRE(ctx, s->head_dim == 64 || s->head_dim == 128, WF_ERR_UNSUPPORTED_SHAPE,
             "wf_kv_create: head_dim must be 64 or 128");
  WF_REQUIRE(ctx, n_free >= 0 && n_free <= s->num_pages && (n_free == 0 || free_pages_host),
             WF_ERR_INVALID_ARG, "wf_kv_create: bad free list");
  WF_REQUIRE(ctx, ((uintptr_t)k_pool % 16 == 0) && ((uintptr_t)v_pool % 16 == 0), WF_ERR_INVALID_ARG,
             "wf_kv_create: pools must be 16-byte aligned");
  std::vector<char> seen(s->num_pages, 0);
  for (int i = 0; i < n_free; ++i) {
    int p = free_pages_host[i];
    WF_REQUIRE(ctx, p >= 0 && p < s->num_pages && !seen[p], WF_ERR_INVALID_ARG,
               "wf_kv_create: free list entry %d invalid or duplicated", i);
    seen[p] = 1;
  }
  wf_paged_kv* kv = new (std::nothrow) wf_paged_kv();
  if (!kv) return wf_set_error(ctx, WF_ERR_INVALID_ARG, "wf_kv_create: host allocation failed");
  kv->ctx = ctx;
  kv->s = *s;
  kv->k_pool = (__nv_bfloat16*)k_pool;
  kv->v_pool = (__nv_bfloat16*)v_pool;
  kv->block_table = block_table;
  kv->seq_len = seq_len;
  kv->pages_held = kv->free_ring = kv->ring_state = kv->scratch = nullptr;
  kv->d_tmaps = nullptr;
  kv->h_tiles_hint = nullptr;
  CUtensorMap maps[2];
  {
    const uint64_t rows = (uint64_t)s->n_layers * s->num_pages * s->n_kv_heads * s->page_size;
    int rc = wf_make_tmap_2d(ctx, &maps[0], k_pool, rows, s->head_dim, 64, 16);
    if (rc == WF_OK) rc = wf_make_tmap_2d(ctx, &maps[1], v_pool, rows, s->head_dim, 64, 16);
    if (rc != WF_OK) { delete kv; return rc; }
  }
  cudaError_t e = cudaMalloc(&kv->pages_held, sizeof(int32_t) * s->max_seqs);
  if (e == cudaSuccess) e = cudaMalloc(&kv->free_ring, sizeof(int32_t) * s->num_pages);
  if (e == cudaSuccess) e = cudaMalloc(&kv->ring_state, sizeof(int32_t) * 2);
  if (e == cudaSuccess) e = cudaMalloc(&kv->scratch, sizeof(int32_t) * 2 * s->max_seqs);
  if (e == cudaSuccess) e = cudaMalloc(&kv->d_tmaps, sizeof(maps));
  if (e == cudaSuccess) e = cudaHostAlloc(&kv->h_tiles_hint, sizeof(int), cudaHostAllocMapped);
  if (e == cudaSuccess) *kv->h_tiles_hint = -1;
  if (e == cudaSuccess) e = cudaMemcpy(kv->d_tmaps, maps, sizeof(maps), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemset(kv->pages_held, 0, sizeof(int32_t) * s->max_seqs);
  if (e == cudaSuccess) e = cudaMemset(kv->free_ring, 0xff, sizeof(int32_t) * s->num_pages);
  if (e == cudaSuccess && n_free)
    e = cudaMemcpy(kv->free_ring, free_pages_host, sizeof(int32_t) * n_free, cudaMemcpyHostToDevice);
  int32_t st[2] = {0, n_free};
  if (e == cudaSuccess) e = cudaMemcpy(kv->ring_state, st, sizeof(st), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    wf_kv_destroy(kv);
    return wf_set_error(ctx, WF_ERR_CUDA, "wf_kv_create: %s", cudaGetErrorString(e));
  }
  *out = kv;
  return WF_OK;
}

extern "C" int wf_kv_destroy(wf_paged_kv* kv) {
  if (!kv) return WF_ERR_INVALID_ARG;
  cudaFree(kv->pages_held);
  cudaFree(kv->free_ring);
  cudaFree(kv->ring_state);
  cudaFree(kv->scratch);
  cudaFree(kv->d_tmaps);
  if (kv->h_tiles_hint) cudaFreeHost(kv->h_tiles_hint);
  delete kv;
  return WF_OK;
}

extern "C" const int32_t* wf_kv_pages_held(const wf_paged_kv* kv) { return kv ? kv->pages_held : nullptr; }

__global__ void __launch_bounds__(1024) wf_kv_reserve_kernel(KvView kv, const int32_t* __restrict__ add_tokens,
                                                             int B, int* status) {
  wf_pdl_wait();
  wf_pdl_trigger();
  kv_reserve_block(kv, B, [&](int b) { return add_tokens[b]; }, [](int b) { return b; }, status);
}

extern "C" int wf_kv_reserve(wf_paged_kv* kv, const int32_t* add_tokens, int B, void* stream) {
  if (!kv) return WF_ERR_INVALID_ARG;
  wf_ctx* ctx = kv->ctx;
  WF_REQUIRE(ctx, add_tokens && B >= 0 && B <= kv->s.max_seqs, WF_ERR_INVALID_ARG, "wf_kv_reserve: bad arguments");
  if (B == 0) return WF_OK;
  wf_launch(wf_kv_reserve_kernel, dim3(1), dim3(1024), 0, (cudaStream_t)stream, kv_view(kv), add_tokens, B, ctx->d_status);
  return wf_check_launch(ctx, "wf_kv_reserve");
}

__global__ void wf_kv_release_kernel(KvView kv, int seq) {
  // pages return to the ring tail in block-table order
  wf_pdl_wait();
  wf_pdl_trigger();
  const int held = kv.pages_held[seq];
  const int head = kv.ring_state[0], count = kv.ring_state[1];
  int32_t* row = kv.block_table + (size_t)seq * kv.max_pages_per_seq;
  for (int i = threadIdx.x; i < held; i += blockDim.x) {
    kv.free_ring[(head + count + i) % kv.num_pages] = row[i];
    row[i] = -1;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    kv.ring_state[1] = count + held;
    kv.pages_held[seq] = 0;
    kv.seq_len[seq] = 0;
  }
}

extern "C" int wf_kv_release_seq(wf_paged_kv* kv, int seq, void* stream) {
  if (!kv) return WF_ERR_INVALID_ARG;
  wf_ctx* ctx = kv->ctx;
  WF_REQUIRE(ctx, seq >= 0 && seq < kv->s.max_seqs, WF_ERR_INVALID_ARG, "wf_kv_release_seq: bad sequence index");
  wf_launch(wf_kv_release_kernel, dim3(1), dim3(256), 0, (cudaStream_t)stream, kv_view(kv), seq);
  return wf_check_launch(ctx, "wf_kv_release_seq");
}

// ---------------------------------------------------------------------------------------------
// Tree verification, step 3: path compaction (reading T5).  One CTA per (sequence, layer).
// A thread owns one 16-byte column (K or V, kv head, 8 elements) of the rows and moves it for every
// step k of the path: position ctx + path[k] -> ctx + k.  The only overlap between the moves is a
// destination that is another step's source, always in the same column, i.e. in the same thread:
// it reads a batch of 8 sources before it writes the batch, and batches ascend (path[j] > j, so a
// later source is never an earlier destination).  No barrier, no second buffer.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) wf_kv_compact_path_kernel(KvView kv, const int32_t* __restrict__ path,
                                                                 int path_stride, const int32_t* __restrict__ n_commit,
                                                                 int* status) {
  __shared__ int s_src[64], s_dst[64];                      // row index in the pool's [page][head][slot] order, head 0
  wf_pdl_wait();
  wf_pdl_trigger();
  const int b = blockIdx.x, layer = blockIdx.y;
  const int nc = min(n_commit[b], 64);
  if (nc <= 1) return;                                      // the root is in place
  const int ctx = kv.seq_len[b];
  const int32_t* bt = kv.block_table + (size_t)b * kv.max_pages_per_seq;
  if (threadIdx.x < nc) {
    const int k = threadIdx.x;
    const int node = path[(size_t)b * path_stride + k];
    const bool ok = node >= k && node < 64 && (ctx + node) / 16 < kv.max_pages_per_seq;
    if (!ok && layer == 0) atomicCAS(status, 0, (int)WF_ERR_INVALID_ARG);
    const int ps = ok ? ctx + node : ctx + k, pd = ctx + k;
    s_src[k] = (bt[ps >> 4] * kv.n_kv_heads) * 16 + (ps & 15);
    s_dst[k] = (bt[pd >> 4] * kv.n_kv_heads) * 16 + (pd & 15);
  }
  __syncthreads();
  const int cpr = kv.head_dim / 8;                          // 16-byte chunks per row
  const int cols = 2 * kv.n_kv_heads * cpr;
  const size_t layer_rows = (size_t)layer * kv.num_pages * kv.n_kv_heads * 16;
  for (int col = threadIdx.x; col < cols; col += blockDim.x) {
    const int which = col / (kv.n_kv_heads * cpr), rem = col % (kv.n_kv_heads * cpr);
    const int head = rem / cpr, chunk = rem % cpr;
    uint4* pool = reinterpret_cast<uint4*>(which ? kv.v_pool : kv.k_pool);
    auto at = [&](int row0) { return pool + (layer_rows + (size_t)row0 + (size_t)head * 16) * cpr + chunk; };
    for (int k0 = 1; k0 < nc; k0 += 8) {
      uint4 x[8];
#pragma unroll
      for (int u = 0; u < 8; ++u)
        if (k0 + u < nc) x[u] = *at(s_src[k0 + u]);
#pragma unroll
      for (int u = 0; u < 8; ++u)
        if (k0 + u < nc && s_src[k0 + u] != s_dst[k0 + u]) *at(s_dst[k0 + u]) = x[u];
    }
  }
}

__global__ void wf_kv_advance_kernel(int32_t* __restrict__ seq_len, const int32_t* __restrict__ n_commit, int B) {
  wf_pdl_wait();
  wf_pdl_trigger();
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < B) seq_len[b] += n_commit[b];
}

extern "C" int wf_kv_compact_path(wf_paged_kv* kv, const int32_t* path, int path_stride, const int32_t* n_commit, int B,
                                  void* stream) {
  if (!kv) return WF_ERR_INVALID_ARG;
  wf_ctx* ctx = kv->ctx;
  WF_REQUIRE(ctx, path && n_commit && path_stride >= 1 && B >= 0 && B <= kv->s.max_seqs, WF_ERR_INVALID_ARG,
             "wf_kv_compact_path: bad arguments");
  if (B == 0) return WF_OK;
  cudaStream_t st = (cudaStream_t)stream;
  wf_launch(wf_kv_compact_path_kernel, dim3(B, kv->s.n_layers), dim3(256), 0, st, kv_view(kv), path, path_stride,
            n_commit, ctx->d_status);
  int rc = wf_check_launch(ctx, "wf_kv_compact_path_kernel");
  if (rc != WF_OK) return rc;
  wf_launch(wf_kv_advance_kernel, dim3((B + 255) / 256), dim3(256), 0, st, kv->seq_len, n_commit, B);
  return wf_check_launch(ctx, "wf_kv_advance_kernel");
}

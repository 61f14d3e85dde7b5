// (c) KV-only prefill and (d) Lazy Catch-up.  TEMPORARY placeholder while the tcgen05 GEMM is written.
#include "wf_internal.cuh"
extern "C" int wf_drafter_create(wf_ctx* ctx, const wf_drafter_shape*, const void* const*, const void* const*,
                                 wf_paged_kv*, void*, int32_t*, wf_drafter** out) {
  if (out) *out = nullptr;
  return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "not built yet");
}
extern "C" int wf_drafter_destroy(wf_drafter*) { return WF_ERR_INVALID_ARG; }
extern "C" int wf_kv_only_prefill(wf_ctx* ctx, wf_drafter*, const void*, const int32_t*, const int32_t*,
                                  const int32_t*, int, int, void*) { return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "not built yet"); }
extern "C" int wf_lazy_catchup_enqueue(wf_ctx* ctx, wf_drafter*, const void*, const int32_t*, const int32_t*,
                                       const int32_t*, const int32_t*, int, int, void*) { return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "not built yet"); }
extern "C" int wf_lazy_catchup_flush(wf_ctx* ctx, wf_drafter*, const int32_t*, int, void*) { return wf_set_error(ctx, WF_ERR_UNSUPPORTED_SHAPE, "not built yet"); }

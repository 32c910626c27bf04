// Decode entry points (placeholder until decode_kernel.cu lands).
#include "ctx.h"
using namespace kam;
extern "C" {
kam_status kam_paged_decode_merge(kam_ctx* c, const void*, const kam_pool*, const int32_t*, int32_t, const int32_t*,
                                  const int64_t*, const int32_t*, int32_t, const kam_patch_ref*, int32_t, int32_t, float,
                                  void*, float*, void*) { return fail(c, KAM_ERR_UNSUPPORTED, "decode not built yet"); }
kam_status kam_window_decode(kam_ctx* c, const void*, const int32_t*, int32_t, int32_t, float, void*, float*, void*) {
  return fail(c, KAM_ERR_UNSUPPORTED, "decode not built yet"); }
kam_status kam_paged_decode_merge_host(kam_ctx* c, const void*, const kam_pool*, const int32_t*, int32_t, const int32_t*,
                                       const int64_t*, const int32_t*, int32_t, const kam_patch_ref*, int32_t, int32_t,
                                       float, void*, float*, void*) { return fail(c, KAM_ERR_UNSUPPORTED, "decode not built yet"); }
kam_status kam_relocate_patch_host(kam_ctx* c, const kam_pool*, const int32_t*, int64_t, int32_t, int64_t, int64_t,
                                   const void* const*, const void* const*, const void* const*, const void* const*,
                                   const void* const*, const void* const*, int32_t, int32_t, void*) {
  return fail(c, KAM_ERR_UNSUPPORTED, "host path not built yet"); }
}

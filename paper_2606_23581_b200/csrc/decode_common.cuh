// Device helpers and launch plumbing shared by the decode kernels (decode_kernel.cu, decode_mla_kernel.cu).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace kam {
namespace {
enum : int { HDR_FIRST = 1, HDR_LAST = 2, HDR_PARTIAL = 4 };

__device__ __forceinline__ float ex2(float x) {                  // 2^x, ex2(-inf) = 0
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {   // 8x8 b16 transpose across the warp
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}
__device__ __forceinline__ float col_max(float v) {              // over the 8 lanes that share lane % 4
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 4));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 8));
  return fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 16));
}
__device__ __forceinline__ float col_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  v += __shfl_xor_sync(0xffffffffu, v, 8);
  return v + __shfl_xor_sync(0xffffffffu, v, 16);
}
__device__ __forceinline__ uint32_t ldg_u32(const void* p) { return __ldg(reinterpret_cast<const unsigned int*>(p)); }
__device__ __forceinline__ uint32_t ldg_u16(const void* p) { return __ldg(reinterpret_cast<const unsigned short*>(p)); }

// On-read patch of one segment: rank of the chunk's kam_patch_ref if the record is well formed and the kernel is specialised
// for it (KT rank tiles), else 0 (no patch; malformed records are counted once per segment by the producer warp).
struct SegPatch { const char* Uk; const char* Uv; const __nv_bfloat16* Wk; const __nv_bfloat16* Wv; long long uts, uhs; int rank, frame; };
__device__ __forceinline__ SegPatch seg_patch(const kam_patch_ref* refs, int idx, int KT, bool need_v, bool* malformed) {
  SegPatch sp{};
  *malformed = false;
  if (!refs || idx < 0) return sp;
  const kam_patch_ref r = refs[idx];
  if (r.rank == 0 || (!r.Uk && !r.Wk && !r.Uv && !r.Wv)) return sp;
  const bool ok = r.rank > 0 && r.rank % 16 == 0 && r.rank <= KT * 16 && r.Uk && r.Wk && (!need_v || (r.Uv && r.Wv)) &&
                  (r.u_token_stride & 7) == 0 && (r.u_head_stride & 7) == 0 && (r.u_head_stride == 0 || r.u_head_stride >= r.rank) &&
                  ((reinterpret_cast<uintptr_t>(r.Uk) | reinterpret_cast<uintptr_t>(r.Wk) |
                    (need_v ? (reinterpret_cast<uintptr_t>(r.Uv) | reinterpret_cast<uintptr_t>(r.Wv)) : 0)) & 15) == 0;
  if (!ok) { *malformed = true; return sp; }
  sp.Uk = static_cast<const char*>(r.Uk); sp.Uv = static_cast<const char*>(r.Uv);
  sp.Wk = static_cast<const __nv_bfloat16*>(r.Wk); sp.Wv = static_cast<const __nv_bfloat16*>(r.Wv);
  sp.uts = r.u_token_stride; sp.uhs = r.u_head_stride; sp.rank = r.rank; sp.frame = r.frame;
  return sp;
}

template <typename K, typename... A>
void launch_ex(K kern, int grid, int block, int smem, bool pdl, cudaStream_t st, const A&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kern, args...);
}
}  // namespace
}  // namespace kam

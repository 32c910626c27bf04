// kam_form_patch: the compile-side step of the method on the GPU (Eq. 2).
//
//   Delta = KV(B|A) - R(delta) KV(B|0)          per layer and KV head, [T x D]   (V: no rotation)
//   Delta ~= U W,  U = U_m S (T x m),  W = V_m^T (m x D)                           top-m singular triplets, S folded into U
//
// The conditioned forward that produces KV(B|A) needs model weights and stays outside; this entry takes
// KV(B|A) as an input.  Algorithm (restated, not ported - the paper only says "SVD"): block subspace iteration on
// Delta^T Delta with oversampling (Halko, Martinsson, Tropp 2011, Alg. 4.4), then Rayleigh-Ritz on the small block:
//   Q0 = fixed pseudo-random [D x b], b = m + 8;   repeat n_iter times:  Q <- orth( Delta^T (Delta Q) )
//   B = Delta Q [T x b];  C = B^T B = Z diag(lambda) Z^T (cyclic Jacobi, one warp);  sigma_j = sqrt(lambda_j), descending
//   W = (Q Z[:, :m])^T,   U S = B Z[:, :m]
// For Delta of rank <= b the result is the exact truncated SVD after one iteration; otherwise the subspace error shrinks by
// (sigma_{b+1} / sigma_m)^2 per iteration.  Everything is fp32 on CUDA cores: one CTA per (layer, KV head), a few MFLOP
// each, paid once per chunk - this is not a hot path and is not tuned like one.
#include <cuda_runtime.h>

#include <algorithm>
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace kam {

namespace {
constexpr int kFpThreads = 256;
constexpr int kFpRows = 16;                // tokens of Delta staged per pass

__device__ __forceinline__ float block_sum(float v, float* red) {      // sum over the CTA, result in every thread
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();                                                     // red[] may still be read from the previous call
  if (lane == 0) red[warp] = v;
  __syncthreads();
  float t = 0.f;
#pragma unroll
  for (int w = 0; w < kFpThreads / 32; ++w) t += red[w];
  return t;
}

__device__ __forceinline__ float hash_unit(uint32_t x) {               // fixed pseudo-random start in (-1, 1)
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return static_cast<float>(static_cast<int32_t>(x)) * (1.0f / 2147483648.0f);
}
}  // namespace

// Delta[l][h][t][c] = cond - R(delta) solo (fp32).  One thread per (token, head, rope pair or plain column).
__global__ void __launch_bounds__(256) kam_delta_kernel(const __grid_constant__ FormPatchParams p) {
  const int l = blockIdx.y;
  const long long n = static_cast<long long>(p.T) * p.H * p.D;
  const __nv_bfloat16* cond = static_cast<const __nv_bfloat16*>(p.cond[l]);
  const __nv_bfloat16* solo = static_cast<const __nv_bfloat16*>(p.solo[l]);
  float* out = p.delta_ws + static_cast<size_t>(l) * n;
  const int half = p.d_r >> 1;
  for (long long idx = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; idx < n; idx += static_cast<long long>(gridDim.x) * blockDim.x) {
    const int c = static_cast<int>(idx % p.D);
    const long long th = idx / p.D;
    const int h = static_cast<int>(th % p.H);
    const long long t = th / p.H;
    float v = __bfloat162float(solo[idx]);
    const int rel = c - p.rope_off;
    if (p.rotate && rel >= 0 && rel < p.d_r) {
      int i, partner; bool first;
      if (p.rope_style == KAM_ROPE_HALF) { first = rel < half; i = first ? rel : rel - half; partner = first ? c + half : c - half; }
      else { first = (rel & 1) == 0; i = rel >> 1; partner = first ? c + 1 : c - 1; }
      const float w = __bfloat162float(solo[idx - c + partner]);
      double sn, cs;
      sincos(static_cast<double>(p.delta) * p.inv_freq[i], &sn, &cs);
      const float cf = static_cast<float>(cs), sf = static_cast<float>(sn);
      v = first ? fmaf(v, cf, -w * sf) : fmaf(w, sf, v * cf);       // a' = a c - b s ; b' = a s + b c
    }
    // workspace layout [l][h][t][c]: one contiguous T x D matrix per (layer, head)
    out[(static_cast<size_t>(h) * p.T + t) * p.D + c] = __bfloat162float(cond[idx]) - v;
  }
}

namespace {
// Orthonormalise the b columns of Q [D][ldq] in shared memory: classical Gram-Schmidt, applied twice per column (CGS2).
// A column with no component left outside the previous ones (Delta of lower rank) becomes zero.
__device__ void orthonormalise(float* Q, int D, int b, int ldq, float* rv, float* red) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int j = 0; j < b; ++j) {
    float n0 = 0.f;
    for (int c = tid; c < D; c += kFpThreads) n0 += Q[c * ldq + j] * Q[c * ldq + j];
    n0 = block_sum(n0, red);
    for (int pass = 0; pass < 2; ++pass) {
      for (int i = warp; i < j; i += kFpThreads / 32) {
        float s = 0.f;
        for (int c = lane; c < D; c += 32) s += Q[c * ldq + i] * Q[c * ldq + j];
#pragma unroll
        for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) rv[i] = s;
      }
      __syncthreads();
      for (int c = tid; c < D; c += kFpThreads) {
        float acc = Q[c * ldq + j];
        for (int i = 0; i < j; ++i) acc = fmaf(-rv[i], Q[c * ldq + i], acc);
        Q[c * ldq + j] = acc;
      }
      __syncthreads();
    }
    float n1 = 0.f;
    for (int c = tid; c < D; c += kFpThreads) n1 += Q[c * ldq + j] * Q[c * ldq + j];
    n1 = block_sum(n1, red);
    const float inv = (n1 > 1e-12f * n0 && n1 > 0.f) ? rsqrtf(n1) : 0.f;
    for (int c = tid; c < D; c += kFpThreads) Q[c * ldq + j] *= inv;
    __syncthreads();
  }
}

// Y[r][j] = sum_c Dblk[r][c] Q[c][j] for the staged rows.
__device__ __forceinline__ void rows_times_q(const float* Dblk, const float* Q, float* Y, int rows, int D, int b, int ldq) {
  for (int idx = threadIdx.x; idx < rows * b; idx += kFpThreads) {
    const int r = idx / b, j = idx - r * b;
    const float* d = Dblk + r * D;
    float acc = 0.f;
    for (int c = 0; c < D; ++c) acc = fmaf(d[c], Q[c * ldq + j], acc);
    Y[r * b + j] = acc;
  }
}
}  // namespace

// One CTA per (layer, KV head): subspace iteration, Rayleigh-Ritz, factors out.
__global__ void __launch_bounds__(kFpThreads) kam_form_patch_kernel(const __grid_constant__ FormPatchParams p) {
  extern __shared__ __align__(16) float sm[];
  const int l = blockIdx.x / p.H, h = blockIdx.x - l * p.H;
  const int D = p.D, b = p.b, ldq = p.ldq, T = p.T, m = p.m;
  const int tid = threadIdx.x;
  float* Q = sm;                           // [D][ldq]
  float* Qn = Q + D * ldq;                 // [D][ldq]   Delta^T (Delta Q); later reused for Z-rotated bases
  float* Dblk = Qn + D * ldq;              // [kFpRows][D]
  float* Y = Dblk + kFpRows * D;           // [kFpRows][b]
  float* C = Y + kFpRows * b;              // [b][b+1]
  float* Z = C + b * (b + 1);              // [b][b+1]
  float* rv = Z + b * (b + 1);             // [b]
  float* red = rv + b;                     // [8]
  int* order = reinterpret_cast<int*>(red + 8);   // [b]
  const float* Delta = p.delta_ws + (static_cast<size_t>(l) * p.H + h) * T * D;
  float* Bws = p.b_ws + (static_cast<size_t>(l) * p.H + h) * T * b;
  const int ldc = b + 1;

  for (int i = tid; i < D * b; i += kFpThreads) { const int c = i / b, j = i - c * b; Q[c * ldq + j] = hash_unit(static_cast<uint32_t>(i) * 2654435761u + 12345u); }
  __syncthreads();
  orthonormalise(Q, D, b, ldq, rv, red);

  for (int it = 0; it < p.n_iter; ++it) {
    for (int i = tid; i < D * ldq; i += kFpThreads) Qn[i] = 0.f;
    for (int t0 = 0; t0 < T; t0 += kFpRows) {
      const int rows = min(kFpRows, T - t0);
      __syncthreads();
      for (int i = tid; i < rows * D; i += kFpThreads) Dblk[i] = Delta[static_cast<size_t>(t0) * D + i];
      __syncthreads();
      rows_times_q(Dblk, Q, Y, rows, D, b, ldq);
      __syncthreads();
      for (int idx = tid; idx < D * b; idx += kFpThreads) {       // Qn += Dblk^T Y
        const int c = idx / b, j = idx - c * b;
        float acc = Qn[c * ldq + j];
        for (int r = 0; r < rows; ++r) acc = fmaf(Dblk[r * D + c], Y[r * b + j], acc);
        Qn[c * ldq + j] = acc;
      }
    }
    __syncthreads();
    for (int i = tid; i < D * ldq; i += kFpThreads) Q[i] = Qn[i];
    __syncthreads();
    orthonormalise(Q, D, b, ldq, rv, red);
  }

  // ---- B = Delta Q (kept in global memory), C = B^T B
  for (int i = tid; i < b * ldc; i += kFpThreads) { C[i] = 0.f; Z[i] = 0.f; }
  for (int t0 = 0; t0 < T; t0 += kFpRows) {
    const int rows = min(kFpRows, T - t0);
    __syncthreads();
    for (int i = tid; i < rows * D; i += kFpThreads) Dblk[i] = Delta[static_cast<size_t>(t0) * D + i];
    __syncthreads();
    rows_times_q(Dblk, Q, Y, rows, D, b, ldq);
    __syncthreads();
    for (int i = tid; i < rows * b; i += kFpThreads) Bws[static_cast<size_t>(t0) * b + i] = Y[i];
    for (int idx = tid; idx < b * b; idx += kFpThreads) {
      const int i = idx / b, j = idx - i * b;
      float acc = C[i * ldc + j];
      for (int r = 0; r < rows; ++r) acc = fmaf(Y[r * b + i], Y[r * b + j], acc);
      C[i * ldc + j] = acc;
    }
  }
  __syncthreads();
  for (int i = tid; i < b; i += kFpThreads) Z[i * ldc + i] = 1.f;
  __syncthreads();

  // ---- C = Z diag(lambda) Z^T: cyclic Jacobi by one warp (b <= 72; lanes own rows/columns k = lane, lane + 32, ...)
  if (tid < 32) {
    const int lane = tid;
    for (int sweep = 0; sweep < 16; ++sweep) {
      float off = 0.f;
      for (int i = lane; i < b; i += 32)
        for (int j = 0; j < b; ++j) if (j != i) off += C[i * ldc + j] * C[i * ldc + j];
#pragma unroll
      for (int o = 16; o; o >>= 1) off += __shfl_xor_sync(0xffffffffu, off, o);
      float diag = 0.f;
      for (int i = lane; i < b; i += 32) diag += C[i * ldc + i] * C[i * ldc + i];
#pragma unroll
      for (int o = 16; o; o >>= 1) diag += __shfl_xor_sync(0xffffffffu, diag, o);
      if (off <= 1e-14f * diag) break;
      for (int pp = 0; pp < b - 1; ++pp) {
        for (int qq = pp + 1; qq < b; ++qq) {
          const float apq = C[pp * ldc + qq];
          const float app = C[pp * ldc + pp], aqq = C[qq * ldc + qq];
          if (fabsf(apq) <= 1e-9f * sqrtf(fabsf(app * aqq)) || apq == 0.f) continue;        // warp-uniform: all lanes read the same values
          const float tau = (aqq - app) / (2.f * apq);
          const float t = (tau >= 0.f ? 1.f : -1.f) / (fabsf(tau) + sqrtf(1.f + tau * tau));
          const float cs = rsqrtf(1.f + t * t), sn = t * cs;
          for (int k = lane; k < b; k += 32) {                  // columns p, q
            const float ckp = C[k * ldc + pp], ckq = C[k * ldc + qq];
            C[k * ldc + pp] = cs * ckp - sn * ckq; C[k * ldc + qq] = sn * ckp + cs * ckq;
            const float zkp = Z[k * ldc + pp], zkq = Z[k * ldc + qq];
            Z[k * ldc + pp] = cs * zkp - sn * zkq; Z[k * ldc + qq] = sn * zkp + cs * zkq;
          }
          __syncwarp();
          for (int k = lane; k < b; k += 32) {                  // rows p, q
            const float cpk = C[pp * ldc + k], cqk = C[qq * ldc + k];
            C[pp * ldc + k] = cs * cpk - sn * cqk; C[qq * ldc + k] = sn * cpk + cs * cqk;
          }
          __syncwarp();
        }
      }
    }
    // eigenvalues in descending order (selection; b is tiny)
    if (lane == 0) {
      for (int i = 0; i < b; ++i) order[i] = i;
      for (int i = 0; i < b; ++i) {
        int best = i;
        for (int j = i + 1; j < b; ++j) if (C[order[j] * ldc + order[j]] > C[order[best] * ldc + order[best]]) best = j;
        const int tmp = order[i]; order[i] = order[best]; order[best] = tmp;
      }
    }
  }
  __syncthreads();

  // ---- W[h][j][c] = sum_i Q[c][i] Z[i][o_j];  U[t][h][j] = sum_i B[t][i] Z[i][o_j];  sigma_j = sqrt(lambda_j)
  __nv_bfloat16* W = static_cast<__nv_bfloat16*>(p.W_out[l]) + static_cast<size_t>(h) * m * D;
  for (int idx = tid; idx < m * D; idx += kFpThreads) {
    const int j = idx / D, c = idx - j * D, o = order[j];
    float acc = 0.f;
    for (int i = 0; i < b; ++i) acc = fmaf(Q[c * ldq + i], Z[i * ldc + o], acc);
    W[idx] = __float2bfloat16_rn(acc);
  }
  __nv_bfloat16* U = static_cast<__nv_bfloat16*>(p.U_out[l]) + static_cast<size_t>(h) * m;
  for (int idx = tid; idx < T * m; idx += kFpThreads) {
    const int t = idx / m, j = idx - t * m, o = order[j];
    const float* brow = Bws + static_cast<size_t>(t) * b;
    float acc = 0.f;
    for (int i = 0; i < b; ++i) acc = fmaf(brow[i], Z[i * ldc + o], acc);
    U[static_cast<size_t>(t) * p.H * m + j] = __float2bfloat16_rn(acc);
  }
  if (p.sigma_out)
    for (int j = tid; j < m; j += kFpThreads) p.sigma_out[(static_cast<size_t>(l) * p.H + h) * m + j] = sqrtf(fmaxf(C[order[j] * ldc + order[j]], 0.f));
}

void launch_form_patch(const FormPatchParams& p, cudaStream_t st) {
  const long long n = static_cast<long long>(p.T) * p.H * p.D;
  dim3 g1(static_cast<unsigned>(std::min<long long>((n + 255) / 256, 2048)), p.L);
  kam_delta_kernel<<<g1, 256, 0, st>>>(p);
  cudaFuncSetAttribute(kam_form_patch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, p.smem_bytes);
  kam_form_patch_kernel<<<p.L * p.H, kFpThreads, p.smem_bytes, st>>>(p);
}

}  // namespace kam

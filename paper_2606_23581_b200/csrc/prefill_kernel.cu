// kam_paged_prefill_kernel: the readout of P:44 for a BLOCK of query rows over relocated chunks in the paged pool
// (SURVEY.md 8(f) f4 "chunked-prefill (multi-query) attention over relocated chunks"; the TTFT path of P:105 / P:349: after
// `apply_reuse` has placed the recalled chunks, the appended text turn is prefilled over them).
//
//   row (t, hq) of request b:   s_j = sm_scale * q[t,hq] . k^_j,   k^_j = R(chunk_offset of j's chunk) k_j   (never written)
//                               visible j: all cached tokens (causal = 0) or j <= N_b - Tq + t (causal = 1: the rows are the
//                               last Tq cached tokens, reading R-19)
//                               out = sum_j softmax(s)_j v_j,   lse = ln sum_j e^{s_j}
//
// Unlike decode, where M = the <= 8 query heads of one KV head and the kernel is a pure HBM stream, here M = Tq x G query rows
// per KV head: a dense contraction (4 Tq Hq N D flops against N H D x 4 bytes).  This is the mma.sync formulation - the
// baseline the tcgen05 question is asked of (north_star: tensor memory "only if ncu shows them to be the limiter";
// profiles/ncu_prefill_r02.md has the tensor-pipe figure) - in the FlashAttention-2 shape:
//   * one CTA = 4 warps x 16 rows = 64 rows of the flattened (token, head-in-group) row space of ONE KV head; grid = (row tiles,
//     KV heads, requests); no split over the cached tokens (Tq x G x H x batch row tiles are parallelism enough), hence no
//     partials and no merge kernel: the per-chunk softmax states are merged in registers, tile by tile, by the same
//     log-sum-exp state merge (running reference m, mass l, O rescaled) - P:44's merge, applied online;
//   * the cached tokens of a request are walked chunk by chunk in 64-token tiles (a tile never straddles a chunk, so one
//     rotation serves it); K and V tiles arrive through a two-stage cp.async pipeline, one 16-byte copy per (token, 8
//     columns), slots mapped through the block table per token (A1), rows beyond the chunk zero-filled; 16-byte chunks are
//     XOR-swizzled by the token's low bits so that ldmatrix (K) and ldmatrix.trans (V) are conflict-free;
//   * relocation on read rotates the QUERY, once per chunk: q~ = R(-delta) q, rebuilt in the A fragments from the staged q and
//     carried as bf16 hi + lo (the rotation then costs no precision; chunks with delta = 0 skip the lo products);
//   * causal masking only on the tiles the diagonal crosses; tiles wholly beyond the last row's horizon are never loaded.
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace kam {

namespace {

constexpr int kPfWarps = 4;
constexpr int kPfThreads = kPfWarps * 32;
constexpr int kPfM = 16 * kPfWarps;      // rows per CTA
constexpr int kPfN = 64;                 // cached tokens per tile

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src, bool valid) {
  const int bytes = valid ? 16 : 0;      // src-size 0: the 16 bytes are zero-filled, nothing is read
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ float ex2f(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// Walk over the 64-token tiles of a request's cached tokens, chunk by chunk, up to the horizon `vis_hi`.
struct PfTiles {
  const int32_t* cs;       // the request's CSR row
  const long long* offs;   // the request's chunk offsets or nullptr
  int nc, base0, vis_hi;
  int c, lo, hi, pos;      // current chunk, its logical token range, the tile's first token
  __device__ __forceinline__ bool enter(int chunk) {      // first tile of the first non-empty chunk >= chunk below the horizon
    for (c = chunk; c < nc; ++c) {
      lo = cs[c] - base0; hi = cs[c + 1] - base0;
      if (lo >= vis_hi) return false;
      if (hi > lo) { pos = lo; return true; }
    }
    return false;
  }
  __device__ __forceinline__ bool next() {
    pos += kPfN;
    if (pos < hi && pos < vis_hi) return true;
    return enter(c + 1);
  }
  __device__ __forceinline__ long long delta() const { return offs ? offs[c] : 0; }
};

}  // namespace

template <int D>
__global__ void __launch_bounds__(kPfThreads, 2) kam_paged_prefill_kernel(const __grid_constant__ PrefillParams p) {
  constexpr int KS = D / 16;               // k-steps of QK^T
  constexpr int CPR = D / 8;               // 16-byte chunks per row
  constexpr int ROWB = D * 2;              // bytes per row
  constexpr int TILEB = kPfN * ROWB;
  extern __shared__ __align__(128) uint8_t smem[];
  uint8_t* sQ = smem;                                    // [64 rows][D] bf16, swizzled
  uint8_t* sK = sQ + kPfM * ROWB;                        // 2 x [64 tokens][D]
  uint8_t* sV = sK + 2 * TILEB;
  float2* cs_tab = reinterpret_cast<float2*>(sV + 2 * TILEB);   // (cos, sin)(delta f_i), i < D / 2

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gq = lane >> 2, t4 = lane & 3;
  const int b = blockIdx.z, h = blockIdx.y, G = p.G;
  const int row0 = blockIdx.x * kPfM;                    // first flattened row (t * G + g) of this CTA
  const int n_rows = p.Tq * G;
  const int32_t* cs = p.chunk_starts + static_cast<size_t>(b) * (p.max_chunks + 1);
  const int nc = min(p.n_chunks[b], p.max_chunks);
  const int base0 = cs[0];
  const int N = nc > 0 ? cs[nc] - base0 : 0;             // cached tokens of the request
  const int32_t* bt = p.block_tables + static_cast<size_t>(b) * p.max_pages;
  const char* pool_k = static_cast<const char*>(p.pool_k_layers[p.layer]);
  const char* pool_v = static_cast<const char*>(p.pool_v_layers[p.layer]);
  const size_t tok_bytes = static_cast<size_t>(p.H) * ROWB;     // one token's row of all KV heads in the pool
  const size_t head_off = static_cast<size_t>(h) * ROWB;

  // ---- stage this CTA's query rows (rows past the end are zeros)
  for (int idx = threadIdx.x; idx < kPfM * CPR; idx += kPfThreads) {
    const int r = idx / CPR, c = idx - r * CPR;
    const int fr = row0 + r;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (fr < n_rows) {
      const int t = fr / G, g = fr - t * G;
      v = *reinterpret_cast<const uint4*>(static_cast<const char*>(p.q) + ((static_cast<size_t>(b) * p.Tq + t) * p.Hq + h * G + g) * ROWB + c * 16);
    }
    *reinterpret_cast<uint4*>(sQ + r * ROWB + ((c ^ (r & 7)) << 4)) = v;
  }

  // ---- horizon of this CTA: the last row's, and whether any masking can occur
  const int t_lo = row0 / G, t_hi = min(row0 + kPfM - 1, n_rows - 1) / G;
  const int shift = N - p.Tq;                             // causal: row of token t sees j <= shift + t
  PfTiles cur;
  cur.cs = cs; cur.offs = p.chunk_offsets ? p.chunk_offsets + static_cast<size_t>(b) * p.max_chunks : nullptr;
  cur.nc = nc; cur.base0 = base0;
  cur.vis_hi = p.causal ? min(N, max(0, shift + t_hi + 1)) : N;
  bool more = cur.enter(0);

  const uint32_t sK_u = smem_u32(sK), sV_u = smem_u32(sV);
  // loader: thread -> 16-byte chunk lc of rows lr0 + 8 i (D = 128: 16 chunks per row, 8 rows per pass)
  constexpr int RPP = kPfThreads / CPR;                   // rows per pass
  const int lc = threadIdx.x % CPR, lr0 = threadIdx.x / CPR;
  auto issue = [&](const PfTiles& tl, int buf) {
#pragma unroll
    for (int i = 0; i < kPfN / RPP; ++i) {
      const int r = lr0 + i * RPP;
      const int tok = tl.pos + r;
      bool valid = tok < tl.hi;
      size_t src = 0;
      if (valid) {
        const int pg = p.P_shift >= 0 ? (tok >> p.P_shift) : tok / p.P;
        const int page = pg < p.max_pages ? bt[pg] : -1;
        if (page >= 0 && page < p.num_pages) {
          src = (static_cast<size_t>(page) * p.P + (tok - pg * p.P)) * tok_bytes + head_off + lc * 16;     // A1 slot mapping
        } else {                                              // inconsistent metadata: a zero row, never a wild read
          valid = false;
          if (lc == 0 && (tok == tl.pos || tok == pg * p.P)) atomicAdd(p.err, 1);
        }
      }
      const uint32_t d = static_cast<uint32_t>(buf * TILEB + r * ROWB + ((lc ^ (r & 7)) << 4));
      cp_async_16(sK_u + d, pool_k + src, valid);
      cp_async_16(sV_u + d, pool_v + src, valid);
    }
    cp_async_commit();
  };
  if (more) issue(cur, 0);

  // ---- per-warp state: 16 rows (gq, gq + 8)
  uint32_t qh[KS][4], ql[KS][4];
  float O[D / 8][4];
#pragma unroll
  for (int n = 0; n < D / 8; ++n) O[n][0] = O[n][1] = O[n][2] = O[n][3] = 0.f;
  float m_run[2] = {-CUDART_INF_F, -CUDART_INF_F}, l_run[2] = {0.f, 0.f};
  const float scale_log2 = p.sm_scale * 1.4426950408889634f;
  const int fr0 = row0 + warp * 16 + gq, fr1 = fr0 + 8;     // this lane's two flattened rows
  const int tq0 = fr0 / G, tq1 = fr1 / G;
  const int lim0 = p.causal ? shift + tq0 : N, lim1 = p.causal ? shift + tq1 : N;     // largest visible j of each row
  const int cta_lim_lo = p.causal ? shift + t_lo : N;      // a tile whose last token is <= this needs no causal mask
  bool use_lo = false;
  int cur_chunk = -1, buf = 0;
  const uint32_t sQ_u = smem_u32(sQ);
  // ldmatrix lane addressing: A (q rows), B (K rows: token-major), B^T (V rows through .trans)
  const int a_row = warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, a_ch = lane >> 4;
  const int k_row = (lane & 7) + ((lane >> 4) << 3), k_ch = (lane >> 3) & 1;
  const int v_row = (lane & 7) + ((lane >> 3) & 1) * 8, v_ch = lane >> 4;

  __syncthreads();                                         // sQ is staged
  while (more) {
    PfTiles nxt = cur;
    const bool has_next = nxt.next();
    if (has_next) issue(nxt, buf ^ 1);
    if (has_next) cp_async_wait<1>(); else cp_async_wait<0>();
    __syncthreads();                                       // tile `cur` has landed for every thread

    if (cur.c != cur_chunk) {
      // ---- new chunk: q~ = R(-delta) q in the A fragments (hi + lo); delta = 0 keeps the staged bits
      cur_chunk = cur.c;
      const long long delta = cur.delta();
      use_lo = delta != 0;
      if (use_lo) {
        if (threadIdx.x < D / 2) {
          double sn, csn;
          sincos(static_cast<double>(delta) * p.inv_freq[threadIdx.x], &sn, &csn);       // fp64 angle (R-18)
          cs_tab[threadIdx.x] = make_float2(static_cast<float>(csn), static_cast<float>(sn));
        }
        __syncthreads();
      }
#pragma unroll
      for (int ks = 0; ks < KS; ++ks)
        ldmatrix_x4(qh[ks][0], qh[ks][1], qh[ks][2], qh[ks][3], sQ_u + a_row * ROWB + (((2 * ks + a_ch) ^ (a_row & 7)) << 4));
      if (use_lo) {
        auto rot = [&](float x, float y, float2 u, float& xo, float& yo) { xo = fmaf(x, u.x, y * u.y); yo = fmaf(y, u.x, -x * u.y); };
        auto split = [&](float a, float bq, uint32_t& hi, uint32_t& lo) {
          hi = pack_bf16x2(a, bq);
          lo = pack_bf16x2(a - bf_lo(hi), bq - bf_hi(hi));
        };
        if (p.rope_style == KAM_ROPE_HALF) {
#pragma unroll
          for (int ks = 0; ks < KS / 2; ++ks)
#pragma unroll
            for (int r = 0; r < 4; ++r) {
              const int i0 = 16 * ks + (r >> 1) * 8 + 2 * t4;                  // frequency of the register's first column
              const float2 u0 = cs_tab[i0], u1 = cs_tab[i0 + 1];
              const uint32_t xw = qh[ks][r], yw = qh[ks + KS / 2][r];
              float x0, y0, x1, y1;
              rot(bf_lo(xw), bf_lo(yw), u0, x0, y0);
              rot(bf_hi(xw), bf_hi(yw), u1, x1, y1);
              split(x0, x1, qh[ks][r], ql[ks][r]);
              split(y0, y1, qh[ks + KS / 2][r], ql[ks + KS / 2][r]);
            }
        } else {
#pragma unroll
          for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int r = 0; r < 4; ++r) {
              const float2 u = cs_tab[8 * ks + (r >> 1) * 4 + t4];              // pair (2i, 2i+1) sits in one register
              float x, y;
              rot(bf_lo(qh[ks][r]), bf_hi(qh[ks][r]), u, x, y);
              split(x, y, qh[ks][r], ql[ks][r]);
            }
        }
      }
    }

    // ---- S[16 rows][64 tokens] = q~ K^T
    float S[kPfN / 8][4];
#pragma unroll
    for (int j = 0; j < kPfN / 8; ++j) S[j][0] = S[j][1] = S[j][2] = S[j][3] = 0.f;
    const uint32_t kb = sK_u + buf * TILEB, vb = sV_u + buf * TILEB;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
#pragma unroll
      for (int jp = 0; jp < kPfN / 16; ++jp) {
        uint32_t b0, b1, b2, b3;
        const int r = jp * 16 + k_row;
        ldmatrix_x4(b0, b1, b2, b3, kb + r * ROWB + (((2 * ks + k_ch) ^ (r & 7)) << 4));
        mma_bf16_16816(S[2 * jp][0], S[2 * jp][1], S[2 * jp][2], S[2 * jp][3], qh[ks][0], qh[ks][1], qh[ks][2], qh[ks][3], b0, b1);
        mma_bf16_16816(S[2 * jp + 1][0], S[2 * jp + 1][1], S[2 * jp + 1][2], S[2 * jp + 1][3], qh[ks][0], qh[ks][1], qh[ks][2], qh[ks][3], b2, b3);
        if (use_lo) {
          mma_bf16_16816(S[2 * jp][0], S[2 * jp][1], S[2 * jp][2], S[2 * jp][3], ql[ks][0], ql[ks][1], ql[ks][2], ql[ks][3], b0, b1);
          mma_bf16_16816(S[2 * jp + 1][0], S[2 * jp + 1][1], S[2 * jp + 1][2], S[2 * jp + 1][3], ql[ks][0], ql[ks][1], ql[ks][2], ql[ks][3], b2, b3);
        }
      }
    }

    // ---- mask (only where the chunk ends inside the tile or the diagonal crosses it), then the online state merge
    const int tile_hi = min(cur.pos + kPfN, cur.hi) - 1;            // last real token of the tile
    const bool masked = (cur.pos + kPfN > cur.hi) || (tile_hi > cta_lim_lo);
    float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
#pragma unroll
    for (int j = 0; j < kPfN / 8; ++j) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        float v = S[j][e] * scale_log2;
        if (masked) {
          const int tok = cur.pos + 8 * j + 2 * t4 + (e & 1);
          if (tok > tile_hi || tok > ((e & 2) ? lim1 : lim0)) v = -CUDART_INF_F;
        }
        S[j][e] = v;
        if (e & 2) mx1 = fmaxf(mx1, v); else mx0 = fmaxf(mx0, v);
      }
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1)); mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1)); mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(m_run[0], mx0), mn1 = fmaxf(m_run[1], mx1);
    const float ref0 = mn0 == -CUDART_INF_F ? 0.f : mn0, ref1 = mn1 == -CUDART_INF_F ? 0.f : mn1;   // a row that has seen nothing yet
    const float al0 = ex2f(m_run[0] - ref0), al1 = ex2f(m_run[1] - ref1);                             // e^{-inf} = 0 on the first tile
    m_run[0] = mn0; m_run[1] = mn1;
    float sum0 = 0.f, sum1 = 0.f;
    uint32_t P[kPfN / 16][4];
#pragma unroll
    for (int j = 0; j < kPfN / 8; ++j) {
      const float p0 = ex2f(S[j][0] - ref0), p1 = ex2f(S[j][1] - ref0), p2 = ex2f(S[j][2] - ref1), p3 = ex2f(S[j][3] - ref1);
      sum0 += p0 + p1; sum1 += p2 + p3;
      P[j >> 1][(j & 1) * 2] = pack_bf16x2(p0, p1);
      P[j >> 1][(j & 1) * 2 + 1] = pack_bf16x2(p2, p3);
    }
    l_run[0] = fmaf(l_run[0], al0, sum0); l_run[1] = fmaf(l_run[1], al1, sum1);     // quad-partial masses; reduced at the end
#pragma unroll
    for (int n = 0; n < D / 8; ++n) { O[n][0] *= al0; O[n][1] *= al0; O[n][2] *= al1; O[n][3] *= al1; }

    // ---- O[16 rows][D] += P V
#pragma unroll
    for (int kk = 0; kk < kPfN / 16; ++kk) {
#pragma unroll
      for (int np = 0; np < D / 16; ++np) {
        uint32_t b0, b1, b2, b3;
        const int r = kk * 16 + v_row;
        ldmatrix_x4_trans(b0, b1, b2, b3, vb + r * ROWB + (((2 * np + v_ch) ^ (r & 7)) << 4));
        mma_bf16_16816(O[2 * np][0], O[2 * np][1], O[2 * np][2], O[2 * np][3], P[kk][0], P[kk][1], P[kk][2], P[kk][3], b0, b1);
        mma_bf16_16816(O[2 * np + 1][0], O[2 * np + 1][1], O[2 * np + 1][2], O[2 * np + 1][3], P[kk][0], P[kk][1], P[kk][2], P[kk][3], b2, b3);
      }
    }
    __syncthreads();                                       // every warp is done with `buf` before the next issue overwrites it
    cur = nxt; more = has_next; buf ^= 1;
  }

  // ---- write out: out = O / l (bf16), lse = ln 2 * m + ln l; a row that saw nothing: 0 and -inf
  float l0 = l_run[0], l1 = l_run[1];
  l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
  const float inv0 = l0 > 0.f ? 1.f / l0 : 0.f, inv1 = l1 > 0.f ? 1.f / l1 : 0.f;
  constexpr float kLn2 = 0.6931471805599453f;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int fr = half ? fr1 : fr0;
    if (fr >= n_rows) continue;
    const int t = fr / G, g = fr - t * G;
    const size_t row = (static_cast<size_t>(b) * p.Tq + t) * p.Hq + h * G + g;
    uint32_t* o = reinterpret_cast<uint32_t*>(static_cast<char*>(p.out) + row * ROWB) + t4;
    const float inv = half ? inv1 : inv0;
#pragma unroll
    for (int n = 0; n < D / 8; ++n) o[n * 4] = pack_bf16x2(O[n][2 * half] * inv, O[n][2 * half + 1] * inv);
    if (t4 == 0) {
      const float l = half ? l1 : l0, m = half ? m_run[1] : m_run[0];
      p.lse[row] = l > 0.f ? m * kLn2 + logf(l) : -CUDART_INF_F;
    }
  }
}

int prefill_smem_bytes(int D) { return kPfM * D * 2 + 4 * kPfN * D * 2 + (D / 2) * 8; }

void launch_prefill(const PrefillParams& p, int D, cudaStream_t st) {
  const int smem = prefill_smem_bytes(D);
  dim3 grid((p.Tq * p.G + kPfM - 1) / kPfM, p.H, p.batch);
  static std::atomic<uint64_t> attr_done{0};          // per device: the attribute is not shared between GPUs
  if (first_launch_on_this_device(attr_done)) {
    cudaFuncSetAttribute(kam_paged_prefill_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, prefill_smem_bytes(128));
    cudaFuncSetAttribute(kam_paged_prefill_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, prefill_smem_bytes(64));
  }
  if (D == 128) kam_paged_prefill_kernel<128><<<grid, kPfThreads, smem, st>>>(p);
  else kam_paged_prefill_kernel<64><<<grid, kPfThreads, smem, st>>>(p);
}

}  // namespace kam

// kam_mla_decode_kernel: fused-on-read paged decode over an MLA latent pool in absorbed form.
//
// A cached token is ONE row [c_KV (512, position-free) | k_pe (64, RoPE)]; with the up-projections absorbed into the query
// and output sides (outside this library) a query head is q = [q_lat 512 | q_pe 64], the score is the 576-wide dot product
// and the value is the latent itself:      s_t = sm_scale * q . k^_t ,   o = sum_t p_t k^_t[0:512]
// so every cached byte is read ONCE and serves both QK^T and PV.  Relocation on read touches only q_pe (q~ = R(-delta) q on
// the rope band, bf16 hi + lo); the rank-m patch on read is one U (the key's): s_t += U[t,:].(W q),  o += (sum_t p_t U[t,:]) W[:, 0:512].
//
// This k-split kernel carries the calls WITH an on-read patch (and KAM_MLA_KSPLIT=1); patch-free calls run the token-split kernel
// (decode_mla_ts_kernel.cu), which is faster (0.129 vs 0.152 ms per layer at batch 64 x 8192 tokens).
// Same plan, partials and merge as the GQA kernel (decode_kernel.cu).  Work unit = (16 query heads, run of 16-token tiles of
// one chunk).  CTA = 1 producer warp (slot mapping A1 + one TMA box [9 x 64 columns][16 tokens][128 B, swizzled] per tile) +
// 4 compute warps.  30 flop per byte is ~35 % of the mma.sync rate at the HBM roofline, so nothing may be computed twice:
//   S^T[16 tokens][16 heads]: the 36 k-steps are split 9 per warp (8 latent + 1 rope); the four partial S fragments meet
//     in a double-buffered shared-memory exchange (one named barrier per tile) and every warp adds them in the same order.
//   softmax: tiny, done by every warp identically (so m, l, P need no second exchange).
//   O^T[512][16 heads]: warp w owns value columns [128 w, 128 w + 128), A = the same box through ldmatrix.trans.
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "decode_common.cuh"
#include "internal.h"

namespace kam {

namespace {
constexpr int kLatSteps = 8;               // latent k-steps per warp: 4 warps x 8 x 16 = 512 columns
constexpr int kSteps = kLatSteps + 1;      // + one 16-column step of the 64-wide rope band
constexpr int kDvTiles = 8;                // 16-row tiles of the value columns a warp owns (128)
constexpr int kD = 576, kDv = 512, kRopeOff = 512, kRopeDim = 64;
}  // namespace

template <int KT>
__global__ void __launch_bounds__((kMlaWarps + 1) * 32, 2)
kam_mla_decode_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + g.n_boxes;
  int4* hdrs = reinterpret_cast<int4*>(smem + g.off_hdr);
  float* xch = reinterpret_cast<float*>(smem + g.off_xch);          // [2 buffers][4 warps][8 values][32 lanes]
  uint8_t* box0 = smem + g.off_box0;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < g.n_boxes; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], kMlaWarps); }
    mbar_fence_init();
  }
  __syncthreads();

  grid_dep_launch();
  if (p.plan_fresh) grid_dep_wait();                             // the plan comes from the kernel right before this one
  const int seg_begin = p.plan.cta_seg[blockIdx.x], seg_end = p.plan.cta_seg[blockIdx.x + 1];
  if (seg_begin >= seg_end) return;

  if (warp == kMlaWarps) {
    // ================================================================ producer warp: slot-map (A1), one box per tile
    int box = 0; uint32_t phase = 0;
    const char* tm_k = static_cast<const char*>(p.tmaps) + static_cast<size_t>(p.layer) * kTmapLayerBytes;
    DecSeg S_next = p.plan.segs[seg_begin];
    grid_dep_wait();
    for (int seg = seg_begin; seg < seg_end; ++seg) {
      const DecSeg S = S_next;
      if (seg + 1 < seg_end) S_next = p.plan.segs[seg + 1];
      const int32_t* bt = p.block_tables + S.bt_off;
      [[maybe_unused]] SegPatch sp{};
      [[maybe_unused]] uint32_t u_row_bytes = 0;
      if constexpr (KT > 0) {
        bool bad;
        sp = seg_patch(p.patches, S.patch, KT, false, &bad);
        if (bad && lane == 0 && S.tile0 * kDecTile <= S.tok_lo && S.hg == 0) atomicAdd(p.err, 1);
        u_row_bytes = static_cast<uint32_t>(sp.rank * 2);
      }
      for (int t0 = 0; t0 < S.n_tiles; t0 += 32) {
        int slot = 0;
        if (t0 + lane < S.n_tiles && t0 + lane > 0) {
          const int tok = (S.tile0 + t0 + lane) * kDecTile;
          const int pg = g.P_shift >= 0 ? (tok >> g.P_shift) : tok / g.P;
          slot = bt[pg] * g.P + (tok - pg * g.P);
        }
        const int nb = min(32, S.n_tiles - t0);
        for (int i = 0; i < nb; ++i) {
          const int s0 = (t0 + i == 0) ? S.slot0 : __shfl_sync(0xffffffffu, slot, i);
          const int tl = t0 + i;
          const int tok = (S.tile0 + tl) * kDecTile;
          const int row_lo = max(S.tok_lo - tok, 0), row_hi = min(S.tok_hi - tok, kDecTile);
          mbar_wait(&empty_bar[box], phase ^ 1);
          uint8_t* dst = box0 + static_cast<size_t>(box) * g.box_bytes;
          const uint32_t u_bytes = static_cast<uint32_t>(row_hi - row_lo) * u_row_bytes;
          if (lane == 0) {
            const int flags = (tl == 0 ? HDR_FIRST : 0) | (tl == S.n_tiles - 1 ? HDR_LAST : 0) |
                              ((row_lo > 0 || row_hi < kDecTile) ? HDR_PARTIAL : 0);
            hdrs[box] = make_int4(seg, flags, row_lo | (row_hi << 8), tok - S.tok_lo);
            mbar_arrive_expect_tx(&full_bar[box], static_cast<uint32_t>(g.kv_bytes) + u_bytes);
            tma_load_3d(dst, tm_k, 0, s0, 0, &full_bar[box]);
          }
          if constexpr (KT > 0) {
            if (u_bytes) {
              __syncwarp();
              if (lane >= row_lo && lane < row_hi)
                bulk_g2s(dst + g.u_off + lane * g.su_row, sp.Uk + static_cast<long long>(tok - S.tok_lo + lane) * sp.uts * 2, u_row_bytes, &full_bar[box]);
            }
          }
          if (++box == g.n_boxes) { box = 0; phase ^= 1; }
        }
      }
    }
    mbar_wait(&empty_bar[box], phase ^ 1);
    if (lane == 0) { hdrs[box] = make_int4(-1, 0, 0, 0); mbar_arrive(&full_bar[box]); }
    return;
  }

  // ================================================================ compute warps
  const int gq = lane >> 2, t4 = lane & 3;
  const float scale_log2 = p.sm_scale * 1.4426950408889634f;
  // this warp's k-steps, as first column: latent [128 w + 16 i), rope band 512 + 16 w
  auto step_col = [&](int i) { return i < kLatSteps ? warp * (kLatSteps * 16) + i * 16 : kRopeOff + warp * 16; };

  uint32_t qhi[2][kSteps][2], qlo[2][2];
  float O[2][kDvTiles][4];
  float m_run[2][2], l_run[2][2];
  bool use_lo = false;
  int n_rows = 0;                                                // query heads of this work unit (16, fewer in the last one)
  constexpr int KTA = KT > 0 ? KT : 1;
  [[maybe_unused]] uint32_t wqh[2][KTA][2], wql[2][KTA][2];
  [[maybe_unused]] float Z[2][KTA][4];
  [[maybe_unused]] int kt_seg = 0;
  [[maybe_unused]] const __nv_bfloat16* W_seg = nullptr;

  const int k_row = (lane & 7) + ((lane >> 3) & 1) * 8, k_hi = lane >> 4;
  const int v_row = (lane & 7) + (lane >> 4) * 8, v_hi = (lane >> 3) & 1;
  const uint32_t k_sw = (k_hi ^ (lane & 7)) << 4, v_sw = (v_hi ^ (lane & 7)) << 4;
  // box address of 16-column step starting at column c (multiple of 16): block c / 64, chunk pair (c / 16) & 3
  auto k_addr = [&](uint32_t base, int c) { return base + (c >> 6) * 2048 + k_row * 128 + (k_sw ^ (((c >> 4) & 3) << 5)); };
  auto v_addr = [&](uint32_t base, int c) { return base + (c >> 6) * 2048 + v_row * 128 + (v_sw ^ (((c >> 4) & 3) << 5)); };

  int box = 0; uint32_t phase = 0;
  int seg = 0, xbuf = 0;
  grid_dep_wait();
  while (true) {
    mbar_wait(&full_bar[box], phase);
    const int4 hdr = hdrs[box];
    if (hdr.x < 0) break;
    uint8_t* bptr = box0 + static_cast<size_t>(box) * g.box_bytes;
    const uint32_t bb = smem_u32(bptr);
    const int cbox = box;
    if (++box == g.n_boxes) { box = 0; phase ^= 1; }

    if (hdr.y & HDR_FIRST) {
      // ---- new segment: this warp's slice of the 16 query rows; the rope step rotated by -delta (hi + lo)
      seg = hdr.x;
      const DecSeg S = p.plan.segs[seg];
      use_lo = S.rotate;
      constexpr int half = kRopeDim / 2;
      const float2* cs = p.plan.cs + static_cast<size_t>(S.chunk) * half;
      const __nv_bfloat16* qb = static_cast<const __nv_bfloat16*>(p.q) + (static_cast<size_t>(S.b) * g.Hq + static_cast<size_t>(S.hg) * kMlaHeads) * kD;
      n_rows = min(kMlaHeads, g.Hq - S.hg * kMlaHeads);
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        const int row = nt * 8 + gq;
        const __nv_bfloat16* qr = qb + static_cast<size_t>(row) * kD;
#pragma unroll
        for (int i = 0; i < kSteps; ++i) {
#pragma unroll
          for (int part = 0; part < 2; ++part) {
            const int c0 = step_col(i) + part * 8 + 2 * t4;
            float x0 = 0.f, x1 = 0.f;
            if (row < n_rows) {
              const uint32_t xv = ldg_u32(qr + c0);
              x0 = bf_lo(xv); x1 = bf_hi(xv);
              if (i == kLatSteps && use_lo) {                    // q~ = R(-delta) q on the rope band
                const int rel = c0 - kRopeOff;
                if (g.rope_style == KAM_ROPE_HALF) {
                  if (rel < half) {
                    const uint32_t yv = ldg_u32(qr + c0 + half);
                    const float2 u0 = cs[rel], u1 = cs[rel + 1];
                    x0 = fmaf(x0, u0.x, bf_lo(yv) * u0.y);
                    x1 = fmaf(x1, u1.x, bf_hi(yv) * u1.y);
                  } else {
                    const uint32_t yv = ldg_u32(qr + c0 - half);
                    const float2 u0 = cs[rel - half], u1 = cs[rel - half + 1];
                    x0 = fmaf(x0, u0.x, -bf_lo(yv) * u0.y);
                    x1 = fmaf(x1, u1.x, -bf_hi(yv) * u1.y);
                  }
                } else {
                  const float2 u0 = cs[rel >> 1];
                  const float a = x0, b = x1;
                  x0 = fmaf(a, u0.x, b * u0.y);
                  x1 = fmaf(b, u0.x, -a * u0.y);
                }
              }
            }
            const uint32_t hi = pack_bf16x2(x0, x1);
            qhi[nt][i][part] = hi;
            if (i == kLatSteps) qlo[nt][part] = pack_bf16x2(x0 - bf_lo(hi), x1 - bf_hi(hi));
          }
        }
#pragma unroll
        for (int n = 0; n < kDvTiles; ++n) { O[nt][n][0] = O[nt][n][1] = O[nt][n][2] = O[nt][n][3] = 0.f; }
        m_run[nt][0] = m_run[nt][1] = -CUDART_INF_F;
        l_run[nt][0] = l_run[nt][1] = 0.f;
      }
      if constexpr (KT > 0) {
        // ---- (W q)^T [rank][16 heads]: this warp contracts its own 9 k-steps; the four partial results meet in the
        // exchange buffer like the scores do.  TARGET frame contracts the UNrotated q, CANONICAL the rotated one.
        bool bad;
        const SegPatch sp = seg_patch(p.patches, S.patch, KT, false, &bad);
        kt_seg = sp.rank >> 4;
        W_seg = sp.Wk;
        const bool raw_q = use_lo && sp.frame != KAM_PATCH_CANONICAL_FRAME;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {                                     // kt_seg is the same in all four warps: barriers below are uniform
            float acc[2][4];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
            const __nv_bfloat16* w0 = sp.Wk + static_cast<size_t>(kt * 16 + gq) * kD + 2 * t4;
#pragma unroll
            for (int i = 0; i < kSteps; ++i) {
              const int c = step_col(i);
              const uint32_t a0 = ldg_u32(w0 + c), a1 = ldg_u32(w0 + 8 * kD + c), a2 = ldg_u32(w0 + c + 8), a3 = ldg_u32(w0 + 8 * kD + c + 8);
#pragma unroll
              for (int nt = 0; nt < 2; ++nt) {
                uint32_t b0 = qhi[nt][i][0], b1 = qhi[nt][i][1];
                if (i == kLatSteps && raw_q) {
                  const int row = nt * 8 + gq;
                  b0 = b1 = 0u;
                  if (row < n_rows) { const __nv_bfloat16* qr = qb + static_cast<size_t>(row) * kD + c + 2 * t4; b0 = ldg_u32(qr); b1 = ldg_u32(qr + 8); }
                }
                mma_bf16_16816(acc[nt][0], acc[nt][1], acc[nt][2], acc[nt][3], a0, a1, a2, a3, b0, b1);
                if (i == kLatSteps && use_lo && !raw_q) mma_bf16_16816(acc[nt][0], acc[nt][1], acc[nt][2], acc[nt][3], a0, a1, a2, a3, qlo[nt][0], qlo[nt][1]);
              }
            }
            float* xw = xch + (xbuf * kMlaWarps + warp) * 256 + lane;
#pragma unroll
            for (int nt = 0; nt < 2; ++nt)
#pragma unroll
              for (int e = 0; e < 4; ++e) xw[(nt * 4 + e) * 32] = acc[nt][e];
            named_bar_sync(1, kMlaWarps * 32);
            const float* xr = xch + xbuf * kMlaWarps * 256 + lane;
            xbuf ^= 1;
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
              float t[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) t[e] = (xr[(nt * 4 + e) * 32] + xr[256 + (nt * 4 + e) * 32]) + (xr[512 + (nt * 4 + e) * 32] + xr[768 + (nt * 4 + e) * 32]);
              const uint32_t h01 = pack_bf16x2(t[0], t[1]), h23 = pack_bf16x2(t[2], t[3]);
              const uint32_t l01 = pack_bf16x2(t[0] - bf_lo(h01), t[1] - bf_hi(h01)), l23 = pack_bf16x2(t[2] - bf_lo(h23), t[3] - bf_hi(h23));
              wqh[nt][kt][0] = movmatrix_trans(h01); wqh[nt][kt][1] = movmatrix_trans(h23);
              wql[nt][kt][0] = movmatrix_trans(l01); wql[nt][kt][1] = movmatrix_trans(l23);
              Z[nt][kt][0] = Z[nt][kt][1] = Z[nt][kt][2] = Z[nt][kt][3] = 0.f;
            }
          }
        }
      }
    }

    // ---- this warp's share of S^T[16 tokens][16 heads] = K q~^T (9 of the 36 k-steps)
    float sa[2][4], sb[2][4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) { sa[nt][0] = sa[nt][1] = sa[nt][2] = sa[nt][3] = 0.f; sb[nt][0] = sb[nt][1] = sb[nt][2] = sb[nt][3] = 0.f; }
    {
      // the asm statements are volatile (ordered as written): fragments are fetched two steps ahead of the MMAs that use them
      uint32_t a[3][4];
      ldmatrix_x4(a[0][0], a[0][1], a[0][2], a[0][3], k_addr(bb, step_col(0)));
      ldmatrix_x4(a[1][0], a[1][1], a[1][2], a[1][3], k_addr(bb, step_col(1)));
#pragma unroll
      for (int i = 0; i < kSteps; ++i) {
        if (i + 2 < kSteps) ldmatrix_x4(a[(i + 2) % 3][0], a[(i + 2) % 3][1], a[(i + 2) % 3][2], a[(i + 2) % 3][3], k_addr(bb, step_col(i + 2)));
        const uint32_t a0 = a[i % 3][0], a1 = a[i % 3][1], a2 = a[i % 3][2], a3 = a[i % 3][3];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
          if (i & 1) mma_bf16_16816(sb[nt][0], sb[nt][1], sb[nt][2], sb[nt][3], a0, a1, a2, a3, qhi[nt][i][0], qhi[nt][i][1]);
          else       mma_bf16_16816(sa[nt][0], sa[nt][1], sa[nt][2], sa[nt][3], a0, a1, a2, a3, qhi[nt][i][0], qhi[nt][i][1]);
          if (i == kLatSteps && use_lo) mma_bf16_16816(sb[nt][0], sb[nt][1], sb[nt][2], sb[nt][3], a0, a1, a2, a3, qlo[nt][0], qlo[nt][1]);
        }
      }
    }
    if constexpr (KT > 0) {
      if (kt_seg && warp == 0) {                                // s_t += U[t,:] . (W q), added once (warp 0's share)
        const uint32_t ub = bb + g.u_off + k_row * g.su_row + k_hi * 16;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t a0, a1, a2, a3;
            ldmatrix_x4(a0, a1, a2, a3, ub + kt * 32);
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
              mma_bf16_16816(sa[nt][0], sa[nt][1], sa[nt][2], sa[nt][3], a0, a1, a2, a3, wqh[nt][kt][0], wqh[nt][kt][1]);
              mma_bf16_16816(sb[nt][0], sb[nt][1], sb[nt][2], sb[nt][3], a0, a1, a2, a3, wql[nt][kt][0], wql[nt][kt][1]);
            }
          }
        }
      }
    }
    {
      float* xw = xch + (xbuf * kMlaWarps + warp) * 256 + lane;
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int e = 0; e < 4; ++e) xw[(nt * 4 + e) * 32] = sa[nt][e] + sb[nt][e];
    }
    named_bar_sync(1, kMlaWarps * 32);
    const float* xr = xch + xbuf * kMlaWarps * 256 + lane;
    xbuf ^= 1;

    // ---- online softmax, identical in the four warps (same sums in the same order)
    const bool partial = hdr.y & HDR_PARTIAL;
    const int row_lo = hdr.z & 0xff, row_hi = hdr.z >> 8;
    const bool ok0 = !partial || (gq >= row_lo && gq < row_hi);
    const bool ok1 = !partial || (gq + 8 >= row_lo && gq + 8 < row_hi);
    uint32_t pb[2][2];
    float al[2][2];
    bool rescale = false;
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      float v[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float sv = ((xr[(nt * 4 + e) * 32] + xr[256 + (nt * 4 + e) * 32]) + (xr[512 + (nt * 4 + e) * 32] + xr[768 + (nt * 4 + e) * 32])) * scale_log2;
        v[e] = ((e < 2) ? ok0 : ok1) ? sv : -CUDART_INF_F;
      }
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const float mx = col_max(fmaxf(v[e], v[2 + e]));
        // lazy rescale: the running reference only moves when the tile's max exceeds it by more than 2^8 (p stays <= 256, exact
        // enough in bf16 / fp32; l and lse are relative to the reference, so the result is unchanged) - O is rarely rescaled
        const float mn = mx > m_run[nt][e] + 8.f ? mx : m_run[nt][e];
        const float ms = (mn == -CUDART_INF_F) ? 0.f : mn;
        al[nt][e] = ex2(m_run[nt][e] - ms);
        m_run[nt][e] = mn;
        v[e] = ex2(v[e] - ms); v[2 + e] = ex2(v[2 + e] - ms);
        l_run[nt][e] = fmaf(l_run[nt][e], al[nt][e], v[e] + v[2 + e]);
        rescale |= (al[nt][e] != 1.f);
      }
      pb[nt][0] = movmatrix_trans(pack_bf16x2(v[0], v[1]));
      pb[nt][1] = movmatrix_trans(pack_bf16x2(v[2], v[3]));
    }
    if (__any_sync(0xffffffffu, rescale)) {
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
        for (int n = 0; n < kDvTiles; ++n) { O[nt][n][0] *= al[nt][0]; O[nt][n][1] *= al[nt][1]; O[nt][n][2] *= al[nt][0]; O[nt][n][3] *= al[nt][1]; }
        if constexpr (KT > 0) {
#pragma unroll
          for (int kt = 0; kt < KT; ++kt) { Z[nt][kt][0] *= al[nt][0]; Z[nt][kt][1] *= al[nt][1]; Z[nt][kt][2] *= al[nt][0]; Z[nt][kt][3] *= al[nt][1]; }
        }
      }
    }

    // ---- O^T[this warp's 128 value columns][16 heads] += V^T P^T, V = the latent columns of the same box
    if (partial) {
      // rows outside the chunk may hold anything: 0 * NaN must not reach O.  Each warp clears its own value columns (and the
      // U rows, all warps the same zeros); the other warps' score MMAs may still read those rows - their scores are masked.
      for (int idx = lane; idx < 16 * 16; idx += 32) {
        const int r = idx >> 4, j = idx & 15;                   // token row, 16-byte chunk of this warp's 128 columns
        if (r < row_lo || r >= row_hi)
          *reinterpret_cast<uint4*>(bptr + ((warp * 2 + (j >> 3)) * 16 + r) * 128 + (((j & 7) ^ (r & 7)) << 4)) = make_uint4(0, 0, 0, 0);
      }
      if constexpr (KT > 0) {
        if (kt_seg) {
          const int cpr = kt_seg * 2;
          for (int idx = lane; idx < 16 * cpr; idx += 32) {
            const int r = idx / cpr, j = idx - r * cpr;
            if (r < row_lo || r >= row_hi) *reinterpret_cast<uint4*>(bptr + g.u_off + r * g.su_row + j * 16) = make_uint4(0, 0, 0, 0);
          }
        }
      }
      __syncwarp();
    }
    {
      uint32_t a[3][4];
      ldmatrix_x4_trans(a[0][0], a[0][1], a[0][2], a[0][3], v_addr(bb, warp * 128));
      ldmatrix_x4_trans(a[1][0], a[1][1], a[1][2], a[1][3], v_addr(bb, warp * 128 + 16));
#pragma unroll
      for (int dp = 0; dp < kDvTiles; ++dp) {
        if (dp + 2 < kDvTiles) ldmatrix_x4_trans(a[(dp + 2) % 3][0], a[(dp + 2) % 3][1], a[(dp + 2) % 3][2], a[(dp + 2) % 3][3], v_addr(bb, warp * 128 + (dp + 2) * 16));
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
          mma_bf16_16816(O[nt][dp][0], O[nt][dp][1], O[nt][dp][2], O[nt][dp][3], a[dp % 3][0], a[dp % 3][1], a[dp % 3][2], a[dp % 3][3], pb[nt][0], pb[nt][1]);
      }
    }
    if constexpr (KT > 0) {
      if (kt_seg) {                                             // z^T[j][head] += U^T P^T (every warp keeps the whole z: it is tiny)
        const uint32_t ub = bb + g.u_off + v_row * g.su_row + v_hi * 16;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t a0, a1, a2, a3;
            ldmatrix_x4_trans(a0, a1, a2, a3, ub + kt * 32);
#pragma unroll
            for (int nt = 0; nt < 2; ++nt)
              mma_bf16_16816(Z[nt][kt][0], Z[nt][kt][1], Z[nt][kt][2], Z[nt][kt][3], a0, a1, a2, a3, pb[nt][0], pb[nt][1]);
          }
        }
      }
    }
    if (partial) fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[cbox]);

    if constexpr (KT > 0) {
      if ((hdr.y & HDR_LAST) && kt_seg) {
        // ---- o^T[d][head] += W[:, d]^T z^T for this warp's value columns: A[d][j] = W[j][d] gathered from global
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t bh[2][2], bl[2][2];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
              const uint32_t h01 = pack_bf16x2(Z[nt][kt][0], Z[nt][kt][1]), h23 = pack_bf16x2(Z[nt][kt][2], Z[nt][kt][3]);
              const uint32_t l01 = pack_bf16x2(Z[nt][kt][0] - bf_lo(h01), Z[nt][kt][1] - bf_hi(h01));
              const uint32_t l23 = pack_bf16x2(Z[nt][kt][2] - bf_lo(h23), Z[nt][kt][3] - bf_hi(h23));
              bh[nt][0] = movmatrix_trans(h01); bh[nt][1] = movmatrix_trans(h23);
              bl[nt][0] = movmatrix_trans(l01); bl[nt][1] = movmatrix_trans(l23);
            }
            const __nv_bfloat16* w0 = W_seg + static_cast<size_t>(kt * 16 + 2 * t4) * kD + warp * 128 + gq;
#pragma unroll
            for (int dp = 0; dp < kDvTiles; ++dp) {
              const __nv_bfloat16* w = w0 + dp * 16;
              const uint32_t a0 = ldg_u16(w) | (ldg_u16(w + kD) << 16), a1 = ldg_u16(w + 8) | (ldg_u16(w + kD + 8) << 16);
              const uint32_t a2 = ldg_u16(w + 8 * kD) | (ldg_u16(w + 9 * kD) << 16), a3 = ldg_u16(w + 8 * kD + 8) | (ldg_u16(w + 9 * kD + 8) << 16);
#pragma unroll
              for (int nt = 0; nt < 2; ++nt) {
                mma_bf16_16816(O[nt][dp][0], O[nt][dp][1], O[nt][dp][2], O[nt][dp][3], a0, a1, a2, a3, bh[nt][0], bh[nt][1]);
                mma_bf16_16816(O[nt][dp][0], O[nt][dp][1], O[nt][dp][2], O[nt][dp][3], a0, a1, a2, a3, bl[nt][0], bl[nt][1]);
              }
            }
          }
        }
      }
    }
    if (hdr.y & HDR_LAST) {
      // ---- per-(segment, head) softmax state -> partials (this warp's 128 value columns; warp 0 also the lse)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int hq = nt * 8 + 2 * t4 + e;
          const float l = col_sum(l_run[nt][e]);
          if (hq < n_rows) {
            const float inv = l > 0.f ? 1.f / l : 0.f;
            const size_t row = static_cast<size_t>(seg) * g.R + hq;
            float* po = p.part_o + row * kDv + warp * 128 + gq;
#pragma unroll
            for (int n = 0; n < kDvTiles; ++n) { po[n * 16] = O[nt][n][e] * inv; po[n * 16 + 8] = O[nt][n][2 + e] * inv; }
            if (warp == 0 && gq == 0) p.part_lse[row] = l > 0.f ? (m_run[nt][e] + log2f(l)) * 0.6931471805599453f : -CUDART_INF_F;
          }
        }
      }
    }
  }
}

namespace {
template <typename F> void mla_dispatch(const DecodeGeom& g, F&& f) {
  switch (g.KT) {
    case 0: f(kam_mla_decode_kernel<0>); break;
    case 1: f(kam_mla_decode_kernel<1>); break;
    case 2: f(kam_mla_decode_kernel<2>); break;
    default: f(kam_mla_decode_kernel<4>); break;
  }
}
}  // namespace

int mla_decode_occupancy(const DecodeGeom& g) {
  int n = 0;
  mla_dispatch(g, [&](auto kern) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, (kMlaWarps + 1) * 32, g.smem_bytes) != cudaSuccess) { cudaGetLastError(); n = 0; }
  });
  return n;
}

void launch_mla_decode(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st) {
  mla_dispatch(g, [&](auto kern) { launch_ex(kern, g.n_ctas, (kMlaWarps + 1) * 32, g.smem_bytes, pdl, st, g, p); });
}

}  // namespace kam

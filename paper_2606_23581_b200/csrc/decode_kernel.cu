// kam_paged_decode_merge: fused-on-read paged decode attention with per-chunk LSE merge.
//
//   plan    (1 CTA)      device chunk metadata -> a flat list of splits (token ranges inside one chunk), so that
//                        nothing about the batch has to be known on the host (CUDA-graph friendly)
//   decode  (persistent) one CTA per SM pulls (split, KV-head-group) work units from an atomic counter.  A producer
//                        warp resolves the block table and streams 32-token K and V tiles into shared memory with
//                        1-D bulk async copies behind an mbarrier ring that runs ACROSS work units (no drain between
//                        them); one compute warp per KV head runs QK^T and PV as m16n8k16 bf16 MMAs with the G query
//                        heads of the group as the M dimension (online softmax in fp32, exp2 domain).
//                        The cached keys are NOT rewritten: relocation is applied on read as q~ = R(-delta) q
//                        (q.(R(delta)k) = (R(-delta)q).k), carried as a bf16 hi+lo pair so that the rotation costs
//                        no precision; per (split, head) state (o, lse) goes to a partials buffer
//   merge   (B*Hq CTAs)  lse = ln sum_s e^{lse_s}; out = sum_s e^{lse_s - lse} o_s   (the paper's state merge)
//
// Decode is HBM-bound: every K and V byte is read exactly once; MMA work is G flop/byte, far below the
// legacy tensor pipe's rate, which is why mma.sync (not tcgen05/TMEM) carries it - see DESIGN.md.
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace kam {

// ---------------------------------------------------------------------------------------------------- plan
__global__ void __launch_bounds__(1024) kam_decode_plan_kernel(const int32_t* __restrict__ chunk_starts,
                                                               const long long* __restrict__ chunk_offsets,
                                                               const int32_t* __restrict__ n_chunks, int max_chunks,
                                                               int max_pages, int batch, int split_tokens, int max_splits,
                                                               DecodeItem* items, int32_t* n_items, int32_t* n_splits,
                                                               int32_t* work_counter) {
  __shared__ int scan[1024];
  __shared__ int carry;
  const int tid = threadIdx.x;
  if (tid == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < batch; base += 1024) {
    const int b = base + tid;
    int cnt = 0, nc = 0;
    const int32_t* cs = nullptr;
    if (b < batch) {
      nc = min(n_chunks[b], max_chunks);
      cs = chunk_starts + static_cast<size_t>(b) * (max_chunks + 1);
      for (int c = 0; c < nc; ++c) cnt += (cs[c + 1] - cs[c] + split_tokens - 1) / split_tokens;
      cnt = min(cnt, max_splits);
    }
    scan[tid] = cnt;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {          // inclusive Hillis-Steele scan
      const int v = tid >= off ? scan[tid - off] : 0;
      __syncthreads();
      scan[tid] += v;
      __syncthreads();
    }
    int idx = carry + scan[tid] - cnt;
    if (b < batch) {
      n_splits[b] = cnt;
      int sp = 0;
      for (int c = 0; c < nc && sp < cnt; ++c) {
        const int len = cs[c + 1] - cs[c];
        for (int o = 0; o < len && sp < cnt; o += split_tokens) {
          DecodeItem it;
          it.bt_off = static_cast<long long>(b) * max_pages;
          it.delta = chunk_offsets ? chunk_offsets[static_cast<size_t>(b) * max_chunks + c] : 0;
          it.b = b; it.chunk = c;
          it.tok0 = cs[c] - cs[0] + o;
          it.n_tok = min(split_tokens, len - o);
          it.split = sp++;
          it.ctok0 = o;
          items[idx++] = it;
        }
      }
    }
    __syncthreads();
    if (tid == 1023) carry += scan[1023];
    __syncthreads();
  }
  if (tid == 0) { *n_items = carry; *work_counter = 0; }
}

void launch_decode_plan(const int32_t* chunk_starts, const long long* chunk_offsets, const int32_t* n_chunks,
                        int32_t max_chunks, int32_t max_pages, int32_t batch, int32_t split_tokens, int32_t max_splits,
                        DecodeItem* items, int32_t* n_items, int32_t* n_splits, int32_t* work_counter, cudaStream_t st) {
  kam_decode_plan_kernel<<<1, 1024, 0, st>>>(chunk_starts, chunk_offsets, n_chunks, max_chunks, max_pages, batch,
                                             split_tokens, max_splits, items, n_items, n_splits, work_counter);
}

// ---------------------------------------------------------------------------------------------------- decode
namespace {
enum : int { HDR_FIRST = 1, HDR_LAST = 2 };

__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  return fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
}
__device__ __forceinline__ float quad_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v + __shfl_xor_sync(0xffffffffu, v, 2);
}
}  // namespace

// KS = D / 16 (k-steps of QK^T; D = Dv).  TMA: pool pages arrive as swizzled 16-token tensor-map boxes.
//
// TMA path shared-memory layout of one box: [64-column block c][token r (16)][128 bytes], SWIZZLE_128B, i.e. the 16-byte
// chunk j of (c, r) sits at (c*16 + r)*128 + ((j ^ (r & 7)) << 4): eight consecutive tokens of one chunk hit eight
// different bank groups, so ldmatrix (K) and ldmatrix.trans (V) are conflict-free without padding.  Tiles are aligned
// to 16 tokens of the page list (a box never straddles a page because P % 16 == 0); rows outside the split's token
// range are masked in the softmax.
template <int KS, bool TMA>
__global__ void __launch_bounds__((kDecMaxHG + 1) * 32, 1)
kam_paged_decode_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + g.n_stages;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_threads = blockDim.x;

  if (threadIdx.x == 0) {
    for (int s = 0; s < g.n_stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], g.HG); }
    mbar_fence_init();
  }
  // Rows beyond a tile's valid tokens are never copied; they must hold finite values (0 * NaN would poison PV).
  for (int i = threadIdx.x * 16; i < g.n_stages * g.stage_bytes; i += n_threads * 16)
    *reinterpret_cast<uint4*>(smem + g.off_stage0 + i) = make_uint4(0, 0, 0, 0);
  fence_proxy_async();
  __syncthreads();

  const int total = *p.n_items * g.n_hg;

  if (warp == g.HG) {
    // ================================================================ producer warp: schedule, slot-map, copy
    int stage = 0; uint32_t phase = 0;
    const char* pk = static_cast<const char*>(p.pool_k_layers[p.layer]);
    const char* pv = static_cast<const char*>(p.pool_v_layers[p.layer]);
    while (true) {
      int w = 0;
      if (lane == 0) w = atomicAdd(p.work_counter, 1);
      w = __shfl_sync(0xffffffffu, w, 0);
      if (w >= total) {
        mbar_wait(&empty_bar[stage], phase ^ 1);
        if (lane == 0) {
          *reinterpret_cast<int4*>(smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes + g.st_hdr) = make_int4(-1, 0, 0, 0);
          mbar_arrive(&full_bar[stage]);
        }
        break;
      }
      const int item_idx = w / g.n_hg, hg = w - item_idx * g.n_hg;
      const DecodeItem it = p.items[item_idx];
      const int32_t* bt = p.block_tables + it.bt_off;
      if constexpr (TMA) {
        const char* tm_k = static_cast<const char*>(p.tmaps) + static_cast<size_t>(p.layer) * 256;
        const char* tm_v = tm_k + 128;
        const int a0 = it.tok0 & ~15, end = it.tok0 + it.n_tok;
        const int n_tiles = (end - a0 + kDecTT - 1) / kDecTT;
        for (int t = 0; t < n_tiles; ++t) {
          const int base = a0 + t * kDecTT;
          const int n_box = min(2, (end - base + 15) >> 4);
          int slot0 = 0;
          if (lane < n_box) {
            const int tok = base + lane * 16;
            const int pg = g.P_shift >= 0 ? (tok >> g.P_shift) : tok / g.P;
            slot0 = bt[pg] * g.P + (tok - pg * g.P);
          }
          const int slot1 = __shfl_sync(0xffffffffu, slot0, 1);
          mbar_wait(&empty_bar[stage], phase ^ 1);
          if (lane == 0) {
            uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
            const int lo = max(it.tok0 - base, 0), hi = min(end - base, kDecTT);
            *reinterpret_cast<int4*>(st + g.st_hdr) = make_int4(w, t, lo | (hi << 16), (t == 0 ? HDR_FIRST : 0) | (t == n_tiles - 1 ? HDR_LAST : 0));
            mbar_arrive_expect_tx(&full_bar[stage], static_cast<uint32_t>(n_box) * g.box_bytes * 2u);
            tma_load_3d(st + g.st_k, tm_k, 0, slot0, hg * g.ncb, &full_bar[stage]);
            tma_load_3d(st + g.st_v, tm_v, 0, slot0, hg * g.ncb, &full_bar[stage]);
            if (n_box > 1) {
              tma_load_3d(st + g.st_k + g.box_bytes, tm_k, 0, slot1, hg * g.ncb, &full_bar[stage]);
              tma_load_3d(st + g.st_v + g.box_bytes, tm_v, 0, slot1, hg * g.ncb, &full_bar[stage]);
            }
          }
          if (++stage == g.n_stages) { stage = 0; phase ^= 1; }
        }
        continue;
      }
      const int n_tiles = (it.n_tok + kDecTT - 1) / kDecTT;
      const size_t off = static_cast<size_t>(hg) * g.slice_bytes;
      for (int t = 0; t < n_tiles; ++t) {
        // A1 slot mapping for the tile's 32 tokens, one per lane (issued before waiting for the stage)
        const int rel = t * kDecTT + lane;
        int slot = 0;
        if (rel < it.n_tok) {
          const int tok = it.tok0 + rel;
          const int pg = g.P_shift >= 0 ? (tok >> g.P_shift) : tok / g.P;
          slot = bt[pg] * g.P + (tok - pg * g.P);
        }
        const int nvalid = min(kDecTT, it.n_tok - t * kDecTT);
        mbar_wait(&empty_bar[stage], phase ^ 1);
        uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
        if (lane == 0) {
          *reinterpret_cast<int4*>(st + g.st_hdr) = make_int4(w, t, nvalid << 16, (t == 0 ? HDR_FIRST : 0) | (t == n_tiles - 1 ? HDR_LAST : 0));
          mbar_arrive_expect_tx(&full_bar[stage], static_cast<uint32_t>(nvalid) * g.slice_bytes * 2u);
        }
        __syncwarp();
        for (int r = 0; r < nvalid; ++r) {
          const int s = __shfl_sync(0xffffffffu, slot, r);
          if (lane == 0) {
            const size_t row = static_cast<size_t>(s) * g.row_bytes + off;
            bulk_g2s(st + g.st_k + r * g.s_row, pk + row, g.slice_bytes, &full_bar[stage]);
            bulk_g2s(st + g.st_v + r * g.s_row, pv + row, g.slice_bytes, &full_bar[stage]);
          }
        }
        if (++stage == g.n_stages) { stage = 0; phase ^= 1; }
      }
    }
    return;
  }

  // ================================================================ compute warps: one KV head each
  const int gq = lane >> 2, t4 = lane & 3;
  const int D = KS * 16;
  float2* cs_w = reinterpret_cast<float2*>(smem + g.off_warp + warp * g.warp_bytes);
  const float scale_log2 = p.sm_scale * 1.4426950408889634f;

  uint32_t qhi[KS][4], qlo[KS][4];
  float O[2 * KS][4];
  float m_run[2] = {-CUDART_INF_F, -CUDART_INF_F}, l_run[2] = {0.f, 0.f};
  bool use_lo = false;
  int item_b = 0, item_split = 0, head = 0;

  // ldmatrix lane addressing inside a stage (bytes relative to the K / V region)
  //   K (non-trans): matrices = (tokens 0-7 | 8-15 of a 16-token block) x (first | second 16-byte chunk of the k-step)
  //   V (trans):     matrices = (tokens 0-7 | 8-15) x (first | second d n-tile of the pair)
  const int k_row = (lane & 7) + ((lane >> 4) & 1) * 8, k_hi = (lane >> 3) & 1;
  const int v_row = (lane & 7) + ((lane >> 3) & 1) * 8, v_hi = (lane >> 4) & 1;
  const uint32_t k_lane = TMA ? (warp * (D / 64) * 16 + k_row) * 128 : k_row * g.s_row + warp * D * 2 + k_hi * 16;
  const uint32_t v_lane = TMA ? (warp * (D / 64) * 16 + v_row) * 128 : v_row * g.s_row + warp * D * 2 + v_hi * 16;
  const uint32_t k_sw = (k_hi ^ (lane & 7)) << 4, v_sw = (v_hi ^ (lane & 7)) << 4;   // swizzled chunk of k-step 0
  const uint32_t blk16 = TMA ? g.box_bytes : 16 * g.s_row;                            // bytes between 16-token blocks

  int stage = 0; uint32_t phase = 0;
  while (true) {
    mbar_wait(&full_bar[stage], phase);
    const uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
    const int4 hdr = *reinterpret_cast<const int4*>(st + g.st_hdr);
    if (hdr.x < 0) break;
    const int row_lo = hdr.z & 0xffff, row_hi = hdr.z >> 16;        // valid token rows of this tile

    if (hdr.w & HDR_FIRST) {
      // ---- new work unit: load the G query rows of this KV head, rotate them by -delta, split into bf16 hi + lo
      const int item_idx = hdr.x / g.n_hg, hg = hdr.x - item_idx * g.n_hg;
      const DecodeItem it = p.items[item_idx];
      item_b = it.b; item_split = it.split;
      head = hg * g.HG + warp;
      use_lo = (it.delta != 0) && g.d_r > 0;
      const int half = g.d_r >> 1;
      if (use_lo) {
        for (int i = lane; i < half; i += 32) {
          const double f = pow(g.theta, -2.0 * i / g.d_r);
          double s, c;
          sincos(static_cast<double>(it.delta) * f, &s, &c);
          cs_w[i] = make_float2(static_cast<float>(c), static_cast<float>(s));
        }
        __syncwarp();
      }
      const __nv_bfloat16* qb = static_cast<const __nv_bfloat16*>(p.q) + (static_cast<size_t>(it.b) * g.Hq + static_cast<size_t>(head) * g.G) * D;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
#pragma unroll
        for (int part = 0; part < 2; ++part) {
          const int c0 = ks * 16 + part * 8 + 2 * t4;
#pragma unroll
          for (int rs = 0; rs < 2; ++rs) {
            const int row = gq + rs * 8;
            float x0 = 0.f, x1 = 0.f;
            if (row < g.G) {
              const __nv_bfloat16* qr = qb + static_cast<size_t>(row) * D;
              const uint32_t xv = *reinterpret_cast<const uint32_t*>(qr + c0);
              x0 = bf_lo(xv); x1 = bf_hi(xv);
              const int rel = c0 - g.rope_off;
              if (use_lo && rel >= 0 && rel < g.d_r) {
                // q~ = R(-delta) q : with (c, s) = (cos, sin)(delta f):  a' = a c + b s ,  b' = -a s + b c
                if (g.rope_style == KAM_ROPE_HALF) {
                  if (rel < half) {
                    const uint32_t yv = *reinterpret_cast<const uint32_t*>(qr + c0 + half);
                    const float2 t0 = cs_w[rel], t1 = cs_w[rel + 1];
                    x0 = fmaf(x0, t0.x, bf_lo(yv) * t0.y);
                    x1 = fmaf(x1, t1.x, bf_hi(yv) * t1.y);
                  } else {
                    const uint32_t yv = *reinterpret_cast<const uint32_t*>(qr + c0 - half);
                    const float2 t0 = cs_w[rel - half], t1 = cs_w[rel - half + 1];
                    x0 = fmaf(x0, t0.x, -bf_lo(yv) * t0.y);
                    x1 = fmaf(x1, t1.x, -bf_hi(yv) * t1.y);
                  }
                } else {
                  const float2 t0 = cs_w[rel >> 1];
                  const float a = x0, b = x1;
                  x0 = fmaf(a, t0.x, b * t0.y);
                  x1 = fmaf(b, t0.x, -a * t0.y);
                }
              }
            }
            const uint32_t hi = pack_bf16x2(x0, x1);
            qhi[ks][part * 2 + rs] = hi;
            qlo[ks][part * 2 + rs] = pack_bf16x2(x0 - bf_lo(hi), x1 - bf_hi(hi));
          }
        }
      }
#pragma unroll
      for (int n = 0; n < 2 * KS; ++n) { O[n][0] = O[n][1] = O[n][2] = O[n][3] = 0.f; }
      m_run[0] = m_run[1] = -CUDART_INF_F;
      l_run[0] = l_run[1] = 0.f;
    }

    // ---- S = q~ K^T for 32 tokens (4 n-tiles)
    float S[4][4];
#pragma unroll
    for (int n = 0; n < 4; ++n) { S[n][0] = S[n][1] = S[n][2] = S[n][3] = 0.f; }
    const uint32_t kb = smem_u32(st + g.st_k) + k_lane;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
#pragma unroll
      for (int np = 0; np < 2; ++np) {
        uint32_t b0, b1, b2, b3;
        // chunk index of this k-step inside its 64-column block: (ks & 3) * 2 (+ k_hi), XOR-swizzled on the TMA path
        ldmatrix_x4(b0, b1, b2, b3, TMA ? kb + np * blk16 + (ks >> 2) * 2048 + (k_sw ^ ((ks & 3) << 5))
                                        : kb + np * blk16 + ks * 32);
        mma_bf16_16816(S[2 * np][0], S[2 * np][1], S[2 * np][2], S[2 * np][3], qhi[ks][0], qhi[ks][1], qhi[ks][2], qhi[ks][3], b0, b1);
        mma_bf16_16816(S[2 * np + 1][0], S[2 * np + 1][1], S[2 * np + 1][2], S[2 * np + 1][3], qhi[ks][0], qhi[ks][1], qhi[ks][2], qhi[ks][3], b2, b3);
        if (use_lo) {
          mma_bf16_16816(S[2 * np][0], S[2 * np][1], S[2 * np][2], S[2 * np][3], qlo[ks][0], qlo[ks][1], qlo[ks][2], qlo[ks][3], b0, b1);
          mma_bf16_16816(S[2 * np + 1][0], S[2 * np + 1][1], S[2 * np + 1][2], S[2 * np + 1][3], qlo[ks][0], qlo[ks][1], qlo[ks][2], qlo[ks][3], b2, b3);
        }
      }
    }
    // ---- online softmax (exp2 domain), rows gq and gq + 8
    float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
#pragma unroll
    for (int n = 0; n < 4; ++n) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int tr = n * 8 + 2 * t4 + e;
        const bool ok = tr >= row_lo && tr < row_hi;
        S[n][e] = ok ? S[n][e] * scale_log2 : -CUDART_INF_F;
        S[n][2 + e] = ok ? S[n][2 + e] * scale_log2 : -CUDART_INF_F;
        mx0 = fmaxf(mx0, S[n][e]); mx1 = fmaxf(mx1, S[n][2 + e]);
      }
    }
    mx0 = quad_max(mx0); mx1 = quad_max(mx1);
    const float mn0 = fmaxf(m_run[0], mx0), mn1 = fmaxf(m_run[1], mx1);
    const float ms0 = (mn0 == -CUDART_INF_F) ? 0.f : mn0, ms1 = (mn1 == -CUDART_INF_F) ? 0.f : mn1;
    const float al0 = exp2f(m_run[0] - ms0), al1 = exp2f(m_run[1] - ms1);
    m_run[0] = mn0; m_run[1] = mn1;
    float ps0 = 0.f, ps1 = 0.f;
#pragma unroll
    for (int n = 0; n < 4; ++n) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        S[n][e] = exp2f(S[n][e] - ms0); ps0 += S[n][e];
        S[n][2 + e] = exp2f(S[n][2 + e] - ms1); ps1 += S[n][2 + e];
      }
    }
    l_run[0] = l_run[0] * al0 + ps0; l_run[1] = l_run[1] * al1 + ps1;
#pragma unroll
    for (int n = 0; n < 2 * KS; ++n) { O[n][0] *= al0; O[n][1] *= al0; O[n][2] *= al1; O[n][3] *= al1; }
    // ---- O += P V
    const uint32_t vb = smem_u32(st + g.st_v) + v_lane;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const uint32_t pa0 = pack_bf16x2(S[2 * j][0], S[2 * j][1]), pa1 = pack_bf16x2(S[2 * j][2], S[2 * j][3]);
      const uint32_t pa2 = pack_bf16x2(S[2 * j + 1][0], S[2 * j + 1][1]), pa3 = pack_bf16x2(S[2 * j + 1][2], S[2 * j + 1][3]);
#pragma unroll
      for (int dp = 0; dp < KS; ++dp) {
        uint32_t v0, v1, v2, v3;
        ldmatrix_x4_trans(v0, v1, v2, v3, TMA ? vb + j * blk16 + (dp >> 2) * 2048 + (v_sw ^ ((dp & 3) << 5))
                                              : vb + j * blk16 + dp * 32);
        mma_bf16_16816(O[2 * dp][0], O[2 * dp][1], O[2 * dp][2], O[2 * dp][3], pa0, pa1, pa2, pa3, v0, v1);
        mma_bf16_16816(O[2 * dp + 1][0], O[2 * dp + 1][1], O[2 * dp + 1][2], O[2 * dp + 1][3], pa0, pa1, pa2, pa3, v2, v3);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[stage]);          // the stage's shared memory is no longer read below
    if (++stage == g.n_stages) { stage = 0; phase ^= 1; }

    if (hdr.w & HDR_LAST) {
      // ---- per-(split, head) softmax state -> partials: o normalised, lse in natural log
      const float l0 = quad_sum(l_run[0]), l1 = quad_sum(l_run[1]);
      const float inv0 = l0 > 0.f ? 1.f / l0 : 0.f, inv1 = l1 > 0.f ? 1.f / l1 : 0.f;
#pragma unroll
      for (int rs = 0; rs < 2; ++rs) {
        const int row = gq + rs * 8;
        if (row < g.G) {
          const size_t slot = (static_cast<size_t>(item_b) * g.Hq + static_cast<size_t>(head) * g.G + row) * p.max_splits + item_split;
          float* po = p.part_o + slot * g.Dv + 2 * t4;
          const float inv = rs ? inv1 : inv0;
#pragma unroll
          for (int n = 0; n < 2 * KS; ++n)
            *reinterpret_cast<float2*>(po + n * 8) = make_float2(O[n][2 * rs] * inv, O[n][2 * rs + 1] * inv);
          if (t4 == 0) {
            const float l = rs ? l1 : l0, m = rs ? m_run[1] : m_run[0];
            p.part_lse[slot] = l > 0.f ? (m + log2f(l)) * 0.6931471805599453f : -CUDART_INF_F;
          }
        }
      }
    }
  }
}

void launch_decode(const DecodeGeom& g, const DecodeParams& p, int grid, cudaStream_t st) {
  const int threads = (g.HG + 1) * 32;
  auto go = [&](auto kern) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    kern<<<grid, threads, g.smem_bytes, st>>>(g, p);
  };
  if (g.D == 128) { if (g.use_tma) go(kam_paged_decode_kernel<8, true>); else go(kam_paged_decode_kernel<8, false>); }
  else            { if (g.use_tma) go(kam_paged_decode_kernel<4, true>); else go(kam_paged_decode_kernel<4, false>); }
}

// ---------------------------------------------------------------------------------------------------- merge
// A9: lse = ln sum_s e^{lse_s};  out = sum_s e^{lse_s - lse} o_s.  Fixed summation order => run-to-run deterministic.
__global__ void __launch_bounds__(128) kam_lse_merge_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  const int bh = blockIdx.x;                      // b * Hq + hq
  const int b = bh / g.Hq;
  const int ns = p.n_splits[b];
  const float* pl = p.part_lse + static_cast<size_t>(bh) * p.max_splits;
  const float* po = p.part_o + static_cast<size_t>(bh) * p.max_splits * g.Dv;
  float m = -CUDART_INF_F;
  for (int s = 0; s < ns; ++s) m = fmaxf(m, pl[s]);
  __nv_bfloat16* out = static_cast<__nv_bfloat16*>(p.out) + static_cast<size_t>(bh) * g.Dv;
  if (m == -CUDART_INF_F) {                       // no tokens at all: out = 0, lse = -inf, no NaN
    for (int c = threadIdx.x; c < g.Dv; c += blockDim.x) out[c] = __float2bfloat16_rn(0.f);
    if (threadIdx.x == 0) p.lse[bh] = -CUDART_INF_F;
    return;
  }
  float tot = 0.f;
  for (int s = 0; s < ns; ++s) tot += __expf(pl[s] - m);
  const float inv = 1.f / tot;
  for (int c = threadIdx.x; c < g.Dv; c += blockDim.x) {
    float acc = 0.f;
    for (int s = 0; s < ns; ++s) acc = fmaf(__expf(pl[s] - m), po[static_cast<size_t>(s) * g.Dv + c], acc);
    out[c] = __float2bfloat16_rn(acc * inv);
  }
  if (threadIdx.x == 0) p.lse[bh] = m + logf(tot);
}

void launch_decode_merge(const DecodeGeom& g, const DecodeParams& p, cudaStream_t st) {
  kam_lse_merge_kernel<<<p.batch * g.Hq, 128, 0, st>>>(g, p);
}

}  // namespace kam

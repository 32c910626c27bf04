// kam_paged_decode_merge: fused-on-read paged decode attention with per-chunk LSE merge.
//
//   plan    (1 + n CTAs)  device chunk metadata -> the flat list of 16-token tiles (head group x request x chunk x tile)
//                         is cut into one equal contiguous range per persistent CTA; a range is a list of SEGMENTS (runs
//                         of tiles inside one chunk).  Everything is computed on the device from device metadata, so a
//                         call never needs the batch on the host (CUDA-graph friendly).  The other CTAs of the launch
//                         write the per-chunk (cos, sin)(delta f_i) tables, fp64 sincos, once for all layers.
//   decode  (persistent)  2-3 CTAs per SM, each = 1 producer warp + one compute warp per KV head of the head group.  The
//                         producer resolves the block table and streams 16-token K and V boxes through a ring of
//                         mbarrier-guarded shared-memory boxes with TMA tensor-map loads (cp.async.bulk.tensor, 128-byte
//                         swizzle); the ring runs ACROSS segments.  A compute warp owns one KV head: S^T = K q~^T and
//                         O^T += V^T P^T as m16n8k16 bf16 MMAs with the TOKENS / head-dim as the M dimension and the (<= 8)
//                         query heads of the group as N - no MMA rows are wasted on padding and the accumulators of a
//                         128-wide head are 32 registers.  Online softmax in fp32 (exp2 domain); P^T goes from the
//                         accumulator layout to the B-operand layout with one movmatrix.trans per 8 tokens.
//                         The cached keys are NOT rewritten: relocation is applied on read as q~ = R(-delta) q
//                         (q.(R(delta)k) = (R(-delta)q).k), carried as a bf16 hi+lo pair so the rotation costs no
//                         precision.  Per (segment, query head) state (o, lse) goes to a partials buffer.
//   merge   (B*Hq CTAs)   lse = ln sum_s e^{lse_s}; out = sum_s e^{lse_s - lse} o_s   (the paper's state merge)
//
// Decode is HBM-bound: every K and V byte is read exactly once.  MMA work is 2 HMMA per 16 tokens x 16 dims, a few percent
// of the legacy tensor pipe, which is why mma.sync (not tcgen05/TMEM, whose M is 64/128) carries it - see DESIGN.md.
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "decode_common.cuh"
#include "internal.h"

namespace kam {

// ---------------------------------------------------------------------------------------------------- plan
namespace {

// Exclusive prefix sum of data[0, M) in place; data[M] = total (also returned).  One block, any M.
__device__ int block_excl_scan(int32_t* data, int M, int* sh) {
  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int per = (M + T - 1) / T;
  const int lo = min(M, tid * per), hi = min(M, lo + per);
  int local = 0;
  for (int i = lo; i < hi; ++i) local += data[i];
  int inc = local;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, inc, off);
    if (lane >= off) inc += v;
  }
  if (lane == 31) sh[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int v = lane < (T >> 5) ? sh[lane] : 0;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, v, off);
      if (lane >= off) v += u;
    }
    sh[lane] = v;                                  // inclusive totals of the warps
  }
  __syncthreads();
  int run = inc - local + (warp ? sh[warp - 1] : 0);
  const int total = sh[(T >> 5) - 1];
  for (int i = lo; i < hi; ++i) { const int v = data[i]; data[i] = run; run += v; }
  if (tid == 0) data[M] = total;
  __syncthreads();
  return total;
}

__device__ __forceinline__ long long ceil_div_ll(long long a, long long b) { return (a + b - 1) / b; }

struct SegCut { long long g0, g1, i_lo; int nseg; };
// Chunk j of head group hg covers global tiles [g0, g1); CTA i starts at tile s_i = i * total / n_eff.
__device__ __forceinline__ SegCut seg_cut(int hg, int j, const int32_t* tile_pre, long long total_hg, long long total, long long n_eff) {
  SegCut c;
  c.g0 = hg * total_hg + tile_pre[j];
  c.g1 = hg * total_hg + tile_pre[j + 1];
  c.nseg = 0; c.i_lo = 0;
  if (c.g1 > c.g0) {
    c.i_lo = ceil_div_ll((c.g0 + 1) * n_eff, total);            // smallest i with s_i > g0
    const long long i_hi = ceil_div_ll(c.g1 * n_eff, total);    // smallest i with s_i >= g1
    c.nseg = 1 + static_cast<int>(max(0ll, i_hi - c.i_lo));
  }
  return c;
}

}  // namespace

__global__ void __launch_bounds__(kDecPlanThreads) kam_decode_plan_kernel(const __grid_constant__ DecodeGeom g,
                                                                          const __grid_constant__ DecodePlan pl,
                                                                          const __grid_constant__ DecodeCsr csr) {
  __shared__ int sh[32];
  const int tid = threadIdx.x;
  const int N = pl.n_chunks;
  grid_dep_launch();                                            // the decode kernel may set itself up while this one runs

  if (blockIdx.x > 0) {
    // ---- A2 for decode: (cos, sin)(delta f_i) per (chunk, frequency); the angle is formed in fp64 (R-18)
    const int half = g.d_r >> 1;
    const long long n = static_cast<long long>(N) * half;
    for (long long idx = static_cast<long long>(blockIdx.x - 1) * blockDim.x + tid; idx < n; idx += static_cast<long long>(gridDim.x - 1) * blockDim.x) {
      const int j = static_cast<int>(idx / half), i = static_cast<int>(idx - static_cast<long long>(j) * half);
      long long delta;
      if (csr.enabled) {
        const int b = j / csr.max_chunks, c = j - b * csr.max_chunks;
        delta = (csr.chunk_offsets && c < csr.n_chunks[b]) ? csr.chunk_offsets[j] : 0;
      } else {
        delta = pl.chunks[j].delta;
      }
      if (delta != 0) {
        double s, c;
        sincos(static_cast<double>(delta) * pl.inv_freq[i], &s, &c);
        pl.cs[idx] = make_float2(static_cast<float>(c), static_cast<float>(s));
      }
    }
    return;
  }

  if (tid == 0) pl.dyn[0] = N;
  // ---- phase 0: chunk records of the stateless call (CSR token boundaries per request)
  if (csr.enabled) {
    for (int j = tid; j < N; j += blockDim.x) {
      const int b = j / csr.max_chunks, c = j - b * csr.max_chunks;
      const int32_t* cs = csr.chunk_starts + static_cast<size_t>(b) * (csr.max_chunks + 1);
      const int nc = min(csr.n_chunks[b], csr.max_chunks);
      DecChunk ch;
      ch.bt_off = static_cast<long long>(b) * csr.max_pages;
      ch.delta = 0; ch.b = b; ch.tok0 = 0; ch.n_tok = 0; ch.patch = -1;
      if (c < nc) {
        ch.tok0 = cs[c] - cs[0];
        ch.n_tok = max(0, cs[c + 1] - cs[c]);
        ch.delta = csr.chunk_offsets ? csr.chunk_offsets[j] : 0;
        ch.patch = csr.has_patches ? j : -1;
      }
      pl.chunks[j] = ch;
    }
    for (int b = tid; b <= pl.batch; b += blockDim.x) pl.rcb[b] = b * csr.max_chunks;
    __syncthreads();
  }

  // ---- phase 1: 16-token tiles per chunk (tiles are aligned to the page list, so a box never straddles a page)
  for (int j = tid; j < N; j += blockDim.x) {
    const DecChunk& ch = pl.chunks[j];
    pl.tile_pre[j] = ch.n_tok > 0 ? ((ch.tok0 + ch.n_tok + kDecTile - 1) / kDecTile) - (ch.tok0 / kDecTile) : 0;
  }
  __syncthreads();
  const long long total_hg = block_excl_scan(pl.tile_pre, N, sh);
  const long long total = total_hg * g.n_hg;
  const long long n_eff = min(static_cast<long long>(g.n_ctas), total);
  const int M = g.n_hg * N;

  // ---- phase 2: segments per (head group, chunk) = 1 + CTA cuts strictly inside it
  for (int e = tid; e < M; e += blockDim.x) {
    const int hg = e / N, j = e - hg * N;
    pl.seg_base[e] = total ? seg_cut(hg, j, pl.tile_pre, total_hg, total, n_eff).nseg : 0;
  }
  __syncthreads();
  const int n_segs = block_excl_scan(pl.seg_base, M, sh);

  // ---- phase 3: emit the segments and each CTA's first segment
  for (int i = tid; i <= g.n_ctas; i += blockDim.x)
    if (i >= n_eff) pl.cta_seg[i] = n_segs;
  for (int e = tid; e < M; e += blockDim.x) {
    if (!total) break;
    const int hg = e / N, j = e - hg * N;
    const SegCut c = seg_cut(hg, j, pl.tile_pre, total_hg, total, n_eff);
    if (c.nseg == 0) continue;
    const DecChunk ch = pl.chunks[j];
    const int base = pl.seg_base[e];
    for (int k = 0; k < c.nseg; ++k) {
      const long long start = k == 0 ? c.g0 : ((c.i_lo + k - 1) * total) / n_eff;
      const long long end = k == c.nseg - 1 ? c.g1 : ((c.i_lo + k) * total) / n_eff;
      DecSeg s;
      s.bt_off = ch.bt_off; s.chunk = j; s.b = ch.b; s.hg = hg;
      s.tile0 = ch.tok0 / kDecTile + static_cast<int>(start - c.g0);
      s.n_tiles = static_cast<int>(end - start);
      s.tok_lo = ch.tok0; s.tok_hi = ch.tok0 + ch.n_tok;
      s.rotate = (ch.delta != 0) && g.d_r > 0;
      s.patch = ch.patch;
      {
        const int tok = s.tile0 * kDecTile;
        const int pg = g.P_shift >= 0 ? (tok >> g.P_shift) : tok / g.P;
        s.slot0 = pl.block_tables[ch.bt_off + pg] * g.P + (tok - pg * g.P);
      }
      pl.segs[base + k] = s;
      const long long i = k == 0 ? ceil_div_ll(start * n_eff, total) : c.i_lo + k - 1;   // the CTA starting exactly here, if any
      if (i < n_eff && (i * total) / n_eff == start) pl.cta_seg[i] = base + k;
    }
  }
}

void launch_decode_plan(const DecodeGeom& g, const DecodePlan& plan, const DecodeCsr& csr, cudaStream_t st) {
  const long long n_cs = static_cast<long long>(plan.n_chunks) * (g.d_r / 2);
  const int cs_blocks = static_cast<int>(min(64ll, (n_cs + kDecPlanThreads - 1) / kDecPlanThreads));
  kam_decode_plan_kernel<<<1 + cs_blocks, kDecPlanThreads, 0, st>>>(g, plan, csr);
}

// ---------------------------------------------------------------------------------------------------- decode

// KS = D / 16 (k-steps of QK^T; D = Dv).  NT = ceil(G / 8) query-head tiles.  TMA: pool pages arrive as swizzled boxes.
//
// Box layout, TMA path: [64-column block c][token r (16)][128 bytes], SWIZZLE_128B: the 16-byte chunk j of (c, r) sits at
// (c*16 + r)*128 + ((j ^ (r & 7)) << 4), so eight consecutive tokens of one chunk column hit eight different bank groups
// and ldmatrix (K) / ldmatrix.trans (V) are conflict-free without padding.  Bulk-copy path: [token r][s_row bytes], s_row
// padded so that (s_row / 16) is odd.  Tiles are aligned to 16 tokens of the page list (P % 16 == 0 on the TMA path, so a
// box never straddles a page); rows outside the chunk's token range are masked in the softmax and zeroed in V.
//
// KT > 0: on-read patch (Eq. 1 applied to what is read; the pool is never written).  Behind the K rows of a box rides the
// tile's U_k rows, behind the V rows its U_v rows ([16 tokens][su_row bytes], one run of `rank` values per KV head).  With
// wq = W_k q (per segment, m x G, carried as bf16 hi + lo):   s_t += U_k[t,:] . wq          (rank/16 MMAs per tile)
// and z += U_v^T P^T accumulated like O (rank/16 MMAs per tile); at the end of the segment o += W_v^T z.
template <int KS, int NT, bool TMA, int KT>
__global__ void __launch_bounds__((kDecMaxHG + 1) * 32, (NT == 1 && KT == 0) ? 3 : (NT == 1 ? 2 : 1))
kam_paged_decode_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + g.n_boxes;
  int4* hdrs = reinterpret_cast<int4*>(smem + g.off_hdr);
  uint8_t* box0 = smem + g.off_box0;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < g.n_boxes; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], g.HG); }
    mbar_fence_init();
  }
  __syncthreads();

  grid_dep_launch();
  if (p.plan_fresh) grid_dep_wait();                             // the plan comes from the kernel right before this one
  const int seg_begin = p.plan.cta_seg[blockIdx.x], seg_end = p.plan.cta_seg[blockIdx.x + 1];
  if (seg_begin >= seg_end) return;

  if (warp == g.HG) {
    // ================================================================ producer warp: slot-map (A1), stream K / V boxes
    int box = 0; uint32_t phase = 0;
    const char* pk = static_cast<const char*>(p.pool_k_layers[p.layer]);
    const char* pv = static_cast<const char*>(p.pool_v_layers[p.layer]);
    const char* tm_k = static_cast<const char*>(p.tmaps) + static_cast<size_t>(p.layer) * kTmapLayerBytes;
    const char* tm_v = tm_k + 128;
    DecSeg S_next = p.plan.segs[seg_begin];
    grid_dep_wait();                                            // nothing of the pool is read before the stream's earlier work is done
    for (int seg = seg_begin; seg < seg_end; ++seg) {
      const DecSeg S = S_next;
      if (seg + 1 < seg_end) S_next = p.plan.segs[seg + 1];     // in flight while this segment streams
      const int32_t* bt = p.block_tables + S.bt_off;
      const size_t col_off = static_cast<size_t>(S.hg) * g.slice_bytes;
      [[maybe_unused]] SegPatch sp{};
      [[maybe_unused]] uint32_t u_row_bytes = 0, u_run_bytes = 0; [[maybe_unused]] int u_runs = 0;
      if constexpr (KT > 0) {
        bool bad;
        sp = seg_patch(p.patches, S.patch, KT, true, &bad);
        if (bad && lane == 0 && S.tile0 * kDecTile <= S.tok_lo && S.hg == 0) atomicAdd(p.err, 1);   // once per chunk
        if (sp.rank) {
          // a token's U run of this head group: HG heads x rank (one copy if the heads are contiguous), or rank (shared U)
          const int nh = sp.uhs == 0 ? 1 : g.HG;
          const bool one = nh == 1 || sp.uhs == sp.rank;
          u_runs = one ? 1 : nh;
          u_run_bytes = static_cast<uint32_t>((one ? nh : 1) * sp.rank * 2);
          u_row_bytes = static_cast<uint32_t>(nh * sp.rank * 2);
        }
      }
      for (int t0 = 0; t0 < S.n_tiles; t0 += 32) {
        int slot = 0;
        if (t0 + lane < S.n_tiles && t0 + lane > 0) {           // A1: page = block_table[tok / P], slot = page * P + tok % P
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
          int rslot = 0;
          if constexpr (!TMA) {                                 // any page size: every row of the tile is slot-mapped
            if (lane >= row_lo && lane < row_hi) {
              const int tk = tok + lane;
              const int pg = g.P_shift >= 0 ? (tk >> g.P_shift) : tk / g.P;
              rslot = bt[pg] * g.P + (tk - pg * g.P);
            }
          }
#pragma unroll
          for (int kv = 0; kv < 2; ++kv) {
            mbar_wait(&empty_bar[box], phase ^ 1);
            uint8_t* dst = box0 + static_cast<size_t>(box) * g.box_bytes;
            const uint32_t u_bytes = static_cast<uint32_t>(row_hi - row_lo) * u_row_bytes;      // 0 without a patch
            if (lane == 0) {
              if (kv == 0) {
                const int flags = (tl == 0 ? HDR_FIRST : 0) | (tl == S.n_tiles - 1 ? HDR_LAST : 0) |
                                  ((row_lo > 0 || row_hi < kDecTile) ? HDR_PARTIAL : 0);
                hdrs[box] = make_int4(seg, flags, row_lo | (row_hi << 8), tok - S.tok_lo);
              }
              if constexpr (TMA) {
                mbar_arrive_expect_tx(&full_bar[box], static_cast<uint32_t>(g.kv_bytes) + u_bytes);
                tma_load_3d(dst, kv ? tm_v : tm_k, 0, s0, S.hg * g.ncb, &full_bar[box]);
              } else {
                mbar_arrive_expect_tx(&full_bar[box], static_cast<uint32_t>(row_hi - row_lo) * g.slice_bytes + u_bytes);
              }
            }
            if constexpr (KT > 0) {
              if (u_bytes) {                                       // lane r copies token row r's U run(s): chunk-local token tok - tok_lo + r
                __syncwarp();
                if (lane >= row_lo && lane < row_hi) {
                  const char* src = (kv ? sp.Uv : sp.Uk) +
                                    ((static_cast<long long>(tok - S.tok_lo + lane)) * sp.uts + static_cast<long long>(S.hg) * g.HG * sp.uhs) * 2;
                  uint8_t* ud = dst + g.u_off + lane * g.su_row;
                  for (int r = 0; r < u_runs; ++r) bulk_g2s(ud + r * sp.rank * 2, src + r * sp.uhs * 2, u_run_bytes, &full_bar[box]);
                }
              }
            }
            if constexpr (!TMA) {
              const char* src = (kv ? pv : pk) + col_off;
              for (int r = row_lo; r < row_hi; ++r) {
                const int sr = __shfl_sync(0xffffffffu, rslot, r);
                if (lane == 0) bulk_g2s(dst + r * g.s_row, src + static_cast<size_t>(sr) * g.row_bytes, g.slice_bytes, &full_bar[box]);
              }
            }
            if (++box == g.n_boxes) { box = 0; phase ^= 1; }
          }
        }
      }
    }
    mbar_wait(&empty_bar[box], phase ^ 1);
    if (lane == 0) { hdrs[box] = make_int4(-1, 0, 0, 0); mbar_arrive(&full_bar[box]); }
    return;
  }

  // ================================================================ compute warps: one KV head each
  const int gq = lane >> 2, t4 = lane & 3;
  constexpr int D = KS * 16;
  const float scale_log2 = p.sm_scale * 1.4426950408889634f;

  uint32_t qhi[NT][KS][2], qlo[NT][KS][2];
  float O[NT][KS][4];
  float m_run[NT][2], l_run[NT][2];
  bool use_lo = false;
  constexpr int KTA = KT > 0 ? KT : 1;
  [[maybe_unused]] uint32_t wqh[NT][KTA][2], wql[NT][KTA][2];     // (W_k q)^T as the B operand of the score MMA, bf16 hi + lo
  [[maybe_unused]] float Z[NT][KTA][4];                           // z^T[j][head] = sum_t p_t U_v[t][j]
  [[maybe_unused]] int kt_seg = 0;                                // rank / 16 of this segment's patch (0: none)
  [[maybe_unused]] const __nv_bfloat16* Wv_seg = nullptr;
  [[maybe_unused]] uint32_t u_head_off = 0;                       // bytes: this warp's KV head inside a U row

  // ldmatrix lane addressing inside a box (bytes)
  //   K (A operand, rows = tokens): matrices (tokens 0-7 | 8-15) x (first | second 16-byte chunk of the k-step)
  //   V (A operand via .trans, rows = head dims): matrices (first | second d chunk) x (tokens 0-7 | 8-15)
  const int k_row = (lane & 7) + ((lane >> 3) & 1) * 8, k_hi = lane >> 4;
  const int v_row = (lane & 7) + (lane >> 4) * 8, v_hi = (lane >> 3) & 1;
  const uint32_t k_lane = TMA ? (warp * (D / 64) * 16 + k_row) * 128 : k_row * g.s_row + warp * D * 2 + k_hi * 16;
  const uint32_t v_lane = TMA ? (warp * (D / 64) * 16 + v_row) * 128 : v_row * g.s_row + warp * D * 2 + v_hi * 16;
  const uint32_t k_sw = (k_hi ^ (lane & 7)) << 4, v_sw = (v_hi ^ (lane & 7)) << 4;   // swizzled chunk of step 0

  int box = 0; uint32_t phase = 0;
  int seg = 0;
  grid_dep_wait();                                              // q and the partials buffer belong to earlier work until here
  while (true) {
    mbar_wait(&full_bar[box], phase);
    const int4 hdr = hdrs[box];
    if (hdr.x < 0) break;
    const uint32_t kb = smem_u32(box0 + static_cast<size_t>(box) * g.box_bytes) + k_lane;
    const int kbox = box;
    if (++box == g.n_boxes) { box = 0; phase ^= 1; }

    if (hdr.y & HDR_FIRST) {
      // ---- new segment: the G query rows of this KV head, rotated by -delta (A8), split into bf16 hi + lo
      seg = hdr.x;
      const DecSeg S = p.plan.segs[seg];
      const int head = S.hg * g.HG + warp;
      use_lo = S.rotate;
      const int half = g.d_r >> 1;
      const float2* cs = p.plan.cs + static_cast<size_t>(S.chunk) * half;
      const __nv_bfloat16* qb = static_cast<const __nv_bfloat16*>(p.q) + (static_cast<size_t>(S.b) * g.Hq + static_cast<size_t>(head) * g.G) * D;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const int row = nt * 8 + gq;                              // query head inside the group = column of S^T
        const __nv_bfloat16* qr = qb + static_cast<size_t>(row) * D;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
#pragma unroll
          for (int part = 0; part < 2; ++part) {
            const int c0 = ks * 16 + part * 8 + 2 * t4;
            float x0 = 0.f, x1 = 0.f;
            if (row < g.G) {
              const uint32_t xv = *reinterpret_cast<const uint32_t*>(qr + c0);
              x0 = bf_lo(xv); x1 = bf_hi(xv);
              const int rel = c0 - g.rope_off;
              if (use_lo && rel >= 0 && rel < g.d_r) {
                // q~ = R(-delta) q : with (c, s) = (cos, sin)(delta f):  a' = a c + b s ,  b' = -a s + b c
                if (g.rope_style == KAM_ROPE_HALF) {
                  if (rel < half) {
                    const uint32_t yv = *reinterpret_cast<const uint32_t*>(qr + c0 + half);
                    const float2 u0 = cs[rel], u1 = cs[rel + 1];
                    x0 = fmaf(x0, u0.x, bf_lo(yv) * u0.y);
                    x1 = fmaf(x1, u1.x, bf_hi(yv) * u1.y);
                  } else {
                    const uint32_t yv = *reinterpret_cast<const uint32_t*>(qr + c0 - half);
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
            qhi[nt][ks][part] = hi;
            qlo[nt][ks][part] = pack_bf16x2(x0 - bf_lo(hi), x1 - bf_hi(hi));
          }
        }
#pragma unroll
        for (int n = 0; n < KS; ++n) { O[nt][n][0] = O[nt][n][1] = O[nt][n][2] = O[nt][n][3] = 0.f; }
        m_run[nt][0] = m_run[nt][1] = -CUDART_INF_F;
        l_run[nt][0] = l_run[nt][1] = 0.f;
      }
      if constexpr (KT > 0) {
        // ---- on-read patch of this segment: (W_k q)^T [rank][G] by MMA (A = W_k rows from global, B = the q fragments).
        // TARGET frame (Eq. 1: rotate, then add) contracts W_k with the UNrotated q; CANONICAL with the rotated one.
        bool bad;
        const SegPatch sp = seg_patch(p.patches, S.patch, KT, true, &bad);
        kt_seg = sp.rank >> 4;
        if (kt_seg) {
          const __nv_bfloat16* Wk = sp.Wk + static_cast<size_t>(head) * sp.rank * D;
          Wv_seg = sp.Wv + static_cast<size_t>(head) * sp.rank * D;
          u_head_off = sp.uhs ? static_cast<uint32_t>(warp * sp.rank * 2) : 0u;
          const bool raw_q = use_lo && sp.frame != KAM_PATCH_CANONICAL_FRAME;
#pragma unroll
          for (int kt = 0; kt < KT; ++kt) {
            if (kt < kt_seg) {
              float acc[NT][4];
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
              const __nv_bfloat16* w0 = Wk + static_cast<size_t>(kt * 16 + gq) * D + 2 * t4;
#pragma unroll
              for (int ks = 0; ks < KS; ++ks) {
                const uint32_t a0 = ldg_u32(w0 + ks * 16), a1 = ldg_u32(w0 + 8 * D + ks * 16);
                const uint32_t a2 = ldg_u32(w0 + ks * 16 + 8), a3 = ldg_u32(w0 + 8 * D + ks * 16 + 8);
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                  uint32_t b0 = qhi[nt][ks][0], b1 = qhi[nt][ks][1];
                  if (raw_q) {
                    const int row = nt * 8 + gq;
                    b0 = b1 = 0u;
                    if (row < g.G) { const __nv_bfloat16* qr = qb + static_cast<size_t>(row) * D + ks * 16 + 2 * t4; b0 = ldg_u32(qr); b1 = ldg_u32(qr + 8); }
                  }
                  mma_bf16_16816(acc[nt][0], acc[nt][1], acc[nt][2], acc[nt][3], a0, a1, a2, a3, b0, b1);
                  if (use_lo && !raw_q) mma_bf16_16816(acc[nt][0], acc[nt][1], acc[nt][2], acc[nt][3], a0, a1, a2, a3, qlo[nt][ks][0], qlo[nt][ks][1]);
                }
              }
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) {
                const uint32_t h01 = pack_bf16x2(acc[nt][0], acc[nt][1]), h23 = pack_bf16x2(acc[nt][2], acc[nt][3]);
                const uint32_t l01 = pack_bf16x2(acc[nt][0] - bf_lo(h01), acc[nt][1] - bf_hi(h01));
                const uint32_t l23 = pack_bf16x2(acc[nt][2] - bf_lo(h23), acc[nt][3] - bf_hi(h23));
                wqh[nt][kt][0] = movmatrix_trans(h01); wqh[nt][kt][1] = movmatrix_trans(h23);
                wql[nt][kt][0] = movmatrix_trans(l01); wql[nt][kt][1] = movmatrix_trans(l23);
                Z[nt][kt][0] = Z[nt][kt][1] = Z[nt][kt][2] = Z[nt][kt][3] = 0.f;
              }
            }
          }
        }
      }
    }

    // ---- S^T[16 tokens][8 heads] = K q~^T : two interleaved accumulator chains per head tile
    float sa[NT][4], sb[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) { sa[nt][0] = sa[nt][1] = sa[nt][2] = sa[nt][3] = 0.f; sb[nt][0] = sb[nt][1] = sb[nt][2] = sb[nt][3] = 0.f; }
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      uint32_t a0, a1, a2, a3;
      // chunk index of this k-step inside its 64-column block: (ks & 3) * 2 (+ k_hi), XOR-swizzled on the TMA path
      ldmatrix_x4(a0, a1, a2, a3, TMA ? kb + (ks >> 2) * 2048 + (k_sw ^ ((ks & 3) << 5)) : kb + ks * 32);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        if (ks & 1) mma_bf16_16816(sb[nt][0], sb[nt][1], sb[nt][2], sb[nt][3], a0, a1, a2, a3, qhi[nt][ks][0], qhi[nt][ks][1]);
        else        mma_bf16_16816(sa[nt][0], sa[nt][1], sa[nt][2], sa[nt][3], a0, a1, a2, a3, qhi[nt][ks][0], qhi[nt][ks][1]);
        if (use_lo) {
          if (ks & 1) mma_bf16_16816(sa[nt][0], sa[nt][1], sa[nt][2], sa[nt][3], a0, a1, a2, a3, qlo[nt][ks][0], qlo[nt][ks][1]);
          else        mma_bf16_16816(sb[nt][0], sb[nt][1], sb[nt][2], sb[nt][3], a0, a1, a2, a3, qlo[nt][ks][0], qlo[nt][ks][1]);
        }
      }
    }
    if constexpr (KT > 0) {
      if (kt_seg) {                                             // s_t += U_k[t,:] . (W_k q): A = the tile's U_k rows (tokens x rank)
        const uint32_t ub = kb - k_lane + g.u_off + k_row * g.su_row + u_head_off + k_hi * 16;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t a0, a1, a2, a3;
            ldmatrix_x4(a0, a1, a2, a3, ub + kt * 32);
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              mma_bf16_16816(sa[nt][0], sa[nt][1], sa[nt][2], sa[nt][3], a0, a1, a2, a3, wqh[nt][kt][0], wqh[nt][kt][1]);
              mma_bf16_16816(sb[nt][0], sb[nt][1], sb[nt][2], sb[nt][3], a0, a1, a2, a3, wql[nt][kt][0], wql[nt][kt][1]);
            }
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[kbox]);               // the K box is no longer read

    // ---- online softmax (exp2 domain) per query head (column); thread holds tokens gq, gq+8 x heads 2*t4, 2*t4+1
    const bool partial = hdr.y & HDR_PARTIAL;
    const int row_lo = hdr.z & 0xff, row_hi = hdr.z >> 8;
    const bool ok0 = !partial || (gq >= row_lo && gq < row_hi);
    const bool ok1 = !partial || (gq + 8 >= row_lo && gq + 8 < row_hi);
    uint32_t pb[NT][2];
    float al[NT][2];
    bool rescale = false;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      float v[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float sv = (sa[nt][e] + sb[nt][e]) * scale_log2;
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
      // P^T as the B operand: b0 = P[tokens 2t,2t+1][head g], b1 = P[tokens 2t+8,2t+9][head g]
      pb[nt][0] = movmatrix_trans(pack_bf16x2(v[0], v[1]));
      pb[nt][1] = movmatrix_trans(pack_bf16x2(v[2], v[3]));
    }
    if (__any_sync(0xffffffffu, rescale)) {
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int n = 0; n < KS; ++n) { O[nt][n][0] *= al[nt][0]; O[nt][n][1] *= al[nt][1]; O[nt][n][2] *= al[nt][0]; O[nt][n][3] *= al[nt][1]; }
      if constexpr (KT > 0) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int kt = 0; kt < KT; ++kt) { Z[nt][kt][0] *= al[nt][0]; Z[nt][kt][1] *= al[nt][1]; Z[nt][kt][2] *= al[nt][0]; Z[nt][kt][3] *= al[nt][1]; }
      }
    }

    // ---- O^T[d][head] += V^T P^T
    mbar_wait(&full_bar[box], phase);
    uint8_t* vbox = box0 + static_cast<size_t>(box) * g.box_bytes;
    const int vboxi = box;
    if (++box == g.n_boxes) { box = 0; phase ^= 1; }
    if (partial) {
      // rows outside the chunk may hold anything (another chunk's tokens, uninitialised pages): 0 * NaN must not reach O
      for (int idx = lane; idx < 16 * (D / 8); idx += 32) {
        const int r = idx / (D / 8), j = idx - r * (D / 8);       // token row, 16-byte chunk of this head's D columns
        if (r < row_lo || r >= row_hi) {
          uint8_t* dst = TMA ? vbox + ((warp * (D / 64) + (j >> 3)) * 16 + r) * 128 + (((j & 7) ^ (r & 7)) << 4)
                             : vbox + r * g.s_row + warp * D * 2 + j * 16;
          *reinterpret_cast<uint4*>(dst) = make_uint4(0, 0, 0, 0);
        }
      }
      if constexpr (KT > 0) {
        if (kt_seg) {                                           // same for the U_v rows of this warp's head (2 chunks per rank tile)
          const int cpr = kt_seg * 2;
          for (int idx = lane; idx < 16 * cpr; idx += 32) {
            const int r = idx / cpr, j = idx - r * cpr;
            if (r < row_lo || r >= row_hi) *reinterpret_cast<uint4*>(vbox + g.u_off + r * g.su_row + u_head_off + j * 16) = make_uint4(0, 0, 0, 0);
          }
        }
      }
      __syncwarp();
    }
    const uint32_t vb = smem_u32(vbox) + v_lane;
#pragma unroll
    for (int dp = 0; dp < KS; ++dp) {
      uint32_t a0, a1, a2, a3;
      ldmatrix_x4_trans(a0, a1, a2, a3, TMA ? vb + (dp >> 2) * 2048 + (v_sw ^ ((dp & 3) << 5)) : vb + dp * 32);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
        mma_bf16_16816(O[nt][dp][0], O[nt][dp][1], O[nt][dp][2], O[nt][dp][3], a0, a1, a2, a3, pb[nt][0], pb[nt][1]);
    }
    if constexpr (KT > 0) {
      if (kt_seg) {                                             // z^T[j][head] += U_v^T P^T: A = the tile's U_v rows, transposed on load
        const uint32_t ub = smem_u32(vbox) + g.u_off + v_row * g.su_row + u_head_off + v_hi * 16;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t a0, a1, a2, a3;
            ldmatrix_x4_trans(a0, a1, a2, a3, ub + kt * 32);
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
              mma_bf16_16816(Z[nt][kt][0], Z[nt][kt][1], Z[nt][kt][2], Z[nt][kt][3], a0, a1, a2, a3, pb[nt][0], pb[nt][1]);
          }
        }
      }
    }
    if (partial) fence_proxy_async();                           // the zeroed rows were generic-proxy writes; the next fill is TMA
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[vboxi]);

    if constexpr (KT > 0) {
      if ((hdr.y & HDR_LAST) && kt_seg) {
        // ---- o^T[d][head] += W_v^T[d][j] z^T[j][head]: A[d][j] = W_v[j][d] gathered from global, B = z^T as bf16 hi + lo
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t bh[NT][2], bl[NT][2];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              const uint32_t h01 = pack_bf16x2(Z[nt][kt][0], Z[nt][kt][1]), h23 = pack_bf16x2(Z[nt][kt][2], Z[nt][kt][3]);
              const uint32_t l01 = pack_bf16x2(Z[nt][kt][0] - bf_lo(h01), Z[nt][kt][1] - bf_hi(h01));
              const uint32_t l23 = pack_bf16x2(Z[nt][kt][2] - bf_lo(h23), Z[nt][kt][3] - bf_hi(h23));
              bh[nt][0] = movmatrix_trans(h01); bh[nt][1] = movmatrix_trans(h23);
              bl[nt][0] = movmatrix_trans(l01); bl[nt][1] = movmatrix_trans(l23);
            }
            const __nv_bfloat16* w0 = Wv_seg + static_cast<size_t>(kt * 16 + 2 * t4) * D + gq;
#pragma unroll
            for (int dp = 0; dp < KS; ++dp) {
              const __nv_bfloat16* w = w0 + dp * 16;
              const uint32_t a0 = ldg_u16(w) | (ldg_u16(w + D) << 16), a1 = ldg_u16(w + 8) | (ldg_u16(w + D + 8) << 16);
              const uint32_t a2 = ldg_u16(w + 8 * D) | (ldg_u16(w + 9 * D) << 16), a3 = ldg_u16(w + 8 * D + 8) | (ldg_u16(w + 9 * D + 8) << 16);
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) {
                mma_bf16_16816(O[nt][dp][0], O[nt][dp][1], O[nt][dp][2], O[nt][dp][3], a0, a1, a2, a3, bh[nt][0], bh[nt][1]);
                mma_bf16_16816(O[nt][dp][0], O[nt][dp][1], O[nt][dp][2], O[nt][dp][3], a0, a1, a2, a3, bl[nt][0], bl[nt][1]);
              }
            }
          }
        }
      }
    }
    if (hdr.y & HDR_LAST) {
      // ---- per-(segment, head) softmax state -> partials: o normalised, lse in natural log
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int hq = nt * 8 + 2 * t4 + e;
          const float l = col_sum(l_run[nt][e]);
          if (hq < g.G) {
            const float inv = l > 0.f ? 1.f / l : 0.f;
            const size_t row = static_cast<size_t>(seg) * g.R + warp * g.G + hq;
            float* po = p.part_o + row * g.Dv + gq;
#pragma unroll
            for (int n = 0; n < KS; ++n) { po[n * 16] = O[nt][n][e] * inv; po[n * 16 + 8] = O[nt][n][2 + e] * inv; }
            if (gq == 0) p.part_lse[row] = l > 0.f ? (m_run[nt][e] + log2f(l)) * 0.6931471805599453f : -CUDART_INF_F;
          }
        }
      }
    }
  }
}

namespace {
template <int KS, int NT, typename F> void decode_dispatch_kt(const DecodeGeom& g, F&& f) {
  if (g.use_tma) {
    switch (g.KT) {
      case 0: f(kam_paged_decode_kernel<KS, NT, true, 0>); break;
      case 1: f(kam_paged_decode_kernel<KS, NT, true, 1>); break;
      case 2: f(kam_paged_decode_kernel<KS, NT, true, 2>); break;
      default: f(kam_paged_decode_kernel<KS, NT, true, 4>); break;
    }
  } else {
    switch (g.KT) {
      case 0: f(kam_paged_decode_kernel<KS, NT, false, 0>); break;
      case 1: f(kam_paged_decode_kernel<KS, NT, false, 1>); break;
      case 2: f(kam_paged_decode_kernel<KS, NT, false, 2>); break;
      default: f(kam_paged_decode_kernel<KS, NT, false, 4>); break;
    }
  }
}
template <typename F> void decode_dispatch(const DecodeGeom& g, F&& f) {
  if (g.D == 128) { if (g.NT == 1) decode_dispatch_kt<8, 1>(g, f); else decode_dispatch_kt<8, 2>(g, f); }
  else            { if (g.NT == 1) decode_dispatch_kt<4, 1>(g, f); else decode_dispatch_kt<4, 2>(g, f); }
}
}  // namespace

int decode_occupancy(const DecodeGeom& g) {
  int n = 0;
  decode_dispatch(g, [&](auto kern) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);   // the launch passes the real size
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, (g.HG + 1) * 32, g.smem_bytes) != cudaSuccess) { cudaGetLastError(); n = 0; }
  });
  return n;
}



void launch_decode(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st) {
  decode_dispatch(g, [&](auto kern) { launch_ex(kern, g.n_ctas, (g.HG + 1) * 32, g.smem_bytes, pdl, st, g, p); });
}

// ---------------------------------------------------------------------------------------------------- merge
// A9: lse = ln sum_s e^{lse_s};  out = sum_s e^{lse_s - lse} o_s over the request's segments of this head's group.
// One CTA per (request, query head); warp w folds segments s0 + w, s0 + w + 8, ... (four independent loads in flight per
// lane), then the 8 warp states are folded in warp order.  Fixed assignment and order => run-to-run deterministic.

// CPL: columns per lane = Dv / 32.  WARPS x UNROLL segments are in flight per CTA; the three instantiations are sized so that
// the whole grid (one CTA per query head) is resident at once: a second wave would repeat the kernel's latency chain (plan read
// -> partials read -> reduce -> write), which is all this kernel's time (measured: 896 CTAs at 5 per SM = 2 waves, 9.7 us).
template <int CPL, int WARPS, int UNROLL, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) kam_lse_merge_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  __shared__ float sm_m[WARPS], sm_l[WARPS];
  __shared__ float sm_acc[WARPS][32 * CPL];
  // stateless call: the decode kernel before this one may itself have started under the plan kernel (it signals its dependents
  // at once), so the plan is only safe to read once the decode kernel - and with it the plan kernel - has completed
  if (p.plan_fresh) grid_dep_wait();
  const int bh = blockIdx.x;                      // b * Hq + hq
  const int b = bh / g.Hq, hq = bh - b * g.Hq;
  const int hg = hq / g.R, r = hq - hg * g.R;
  const int N = p.plan.dyn[0];                    // see DecodePlan::dyn
  const int s0 = p.plan.seg_base[hg * N + p.plan.rcb[b]], s1 = p.plan.seg_base[hg * N + p.plan.rcb[b + 1]];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  grid_dep_wait();                                // the partials are complete and visible from here
  // the next kernel on the stream (the next layer's decode) is released only now: released at the top of this kernel its CTAs
  // become resident during the TAIL of the decode before this merge and hold SM slots its last CTAs' merge needs - measured
  // with the whole merge grid resident at once: 28 layers 3.08 ms instead of 2.71 ms
  grid_dep_launch();
  const float* pl = p.part_lse + r;
  const float* po = p.part_o + static_cast<size_t>(r) * g.Dv + lane * CPL;
  const size_t so = static_cast<size_t>(g.R) * g.Dv;

  float m = -CUDART_INF_F, l = 0.f, acc[CPL];
#pragma unroll
  for (int c = 0; c < CPL; ++c) acc[c] = 0.f;
  for (int base = s0 + warp; base < s1; base += WARPS * UNROLL) {
    float ls[UNROLL], o[UNROLL][CPL];
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
      const int s = base + u * WARPS;
      ls[u] = -CUDART_INF_F;
#pragma unroll
      for (int c = 0; c < CPL; ++c) o[u][c] = 0.f;
      if (s < s1) {
        ls[u] = pl[static_cast<size_t>(s) * g.R];
        if constexpr (CPL % 4 == 0) {
#pragma unroll
          for (int c4 = 0; c4 < CPL / 4; ++c4) {
            const float4 v = *reinterpret_cast<const float4*>(po + s * so + c4 * 4);
            o[u][c4 * 4] = v.x; o[u][c4 * 4 + 1] = v.y; o[u][c4 * 4 + 2] = v.z; o[u][c4 * 4 + 3] = v.w;
          }
        } else { const float2 v = *reinterpret_cast<const float2*>(po + s * so); o[u][0] = v.x; o[u][1] = v.y; }
      }
    }
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
      if (ls[u] == -CUDART_INF_F) continue;
      const float mn = fmaxf(m, ls[u]);
      const float a = __expf(m - mn), w = __expf(ls[u] - mn);
      l = fmaf(l, a, w);
#pragma unroll
      for (int c = 0; c < CPL; ++c) acc[c] = fmaf(acc[c], a, w * o[u][c]);
      m = mn;
    }
  }
  if (lane == 0) { sm_m[warp] = m; sm_l[warp] = l; }
#pragma unroll
  for (int c = 0; c < CPL; ++c) sm_acc[warp][lane * CPL + c] = acc[c];
  __syncthreads();

  float M = -CUDART_INF_F;
#pragma unroll
  for (int w = 0; w < WARPS; ++w) M = fmaxf(M, sm_m[w]);
  __nv_bfloat16* out = static_cast<__nv_bfloat16*>(p.out) + static_cast<size_t>(bh) * g.Dv;
  float* outf = static_cast<float*>(p.out) + static_cast<size_t>(bh) * g.Dv;
  if (M == -CUDART_INF_F) {                       // no tokens at all: out = 0, lse = -inf, no NaN
    for (int c = threadIdx.x; c < g.Dv; c += WARPS * 32) { if (p.out_f32) outf[c] = 0.f; else out[c] = __float2bfloat16_rn(0.f); }
    if (threadIdx.x == 0) p.lse[bh] = -CUDART_INF_F;
    return;
  }
  float tot = 0.f, ew[WARPS];
#pragma unroll
  for (int w = 0; w < WARPS; ++w) {
    ew[w] = sm_m[w] == -CUDART_INF_F ? 0.f : __expf(sm_m[w] - M);
    tot = fmaf(sm_l[w], ew[w], tot);
  }
  for (int c = threadIdx.x; c < g.Dv; c += WARPS * 32) {
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) v = fmaf(sm_acc[w][c], ew[w], v);
    if (p.out_f32) outf[c] = v / tot; else out[c] = __float2bfloat16_rn(v / tot);
  }
  if (threadIdx.x == 0) p.lse[bh] = M + logf(tot);
}

// A9 across ranks (S 8(e), f4): the same state merge over n_parts (o_p, lse_p) pairs, fixed order p = 0, 1, ... (deterministic
// and identical on every rank).  One CTA per query row; a part whose lse is -inf (a rank that held none of the request's
// chunks) contributes nothing.
__global__ void __launch_bounds__(128) kam_state_merge_kernel(const __grid_constant__ StateMergeParams p) {
  const int row = blockIdx.x;
  float M = -CUDART_INF_F;
  for (int i = 0; i < p.n_parts; ++i) M = fmaxf(M, p.lse[i][row]);
  __nv_bfloat16* out = static_cast<__nv_bfloat16*>(p.out) + static_cast<size_t>(row) * p.Dv;
  if (M == -CUDART_INF_F) {
    for (int c = threadIdx.x; c < p.Dv; c += blockDim.x) out[c] = __float2bfloat16_rn(0.f);
    if (threadIdx.x == 0) p.lse_out[row] = -CUDART_INF_F;
    return;
  }
  float tot = 0.f;
  for (int i = 0; i < p.n_parts; ++i) { const float l = p.lse[i][row]; tot += l == -CUDART_INF_F ? 0.f : __expf(l - M); }
  for (int c = threadIdx.x; c < p.Dv; c += blockDim.x) {
    float v = 0.f;
    for (int i = 0; i < p.n_parts; ++i) {
      const float l = p.lse[i][row];
      if (l != -CUDART_INF_F) v = fmaf(p.o[i][static_cast<size_t>(row) * p.Dv + c], __expf(l - M), v);
    }
    out[c] = __float2bfloat16_rn(v / tot);
  }
  if (threadIdx.x == 0) p.lse_out[row] = M + logf(tot);
}

void launch_state_merge(const StateMergeParams& p, cudaStream_t st) {
  kam_state_merge_kernel<<<p.rows, 128, 0, st>>>(p);
}

void launch_decode_merge(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st) {
  const int grid = p.plan.batch * g.Hq;
  if (g.Dv == 512)      launch_ex(kam_lse_merge_kernel<16, 4, 2, 7>, grid, 128, 0, pdl, st, g, p);
  else if (g.Dv == 128) launch_ex(kam_lse_merge_kernel<4, 4, 4, 8>, grid, 128, 0, pdl, st, g, p);
  else                  launch_ex(kam_lse_merge_kernel<2, 4, 4, 8>, grid, 128, 0, pdl, st, g, p);
}

}  // namespace kam

// kam_mla_ts_decode_kernel<KT>: absorbed MLA decode, TOKEN-split form, with the rank-m patch of
// Eq. 1 applied ON READ (KT = 16-wide rank tiles the instantiation carries; 0 = calls without patch refs).
//
// A cached token is ONE row [c_KV (512, position-free) | k_pe (64, RoPE)]; with the up-projections absorbed into the query
// and output sides (outside this library) a query head is q = [q_lat 512 | q_pe 64], the score is the 576-wide dot product
// and the value is the latent itself:      s_t = sm_scale * q . k^_t ,   o = sum_t p_t k^_t[0:512]
// so every cached byte is read ONCE and serves both QK^T and PV.  Relocation on read touches only q_pe (q~ = R(-delta) q on
// the rope band, bf16 hi + lo).  Same plan, partials and merge as the GQA kernel (decode_kernel.cu).
//
// (Round 1 also had a k-split formulation - the 576-deep contraction cut over four warps for EVERY 16-token tile, a score
// exchange, a CTA barrier and a 4x repeated softmax per tile, ~600 instructions per warp and tile - and a tcgen05 one; both
// measured slower at every shape this library runs and were removed, profiles/HISTORY.md.)  One ITERATION is 64 tokens
// (four 16-token TMA boxes) and the work is split by TOKENS first:
//
//   warp w of 8:  tg = w & 3 (which box of the iteration), kh = w >> 2 (which half of the contraction / of the heads)
//   S^T[16 tokens of box tg][16 heads] over k-steps [18 kh, 18 kh + 18): 18 ldmatrix + 36 HMMA, q~ fragments in 72 registers;
//     the two warps of a box swap the head half the other one owns (4 floats per lane, one 64-thread barrier), so each warp
//     ends with COMPLETE scores of 8 heads x 16 tokens and every softmax value is computed once
//   P^T (bf16) -> shared memory [64 tokens][16 heads]
//   ONE CTA barrier per iteration (barrier.red.or: it also tells whether any score ran 2^8 past its head's reference)
//   O^T[64 w .. 64 w + 64][16 heads] += V^T P^T over the iteration's 64 tokens: warp w owns 64-column block w of every box
//
// The reference of the lazy softmax (decode_kernel.cu) is common to the CTA and moves only through a slow path (two more
// barriers: tile maxima -> new references, rescale factors -> O), taken on the first iteration of a segment and then rarely.
// Per warp and 64 tokens: 68 HMMA, 38 LDSM, ~250 instructions in all (the k-split kernel: ~1200).
// CTA = 8 compute warps + 1 producer warp (slot mapping A1 + one TMA box [9 x 64 columns][16 tokens][128 B swizzled] per
// tile) inside a third warpgroup that gives its registers away (setmaxnreg: 12 warps launch at 168 registers, the compute
// warps run at 232, the producer at 40).  One CTA per SM, flat ring of 11 boxes (an iteration takes the next 1-4 slots).
//
// Two things measured on B200 while building this (both shaped the code, both are in DESIGN.md 7.2):
//  * With ~200 KB of bulk copies in flight per SM, a DEMAND load from the same SM waits microseconds (it queues behind them);
//    two dependent ones per segment (the segment record, then q) cost 28 of 133 us.  So the compute warps never load from
//    global memory: the producer stages q (16 rows x 1152 B, one bulk copy) and the chunk's (cos, sin) row into shared memory
//    IN the copy stream, right before the segment's first box, and the segment's fields ride in the box headers.
//  * mbarrier.try_wait costs 100+ cycles even on a phase that completed long ago.  Three of them in a row before PV (the boxes
//    of the other warps) cost 11 of 123 us; so a warp waits ONCE per iteration (its own box, whose header repeats the
//    iteration's fields and the next iteration's size) and lanes 0-3 check the other boxes' barriers in one pass before PV.
//    (Doing that one-pass check where the data may really be late - at the top of the iteration - is slow: the lanes spin
//    one after the other.)
// Measured and rejected: computing the next iteration's scores inside this iteration's PV (two independent ldmatrix -> HMMA
// streams per warp): 123 -> 133 us, whether or not it waited for the next boxes.
//
// On-read patch (KT > 0; Eq. 1 substituted into P:44; "a small added k_pe-band patch").  One U, W pair per chunk (the
// key's; its latent columns patch the value):   s_t += U[t,:] . (W q)        o += (sum_t p_t U[t,:]) W[:, 0:512]
// Nothing of it is fetched by a demand load either.  W travels THROUGH THE BOX RING: a patched segment is bracketed by two
// "W iterations" of rank/16 boxes each, one box = the 16 x 1152-byte rows of one rank tile of W (bulk copies, rows padded to
// 1168 bytes so that ldmatrix is conflict-free), flagged HDR_W in the header:
//   head (HDR_W | HDR_FIRST)  warp (tg, kh) contracts rank tile tg of W with its k-half of q exactly as it computes scores
//                             (TARGET frame: the un-rotated q; CANONICAL: q~ hi + lo); the two halves meet in shared memory and
//                             wq^T [16 heads][rank] is left there as bf16 hi + lo                       (2 CTA barriers)
//   data iterations           the tile's U rows ride behind their box (one bulk copy when U is token-contiguous);
//                             s += U wq: 1 LDSM (U) + 1 LDSM (wq) + 2 HMMA per rank tile on the warp's own 8 heads x 16 tokens;
//                             z^T [rank][8 heads] += U^T P^T for the warp's own box and head tile: 1 LDSM.T + 1 HMMA per rank tile
//   tail (HDR_W | HDR_LAST)   the eight partial z meet in shared memory -> z^T bf16 hi + lo; O^T += W_lat^T z^T with the W boxes
//                             as the A operand through ldmatrix.trans (like V^T); then the segment's state is written
// so W costs two extra box copies per rank tile and segment (the second one an L2 hit) and no dedicated buffer: the ring keeps
// 10 / 9 / 8 boxes at rank <= 16 / 32 / 64.
#include <cuda_runtime.h>
#include <math_constants.h>

#include <type_traits>

#include "common.cuh"
#include "decode_common.cuh"
#include "internal.h"

// diagnostic builds (KAM_NVCC_EXTRA=-DKAM_TS_DIAG=n; wrong results): 1 no W-iteration compute, 2 no per-iteration patch MMAs,
// 4 no U copies
#ifndef KAM_TS_DIAG
#define KAM_TS_DIAG 0
#endif
#if KAM_TS_DIAG & 2
#define KAM_TS_SKIP_ITER && false
#else
#define KAM_TS_SKIP_ITER
#endif
#if KAM_TS_DIAG & 8
#define KAM_TS_SKIP_S && false
#else
#define KAM_TS_SKIP_S
#endif
#if KAM_TS_DIAG & 16
#define KAM_TS_SKIP_Z && false
#else
#define KAM_TS_SKIP_Z
#endif

namespace kam {

namespace {
constexpr int kTsWarps = 8;                 // compute warps
constexpr int kTsThreads = kTsWarps * 32;   // threads at the compute warps' named barriers
constexpr int kTsBlock = 384;               // 2 compute warpgroups + 1 warpgroup whose first warp is the producer (registers move
                                            // between warpgroups: 12 warps launch at 168 registers, the compute warps take 232, the producer keeps 40)
constexpr int kTsIter = 4;                  // boxes (16-token tiles) per full iteration
constexpr int kTsSteps = 36;                // 16-column k-steps of a 576-wide row (32 latent + 4 rope)
constexpr int kTsBox = kDecTile * 576 * 2;  // 18432 bytes
constexpr int kTsPRow = 32;                 // bytes of one token's row of P^T: 16 heads x bf16, 16-byte halves swapped in rows 4-7 of 8
constexpr int kTsPBuf = kTsIter * kDecTile * kTsPRow;
constexpr int kTsWRow = 1168;               // bytes between two rank rows of a W box: 1152 + 16, (kTsWRow / 16) odd
constexpr int kTsWqRow = 144;               // bytes of one head's row of wq^T / z^T (64 ranks x bf16 + 16)
// shared-memory map (bytes)
constexpr int kTsOffHdr = 256;              // int4[<= 16]
constexpr int kTsOffRed = 512;              // float[8 warps][8 heads]: tile maxima (slow path)
constexpr int kTsOffAlpha = 768;            // float[16 heads]: rescale factors (slow path)
constexpr int kTsOffLsum = 1024;            // float[8 warps][8 heads]: softmax masses at the end of a segment
constexpr int kTsOffCs = 1280;              // float2[32]: (cos, sin)(delta f_i) of the segment's chunk
constexpr int kTsOffP = 2048;               // 2 x kTsPBuf
constexpr int kTsOffXch = kTsOffP + 2 * kTsPBuf;            // float[8 warps][4][32 lanes]: partial scores between the k-halves
constexpr int kTsOffQ = kTsOffXch + 4096;   // q of the segment: [16 heads][1152 B], as in global memory
constexpr int kTsOffWq = kTsOffQ + kTsBox;  // 28672; KT > 0: wq^T, later z^T: [hi | lo][16 heads][kTsWqRow]
constexpr int kTsOffZp = kTsOffWq + 2 * 16 * kTsWqRow;      // KT > 0: float[4][KT * 16 ranks][16 heads]: partial wq (2 k-halves) / partial z (4 boxes)
template <int KT> struct TsMap {
  static constexpr int off_box = KT == 0 ? kTsOffWq : (kTsOffZp + 4096 * KT + 1023) / 1024 * 1024;
  static constexpr int box_stride = KT == 0 ? kTsBox : kTsBox + (KT <= 2 ? 1024 : 2048);   // + the U tile: 16 tokens x KT x 32 B
  static constexpr int slots = (227 * 1024 - off_box) / box_stride;                         // 11 | 10 | 9 | 8
  static constexpr int smem = off_box + slots * box_stride;
  static_assert(off_box % 1024 == 0 && box_stride % 1024 == 0 && slots >= 2 * kTsIter && slots <= 16, "shared-memory map");
  static_assert(KT == 0 || 16 * kTsWRow <= box_stride, "a W box is 16 padded rank rows");
};
enum : int { HDR_ROTATE = 8, HDR_W = 16, HDR_CANON = 32 };   // header flags beyond decode_common.cuh's; bits 8-10: rank tiles of the
                                                              // segment's patch; bits 16+: head group

__device__ __forceinline__ bool bar_or(int id, bool pred) {      // barrier over the compute warps + OR of pred
  uint32_t out;
  asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.b32 q, %2, 0;\n\tbarrier.cta.red.or.pred p, %1, %3, q;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(out) : "r"(id), "r"(static_cast<uint32_t>(pred)), "n"(kTsThreads) : "memory");
  return out != 0;
}
// 4 x 4 transpose of 32-bit words across a quad (lanes t4 = 0-3): in, lane r holds row r = (x, y, z, w); out, lane c holds
// column c.  Two butterfly stages (xor 2, xor 1), two shuffles each.
__device__ __forceinline__ void quad_transpose(uint4& v, int t4) {
  const bool h2 = t4 & 2, h1 = t4 & 1;
  uint32_t s0 = h2 ? v.x : v.z, s1 = h2 ? v.y : v.w;
  s0 = __shfl_xor_sync(0xffffffffu, s0, 2); s1 = __shfl_xor_sync(0xffffffffu, s1, 2);
  if (h2) { v.x = s0; v.y = s1; } else { v.z = s0; v.w = s1; }
  s0 = h1 ? v.x : v.y; s1 = h1 ? v.z : v.w;
  s0 = __shfl_xor_sync(0xffffffffu, s0, 1); s1 = __shfl_xor_sync(0xffffffffu, s1, 1);
  if (h1) { v.x = s0; v.z = s1; } else { v.y = s0; v.w = s1; }
}
}  // namespace

template <int KT>
__global__ void __launch_bounds__(kTsBlock, 1)
kam_mla_ts_decode_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  using M = TsMap<KT>;
  constexpr int kSlots = M::slots, kStride = M::box_stride, kOffBox = M::off_box;
  constexpr int kURow = KT * 32;                                 // bytes between two token rows of a box's U tile (whatever the segment's rank)
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + kSlots;
  uint64_t* q_full = empty_bar + kSlots;                         // q (+ cos/sin) of a segment staged / read into registers by all warps
  uint64_t* q_empty = q_full + 1;
  int4* hdrs = reinterpret_cast<int4*>(smem + kTsOffHdr);
  float* red = reinterpret_cast<float*>(smem + kTsOffRed);
  float* alpha_s = reinterpret_cast<float*>(smem + kTsOffAlpha);
  float* lsum = reinterpret_cast<float*>(smem + kTsOffLsum);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kSlots; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], kTsWarps); }
    mbar_init(q_full, 1); mbar_init(q_empty, kTsWarps);
    mbar_fence_init();
  }
  __syncthreads();

  grid_dep_launch();
  if (p.plan_fresh) grid_dep_wait();                             // the plan comes from the kernel right before this one
  const int seg_begin = p.plan.cta_seg[blockIdx.x], seg_end = p.plan.cta_seg[blockIdx.x + 1];
  if (seg_begin >= seg_end) return;

  if (warp >= kTsWarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp > kTsWarps) return;                                 // the rest of the producer warpgroup only gives its registers away
    // ================================================================ producer warp: lanes 0-3 issue the boxes of an iteration
    int slot = 0; uint32_t phase = 0, q_phase = 0;
    const char* tm_k = static_cast<const char*>(p.tmaps) + static_cast<size_t>(p.layer) * kTmapLayerBytes;
    auto tile_slot = [&](const DecSeg& S, const int32_t* bt, int tl) {       // pool slot of tile tl of the segment (A1)
      if (tl == 0) return S.slot0;
      const int tok = (S.tile0 + tl) * kDecTile;
      const int pg = g.P_shift >= 0 ? (tok >> g.P_shift) : tok / g.P;
      return bt[pg] * g.P + (tok - pg * g.P);
    };
    // the segment's patch, if its record is well formed (malformed ones are ignored, and counted once per chunk by `count`)
    auto patch_of = [&](const DecSeg& S, bool count) {
      SegPatch sp{};
      if constexpr (KT > 0) {
        bool bad;
        sp = seg_patch(p.patches, S.patch, KT, false, &bad);
        if (count && bad && lane == 0 && S.tile0 * kDecTile <= S.tok_lo && S.hg == 0) atomicAdd(p.err, 1);
      }
      return sp;
    };
    grid_dep_wait();
    DecSeg S_next = p.plan.segs[seg_begin];
    for (int seg = seg_begin; seg < seg_end; ++seg) {
      const DecSeg S = S_next;
      const SegPatch sp = patch_of(S, true);
      const int kt = sp.rank >> 4;                                 // rank tiles of this segment's patch (0: none)
      int nb_after = 0;                                            // boxes of the next segment's first iteration
      if (seg + 1 < seg_end) {
        S_next = p.plan.segs[seg + 1];                             // in flight while this segment streams
        const int kt_next = patch_of(S_next, false).rank >> 4;     // (the record is read again, from cache, when its turn comes)
        nb_after = kt_next ? kt_next : min(kTsIter, S_next.n_tiles);
      }
      const int seg_flags = (S.rotate ? HDR_ROTATE : 0) | (kt << 8) | (sp.frame == KAM_PATCH_CANONICAL_FRAME ? HDR_CANON : 0) | (S.hg << 16);
      const int32_t* bt = p.block_tables + S.bt_off;
      const int n_rows = min(kMlaHeads, g.Hq - S.hg * kMlaHeads);
      if (lane == 0) {
        // q and the cos/sin row travel in the stream, ahead of the segment's first box
        mbar_wait(q_empty, q_phase ^ 1);
        mbar_arrive_expect_tx(q_full, static_cast<uint32_t>(n_rows * 1152 + (S.rotate ? 256 : 0)));
        bulk_g2s(smem + kTsOffQ, static_cast<const char*>(p.q) + (static_cast<size_t>(S.b) * g.Hq + static_cast<size_t>(S.hg) * kMlaHeads) * 1152,
                 static_cast<uint32_t>(n_rows * 1152), q_full);
        if (S.rotate) bulk_g2s(smem + kTsOffCs, p.plan.cs + static_cast<size_t>(S.chunk) * 32, 256, q_full);
      }
      q_phase ^= 1;
      // a W iteration: box j takes rank tile j of W, one 1152-byte bulk copy per rank row (lanes 0-15)
      auto issue_w = [&](int edge_flag, int nb_next) {
        if constexpr (KT > 0) {
#pragma unroll 1
          for (int j = 0; j < kt; ++j) {
            uint8_t* dst = smem + kOffBox + slot * kStride;
            if (lane == 0) {
              mbar_wait(&empty_bar[slot], phase ^ 1);
              hdrs[slot] = make_int4(seg, seg_flags | HDR_W | edge_flag, 0, kt | (nb_next << 8));
              mbar_arrive_expect_tx(&full_bar[slot], 16u * 1152u);
            }
            __syncwarp();
            if (lane < 16)
              bulk_g2s(dst + lane * kTsWRow, reinterpret_cast<const char*>(sp.Wk) + static_cast<size_t>(j * 16 + lane) * 1152, 1152u, &full_bar[slot]);
            if (++slot == kSlots) { slot = 0; phase ^= 1; }
          }
        }
      };
      if (kt) issue_w(HDR_FIRST, min(kTsIter, S.n_tiles));
      int my_next = (lane < S.n_tiles) ? tile_slot(S, bt, lane) : 0;          // slots of tiles t0 + lane, one batch ahead
      for (int t0 = 0; t0 < S.n_tiles; t0 += 32) {
        const int my_slot = my_next;
        if (t0 + 32 + lane < S.n_tiles) my_next = tile_slot(S, bt, t0 + 32 + lane);
        const int nbatch = min(32, S.n_tiles - t0);
        for (int i0 = 0; i0 < nbatch; i0 += kTsIter) {
          const int nb = min(kTsIter, nbatch - i0);
          const int s0 = __shfl_sync(0xffffffffu, my_slot, i0 + (lane & 3));
          if (lane < nb) {
            int sl = slot + lane; uint32_t ph = phase;
            if (sl >= kSlots) { sl -= kSlots; ph ^= 1; }
            mbar_wait(&empty_bar[sl], ph ^ 1);
            const int tl = t0 + i0 + lane;
            const int tok = (S.tile0 + tl) * kDecTile;
            const int row_lo = max(S.tok_lo - tok, 0), row_hi = min(S.tok_hi - tok, kDecTile);
            // FIRST / LAST belong to the ITERATION (all its headers carry them); a patched segment has them on its W iterations
            const int flags = ((t0 + i0 == 0 && !kt) ? HDR_FIRST : 0) | ((t0 + i0 + nb >= S.n_tiles && !kt) ? HDR_LAST : 0) |
                              ((row_lo > 0 || row_hi < kDecTile) ? HDR_PARTIAL : 0) | seg_flags;
            // .w: boxes of this iteration | boxes of the NEXT one << 8 (0: the CTA's work ends) - the compute warps then know which
            // barriers to look at before any header of that iteration is readable (the plan emits no empty segment)
            const int rem = S.n_tiles - (t0 + i0 + nb);
            const int nb_next = rem > 0 ? min(kTsIter, rem) : (kt ? kt : nb_after);
            hdrs[sl] = make_int4(seg, flags, row_lo | (row_hi << 8), nb | (nb_next << 8));
            uint8_t* dst = smem + kOffBox + sl * kStride;
            const uint32_t u_row = static_cast<uint32_t>(sp.rank) * 2u;          // bytes of one token's U row (0 without a patch)
            mbar_arrive_expect_tx(&full_bar[sl], static_cast<uint32_t>(kTsBox) + ((KAM_TS_DIAG & 4) ? 0u : static_cast<uint32_t>(row_hi - row_lo) * u_row));
            tma_load_3d(dst, tm_k, 0, s0, 0, &full_bar[sl]);
            if constexpr (KT > 0) {
              if (kt && row_hi > row_lo && !(KAM_TS_DIAG & 4)) {
                // the tile's U rows (chunk-local tokens tok - tok_lo + r) land behind the box, kURow bytes apart: ONE copy when U is
                // token-contiguous and the segment's rank is the instantiation's
                const char* us = sp.Uk + static_cast<long long>(tok - S.tok_lo + row_lo) * sp.uts * 2;
                uint8_t* ud = dst + kTsBox + row_lo * kURow;
                if (sp.uts == sp.rank && u_row == kURow) bulk_g2s(ud, us, static_cast<uint32_t>(row_hi - row_lo) * u_row, &full_bar[sl]);
                else for (int r = 0; r < row_hi - row_lo; ++r) bulk_g2s(ud + r * kURow, us + static_cast<long long>(r) * sp.uts * 2, u_row, &full_bar[sl]);
              }
            }
          }
          __syncwarp();
          slot += nb;
          if (slot >= kSlots) { slot -= kSlots; phase ^= 1; }
        }
      }
      if (kt) issue_w(HDR_LAST, nb_after);
    }
    return;
  }

  // ================================================================ compute warps
  asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
  const int tg = warp & 3, kh = warp >> 2;   // box of the iteration; k-half of the scores = head half of the softmax
  const int hh = kh;
  const int gq = lane >> 2, t4 = lane & 3;
  const float scale_log2 = p.sm_scale * 1.4426950408889634f;
  constexpr float kLn2 = 0.6931471805599453f;

  // lane offsets inside a box: K rows through ldmatrix (A of S^T), V^T through ldmatrix.trans (A of O^T); 128-byte swizzle
  const int k_row = (lane & 7) + ((lane >> 3) & 1) * 8, k_hi = lane >> 4;
  const int v_row = (lane & 7) + (lane >> 4) * 8, v_hi = (lane >> 3) & 1;
  uint32_t koff[4], voff[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    koff[j] = static_cast<uint32_t>(k_row * 128) + ((static_cast<uint32_t>(k_hi ^ (lane & 7)) << 4) ^ (static_cast<uint32_t>(j) << 5));
    voff[j] = static_cast<uint32_t>(warp * 2048 + v_row * 128) + ((static_cast<uint32_t>(v_hi ^ (lane & 7)) << 4) ^ (static_cast<uint32_t>(j) << 5));
  }
  const uint32_t sm0 = smem_u32(smem);
  // P^T [token][16 heads]: this lane's stores (token rows gq and gq + 8 of box tg, heads hh * 8 + 2 t4, +1) and its
  // ldmatrix.trans rows; the two 16-byte halves of a row are swapped in rows 4-7 of every 8, so that eight rows cover all banks
  const uint32_t p_st = static_cast<uint32_t>(kTsOffP + (tg * kDecTile + gq) * kTsPRow + ((hh ^ ((gq >> 2) & 1)) << 4) + t4 * 4);
  const int p_row = (lane & 7) + ((lane >> 3) & 1) * 8;
  const uint32_t p_ld = sm0 + static_cast<uint32_t>(kTsOffP + p_row * kTsPRow + (((lane >> 4) ^ ((p_row >> 2) & 1)) << 4));
  float* xch_w = reinterpret_cast<float*>(smem + kTsOffXch) + warp * 128 + lane;          // this warp's partial scores out
  const float* xch_r = reinterpret_cast<const float*>(smem + kTsOffXch) + (warp ^ 4) * 128 + lane;   // the other k-half's in
  // KT > 0: B fragments (hi b0, b1 | lo b0, b1) of wq^T / z^T for head tile nt and rank tile kt through one ldmatrix.x4:
  // matrices (hi, ranks 0-7) (hi, ranks 8-15) (lo, 0-7) (lo, 8-15), rows = the tile's 8 heads
  const uint32_t wq_ld = sm0 + static_cast<uint32_t>(kTsOffWq + (lane >> 4) * 16 * kTsWqRow + (lane & 7) * kTsWqRow + ((lane >> 3) & 1) * 16);
  // and the B fragments of BOTH head tiles from one plane (+ 16 rows: the lo plane): (heads 0-7 | 8-15) x (ranks 0-7 | 8-15)
  const uint32_t wq_ld2 = sm0 + static_cast<uint32_t>(kTsOffWq + ((lane >> 4) * 8 + (lane & 7)) * kTsWqRow + ((lane >> 3) & 1) * 16);
  float* zp = reinterpret_cast<float*>(smem + kTsOffZp);

  uint32_t qf[kTsSteps / 2][2][2], ql[4][2][2];      // [k-step of this half][head tile][b0, b1]; lo: the rope k-steps (k-half 1)
  float O[2][4][4];
  float m_ref[2] = {-CUDART_INF_F, -CUDART_INF_F}, l_run[2] = {0.f, 0.f};
  constexpr int KTA = KT > 0 ? KT : 1;
  [[maybe_unused]] float Z[KTA][4];                  // z^T[16 ranks of tile kt][heads hh * 8 + 2 t4, +1] over this warp's boxes
  [[maybe_unused]] int kt_seg = 0;
  bool use_lo = false;
  int n_rows = 0, seg = 0;
  int slot = 0, pbuf = 0; uint32_t phase = 0, q_phase = 0;
  // ring slot j of the current iteration (slots slot .. slot + 3, wrapping) and its mbarrier parity
  auto slot_of = [&](int j) { const int sl = slot + j; return sl >= kSlots ? sl - kSlots : sl; };
  auto phase_of = [&](int j) { return slot + j >= kSlots ? (phase ^ 1u) : phase; };
  // the segment's softmax state -> partials: o normalised, lse in natural log
  auto publish_mass = [&]() {                                    // this warp's softmax masses; a CTA barrier must follow
    const float l0 = col_sum(l_run[0]), l1 = col_sum(l_run[1]);
    if (gq == 0) { lsum[warp * 8 + 2 * t4] = l0; lsum[warp * 8 + 2 * t4 + 1] = l1; }
  };
  auto write_state = [&]() {
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const float* r0 = lsum + nt * 32 + 2 * t4 + e;
        const float tot = (r0[0] + r0[8]) + (r0[16] + r0[24]);
        const int hq = nt * 8 + 2 * t4 + e;
        if (hq < n_rows) {
          const float inv = tot > 0.f ? 1.f / tot : 0.f;
          const size_t row = static_cast<size_t>(seg) * g.R + hq;
          float* po = p.part_o + row * 512 + warp * 64 + gq;
#pragma unroll
          for (int n = 0; n < 4; ++n) { po[n * 16] = O[nt][n][e] * inv; po[n * 16 + 8] = O[nt][n][2 + e] * inv; }
          if (nt == hh && tg == 0 && gq == 0) p.part_lse[row] = tot > 0.f ? (m_ref[e] + log2f(tot)) * kLn2 : -CUDART_INF_F;
        }
      }
    }
  };
  mbar_wait(&full_bar[0], 0);                                    // bootstrap: the first iteration's header tells its own size
  int nb = hdrs[0].w & 0xff;
  while (nb > 0) {
    // a try_wait costs ~100+ cycles even when the phase is long complete, so a warp waits ONCE here: for its own box, whose
    // header repeats the iteration's fields (a warp without a box in a short iteration waits for the first one)
    const int my_box = slot_of(tg < nb ? tg : 0);
    mbar_wait(&full_bar[my_box], phase_of(tg < nb ? tg : 0));
    const int4 hdr = hdrs[my_box];
    const int nb_next = (hdr.w >> 8) & 0xff;
    const bool first = hdr.y & HDR_FIRST;

    if (first) {
      // ---- new segment: q~ fragments of all 16 heads for this warp's 18 k-steps; the rope band rotated by -delta (hi + lo)
      seg = hdr.x;
      use_lo = hdr.y & HDR_ROTATE;
      n_rows = min(kMlaHeads, g.Hq - (hdr.y >> 16) * kMlaHeads);
      mbar_wait(q_full, q_phase); q_phase ^= 1;
      const float2* cs = reinterpret_cast<const float2*>(smem + kTsOffCs);
      // lane (gq, t4) reads 16-byte chunks 36 kh + 4 j + t4 (j < 9: this k-half's 18 k-steps) of rows gq and gq + 8 of the staged
      // q; a 4 x 4 transpose of 32-bit words across the quad turns four chunks into the B fragments of k-steps 2 j and 2 j + 1.
      // In k-half 1, j = 7 holds rope columns rel = 8 t4 .. + 7 and j = 8 their HALF-style partners rel + 32.
      const uint4 zero4 = make_uint4(0, 0, 0, 0);
      [[maybe_unused]] uint32_t raw[4][2][2];                      // KT > 0: the UNrotated rope k-steps (TARGET frame contracts W with q)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        const int row = nt * 8 + gq;
        const uint4* qr = reinterpret_cast<const uint4*>(smem + kTsOffQ + row * 1152) + 36 * kh + t4;
        const bool live = row < n_rows;
#pragma unroll
        for (int j = 0; j < 7; ++j) {
          uint4 w = live ? qr[4 * j] : zero4;
          quad_transpose(w, t4);
          qf[2 * j][nt][0] = w.x; qf[2 * j][nt][1] = w.y; qf[2 * j + 1][nt][0] = w.z; qf[2 * j + 1][nt][1] = w.w;
        }
        uint4 wx = live ? qr[28] : zero4, wy = live ? qr[32] : zero4;
        uint4 lx = zero4, ly = zero4;
        if constexpr (KT > 0) {
          uint4 rx = wx, ry = wy;
          quad_transpose(rx, t4); quad_transpose(ry, t4);
          raw[0][nt][0] = rx.x; raw[0][nt][1] = rx.y; raw[1][nt][0] = rx.z; raw[1][nt][1] = rx.w;
          raw[2][nt][0] = ry.x; raw[2][nt][1] = ry.y; raw[3][nt][0] = ry.z; raw[3][nt][1] = ry.w;
        }
        if (kh == 1 && use_lo) {                                   // q~ = R(-delta) q, carried as bf16 hi + lo
          float x[8], y[8], rx[8], ry[8];
          unpack8(wx, x); unpack8(wy, y);
          if (g.rope_style == KAM_ROPE_HALF) {
#pragma unroll
            for (int e = 0; e < 8; ++e) {
              const float2 u = cs[8 * t4 + e];
              rx[e] = fmaf(x[e], u.x, y[e] * u.y);
              ry[e] = fmaf(y[e], u.x, -x[e] * u.y);
            }
          } else {
#pragma unroll
            for (int e = 0; e < 8; e += 2) {
              const float2 u = cs[4 * t4 + (e >> 1)], v = cs[16 + 4 * t4 + (e >> 1)];
              rx[e] = fmaf(x[e], u.x, x[e + 1] * u.y); rx[e + 1] = fmaf(x[e + 1], u.x, -x[e] * u.y);
              ry[e] = fmaf(y[e], v.x, y[e + 1] * v.y); ry[e + 1] = fmaf(y[e + 1], v.x, -y[e] * v.y);
            }
          }
          wx = pack8(rx); wy = pack8(ry);
          unpack8(wx, x); unpack8(wy, y);
#pragma unroll
          for (int e = 0; e < 8; ++e) { rx[e] -= x[e]; ry[e] -= y[e]; }
          lx = pack8(rx); ly = pack8(ry);
        }
        quad_transpose(wx, t4); quad_transpose(wy, t4); quad_transpose(lx, t4); quad_transpose(ly, t4);
        qf[14][nt][0] = wx.x; qf[14][nt][1] = wx.y; qf[15][nt][0] = wx.z; qf[15][nt][1] = wx.w;
        qf[16][nt][0] = wy.x; qf[16][nt][1] = wy.y; qf[17][nt][0] = wy.z; qf[17][nt][1] = wy.w;
        ql[0][nt][0] = lx.x; ql[0][nt][1] = lx.y; ql[1][nt][0] = lx.z; ql[1][nt][1] = lx.w;
        ql[2][nt][0] = ly.x; ql[2][nt][1] = ly.y; ql[3][nt][0] = ly.z; ql[3][nt][1] = ly.w;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(q_empty);                       // the staging buffers may take the next segment's q
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int n = 0; n < 4; ++n) O[nt][n][0] = O[nt][n][1] = O[nt][n][2] = O[nt][n][3] = 0.f;
      m_ref[0] = m_ref[1] = -CUDART_INF_F;
      l_run[0] = l_run[1] = 0.f;
      if constexpr (KT > 0) {
        kt_seg = (hdr.y & HDR_W) ? ((hdr.y >> 8) & 7) : 0;
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) Z[kt][0] = Z[kt][1] = Z[kt][2] = Z[kt][3] = 0.f;
        if (hdr.y & HDR_W) {
          // ---- head W iteration: (W q)^T.  Warp (tg, kh) contracts rank tile tg of W with its k-half of q; TARGET frame (Eq. 1:
          // rotate, then add) takes the UNrotated q, CANONICAL the rotated one (hi + lo)
          if (tg < nb && !(KAM_TS_DIAG & 1)) {
            const uint32_t wb = sm0 + static_cast<uint32_t>(kOffBox + my_box * kStride + k_row * kTsWRow + k_hi * 16 + 18 * kh * 32);
            const bool use_raw = use_lo && !(hdr.y & HDR_CANON);
            float acc[2][4];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
#pragma unroll
            for (int i = 0; i < kTsSteps / 2; ++i) {
              uint32_t a0, a1, a2, a3;
              ldmatrix_x4(a0, a1, a2, a3, wb + i * 32);
#pragma unroll
              for (int nt = 0; nt < 2; ++nt) {
                uint32_t b0 = qf[i][nt][0], b1 = qf[i][nt][1];
                if (i >= 14 && kh == 1 && use_raw) { b0 = raw[i - 14][nt][0]; b1 = raw[i - 14][nt][1]; }
                mma_bf16_16816(acc[nt][0], acc[nt][1], acc[nt][2], acc[nt][3], a0, a1, a2, a3, b0, b1);
                if (i >= 14 && kh == 1 && use_lo && !use_raw)
                  mma_bf16_16816(acc[nt][0], acc[nt][1], acc[nt][2], acc[nt][3], a0, a1, a2, a3, ql[i - 14][nt][0], ql[i - 14][nt][1]);
              }
            }
            // the two k-halves swap the head tile the other one owns (as the scores do); each warp then holds the complete
            // wq^T[ranks gq, gq + 8 of tile tg][heads hh * 8 + 2 t4, + 1] and leaves it in shared memory as bf16 hi + lo
#pragma unroll
            for (int e = 0; e < 4; ++e) xch_w[e * 32] = hh ? acc[0][e] : acc[1][e];
            named_bar_sync(4 + tg, 64);
            __nv_bfloat16* w = reinterpret_cast<__nv_bfloat16*>(smem + kTsOffWq + (hh * 8 + 2 * t4) * kTsWqRow) + tg * 16 + gq;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float v = (hh ? acc[1][e] : acc[0][e]) + xch_r[e * 32];
              const __nv_bfloat16 hi = __float2bfloat16_rn(v);
              __nv_bfloat16* we = w + (e & 1) * (kTsWqRow / 2) + (e >> 1) * 8;
              we[0] = hi;
              we[16 * kTsWqRow / 2] = __float2bfloat16_rn(v - __bfloat162float(hi));
            }
          }
          __syncwarp();
          if (lane < nb) mbar_arrive(&empty_bar[slot_of(lane)]);   // this warp is done with the W boxes (it read at most its own)
          named_bar_sync(2, kTsThreads);
          slot += nb;
          if (slot >= kSlots) { slot -= kSlots; phase ^= 1; }
          nb = nb_next;
          continue;
        }
      }
    }

    if constexpr (KT > 0) {
      if ((hdr.y & HDR_W) && (KAM_TS_DIAG & 1)) {
        __syncwarp();
        if (lane < nb) mbar_arrive(&empty_bar[slot_of(lane)]);
        publish_mass();
        named_bar_sync(2, kTsThreads);
        write_state();
        slot += nb;
        if (slot >= kSlots) { slot -= kSlots; phase ^= 1; }
        nb = nb_next;
        continue;
      }
      if (hdr.y & HDR_W) {
        // ---- tail W iteration: z^T = sum of the eight warps' partials (four boxes x two head tiles) -> bf16 hi + lo;
        // O^T[this warp's 64 value columns][16 heads] += W[:, columns]^T z^T, A = the W boxes through ldmatrix.trans
        {
          float* zw = zp + (tg * KT * 16 + gq) * 16 + kh * 8 + 2 * t4;          // [box][rank][head]
#pragma unroll
          for (int kt = 0; kt < KT; ++kt) {
            if (kt < kt_seg) {
              *reinterpret_cast<float2*>(zw + kt * 256) = make_float2(Z[kt][0], Z[kt][1]);
              *reinterpret_cast<float2*>(zw + kt * 256 + 128) = make_float2(Z[kt][2], Z[kt][3]);
            }
          }
        }
        publish_mass();
        named_bar_sync(2, kTsThreads);
        for (int idx = threadIdx.x; idx < kt_seg * 256; idx += kTsThreads) {
          const int r = idx >> 4, h = idx & 15;
          const float v = (zp[idx] + zp[KT * 256 + idx]) + (zp[2 * KT * 256 + idx] + zp[3 * KT * 256 + idx]);
          const __nv_bfloat16 hi = __float2bfloat16_rn(v);
          __nv_bfloat16* w = reinterpret_cast<__nv_bfloat16*>(smem + kTsOffWq + h * kTsWqRow) + r;
          w[0] = hi;
          w[16 * kTsWqRow / 2] = __float2bfloat16_rn(v - __bfloat162float(hi));
        }
        named_bar_sync(2, kTsThreads);
        if (lane < nb && lane != tg) mbar_wait(&full_bar[slot_of(lane)], phase_of(lane));   // the other rank tiles' boxes
        __syncwarp();
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) {
          if (kt < kt_seg) {
            uint32_t zb[2][4];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) ldmatrix_x4(zb[nt][0], zb[nt][1], zb[nt][2], zb[nt][3], wq_ld + nt * 8 * kTsWqRow + kt * 32);
            const uint32_t wv = sm0 + static_cast<uint32_t>(kOffBox + slot_of(kt) * kStride + v_row * kTsWRow + warp * 128 + v_hi * 16);
#pragma unroll
            for (int n = 0; n < 4; ++n) {
              uint32_t a0, a1, a2, a3;
              ldmatrix_x4_trans(a0, a1, a2, a3, wv + n * 32);
#pragma unroll
              for (int nt = 0; nt < 2; ++nt) {
                mma_bf16_16816(O[nt][n][0], O[nt][n][1], O[nt][n][2], O[nt][n][3], a0, a1, a2, a3, zb[nt][0], zb[nt][1]);
                mma_bf16_16816(O[nt][n][0], O[nt][n][1], O[nt][n][2], O[nt][n][3], a0, a1, a2, a3, zb[nt][2], zb[nt][3]);
              }
            }
          }
        }
        __syncwarp();
        if (lane < nb) mbar_arrive(&empty_bar[slot_of(lane)]);
        write_state();
        slot += nb;
        if (slot >= kSlots) { slot -= kSlots; phase ^= 1; }
        nb = nb_next;
        continue;
      }
    }

    // ---- S^T[16 tokens of box tg][16 heads] over this warp's 18 k-steps; the two k-halves of a box swap the head half the
    // other one owns (4 values per lane through shared memory, one 64-thread barrier): complete scores of 8 heads per warp
    float s[4] = {-CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F};
    if (tg < nb) {
      const int4 h2 = hdr;
      const uint32_t kb = sm0 + static_cast<uint32_t>(kOffBox + my_box * kStride);
      const bool partial = h2.y & HDR_PARTIAL;
      const int row_lo = h2.z & 0xff, row_hi = h2.z >> 8;
      float sc[2][2][4];                                           // [head tile][chain: k-step parity]
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int c = 0; c < 2; ++c) sc[nt][c][0] = sc[nt][c][1] = sc[nt][c][2] = sc[nt][c][3] = 0.f;
      [[maybe_unused]] uint32_t ua = 0;                              // this lane's ldmatrix row of the box's U tile; 0: no patch here
      if constexpr (KT > 0) {
        if (kt_seg KAM_TS_SKIP_ITER KAM_TS_SKIP_S) {
          // s_t += U[t,:] . (W q): the tile's U rows are rank/16 more k-steps of the score contraction (A = U rows, B = wq^T) -
          // k-half 0 takes wq's bf16 hi part, k-half 1 the lo part, each for all 16 heads, inside the same accumulator chains.
          // Rows outside the chunk were not copied: both warps of the box clear them first (the same zeros): 0 * NaN must not reach z
          uint8_t* ub = smem + kOffBox + my_box * kStride + kTsBox;
          if (partial) {
            constexpr int cpr = KT * 2;                            // 16-byte chunks per U row
            for (int idx = lane; idx < 16 * cpr; idx += 32) {
              const int r = idx / cpr;
              if (r < row_lo || r >= row_hi) *reinterpret_cast<uint4*>(ub + idx * 16) = make_uint4(0, 0, 0, 0);
            }
            __syncwarp();
          }
          ua = kb + static_cast<uint32_t>(kTsBox + k_row * kURow + k_hi * 16);
        }
      }
      auto qk_half = [&](auto KH) {
        constexpr int H = decltype(KH)::value;                     // compile-time k-half: every ldmatrix address is base + immediate
        constexpr int NB6 = 3;                                     // 18 k-steps in 3 batches of 6: batch c + 1 is fetched under the MMAs of batch c
        uint32_t a[2][6][4];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
          const int c = 18 * H + k;
          ldmatrix_x4(a[0][k][0], a[0][k][1], a[0][k][2], a[0][k][3], kb + koff[c & 3] + (c >> 2) * 2048);
        }
        if constexpr (KT > 0) {
          if (ua) {
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) {
              if (kt < kt_seg) {
                uint32_t uf[4], wf[4];
                ldmatrix_x4(uf[0], uf[1], uf[2], uf[3], ua + kt * 32);
                ldmatrix_x4(wf[0], wf[1], wf[2], wf[3], wq_ld2 + H * 16 * kTsWqRow + kt * 32);
                mma_bf16_16816(sc[0][kt & 1][0], sc[0][kt & 1][1], sc[0][kt & 1][2], sc[0][kt & 1][3], uf[0], uf[1], uf[2], uf[3], wf[0], wf[1]);
                mma_bf16_16816(sc[1][kt & 1][0], sc[1][kt & 1][1], sc[1][kt & 1][2], sc[1][kt & 1][3], uf[0], uf[1], uf[2], uf[3], wf[2], wf[3]);
              }
            }
          }
        }
#pragma unroll
        for (int bt6 = 0; bt6 < NB6; ++bt6) {
          if (bt6 + 1 < NB6) {
#pragma unroll
            for (int k = 0; k < 6; ++k) {
              const int c = 18 * H + 6 * (bt6 + 1) + k;
              ldmatrix_x4(a[(bt6 + 1) & 1][k][0], a[(bt6 + 1) & 1][k][1], a[(bt6 + 1) & 1][k][2], a[(bt6 + 1) & 1][k][3], kb + koff[c & 3] + (c >> 2) * 2048);
            }
          }
#pragma unroll
          for (int k = 0; k < 6; ++k) {
            const int i = 6 * bt6 + k;
            const uint32_t* f = a[bt6 & 1][k];
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
              mma_bf16_16816(sc[nt][i & 1][0], sc[nt][i & 1][1], sc[nt][i & 1][2], sc[nt][i & 1][3], f[0], f[1], f[2], f[3], qf[i][nt][0], qf[i][nt][1]);
              if (H == 1 && i >= 14 && use_lo)
                mma_bf16_16816(sc[nt][(i & 1) ^ 1][0], sc[nt][(i & 1) ^ 1][1], sc[nt][(i & 1) ^ 1][2], sc[nt][(i & 1) ^ 1][3], f[0], f[1], f[2], f[3], ql[i - 14][nt][0], ql[i - 14][nt][1]);
            }
          }
        }
      };
      if (kh) qk_half(std::integral_constant<int, 1>{}); else qk_half(std::integral_constant<int, 0>{});
      float own[4], oth[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float s0 = sc[0][0][e] + sc[0][1][e], s1 = sc[1][0][e] + sc[1][1][e];
        own[e] = kh ? s1 : s0;
        oth[e] = kh ? s0 : s1;
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) xch_w[e * 32] = oth[e];
      named_bar_sync(4 + tg, 64);
      float sa[4], sb[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) { sa[e] = own[e]; sb[e] = xch_r[e * 32]; }
      const bool ok0 = !partial || (gq >= row_lo && gq < row_hi);
      const bool ok1 = !partial || (gq + 8 >= row_lo && gq + 8 < row_hi);
      s[0] = ok0 ? (sa[0] + sb[0]) * scale_log2 : -CUDART_INF_F;
      s[1] = ok0 ? (sa[1] + sb[1]) * scale_log2 : -CUDART_INF_F;
      s[2] = ok1 ? (sa[2] + sb[2]) * scale_log2 : -CUDART_INF_F;
      s[3] = ok1 ? (sa[3] + sb[3]) * scale_log2 : -CUDART_INF_F;
      if (partial) {
        // rows outside the chunk may hold anything (a neighbouring chunk, an unwritten page): 0 * NaN must not reach O.  The two
        // warps of this box clear the latent columns of those rows (4 blocks each); the other warp's score MMAs may still read
        // them - its scores of those rows are masked too.
        uint8_t* bptr = smem + kOffBox + my_box * kStride + hh * 4 * 2048;
        for (int idx = lane; idx < 16 * 32; idx += 32) {
          const int r = idx >> 5, j = idx & 31;                  // token row, 16-byte chunk of this warp's 4 blocks
          if (r < row_lo || r >= row_hi) *reinterpret_cast<uint4*>(bptr + (j >> 3) * 2048 + r * 128 + ((j & 7) << 4)) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async();
      }
    }

    // ---- P^T with the current references; one barrier publishes it and tells whether a reference must move
    bool need = false;
    float pv[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      need |= s[e] > m_ref[e & 1] + 8.f;
      pv[e] = ex2(s[e] - (m_ref[e & 1] == -CUDART_INF_F ? 0.f : m_ref[e & 1]));
    }
    uint8_t* pb = smem + pbuf * kTsPBuf;
    if (tg < nb) {
      *reinterpret_cast<uint32_t*>(pb + p_st) = pack_bf16x2(pv[0], pv[1]);
      *reinterpret_cast<uint32_t*>(pb + p_st + 8 * kTsPRow) = pack_bf16x2(pv[2], pv[3]);
    }
    if (bar_or(1, need)) {
      // ---- slow path (first iteration of a segment, then rare): tile maxima -> new references -> P again, O rescaled
      float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
      mx0 = col_max(mx0); mx1 = col_max(mx1);
      if (gq == 0) { red[warp * 8 + 2 * t4] = mx0; red[warp * 8 + 2 * t4 + 1] = mx1; }
      named_bar_sync(2, kTsThreads);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const float* r0 = red + hh * 32 + 2 * t4 + e;
        const float tm = fmaxf(fmaxf(r0[0], r0[8]), fmaxf(r0[16], r0[24]));
        const float mn = tm > m_ref[e] + 8.f ? tm : m_ref[e];
        const float al = mn == m_ref[e] ? 1.f : ex2(m_ref[e] - mn);
        l_run[e] *= al;
        if constexpr (KT > 0) {                                    // z of this warp's head tile follows its own heads' references
#pragma unroll
          for (int kt = 0; kt < KT; ++kt) { Z[kt][e] *= al; Z[kt][2 + e] *= al; }
        }
        m_ref[e] = mn;
        if (tg == 0 && gq == 0) alpha_s[hh * 8 + 2 * t4 + e] = al;
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) pv[e] = ex2(s[e] - (m_ref[e & 1] == -CUDART_INF_F ? 0.f : m_ref[e & 1]));
      if (tg < nb) {
        *reinterpret_cast<uint32_t*>(pb + p_st) = pack_bf16x2(pv[0], pv[1]);
        *reinterpret_cast<uint32_t*>(pb + p_st + 8 * kTsPRow) = pack_bf16x2(pv[2], pv[3]);
      }
      named_bar_sync(2, kTsThreads);
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        const float a0 = alpha_s[nt * 8 + 2 * t4], a1 = alpha_s[nt * 8 + 2 * t4 + 1];
#pragma unroll
        for (int n = 0; n < 4; ++n) { O[nt][n][0] *= a0; O[nt][n][1] *= a1; O[nt][n][2] *= a0; O[nt][n][3] *= a1; }
      }
    }
    l_run[0] += pv[0] + pv[2];
    l_run[1] += pv[1] + pv[3];

    // ---- O^T[this warp's 64 value columns][16 heads] += V^T P^T over the iteration's boxes; a box returns to the producer
    // as soon as this warp's MMAs on it are issued (they consumed its fragments)
    {
      const uint32_t pl = p_ld + static_cast<uint32_t>(pbuf * kTsPBuf);
      const uint32_t box0 = sm0 + static_cast<uint32_t>(kOffBox);
      // KT > 0: z^T[rank][this warp's head tile] += U^T P^T over the 16 tokens of this warp's OWN box: A = its U rows through
      // ldmatrix.trans, B = the P^T fragment of (box tg, head tile hh).  The fragments are fetched with the PV prologue and
      // multiplied behind the first box's MMAs (their latency stays off the iteration's critical path)
      [[maybe_unused]] uint32_t zu = 0;
      if constexpr (KT > 0) {
        if (kt_seg && tg < nb KAM_TS_SKIP_ITER KAM_TS_SKIP_Z)
          zu = box0 + static_cast<uint32_t>(my_box * kStride + kTsBox + v_row * kURow + v_hi * 16);
      }
      [[maybe_unused]] uint32_t zb[4], za[KTA][4];
      auto z_fetch = [&]() {
        if constexpr (KT > 0) {
          if (zu) {
            ldmatrix_x4_trans(zb[0], zb[1], zb[2], zb[3], pl + tg * (kDecTile * kTsPRow));
#pragma unroll
            for (int kt = 0; kt < KT; ++kt)
              if (kt < kt_seg) ldmatrix_x4_trans(za[kt][0], za[kt][1], za[kt][2], za[kt][3], zu + kt * 32);
          }
        }
      };
      auto z_mma = [&]() {
        if constexpr (KT > 0) {
          if (zu) {
#pragma unroll
            for (int kt = 0; kt < KT; ++kt)
              if (kt < kt_seg) mma_bf16_16816(Z[kt][0], Z[kt][1], Z[kt][2], Z[kt][3], za[kt][0], za[kt][1], za[kt][2], za[kt][3], hh ? zb[2] : zb[0], hh ? zb[3] : zb[1]);
          }
        }
      };
      if (nb == kTsIter) {
        // full iteration, straight-line,
        // P^T fragments of all four k-steps up front, V^T fragments of box j + 1 fetched under the MMAs of box j
        // the other boxes: their owners waited for them before the barrier above, this look orders OUR reads - lanes 0-3 take one
        // barrier each (one pass instead of three waits in a row), __syncwarp orders the other lanes behind them
        if (lane < kTsIter && lane != tg) mbar_wait(&full_bar[slot_of(lane)], phase_of(lane));
        __syncwarp();
        uint32_t vb[kTsIter];
#pragma unroll
        for (int j = 0; j < kTsIter; ++j) vb[j] = box0 + static_cast<uint32_t>(slot_of(j) * kStride);
        uint32_t b[kTsIter][4];
#pragma unroll
        for (int j = 0; j < kTsIter; ++j) ldmatrix_x4_trans(b[j][0], b[j][1], b[j][2], b[j][3], pl + j * (kDecTile * kTsPRow));
        uint32_t a[2][4][4];
#pragma unroll
        for (int n = 0; n < 4; ++n) ldmatrix_x4_trans(a[0][n][0], a[0][n][1], a[0][n][2], a[0][n][3], vb[0] + voff[n]);
        z_fetch();
#pragma unroll
        for (int j = 0; j < kTsIter; ++j) {
          if (j + 1 < kTsIter) {
#pragma unroll
            for (int n = 0; n < 4; ++n)
              ldmatrix_x4_trans(a[(j + 1) & 1][n][0], a[(j + 1) & 1][n][1], a[(j + 1) & 1][n][2], a[(j + 1) & 1][n][3], vb[j + 1] + voff[n]);
          }
#pragma unroll
          for (int n = 0; n < 4; ++n) {
            const uint32_t* f = a[j & 1][n];
            mma_bf16_16816(O[0][n][0], O[0][n][1], O[0][n][2], O[0][n][3], f[0], f[1], f[2], f[3], b[j][0], b[j][1]);
            mma_bf16_16816(O[1][n][0], O[1][n][1], O[1][n][2], O[1][n][3], f[0], f[1], f[2], f[3], b[j][2], b[j][3]);
          }
          if (j == 0) z_mma();                                    // before any box of the iteration is released
          if (lane == 0) mbar_arrive(&empty_bar[slot_of(j)]);
        }
      } else {
        // short iteration at the end of a segment
        z_fetch();
        z_mma();
        for (int j = 0; j < nb; ++j) {
          const int sl = slot_of(j);
          if (j != tg) mbar_wait(&full_bar[sl], phase_of(j));
          const uint32_t vbj = box0 + static_cast<uint32_t>(sl * kStride);
          uint32_t b[4];
          ldmatrix_x4_trans(b[0], b[1], b[2], b[3], pl + j * (kDecTile * kTsPRow));
#pragma unroll
          for (int n = 0; n < 4; ++n) {
            uint32_t f[4];
            ldmatrix_x4_trans(f[0], f[1], f[2], f[3], vbj + voff[n]);
            mma_bf16_16816(O[0][n][0], O[0][n][1], O[0][n][2], O[0][n][3], f[0], f[1], f[2], f[3], b[0], b[1]);
            mma_bf16_16816(O[1][n][0], O[1][n][1], O[1][n][2], O[1][n][3], f[0], f[1], f[2], f[3], b[2], b[3]);
          }
          if (lane == 0) mbar_arrive(&empty_bar[sl]);
        }
      }
    }
    pbuf ^= 1;
    slot += nb;
    if (slot >= kSlots) { slot -= kSlots; phase ^= 1; }
    nb = nb_next;

    if (hdr.y & HDR_LAST) {                                     // (a patched segment ends with its tail W iteration instead)
      publish_mass();
      named_bar_sync(2, kTsThreads);
      write_state();
    }
  }
}

namespace {
template <typename F> void mla_ts_dispatch(int kt, F&& f) {
  switch (kt) {
    case 0: f(kam_mla_ts_decode_kernel<0>, TsMap<0>::smem); break;
    case 1: f(kam_mla_ts_decode_kernel<1>, TsMap<1>::smem); break;
    case 2: f(kam_mla_ts_decode_kernel<2>, TsMap<2>::smem); break;
    default: f(kam_mla_ts_decode_kernel<4>, TsMap<4>::smem); break;
  }
}
}  // namespace

int mla_ts_smem_bytes(int kt) {
  int n = 0;
  mla_ts_dispatch(kt, [&](auto, int smem) { n = smem; });
  return n;
}

void launch_mla_ts_decode(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st) {
  mla_ts_dispatch(g.KT, [&](auto kern, int smem) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    launch_ex(kern, g.n_ctas, kTsBlock, smem, pdl, st, g, p);
  });
}

}  // namespace kam

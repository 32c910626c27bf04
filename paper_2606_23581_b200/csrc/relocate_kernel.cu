// kam_relocate_patch / kam_rotate_inplace: Eq. 1 of the paper written into the paged pool.
//
// One persistent launch covers layers x chunks x token tiles.  The step is HBM-bound: every
// element of the chunk's K/V is read once and written once, plus the factors.  Design for sm_100a:
//   * 4 producer warps (K rows | V rows | U_k | U_v) stream 16*RB-token tiles into shared memory with 1-D bulk
//     async copies (cp.async.bulk, the TMA engine) behind an mbarrier ring: deep memory-level parallelism without
//     spending registers.  One elected lane issues the copies from a scalar loop (uniform registers); rows are
//     padded so that every later shared-memory access is conflict-free;
//   * 8 consumer warps take (16 tokens x <=128 columns) slabs: unpack bf16, rotate the rope band with the
//     chunk's (cos, sin) table (one fp64 sincos per (chunk, frequency), reused over tokens, heads, layers),
//     add the rank-m patch as m16n8k16 bf16 tensor-core MMAs whose accumulators START as the rotated rows
//     (so the add is free and accumulation is fp32), round to bf16 (RNE) and store 128-bit vectors straight to
//     the pool page the block table names;
//   * W (the paper's V_m^T) is staged once per (chunk, layer, head group) in shared memory with the columns of
//     each 32-group in MMA order; the permutation is chosen so that each thread owns 8 contiguous columns
//     (128-bit loads/stores) AND both members of every rope pair (so in-place rotation is race-free);
//   * the flat tile list is cut into equal contiguous ranges, one per SM; no integer division in the tile loop.
// Why not FP32 FMAs for the patch: at m=16 the patch needs 51 TFLOP/s at the HBM roofline and at m=32 95 TFLOP/s,
// against a 74 TFLOP/s FFMA peak; on the tensor pipe it is <10 % of the legacy-MMA rate.
#include <cuda_runtime.h>

#include "common.cuh"
#include "internal.h"

namespace kam {

namespace {

// Incremental (division-free) walk over the flat tile list: chunk d -> layer l -> head group hg -> kv -> token tile tt.
// kv level: only in kv-split geometry (a tile carries K rows or V rows), and only for chunks that have V rows to write.
// Survivors rotated in place inside a K+V launch use the V half of a stage for K rows too: their tiles hold 2 * TT tokens.
struct TileWalk {
  int d, l, hg, kv, tt, n_tt, n_kv, n_tokens, tile_tok;
  long long d_end;                       // first tile index of the next chunk
  __device__ __forceinline__ void set_desc(const RelocGeom& g, const RelocDescDev& desc) {
    n_tokens = desc.n_tokens;
    const bool inplace = desc.flags & FLAG_INPLACE;
    tile_tok = (inplace && g.nkv == 2 && !g.kv_split) ? 2 * g.TT : g.TT;
    n_tt = (n_tokens + tile_tok - 1) / tile_tok;
    n_kv = (g.kv_split && g.nkv == 2 && !inplace) ? 2 : 1;
  }
  __device__ __forceinline__ void init(const RelocGeom& g, int n_descs, const RelocDescDev* descs, const long long* tile_prefix, long long tile) {
    int lo = 0, hi = n_descs;            // largest d with prefix[d] <= tile
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (tile_prefix[mid] <= tile) lo = mid; else hi = mid; }
    d = lo;
    while (tile_prefix[d + 1] <= tile) ++d;            // skip empty chunks
    set_desc(g, descs[d]);
    d_end = tile_prefix[d + 1];
    const int local = static_cast<int>(tile - tile_prefix[d]);
    tt = local % n_tt;
    int uu = local / n_tt;
    kv = uu % n_kv; uu /= n_kv;
    hg = uu % g.n_hg;
    l = uu / g.n_hg;
  }
  __device__ __forceinline__ void next(const RelocGeom& g, const RelocDescDev* descs, const long long* tile_prefix, long long new_tile) {
    if (++tt < n_tt) return;
    tt = 0;
    if (++kv < n_kv) return;
    kv = 0;
    if (++hg < g.n_hg) return;
    hg = 0;
    if (++l < g.L) return;
    l = 0;
    do { ++d; } while (tile_prefix[d + 1] <= new_tile);
    set_desc(g, descs[d]);
    d_end = tile_prefix[d + 1];
  }
};

// ---- packed fp32 pairs (sm_100a FFMA2 / FMUL2): two fp32 lanes per 64-bit register pair
__device__ __forceinline__ uint64_t pk2(float lo, float hi) { uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) { uint64_t r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) { uint64_t r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

// The (cos, sin) table of a chunk is planar in shared memory: c[half] | s[half] | -s[half]  (half = d_r / 2).
// HALF: element e of `a` (column i) pairs with element e of `b` (column i + d_r/2); tab points at the thread's first
// frequency.  a' = a c - b s ; b' = a s + b c, two pairs per packed instruction.
__device__ __forceinline__ void rotate_half8(float* a, float* b, const float* tab, int half) {
  const float4 c0 = *reinterpret_cast<const float4*>(tab), c1 = *reinterpret_cast<const float4*>(tab + 4);
  const float4 s0 = *reinterpret_cast<const float4*>(tab + half), s1 = *reinterpret_cast<const float4*>(tab + half + 4);
  const float4 n0 = *reinterpret_cast<const float4*>(tab + 2 * half), n1 = *reinterpret_cast<const float4*>(tab + 2 * half + 4);
  const uint64_t C[4] = {pk2(c0.x, c0.y), pk2(c0.z, c0.w), pk2(c1.x, c1.y), pk2(c1.z, c1.w)};
  const uint64_t S[4] = {pk2(s0.x, s0.y), pk2(s0.z, s0.w), pk2(s1.x, s1.y), pk2(s1.z, s1.w)};
  const uint64_t N[4] = {pk2(n0.x, n0.y), pk2(n0.z, n0.w), pk2(n1.x, n1.y), pk2(n1.z, n1.w)};
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const uint64_t A = pk2(a[2 * e], a[2 * e + 1]), B = pk2(b[2 * e], b[2 * e + 1]);
    upk2(fma2(B, N[e], mul2(A, C[e])), a[2 * e], a[2 * e + 1]);
    upk2(fma2(A, S[e], mul2(B, C[e])), b[2 * e], b[2 * e + 1]);
  }
}
__device__ __forceinline__ void rotate_half8x2(float* a0, float* b0, float* a1, float* b1, const float* tab, int half) {
  const float4 c0 = *reinterpret_cast<const float4*>(tab), c1 = *reinterpret_cast<const float4*>(tab + 4);
  const float4 s0 = *reinterpret_cast<const float4*>(tab + half), s1 = *reinterpret_cast<const float4*>(tab + half + 4);
  const float4 n0 = *reinterpret_cast<const float4*>(tab + 2 * half), n1 = *reinterpret_cast<const float4*>(tab + 2 * half + 4);
  const uint64_t C[4] = {pk2(c0.x, c0.y), pk2(c0.z, c0.w), pk2(c1.x, c1.y), pk2(c1.z, c1.w)};
  const uint64_t S[4] = {pk2(s0.x, s0.y), pk2(s0.z, s0.w), pk2(s1.x, s1.y), pk2(s1.z, s1.w)};
  const uint64_t N[4] = {pk2(n0.x, n0.y), pk2(n0.z, n0.w), pk2(n1.x, n1.y), pk2(n1.z, n1.w)};
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    uint64_t A = pk2(a0[2 * e], a0[2 * e + 1]), B = pk2(b0[2 * e], b0[2 * e + 1]);
    upk2(fma2(B, N[e], mul2(A, C[e])), a0[2 * e], a0[2 * e + 1]);
    upk2(fma2(A, S[e], mul2(B, C[e])), b0[2 * e], b0[2 * e + 1]);
    A = pk2(a1[2 * e], a1[2 * e + 1]); B = pk2(b1[2 * e], b1[2 * e + 1]);
    upk2(fma2(B, N[e], mul2(A, C[e])), a1[2 * e], a1[2 * e + 1]);
    upk2(fma2(A, S[e], mul2(B, C[e])), b1[2 * e], b1[2 * e + 1]);
  }
}
// INTERLEAVED: columns (2i, 2i+1) are adjacent inside one 8-vector; tab points at the thread's first frequency.
__device__ __forceinline__ void rotate_inter8x2(float* a0, float* a1, const float* tab, int half) {
  const float4 c = *reinterpret_cast<const float4*>(tab), s = *reinterpret_cast<const float4*>(tab + half);
  const float cc[4] = {c.x, c.y, c.z, c.w}, ss[4] = {s.x, s.y, s.z, s.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float x = a0[2 * i], y = a0[2 * i + 1];
    a0[2 * i] = fmaf(x, cc[i], -y * ss[i]);
    a0[2 * i + 1] = fmaf(x, ss[i], y * cc[i]);
    x = a1[2 * i]; y = a1[2 * i + 1];
    a1[2 * i] = fmaf(x, cc[i], -y * ss[i]);
    a1[2 * i + 1] = fmaf(x, ss[i], y * cc[i]);
  }
}

// One 32-column group: 4 n-tiles of m16n8k16.  w01 / w23 = B fragments (b0, b1) of n-tiles (0,1) / (2,3).
__device__ __forceinline__ void mma_group(float* r0, float* r1, const uint32_t* a, const uint32_t* w01, const uint32_t* w23) {
  mma_bf16_16816(r0[0], r0[1], r1[0], r1[1], a[0], a[1], a[2], a[3], w01[0], w01[1]);
  mma_bf16_16816(r0[2], r0[3], r1[2], r1[3], a[0], a[1], a[2], a[3], w01[2], w01[3]);
  mma_bf16_16816(r0[4], r0[5], r1[4], r1[5], a[0], a[1], a[2], a[3], w23[0], w23[1]);
  mma_bf16_16816(r0[6], r0[7], r1[6], r1[7], a[0], a[1], a[2], a[3], w23[2], w23[3]);
}

enum : int { ROPE_NONE = 0, ROPE_HALF = 1, ROPE_INTER = 2 };

// What one consumer warp needs to process a slab (16 tokens x one column block), beyond the template parameters.
struct SlabArgs {
  const uint8_t* rows;       // this thread's first vector: token row (lane / 4), 16-byte column slot (lane % 4) of group 0
  char* dst0;                // pool address of the same vector for token row lane/4, and for row lane/4 + 8
  char* dst1;
  const float* tab;          // the thread's first table entry for group 0 of the block (HALF: frequency; INTER: column / 2)
  uint32_t wb;               // shared address of this lane's ldmatrix row of W (k-tile 0, group 0)
  int s_row, w_row16, half;  // token stride in the stage; bytes of 16 k-rows of W; d_r / 2
  int steps;                 // pairs of 32-column groups
  bool ok0, ok1, canonical;
  // ranks that are not a multiple of 16: the A fragments are gathered element by element, columns >= m_rag read as zero
  // (the W rows behind them are zero in shared memory too, so the padded products vanish exactly)
  const uint8_t* ug;         // U[token row lane/4][head][0] of this slab in the stage
  int su;                    // token stride of U in the stage (bytes)
  int m_rag;                 // 0: rank is a multiple of 16 (ldmatrix path); else the rank
};

// A step = two 32-column groups (gA, gB) x 16 tokens: HALF pairs group sp with group sp + steps (column i with i + d_r/2).
template <int KT, int ROPE, int STEPS>
__device__ __forceinline__ void slab_steps(const SlabArgs& s, const uint32_t (*afr)[4]) {
#pragma unroll
  for (int sp = 0; sp < STEPS; ++sp) {                                          // independent steps: unrolled for ILP
    const int offA = (ROPE == ROPE_HALF ? sp : 2 * sp) * 64;
    const int offB = (ROPE == ROPE_HALF ? sp + STEPS : 2 * sp + 1) * 64;
    float a0[8], a1[8], b0[8], b1[8];
    unpack8(*reinterpret_cast<const uint4*>(s.rows + offA), a0);
    unpack8(*reinterpret_cast<const uint4*>(s.rows + 8 * s.s_row + offA), a1);
    unpack8(*reinterpret_cast<const uint4*>(s.rows + offB), b0);
    unpack8(*reinterpret_cast<const uint4*>(s.rows + 8 * s.s_row + offB), b1);
    auto rotate = [&]() {
      if constexpr (ROPE == ROPE_HALF) {
        rotate_half8x2(a0, b0, a1, b1, s.tab + (offA >> 1), s.half);            // 32 frequencies per group
      } else if constexpr (ROPE == ROPE_INTER) {
        rotate_inter8x2(a0, a1, s.tab + (offA >> 2), s.half);                   // 16 frequencies per group
        rotate_inter8x2(b0, b1, s.tab + (offB >> 2), s.half);
      }
    };
    if (ROPE != ROPE_NONE && !s.canonical) rotate();                            // Eq. 1: rotate, then add the patch
#pragma unroll
    for (int kt = 0; kt < KT; ++kt) {
      uint32_t wA[8], wB[8];
      const uint32_t base = s.wb + kt * s.w_row16;
      ldmatrix_x4_trans(wA[0], wA[1], wA[2], wA[3], base + offA);
      ldmatrix_x4_trans(wA[4], wA[5], wA[6], wA[7], base + offA + 32);
      ldmatrix_x4_trans(wB[0], wB[1], wB[2], wB[3], base + offB);
      ldmatrix_x4_trans(wB[4], wB[5], wB[6], wB[7], base + offB + 32);
      mma_group(a0, a1, afr[kt], wA, wA + 4);
      mma_group(b0, b1, afr[kt], wB, wB + 4);
    }
    if (ROPE != ROPE_NONE && s.canonical) rotate();                             // patch stored in the chunk's own frame (R-4)
    if (s.ok0) { st_global_v4(s.dst0 + offA, pack8(a0)); st_global_v4(s.dst0 + offB, pack8(b0)); }
    if (s.ok1) { st_global_v4(s.dst1 + offA, pack8(a1)); st_global_v4(s.dst1 + offB, pack8(b1)); }
  }
}

template <int KT>
__device__ __forceinline__ void slab_run(const SlabArgs& s, int rope, uint32_t ua) {
  uint32_t afr[KT > 0 ? KT : 1][4];
#ifdef KAM_VAR_NORAG
  if (false) {
#else
  if (KT > 0 && s.m_rag) {
#endif
    const int t4 = threadIdx.x & 3;
#pragma unroll
    for (int kt = 0; kt < KT; ++kt)
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int k0 = kt * 16 + 2 * t4 + (r >> 1) * 8;
        const uint16_t* row = reinterpret_cast<const uint16_t*>(s.ug + (r & 1) * 8 * s.su);
        const uint32_t lo = k0 < s.m_rag ? row[k0] : 0u, hi = k0 + 1 < s.m_rag ? row[k0 + 1] : 0u;
        afr[kt][r] = lo | (hi << 16);
      }
  } else {
#pragma unroll
    for (int kt = 0; kt < KT; ++kt) ldmatrix_x4(afr[kt][0], afr[kt][1], afr[kt][2], afr[kt][3], ua + kt * 32);
  }
  if (s.steps == 2) {
    if (rope == ROPE_NONE) slab_steps<KT, ROPE_NONE, 2>(s, afr);
    else if (rope == ROPE_HALF) slab_steps<KT, ROPE_HALF, 2>(s, afr);
    else slab_steps<KT, ROPE_INTER, 2>(s, afr);
  } else {
    if (rope == ROPE_NONE) slab_steps<KT, ROPE_NONE, 1>(s, afr);
    else if (rope == ROPE_HALF) slab_steps<KT, ROPE_HALF, 1>(s, afr);
    else slab_steps<KT, ROPE_INTER, 1>(s, afr);
  }
}

}  // namespace

// Shared-memory map (dynamic): [0,128) mbarriers | slab table | cos/sin table | W (column-permuted, padded rows) | stages.
// W in shared memory is [kv][head-in-group][k < 16 * KT][D + 8] bf16 (rows k >= m are zero: the rank is padded to a multiple of
// 16 there, never in HBM) with the columns of every 32-group stored in MMA order (position 8j + 2i + e holds column
// 8i + 2j + e), so that ldmatrix.trans yields B fragments whose accumulator columns are 8 CONTIGUOUS columns per thread.
// A stage is [K rows | V rows | U_k | U_v | slots]; three tile forms share it:
//   K+V tile     (a chunk with V, plain geometry)   : TT tokens, K rows and V rows of the same tokens
//   in-place x2  (a survivor inside a K+V launch)   : 2 * TT tokens of K; the second half lands in the V area, so a slide's
//                                                     survivors keep a full stage of bytes in flight beside the recalled chunk
//   kv-split     (ranks 48 / 64)                    : TT tokens of K or of V in the K area, its U in the U_k area
namespace {
// pages: the page list of a chunk being admitted to a window, or nullptr (the stateless calls: their kernel has no such parameter)
__device__ __forceinline__ void relocate_body(const RelocGeom& g, const RelocParams& p, const RelocInline& inl, const RelocPages* pages) {
  extern __shared__ __align__(128) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + g.n_stages;
  int4* slab_tab = reinterpret_cast<int4*>(smem + g.off_tab);
  float* tab = reinterpret_cast<float*>(smem + g.off_cs);
  uint8_t* wsm = smem + g.off_w;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < g.n_stages; ++s) { mbar_init(&full_bar[s], kRelocProducerWarps); mbar_init(&empty_bar[s], kRelocConsumerWarps); }
    mbar_fence_init();
  }
  if (threadIdx.x < 2 * g.RB * g.n_blocks) {
    // slab s -> (half, row block, column block); everything a consumer needs, as byte offsets.  half = 1: the V rows of a
    // K+V tile, or the second TT tokens of an in-place x2 tile.  The rope kind is the block's; V slabs ignore it.
    const int s = threadIdx.x, per = g.RB * g.n_blocks;
    const int kv = s / per, rem = s - kv * per, rb = rem / g.n_blocks;
    const ColBlock cb = g.blk[rem % g.n_blocks];
    const int rope = cb.rope ? (g.rope_style == KAM_ROPE_HALF ? ROPE_HALF : ROPE_INTER) : ROPE_NONE;
    const int tab_off = g.rope_style == KAM_ROPE_HALF ? cb.band_col0 : cb.band_col0 >> 1;       // first frequency of the block
    slab_tab[s] = make_int4(kv | (rb << 4) | (cb.fhead << 8) | (rope << 16) | ((cb.n_groups >> 1) << 20),
                            cb.col_off * 2, cb.w_col_off * 2, tab_off);
  }
  __syncthreads();
  // Programmatic dependent launch: everything above (barrier init, slab table) may run under the tail of the previous kernel on
  // the stream; nothing below - the first global read or write - starts before that kernel has completed.  The next kernel is
  // released at once: its prologue then hides under this kernel's tail in the same way (one CTA per SM and ~220 KB of shared
  // memory: it cannot become resident before a CTA of this kernel has left).
  grid_dep_wait();
  grid_dep_launch();

  // small batches carry their descriptors in the kernel parameters (no H2D staging copy, no global loads to read them)
  const RelocDescDev* descs = p.descs ? p.descs : inl.d;
  const long long* tile_prefix = p.descs ? p.tile_prefix : inl.prefix;
  const long long* w_prefix = p.descs ? p.w_prefix : inl.wprefix;
  // the page list of a chunk just admitted to a window: CTA 0 publishes it to the device mirror (read by later launches only)
  if (pages && blockIdx.x == 0)
    for (int i = threadIdx.x; i < pages->n; i += blockDim.x) pages->mirror_dst[i] = pages->pages[i];
  // CTA i owns the tiles whose cumulative WEIGHT falls in [W i / n, W (i+1) / n): tiles of one chunk weigh the same, tiles of
  // different chunks do not (a survivor rotated in place moves K only and runs no MMA; a recalled chunk moves K, V, U and runs
  // the patch) - equal COUNTS left the CTAs of a slide 13 % apart (profiles/ncu_slide_r02.md)
  auto cut = [&](unsigned i) -> long long {
    if (i >= gridDim.x) return p.total_tiles;
    const long long b = p.total_weight * i / gridDim.x;
    int lo = 0, hi = p.n_descs;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (w_prefix[mid] <= b) lo = mid; else hi = mid; }
    while (lo + 1 < p.n_descs && w_prefix[lo + 1] <= b) ++lo;
    const int tw = descs[lo].tile_weight;
    const long long t = tile_prefix[lo] + (tw > 0 ? (b - w_prefix[lo]) / tw : 0);
    return t < tile_prefix[lo + 1] ? t : tile_prefix[lo + 1];
  };
  const long long t_begin = cut(blockIdx.x), t_end = cut(blockIdx.x + 1);
  if (t_begin >= t_end) return;
  TileWalk w;
  w.init(g, p.n_descs, descs, tile_prefix, t_begin);
  const bool split = g.kv_split;

  if (warp >= kRelocConsumerWarps) {
    // ================================================================ producer warps: K | V | U_k | U_v
    // Copies are issued lane-parallel (lane r owns token row r, or the run of rows that starts at r); the block-table
    // entries of a tile are loaded BEFORE the wait for a free stage, so their latency hides behind it.
    const int role = warp - kRelocConsumerWarps;
    int stage = 0; uint32_t phase = 0;
    int cur_d = -1, cur_l = -1, cur_kv = -1;
    // per (chunk, layer[, kv]) state
    const char* src = nullptr; const int32_t* bt = nullptr;
    long long u_tok_stride = 0, u_head_stride = 0;
    int dst0 = 0, m = 0, flags = 0;
    bool dbl = false;                      // in-place x2 tile form
    for (long long tile = t_begin; tile < t_end; ++tile) {
      if (w.d != cur_d || w.l != cur_l || w.kv != cur_kv) {
        cur_d = w.d; cur_l = w.l; cur_kv = w.kv;
        const RelocDescDev& desc = descs[w.d];
        flags = desc.flags; m = desc.rank_l[w.l]; dst0 = static_cast<int>(desc.dst_token_start);
        bt = (pages && (flags & FLAG_INLINE_PAGES)) ? pages->pages : desc.block_table;
        u_tok_stride = desc.u_token_stride; u_head_stride = desc.u_head_stride;
        const bool inplace = flags & FLAG_INPLACE;
        dbl = inplace && g.nkv == 2 && !split;
        // what this warp streams for this (chunk, layer, kv): sel 0 = K rows, 1 = V rows, 2 = U_k, 3 = U_v, -1 = nothing
        int sel = role;
        if (split) sel = (role & 1) ? -1 : role + w.kv;
        src = nullptr;
        if (sel == 0) src = inplace ? static_cast<const char*>(p.pool_k[w.l]) : static_cast<const char*>(desc.k_src[w.l]);
        else if (sel == 1) {
          if (dbl) src = static_cast<const char*>(p.pool_k[w.l]);
          else if (!inplace && g.nkv == 2) src = static_cast<const char*>(desc.v_src[w.l]);
        } else if (sel >= 2) {
          const void* const* tab_l = sel == 2 ? desc.Uk : desc.Uv;
          if (m && tab_l && !inplace && (sel == 2 || g.nkv == 2)) src = static_cast<const char*>(tab_l[w.l]);
          if (src) {
            // the consumers stage this (chunk, layer)'s W a few tiles from now: pull it into L2 ahead of them
            const void* const* Wt = sel == 2 ? desc.Wk : desc.Wv;
            const size_t wbytes = static_cast<size_t>(g.HG) * m * g.D * 2;
            const char* wp = static_cast<const char*>(Wt[w.l]) + static_cast<size_t>(w.hg) * wbytes;
            for (size_t o = static_cast<size_t>(lane) * 128; o < wbytes; o += 32 * 128)
              asm volatile("prefetch.global.L2 [%0];" ::"l"(wp + o));
          }
        }
      }
      const bool inplace = flags & FLAG_INPLACE;
      const bool rows_role = role <= 1;
      const bool second = dbl && role == 1;                      // this warp streams tokens [TT, 2 TT) of the tile
      const int tok0 = w.tt * w.tile_tok + (second ? g.TT : 0);
      const int nvalid = max(0, min(g.TT, w.n_tokens - tok0));
      // A1 slot mapping: g = dst_token_start + t -> page = block_table[g / P], slot = page * P + g % P   (TT <= 64: 2 rows per lane)
      // A page outside the pool is never written (slot -1) and never read (row 0 stands in); it is counted once per table entry.
      int slot_lo = -1, slot_hi = -1, rd_lo = 0, rd_hi = 0;
      if (role == 0 || second) {
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          const int r = lane + 32 * hf;
          if (r < nvalid) {
            const int gt = dst0 + tok0 + r;
            const int pg = g.P_shift >= 0 ? (gt >> g.P_shift) : gt / g.P;
            const int in_pg = gt - pg * g.P;
#ifdef KAM_VAR_LDG
            const int page = (flags & FLAG_INLINE_PAGES) ? bt[pg] : __ldg(bt + pg);
#else
            const int page = bt[pg];             // generic load: the list may sit in the kernel parameters
#endif
            int slot = -1, rd = 0;
            if (static_cast<unsigned>(page) < static_cast<unsigned>(p.num_pages)) { slot = page * g.P + in_pg; rd = slot; }
            else if (p.err && w.l == 0 && w.hg == 0 && w.kv == 0 && (in_pg == 0 || tok0 + r == 0)) atomicAdd(p.err, 1);
            if (hf) { slot_hi = slot; rd_hi = rd; } else { slot_lo = slot; rd_lo = rd; }
          }
        }
      }
      mbar_wait(&empty_bar[stage], phase ^ 1);
      uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
      uint64_t* fb = &full_bar[stage];
      if (rows_role) {
        if (role == 0 || second) {
          int32_t* slots = reinterpret_cast<int32_t*>(st + g.st_slot) + (second ? g.TT : 0);
          if (lane < g.TT) slots[lane] = slot_lo;
          if (lane + 32 < g.TT) slots[lane + 32] = slot_hi;
          __syncwarp();                              // every lane's slots are written before lane 0 arrives on the barrier
        }
        if (src == nullptr || nvalid == 0) {
          if (lane == 0) mbar_arrive(fb);
        } else {
          if (lane == 0) mbar_arrive_expect_tx(fb, static_cast<uint32_t>(nvalid) * g.slice_bytes);
          __syncwarp();
          const size_t off = static_cast<size_t>(w.hg) * g.slice_bytes;
          uint8_t* dst = st + (role == 0 ? g.st_k : g.st_v);
          if (!inplace) {
            const char* s0 = src + static_cast<size_t>(tok0) * g.row_bytes + off;
            if (g.contig) {
              if (lane == 0) {
                if (g.load_hint) bulk_g2s_hint(dst, s0, static_cast<uint32_t>(nvalid) * g.slice_bytes, fb, make_policy_evict_first());
                else bulk_g2s(dst, s0, static_cast<uint32_t>(nvalid) * g.slice_bytes, fb);
              }
            }
            else for (int r = lane; r < nvalid; r += 32) bulk_g2s(dst + r * g.s_row, s0 + static_cast<size_t>(r) * g.row_bytes, g.slice_bytes, fb);
          } else if (g.contig) {
            // pool rows are contiguous inside a page: one copy per run of consecutive slots, issued by the run's first lane
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
              const int r = lane + 32 * hf;
              const int mine = hf ? rd_hi : rd_lo;
              const int prev = __shfl_up_sync(0xffffffffu, mine, 1);
              const bool valid = r < nvalid;
              const bool head = valid && (lane == 0 || mine != prev + 1);          // a run never spans the two halves
              const uint32_t heads = __ballot_sync(0xffffffffu, head), valids = __ballot_sync(0xffffffffu, valid);
              if (head) {
                const uint32_t above = heads & ~((2u << lane) - 1u);                  // run heads after this lane
                const int end = above ? __ffs(above) - 1 : __popc(valids);           // rows of this half are valid from lane 0 up
                bulk_g2s(dst + r * g.s_row, src + static_cast<size_t>(mine) * g.row_bytes, static_cast<uint32_t>(end - lane) * g.slice_bytes, fb);
              }
            }
          } else {
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
              const int r = lane + 32 * hf;
              if (r < nvalid) bulk_g2s(dst + r * g.s_row, src + static_cast<size_t>(hf ? rd_hi : rd_lo) * g.row_bytes + off, g.slice_bytes, fb);
            }
          }
        }
      } else {
        if (src == nullptr || nvalid == 0) {
          if (lane == 0) mbar_arrive(fb);
        } else {
          // U rows of this tile.  Native form: the tile's rows are one contiguous run of the caller's array ([T][..] with its own
          // token stride, all heads of the row in this slice) - ONE copy, and the consumers index it with the caller's strides.
          // Otherwise one run of (heads-in-slice * m) elements per token when the heads are adjacent, else one run per head.
          const int hf_n = (u_head_stride == 0) ? 1 : g.HG;
          const uint32_t u_run = static_cast<uint32_t>(m) * 2u, u_tok_bytes = u_run * hf_n;
          const long long h0 = (u_head_stride == 0) ? 0 : static_cast<long long>(w.hg) * g.HG;
          const char* s0 = src + (static_cast<long long>(tok0) * u_tok_stride + h0 * u_head_stride) * 2;
          uint8_t* dst = st + (role == 2 ? g.st_uk : g.st_uv);
          const bool heads_adjacent = hf_n == 1 || u_head_stride == m;
          if (u_form(g.su_row, g.HG, g.n_hg, m, u_tok_stride, u_head_stride) == U_NATIVE) {
            if (lane == 0) {
              // a ragged rank can leave < 16 bytes at the end of a chunk's last tile: those travel as plain 2-byte accesses
              const uint32_t total = static_cast<uint32_t>(nvalid) * static_cast<uint32_t>(u_tok_stride) * 2u, bulk = total & ~15u;
              for (uint32_t o = bulk; o < total; o += 2)
                *reinterpret_cast<uint16_t*>(dst + o) = __ldg(reinterpret_cast<const uint16_t*>(s0 + o));
              if (bulk) { mbar_arrive_expect_tx(fb, bulk); bulk_g2s(dst, s0, bulk, fb); }
              else mbar_arrive(fb);
            }
          } else {
            if (lane == 0) mbar_arrive_expect_tx(fb, static_cast<uint32_t>(nvalid) * u_tok_bytes);
            __syncwarp();
            if (heads_adjacent) {
              for (int r = lane; r < nvalid; r += 32) bulk_g2s(dst + r * g.su_row, s0 + r * u_tok_stride * 2, u_tok_bytes, fb);
            } else {
              for (int r = lane; r < nvalid; r += 32)
                for (int h = 0; h < hf_n; ++h)
                  bulk_g2s(dst + r * g.su_row + h * u_run, s0 + (r * u_tok_stride + h * u_head_stride) * 2, u_run, fb);
            }
          }
        }
      }
      if (++stage == g.n_stages) { stage = 0; phase ^= 1; }
      if (tile + 1 < t_end) w.next(g, descs, tile_prefix, tile + 1);
    }
    return;
  }

  // ================================================================ consumer warps
  const int gq = lane >> 2, t4 = lane & 3;
  const int ctid = threadIdx.x;                                   // 0 .. 255
  int stage = 0; uint32_t phase = 0;
  int cur_d = -1, cur_l = -1, cur_hg = -1, cur_kv = -1;
  int m = 0, m_pad = 0, flags = 0, KT = 0, su = 0, uhs = 0; bool u_shared = false, has_uk = false, has_uv = false;
  char* pool_k = nullptr; char* pool_v = nullptr;
  const int half = g.d_r >> 1;
  // ldmatrix lane addressing
  const int a_row = lane & 15, a_koff = (lane >> 4) * 8;                       // A: rows of U, k offset
  const int b_k = (lane & 7) + ((lane >> 3) & 1) * 8, b_nt = lane >> 4;         // B: k row of W, n-tile 0/1 of the pair

  for (long long tile = t_begin; tile < t_end; ++tile) {
    if (w.d != cur_d || w.l != cur_l || w.hg != cur_hg || w.kv != cur_kv) {
      // ---- new (chunk, layer, head group[, kv]): rebuild the sin/cos table (new chunk) and stage W
      const bool new_chunk = (w.d != cur_d);
      cur_d = w.d; cur_l = w.l; cur_hg = w.hg; cur_kv = w.kv;
      const RelocDescDev& desc = descs[w.d];
      flags = desc.flags; m = desc.rank_l[w.l]; KT = (m + 15) >> 4; m_pad = KT << 4;
      u_shared = desc.u_head_stride == 0;
      const bool inplace = flags & FLAG_INPLACE;
      has_uk = m && desc.Uk && !inplace; has_uv = m && desc.Uv && !inplace && g.nkv == 2;
      // strides of U in the stage: the caller's own when the tile arrived as one copy (see the producer), else padded rows of
      // head runs of m elements
      if (u_form(g.su_row, g.HG, g.n_hg, m, desc.u_token_stride, desc.u_head_stride) == U_NATIVE) { su = static_cast<int>(desc.u_token_stride) * 2; uhs = static_cast<int>(desc.u_head_stride); }
      else { su = g.su_row; uhs = m; }
      pool_k = static_cast<char*>(p.pool_k[w.l]) + static_cast<size_t>(w.hg) * g.slice_bytes;
      pool_v = g.nkv == 2 ? static_cast<char*>(p.pool_v[w.l]) + static_cast<size_t>(w.hg) * g.slice_bytes : nullptr;
      named_bar_sync(1, kRelocConsumerWarps * 32);                // everyone is done with the old tables
      if (new_chunk && ctid < half) {
        // A2: f_i = theta^(-2i/d_r); angle = delta * f_i in fp64 (positions reach 1e5: fp32 angles would cost 2 bf16 ulp)
        const double f = p.inv_freq ? p.inv_freq[ctid] : pow(g.theta, -2.0 * ctid / g.d_r);
        double sn, cs;
        sincos(static_cast<double>(desc.delta) * f, &sn, &cs);
        tab[ctid] = static_cast<float>(cs);
        tab[half + ctid] = static_cast<float>(sn);
        tab[2 * half + ctid] = -static_cast<float>(sn);
      }
      // which of W_k / W_v go to shared memory now: both (plain geometry) or the one of this tile's kv (kv-split)
      const int kv_lo = split ? w.kv : 0;
      const int kv_n = split ? ((w.kv ? has_uv : has_uk) ? 1 : 0) : (has_uk ? (has_uv ? 2 : 1) : 0);
      if (kv_n) {
        // W[l] is [H][m][D]; copy this head group's rows, 16 bytes (8 columns = 4 pairs) per thread, scattering the pairs
        // to their MMA-order positions inside the 32-column group; rows m .. m_pad-1 of every head are written as zeros.
        const int vec_per_row = g.D >> 3;
        const int per_kv = g.HG * m_pad * vec_per_row;
        const int n_vec = kv_n * per_kv;
        constexpr int kCT = kRelocConsumerWarps * 32, kBatch = 8;      // 8 independent 16-byte loads in flight per thread
        for (int e0 = ctid; e0 < n_vec; e0 += kCT * kBatch) {
          uint4 x[kBatch];
#pragma unroll
          for (int u = 0; u < kBatch; ++u) {
            const int e = e0 + u * kCT;
            x[u] = make_uint4(0u, 0u, 0u, 0u);
            if (e < n_vec) {
              const int kv = e >= per_kv;
              int r = e - kv * per_kv;
              const int v = r % vec_per_row; r /= vec_per_row;     // r = head-in-group * m_pad + k
              const int hd = r / m_pad, k = r - hd * m_pad;
              if (k < m) {
                const void* const* Wl = (kv_lo + kv) ? desc.Wv : desc.Wk;
                x[u] = __ldg(reinterpret_cast<const uint4*>(static_cast<const char*>(Wl[w.l]) +
                                                            (static_cast<size_t>(w.hg) * g.HG + hd) * m * g.D * 2 + static_cast<size_t>(k) * g.D * 2) + v);
              }
            }
          }
#pragma unroll
          for (int u = 0; u < kBatch; ++u) {
            const int e = e0 + u * kCT;
            if (e < n_vec) {
              const int kv = e >= per_kv;
              int r = e - kv * per_kv;
              const int v = r % vec_per_row; r /= vec_per_row;     // r = head-in-group * m_pad + k
              const int q = v >> 2, i = v & 3;                       // columns 32q + 8i .. +7 = pairs j = 0..3
              uint32_t* dst = reinterpret_cast<uint32_t*>(wsm + static_cast<size_t>(kv) * g.w_kv_stride + static_cast<size_t>(r) * g.w_row) + q * 16 + i;
              dst[0] = x[u].x; dst[4] = x[u].y; dst[8] = x[u].z; dst[12] = x[u].w;   // pair j lands at 32-bit position 4j + i
            }
          }
        }
      }
      named_bar_sync(1, kRelocConsumerWarps * 32);
    }

    mbar_wait(&full_bar[stage], phase);

    const uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
    const int32_t* slots = reinterpret_cast<const int32_t*>(st + g.st_slot);
    const bool inplace = flags & FLAG_INPLACE;
    const bool dbl = inplace && g.nkv == 2 && !split;
    const int n_slabs = ((g.nkv == 2 && !split && (!inplace || dbl)) ? 2 : 1) * g.RB * g.n_blocks;

    for (int s = warp; s < n_slabs; s += kRelocConsumerWarps) {
      const int4 e = slab_tab[s];
      const int hf = e.x & 0xf, rb = (e.x >> 4) & 0xf, fhead = (e.x >> 8) & 0xff;
      const int kv = split ? w.kv : (dbl ? 0 : hf);                // what the rows are: 0 = keys, 1 = values
      const int rope = kv ? ROPE_NONE : (e.x >> 16) & 0xf;
      const int row0 = rb * 16 + gq;
      const int srow = row0 + (dbl && hf ? g.TT : 0);
      const int slot0 = slots[srow], slot1 = slots[srow + 8];
      char* pool = (kv ? pool_v : pool_k) + e.y + t4 * 16;
      SlabArgs a;
      a.rows = st + (hf ? g.st_v : g.st_k) + row0 * g.s_row + e.y + t4 * 16;
      a.dst0 = pool + static_cast<size_t>(slot0 < 0 ? 0 : slot0) * g.row_bytes;
      a.dst1 = pool + static_cast<size_t>(slot1 < 0 ? 0 : slot1) * g.row_bytes;
      a.tab = tab + e.w + (rope == ROPE_HALF ? 8 * t4 : 4 * t4);
      a.s_row = g.s_row; a.w_row16 = 16 * g.w_row; a.half = half;
      a.steps = e.x >> 20;
      a.ok0 = slot0 >= 0; a.ok1 = slot1 >= 0; a.canonical = flags & FLAG_CANONICAL_FRAME;
      const int wkv = split ? 0 : kv;                               // which resident W table
      a.wb = smem_u32(wsm + static_cast<size_t>(wkv) * g.w_kv_stride + static_cast<size_t>(fhead * m_pad + b_k) * g.w_row + e.z + b_nt * 16);
      const int kt = (kv ? has_uv : has_uk) ? KT : 0;
      // A fragments of U for this slab's 16 tokens and head: one ldmatrix.x4 per 16 ranks
      const uint8_t* ubase = st + ((kv && !split) ? g.st_uv : g.st_uk) + ((u_shared ? 0 : fhead) * uhs) * 2;
      const uint32_t ua = smem_u32(ubase + (rb * 16 + a_row) * su + a_koff * 2);
      // ldmatrix needs 16-byte aligned rows of 16 k-values; anything else is gathered element by element
      a.ug = ubase + row0 * su; a.su = su; a.m_rag = ((m | (su >> 1) | uhs) & 7 || (m & 15)) ? m : 0;
      switch (kt) {
        case 0: slab_run<0>(a, rope, ua); break;
        case 1: slab_run<1>(a, rope, ua); break;
        case 2: slab_run<2>(a, rope, ua); break;
        case 3: slab_run<3>(a, rope, ua); break;
        default: slab_run<4>(a, rope, ua); break;
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[stage]);
    if (++stage == g.n_stages) { stage = 0; phase ^= 1; }
    if (tile + 1 < t_end) w.next(g, descs, tile_prefix, tile + 1);
  }
}

}  // namespace

__global__ void __launch_bounds__(kRelocThreads, 1)
kam_relocate_patch_kernel(const __grid_constant__ RelocGeom g, const __grid_constant__ RelocParams p, const __grid_constant__ RelocInline inl) {
  relocate_body(g, p, inl, nullptr);
}
// the same kernel with the admitted chunk's page list as a fourth parameter (kam_admit / kam_slide)
__global__ void __launch_bounds__(kRelocThreads, 1)
kam_relocate_admit_kernel(const __grid_constant__ RelocGeom g, const __grid_constant__ RelocParams p, const __grid_constant__ RelocInline inl,
                          const __grid_constant__ RelocPages pages) {
  relocate_body(g, p, inl, &pages);
}

void launch_relocate_fast(const RelocGeom& g, const RelocParams& p, const RelocInline& inl, const RelocPages* pages, int grid, bool pdl, cudaStream_t st) {
  static std::atomic<uint64_t> attr_done{0};          // per device: the attribute is not shared between GPUs
  if (first_launch_on_this_device(attr_done)) {
    cudaFuncSetAttribute(kam_relocate_patch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    cudaFuncSetAttribute(kam_relocate_admit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kRelocThreads); cfg.dynamicSmemBytes = g.smem_bytes; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  if (pages) cudaLaunchKernelEx(&cfg, kam_relocate_admit_kernel, g, p, inl, *pages);
  else cudaLaunchKernelEx(&cfg, kam_relocate_patch_kernel, g, p, inl);
}

// ---------------------------------------------------------------------------------------------------------------
// Generic element-wise path: any element / factor dtype, any rank <= KAM_MAX_RANK, any even rope band.  One thread
// owns a non-rotated column or BOTH columns of a rope pair (in-place safe).  Correctness path for fp32 tensors (config 1
// as written), row regions that are not multiples of 64 columns and U layouts bulk copies cannot address; every bf16
// rank <= KAM_MAX_RANK runs on the tiled kernel above, which is the one the roofline is quoted on.
template <typename T> __device__ __forceinline__ float ld_as_float(const void* p, size_t i);
template <> __device__ __forceinline__ float ld_as_float<float>(const void* p, size_t i) { return static_cast<const float*>(p)[i]; }
template <> __device__ __forceinline__ float ld_as_float<__nv_bfloat16>(const void* p, size_t i) {
  return __bfloat162float(static_cast<const __nv_bfloat16*>(p)[i]);
}
template <typename T> __device__ __forceinline__ void st_from_float(void* p, size_t i, float v);
template <> __device__ __forceinline__ void st_from_float<float>(void* p, size_t i, float v) { static_cast<float*>(p)[i] = v; }
template <> __device__ __forceinline__ void st_from_float<__nv_bfloat16>(void* p, size_t i, float v) {
  static_cast<__nv_bfloat16*>(p)[i] = __float2bfloat16_rn(v);
}

template <typename ET, typename FT>
__global__ void __launch_bounds__(256) kam_relocate_patch_generic_kernel(const __grid_constant__ GenericParams p) {
  __shared__ float2 cs[256];
  const int d = blockIdx.x / p.L, l = blockIdx.x - d * p.L;
  const RelocDescDev& desc = p.descs[d];
  const int half = p.d_r / 2;
  for (int i = threadIdx.x; i < half; i += blockDim.x) {
    const double f = pow(p.theta, -2.0 * i / p.d_r);
    double s, c;
    sincos(static_cast<double>(desc.delta) * f, &s, &c);
    cs[i] = make_float2(static_cast<float>(c), static_cast<float>(s));
  }
  __syncthreads();
  const bool inplace = desc.flags & FLAG_INPLACE;
  const bool canonical = desc.flags & FLAG_CANONICAL_FRAME;
  const int m = desc.rank_l[l];
  const int wcols = p.D - half;                       // work columns: a plain column, or a rope pair
  const int t_per_block = 8;
  const int tok0 = blockIdx.y * t_per_block;
  const int n_work = t_per_block * p.H * wcols;
  char* pk = static_cast<char*>(p.pool_k[l]);
  char* pv = p.has_v ? static_cast<char*>(p.pool_v[l]) : nullptr;
  for (int w = threadIdx.x; w < n_work; w += blockDim.x) {
    const int wc = w % wcols; int r = w / wcols;
    const int h = r % p.H; const int t = tok0 + r / p.H;
    if (t >= desc.n_tokens) continue;
    const long long gt = desc.dst_token_start + t;
    const long long pg = gt / p.P;
    const int page = desc.block_table[pg];
    if (static_cast<unsigned>(page) >= static_cast<unsigned>(p.num_pages)) {      // a page outside the pool: skipped, counted once
      if (p.err && l == 0 && h == 0 && wc == 0 && (gt == pg * p.P || t == 0)) atomicAdd(p.err, 1);
      continue;
    }
    const size_t slot = static_cast<size_t>(page) * p.P + static_cast<size_t>(gt - pg * p.P);
    const size_t dst_row = (slot * p.H + h) * p.D;
    const size_t src_row = inplace ? dst_row : (static_cast<size_t>(t) * p.H + h) * p.D;
    const void* ksrc = inplace ? static_cast<const void*>(pk) : desc.k_src[l];
    // which columns does this work item cover?
    int ca, cb = -1, fi = 0;
    if (wc < p.rope_off) ca = wc;
    else if (wc < p.rope_off + half) {
      fi = wc - p.rope_off;
      if (p.rope_style == KAM_ROPE_HALF) { ca = p.rope_off + fi; cb = ca + half; }
      else { ca = p.rope_off + 2 * fi; cb = ca + 1; }
    } else ca = wc + half;
    const size_t ubase = static_cast<size_t>(t) * desc.u_token_stride + static_cast<size_t>(h) * desc.u_head_stride;
    auto patch = [&](const void* const* U, const void* const* W, int c) -> float {
      if (!m || !U || !W) return 0.f;
      float acc = 0.f;
      const void* Ul = U[l]; const void* Wl = W[l];
      for (int j = 0; j < m; ++j)
        acc = fmaf(ld_as_float<FT>(Ul, ubase + j), ld_as_float<FT>(Wl, (static_cast<size_t>(h) * m + j) * p.D + c), acc);
      return acc;
    };
    float a = ld_as_float<ET>(ksrc, src_row + ca);
    if (cb < 0) {
      st_from_float<ET>(pk, dst_row + ca, a + patch(desc.Uk, desc.Wk, ca));
    } else {
      float b = ld_as_float<ET>(ksrc, src_row + cb);
      const float2 t2 = cs[fi];
      const float pa = patch(desc.Uk, desc.Wk, ca), pb = patch(desc.Uk, desc.Wk, cb);
      if (canonical) { a += pa; b += pb; }
      float ra = fmaf(a, t2.x, -b * t2.y), rb = fmaf(a, t2.y, b * t2.x);
      if (!canonical) { ra += pa; rb += pb; }
      st_from_float<ET>(pk, dst_row + ca, ra);
      st_from_float<ET>(pk, dst_row + cb, rb);
    }
    if (p.has_v && !inplace) {                          // V: copy + patch, every column of the work item
      const void* vsrc = desc.v_src[l];
      st_from_float<ET>(pv, dst_row + ca, ld_as_float<ET>(vsrc, src_row + ca) + patch(desc.Uv, desc.Wv, ca));
      if (cb >= 0) st_from_float<ET>(pv, dst_row + cb, ld_as_float<ET>(vsrc, src_row + cb) + patch(desc.Uv, desc.Wv, cb));
    }
  }
}

void launch_relocate_generic(const GenericParams& p, int max_tokens, cudaStream_t st) {
  dim3 grid(p.n_descs * p.L, (max_tokens + 7) / 8);
  if (grid.y == 0) return;
  if (p.elem_f32 && p.factor_f32) kam_relocate_patch_generic_kernel<float, float><<<grid, 256, 0, st>>>(p);
  else if (p.elem_f32) kam_relocate_patch_generic_kernel<float, __nv_bfloat16><<<grid, 256, 0, st>>>(p);
  else if (p.factor_f32) kam_relocate_patch_generic_kernel<__nv_bfloat16, float><<<grid, 256, 0, st>>>(p);
  else kam_relocate_patch_generic_kernel<__nv_bfloat16, __nv_bfloat16><<<grid, 256, 0, st>>>(p);
}

}  // namespace kam

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

// Incremental (division-free) walk over the flat tile list: chunk d -> layer l -> head group hg -> token tile tt.
struct TileWalk {
  int d, l, hg, tt, n_tt, n_tokens;
  long long d_end;                       // first tile index of the next chunk
  __device__ __forceinline__ void init(const RelocGeom& g, const RelocParams& p, long long tile) {
    int lo = 0, hi = p.n_descs;          // largest d with prefix[d] <= tile
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (p.tile_prefix[mid] <= tile) lo = mid; else hi = mid; }
    d = lo;
    while (p.tile_prefix[d + 1] <= tile) ++d;          // skip empty chunks
    n_tokens = p.descs[d].n_tokens;
    n_tt = (n_tokens + g.TT - 1) / g.TT;
    d_end = p.tile_prefix[d + 1];
    const int local = static_cast<int>(tile - p.tile_prefix[d]);
    tt = local % n_tt;
    const int uu = local / n_tt;
    hg = uu % g.n_hg;
    l = uu / g.n_hg;
  }
  __device__ __forceinline__ void next(const RelocGeom& g, const RelocParams& p, long long new_tile) {
    if (++tt < n_tt) return;
    tt = 0;
    if (++hg < g.n_hg) return;
    hg = 0;
    if (++l < g.L) return;
    l = 0;
    do { ++d; } while (p.tile_prefix[d + 1] <= new_tile);
    n_tokens = p.descs[d].n_tokens;
    n_tt = (n_tokens + g.TT - 1) / g.TT;
    d_end = p.tile_prefix[d + 1];
  }
};

// Rotate 8 column pairs.  HALF: element e of `a` pairs with element e of `b` (columns i and i + d_r/2).
__device__ __forceinline__ void rotate_half8(float* a, float* b, const float2* cs) {
#pragma unroll
  for (int e = 0; e < 8; e += 2) {
    const float4 t = *reinterpret_cast<const float4*>(cs + e);   // (c0, s0, c1, s1)
    float x = a[e], y = b[e];
    a[e] = fmaf(x, t.x, -y * t.y);
    b[e] = fmaf(x, t.y, y * t.x);
    x = a[e + 1]; y = b[e + 1];
    a[e + 1] = fmaf(x, t.z, -y * t.w);
    b[e + 1] = fmaf(x, t.w, y * t.z);
  }
}
// INTERLEAVED: columns (2i, 2i+1) are adjacent inside one 8-vector.
__device__ __forceinline__ void rotate_inter8(float* a, const float2* cs) {
#pragma unroll
  for (int e = 0; e < 8; e += 4) {
    const float4 t = *reinterpret_cast<const float4*>(cs + e / 2);
    float x = a[e], y = a[e + 1];
    a[e] = fmaf(x, t.x, -y * t.y);
    a[e + 1] = fmaf(x, t.y, y * t.x);
    x = a[e + 2]; y = a[e + 3];
    a[e + 2] = fmaf(x, t.z, -y * t.w);
    a[e + 3] = fmaf(x, t.w, y * t.z);
  }
}

// One 32-column group: 4 n-tiles of m16n8k16.  w01 / w23 = B fragments (b0, b1) of n-tiles (0,1) / (2,3).
__device__ __forceinline__ void mma_group(float* r0, float* r1, const uint32_t* a, const uint32_t* w01, const uint32_t* w23) {
  mma_bf16_16816(r0[0], r0[1], r1[0], r1[1], a[0], a[1], a[2], a[3], w01[0], w01[1]);
  mma_bf16_16816(r0[2], r0[3], r1[2], r1[3], a[0], a[1], a[2], a[3], w01[2], w01[3]);
  mma_bf16_16816(r0[4], r0[5], r1[4], r1[5], a[0], a[1], a[2], a[3], w23[0], w23[1]);
  mma_bf16_16816(r0[6], r0[7], r1[6], r1[7], a[0], a[1], a[2], a[3], w23[2], w23[3]);
}

}  // namespace

// Shared-memory map (dynamic): [0,128) mbarriers | slab table | column-block table | cs | W (column-permuted, padded
// rows) | stages.  W in shared memory is [kv][head-in-group][k][D + 8] bf16 with the columns of every 32-group stored
// in MMA order (position 8j + 2i + e holds column 8i + 2j + e), so that ldmatrix.trans yields B fragments whose
// accumulator columns are 8 CONTIGUOUS columns per thread.
__global__ void __launch_bounds__(kRelocThreads, 1)
kam_relocate_patch_kernel(const __grid_constant__ RelocGeom g, const __grid_constant__ RelocParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + g.n_stages;
  uint32_t* slab_tab = reinterpret_cast<uint32_t*>(smem + g.off_tab);
  int4* blk_tab = reinterpret_cast<int4*>(smem + g.off_tab + 256);
  float2* cs = reinterpret_cast<float2*>(smem + g.off_cs);
  uint8_t* wsm = smem + g.off_w;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < g.n_stages; ++s) { mbar_init(&full_bar[s], kRelocProducerWarps); mbar_init(&empty_bar[s], kRelocConsumerWarps); }
    mbar_fence_init();
  }
  if (threadIdx.x < 2 * g.RB * g.n_blocks && threadIdx.x < 64) {     // slab s -> (kv, row block, column block); K slabs first
    const int s = threadIdx.x, per = g.RB * g.n_blocks;
    const int kv = s / per, rem = s - kv * per;
    slab_tab[s] = kv | ((rem / g.n_blocks) << 8) | ((rem % g.n_blocks) << 16);
  }
  if (threadIdx.x >= 64 && threadIdx.x < 64 + g.n_blocks) {
    const ColBlock cb = g.blk[threadIdx.x - 64];
    blk_tab[threadIdx.x - 64] = make_int4(cb.col_off, cb.w_col_off | (cb.band_col0 << 16), cb.n_groups | (cb.fhead << 8) | (cb.rope << 16), 0);
  }
  __syncthreads();

  const long long t_begin = p.total_tiles * blockIdx.x / gridDim.x;
  const long long t_end = p.total_tiles * (blockIdx.x + 1) / gridDim.x;
  if (t_begin >= t_end) return;
  TileWalk w;
  w.init(g, p, t_begin);

  if (warp >= kRelocConsumerWarps) {
    // ================================================================ producer warps: K | V | U_k | U_v
    const int role = warp - kRelocConsumerWarps;
    int stage = 0; uint32_t phase = 0;
    int cur_d = -1, cur_l = -1;
    // per (chunk, layer) state
    const char* src = nullptr; const int32_t* bt = nullptr;
    long long u_tok_stride = 0, u_head_stride = 0;
    int dst0 = 0, m = 0, flags = 0;
    for (long long tile = t_begin; tile < t_end; ++tile) {
      if (w.d != cur_d || w.l != cur_l) {
        cur_d = w.d; cur_l = w.l;
        const RelocDescDev& desc = p.descs[w.d];
        flags = desc.flags; m = desc.rank_l[w.l]; bt = desc.block_table; dst0 = static_cast<int>(desc.dst_token_start);
        u_tok_stride = desc.u_token_stride; u_head_stride = desc.u_head_stride;
        const bool inplace = flags & FLAG_INPLACE;
        const void* const* tab = role == 0 ? desc.k_src : role == 1 ? desc.v_src : role == 2 ? desc.Uk : desc.Uv;
        src = nullptr;
        if (role == 0) src = inplace ? static_cast<const char*>(p.pool_k[w.l]) : static_cast<const char*>(tab[w.l]);
        else if (role == 1) { if (!inplace && g.nkv == 2) src = static_cast<const char*>(tab[w.l]); }
        else if (m && tab && !inplace && (role == 2 || g.nkv == 2)) src = static_cast<const char*>(tab[w.l]);
      }
      mbar_wait(&empty_bar[stage], phase ^ 1);
      uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
      const int tok0 = w.tt * g.TT;
      const int nvalid = min(g.TT, w.n_tokens - tok0);
      const bool inplace = flags & FLAG_INPLACE;
      if (role == 0) {
        // A1 slot mapping: g = dst_token_start + t -> page = block_table[g / P], slot = page * P + g % P
        int32_t* slots = reinterpret_cast<int32_t*>(st + g.st_slot);
        for (int r = lane; r < g.TT; r += 32) {
          int slot = -1;
          if (r < nvalid) {
            const int gt = dst0 + tok0 + r;
            const int pg = g.P_shift >= 0 ? (gt >> g.P_shift) : gt / g.P;
            slot = bt[pg] * g.P + (gt - pg * g.P);
          }
          slots[r] = slot;
        }
        __syncwarp();
        if (lane == 0) {
          const uint32_t bytes = static_cast<uint32_t>(nvalid) * g.slice_bytes;
          mbar_arrive_expect_tx(&full_bar[stage], bytes);
          const size_t off = static_cast<size_t>(w.hg) * g.slice_bytes;
          uint8_t* dst = st + g.st_k;
          if (!inplace) {
            const char* s0 = src + static_cast<size_t>(tok0) * g.row_bytes + off;
            if (g.contig) bulk_g2s(dst, s0, bytes, &full_bar[stage]);
            else for (int r = 0; r < nvalid; ++r) bulk_g2s(dst + r * g.s_row, s0 + static_cast<size_t>(r) * g.row_bytes, g.slice_bytes, &full_bar[stage]);
          } else if (g.contig) {                     // pool rows: contiguous inside a page -> one copy per run of slots
            int r = 0;
            while (r < nvalid) {
              const int s_first = slots[r];
              int n = 1;
              while (r + n < nvalid && slots[r + n] == s_first + n) ++n;
              bulk_g2s(dst + r * g.s_row, src + static_cast<size_t>(s_first) * g.row_bytes, n * g.slice_bytes, &full_bar[stage]);
              r += n;
            }
          } else {
            for (int r = 0; r < nvalid; ++r)
              bulk_g2s(dst + r * g.s_row, src + static_cast<size_t>(slots[r]) * g.row_bytes + off, g.slice_bytes, &full_bar[stage]);
          }
        }
      } else if (lane == 0) {
        if (src == nullptr) {
          mbar_arrive(&full_bar[stage]);
        } else if (role == 1) {
          const uint32_t bytes = static_cast<uint32_t>(nvalid) * g.slice_bytes;
          mbar_arrive_expect_tx(&full_bar[stage], bytes);
          const char* s0 = src + static_cast<size_t>(tok0) * g.row_bytes + static_cast<size_t>(w.hg) * g.slice_bytes;
          uint8_t* dst = st + g.st_v;
          if (g.contig) bulk_g2s(dst, s0, bytes, &full_bar[stage]);
          else for (int r = 0; r < nvalid; ++r) bulk_g2s(dst + r * g.s_row, s0 + static_cast<size_t>(r) * g.row_bytes, g.slice_bytes, &full_bar[stage]);
        } else {
          // U rows of this tile: one run of (heads-in-slice * m) elements per token when the heads are adjacent
          const int hf_n = (u_head_stride == 0) ? 1 : g.HG;
          const uint32_t u_run = static_cast<uint32_t>(m) * 2u, u_tok_bytes = u_run * hf_n;
          mbar_arrive_expect_tx(&full_bar[stage], static_cast<uint32_t>(nvalid) * u_tok_bytes);
          const long long h0 = (u_head_stride == 0) ? 0 : static_cast<long long>(w.hg) * g.HG;
          const char* s0 = src + (static_cast<long long>(tok0) * u_tok_stride + h0 * u_head_stride) * 2;
          uint8_t* dst = st + (role == 2 ? g.st_uk : g.st_uv);
          if (hf_n == 1 || u_head_stride == m) {
            for (int r = 0; r < nvalid; ++r) bulk_g2s(dst + r * g.su_row, s0 + r * u_tok_stride * 2, u_tok_bytes, &full_bar[stage]);
          } else {
            for (int r = 0; r < nvalid; ++r)
              for (int h = 0; h < hf_n; ++h)
                bulk_g2s(dst + r * g.su_row + h * u_run, s0 + (r * u_tok_stride + h * u_head_stride) * 2, u_run, &full_bar[stage]);
          }
        }
      }
      if (++stage == g.n_stages) { stage = 0; phase ^= 1; }
      if (tile + 1 < t_end) w.next(g, p, tile + 1);
    }
    return;
  }

  // ================================================================ consumer warps
  const int gq = lane >> 2, t4 = lane & 3;
  const int ctid = threadIdx.x;                                   // 0 .. 255
  int stage = 0; uint32_t phase = 0;
  int cur_d = -1, cur_l = -1, cur_hg = -1;
  int m = 0, flags = 0; bool u_shared = false, has_uk = false, has_uv = false;
  // ldmatrix lane addressing
  const int a_row = lane & 15, a_koff = (lane >> 4) * 8;                       // A: rows of U, k offset
  const int b_k = (lane & 7) + ((lane >> 3) & 1) * 8, b_nt = lane >> 4;         // B: k row of W, n-tile 0/1 of the pair

  for (long long tile = t_begin; tile < t_end; ++tile) {
    if (w.d != cur_d || w.l != cur_l || w.hg != cur_hg) {
      // ---- new (chunk, layer, head group): rebuild the sin/cos table (new chunk) and stage W
      const bool new_chunk = (w.d != cur_d);
      cur_d = w.d; cur_l = w.l; cur_hg = w.hg;
      const RelocDescDev& desc = p.descs[w.d];
      flags = desc.flags; m = desc.rank_l[w.l];
      u_shared = desc.u_head_stride == 0;
      const bool inplace = flags & FLAG_INPLACE;
      has_uk = m && desc.Uk && !inplace; has_uv = m && desc.Uv && !inplace && g.nkv == 2;
      named_bar_sync(1, kRelocConsumerWarps * 32);                // everyone is done with the old tables
      if (new_chunk && ctid < g.d_r / 2) {
        // A2: f_i = theta^(-2i/d_r); angle = delta * f_i in fp64 (positions reach 1e5: fp32 angles would cost 2 bf16 ulp)
        const double f = pow(g.theta, -2.0 * ctid / g.d_r);
        double s, c;
        sincos(static_cast<double>(desc.delta) * f, &s, &c);
        cs[ctid] = make_float2(static_cast<float>(c), static_cast<float>(s));
      }
      if (has_uk) {
        // W[l] is [H][m][D]; copy this head group's rows, 16 bytes (8 columns = 4 pairs) per thread, scattering the pairs
        // to their MMA-order positions inside the 32-column group.
        const int vec_per_row = g.D >> 3;
        const int per_kv = g.HG * m * vec_per_row;
        const int nkv_w = has_uv ? 2 : 1;
        for (int e = ctid; e < nkv_w * per_kv; e += kRelocConsumerWarps * 32) {
          const int kv = e >= per_kv;
          int r = e - kv * per_kv;
          const int v = r % vec_per_row; r /= vec_per_row;       // r = head-in-group * m + k
          const void* const* Wl = kv ? desc.Wv : desc.Wk;
          const uint4 x = __ldg(reinterpret_cast<const uint4*>(static_cast<const char*>(Wl[w.l]) +
                                (static_cast<size_t>(w.hg) * g.HG * m + r) * g.D * 2) + v);
          const int q = v >> 2, i = v & 3;                         // columns 32q + 8i .. +7 = pairs j = 0..3
          uint32_t* dst = reinterpret_cast<uint32_t*>(wsm + static_cast<size_t>(kv) * g.w_kv_stride + static_cast<size_t>(r) * g.w_row) + q * 16 + i;
          dst[0] = x.x; dst[4] = x.y; dst[8] = x.z; dst[12] = x.w; // pair j lands at 32-bit position 4j + i
        }
      }
      named_bar_sync(1, kRelocConsumerWarps * 32);
    }

    mbar_wait(&full_bar[stage], phase);

    const uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
    const int32_t* slots = reinterpret_cast<const int32_t*>(st + g.st_slot);
    const bool inplace = flags & FLAG_INPLACE;
    const bool canonical = flags & FLAG_CANONICAL_FRAME;
    const int KT = m >> 4;
    const int n_slabs = ((g.nkv == 2 && !inplace) ? 2 : 1) * g.RB * g.n_blocks;

    for (int s = warp; s < n_slabs; s += kRelocConsumerWarps) {
      const uint32_t se = slab_tab[s];
      const int kv = se & 0xff, rb = (se >> 8) & 0xff, b = se >> 16;
      const int4 cbv = blk_tab[b];
      const int col_off = cbv.x, w_col_off = cbv.y & 0xffff, band_col0 = cbv.y >> 16;
      const int n_groups = cbv.z & 0xff, fhead = (cbv.z >> 8) & 0xff;
      const bool rope = (kv == 0) && ((cbv.z >> 16) & 1);
      const int row0 = rb * 16 + gq;
      const int slot0 = slots[row0], slot1 = slots[row0 + 8];
      char* pool = static_cast<char*>(kv ? p.pool_v[w.l] : p.pool_k[w.l]) + static_cast<size_t>(w.hg) * g.slice_bytes + col_off * 2 + t4 * 16;
      char* dst0 = pool + static_cast<size_t>(slot0 < 0 ? 0 : slot0) * g.row_bytes;
      char* dst1 = pool + static_cast<size_t>(slot1 < 0 ? 0 : slot1) * g.row_bytes;
      const uint8_t* rows = st + (kv ? g.st_v : g.st_k) + row0 * g.s_row + col_off * 2 + t4 * 16;
      const bool patched = KT > 0 && (kv ? has_uv : has_uk);

      // A fragments of U for this slab's 16 tokens and head: one ldmatrix.x4 per 16 ranks
      uint32_t afr[4][4];
      if (patched) {
        const int hf = u_shared ? 0 : fhead;
        const uint32_t ua = smem_u32(st + (kv ? g.st_uv : g.st_uk) + (rb * 16 + a_row) * g.su_row + (hf * m + a_koff) * 2);
#pragma unroll
        for (int kt = 0; kt < 4; ++kt)
          if (kt < KT) ldmatrix_x4(afr[kt][0], afr[kt][1], afr[kt][2], afr[kt][3], ua + kt * 32);
      }
      // B fragments come from W rows k of this head: address of (k = b_k, 32-bit position 0 of n-tile b_nt)
      const uint32_t wb = smem_u32(wsm + static_cast<size_t>(kv) * g.w_kv_stride + static_cast<size_t>(fhead * m + b_k) * g.w_row + (w_col_off + b_nt * 8) * 2);

      const bool half_rope = rope && g.rope_style == KAM_ROPE_HALF;
      const int steps = n_groups >> 1;
#pragma unroll 1
      for (int sp = 0; sp < steps; ++sp) {
        const int gA = half_rope ? sp : 2 * sp;
        const int gB = half_rope ? sp + steps : 2 * sp + 1;
        float a0[8], a1[8], b0[8], b1[8];
        unpack8(*reinterpret_cast<const uint4*>(rows + gA * 64), a0);
        unpack8(*reinterpret_cast<const uint4*>(rows + 8 * g.s_row + gA * 64), a1);
        unpack8(*reinterpret_cast<const uint4*>(rows + gB * 64), b0);
        unpack8(*reinterpret_cast<const uint4*>(rows + 8 * g.s_row + gB * 64), b1);

        const float2* csA = cs;
        const float2* csB = cs;
        if (rope) {
          if (half_rope) csA = cs + band_col0 + 32 * gA + 8 * t4;
          else { csA = cs + ((band_col0 + 32 * gA + 8 * t4) >> 1); csB = cs + ((band_col0 + 32 * gB + 8 * t4) >> 1); }
        }
        if (rope && !canonical) {                                  // Eq. 1: rotate, then add the patch
          if (half_rope) { rotate_half8(a0, b0, csA); rotate_half8(a1, b1, csA); }
          else { rotate_inter8(a0, csA); rotate_inter8(a1, csA); rotate_inter8(b0, csB); rotate_inter8(b1, csB); }
        }
        if (patched) {
#pragma unroll
          for (int kt = 0; kt < 4; ++kt) {
            if (kt < KT) {
              uint32_t wA[8], wB[8];
              const uint32_t base = wb + kt * 16 * g.w_row;
              ldmatrix_x4_trans(wA[0], wA[1], wA[2], wA[3], base + gA * 64);
              ldmatrix_x4_trans(wA[4], wA[5], wA[6], wA[7], base + gA * 64 + 32);
              ldmatrix_x4_trans(wB[0], wB[1], wB[2], wB[3], base + gB * 64);
              ldmatrix_x4_trans(wB[4], wB[5], wB[6], wB[7], base + gB * 64 + 32);
              mma_group(a0, a1, afr[kt], wA, wA + 4);
              mma_group(b0, b1, afr[kt], wB, wB + 4);
            }
          }
        }
        if (rope && canonical) {                                   // patch stored in the chunk's own frame (R-4)
          if (half_rope) { rotate_half8(a0, b0, csA); rotate_half8(a1, b1, csA); }
          else { rotate_inter8(a0, csA); rotate_inter8(a1, csA); rotate_inter8(b0, csB); rotate_inter8(b1, csB); }
        }
        if (slot0 >= 0) { st_global_v4(dst0 + gA * 64, pack8(a0)); st_global_v4(dst0 + gB * 64, pack8(b0)); }
        if (slot1 >= 0) { st_global_v4(dst1 + gA * 64, pack8(a1)); st_global_v4(dst1 + gB * 64, pack8(b1)); }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[stage]);
    if (++stage == g.n_stages) { stage = 0; phase ^= 1; }
    if (tile + 1 < t_end) w.next(g, p, tile + 1);
  }
}

void launch_relocate_fast(const RelocGeom& g, const RelocParams& p, int grid, cudaStream_t st) {
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(kam_relocate_patch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    attr_set = true;
  }
  kam_relocate_patch_kernel<<<grid, kRelocThreads, g.smem_bytes, st>>>(g, p);
}

// ---------------------------------------------------------------------------------------------------------------
// Generic element-wise path: any element / factor dtype, any rank <= KAM_MAX_RANK, any even rope band.  One thread
// owns a non-rotated column or BOTH columns of a rope pair (in-place safe).  Correctness path for small or odd
// shapes (config 1's fp32 tensors and rank 4); the tiled kernel above is the one the roofline is quoted on.
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
    const size_t slot = static_cast<size_t>(desc.block_table[pg]) * p.P + static_cast<size_t>(gt - pg * p.P);
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

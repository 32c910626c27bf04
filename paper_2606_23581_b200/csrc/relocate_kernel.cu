// kam_relocate_patch / kam_rotate_inplace: Eq. 1 of the paper written into the paged pool.
//
// One persistent launch covers layers x chunks x token tiles.  The step is HBM-bound: every
// element of the chunk's K/V is read once and written once, plus the factors.  Design for sm_100a:
//   * a producer warp streams 16*RB-token tiles of the canonical rows and the U factors into shared memory with
//     1-D bulk async copies (cp.async.bulk, the TMA engine) behind an mbarrier ring: deep memory-level
//     parallelism without spending registers, one copy per token slice, padded rows => no bank conflicts;
//   * 8 consumer warps take (16 tokens x <=128 columns) slabs: unpack bf16, rotate the rope band with the
//     chunk's (cos, sin) table (one fp64 sincos per (chunk, frequency), reused over tokens, heads, layers),
//     add the rank-m patch as m16n8k16 bf16 tensor-core MMAs whose accumulators START as the rotated rows
//     (so the add is free and accumulation is fp32), round to bf16 (RNE) and store 128-bit vectors straight to
//     the pool page the block table names;
//   * W (the paper's V_m^T) is re-laid out once per (chunk, layer, head group) into MMA-fragment order in shared
//     memory; the column<->fragment permutation is chosen so that each thread owns 8 contiguous columns
//     (128-bit loads/stores) AND both members of every rope pair (so in-place rotation is race-free).
// Why not FP32 FMAs for the patch: at m=16 the patch needs 51 TFLOP/s at the HBM roofline and at m=32 95 TFLOP/s,
// against a 74 TFLOP/s FFMA peak; on the tensor pipe it is <10 % of the legacy-MMA rate.
#include <cuda_runtime.h>

#include "common.cuh"
#include "internal.h"

namespace kam {

namespace {

struct UnitState {          // what is constant over the tiles of one (chunk, layer)
  const char* k_src; const char* v_src;
  const char* uk; const char* uv;
  const int32_t* bt;
  long long dst0, u_tok_stride, u_head_stride;
  int n_tokens, n_tt, m, flags;
};

__device__ __forceinline__ void load_unit(UnitState& u, const RelocDescDev& d, int l, int TT) {
  u.flags = d.flags;
  u.n_tokens = d.n_tokens;
  u.n_tt = (d.n_tokens + TT - 1) / TT;
  u.m = d.rank_l[l];
  u.bt = d.block_table;
  u.dst0 = d.dst_token_start;
  u.u_tok_stride = d.u_token_stride;
  u.u_head_stride = d.u_head_stride;
  const bool inplace = d.flags & FLAG_INPLACE;
  u.k_src = inplace ? nullptr : static_cast<const char*>(d.k_src[l]);
  u.v_src = (inplace || d.v_src == nullptr) ? nullptr : static_cast<const char*>(d.v_src[l]);
  u.uk = (u.m && d.Uk) ? static_cast<const char*>(d.Uk[l]) : nullptr;
  u.uv = (u.m && d.Uv) ? static_cast<const char*>(d.Uv[l]) : nullptr;
}

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

__device__ __forceinline__ void mma_group(float* r0, float* r1, const uint32_t* a, const uint4& w0, const uint4& w1) {
  mma_bf16_16816(r0[0], r0[1], r1[0], r1[1], a[0], a[1], a[2], a[3], w0.x, w0.y);
  mma_bf16_16816(r0[2], r0[3], r1[2], r1[3], a[0], a[1], a[2], a[3], w0.z, w0.w);
  mma_bf16_16816(r0[4], r0[5], r1[4], r1[5], a[0], a[1], a[2], a[3], w1.x, w1.y);
  mma_bf16_16816(r0[6], r0[7], r1[6], r1[7], a[0], a[1], a[2], a[3], w1.z, w1.w);
}

}  // namespace

__global__ void __launch_bounds__(kRelocThreads, 1)
kam_relocate_patch_kernel(const __grid_constant__ RelocGeom g, const __grid_constant__ RelocParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty_bar = full_bar + g.n_stages;
  float2* cs = reinterpret_cast<float2*>(smem + g.off_cs);
  uint8_t* wfrag = smem + g.off_w;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < g.n_stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], kRelocConsumerWarps); }
    mbar_fence_init();
  }
  __syncthreads();

  const long long t_begin = p.total_tiles * blockIdx.x / gridDim.x;
  const long long t_end = p.total_tiles * (blockIdx.x + 1) / gridDim.x;
  if (t_begin >= t_end) return;

  // first chunk of this CTA's tile range
  int d = 0;
  {
    int lo = 0, hi = p.n_descs;                    // largest d with prefix[d] <= t_begin
    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (p.tile_prefix[mid] <= t_begin) lo = mid; else hi = mid; }
    d = lo;
  }
  long long d_first = p.tile_prefix[d], d_next = p.tile_prefix[d + 1];
  int cur_d = -1, cur_l = -1, cur_hg = -1;
  UnitState u;
  const int tiles_per_layer_div = g.n_hg;

  if (warp == kRelocConsumerWarps) {
    // ================================================================ producer warp
    uint32_t it = 0;
    for (long long tile = t_begin; tile < t_end; ++tile, ++it) {
      while (tile >= d_next) { ++d; d_first = d_next; d_next = p.tile_prefix[d + 1]; }
      if (d != cur_d) { cur_d = d; cur_l = -1; }
      const RelocDescDev& desc = p.descs[d];
      const int n_tt = (desc.n_tokens + g.TT - 1) / g.TT;
      const int local = static_cast<int>(tile - d_first);
      const int tt = local % n_tt, uu = local / n_tt;
      const int hg = uu % tiles_per_layer_div, l = uu / tiles_per_layer_div;
      if (l != cur_l) { cur_l = l; load_unit(u, desc, l, g.TT); }

      const int stage = it % g.n_stages;
      const uint32_t phase = (it / g.n_stages) & 1;
      mbar_wait(&empty_bar[stage], phase ^ 1);

      uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
      int32_t* slots = reinterpret_cast<int32_t*>(st + g.st_slot);
      const int tok0 = tt * g.TT;
      const int nvalid = min(g.TT, u.n_tokens - tok0);
      const bool inplace = u.flags & FLAG_INPLACE;
      const char* pk = static_cast<const char*>(p.pool_k[l]);

      // slot mapping: g = dst_token_start + t -> page = block_table[g / P], slot = page*P + g % P
      for (int r = lane; r < g.TT; r += 32) {
        int slot = -1;
        if (r < nvalid) {
          const long long gt = u.dst0 + tok0 + r;
          const long long pg = gt / g.P;
          slot = u.bt[pg] * g.P + static_cast<int>(gt - pg * g.P);
        }
        slots[r] = slot;
      }
      const bool has_v = (g.nkv == 2) && !inplace;
      const int hf_n = (u.u_head_stride == 0) ? 1 : g.HG;              // factor heads in this slice
      const uint32_t u_run = static_cast<uint32_t>(u.m) * 2u;           // bytes of one (token, head) run of U
      const uint32_t u_tok_bytes = u_run * hf_n;
      uint32_t bytes = static_cast<uint32_t>(nvalid) * (g.slice_bytes * (has_v ? 2u : 1u));
      if (u.uk) bytes += nvalid * u_tok_bytes;
      if (u.uv && has_v) bytes += nvalid * u_tok_bytes;
      __syncwarp();
      if (lane == 0) mbar_arrive_expect_tx(&full_bar[stage], bytes);
      __syncwarp();

      const bool u_one_run = (hf_n == 1) || (u.u_head_stride == u.m);
      const long long h0 = (u.u_head_stride == 0) ? 0 : static_cast<long long>(hg) * g.HG;
      for (int r = lane; r < nvalid; r += 32) {
        const long long t = tok0 + r;
        const size_t off = static_cast<size_t>(hg) * g.slice_bytes;
        const char* ksrc = inplace ? pk + static_cast<size_t>(slots[r]) * g.row_bytes + off
                                   : u.k_src + static_cast<size_t>(t) * g.row_bytes + off;
        bulk_g2s(st + g.st_k + r * g.s_row, ksrc, g.slice_bytes, &full_bar[stage]);
        if (has_v)
          bulk_g2s(st + g.st_v + r * g.s_row, u.v_src + static_cast<size_t>(t) * g.row_bytes + off, g.slice_bytes,
                   &full_bar[stage]);
        if (u.uk) {
          const char* src = u.uk + (t * u.u_tok_stride + h0 * u.u_head_stride) * 2;
          uint8_t* dst = st + g.st_uk + r * g.su_row;
          if (u_one_run) bulk_g2s(dst, src, u_tok_bytes, &full_bar[stage]);
          else
            for (int h = 0; h < hf_n; ++h) bulk_g2s(dst + h * u_run, src + h * u.u_head_stride * 2, u_run, &full_bar[stage]);
        }
        if (u.uv && has_v) {
          const char* src = u.uv + (t * u.u_tok_stride + h0 * u.u_head_stride) * 2;
          uint8_t* dst = st + g.st_uv + r * g.su_row;
          if (u_one_run) bulk_g2s(dst, src, u_tok_bytes, &full_bar[stage]);
          else
            for (int h = 0; h < hf_n; ++h) bulk_g2s(dst + h * u_run, src + h * u.u_head_stride * 2, u_run, &full_bar[stage]);
        }
      }
    }
    return;
  }

  // ================================================================ consumer warps
  const int gq = lane >> 2, t4 = lane & 3;
  const int ctid = threadIdx.x;                                   // 0 .. 255
  uint32_t it = 0;
  for (long long tile = t_begin; tile < t_end; ++tile, ++it) {
    while (tile >= d_next) { ++d; d_first = d_next; d_next = p.tile_prefix[d + 1]; }
    const RelocDescDev& desc = p.descs[d];
    const int n_tt = (desc.n_tokens + g.TT - 1) / g.TT;
    const int local = static_cast<int>(tile - d_first);
    const int uu = local / n_tt;
    const int hg = uu % tiles_per_layer_div, l = uu / tiles_per_layer_div;

    if (d != cur_d || l != cur_l || hg != cur_hg) {
      // ---- new (chunk, layer, head group): rebuild the sin/cos table (new chunk) and W's fragment table
      const bool new_chunk = (d != cur_d);
      cur_d = d; cur_l = l; cur_hg = hg;
      load_unit(u, desc, l, g.TT);
      named_bar_sync(1, kRelocConsumerWarps * 32);                // everyone is done with the old tables
      if (new_chunk && ctid < g.d_r / 2) {
        // A2: f_i = theta^(-2i/d_r); angle = delta * f_i in fp64 (positions reach 1e5: fp32 angles would cost 2 bf16 ulp)
        const double f = pow(g.theta, -2.0 * ctid / g.d_r);
        double s, c;
        sincos(static_cast<double>(desc.delta) * f, &s, &c);
        cs[ctid] = make_float2(static_cast<float>(c), static_cast<float>(s));
      }
      if (u.m) {
        const int KT = u.m >> 4;
        const int per_kv = g.n_blocks * KT * 256;                  // (blk, kt, grp(4), half(2), lane(32)) entries
        const int nkv_w = (g.nkv == 2 && !(u.flags & FLAG_INPLACE)) ? 2 : 1;
        for (int e = ctid; e < nkv_w * per_kv; e += kRelocConsumerWarps * 32) {
          const int kv = e / per_kv;
          int r = e - kv * per_kv;
          const int ln = r & 31; r >>= 5;
          const int half = r & 1; r >>= 1;
          const int grp = r & 3; r >>= 2;
          const int kt = r % KT, b = r / KT;
          const ColBlock cb = g.blk[b];
          if (grp >= cb.n_groups) continue;
          const void* const* Wl = kv ? desc.Wv : desc.Wk;
          if (Wl == nullptr) continue;
          const int head = (g.nkv == 1 && g.H == 1) ? 0 : hg * g.HG + cb.fhead;
          const unsigned short* W = static_cast<const unsigned short*>(Wl[l]) + static_cast<size_t>(head) * u.m * g.D;
          const int gg = ln >> 2, tt4 = ln & 3;
          const int k0 = kt * 16 + 2 * tt4;
          uint32_t v[4];
#pragma unroll
          for (int jj = 0; jj < 2; ++jj) {
            const int col = cb.w_col_off + 32 * grp + 8 * (gg >> 1) + 2 * (half * 2 + jj) + (gg & 1);
            const uint32_t w00 = __ldg(W + static_cast<size_t>(k0) * g.D + col);
            const uint32_t w01 = __ldg(W + static_cast<size_t>(k0 + 1) * g.D + col);
            const uint32_t w10 = __ldg(W + static_cast<size_t>(k0 + 8) * g.D + col);
            const uint32_t w11 = __ldg(W + static_cast<size_t>(k0 + 9) * g.D + col);
            v[2 * jj] = w00 | (w01 << 16);
            v[2 * jj + 1] = w10 | (w11 << 16);
          }
          // [kv][blk][kt][grp][half][lane] x 16 B
          uint4* dst = reinterpret_cast<uint4*>(wfrag + static_cast<size_t>(kv) * g.w_kv_stride) +
                       ((((b * KT + kt) * 4 + grp) * 2 + half) * 32 + ln);
          *dst = make_uint4(v[0], v[1], v[2], v[3]);
        }
      }
      named_bar_sync(1, kRelocConsumerWarps * 32);
    }

    const int stage = it % g.n_stages;
    const uint32_t phase = (it / g.n_stages) & 1;
    mbar_wait(&full_bar[stage], phase);

    const uint8_t* st = smem + g.off_stage0 + static_cast<size_t>(stage) * g.stage_bytes;
    const int32_t* slots = reinterpret_cast<const int32_t*>(st + g.st_slot);
    const bool inplace = u.flags & FLAG_INPLACE;
    const bool canonical = u.flags & FLAG_CANONICAL_FRAME;
    const int nkv_eff = (g.nkv == 2 && !inplace) ? 2 : 1;
    const int KT = u.m >> 4;
    const int n_slabs = nkv_eff * g.RB * g.n_blocks;
    const bool u_shared = (u.u_head_stride == 0);

    for (int s = warp; s < n_slabs; s += kRelocConsumerWarps) {
      const int kv = s / (g.RB * g.n_blocks);
      const int rem = s - kv * (g.RB * g.n_blocks);
      const int rb = rem / g.n_blocks, b = rem - rb * g.n_blocks;
      const ColBlock cb = g.blk[b];
      const int row0 = rb * 16 + gq;
      const int slot0 = slots[row0], slot1 = slots[row0 + 8];
      char* pool = static_cast<char*>(kv ? p.pool_v[l] : p.pool_k[l]);
      char* dst0 = slot0 >= 0 ? pool + static_cast<size_t>(slot0) * g.row_bytes + static_cast<size_t>(hg) * g.slice_bytes : nullptr;
      char* dst1 = slot1 >= 0 ? pool + static_cast<size_t>(slot1) * g.row_bytes + static_cast<size_t>(hg) * g.slice_bytes : nullptr;
      const uint8_t* rows = st + (kv ? g.st_v : g.st_k);
      const uint8_t* urows = st + (kv ? g.st_uv : g.st_uk);
      const bool patched = KT > 0 && ((kv ? u.uv : u.uk) != nullptr);
      const bool rope = (kv == 0) && cb.rope;

      // A fragments of U for this slab's 16 tokens and head
      uint32_t afr[4][4];
      if (patched) {
        const int hf = u_shared ? 0 : cb.fhead;
        const uint8_t* ua = urows + row0 * g.su_row + (hf * u.m + 2 * t4) * 2;
#pragma unroll
        for (int kt = 0; kt < 4; ++kt) {
          if (kt < KT) {
            afr[kt][0] = *reinterpret_cast<const uint32_t*>(ua + kt * 32);
            afr[kt][1] = *reinterpret_cast<const uint32_t*>(ua + 8 * g.su_row + kt * 32);
            afr[kt][2] = *reinterpret_cast<const uint32_t*>(ua + kt * 32 + 16);
            afr[kt][3] = *reinterpret_cast<const uint32_t*>(ua + 8 * g.su_row + kt * 32 + 16);
          }
        }
      }
      const uint4* wf = reinterpret_cast<const uint4*>(wfrag + static_cast<size_t>(kv) * g.w_kv_stride) + (b * KT) * 256 + lane;

      const bool half_rope = rope && g.rope_style == KAM_ROPE_HALF;
      const int steps = cb.n_groups >> 1;
#pragma unroll 1
      for (int sp = 0; sp < steps; ++sp) {
        const int gA = half_rope ? sp : 2 * sp;
        const int gB = half_rope ? sp + steps : 2 * sp + 1;
        const int cA = cb.col_off + 32 * gA + 8 * t4, cB = cb.col_off + 32 * gB + 8 * t4;   // slice-relative columns
        float a0[8], a1[8], b0[8], b1[8];
        unpack8(*reinterpret_cast<const uint4*>(rows + row0 * g.s_row + cA * 2), a0);
        unpack8(*reinterpret_cast<const uint4*>(rows + (row0 + 8) * g.s_row + cA * 2), a1);
        unpack8(*reinterpret_cast<const uint4*>(rows + row0 * g.s_row + cB * 2), b0);
        unpack8(*reinterpret_cast<const uint4*>(rows + (row0 + 8) * g.s_row + cB * 2), b1);

        const float2* csA = cs;
        const float2* csB = cs;
        if (rope) {
          if (half_rope) csA = cs + cb.band_col0 + 32 * gA + 8 * t4;
          else { csA = cs + ((cb.band_col0 + 32 * gA + 8 * t4) >> 1); csB = cs + ((cb.band_col0 + 32 * gB + 8 * t4) >> 1); }
        }
        if (rope && !canonical) {                                  // Eq. 1: rotate, then add the patch
          if (half_rope) { rotate_half8(a0, b0, csA); rotate_half8(a1, b1, csA); }
          else { rotate_inter8(a0, csA); rotate_inter8(a1, csA); rotate_inter8(b0, csB); rotate_inter8(b1, csB); }
        }
        if (patched) {
#pragma unroll
          for (int kt = 0; kt < 4; ++kt) {
            if (kt < KT) {
              const uint4* wA = wf + (kt * 4 + gA) * 64;
              const uint4* wB = wf + (kt * 4 + gB) * 64;
              mma_group(a0, a1, afr[kt], wA[0], wA[32]);
              mma_group(b0, b1, afr[kt], wB[0], wB[32]);
            }
          }
        }
        if (rope && canonical) {                                   // patch stored in the chunk's own frame (R-4)
          if (half_rope) { rotate_half8(a0, b0, csA); rotate_half8(a1, b1, csA); }
          else { rotate_inter8(a0, csA); rotate_inter8(a1, csA); rotate_inter8(b0, csB); rotate_inter8(b1, csB); }
        }
        if (dst0) { st_global_v4(dst0 + cA * 2, pack8(a0)); st_global_v4(dst0 + cB * 2, pack8(b0)); }
        if (dst1) { st_global_v4(dst1 + cA * 2, pack8(a1)); st_global_v4(dst1 + cB * 2, pack8(b1)); }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[stage]);
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

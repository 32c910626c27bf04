// kam_mla_tc_decode_kernel: the absorbed MLA decode (decode_mla_kernel.cu) on the 5th-generation tensor cores.
//
// Why tcgen05 here and nowhere else in this library: north_star reserves it for decode tiles "only if ncu shows them to be the
// limiter".  For GQA/MHA the mma.sync kernel is HBM-bound; for MLA (30 flop per byte, one 1152-byte row is key AND value) the
// mma.sync formulation is bound by its own instruction chain at 61 % of the HBM roofline (profiles/ncu_extras_r01.md).  With
// the TOKENS as the M = 128 dimension one tile costs 36 + 32 tcgen05.mma of 8 cycles against a 6640-cycle HBM budget.
//
//   S^T[tokens][16 heads]     = K[tile x 576] q~^T          A = the tile (K-major, 128-byte swizzle, straight from TMA), B = q~ in smem
//   O^T[512][16 heads]       += V^T[512 x 128] P^T        A = the SAME tile read MN-major (no second copy), B = P^T written by softmax
// S and O live in tensor memory (16 + 4 x 16 columns).  CTA = 4 softmax warps (thread = token row: tcgen05.ld, exp2, P^T to
// smem, lazy O rescale, epilogue), 1 TMA producer warp, 1 MMA-issuing warp.  One CTA per SM, persistent over the plan's
// segments.  A tile is 64 tokens (2.6 tiles fit the rings, so the loads run ahead of the softmax; the M = 128 score MMA simply
// has 64 don't-care rows).  It arrives as 16-token TMA boxes (a box never straddles a page) into two rings: 10 slots of a PAIR
// of 64-column blocks (2 x 8 KB: one M = 128 block of V^T) and 3 slots of the rope block (8 KB).  A pair is released by the
// tcgen05.commit of the PV block that read it.
//
// Not covered here (the mma.sync kernel takes those calls): the on-read patch.
//
// STATUS (round 1): parity-green (tests/test_gpu_decode_mla.py::test_tcgen05_kernel_matches_the_oracle) but OPT-IN
// (KAM_MLA_TC=1), because it is slower than the mma.sync kernel on the 16-head shape: 2.5 TB/s against 3.9 TB/s.
// What was measured (ncu, profiles/): the tcgen05 pipe is 43-45 % active at 35 % DRAM; 52 instructions per 64-token tile take
// ~3300 cycles = ~64 cycles per tcgen05.mma whatever was tried - M = 128 or M = 64 for the scores, 8 independent partial
// accumulators instead of one dependent chain, the PV blocks interleaved, QK^T of tile t + 1 issued ahead of PV of tile t,
// 5 page-sized TMA copies per tile instead of 36.  64 cycles is the cost of an M x 128 x 16 instruction (M N / 256 with N = 128):
// an instruction with N = 16 is charged like N = 128, so 7/8 of the tensor pipe is idle by construction, and the instruction
// count alone (52 x 64 = 3328 cycles) equals the 3320-cycle HBM budget of a 64-token tile.  The formulation pays off from
// N >= 64 query heads per work unit (DeepSeek-V2/V3: 128 heads); for 16 heads the tokens must be the N dimension (padded heads
// as M = 64, O^T [64 x 512] packed into 256 tensor-memory columns, softmax rows = heads) - the next round's kernel.
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "decode_common.cuh"
#include "internal.h"

namespace kam {

namespace {
constexpr int kTcTok = 64;                          // tokens per tile (the score MMA is M = 128: its upper 64 rows are don't-care)
constexpr int kTcGroups = kTcTok / kDecTile;        // 16-token TMA boxes per column block
constexpr int kTcPairSlots = 10, kTcRopeSlots = 3, kTcHdrs = 8;
constexpr int kBlkBytes = kTcTok * 128;             // one 64-column block of a tile: 64 rows x 128 B
constexpr int kPairBytes = 2 * kBlkBytes;
// shared-memory map (bytes)
constexpr int kOffBar = 0;                          // mbarriers
constexpr int kOffTmem = 512;                       // tensor-memory base address from tcgen05.alloc
constexpr int kOffHdr = 1024;                       // int4[kTcHdrs]
constexpr int kOffRed = 1280;                       // float[4][16] cross-warp reductions
constexpr int kOffQhi = 2048;                       // q~ hi: 9 blocks x [16 heads][128 B]
constexpr int kOffQlo = kOffQhi + 9 * 2048;         // q~ lo of the rope block
constexpr int kOffP = kOffQlo + 2048;               // P^T: [16 heads][64 tokens = 128 B] (+ 2 KB spare)
constexpr int kOffRope = kOffP + 4096;              // 26624 = 26 x 1024
constexpr int kOffPair = kOffRope + kTcRopeSlots * kBlkBytes;
// + one block of padding: the M = 128 score MMA reads 128 rows from a 64-row block (the extra rows only feed S rows nobody uses)
constexpr int kTcSmem = kOffPair + kTcPairSlots * kPairBytes + kBlkBytes;     // 223232 bytes
static_assert(kOffRope % 1024 == 0 && kTcSmem <= 227 * 1024, "shared-memory map");
enum : int { BAR_FULL_PAIR = 0, BAR_EMPTY_PAIR = 10, BAR_FULL_ROPE = 20, BAR_EMPTY_ROPE = 23, BAR_S_FULL = 26 /* x2 */, BAR_P_FULL = 28,
             BAR_O_DONE = 29, BAR_Q_FULL = 30, BAR_SEG = 31, BAR_COUNT = 32 };
// Tensor-memory columns.  O block b: [16 b, 16 b + 16).  S of tile parity u: kSParts partial sums at [64 + 128 u + 16 p, +16): back-to-back
// MMAs into ONE accumulator serialise on its ~64-cycle pipeline latency (measured: 64 cycles per N = 16 instruction whatever M),
// so consecutive k-steps go to different partial accumulators and the softmax warps add them.
constexpr uint32_t kTmemCols = 512;
constexpr int kSParts = 8;
constexpr uint32_t kTmemS = 64;

// ---- tcgen05 wrappers (PTX as documented in the Blackwell guide / CUTLASS cute/arch/mma_sm100_umma.hpp)
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {     // arrives on bar when all MMAs issued so far by this thread are done
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// shared-memory matrix descriptor, 128-byte swizzle (layout type 2), version 1; offsets in bytes
__device__ __forceinline__ uint64_t tc_desc(uint32_t smem_addr, uint32_t lbo, uint32_t sbo) {
  return static_cast<uint64_t>((smem_addr & 0x3ffff) >> 4) | (static_cast<uint64_t>(lbo >> 4) << 16) |
         (static_cast<uint64_t>(sbo >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: D = f32, A = B = bf16, N = 16, M = m; a_mn: A is MN-major (the V^T read of the tile)
__device__ __forceinline__ constexpr uint32_t tc_idesc(bool a_mn, uint32_t m) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((a_mn ? 1u : 0u) << 15) | ((16u >> 3) << 17) | ((m >> 4) << 24);
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {          // this thread's lane, 16 consecutive columns
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float* v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
               ::"r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])),
                 "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])),
                 "r"(__float_as_uint(v[7])), "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])),
                 "r"(__float_as_uint(v[11])), "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])),
                 "r"(__float_as_uint(v[15]))
               : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// 2-D-in-3-D TMA load of one (64 columns x 16 tokens) box of column block cb
__device__ __forceinline__ bool bar_or_128(int id, bool pred) {                  // OR of pred over the 128 softmax threads
  uint32_t out;
  asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.b32 q, %2, 0;\n\tbarrier.cta.red.or.pred p, %1, 128, q;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(out) : "r"(id), "r"(static_cast<uint32_t>(pred)) : "memory");
  return out != 0;
}
// byte offset of element (row r of 16, column c of 64) inside a [16 rows][128 B] swizzled K-major operand block pair of atoms
__device__ __forceinline__ uint32_t sw_off(int r, int c) {
  return static_cast<uint32_t>((r >> 3) * 1024 + (r & 7) * 128 + ((((c >> 3) ^ (r & 7)) & 7) << 4) + (c & 7) * 2);
}
}  // namespace

__global__ void __launch_bounds__(192, 1)
kam_mla_tc_decode_kernel(const __grid_constant__ DecodeGeom g, const __grid_constant__ DecodeParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kOffBar);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + kOffTmem);
  int4* hdrs = reinterpret_cast<int4*>(smem + kOffHdr);
  float* red = reinterpret_cast<float*>(smem + kOffRed);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  const int seg_begin = p.plan.cta_seg[blockIdx.x], seg_end = p.plan.cta_seg[blockIdx.x + 1];
  if (seg_begin >= seg_end) return;                               // before any allocation: nothing to undo

  if (threadIdx.x == 0) {
    for (int i = 0; i < kTcPairSlots; ++i) { mbar_init(&bars[BAR_FULL_PAIR + i], 1); mbar_init(&bars[BAR_EMPTY_PAIR + i], 1); }
    for (int i = 0; i < kTcRopeSlots; ++i) { mbar_init(&bars[BAR_FULL_ROPE + i], 1); mbar_init(&bars[BAR_EMPTY_ROPE + i], 1); }
    mbar_init(&bars[BAR_S_FULL], 1); mbar_init(&bars[BAR_S_FULL + 1], 1); mbar_init(&bars[BAR_P_FULL], 128); mbar_init(&bars[BAR_O_DONE], 1);
    mbar_init(&bars[BAR_Q_FULL], 128); mbar_init(&bars[BAR_SEG], 1);
    mbar_fence_init();
  }
  // the rings start as zeros: rows a tile never loads (beyond the end of a segment) are read by the PV MMA with P = 0
  for (int i = threadIdx.x; i < (kTcSmem - kOffRope) / 16; i += blockDim.x) reinterpret_cast<uint4*>(smem + kOffRope)[i] = make_uint4(0, 0, 0, 0);
  fence_proxy_async();
  if (warp == 5) {                                                // one warp allocates the tensor memory and owns the deallocation
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(const_cast<uint32_t*>(tmem_slot))), "n"(kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  grid_dep_launch();

  if (warp == 4) {
    // ================================================================ producer: slot-map (A1) + 36 TMA boxes per 64-token tile
    const char* tm = static_cast<const char*>(p.tmaps) + static_cast<size_t>(p.layer) * kTmapLayerBytes + 128;   // (64 col x 16 tok x 1)
    const char* tm_pair = tm + 128;                               // (64 x 64 x 2): a whole pair slot in one copy
    const char* tm_blk = tm + 256;                                // (64 x 64 x 1): the rope block in one copy
    const bool big = g.P % kTcTok == 0;                           // a 64-aligned run of 64 tokens of the page list is one page run
    int pair_slot = 0, rope_slot = 0; uint32_t pair_phase = 0, rope_phase = 0; int hdr_i = 0;
    grid_dep_wait();
    for (int seg = seg_begin; seg < seg_end; ++seg) {
      const DecSeg S = p.plan.segs[seg];
      const int32_t* bt = p.block_tables + S.bt_off;
      // tiles are cut at multiples of 64 tokens of the page list, so every inner tile is one page run (first / last may be short)
      for (int t0 = 0; t0 < S.n_tiles;) {
        const int gpos = S.tile0 + t0;                            // 16-token index in the page list
        const int ng = min(kTcGroups - (gpos % kTcGroups), S.n_tiles - t0);
        int slot = 0;                                             // lane i < ng: pool slot of group i
        if (lane < ng) {
          const int tok = (gpos + lane) * kDecTile;
          const int pg = g.P_shift >= 0 ? (tok >> g.P_shift) : tok / g.P;
          slot = bt[pg] * g.P + (tok - pg * g.P);
        }
        const int slot0 = __shfl_sync(0xffffffffu, slot, 0);
        const bool one = big && ng == kTcGroups;                  // full, aligned tile: 5 copies instead of 36
        const int tok0 = gpos * kDecTile;
        const int row_lo = max(S.tok_lo - tok0, 0), row_hi = min(S.tok_hi - tok0, ng * kDecTile);
        // rope block first (its slot also publishes the tile header)
        mbar_wait(&bars[BAR_EMPTY_ROPE + rope_slot], rope_phase ^ 1);
        if (lane == 0) {
          const int flags = (t0 == 0 ? HDR_FIRST : 0) | (t0 + ng >= S.n_tiles ? HDR_LAST : 0) |
                            ((row_lo > 0 || row_hi < kTcTok) ? HDR_PARTIAL : 0);
          hdrs[hdr_i] = make_int4(seg, flags, row_lo | (row_hi << 16), ng);
          mbar_arrive_expect_tx(&bars[BAR_FULL_ROPE + rope_slot], static_cast<uint32_t>(ng) * 2048u);
          if (one) tma_load_3d(smem + kOffRope + rope_slot * kBlkBytes, tm_blk, 0, slot0, 8, &bars[BAR_FULL_ROPE + rope_slot]);
        }
        __syncwarp();
        if (!one && lane < ng) tma_load_3d(smem + kOffRope + rope_slot * kBlkBytes + lane * 2048, tm, 0, slot, 8, &bars[BAR_FULL_ROPE + rope_slot]);
        if (++rope_slot == kTcRopeSlots) { rope_slot = 0; rope_phase ^= 1; }
        hdr_i = (hdr_i + 1) % kTcHdrs;
        for (int b = 0; b < 4; ++b) {                             // the four pairs of latent blocks
          mbar_wait(&bars[BAR_EMPTY_PAIR + pair_slot], pair_phase ^ 1);
          uint8_t* dst0 = smem + kOffPair + pair_slot * kPairBytes;
          if (lane == 0) {
            mbar_arrive_expect_tx(&bars[BAR_FULL_PAIR + pair_slot], static_cast<uint32_t>(ng) * 4096u);
            if (one) tma_load_3d(dst0, tm_pair, 0, slot0, 2 * b, &bars[BAR_FULL_PAIR + pair_slot]);
          }
          __syncwarp();
          if (!one && lane < ng) {
            tma_load_3d(dst0 + lane * 2048, tm, 0, slot, 2 * b, &bars[BAR_FULL_PAIR + pair_slot]);
            tma_load_3d(dst0 + lane * 2048 + kBlkBytes, tm, 0, slot, 2 * b + 1, &bars[BAR_FULL_PAIR + pair_slot]);
          }
          if (++pair_slot == kTcPairSlots) { pair_slot = 0; pair_phase ^= 1; }
        }
        t0 += ng;
      }
    }
    mbar_wait(&bars[BAR_EMPTY_ROPE + rope_slot], rope_phase ^ 1);
    if (lane == 0) { hdrs[hdr_i] = make_int4(-1, 0, 0, 0); mbar_arrive(&bars[BAR_FULL_ROPE + rope_slot]); }
  } else if (warp == 5) {
    // ================================================================ MMA issuer (one lane).  Tile t: S buffer t & 1, rope slot t % 3,
    // pairs (4 t + b) % 10.  QK^T of tile t + 1 is issued BEFORE the PV of tile t (same segment), so the tensor pipe works
    // while the softmax warps turn S(t) into P(t).
    const uint32_t sm0 = smem_u32(smem);
    constexpr uint32_t idesc_qk = tc_idesc(false, 64), idesc_pv = tc_idesc(true, 128);
    uint32_t p_phase = 0, q_phase = 0;
    auto read_hdr = [&](int t) {
      mbar_wait(&bars[BAR_FULL_ROPE + t % kTcRopeSlots], (t / kTcRopeSlots) & 1);
      return hdrs[t % kTcHdrs];
    };
    auto issue_qk = [&](int t, const int4& hdr) {
      tc_fence_after();
      const uint32_t s_tmem = tmem + kTmemS + 128 * (t & 1);
      const bool rotate = p.plan.segs[hdr.x].rotate;
      // k-step k (0-3 rope, then 8 per pair, then the 4 lo steps of a rotated q~) accumulates into partial k % kSParts
      auto step = [&](int k, uint64_t a, uint64_t b_) { tc_mma(s_tmem + 16 * (k % kSParts), a, b_, idesc_qk, k >= kSParts ? 1u : 0u); };
      if (lane == 0) {
        const uint32_t rope = sm0 + kOffRope + (t % kTcRopeSlots) * kBlkBytes;
        for (int j = 0; j < 4; ++j) step(j, tc_desc(rope + j * 32, 16, 1024), tc_desc(sm0 + kOffQhi + 8 * 2048 + j * 32, 16, 1024));
      }
      __syncwarp();
      for (int b = 0; b < 4; ++b) {
        const int c = 4 * t + b, slot = c % kTcPairSlots;
        mbar_wait(&bars[BAR_FULL_PAIR + slot], (c / kTcPairSlots) & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t base = sm0 + kOffPair + slot * kPairBytes;
          for (int half = 0; half < 2; ++half)
            for (int j = 0; j < 4; ++j)
              step(4 + 8 * b + 4 * half + j, tc_desc(base + half * kBlkBytes + j * 32, 16, 1024), tc_desc(sm0 + kOffQhi + (2 * b + half) * 2048 + j * 32, 16, 1024));
        }
        __syncwarp();
      }
      if (lane == 0) {
        if (rotate) {
          const uint32_t rope = sm0 + kOffRope + (t % kTcRopeSlots) * kBlkBytes;
          for (int j = 0; j < 4; ++j) step(36 + j, tc_desc(rope + j * 32, 16, 1024), tc_desc(sm0 + kOffQlo + j * 32, 16, 1024));
        }
        tc_commit(&bars[BAR_EMPTY_ROPE + t % kTcRopeSlots]);
        tc_commit(&bars[BAR_S_FULL + (t & 1)]);
      }
      __syncwarp();
    };
    auto issue_pv = [&](int t, bool first) {
      mbar_wait(&bars[BAR_P_FULL], p_phase); p_phase ^= 1;     // P^T(t) is in shared memory, O rescaled if the reference moved
      tc_fence_after();
      if (lane == 0) {
        for (int j = 0; j < kTcGroups; ++j)                     // 16 tokens per k-step: A advances 16 rows, B 32 bytes;
          for (int b = 0; b < 4; ++b) {                         // the four O blocks are independent accumulators: interleave them
            const uint32_t base = sm0 + kOffPair + ((4 * t + b) % kTcPairSlots) * kPairBytes;
            tc_mma(tmem + 16 * b, tc_desc(base + j * 2048, kBlkBytes, 1024), tc_desc(sm0 + kOffP + j * 32, 16, 1024), idesc_pv,
                   (!first || j > 0) ? 1u : 0u);
          }
        for (int b = 0; b < 4; ++b) tc_commit(&bars[BAR_EMPTY_PAIR + (4 * t + b) % kTcPairSlots]);   // the pairs return to the producer
        tc_commit(&bars[BAR_O_DONE]);
      }
      __syncwarp();
    };
    int tile = 0;
    int4 hdr = read_hdr(tile);
    while (hdr.x >= 0) {                                        // hdr: the FIRST tile of a segment
      if (lane == 0) mbar_arrive(&bars[BAR_SEG]);               // the softmax warps stage q~ of this segment ...
      mbar_wait(&bars[BAR_Q_FULL], q_phase); q_phase ^= 1;      // ... and say when it is in shared memory
      issue_qk(tile, hdr);
      int4 cur = hdr; int cur_t = tile;
      ++tile;
      while (true) {
        const int4 nxt = read_hdr(tile);
        const bool look = nxt.x >= 0 && !(nxt.y & HDR_FIRST);   // same segment: its scores can be computed ahead
        if (look) issue_qk(tile, nxt);
        issue_pv(cur_t, cur.y & HDR_FIRST);
        if (!look) { hdr = nxt; break; }
        cur = nxt; cur_t = tile;
        ++tile;
      }
    }
    if (lane == 0) mbar_arrive(&bars[BAR_SEG]);                 // terminator
  } else {
    // ================================================================ softmax warps 0-3.  The M = 64 score MMA puts token row t of the tile in
    // tensor-memory lane (t % 16) + 32 (t / 16): the lower 16 lanes of warp t / 16.  For O^T (M = 128) lane = value column.
    const int tid = threadIdx.x;
    const int trow_tok = lane < 16 ? warp * 16 + lane : -1;        // the token row this thread owns (none for the upper lanes)
    const uint32_t trow = tmem + (static_cast<uint32_t>(warp * 32) << 16);     // this thread's tensor-memory lane
    const float scale_log2 = p.sm_scale * 1.4426950408889634f;
    float m_ref[16], l_sum[16];
    uint32_t seg_phase = 0, o_phase = 0;
    bool pending_o = false, need_seg = true;
    int n_rows = 0;
    grid_dep_wait();
    for (int ti = 0;; ++ti) {
      if (need_seg) {                                            // the next tile starts a segment (or is the terminator)
        mbar_wait(&bars[BAR_SEG], seg_phase); seg_phase ^= 1;
        if (hdrs[ti % kTcHdrs].x < 0) break;
      }
      const int4 hdr = hdrs[ti % kTcHdrs];
      const int seg = hdr.x;
      const bool first = need_seg;
      need_seg = false;
      if (first) {
        // ---- q~ of the segment into shared memory as the B operand: [9 blocks][16 heads][128 B], 128-byte swizzle; the rope
        // block rotated by -delta and split into bf16 hi + lo.  The previous segment's MMAs are complete (its epilogue waited).
        const DecSeg S = p.plan.segs[seg];
        n_rows = min(kMlaHeads, g.Hq - S.hg * kMlaHeads);
        const float2* cs = p.plan.cs + static_cast<size_t>(S.chunk) * 32;
        const __nv_bfloat16* qb = static_cast<const __nv_bfloat16*>(p.q) + (static_cast<size_t>(S.b) * g.Hq + static_cast<size_t>(S.hg) * kMlaHeads) * 576;
        for (int id = tid; id < 16 * 72; id += 128) {
          const int h = id / 72, ch = id - h * 72, c0 = ch * 8;
          uint4 hi = make_uint4(0, 0, 0, 0), lo = make_uint4(0, 0, 0, 0);
          if (h < n_rows) {
            const __nv_bfloat16* qr = qb + static_cast<size_t>(h) * 576;
            hi = __ldg(reinterpret_cast<const uint4*>(qr + c0));
            if (c0 >= 512 && S.rotate) {
              float x[8], y[8], r[8];
              unpack8(hi, x);
              const int rel = c0 - 512;
              if (g.rope_style == KAM_ROPE_HALF) {
                const bool lower = rel < 32;
                unpack8(__ldg(reinterpret_cast<const uint4*>(qr + (lower ? c0 + 32 : c0 - 32))), y);
#pragma unroll
                for (int e = 0; e < 8; ++e) { const float2 u = cs[(rel & 31) + e]; r[e] = lower ? fmaf(x[e], u.x, y[e] * u.y) : fmaf(x[e], u.x, -y[e] * u.y); }
              } else {
#pragma unroll
                for (int e = 0; e < 8; e += 2) { const float2 u = cs[(rel + e) >> 1]; r[e] = fmaf(x[e], u.x, x[e + 1] * u.y); r[e + 1] = fmaf(x[e + 1], u.x, -x[e] * u.y); }
              }
              hi = pack8(r);
              float hf[8];
              unpack8(hi, hf);
#pragma unroll
              for (int e = 0; e < 8; ++e) r[e] -= hf[e];
              lo = pack8(r);
            }
          }
          const uint32_t off = static_cast<uint32_t>((h >> 3) * 1024 + (h & 7) * 128 + (((((c0 & 63) >> 3) ^ (h & 7)) & 7) << 4));
          *reinterpret_cast<uint4*>(smem + kOffQhi + (c0 >> 6) * 2048 + off) = hi;
          if (c0 >= 512) *reinterpret_cast<uint4*>(smem + kOffQlo + off) = lo;
        }
        fence_proxy_async();
        mbar_arrive(&bars[BAR_Q_FULL]);
#pragma unroll
        for (int h = 0; h < 16; ++h) { m_ref[h] = -CUDART_INF_F; l_sum[h] = 0.f; }
      }

      // ---- S^T row of this token
      mbar_wait(&bars[BAR_S_FULL + (ti & 1)], (ti >> 1) & 1);
      tc_fence_after();
      float v[16];
      tmem_ld16(trow + kTmemS + 128 * (ti & 1), v);
#pragma unroll
      for (int part = 1; part < kSParts; ++part) {
        float w[16];
        tmem_ld16(trow + kTmemS + 128 * (ti & 1) + 16 * part, w);
#pragma unroll
        for (int h = 0; h < 16; ++h) v[h] += w[h];
      }
      const int row_lo = hdr.z & 0xffff, row_hi = hdr.z >> 16;
      const bool valid = trow_tok >= row_lo && trow_tok < row_hi;
      bool need = false;
#pragma unroll
      for (int h = 0; h < 16; ++h) { v[h] = valid ? v[h] * scale_log2 : -CUDART_INF_F; need |= v[h] > m_ref[h] + 8.f; }
      if (pending_o) { mbar_wait(&bars[BAR_O_DONE], o_phase); o_phase ^= 1; pending_o = false; tc_fence_after(); }   // O and P^T are ours again
      if (bar_or_128(1, need)) {
        // ---- some score exceeds its head's reference by more than 2^8: move the references (lazy rescale, as in decode_kernel.cu)
#pragma unroll
        for (int h = 0; h < 16; ++h) {
          float mx = v[h];
#pragma unroll
          for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
          if (lane == 0) red[warp * 16 + h] = mx;
        }
        named_bar_sync(2, 128);
        float alpha[16];
        bool any = false;
#pragma unroll
        for (int h = 0; h < 16; ++h) {
          const float tm = fmaxf(fmaxf(red[h], red[16 + h]), fmaxf(red[32 + h], red[48 + h]));
          const float mn = tm > m_ref[h] + 8.f ? tm : m_ref[h];
          alpha[h] = mn == m_ref[h] ? 1.f : ex2(m_ref[h] - mn);
          any |= alpha[h] != 1.f;
          l_sum[h] *= alpha[h];
          m_ref[h] = mn;
        }
        named_bar_sync(2, 128);                                   // red[] is free again
        if (!first && any) {                                      // O^T rows d = 128 b + tid hold earlier tiles: scale column h by alpha[h]
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            float o[16];
            tmem_ld16(trow + 16 * b, o);
#pragma unroll
            for (int h = 0; h < 16; ++h) o[h] *= alpha[h];
            tmem_st16(trow + 16 * b, o);
          }
          tmem_st_wait();
        }
      }
      // ---- P^T[head][token] in bf16 as the B operand of the PV MMA: 2 token halves x [16 heads][128 B], swizzled
      {
        uint8_t* pbase = smem + kOffP;
        const int c = trow_tok & 63;
#pragma unroll
        for (int h = 0; h < 16; ++h) {
          const float ms = m_ref[h] == -CUDART_INF_F ? 0.f : m_ref[h];
          const float pv = ex2(v[h] - ms);
          l_sum[h] += pv;
          if (trow_tok >= 0) *reinterpret_cast<__nv_bfloat16*>(pbase + sw_off(h, c)) = __float2bfloat16_rn(pv);
        }
      }
      if ((hdr.y & HDR_PARTIAL) && !valid && trow_tok >= 0) {
        // this token row is outside the chunk: whatever it holds (a neighbouring chunk, an unwritten page) must not reach O as 0 * NaN
        for (int b = 0; b < 4; ++b) {
          uint8_t* rowp = smem + kOffPair + ((4 * ti + b) % kTcPairSlots) * kPairBytes + trow_tok * 128;
#pragma unroll
          for (int j = 0; j < 8; ++j) { reinterpret_cast<uint4*>(rowp)[j] = make_uint4(0, 0, 0, 0); reinterpret_cast<uint4*>(rowp + kBlkBytes)[j] = make_uint4(0, 0, 0, 0); }
        }
      }
      fence_proxy_async();
      tc_fence_before();
      mbar_arrive(&bars[BAR_P_FULL]);
      pending_o = true;

      if (hdr.y & HDR_LAST) {
        // ---- the segment's state -> partials: o normalised, lse in natural log
        mbar_wait(&bars[BAR_O_DONE], o_phase); o_phase ^= 1; pending_o = false;
        tc_fence_after();
#pragma unroll
        for (int h = 0; h < 16; ++h) {
          float s = l_sum[h];
#pragma unroll
          for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
          if (lane == 0) red[warp * 16 + h] = s;
        }
        named_bar_sync(2, 128);
        float inv[16];
#pragma unroll
        for (int h = 0; h < 16; ++h) {
          const float tot = (red[h] + red[16 + h]) + (red[32 + h] + red[48 + h]);
          inv[h] = tot > 0.f ? 1.f / tot : 0.f;
          if (tid == h && h < n_rows)
            p.part_lse[static_cast<size_t>(seg) * g.R + h] = tot > 0.f ? (m_ref[h] + log2f(tot)) * 0.6931471805599453f : -CUDART_INF_F;
        }
        named_bar_sync(2, 128);
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          float o[16];
          tmem_ld16(trow + 16 * b, o);
          float* po = p.part_o + static_cast<size_t>(seg) * g.R * 512 + b * 128 + tid;
#pragma unroll
          for (int h = 0; h < 16; ++h) if (h < n_rows) po[static_cast<size_t>(h) * 512] = o[h] * inv[h];
        }
        tc_fence_before();
        need_seg = true;
      }
    }
  }
  // ---- teardown: every role is past its last tensor-memory access
  tc_fence_before();
  __syncthreads();
  if (warp == 5) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols) : "memory");
}

int mla_tc_smem_bytes() { return kTcSmem; }

void launch_mla_tc_decode(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st) {
  cudaFuncSetAttribute(kam_mla_tc_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmem);
  launch_ex(kam_mla_tc_decode_kernel, g.n_ctas, 192, kTcSmem, pdl, st, g, p);
}

}  // namespace kam

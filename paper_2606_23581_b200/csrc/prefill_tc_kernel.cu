// kam_paged_prefill_tc_kernel: the multi-query readout of prefill_kernel.cu on the 5th-generation tensor cores
// (tcgen05.mma, accumulators in tensor memory).
//
// Why tcgen05 HERE: north_star reserves it for the QK^T / PV tiles "only if ncu shows them to be the limiter".  For decode
// (M = the <= 16 query heads of a KV head) the kernels are HBM streams and an N = 16 tcgen05.mma is charged like N = 128
// (round 1 built that kernel and removed it, profiles/HISTORY.md).  For a BLOCK of query rows M = Tq x G >= 128 and the
// mma.sync formulation is the limiter: 183 TFLOP/s with the legacy tensor pipe 54 % active and the time independent of the
// number of MMAs issued (profiles/ncu_extras_r02.md).  Here one CTA owns 128 rows of the flattened (token, head-in-group) row
// space of one KV head and walks the request's cached tokens in 64-token tiles:
//
//   S[128 rows][64 tokens]  = q~ K^T     A = q~ (smem, K-major), B = the K tile (smem, K-major)          8 x tcgen05.mma M128 N64 K16
//   O[128 rows][D]         += P V        A = P (TENSOR MEMORY: written by the softmax threads over S), B = the V tile read MN-major   4 x M128 N128 K16
//
// S (double-buffered, 2 x 64 columns) and O (D columns) live in tensor memory; a softmax thread owns ONE row (its TMEM lane):
// tcgen05.ld of the row, mask, maximum, exp2, the P row (bf16 pairs) stored with tcgen05.st over the first 32 columns of the
// S buffer it came from - PV reads its A operand from there, no shared-memory round trip and no proxy fence -, and the lazy O rescale of the
// FlashAttention-4 kind (only when the row's reference must move by more than 2^8) through tcgen05.ld / st - row statistics
// never cross threads.  Roles: warps 0-3 softmax (128 threads = 128 rows); warp 4 issues the MMAs and owns the tensor-memory
// allocation - it stays CONVERGED and elects the issuing lane inside each asm block (see tc_mma); warps 5-8 load K / V tiles
// with cp.async (one slot lookup per row, shuffled to the copying lanes; slots mapped through the block table per token, rows
// beyond the chunk zero-filled) into a 4-stage ring in the canonical SWIZZLE_128B operand layout ([64-column block][token]
// [128 B], 16-byte chunk index XOR token & 7) and signal a tile's barrier with cp.async.mbarrier.arrive.noinc (no wait_group on
// their path).  QK^T of tile t + 1 is issued before PV of tile t, so the tensor pipe computes scores while the softmax threads
// turn S(t) into P(t).  Relocation on read: q~ = R(-delta) q is rebuilt in shared memory once per chunk (hi + lo; chunks with
// delta = 0 skip the lo products); no look-ahead across a chunk boundary.  Same arithmetic contract, masks and output as
// prefill_kernel.cu (a call with sm_scale <= 0 runs that kernel: the row maximum here is taken before scaling).
// Measured path and where the cycles go: DESIGN.md 7.4.  Diagnostic builds (KAM_NVCC_EXTRA=-DPF_DIAG=n; wrong results): 1 no
// exp2, 2 no QK^T look-ahead, 8 clock64 counters of the MMA warp's and a softmax thread's waits written over two lse rows.
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace kam {

namespace {

constexpr int kTcRows = 128;               // rows per CTA (= TMEM lanes)
constexpr int kTcTile = 64;                // cached tokens per tile
constexpr int kTcStages = 4;
constexpr bool kTcPInTmem = true;         // P(t) is written over the first 32 columns of S(t) in tensor memory and read from there by PV
constexpr int kTcLoaders = 4;              // loader warps: each takes a quarter of a tile's rows
constexpr int kTcThreads = (5 + kTcLoaders) * 32;   // 4 softmax warps + MMA warp + loader warps
enum : int { BAR_KV_FULL = 0, BAR_KV_EMPTY = kTcStages, BAR_S_FULL = 2 * kTcStages /* x2 */, BAR_P_FULL = 2 * kTcStages + 2 /* x2 */, BAR_O_DONE = 2 * kTcStages + 4,
             BAR_Q_READY = 2 * kTcStages + 5, BAR_COUNT = 2 * kTcStages + 6 };

__device__ __forceinline__ void tcf_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcf_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// The MMA warp runs CONVERGED with warp-uniform operands; the single issuing lane is elected INSIDE each asm block.  (An
// `if (lane == 0)` around tcgen05 instructions makes the compiler wrap every one of them in an ELECT / BRA.U.ANY loop and rebuild
// its descriptors with ~16 uniform-datapath instructions: ~420 instructions per tile in the issuing warp - measured with clock64:
// the warp spent 2 270 of 2 460 cycles per tile ISSUING, not waiting.)
__device__ __forceinline__ void tc_commit(uint64_t* bar) {     // arrives on bar when all MMAs issued so far by the elected lane are done
  asm volatile("{\n\t.reg .pred e;\n\telect.sync _|e, 0xffffffff;\n\t"
               "@e tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
// descriptors travel as (low word, high word): the low word is base + (byte offset >> 4), the high word a constant
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p, e;\n\t.reg .b64 da, db;\n\tsetp.ne.b32 p, %6, 0;\n\tmov.b64 da, {%1, %2};\n\tmov.b64 db, {%3, %4};\n\t"
      "elect.sync _|e, 0xffffffff;\n\t"
      "@e tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %5, p;\n\t}"
      ::"r"(d_tmem), "r"(a_lo), "r"(a_hi), "r"(b_lo), "r"(b_hi), "r"(idesc), "r"(accumulate) : "memory");
}
// the same with the A operand in TENSOR MEMORY (the P row block: lane = row, 16 bf16 of K in 8 columns)
__device__ __forceinline__ void tc_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p, e;\n\t.reg .b64 db;\n\tsetp.ne.b32 p, %5, 0;\n\tmov.b64 db, {%2, %3};\n\t"
      "elect.sync _|e, 0xffffffff;\n\t"
      "@e tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], db, %4, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(b_hi), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* r) {      // this thread's lane, 32 consecutive columns
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
               ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]),
                 "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
                 "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
               : "memory");
}
// Shared-memory matrix descriptors (128-byte swizzle = layout type 2, version 1) are built in the MMA warp as two words:
//   low  = (address >> 4) | (lbo >> 4) << 16      high = (sbo >> 4) | 1 << 14 | 2 << 29
// K-major operand: lbo unused (16), sbo = stride between 8-row groups.  MN-major operand (the V tile): lbo = stride between
// 64-element blocks along MN, sbo = stride between groups of 8 K rows.
// instruction descriptor: D = f32, A = B = bf16, M x N, A K-major; b_mn: B is MN-major (the V tile)
__device__ __forceinline__ constexpr uint32_t tc_idesc(uint32_t m, uint32_t n, bool b_mn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn ? 1u : 0u) << 16) | ((n >> 3) << 17) | ((m >> 4) << 24);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// this thread's lane, 32 consecutive columns; the caller waits (tmem_ld_wait) before it touches v
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, float* v) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]),
                 "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]),
                 "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
               : "r"(taddr));
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
__device__ __forceinline__ void cp_async_16z(uint32_t dst, const void* src, bool valid) {
  const int bytes = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ float ex2a(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// byte offset of 16-byte chunk `ch` (of 8) of row r inside one [rows][128 B] SWIZZLE_128B operand block
__device__ __forceinline__ uint32_t sw_chunk(int r, int ch) {
  return static_cast<uint32_t>((r >> 3) * 1024 + (r & 7) * 128 + (((ch ^ r) & 7) << 4));
}

// the same walk as prefill_kernel.cu: 64-token tiles, chunk by chunk, up to the horizon; every role runs it for itself
struct TcTiles {
  const int32_t* cs; const long long* offs;
  int nc, base0, vis_hi;
  int c, lo, hi, pos;
  __device__ __forceinline__ bool enter(int chunk) {
    for (c = chunk; c < nc; ++c) {
      lo = cs[c] - base0; hi = cs[c + 1] - base0;
      if (lo >= vis_hi) return false;
      if (hi > lo) { pos = lo; return true; }
    }
    return false;
  }
  __device__ __forceinline__ bool next() {
    pos += kTcTile;
    if (pos < hi && pos < vis_hi) return true;
    return enter(c + 1);
  }
  __device__ __forceinline__ long long delta() const { return offs ? offs[c] : 0; }
};

}  // namespace

template <int D>
__global__ void __launch_bounds__(kTcThreads, 1) kam_paged_prefill_tc_kernel(const __grid_constant__ PrefillParams p) {
  constexpr int DB = D / 64;                               // 64-column blocks of a row
  constexpr int QBYTES = kTcRows * D * 2;                  // one q~ operand (hi or lo): [DB][128 rows][128 B]
  constexpr int PBYTES = kTcRows * kTcTile * 2;            // P: [128 rows][128 B], two buffers
  constexpr int KVB = kTcTile * D * 2;                     // one K (or V) tile: [DB][64 tokens][128 B]
  constexpr int OFF_Q = 1024, OFF_QLO = OFF_Q + QBYTES, OFF_P = OFF_QLO + QBYTES, OFF_KV = OFF_P + (kTcPInTmem ? 0 : 2 * PBYTES);
  constexpr uint32_t TM_S = 0, TM_O = 2 * kTcTile, TM_COLS = (TM_O + D <= 256) ? 256 : 512;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + 256);
  float2* cs_tab = reinterpret_cast<float2*>(smem + 512);  // (cos, sin)(delta f_i), i < D / 2  (<= 512 bytes)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.z, h = blockIdx.y, G = p.G;
  const int row0 = blockIdx.x * kTcRows;
  const int n_rows = p.Tq * G;
  const int32_t* cs = p.chunk_starts + static_cast<size_t>(b) * (p.max_chunks + 1);
  const int nc = min(p.n_chunks[b], p.max_chunks);
  const int base0 = cs[0];
  const int N = nc > 0 ? cs[nc] - base0 : 0;
  const int t_lo = row0 / G, t_hi = min(row0 + kTcRows - 1, n_rows - 1) / G;
  const int shift = N - p.Tq;
  TcTiles cur;
  cur.cs = cs; cur.offs = p.chunk_offsets ? p.chunk_offsets + static_cast<size_t>(b) * p.max_chunks : nullptr;
  cur.nc = nc; cur.base0 = base0;
  cur.vis_hi = p.causal ? min(N, max(0, shift + t_hi + 1)) : N;
  bool more = cur.enter(0);

  if (threadIdx.x == 0) {
    for (int i = 0; i < kTcStages; ++i) { mbar_init(&bars[BAR_KV_FULL + i], kTcLoaders * 32); mbar_init(&bars[BAR_KV_EMPTY + i], 1); }
    mbar_init(&bars[BAR_S_FULL], 1); mbar_init(&bars[BAR_S_FULL + 1], 1);
    mbar_init(&bars[BAR_P_FULL], 128); mbar_init(&bars[BAR_P_FULL + 1], 128); mbar_init(&bars[BAR_O_DONE], 1); mbar_init(&bars[BAR_Q_READY], 128);
    mbar_fence_init();
  }
  if (warp == 4) {                                          // one warp allocates the tensor memory and owns the deallocation
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(const_cast<uint32_t*>(tmem_slot))), "n"(TM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tcf_before();
  __syncthreads();
  tcf_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t sm0 = smem_u32(smem);

  if (warp >= 5) {
    // ================================================================ loaders: cp.async of K and V tiles into the ring; warp w takes rows
    // [16 (w - 5), +16) of every tile
    const int32_t* bt = p.block_tables + static_cast<size_t>(b) * p.max_pages;
    const char* pool_k = static_cast<const char*>(p.pool_k_layers[p.layer]);
    const char* pool_v = static_cast<const char*>(p.pool_v_layers[p.layer]);
    const size_t tok_bytes = static_cast<size_t>(p.H) * D * 2, head_off = static_cast<size_t>(h) * D * 2;
    constexpr int CPR = D / 8;                              // 16-byte chunks per row
    constexpr int RPP = 32 / CPR;                           // rows per pass of the warp (2 at D = 128, 4 at D = 64)
    constexpr int RPW = kTcTile / kTcLoaders;               // rows per loader warp
    const int lc = lane % CPR;
    static_assert(RPW <= 32 && (RPW & (RPW - 1)) == 0, "one slot per lane");
    const uint32_t dst_c = static_cast<uint32_t>((lc >> 3) * (kTcTile * 128));       // the chunk's 64-column block
    int issued = 0;
    const char* kbase = pool_k + head_off + lc * 16;
    const char* vbase = pool_v + head_off + lc * 16;
    const int wrow0 = (warp - 5) * RPW;                     // this warp's first row of a tile
    while (more) {
      const int st = issued % kTcStages;
      // A1 slot mapping, once per row: lane l < RPW maps row wrow0 + l; the copy loop below takes it by shuffle
      int myslot = -1;
      {
        const int tok = cur.pos + wrow0 + (lane & (RPW - 1));
        if (tok < cur.hi) {
          const int pg = p.P_shift >= 0 ? (tok >> p.P_shift) : tok / p.P;
          const int page = pg < p.max_pages ? bt[pg] : -1;
          if (page >= 0 && page < p.num_pages) myslot = page * p.P + (tok - pg * p.P);
          else if (lane < RPW && (tok == cur.pos + wrow0 || tok == pg * p.P)) atomicAdd(p.err, 1);   // a zero row, never a wild read
        }
      }
      if (issued >= kTcStages) mbar_wait(&bars[BAR_KV_EMPTY + st], ((issued / kTcStages) - 1) & 1);
      const uint32_t kd = sm0 + OFF_KV + st * 2 * KVB + dst_c, vd = kd + KVB;
#pragma unroll
      for (int i = 0; i < RPW / RPP; ++i) {
        const int rr = lane / CPR + i * RPP;                  // row inside the warp's RPW rows
        const int slot = __shfl_sync(0xffffffffu, myslot, rr);
        const bool valid = slot >= 0;                          // rows beyond the chunk are zero-filled
        const size_t off = valid ? static_cast<size_t>(slot) * tok_bytes : 0;
        const uint32_t d = sw_chunk(wrow0 + rr, lc & 7);
        cp_async_16z(kd + d, kbase + off, valid);
        cp_async_16z(vd + d, vbase + off, valid);
      }
      // the tile's barrier hears from this thread when ITS copies have landed (no wait here: up to kTcStages tiles stay in flight)
      asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(&bars[BAR_KV_FULL + st])) : "memory");
      ++issued;
      more = cur.next();
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
#if defined(PF_DIAG) && (PF_DIAG & 8)
    asm volatile("bar.sync 7, %0;" ::"n"(kTcThreads) : "memory");
#endif
  } else if (warp == 4) {
    // ================================================================ MMA issuer (lane 0 issues; the warp stays converged for dealloc)
    constexpr uint32_t idesc_qk = tc_idesc(kTcRows, kTcTile, false), idesc_pv = tc_idesc(kTcRows, D, true);
    uint32_t q_phase = 0;
    int cur_chunk = -1;
    bool use_lo = false;
#if defined(PF_DIAG) && (PF_DIAG & 8)
    long long dbg_kv = 0, dbg_p = 0, dbg_t0 = clock64();
#define DBG_T(acc, stmt) { const long long c0_ = clock64(); stmt; acc += clock64() - c0_; }
#else
#define DBG_T(acc, stmt) { stmt; }
    long long dbg_kv = 0, dbg_p = 0;
#endif
    // descriptor words: hi = (sbo >> 4) | version 1 << 14 | swizzle-128B << 29 (+ the lbo field in the low word's upper half)
    constexpr uint32_t kHiK = (1024u >> 4) | (1u << 14) | (2u << 29);
    constexpr uint32_t kLoK = (16u >> 4) << 16;                                   // K-major operands: lbo unused (16)
    constexpr uint32_t kLoV = ((kTcTile * 128u) >> 4) << 16;                      // the V tile, MN-major: lbo = stride between 64-column blocks
    const uint32_t q_lo = kLoK | ((sm0 + OFF_Q) >> 4), ql_lo = kLoK | ((sm0 + OFF_QLO) >> 4), p_lo = kLoK | ((sm0 + OFF_P) >> 4);
    const uint32_t kv_lo = (sm0 + OFF_KV) >> 4;
    auto issue_qk = [&](int t) {
      const int st = t % kTcStages;
      DBG_T(dbg_kv, mbar_wait(&bars[BAR_KV_FULL + st], (t / kTcStages) & 1));
      fence_proxy_async();                                  // the tile was written by cp.async (generic proxy), tcgen05.mma reads through the async proxy
      tcf_after();
      const uint32_t k_lo = kLoK | (kv_lo + st * (2 * KVB >> 4));
      const uint32_t s_t = tmem + TM_S + kTcTile * (t & 1);
#pragma unroll
      for (int ks = 0; ks < D / 16; ++ks)
        tc_mma(s_t, q_lo + (((ks >> 2) * (kTcRows * 128) + (ks & 3) * 32) >> 4), kHiK,
               k_lo + (((ks >> 2) * (kTcTile * 128) + (ks & 3) * 32) >> 4), kHiK, idesc_qk, ks > 0 ? 1u : 0u);
      if (use_lo) {
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks)
          tc_mma(s_t, ql_lo + (((ks >> 2) * (kTcRows * 128) + (ks & 3) * 32) >> 4), kHiK,
                 k_lo + (((ks >> 2) * (kTcTile * 128) + (ks & 3) * 32) >> 4), kHiK, idesc_qk, 1u);
      }
      tc_commit(&bars[BAR_S_FULL + (t & 1)]);
    };
    auto issue_pv = [&](int t) {
      DBG_T(dbg_p, mbar_wait(&bars[BAR_P_FULL + (t & 1)], (t >> 1) & 1));   // P(t) is in shared memory, O rescaled if a reference moved
      tcf_after();
      const int st = t % kTcStages;
      const uint32_t v_lo = kLoV | (kv_lo + ((st * 2 * KVB + KVB) >> 4));
      const uint32_t pa_lo = p_lo + (t & 1) * (PBYTES >> 4);
#pragma unroll
      for (int kk = 0; kk < kTcTile / 16; ++kk)
        if (kTcPInTmem) tc_mma_ts(tmem + TM_O, tmem + TM_S + kTcTile * (t & 1) + 8 * kk, v_lo + ((kk * 2048) >> 4), kHiK, idesc_pv, (t > 0 || kk > 0) ? 1u : 0u);
        else tc_mma(tmem + TM_O, pa_lo + ((kk * 32) >> 4), kHiK, v_lo + ((kk * 2048) >> 4), kHiK, idesc_pv, (t > 0 || kk > 0) ? 1u : 0u);
      tc_commit(&bars[BAR_KV_EMPTY + st]);                  // the stage returns to the loader
      tc_commit(&bars[BAR_O_DONE]);
    };
    auto enter_chunk = [&]() {                               // q~ of the tile's chunk is staged by the softmax threads
      if (cur.c != cur_chunk) {
        cur_chunk = cur.c;
        use_lo = cur.delta() != 0;
        mbar_wait(&bars[BAR_Q_READY], q_phase); q_phase ^= 1;
        tcf_after();
      }
    };
    int t = 0;
    if (more) { enter_chunk(); issue_qk(0); }
    while (more) {
      TcTiles nxt = cur;
      const bool has_next = nxt.next();
#if defined(PF_DIAG) && (PF_DIAG & 2)
      const bool look = false;
#else
      const bool look = has_next && nxt.c == cur.c;          // same chunk: its scores are computed ahead of this tile's PV
#endif
      if (look) issue_qk(t + 1);
      issue_pv(t);
      cur = nxt; more = has_next;
      if (has_next && !look) { enter_chunk(); issue_qk(t + 1); }
      ++t;
    }
#if defined(PF_DIAG) && (PF_DIAG & 8)
    __syncwarp();
    asm volatile("bar.sync 7, %0;" ::"n"(kTcThreads) : "memory");          // everyone's results are written: the debug words go on top
    if (lane == 0 && blockIdx.x == 3) {
      float* dbg = p.lse + (static_cast<size_t>(b) * p.Tq + 55) * p.Hq + h * G;
      dbg[0] = static_cast<float>(clock64() - dbg_t0); dbg[1] = static_cast<float>(dbg_kv); dbg[2] = static_cast<float>(dbg_p); dbg[3] = static_cast<float>(t);
    }
#endif
    (void)dbg_kv; (void)dbg_p;
  } else {
    // ================================================================ softmax threads: thread = row = tensor-memory lane
    const int r = threadIdx.x;                               // 0 .. 127
    const uint32_t trow = tmem + (static_cast<uint32_t>(warp * 32) << 16);      // this warp's lane quadrant
    const int fr = row0 + r;
    const bool live = fr < n_rows;
    const int tq = fr / G, gh = fr - tq * G;
    const int lim = p.causal ? shift + tq : N;
    const int cta_lim_lo = p.causal ? shift + t_lo : N;
    const char* qrow = static_cast<const char*>(p.q) + ((static_cast<size_t>(b) * p.Tq + (live ? tq : 0)) * p.Hq + h * G + (live ? gh : 0)) * D * 2;
    const float scale_log2 = p.sm_scale * 1.4426950408889634f;
    float m_ref = -CUDART_INF_F, l_sum = 0.f;
    uint32_t o_phase = 0;
    int cur_chunk = -1, t = 0;
    [[maybe_unused]] long long dbg_s = 0, dbg_s0 = clock64();
    while (more) {
      if (cur.c != cur_chunk) {
        // ---- new chunk: q~ = R(-delta) q of this thread's row into the A operand (hi, and lo when rotated).  Every MMA that
        // read the previous q~ has completed: this thread waited for the S of the previous chunk's last tile.
        cur_chunk = cur.c;
        const long long delta = cur.delta();
        const bool rot = delta != 0;
        if (rot) {
          if (r < D / 2) {
            double sn, csn;
            sincos(static_cast<double>(delta) * p.inv_freq[r], &sn, &csn);      // fp64 angle (R-18)
            cs_tab[r] = make_float2(static_cast<float>(csn), static_cast<float>(sn));
          }
          named_bar_sync(1, 128);
        }
        constexpr int CH = D / 8;                            // 16-byte chunks of a row
        if (!rot) {
#pragma unroll
          for (int c = 0; c < CH; ++c) {
            const uint4 v = live ? __ldg(reinterpret_cast<const uint4*>(qrow) + c) : make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4*>(smem + OFF_Q + (c >> 3) * (kTcRows * 128) + sw_chunk(r, c & 7)) = v;
          }
        } else {
          // HALF: chunk c (columns 8c ..) pairs with chunk c + CH/2; INTERLEAVED: pairs inside the chunk
#pragma unroll
          for (int c = 0; c < CH / 2; ++c) {
            float x[8], y[8], rx[8], ry[8];
            const int ca = p.rope_style == KAM_ROPE_HALF ? c : 2 * c, cb = p.rope_style == KAM_ROPE_HALF ? c + CH / 2 : 2 * c + 1;
            unpack8(live ? __ldg(reinterpret_cast<const uint4*>(qrow) + ca) : make_uint4(0, 0, 0, 0), x);
            unpack8(live ? __ldg(reinterpret_cast<const uint4*>(qrow) + cb) : make_uint4(0, 0, 0, 0), y);
            if (p.rope_style == KAM_ROPE_HALF) {
#pragma unroll
              for (int e = 0; e < 8; ++e) {
                const float2 u = cs_tab[8 * c + e];
                rx[e] = fmaf(x[e], u.x, y[e] * u.y);
                ry[e] = fmaf(y[e], u.x, -x[e] * u.y);
              }
            } else {
#pragma unroll
              for (int e = 0; e < 8; e += 2) {
                const float2 u = cs_tab[8 * c + (e >> 1)], w = cs_tab[8 * c + 4 + (e >> 1)];
                rx[e] = fmaf(x[e], u.x, x[e + 1] * u.y); rx[e + 1] = fmaf(x[e + 1], u.x, -x[e] * u.y);
                ry[e] = fmaf(y[e], w.x, y[e + 1] * w.y); ry[e + 1] = fmaf(y[e + 1], w.x, -y[e] * w.y);
              }
            }
            const uint4 hx = pack8(rx), hy = pack8(ry);
            float fx[8], fy[8];
            unpack8(hx, fx); unpack8(hy, fy);
#pragma unroll
            for (int e = 0; e < 8; ++e) { rx[e] -= fx[e]; ry[e] -= fy[e]; }
            const uint32_t oa = (ca >> 3) * (kTcRows * 128) + sw_chunk(r, ca & 7), ob = (cb >> 3) * (kTcRows * 128) + sw_chunk(r, cb & 7);
            *reinterpret_cast<uint4*>(smem + OFF_Q + oa) = hx; *reinterpret_cast<uint4*>(smem + OFF_Q + ob) = hy;
            *reinterpret_cast<uint4*>(smem + OFF_QLO + oa) = pack8(rx); *reinterpret_cast<uint4*>(smem + OFF_QLO + ob) = pack8(ry);
          }
        }
        fence_proxy_async();
        mbar_arrive(&bars[BAR_Q_READY]);
      }

      // ---- this row of S(t)
#if defined(PF_DIAG) && (PF_DIAG & 8)
      { const long long c0_ = clock64(); mbar_wait(&bars[BAR_S_FULL + (t & 1)], (t >> 1) & 1); dbg_s += clock64() - c0_; }
#else
      mbar_wait(&bars[BAR_S_FULL + (t & 1)], (t >> 1) & 1);
#endif
      tcf_after();
      float s[kTcTile];
#pragma unroll
      for (int j = 0; j < kTcTile / 32; ++j) tmem_ld32_nowait(trow + TM_S + kTcTile * (t & 1) + 32 * j, s + 32 * j);
      tmem_ld_wait();
      const int tile_hi = min(cur.pos + kTcTile, cur.hi) - 1;
      const bool masked = (cur.pos + kTcTile > cur.hi) || (tile_hi > cta_lim_lo);      // CTA-uniform
      if (masked) {                                           // only where the chunk ends inside the tile or the diagonal crosses it
        const int last = min(tile_hi, lim) - cur.pos;         // last visible column of this row in the tile (may be < 0)
#pragma unroll
        for (int j = 0; j < kTcTile; ++j) if (j > last) s[j] = -CUDART_INF_F;
      }
      float mx = s[0];
#pragma unroll
      for (int j = 1; j < kTcTile; ++j) mx = fmaxf(mx, s[j]);
      mx *= scale_log2;                                       // sm_scale > 0: the scaled maximum is the maximum of the scaled scores
      const bool need = mx > m_ref + 8.f;                     // lazy reference: moves only when a score runs 2^8 past it
      // P has two buffers: P(t) may be written while PV(t - 1) still runs (PV(t - 2), the last reader of this buffer, was seen
      // complete during tile t - 1).  Only a rescale of O must wait for PV(t - 1) first; otherwise that wait moves behind the
      // P write, where it has long been satisfied.
      bool o_pending = t > 0;
      if (__any_sync(0xffffffffu, need)) {
        if (o_pending) { mbar_wait(&bars[BAR_O_DONE], o_phase); o_phase ^= 1; tcf_after(); o_pending = false; }
        const float mn = need ? mx : m_ref;
        const float alpha = (mn == m_ref) ? 1.f : ex2a(m_ref - mn);     // m_ref = -inf -> 0
        l_sum *= alpha;
        m_ref = mn;
        if (t > 0) {                                          // O holds earlier tiles: scale this row (warp-collective ld / st)
#pragma unroll
          for (int j = 0; j < D / 16; ++j) {
            float o[16];
            tmem_ld16(trow + TM_O + 16 * j, o);
#pragma unroll
            for (int e = 0; e < 16; ++e) o[e] *= alpha;
            tmem_st16(trow + TM_O + 16 * j, o);
          }
          tmem_st_wait();
        }
      }
      // ---- P row (bf16) as the A operand of PV: [128 rows][128 B], swizzled
      const float nref = m_ref == -CUDART_INF_F ? 0.f : -m_ref;
      float ls0 = 0.f, ls1 = 0.f;
      [[maybe_unused]] uint32_t pw[kTcTile / 2];
#pragma unroll
      for (int c = 0; c < kTcTile / 8; ++c) {
        float pv[8];
#pragma unroll
#if defined(PF_DIAG) && (PF_DIAG & 1)
        for (int e = 0; e < 8; ++e) pv[e] = s[8 * c + e];
#else
        for (int e = 0; e < 8; ++e) pv[e] = ex2a(fmaf(s[8 * c + e], scale_log2, nref));     // e^{s - m}: -inf -> 0
#endif
        ls0 += (pv[0] + pv[1]) + (pv[2] + pv[3]); ls1 += (pv[4] + pv[5]) + (pv[6] + pv[7]);
        const uint4 pk = pack8(pv);
        if (kTcPInTmem) { pw[4 * c] = pk.x; pw[4 * c + 1] = pk.y; pw[4 * c + 2] = pk.z; pw[4 * c + 3] = pk.w; }
        else *reinterpret_cast<uint4*>(smem + OFF_P + (t & 1) * PBYTES + sw_chunk(r, c)) = pk;
      }
      l_sum += ls0 + ls1;
      if (kTcPInTmem) {
        // P(t) over the first 32 columns of S(t): this thread has its S row in registers; the next writer of these columns is
        // QK^T of tile t + 2, issued after PV(t) and executed behind it
#pragma unroll
        for (int j = 0; j < kTcTile / 64; ++j) tmem_st32(trow + TM_S + kTcTile * (t & 1) + 32 * j, pw + 32 * j);
        tmem_st_wait();
      } else {
        fence_proxy_async();
      }
      // O_DONE is ONE barrier read by parity: PV(t - 1)'s completion must be observed BEFORE this thread lets PV(t) go (its P_FULL
      // arrival below).  In the other order a thread held up between the two could see PV(t - 1) and PV(t) both complete - the
      // parity back where it was - and wait for PV(t + 1), which needs this thread's own next arrival: a hang.  Behind the P
      // write the wait has long been satisfied, so it costs one poll.
      if (o_pending) { mbar_wait(&bars[BAR_O_DONE], o_phase); o_phase ^= 1; tcf_after(); }
      tcf_before();
      mbar_arrive(&bars[BAR_P_FULL + (t & 1)]);
      more = cur.next();
      ++t;
    }
    // ---- epilogue: out = O / l, lse = ln 2 * m + ln l; a row that saw nothing: 0 and -inf
    if (t > 0) { mbar_wait(&bars[BAR_O_DONE], o_phase); tcf_after(); }
    const float inv = l_sum > 0.f ? 1.f / l_sum : 0.f;
    const size_t orow = (static_cast<size_t>(b) * p.Tq + (live ? tq : 0)) * p.Hq + h * G + (live ? gh : 0);
    uint4* op = reinterpret_cast<uint4*>(static_cast<char*>(p.out) + orow * D * 2);
#pragma unroll
    for (int j = 0; j < D / 16; ++j) {
      float o[16];
      if (t > 0) tmem_ld16(trow + TM_O + 16 * j, o);
      else {
#pragma unroll
        for (int e = 0; e < 16; ++e) o[e] = 0.f;
      }
#pragma unroll
      for (int e = 0; e < 16; ++e) o[e] *= inv;
      if (live) { op[2 * j] = pack8(o); op[2 * j + 1] = pack8(o + 8); }
    }
    if (live) p.lse[orow] = l_sum > 0.f ? m_ref * 0.6931471805599453f + logf(l_sum) : -CUDART_INF_F;
#if defined(PF_DIAG) && (PF_DIAG & 8)
    const long long dbg_tot = clock64() - dbg_s0;
    asm volatile("bar.sync 7, %0;" ::"n"(kTcThreads) : "memory");
    if (threadIdx.x == 0 && blockIdx.x == 3) {
      float* dbg = p.lse + (static_cast<size_t>(b) * p.Tq + 56) * p.Hq + h * G;
      dbg[0] = static_cast<float>(dbg_tot); dbg[1] = static_cast<float>(dbg_s); dbg[3] = static_cast<float>(t);
    }
#endif
  }
  // ---- teardown: every role is past its last tensor-memory access
  tcf_before();
  __syncthreads();
  if (warp == 4) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TM_COLS) : "memory");
}

int prefill_tc_smem_bytes(int D) { return 1024 + 2 * kTcRows * D * 2 + (kTcPInTmem ? 0 : 2 * kTcRows * kTcTile * 2) + kTcStages * 2 * kTcTile * D * 2; }

void launch_prefill_tc(const PrefillParams& p, int D, cudaStream_t st) {
  const int smem = prefill_tc_smem_bytes(D);
  dim3 grid((p.Tq * p.G + kTcRows - 1) / kTcRows, p.H, p.batch);
  static std::atomic<uint64_t> attr_done{0};          // per device: the attribute is not shared between GPUs
  if (first_launch_on_this_device(attr_done)) {
    cudaFuncSetAttribute(kam_paged_prefill_tc_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, prefill_tc_smem_bytes(128));
    cudaFuncSetAttribute(kam_paged_prefill_tc_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, prefill_tc_smem_bytes(64));
  }
  if (D == 128) kam_paged_prefill_tc_kernel<128><<<grid, kTcThreads, smem, st>>>(p);
  else kam_paged_prefill_tc_kernel<64><<<grid, kTcThreads, smem, st>>>(p);
}

}  // namespace kam

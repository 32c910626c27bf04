// Host/device records shared between the libkamera entry points and its kernels.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/kamera.h"

namespace kam {

// ---------------------------------------------------------------- relocate + patch
// One chunk of a (batched) relocate call, as the kernels see it.
struct RelocDescDev {
  const void* const* k_src;      // device array [L] -> [T][H][D]; unused when FLAG_INPLACE
  const void* const* v_src;
  const void* const* Uk;         // device arrays [L] or nullptr
  const void* const* Wk;
  const void* const* Uv;
  const void* const* Wv;
  const int32_t* block_table;    // device
  long long dst_token_start;
  long long delta;               // p_target - p_base
  long long u_token_stride;      // elements
  long long u_head_stride;       // elements; 0 => U shared by all heads
  int32_t n_tokens;
  int32_t flags;
  int32_t tile_weight;           // relative cost of one tile of this chunk (the CTAs' shares are cut by weight, not by count)
  uint8_t rank_l[KAM_MAX_LAYERS];
};
enum : int32_t { FLAG_INPLACE = 1, FLAG_CANONICAL_FRAME = 2,
                 FLAG_INLINE_PAGES = 4 };   // the chunk's page list is RelocPages in the kernel parameters, not block_table

// A column block of a token's slice: what one warp processes for 16 tokens (up to 4 groups of 32 columns).
struct ColBlock {
  int16_t col_off;      // first column, relative to the slice
  int16_t w_col_off;    // same column, relative to its head's row (index into W's last dim)
  int16_t band_col0;    // column relative to the rope band start (rope blocks only)
  int8_t n_groups;      // 2 or 4
  int8_t fhead;         // head index inside the head group (selects U/W head)
  int8_t rope;          // 1 if the block lies in the rope band
  int8_t pad[3];
};

constexpr int kMaxColBlocks = 24;
constexpr int kRelocConsumerWarps = 8;
constexpr int kRelocProducerWarps = 4;     // K rows | V rows | U_k | U_v
constexpr int kRelocThreads = (kRelocConsumerWarps + kRelocProducerWarps) * 32;

struct RelocGeom {
  int32_t L, H, D, P;
  int32_t P_shift;              // log2(P) if P is a power of two, else -1
  int32_t contig;               // 1: slice == whole token row and shared-memory rows are unpadded (one copy per tile)
  int32_t HG, n_hg;             // KV heads per slice, slices per token row
  int32_t slice_bytes;          // HG * D * 2
  int32_t row_bytes;            // H * D * 2 : one token of one layer in chunk and pool
  int32_t s_row;                // padded shared-memory stride of a token's slice (== 64 mod 128)
  int32_t su_row;               // padded shared-memory stride of a token's U run ((su_row/16) odd)
  int32_t RB, TT;               // 16-token row blocks per tile; TT = 16 * RB tokens
  int32_t nkv;                  // 2 with a V pool, 1 for MLA
  int32_t n_blocks;
  int32_t KT_max;               // 16-wide rank tiles of the largest rank of the call: ceil(max rank / 16)
  int32_t kv_split;             // 1: a tile carries K rows OR V rows (the tile list gets a kv level): only one of W_k / W_v is
                                //    resident at a time, which is what lets three stages fit at ranks 48 / 64
  int32_t rope_style, d_r, half_groups;   // half_groups = d_r / 64 for HALF
  int32_t n_stages;
  int32_t off_tab, off_cs, off_w, off_stage0, stage_bytes;   // byte offsets in dynamic shared memory
  int32_t w_row;                // bytes of one k-row of W in shared memory: (D + 8) * 2
  int32_t st_k, st_v, st_uk, st_uv, st_slot;        // offsets inside a stage
  int32_t w_kv_stride;          // bytes of one of {K,V}'s fragment table
  int32_t smem_bytes;
  int32_t load_hint;            // 1: canonical sources are read with L2 evict_first
  double theta;
  ColBlock blk[kMaxColBlocks];
};

// How the U rows of a (chunk, layer) of rank m travel to shared memory (producer and consumers of the kernel and the host's
// eligibility check all ask this one function).  NATIVE: the tile's rows are one contiguous run of the caller's array - one
// copy, the caller's strides kept in shared memory (ldmatrix then sees rows at a power-of-two stride: 8-way bank conflicts,
// tolerable for the ONE ldmatrix per slab of rank <= 16, and the only form that can carry ranks whose runs are not multiples
// of 16 bytes).  ROWS: one copy per token (heads adjacent) or per (token, head) into rows padded to an odd multiple of 16
// bytes - conflict-free, what ranks > 16 use when their runs are 16-byte multiples.  NONE: the element-wise kernel.
#ifndef KAM_U_NATIVE_BELOW
#define KAM_U_NATIVE_BELOW 17
#endif
enum : int { U_NONE = 0, U_NATIVE = 1, U_ROWS = 2 };
__host__ __device__ inline int u_form(int su_row, int HG, int n_hg, int m, long long uts, long long uhs) {
  const bool native_ok = uts * 2 <= su_row - 16 && (uhs == 0 || n_hg == 1);
  const int hf_n = uhs == 0 ? 1 : HG;
  const bool heads_adjacent = hf_n == 1 || uhs == m;
  const bool rows_ok = (uts * 2) % 16 == 0 && ((long long)HG * uhs * 2) % 16 == 0 &&
                       (heads_adjacent ? ((long long)hf_n * m * 2) % 16 == 0 : (m * 2) % 16 == 0 && (uhs * 2) % 16 == 0);
  if (native_ok && (m < KAM_U_NATIVE_BELOW || !rows_ok)) return U_NATIVE;
  return rows_ok ? U_ROWS : U_NONE;
}

constexpr int kRelocInlineDescs = 8;   // batches up to this size travel in the kernel parameters
struct RelocInline {
  RelocDescDev d[kRelocInlineDescs];
  long long prefix[kRelocInlineDescs + 1];
  long long wprefix[kRelocInlineDescs + 1];
};
// The page list of a chunk admitted to a window travels in the kernel parameters too: the kernel maps its slots from here and
// CTA 0 writes the list to the device mirror of the window's page lists - a slide is one launch and no copy.
constexpr int kRelocInlinePages = 256;
struct RelocPages {
  int32_t pages[kRelocInlinePages];
  int32_t* mirror_dst;           // device mirror row of the chunk's slot, or nullptr (no inline page list in this launch)
  int32_t n;
};

struct RelocParams {
  const RelocDescDev* descs;     // device array, or nullptr => RelocInline
  const long long* tile_prefix;  // [n_descs + 1]
  const long long* w_prefix;     // [n_descs + 1] cumulative tile weights
  long long total_weight;
  void* const* pool_k;
  void* const* pool_v;
  const double* inv_freq;        // [d_r / 2] f_i = theta^(-2i/d_r) in fp64 (written at kam_create), or nullptr
  long long total_tiles;
  int32_t n_descs;
  int32_t num_pages;             // block-table entries outside [0, num_pages) are skipped and counted in *err
  int32_t* err;                  // device counter (kam_stats.device_errors)
};

// generic (any dtype / rank / width) element-wise path
struct GenericParams {
  const RelocDescDev* descs;
  void* const* pool_k;
  void* const* pool_v;
  int32_t n_descs, L, H, D, P, rope_off, d_r, rope_style, has_v, elem_f32, factor_f32;
  int32_t num_pages;
  int32_t* err;
  double theta;
};

void launch_relocate_fast(const RelocGeom& g, const RelocParams& p, const RelocInline& inl, const RelocPages* pages /* or nullptr */, int grid, bool pdl, cudaStream_t st);
void launch_relocate_generic(const GenericParams& p, int max_tokens, cudaStream_t st);

// ---------------------------------------------------------------- decode
constexpr int kTmapLayerBytes = 2 * 128;   // tensor maps per layer: K | V (MLA: one map, the whole 576-wide row x 16 tokens)
constexpr int kDecTile = 16;               // tokens per pipeline box (one TMA box of K or of V)
constexpr int kDecMaxHG = 4;               // KV heads (= compute warps) per CTA
constexpr int kDecPlanThreads = 1024;

struct DecodeGeom {
  int32_t Hq, H, G, D, Dv, P, P_shift;
  int32_t HG, n_hg;              // KV heads per work unit (one compute warp each), units per token row
  int32_t R;                     // query rows per unit = HG * G (rows of one partial)
  int32_t NT;                    // 8-wide query-head tiles per KV head: ceil(G / 8)
  int32_t rope_off, d_r, rope_style;
  int32_t row_bytes, slice_bytes, s_row;      // s_row: padded stride of a token's slice in shared memory (bulk-copy path)
  int32_t n_boxes, box_bytes;    // ring of boxes; K and V tiles alternate (even = K, odd = V)
  int32_t off_hdr, off_box0, smem_bytes;
  int32_t use_tma;               // 1: pool pages arrive as 16-token swizzled TMA boxes; 0: one padded bulk copy per token
  int32_t ncb;                   // TMA path: 64-column blocks per slice
  int32_t n_ctas;                // persistent grid: sm_count * CTAs per SM
  int32_t KT;                    // on-read patch: 16-wide rank tiles the kernel is specialised for (0: no patch in this call)
  int32_t kv_bytes;              // bytes of the K (or V) rows of a box; box_bytes = kv_bytes + the U tile (KT > 0)
  int32_t u_off, su_row;         // U tile inside a box: [16 tokens][su_row bytes], (su_row / 16) odd
  int32_t mla;                   // 1: absorbed MLA decode (one latent+rope row per token, value = its first Dv columns)
};

struct DecChunk {                // plan input: one chunk of one request (flat, request-major)
  long long bt_off;              // index of the chunk's page list (its first entry) in the block-table array
  long long delta;               // RoPE offset to apply on read
  int32_t b;                     // request index in the batch
  int32_t tok0, n_tok;           // tokens [tok0, tok0 + n_tok) of that page list
  int32_t patch;                 // index into the patch-ref array, or -1
};

struct DecSeg {                  // plan output: a run of 16-token tiles inside ONE chunk, owned by one CTA
  long long bt_off;
  int32_t chunk;                 // flat chunk index (row of the cos/sin table, patch lookup)
  int32_t b, hg;
  int32_t tile0, n_tiles;        // tiles [tile0, tile0 + n_tiles) of the page list, 16 tokens each
  int32_t tok_lo, tok_hi;        // the chunk's tokens of that page list: rows outside are masked
  int32_t rotate;                // 1: delta != 0, q is rotated by -delta on read
  int32_t patch;                 // index into the patch-ref array, or -1
  int32_t slot0;                 // pool slot of the segment's first tile (saves the producer one dependent load)
};

struct DecodePlan {              // device pointers into the workspace; filled by the plan kernel
  DecChunk* chunks;              // [n_chunks]
  int32_t* rcb;                  // [batch + 1] request -> first flat chunk
  int32_t* tile_pre;             // [n_chunks + 1]
  int32_t* seg_base;             // [n_hg * n_chunks + 1]
  DecSeg* segs;                  // [max_segs]
  int32_t* cta_seg;              // [n_ctas + 1]
  float2* cs;                    // [n_chunks][d_r / 2] (cos, sin)(delta f_i)
  const double* inv_freq;        // [d_r / 2] f_i = theta^(-2i/d_r), fp64, written at kam_create
  const int32_t* block_tables;   // the call's block-table array (segments record their first slot)
  int32_t* dyn;                  // [0] = n_chunks as the plan kernel saw it.  The merge kernel reads it from HERE, not from its
                                 // parameters: a CUDA graph captured over kam_window_decode replays stale parameters after
                                 // the windows' chunk count changed, the workspace is always current
  int32_t n_chunks, batch, max_segs;
};

struct DecodeParams {
  const void* q;                 // [B][Hq][D] bf16
  void* const* pool_k_layers;    // device arrays of per-layer page bases; the kernel reads entry `layer`
  void* const* pool_v_layers;
  int32_t layer;
  const int32_t* block_tables;
  const void* tmaps;             // device array of CUtensorMap [n_layers][2] over the context's pool (TMA path)
  DecodePlan plan;
  const kam_patch_ref* patches;  // device array or nullptr
  int32_t* err;                  // device counter of malformed patch refs (kam_stats.device_errors)
  float* part_o;                 // [max_segs][R][Dv]
  float* part_lse;               // [max_segs][R]
  float sm_scale;
  void* out;                     // [B][Hq][Dv] bf16 (f32 when out_f32: a softmax STATE for a later cross-rank merge)
  float* lse;                    // [B][Hq]
  int32_t out_f32;
  int32_t plan_fresh;            // 1: the plan is written by the kernel just before this one on the stream (stateless call):
                                 // nothing of it may be read before griddepcontrol.wait
};

// merge of n_parts softmax states (o_p f32 [rows][Dv], lse_p f32 [rows]) of the same queries, e.g. one per rank of a
// chunk-parallel decode; the pointers may be peer memory.
constexpr int kMaxStateParts = 16;
struct StateMergeParams {
  const float* o[kMaxStateParts];
  const float* lse[kMaxStateParts];
  int32_t n_parts, rows, Dv;
  void* out;                     // [rows][Dv] bf16
  float* lse_out;                // [rows]
};
void launch_state_merge(const StateMergeParams& p, cudaStream_t st);

struct DecodeCsr {               // front end of the plan kernel for the stateless call (device metadata)
  const int32_t* chunk_starts;   // [B][max_chunks + 1]
  const long long* chunk_offsets;  // [B][max_chunks] or nullptr
  const int32_t* n_chunks;       // [B]
  int32_t max_chunks, max_pages;
  int32_t enabled;               // 0: plan.chunks / plan.rcb were uploaded by the host (window store)
  int32_t has_patches;           // patch index of chunk (b, c) = b * max_chunks + c
};

// KV heads per decode work unit (= compute warps per CTA): the largest divisor of n_kv_heads <= kDecMaxHG.
inline int decode_head_group(const kam_layout& L) {
  for (int h = L.n_kv_heads < kDecMaxHG ? L.n_kv_heads : kDecMaxHG; h >= 1; --h) if (L.n_kv_heads % h == 0) return h;
  return 1;
}
int decode_occupancy(const DecodeGeom& g);     // resident CTAs per SM of the decode kernel this geometry selects
void launch_decode_plan(const DecodeGeom& g, const DecodePlan& plan, const DecodeCsr& csr, cudaStream_t st);
// pdl: launch with programmatic stream serialization - the kernel's prologue (plan reads, barrier setup) overlaps the
// tail of the previous kernel on the stream; only legal when that kernel does not write the plan.
void launch_decode(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st);
void launch_decode_merge(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st);
// absorbed MLA decode (decode_mla_ts_kernel.cu: token-split mma.sync kernel, one CTA per SM): same plan, same partials, same merge
constexpr int kMlaHeads = 16;              // query heads per work unit (two 8-wide MMA n-tiles)
int mla_ts_smem_bytes(int kt);             // kt: rank tiles of the on-read patch the instantiation carries (0, 1, 2, 4)
void launch_mla_ts_decode(const DecodeGeom& g, const DecodeParams& p, bool pdl, cudaStream_t st);

// ---------------------------------------------------------------- multi-query readout (prefill_kernel.cu)
struct PrefillParams {
  const void* q;                 // [B][Tq][Hq][D] bf16
  void* out;                     // [B][Tq][Hq][D] bf16
  float* lse;                    // [B][Tq][Hq]
  void* const* pool_k_layers;    // device arrays of per-layer page bases
  void* const* pool_v_layers;
  const int32_t* block_tables;   // [B][max_pages]
  const int32_t* chunk_starts;   // [B][max_chunks + 1]
  const long long* chunk_offsets;  // [B][max_chunks] or nullptr
  const int32_t* n_chunks;       // [B]
  const double* inv_freq;        // [D / 2]
  int32_t layer, batch, Tq, Hq, H, G, P, P_shift, max_pages, max_chunks, causal, rope_style;
  float sm_scale;
  int32_t num_pages;             // pool pages: a token whose page index is >= max_pages or whose table entry lies outside
                                 // [0, num_pages) is never dereferenced - it reads as a zero row and is counted in *err
  int32_t* err;                  // device counter (kam_stats.device_errors)
};
void launch_prefill(const PrefillParams& p, int D, cudaStream_t st);        // mma.sync formulation (prefill_kernel.cu)
void launch_prefill_tc(const PrefillParams& p, int D, cudaStream_t st);     // tcgen05 / tensor-memory formulation (prefill_tc_kernel.cu)

// ---------------------------------------------------------------- form_patch (compile side, form_patch.cu)
struct FormPatchParams {
  const void* const* cond;       // device array [L] -> KV(B|A) rows [T][H][D] bf16, at the target position
  const void* const* solo;       // device array [L] -> canonical KV(B|0) rows [T][H][D] bf16
  void* const* U_out;            // device array [L] -> [T][H][m] bf16  (U_m S)
  void* const* W_out;            // device array [L] -> [H][m][D] bf16  (V_m^T)
  float* sigma_out;              // [L][H][m] or nullptr
  float* delta_ws;               // [L][H][T][D] fp32
  float* b_ws;                   // [L][H][T][b] fp32
  const double* inv_freq;        // [d_r / 2]
  long long delta;               // p_target - p_base
  int32_t L, H, T, D, m, b, ldq, n_iter;
  int32_t rope_off, d_r, rope_style, rotate;   // rotate = 0 for V
  int32_t smem_bytes;
};
void launch_form_patch(const FormPatchParams& p, cudaStream_t st);

}  // namespace kam

/* kamera.h - C ABI of libkamera: the serve-time hot path of Kamera's training-free KV-reuse operator
 * (arxiv/paper_2606_23581), hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations: P:NN = line NN of the paper text; R-n = reading n in DESIGN.md.
 *
 *   KV^(B|A) = R(delta) . KV(B|0) + U_m V_m^T                                           (Eq. 1)
 *
 * A cached, position-free chunk is relocated to any target offset by exact RoPE re-rotation (for MLA only
 * the decoupled rope band rotates), its stored rank-m conditioning patch is added to K and V per
 * layer and KV head, and the result is scattered into a paged KV pool through a block table (P:56,
 * P:195-204).  Chunks are admitted / evicted at either end of a window in O(1).  The same
 * operator is available fused-on-read inside a paged decode-attention kernel that merges per-chunk softmax
 * states by log-sum-exp.
 *
 * Conventions
 *  - "device" pointers are CUDA device memory owned by the CALLER (e.g. torch tensors); "host" pointers are
 *    ordinary host memory.  The library owns only kam_ctx and what hangs off it.
 *  - All device base pointers must be 16-byte aligned.
 *  - Every call that takes a `stream` (a cudaStream_t passed as void*; NULL = legacy default stream) enqueues
 *    its work on that stream and returns without synchronising.  Host bookkeeping (windows, free list) is
 *    applied immediately; device effects are stream-ordered.
 *  - A context serves ONE stream at a time: its staging buffers, descriptor rings, decode plans and partials are
 *    reused from call to call and ordered by that stream only.  Use one context per concurrently used stream.
 *  - Errors: every function returns a kam_status; nothing throws or aborts.  Arguments, window state and page
 *    supply are validated before any state changes, so a call that fails with INVALID_ARG / STATE / NO_PAGES /
 *    UNSUPPORTED leaves the context as it was.  KAM_ERR_CUDA reports a failure of the CUDA runtime itself (a
 *    launch, a copy): device state is then undefined as after any CUDA error, and the context should be
 *    destroyed.  kam_last_error() gives the reason.
 *  - There is no CPU fallback: without a CUDA device every compute entry returns KAM_ERR_CUDA.
 *  - The library never reads the process environment; what is tunable goes through kam_set_option.
 */
#ifndef KAMERA_H_
#define KAMERA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KAM_MAX_RANK   64    /* largest rank the paper uses: the rank-64 removal patch */
#define KAM_MAX_LAYERS 128

typedef struct kam_ctx kam_ctx;                       /* opaque; library-owned */

typedef enum { KAM_OK = 0, KAM_ERR_INVALID_ARG = 1, KAM_ERR_NO_PAGES = 2, KAM_ERR_UNSUPPORTED = 3,
               KAM_ERR_STATE = 4, KAM_ERR_CUDA = 5 } kam_status;
typedef enum { KAM_MHA = 0, KAM_GQA = 1, KAM_MLA = 2 } kam_layout_kind;
typedef enum { KAM_ROPE_HALF = 0, KAM_ROPE_INTERLEAVED = 1 } kam_rope_style;  /* pair (i, i+d/2) vs (2i, 2i+1); R-1 */
typedef enum { KAM_PATCH_TARGET_FRAME = 0, KAM_PATCH_CANONICAL_FRAME = 1 } kam_patch_frame; /* Eq. 1 order = 0; R-4 */
typedef enum { KAM_FRONT = 0, KAM_BACK = 1 } kam_end;
typedef enum { KAM_BF16 = 0, KAM_F32 = 1 } kam_dtype;

/* "layout = {MHA, GQA, MLA}" made explicit: one content | rope split covers all three (Fig. 2). */
typedef struct kam_layout {
  int32_t kind;            /* kam_layout_kind */
  int32_t n_layers;        /* <= KAM_MAX_LAYERS */
  int32_t n_q_heads;       /* multiple of n_kv_heads; query head hq reads KV head hq / (n_q_heads/n_kv_heads) (R-12) */
  int32_t n_kv_heads;      /* 1 for MLA */
  int32_t row_dim;         /* elements per token per KV head: head_dim; 576 for MLA (512 latent + 64 rope) */
  int32_t rope_off;        /* first rotated column of a row: 0 for MHA/GQA, 512 for MLA */
  int32_t rope_dim;        /* number of rotated columns (even): row_dim for MHA/GQA, 64 for MLA */
  int32_t has_v;           /* 1: separate V pool (MHA/GQA); 0: MLA, one latent+rope row per token */
  int32_t v_dim;           /* decode only, has_v == 0: a token's value = first v_dim columns of its row (512) */
  int32_t page_size;       /* tokens per page */
  int32_t rope_style;      /* kam_rope_style */
  int32_t elem_dtype;      /* kam_dtype of canonical chunks AND pool pages */
  int32_t factor_dtype;    /* kam_dtype of U and W */
  double  rope_theta;      /* f_i = theta^(-2i/rope_dim) (R-2) */
} kam_layout;

/* Paged KV pool.  k_layers / v_layers: DEVICE arrays [n_layers] of device base pointers; each layer is
 * [num_pages][page_size][n_kv_heads][row_dim] of elem_dtype (token-major pages, R-13).  v_layers NULL iff !has_v. */
typedef struct kam_pool {
  void *const *k_layers;
  void *const *v_layers;
  int32_t num_pages;
} kam_pool;

/* A position-free canonical chunk KV(B|0).  k_layers / v_layers: DEVICE arrays [n_layers] of
 * device pointers to [n_tokens][n_kv_heads][row_dim] rows.  p_base = the RoPE position token 0's key sits
 * at in this stored copy (0 for a chunk prefilled alone); relocation applies the uniform phase advance
 * delta = p_target - p_base to every token (R-3). */
typedef struct kam_chunk {
  const void *const *k_layers;
  const void *const *v_layers;     /* NULL iff !has_v */
  int32_t n_tokens;
  int64_t p_base;
} kam_chunk;

/* Rank-m patch factors {U_m S, V_m^T}: Delta ~= U W per layer and KV head.
 * Uk/Wk/Uv/Wv: DEVICE arrays [n_layers] of device pointers.
 *   U element (t, h, j) at  U[l] + t*u_token_stride + h*u_head_stride + j      (strides in elements;
 *     u_head_stride == 0 => one U shared by all KV heads, the paper's per-layer form, R-6)
 *   W[l] is [n_kv_heads][rank][row_dim], contiguous  (the paper's V_m^T).
 * rank_per_layer: HOST array [n_layers] or NULL (=> the call's `rank` everywhere); 0 => that layer gets the
 * rotation only (the deep-half variant). */
typedef struct kam_patch {
  const void *const *Uk, *const *Wk, *const *Uv, *const *Wv;     /* Uv/Wv NULL iff !has_v */
  int64_t u_token_stride, u_head_stride;
  const int32_t *rank_per_layer;
  int32_t frame;                   /* kam_patch_frame */
} kam_patch;

/* The argument tuple of kam_relocate_patch as a record, so that one launch covers many chunks. */
typedef struct kam_reloc_desc {
  const int32_t *block_table;      /* device */
  int64_t dst_token_start;
  const kam_chunk *chunk;          /* host struct */
  int64_t p_target;
  const kam_patch *patch;          /* host struct or NULL */
  int32_t rank;
} kam_reloc_desc;

/* One layer's factors of one (request, chunk), for patching on read inside the decode kernel (Eq. 1 applied to
 * the keys and values as they are read, the pool is never written).  Uk/Wk/Uv/Wv: device pointers to THIS layer's
 * U [T][..] (token t of the chunk = row t, strides as in kam_patch) and W [H][rank][row_dim]; bf16.  rank: 0 or all
 * pointers NULL => no patch for this chunk; otherwise a multiple of 16, <= the context's max patch rank
 * (kam_decode_set_max_patch_rank), u_token_stride and u_head_stride multiples of 8, pointers 16-byte aligned.
 * u_head_stride is either 0 (one U shared by all KV heads, R-6) or >= rank.  A ref that breaks these rules is ignored
 * by the kernel and counted in kam_stats.device_errors.  MLA (has_v == 0): Uv/Wv are not read - the value patch is the
 * first v_dim columns of the key patch. */
typedef struct kam_patch_ref {
  const void *Uk, *Wk, *Uv, *Wv;
  int64_t u_token_stride, u_head_stride;
  int32_t rank;
  int32_t frame;                   /* kam_patch_frame of the K patch: TARGET (Eq. 1) or CANONICAL (R-4) */
} kam_patch_ref;

typedef struct kam_stats {
  int64_t pages_free, pages_total;
  int64_t table_entries_written;   /* page-table entries written since kam_create (O(1)-per-op evidence) */
  int64_t chunks_live;
  int64_t kernels_launched;        /* CUDA kernels this context has launched since kam_create */
  int64_t device_errors;           /* malformed kam_patch_ref records the decode kernels ignored + block-table entries outside
                                      [0, num_pages) the relocate kernels skipped (reading it synchronises) */
  int64_t generic_launches;        /* of kernels_launched: launches of the element-wise fallback relocate kernel (fp32 tensors,
                                      row regions that are not multiples of 64 columns, U strides bulk copies cannot address);
                                      every bf16 rank in [0, KAM_MAX_RANK] runs on the tiled kernel */
} kam_stats;

/* ---- context -------------------------------------------------------------------------------------------------
 * pool == NULL creates a bookkeeping-only context: window calls update and export host state but launch nothing
 * (used to test the host logic without a GPU); its compute entries return KAM_ERR_CUDA.
 * max_requests / max_chunks_per_request / max_pages_per_chunk size the window store: page lists are kept per chunk
 * ([max_requests * max_chunks_per_request][max_pages_per_chunk] int32, host + device mirror), which is what makes an
 * admit / evict touch only that chunk's entries.  (SURVEY.md 8(b) sketched one max_pages_per_request; the
 * per-chunk table needs the two factors separately.) */
kam_status kam_create(const kam_layout *layout, const kam_pool *pool, int32_t max_requests,
                      int32_t max_chunks_per_request, int32_t max_pages_per_chunk, kam_ctx **out);
kam_status kam_destroy(kam_ctx *ctx);
const char *kam_last_error(const kam_ctx *ctx);     /* ctx may be NULL: error of this thread's last failed kam_create (or context-free call) */
const char *kam_version(void);
/* Tunables, per context; the defaults are the measured choices and nothing reads the environment.  Keys:
 *   reloc_stages 0..8 (0 = automatic)   reloc_head_group 0..4   reloc_head_group_cap 1..8   reloc_kv_split 0 never / 1 automatic / 2 always
 *   reloc_contig 0/1   reloc_row_blocks 0..4   reloc_evict_first 0/1   reloc_patch_cost_pct 50..200   reloc_pdl 0/1
 *   decode_ctas_per_sm 0..8   decode_boxes 0..16
 *   decode_pdl 0/1   decode_tma 0/1   prefill_tcgen05 0/1   host_copy_overlap 0/1   host_entries_sync 0/1
 * Setting any of them drops cached decode plans; CUDA graphs captured over this context's calls must be re-captured.
 * Errors: INVALID_ARG (unknown key, value out of range). */
kam_status kam_set_option(kam_ctx *ctx, const char *key, int64_t value);

/* ---- stateless operator: Eq. 1 written into the paged pool (`apply_reuse`) --------------------
 * For every layer l, token t, head h:
 *     k^ = R(p_target - p_base) k + U_k W_k ,  v^ = v + U_v W_v      (TARGET frame; CANONICAL adds U_k W_k first)
 *     g = dst_token_start + t ; page = block_table[g / P] ; pool[l][page][g % P][h][:] = round_to_elem(k^ / v^)
 * block_table: DEVICE int32[>= ceil((dst_token_start + n_tokens)/P)], logical page -> physical page.
 * dst_token_start need not be page aligned.  patch == NULL or rank == 0 => pure rotation (survivors).
 * p_target is a RoPE phase (any int64; M-RoPE positions are not sequence indices); dst_token_start is the
 * logical index inside the block table - two different things on purpose.
 * A block-table entry outside [0, pool->num_pages) is never dereferenced: its tokens are skipped and the entry is counted
 * once in kam_stats.device_errors.  rank: any value in [0, KAM_MAX_RANK] (ranks that are not multiples of 16 are padded
 * with zeros in shared memory, never in HBM).
 * layout: north_star's `layout = {MHA, GQA, MLA}` argument.  A context is created for ONE layout (kernel geometry, the
 * frequency table and the tensor maps hang off it), so this is a check, not a dispatch: NULL = the context's layout, else it
 * must equal it field by field (INVALID_ARG otherwise).
 * pool == NULL => the context's pool.  Errors: INVALID_ARG (null/misaligned pointers, rank < 0 or > KAM_MAX_RANK,
 * n_tokens < 0, dst_token_start + n_tokens > 2^31 - 1), UNSUPPORTED (layout the kernels do not cover), CUDA. */
kam_status kam_relocate_patch(kam_ctx *ctx, const kam_pool *pool, const int32_t *block_table,
                              int64_t dst_token_start, const kam_chunk *chunk, int64_t p_target,
                              const kam_patch *patch, int32_t rank, const kam_layout *layout, void *stream);
kam_status kam_relocate_patch_batch(kam_ctx *ctx, const kam_pool *pool, int32_t n,
                                    const kam_reloc_desc *descs /* host array [n] */, void *stream);

/* Survivors (P:26(ii)): rotate the rope band of K rows ALREADY in the pool, in place, by delta (may be
 * negative); V is not read.  Tokens [token_start, token_start + n_tokens) of block_table (device). */
kam_status kam_rotate_inplace(kam_ctx *ctx, const kam_pool *pool, const int32_t *block_table,
                              int64_t token_start, int32_t n_tokens, int64_t delta, void *stream);

/* Same operator with the canonical chunk and its factors in HOST memory (a chunk recalled from an off-device
 * canonical store): every k/v/U/W array is a HOST array [n_layers] of HOST pointers with the layouts above
 * (U contiguous [T][H][rank]).  The library copies them to device staging it owns (H2D on `stream`), then runs
 * kam_relocate_patch.  Pinned host memory makes the copies asynchronous.  Copies whose host source continues the previous
 * one are merged: a chunk kept as ONE slab in the order (per layer: K, V, U_k, W_k, U_v, W_v) crosses PCIe in one transfer.
 * By default the copies are enqueued on `stream` like everything else, so host arrays that earlier work on `stream` is still
 * filling (the D2H copy of an eviction to the host store, followed by its recall) are read in stream order.
 * Option host_copy_overlap = 1 (opt-in) moves the copies to a stream of the library's own and alternates two staging buffers, so
 * the transfer of one call overlaps the kernel of the previous one; the kernel still waits for its copies on `stream`.  That copy
 * stream is NOT ordered behind `stream`: with the option on, the CONTENTS of the host arrays must be final when the call is made
 * (written by the host, or by device work the caller has already synchronised with).
 * Either way the host arrays must stay valid until `stream` has passed this call. */
kam_status kam_relocate_patch_host(kam_ctx *ctx, const kam_pool *pool, const int32_t *block_table /* device */,
                                   int64_t dst_token_start, int32_t n_tokens, int64_t p_base, int64_t p_target,
                                   const void *const *k_host, const void *const *v_host,
                                   const void *const *Uk_host, const void *const *Wk_host,
                                   const void *const *Uv_host, const void *const *Wv_host,
                                   int32_t rank, int32_t frame, void *stream);

/* ---- compile side (P:189-193 `form_patch`; Eq. 2) -------------------------------------------------
 * Forms the rank-m patch of ONE chunk from its conditioned rows:  Delta = KV(B|A) - R(delta) KV(B|0) per layer and KV head,
 * top-m singular triplets, singular values folded into U (R-15):  U_out[l] [n_tokens][n_kv_heads][rank] = U_m S,
 * W_out[l] [n_kv_heads][rank][row_dim] = V_m^T (both bf16, contiguous), sigma_out [n_layers][n_kv_heads][rank] f32 or NULL.
 * kv_cond_layers / kv_solo_layers / U_out / W_out: DEVICE arrays [n_layers] of device pointers; rows [n_tokens][H][row_dim]
 * bf16.  is_key = 1: the solo rows are relocated by delta on their rope band first (TARGET frame, Eq. 1); is_key = 0
 * (values; or MLA with delta = 0): plain difference.  The conditioned forward that yields KV(B|A) is the caller's.
 * Method: block subspace iteration on Delta^T Delta with 8 columns of oversampling + Rayleigh-Ritz, n_iter sweeps (0 = 6);
 * exact for rank(Delta) <= rank + 8, otherwise the subspace error shrinks by (sigma_{m+9}/sigma_m)^2 per sweep.
 * What is unique - U W, the best rank-m approximation, and sigma - is what tests compare (signs of U, W columns are free).
 * Errors: INVALID_ARG, UNSUPPORTED (fp32 layouts; row_dim x rank too large for shared memory, e.g. MLA above rank 32), CUDA. */
kam_status kam_form_patch(kam_ctx *ctx, const void *const *kv_cond_layers, const void *const *kv_solo_layers,
                          int32_t n_tokens, int64_t delta, int32_t is_key, int32_t rank, int32_t n_iter,
                          void *const *U_out, void *const *W_out, float *sigma_out, void *stream);

/* ---- the window store as a deque (allocation policy R-13) ------------------------------------------
 * Per request: an ordered list of chunks; logical token order = list order; position of chunk i =
 * window_base + tokens before it.  Pages come from one LIFO free list (first pops give 0,1,2,...; admit pops in
 * logical order; evict pushes back in reverse logical order).  The first `n_front_chunks` pinned chunks (a text
 * prefix) are exempt from FRONT operations.  Chunk lengths must be positive multiples of page_size.
 *   kam_admit  takes pages, places the chunk at p_target = its position via Eq. 1 (relocate + patch into its pages).
 *   kam_evict  returns the chunk's pages.
 * Chunks whose position moved (FRONT ops): materialize = 1 rotates them in place now (delta = position - phase);
 * materialize = 0 touches nothing - the pending delta is applied on read by kam_window_decode.
 * kam_slide = kam_evict(evict_end, lazy) + kam_admit(admit_end, materialize) as ONE call and ONE kernel launch ("as the
 * oldest frame leaves, survivors re-rotate by the slide offset and a later recall rehydrates the dropped frame"): the
 * survivors' in-place rotations (by their NET displacement, rounded once) and the admitted chunk's Eq. 1 ride in the same
 * descriptor list.  kam_admit alone likewise launches once for its survivors and its chunk.  A slide whose admission cannot
 * succeed (pages, sizes) fails before anything is evicted.
 * Errors: INVALID_ARG, STATE (request not open / already open / window empty / too many chunks), NO_PAGES. */
kam_status kam_window_open(kam_ctx *ctx, int32_t req, int64_t window_base);
kam_status kam_window_pin(kam_ctx *ctx, int32_t req, int32_t n_front_chunks);
kam_status kam_window_close(kam_ctx *ctx, int32_t req);
kam_status kam_admit(kam_ctx *ctx, int32_t req, int32_t end /* kam_end */, const kam_chunk *chunk,
                     const kam_patch *patch, int32_t rank, int32_t materialize, int32_t *chunk_handle_out,
                     void *stream);
kam_status kam_evict(kam_ctx *ctx, int32_t req, int32_t end /* kam_end */, int32_t materialize, void *stream);
kam_status kam_slide(kam_ctx *ctx, int32_t req, int32_t evict_end /* kam_end */, int32_t admit_end /* kam_end */,
                     const kam_chunk *chunk, const kam_patch *patch, int32_t rank, int32_t materialize,
                     int32_t *chunk_handle_out, void *stream);
/* Linear host view of one request, for bit-exact checks.  Any output pointer may be NULL.  Capacities are in
 * entries; too small => INVALID_ARG.  chunk_cap counts the entries of EACH chunk array that is not NULL; chunk_starts_out gets
 * n_chunks + 1 entries, so with chunk_starts_out != NULL chunk_cap must be >= n_chunks + 1. */
kam_status kam_window_export(kam_ctx *ctx, int32_t req, int32_t *block_table_out, int32_t block_table_cap,
                             int64_t *slot_mapping_out, int64_t slot_mapping_cap, int32_t *chunk_starts_out,
                             int64_t *chunk_offsets_out, int32_t *chunk_handles_out, int32_t chunk_cap,
                             int32_t *n_pages_out, int32_t *n_chunks_out);
/* Host counters; device_errors is copied back from the device, so this call waits for the context's earlier work. */
kam_status kam_get_stats(kam_ctx *ctx, kam_stats *out);

/* ---- fused-on-read paged decode with LSE merge (R-12) -----------------------------------------------------
 * For request b, query head hq (KV head h = hq / G), over all chunks c of the request:
 *     k^_t = R(chunk_offsets[b][c]) k_t (+ U_k W_k)   v^_t = v_t (+ U_v W_v)          read from the pool, never written
 *     s_t = sm_scale * q . k^_t ;  per chunk (o_c, lse_c) ;  lse = ln sum_c e^{lse_c} ;  out = sum_c e^{lse_c - lse} o_c
 * q [batch][n_q_heads][row_dim] bf16 device, 16-byte aligned like out (q rows travel as bulk copies; else INVALID_ARG).
 * block_tables device int32 [batch][max_pages].  chunk_starts device
 * int32 [batch][max_chunks+1] (CSR token boundaries; only differences to chunk_starts[b][0] are used).
 * chunk_offsets device int64 [batch][max_chunks] (delta to apply on read; 0 if materialised) or NULL (= all 0).
 * n_chunks device int32 [batch].  patches: NULL, or device kam_patch_ref [batch][max_chunks]: the rank-m patch of Eq. 1
 * is applied ON READ in O(m) per token, s_t += sm_scale * U_k[t,:].(W_k q) and o += (sum_t p_t U_v[t,:]) W_v, which is
 * the same readout as attending over k_t + U_k W_k, v_t + U_v W_v (P:44 with Eq. 1 substituted).
 * out [batch][n_q_heads][Dv] bf16 (Dv = row_dim, or v_dim for MLA), lse [batch][n_q_heads] f32 (natural log, scale
 * inside).  A request with no tokens gives out = 0, lse = -inf.  Requires elem_dtype == KAM_BF16; head_dim 64 or 128 and at most
 * 16 query heads per KV head (MHA/GQA); MLA in absorbed form: row_dim 576 = 512 latent + 64 rope, v_dim 512, q rows of 576,
 * page_size % 16 == 0 (any number of query heads).  Otherwise KAM_ERR_UNSUPPORTED.
 * pool: NULL = the context's, or any pool of the context's layout.  Pool pages travel as TMA tensor-map boxes; the maps are
 * built per pool and cached (keyed by the pool's pointer-array addresses and page count): the FIRST decode call that names a
 * new pool reads its layer pointers back, which synchronises; a caller that re-fills a pointer array in place must pass it
 * under a new address. */
/* Largest rank a kam_patch_ref of later decode calls may carry: 16, 32 or 64 (default KAM_MAX_RANK).  The decode kernel
 * is specialised for it (shared memory and registers per tile grow with it), so a caller whose patches are all rank 16
 * should say so.  Errors: INVALID_ARG. */
kam_status kam_decode_set_max_patch_rank(kam_ctx *ctx, int32_t max_rank);
kam_status kam_paged_decode_merge(kam_ctx *ctx, const void *q, const kam_pool *pool, const int32_t *block_tables,
                                  int32_t max_pages, const int32_t *chunk_starts, const int64_t *chunk_offsets,
                                  const int32_t *n_chunks, int32_t max_chunks, const kam_patch_ref *patches,
                                  int32_t layer, int32_t batch, float sm_scale, void *out, float *lse, void *stream);
/* The work split of a decode call (which 16-token tiles each persistent CTA streams, each segment's first pool slot, the
 * per-chunk cos/sin rows) depends on the paging metadata only - not on the layer, the query or the factors.  By default
 * kam_paged_decode_merge rebuilds it on every call (one small kernel).  kam_paged_decode_plan builds it once and PINS it:
 * every later kam_paged_decode_merge / _state / _merge_host call on this context that names the same block_tables,
 * chunk_starts, chunk_offsets, n_chunks arrays, the same pool, max_pages, max_chunks, batch and the same `patches != NULL`
 * reuses the pinned plan (all layers of a decode step share one plan, as kam_window_decode's do).  The caller must call
 * kam_paged_decode_plan again when the CONTENT of those arrays changed; a call with different arrays or sizes rebuilds its own
 * plan and drops the pin; batch == 0 or block_tables == NULL just drops it. */
kam_status kam_paged_decode_plan(kam_ctx *ctx, const kam_pool *pool, const int32_t *block_tables, int32_t max_pages,
                                 const int32_t *chunk_starts, const int64_t *chunk_offsets, const int32_t *n_chunks,
                                 int32_t max_chunks, int32_t has_patches, int32_t batch, void *stream);
/* ---- the same readout for a BLOCK of query rows: chunked prefill over relocated chunks (the TTFT path of
 * P:105 / P:349: after `apply_reuse` has placed the recalled chunks, the appended text turn is prefilled over them).
 * q [batch][n_q_tokens][n_q_heads][row_dim] bf16 device (RoPE already applied at the rows' own positions), out the same shape,
 * lse [batch][n_q_tokens][n_q_heads] f32 (natural log, scale inside).  Paging arguments as kam_paged_decode_merge: the request's
 * cached tokens are the logical tokens [0, N_b) of its block-table row, cut into chunks by chunk_starts; chunk_offsets (or NULL)
 * are applied ON READ, by rotating the query block once per chunk (the pool is never written).
 *   causal = 0: every row sees all N_b cached tokens.
 *   causal = 1: the rows ARE the last n_q_tokens cached tokens (their keys and values were appended to the pool before this
 *               call): row t sees cached token j iff j <= N_b - n_q_tokens + t (reading R-19).  A row that sees nothing
 *               (n_q_tokens > N_b) gives out = 0, lse = -inf.
 * The per-chunk softmax states are merged in registers by the same log-sum-exp state merge as the decode, online.
 * No on-read patch here: on this path the patches were materialised by kam_relocate_patch / kam_admit.
 * Inconsistent paging metadata is never dereferenced: a cached token whose page index is >= max_pages or whose block-table entry
 * lies outside [0, pool->num_pages) reads as a zero key / value row and is counted (at least once) in kam_stats.device_errors.
 * Requires a bf16 MHA / GQA pool, head_dim 64 or 128 rotated over the whole head; else KAM_ERR_UNSUPPORTED.
 * Errors: INVALID_ARG, UNSUPPORTED, CUDA. */
kam_status kam_paged_prefill_merge(kam_ctx *ctx, const void *q, const kam_pool *pool, const int32_t *block_tables,
                                   int32_t max_pages, const int32_t *chunk_starts, const int64_t *chunk_offsets,
                                   const int32_t *n_chunks, int32_t max_chunks, int32_t layer, int32_t batch,
                                   int32_t n_q_tokens, int32_t causal, float sm_scale, void *out, float *lse, void *stream);
/* ---- chunk-parallel decode across GPUs ("the log-sum-exp state merge already used by ... ring/star
 * attention").  When a request's chunks are spread over several GPUs, each rank runs kam_paged_decode_state over the
 * chunks IT holds - same arguments as kam_paged_decode_merge, but the result is the softmax STATE in fp32:
 * o_state [batch][n_q_heads][Dv] (normalised readout over this rank's chunks), lse_state [batch][n_q_heads] (-inf if the
 * rank holds none of the request's tokens).  The states of all ranks are exchanged (one all-gather of (Dv + 1) floats per
 * query head, or peer-memory pointers) and kam_lse_merge_states applies the same merge over them in the fixed order
 * 0 .. n_parts-1:   lse = ln sum_p e^{lse_p},  out = sum_p e^{lse_p - lse} o_p   -> out bf16 [batch][n_q_heads][Dv], lse f32.
 * o_states / lse_states: HOST arrays [n_parts] of DEVICE pointers (they may point into peer GPUs' memory).
 * n_parts <= 16.  Errors: INVALID_ARG, CUDA. */
kam_status kam_paged_decode_state(kam_ctx *ctx, const void *q, const kam_pool *pool, const int32_t *block_tables,
                                  int32_t max_pages, const int32_t *chunk_starts, const int64_t *chunk_offsets,
                                  const int32_t *n_chunks, int32_t max_chunks, const kam_patch_ref *patches,
                                  int32_t layer, int32_t batch, float sm_scale, float *o_state, float *lse_state, void *stream);
kam_status kam_lse_merge_states(kam_ctx *ctx, int32_t n_parts, const float *const *o_states, const float *const *lse_states,
                                int32_t batch, void *out, float *lse, void *stream);
/* Same, over the context's own windows: request ids req_ids[0..batch) (host).  Pending lazy deltas are applied on read.
 * The work split of a step (which 16-token tiles each persistent CTA streams, the per-chunk cos/sin tables) depends on
 * the windows only, not on the layer: kam_window_plan builds it (one small H2D copy + one kernel); kam_window_decode
 * builds it itself when the windows or the request list changed since the last plan and otherwise launches exactly two
 * kernels (decode, merge) and nothing else - in that state it may be captured into a CUDA graph.  The window workspace is
 * laid out once for the largest plan the store can produce (max_requests x max_chunks_per_request chunks) and never moves,
 * and the kernels read the plan's sizes from it: a captured graph stays valid when the windows slide, grow or shrink (re-plan
 * eagerly, then replay).  It is tied, like any graph, to its q / out / lse pointers, its batch size and the options. */
kam_status kam_window_plan(kam_ctx *ctx, const int32_t *req_ids, int32_t batch, void *stream);
kam_status kam_window_decode(kam_ctx *ctx, const void *q, const int32_t *req_ids, int32_t batch, int32_t layer,
                             float sm_scale, void *out, float *lse, void *stream);
/* Same as kam_paged_decode_merge with q, out and lse in HOST memory: H2D of q, the kernels, D2H of out and lse, all enqueued on
 * `stream`; like every other entry it returns without synchronising - out_host / lse_host are valid once `stream` has passed
 * this call (one synchronise per decode step, not per layer).  Each layer has its own device staging, so the calls of a step do
 * not wait for each other.  Option host_entries_sync = 1 restores a cudaStreamSynchronize at the end of every call. */
kam_status kam_paged_decode_merge_host(kam_ctx *ctx, const void *q_host, const kam_pool *pool,
                                       const int32_t *block_tables, int32_t max_pages, const int32_t *chunk_starts,
                                       const int64_t *chunk_offsets, const int32_t *n_chunks, int32_t max_chunks,
                                       const kam_patch_ref *patches, int32_t layer, int32_t batch, float sm_scale,
                                       void *out_host, float *lse_host, void *stream);

/* ---- the fused decode for callers that must not allocate device memory (same readout as kam_paged_decode_merge) -----
 * Who needs this: every other decode entry hangs off a kam_ctx, and a context cudaMallocs - at kam_create (frequency table,
 * error counter, tensor maps) and again whenever a call needs a bigger plan / partials workspace or names a new pool.  Some
 * hosts cannot live with that: a serving engine that hands ALL free HBM to its own KV-pool / caching allocator at start-up (a
 * later cudaMalloc from a library then simply fails with out-of-memory), a plug-in loaded into a process whose memory budget
 * is enforced from outside, a latency-critical loop where cudaMalloc's implicit device-wide synchronisation is not
 * acceptable.  This ONE call needs no context and calls no cudaMalloc / cudaFree / cudaMallocAsync or any other allocating
 * routine, on its first use or later: its plan, its cos/sin tables, its frequency table and the per-segment softmax partials
 * live in a file-scope `static __device__` array of KAM_STATIC_SCRATCH_BYTES inside libkamera.so.
 * The cost: every GPU on which a process loads the library carries that array until the process exits, used or not.
 *
 * Arguments as kam_paged_decode_merge (q, block_tables, chunk_starts, chunk_offsets, n_chunks, out, lse: caller-owned DEVICE
 * memory, same shapes, same alignment rules), with the layout and the pool passed directly instead of through a context.
 * Restrictions: bf16 MHA / GQA pools with head_dim 64 or 128 and at most 16 query heads per KV head, rope_dim <= 256; no on-read
 * patch (materialise patches with kam_relocate_patch first); MLA is KAM_ERR_UNSUPPORTED (its kernel needs tensor maps, which
 * need device memory of their own).  Pool pages are fetched by per-token bulk copies (what option decode_tma = 0 selects on the
 * context path), so any page_size works; the arithmetic, the work split and the merge order are those of the context path.
 *
 * Size limit: the scratch a call needs grows with batch * max_chunks (about (444 + batch * max_chunks) * n_q_heads * (head_dim + 1)
 * * 4 bytes of partials for a 4-KV-head layout, plus the plan); a call that needs more than KAM_STATIC_SCRATCH_BYTES returns
 * KAM_ERR_INVALID_ARG with both figures in kam_last_error(NULL), and nothing is launched.  16 MiB covers BASELINE.json's
 * configs[1] decode step (32 requests x 9 chunks, 28 query heads, head_dim 128: about 11 MB).
 *
 * First call on a device: the library looks up the array's device address (cudaGetSymbolAddress with that device current,
 * once per device, cached).  That lookup may initialise the CUDA module, so make the first call on each device before any
 * stream capture is begun on it and outside any region that must not synchronise; later calls only launch kernels.
 * Sharing: there is ONE array per device, not one per stream or per caller.  Every call overwrites it and finds the previous
 * call's contents in it; the call itself re-writes what it reads (the plan is rebuilt every time, the error word and the frequency
 * table are reset by a small set-up kernel at the head of the call), so calls issued one after another on ONE stream are safe.  Two
 * calls that may run concurrently on the GPU - different streams, or different threads / contexts of one process on the same
 * device - race on the array and give garbage: serialise them (one stream, or an event between them).
 * Errors: INVALID_ARG (NULL / misaligned pointers, bad sizes, scratch limit), UNSUPPORTED (layout), CUDA.  The reason is read with
 * kam_last_error(NULL) (the slot kam_create's failures use: the calling thread's last context-free failure). */
#define KAM_STATIC_SCRATCH_BYTES (16u << 20)
kam_status kam_paged_decode_merge_static(const kam_layout *layout, const void *q, const kam_pool *pool,
                                         const int32_t *block_tables, int32_t max_pages, const int32_t *chunk_starts,
                                         const int64_t *chunk_offsets, const int32_t *n_chunks, int32_t max_chunks,
                                         int32_t layer, int32_t batch, float sm_scale, void *out, float *lse, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* KAMERA_H_ */

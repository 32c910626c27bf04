// Decode entry points: geometry, workspace, plan -> decode -> merge launches.  All arithmetic is in decode_kernel.cu.
#include <algorithm>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <mutex>
#include <vector>

#include "ctx.h"

using namespace kam;

namespace {

inline size_t align_up_sz(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Geometry of the decode kernel for this context's layout; `ctas_per_sm` = 0 picks the densest configuration that fits.
// kt: 16-wide rank tiles of the on-read patch the kernel is specialised for (0 = the call carries no patch refs).
kam_status decode_geom(kam_ctx* c, const kam_pool* pool, int kt, DecodeGeom* out, const void** tmaps_out) {
  const kam_layout& L = c->lay;
  // TMA tensor maps exist per pool (cached; the first call with a new pool reads its layer pointers back, which synchronises)
  const void* tmaps = c->opt.dec_tma ? tmaps_for_pool(c, pool) : nullptr;
  *tmaps_out = tmaps;
  const int variant = tmaps ? 1 : 0;
  if (c->dec_geom_ok[variant][kt]) { *out = c->dec_geom[variant][kt]; return KAM_OK; }
  if (L.elem_dtype != KAM_BF16) return fail(c, KAM_ERR_UNSUPPORTED, "decode needs a bf16 pool");
  if (!L.has_v) {
    // absorbed MLA decode: one latent+rope row per token, value = its first v_dim columns
    if (L.n_kv_heads != 1 || L.row_dim != 576 || L.v_dim != 512 || L.rope_off != 512 || L.rope_dim != 64)
      return fail(c, KAM_ERR_UNSUPPORTED, "MLA decode is built for rows of 512 latent + 64 rope columns with v_dim 512");
    if (!variant) return fail(c, KAM_ERR_UNSUPPORTED, "MLA decode needs TMA tensor maps over the pool: page_size %% 16 == 0, option decode_tma = 1 (%s)", c->tmap_why.c_str());
    // token-split kernel (decode_mla_ts_kernel.cu): one CTA per SM, 64-token iterations, the on-read patch rides in the ring
    DecodeGeom g{};
    g.mla = 1;
    g.Hq = L.n_q_heads; g.H = 1; g.D = 576; g.Dv = 512; g.P = L.page_size;
    g.G = std::min(L.n_q_heads, kMlaHeads);
    g.P_shift = -1;
    for (int s = 0; s < 31; ++s) if ((1 << s) == g.P) g.P_shift = s;
    g.HG = 1; g.n_hg = (L.n_q_heads + kMlaHeads - 1) / kMlaHeads; g.R = g.G; g.NT = 2;
    g.rope_off = L.rope_off; g.d_r = L.rope_dim; g.rope_style = L.rope_style;
    g.row_bytes = g.slice_bytes = 576 * 2; g.use_tma = 1; g.ncb = 9;
    g.kv_bytes = 2048 * g.ncb; g.box_bytes = g.kv_bytes; g.KT = kt;
    g.smem_bytes = mla_ts_smem_bytes(kt);
    g.n_ctas = c->sm_count;
    c->dec_geom[variant][kt] = g; c->dec_geom_ok[variant][kt] = true;
    *out = g;
    return KAM_OK;
  }
  if (L.row_dim != 64 && L.row_dim != 128) return fail(c, KAM_ERR_UNSUPPORTED, "decode supports head_dim 64 or 128");
  const int G = L.n_q_heads / L.n_kv_heads;
  if (G > 16) return fail(c, KAM_ERR_UNSUPPORTED, "decode supports up to 16 query heads per KV head");
  if (L.rope_style == KAM_ROPE_HALF && (L.rope_dim / 2) % 2) return fail(c, KAM_ERR_UNSUPPORTED, "rope_dim/2 must be even");
  DecodeGeom g{};
  g.Hq = L.n_q_heads; g.H = L.n_kv_heads; g.G = G; g.D = L.row_dim; g.Dv = L.row_dim; g.P = L.page_size;
  g.P_shift = -1;
  for (int s = 0; s < 31; ++s) if ((1 << s) == g.P) g.P_shift = s;
  g.HG = decode_head_group(L);
  g.n_hg = g.H / g.HG;
  g.R = g.HG * g.G;
  g.NT = (G + 7) / 8;
  g.rope_off = L.rope_off; g.d_r = L.rope_dim; g.rope_style = L.rope_style;
  g.row_bytes = g.H * g.D * 2; g.slice_bytes = g.HG * g.D * 2;
  g.use_tma = variant;
  g.ncb = g.HG * g.D / 64;
  g.s_row = g.slice_bytes + 16;                                   // (s_row / 16) odd: ldmatrix rows never share a bank group
  g.kv_bytes = g.use_tma ? 2048 * g.ncb : (int)align_up_sz((size_t)kDecTile * g.s_row, 128);
  g.box_bytes = g.kv_bytes;
  g.KT = kt;
  if (kt > 0) {                                                   // the U tile rides behind the K / V rows of its box
    g.u_off = g.kv_bytes;
    g.su_row = g.HG * kt * 16 * 2;
    if ((g.su_row / 16) % 2 == 0) g.su_row += 16;                 // (su_row / 16) odd: conflict-free ldmatrix over 8 token rows
    g.box_bytes = (int)align_up_sz((size_t)g.kv_bytes + (size_t)kDecTile * g.su_row, g.use_tma ? 1024 : 128);
  }
  g.off_hdr = 128; g.off_box0 = 1024;
  // CTAs per SM x ring depth: 3 CTAs with 2 K + 2 V boxes each when that fits, else fewer CTAs with a deeper ring
  const int sm_total = 227 * 1024;
  int want = c->opt.dec_ctas_per_sm > 0 ? c->opt.dec_ctas_per_sm : (kt > 0 ? 2 : 3);
  for (; want >= 1; --want) {
    const int budget = sm_total / want - 1024 - g.off_box0;
    int nb = std::min(8, budget / g.box_bytes) & ~1;
    if (c->opt.dec_boxes > 0) nb = std::min(nb, c->opt.dec_boxes & ~1);
    if (nb < 2) continue;
    if (nb < 4 && want > 1) continue;
    g.n_boxes = nb;
    g.smem_bytes = g.off_box0 + nb * g.box_bytes;
    if (decode_occupancy(g) >= want) break;
  }
  if (want < 1) return fail(c, KAM_ERR_UNSUPPORTED, "decode tile does not fit shared memory");
  g.n_ctas = c->sm_count * want;
  c->dec_geom[variant][kt] = g; c->dec_geom_ok[variant][kt] = true;
  *out = g;
  return KAM_OK;
}

// workspace layout: plan arrays first (chunks | rcb are what the window path uploads), then the partials
struct WsLayout { size_t chunks, rcb, dyn, tile_pre, seg_base, cta_seg, segs, cs, part_lse, part_o, total; int max_segs; };
WsLayout ws_layout(const DecodeGeom& g, int n_chunks, int batch) {
  WsLayout w{};
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up_sz(off + bytes, 256); return o; };
  w.max_segs = g.n_ctas + g.n_hg * n_chunks;
  w.chunks = take((size_t)n_chunks * sizeof(DecChunk));
  w.rcb = take((size_t)(batch + 1) * 4);
  w.dyn = take(16);
  w.tile_pre = take((size_t)(n_chunks + 1) * 4);
  w.seg_base = take(((size_t)g.n_hg * n_chunks + 1) * 4);
  w.cta_seg = take((size_t)(g.n_ctas + 1) * 4);
  w.segs = take((size_t)w.max_segs * sizeof(DecSeg));
  w.cs = take((size_t)n_chunks * std::max(1, g.d_r / 2) * sizeof(float2));
  w.part_lse = take((size_t)w.max_segs * g.R * 4);
  w.part_o = take((size_t)w.max_segs * g.R * g.Dv * 4);
  w.total = off;
  return w;
}

DecodePlan plan_of(kam_ctx* c, void* base, const WsLayout& w, int n_chunks, int batch) {
  char* ws = static_cast<char*>(base);
  DecodePlan pl{};
  pl.chunks = reinterpret_cast<DecChunk*>(ws + w.chunks);
  pl.rcb = reinterpret_cast<int32_t*>(ws + w.rcb);
  pl.dyn = reinterpret_cast<int32_t*>(ws + w.dyn);
  pl.tile_pre = reinterpret_cast<int32_t*>(ws + w.tile_pre);
  pl.seg_base = reinterpret_cast<int32_t*>(ws + w.seg_base);
  pl.cta_seg = reinterpret_cast<int32_t*>(ws + w.cta_seg);
  pl.segs = reinterpret_cast<DecSeg*>(ws + w.segs);
  pl.cs = reinterpret_cast<float2*>(ws + w.cs);
  pl.inv_freq = c->d_inv_freq;
  pl.block_tables = nullptr;                                      // set by the caller
  pl.n_chunks = n_chunks; pl.batch = batch; pl.max_segs = w.max_segs;
  return pl;
}

struct PlanKey {                 // what a stateless plan was built from (kam_paged_decode_plan)
  const void *bt, *starts, *offs, *nc, *pool_k;
  int32_t max_pages, max_chunks, batch, kt;
  bool operator==(const PlanKey& o) const {
    return bt == o.bt && starts == o.starts && offs == o.offs && nc == o.nc && pool_k == o.pool_k && max_pages == o.max_pages &&
           max_chunks == o.max_chunks && batch == o.batch && kt == o.kt;
  }
};
static_assert(sizeof(PlanKey) <= sizeof(((kam_ctx*)nullptr)->decplan_key), "plan key storage");

inline int patch_tiles(const kam_ctx* c, bool has_patches) {
  return has_patches ? (c->dec_max_rank <= 16 ? 1 : c->dec_max_rank <= 32 ? 2 : 4) : 0;
}

}  // namespace

// plan_only: build and pin the plan, launch nothing else.  q == NULL is only legal then.
static kam_status decode_stateless(kam_ctx* c, const void* q, const kam_pool* pool, const int32_t* block_tables,
                                   int32_t max_pages, const int32_t* chunk_starts, const int64_t* chunk_offsets,
                                   const int32_t* n_chunks, int32_t max_chunks, const kam_patch_ref* patches, bool has_patches,
                                   int32_t layer, int32_t batch, float sm_scale, void* out, float* lse, bool out_f32,
                                   bool plan_only, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  kam_status s = check_pool(c, &pool);
  if (s != KAM_OK) return s;
  if (!block_tables || !chunk_starts || !n_chunks) return fail(c, KAM_ERR_INVALID_ARG, "decode: NULL metadata argument");
  if (!plan_only) {
    if (!q || !out || !lse) return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge: NULL argument");
    if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(out)) & 15) return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge: q and out must be 16-byte aligned");
    if (layer < 0 || layer >= c->lay.n_layers) return fail(c, KAM_ERR_INVALID_ARG, "layer %d outside [0, %d)", layer, c->lay.n_layers);
  }
  if (batch < 0 || max_pages < 1 || max_chunks < 1) return fail(c, KAM_ERR_INVALID_ARG, "bad batch / max_pages / max_chunks");
  if (batch == 0) return KAM_OK;
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  if ((long long)batch * max_chunks > (1ll << 24)) return fail(c, KAM_ERR_UNSUPPORTED, "batch * max_chunks too large");
  DecodeGeom g; const void* tmaps = nullptr;
  const int kt = patch_tiles(c, has_patches);
  if ((s = decode_geom(c, pool, kt, &g, &tmaps)) != KAM_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  const int N = batch * max_chunks;
  const WsLayout w = ws_layout(g, N, batch);
  if (c->ws_cap < w.total) {
    c->decplan_valid = false;                                     // a pinned plan lives in the old buffer
    if ((s = grow_device(c, &c->d_ws, &c->ws_cap, w.total + w.total / 4, "cudaMalloc(decode workspace)", st)) != KAM_OK) return s;
  }
  // The plan depends on the paging metadata only, not on the layer or the query: a plan pinned by kam_paged_decode_plan is
  // reused by every call that names the same arrays and sizes (the caller re-plans when their CONTENT changes).
  PlanKey key{block_tables, chunk_starts, chunk_offsets, n_chunks, pool->k_layers, max_pages, max_chunks, batch, kt};
  const bool reuse = !plan_only && c->decplan_valid && key == *reinterpret_cast<const PlanKey*>(c->decplan_key);

  DecodeParams p{};
  p.q = q; p.pool_k_layers = pool->k_layers; p.pool_v_layers = pool->v_layers; p.layer = layer;
  p.block_tables = block_tables; p.tmaps = tmaps;
  p.plan = plan_of(c, c->d_ws, w, N, batch);
  p.plan.block_tables = block_tables;
  p.patches = patches; p.err = c->d_err;
  p.part_o = reinterpret_cast<float*>(static_cast<char*>(c->d_ws) + w.part_o);
  p.part_lse = reinterpret_cast<float*>(static_cast<char*>(c->d_ws) + w.part_lse);
  p.sm_scale = sm_scale; p.out = out; p.lse = lse; p.out_f32 = out_f32 ? 1 : 0;

  const bool pdl = c->opt.use_pdl != 0;
  if (!reuse) {
    DecodeCsr csr{};
    csr.chunk_starts = chunk_starts; csr.chunk_offsets = reinterpret_cast<const long long*>(chunk_offsets); csr.n_chunks = n_chunks;
    csr.max_chunks = max_chunks; csr.max_pages = max_pages; csr.enabled = 1; csr.has_patches = has_patches ? 1 : 0;
    launch_decode_plan(g, p.plan, csr, st);
    ++c->kernels_launched;
    c->decplan_valid = plan_only;
    if (plan_only) { memcpy(c->decplan_key, &key, sizeof key); c->decplan_unread = true; }
  }
  if (!plan_only) {
    // a plan written by the kernel just before this one: with programmatic dependent launch only the decode kernel's prologue
    // (barrier setup, shared-memory carve-up, launch latency) overlaps the plan kernel - plan_fresh makes it wait before the
    // first plan read.  A reused plan is older than anything on the stream that could still be writing it - except on the FIRST
    // decode behind kam_paged_decode_plan, whose plan kernel may be the launch right before this one and still running.
    p.plan_fresh = (reuse && !c->decplan_unread) ? 0 : 1;
    c->decplan_unread = false;
    if (g.mla) launch_mla_ts_decode(g, p, pdl, st);
    else launch_decode(g, p, pdl, st);
    launch_decode_merge(g, p, pdl, st);
    c->kernels_launched += 2;
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "decode launch");
  return KAM_OK;
}

extern "C" {

kam_status kam_paged_decode_plan(kam_ctx* c, const kam_pool* pool, const int32_t* block_tables, int32_t max_pages,
                                 const int32_t* chunk_starts, const int64_t* chunk_offsets, const int32_t* n_chunks,
                                 int32_t max_chunks, int32_t has_patches, int32_t batch, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  c->decplan_valid = false;
  if (batch == 0 || !block_tables) return KAM_OK;                  // release
  return decode_stateless(c, nullptr, pool, block_tables, max_pages, chunk_starts, chunk_offsets, n_chunks, max_chunks, nullptr,
                          has_patches != 0, 0, batch, 0.f, nullptr, nullptr, false, true, stream);
}

kam_status kam_paged_decode_merge(kam_ctx* c, const void* q, const kam_pool* pool, const int32_t* block_tables,
                                  int32_t max_pages, const int32_t* chunk_starts, const int64_t* chunk_offsets,
                                  const int32_t* n_chunks, int32_t max_chunks, const kam_patch_ref* patches, int32_t layer,
                                  int32_t batch, float sm_scale, void* out, float* lse, void* stream) {
  return decode_stateless(c, q, pool, block_tables, max_pages, chunk_starts, chunk_offsets, n_chunks, max_chunks, patches,
                          patches != nullptr, layer, batch, sm_scale, out, lse, false, false, stream);
}

kam_status kam_paged_decode_state(kam_ctx* c, const void* q, const kam_pool* pool, const int32_t* block_tables,
                                  int32_t max_pages, const int32_t* chunk_starts, const int64_t* chunk_offsets,
                                  const int32_t* n_chunks, int32_t max_chunks, const kam_patch_ref* patches, int32_t layer,
                                  int32_t batch, float sm_scale, float* o_state, float* lse_state, void* stream) {
  return decode_stateless(c, q, pool, block_tables, max_pages, chunk_starts, chunk_offsets, n_chunks, max_chunks, patches,
                          patches != nullptr, layer, batch, sm_scale, o_state, lse_state, true, false, stream);
}

kam_status kam_lse_merge_states(kam_ctx* c, int32_t n_parts, const float* const* o_states, const float* const* lse_states,
                                int32_t batch, void* out, float* lse, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (n_parts < 1 || n_parts > kMaxStateParts) return fail(c, KAM_ERR_INVALID_ARG, "n_parts outside [1, %d]", kMaxStateParts);
  if (!o_states || !lse_states || !out || !lse || batch < 0) return fail(c, KAM_ERR_INVALID_ARG, "kam_lse_merge_states: bad argument");
  for (int i = 0; i < n_parts; ++i)
    if (!o_states[i] || !lse_states[i]) return fail(c, KAM_ERR_INVALID_ARG, "kam_lse_merge_states: part %d is NULL", i);
  if (batch == 0) return KAM_OK;
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  StateMergeParams p{};
  for (int i = 0; i < n_parts; ++i) { p.o[i] = o_states[i]; p.lse[i] = lse_states[i]; }
  p.n_parts = n_parts; p.rows = batch * c->lay.n_q_heads; p.Dv = c->lay.has_v ? c->lay.row_dim : c->lay.v_dim;
  p.out = out; p.lse_out = lse;
  launch_state_merge(p, static_cast<cudaStream_t>(stream));
  ++c->kernels_launched;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "kam_state_merge_kernel launch");
  return KAM_OK;
}

}  // extern "C"

// The plan (segments, first slots, cos/sin tables) depends only on the windows, not on the layer or the query: it is
// rebuilt when a window changed (epoch) or the request list differs, and reused by every layer of the same step.
// The window path has a workspace of its own, laid out ONCE for the largest plan the window store can produce
// (max_requests x max_chunks_per_request chunks): the addresses a decode launch carries never depend on how many chunks the
// windows hold right now, so a CUDA graph captured over kam_window_decode stays valid while windows grow, shrink and slide.
static kam_status window_plan(kam_ctx* c, const int32_t* req_ids, int32_t batch, cudaStream_t st, DecodeGeom* g_out,
                              WsLayout* w_out, bool* was_cached) {
  if (!c->win) return fail(c, KAM_ERR_STATE, "context was created without a window store");
  if (!c->has_pool || !c->cuda_ok) return fail(c, KAM_ERR_CUDA, "window decode needs a context with a pool on a CUDA device");
  if (!req_ids || batch < 1 || batch > c->max_requests) return fail(c, KAM_ERR_INVALID_ARG, "window decode: bad request list");
  for (int b = 0; b < batch; ++b)
    if (!c->win->is_open(req_ids[b])) return fail(c, KAM_ERR_STATE, "request %d is not open", req_ids[b]);
  DecodeGeom g; const void* tmaps = nullptr;
  kam_status s = decode_geom(c, &c->pool, 0, &g, &tmaps);
  if (s != KAM_OK) return s;
  const bool cached = c->winplan_epoch == c->win->epoch() && c->winplan_reqs.size() == (size_t)batch &&
                      std::equal(c->winplan_reqs.begin(), c->winplan_reqs.end(), req_ids);
  const int n_max = c->max_requests * c->max_chunks;
  const WsLayout w = ws_layout(g, n_max, c->max_requests);
  *g_out = g; *w_out = w; *was_cached = cached;
  if (cached) return KAM_OK;
  // (re)allocation happens on the first plan only - or after kam_set_option changed the kernel's geometry, which invalidates
  // captured graphs anyway (kamera.h)
  if ((s = grow_device(c, &c->d_ws_win, &c->ws_win_cap, w.total, "cudaMalloc(window decode workspace)", st)) != KAM_OK) return s;
  int N = 0;
  for (int b = 0; b < batch; ++b) N += (int)c->win->chunks(req_ids[b]).size();
  // host -> device: the flat chunk list (pending lazy deltas become on-read rotations) and the request index
  const size_t up_bytes = w.rcb + (size_t)(batch + 1) * 4;
  Staging* sg;
  if ((s = staging_acquire(c, up_bytes, &sg)) != KAM_OK) return s;
  char* h = static_cast<char*>(sg->host);
  DecChunk* hc = reinterpret_cast<DecChunk*>(h + w.chunks);
  int32_t* hr = reinterpret_cast<int32_t*>(h + w.rcb);
  int j = 0;
  for (int b = 0; b < batch; ++b) {
    hr[b] = j;
    int64_t pos = c->win->window_base(req_ids[b]);
    for (const ChunkRec& r : c->win->chunks(req_ids[b])) {
      DecChunk ch{};
      ch.bt_off = (long long)r.slot * c->max_ppc; ch.delta = pos - r.phase;
      ch.b = b; ch.tok0 = 0; ch.n_tok = r.n_tokens; ch.patch = -1;
      hc[j++] = ch;
      pos += r.n_tokens;
    }
  }
  hr[batch] = j;
  // two copies: the chunk records are N entries, the request index sits at its fixed offset behind room for n_max of them
  cudaError_t e = cudaMemcpyAsync(c->d_ws_win, h, (size_t)N * sizeof(DecChunk), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(static_cast<char*>(c->d_ws_win) + w.rcb, h + w.rcb, (size_t)(batch + 1) * 4, cudaMemcpyHostToDevice, st);
  staging_release(sg, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(window plan)");
  DecodePlan pl = plan_of(c, c->d_ws_win, w, N, batch);
  pl.block_tables = c->d_slot_pages;
  DecodeCsr csr{};
  launch_decode_plan(g, pl, csr, st);
  ++c->kernels_launched;
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(c, e, "decode plan launch");
  c->winplan_unread = true;
  c->winplan_epoch = c->win->epoch();
  c->winplan_reqs.assign(req_ids, req_ids + batch);
  c->winplan_chunks = N;
  return KAM_OK;
}

extern "C" {

kam_status kam_decode_set_max_patch_rank(kam_ctx* c, int32_t max_rank) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (max_rank != 16 && max_rank != 32 && max_rank != 64) return fail(c, KAM_ERR_INVALID_ARG, "max patch rank must be 16, 32 or 64 (got %d)", max_rank);
  c->dec_max_rank = max_rank;
  c->decplan_valid = false;
  return KAM_OK;
}

kam_status kam_window_plan(kam_ctx* c, const int32_t* req_ids, int32_t batch, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (batch == 0) return KAM_OK;
  DecodeGeom g; WsLayout w; bool cached;
  return window_plan(c, req_ids, batch, static_cast<cudaStream_t>(stream), &g, &w, &cached);
}

kam_status kam_window_decode(kam_ctx* c, const void* q, const int32_t* req_ids, int32_t batch, int32_t layer, float sm_scale,
                             void* out, float* lse, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (batch == 0) return KAM_OK;
  if (!q || !out || !lse) return fail(c, KAM_ERR_INVALID_ARG, "kam_window_decode: NULL argument");
  if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(out)) & 15) return fail(c, KAM_ERR_INVALID_ARG, "kam_window_decode: q and out must be 16-byte aligned");
  if (layer < 0 || layer >= c->lay.n_layers) return fail(c, KAM_ERR_INVALID_ARG, "layer %d outside [0, %d)", layer, c->lay.n_layers);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DecodeGeom g; WsLayout w; bool cached;
  kam_status s = window_plan(c, req_ids, batch, st, &g, &w, &cached);
  if (s != KAM_OK) return s;
  DecodeParams p{};
  p.q = q; p.pool_k_layers = c->pool.k_layers; p.pool_v_layers = c->pool.v_layers; p.layer = layer;
  p.block_tables = c->d_slot_pages; p.tmaps = c->opt.dec_tma ? tmaps_for_pool(c, &c->pool) : nullptr;
  // the one plan size a kernel needs (the chunk count, in the merge) is read from the workspace (DecodePlan::dyn), so the
  // parameters a captured graph replays stay right when the windows change
  p.plan = plan_of(c, c->d_ws_win, w, c->winplan_chunks, batch);
  p.plan.block_tables = c->d_slot_pages;
  p.part_o = reinterpret_cast<float*>(static_cast<char*>(c->d_ws_win) + w.part_o);
  p.part_lse = reinterpret_cast<float*>(static_cast<char*>(c->d_ws_win) + w.part_lse);
  p.sm_scale = sm_scale; p.out = out; p.lse = lse; p.err = c->d_err;
  const bool pdl = c->opt.use_pdl != 0;
  // with a plan an earlier decode already ran on, the decode prologue may overlap whatever precedes it on the stream (it only reads
  // the plan).  The first decode behind a plan kernel - built by this call, or by kam_window_plan just before it - starts in plain
  // stream order: that kernel may be the launch right before this one and still writing the plan.
  const bool settled = cached && !c->winplan_unread;
  c->winplan_unread = false;
  if (g.mla) launch_mla_ts_decode(g, p, settled && pdl, st);
  else launch_decode(g, p, settled && pdl, st);
  launch_decode_merge(g, p, pdl, st);
  c->kernels_launched += 2;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "decode launch");
  return KAM_OK;
}

// The readout for a block of query rows: arithmetic in prefill_kernel.cu.
kam_status kam_paged_prefill_merge(kam_ctx* c, const void* q, const kam_pool* pool, const int32_t* block_tables, int32_t max_pages,
                                   const int32_t* chunk_starts, const int64_t* chunk_offsets, const int32_t* n_chunks,
                                   int32_t max_chunks, int32_t layer, int32_t batch, int32_t n_q_tokens, int32_t causal,
                                   float sm_scale, void* out, float* lse, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  kam_status s = check_pool(c, &pool);
  if (s != KAM_OK) return s;
  if (!q || !block_tables || !chunk_starts || !n_chunks || !out || !lse) return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_prefill_merge: NULL argument");
  if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(out)) & 15) return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_prefill_merge: q and out must be 16-byte aligned");
  const kam_layout& L = c->lay;
  if (layer < 0 || layer >= L.n_layers) return fail(c, KAM_ERR_INVALID_ARG, "layer %d outside [0, %d)", layer, L.n_layers);
  if (batch < 0 || n_q_tokens < 0 || max_pages < 1 || max_chunks < 1 || (causal != 0 && causal != 1))
    return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_prefill_merge: bad batch / n_q_tokens / max_pages / max_chunks / causal");
  if (batch > 65535 || L.n_kv_heads > 65535) return fail(c, KAM_ERR_UNSUPPORTED, "kam_paged_prefill_merge: batch or KV heads beyond 65535");
  if (batch == 0 || n_q_tokens == 0) return KAM_OK;
  if (L.elem_dtype != KAM_BF16 || !L.has_v || (L.row_dim != 64 && L.row_dim != 128) || L.rope_off != 0 || L.rope_dim != L.row_dim)
    return fail(c, KAM_ERR_UNSUPPORTED, "kam_paged_prefill_merge covers bf16 MHA / GQA pools with head_dim 64 or 128 rotated over the whole head");
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  PrefillParams p{};
  p.q = q; p.out = out; p.lse = lse; p.pool_k_layers = pool->k_layers; p.pool_v_layers = pool->v_layers;
  p.block_tables = block_tables; p.chunk_starts = chunk_starts; p.chunk_offsets = reinterpret_cast<const long long*>(chunk_offsets);
  p.n_chunks = n_chunks; p.inv_freq = c->d_inv_freq;
  p.layer = layer; p.batch = batch; p.Tq = n_q_tokens; p.Hq = L.n_q_heads; p.H = L.n_kv_heads; p.G = L.n_q_heads / L.n_kv_heads;
  p.P = L.page_size; p.P_shift = -1;
  for (int sft = 0; sft < 31; ++sft) if ((1 << sft) == p.P) p.P_shift = sft;
  p.max_pages = max_pages; p.max_chunks = max_chunks; p.causal = causal; p.rope_style = L.rope_style; p.sm_scale = sm_scale;
  p.num_pages = pool->num_pages; p.err = c->d_err;
  if (c->opt.prefill_tc && sm_scale > 0.f) launch_prefill_tc(p, L.row_dim, static_cast<cudaStream_t>(stream));
  else launch_prefill(p, L.row_dim, static_cast<cudaStream_t>(stream));
  ++c->kernels_launched;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "kam_paged_prefill_kernel launch");
  return KAM_OK;
}

kam_status kam_paged_decode_merge_host(kam_ctx* c, const void* q_host, const kam_pool* pool, const int32_t* block_tables,
                                       int32_t max_pages, const int32_t* chunk_starts, const int64_t* chunk_offsets,
                                       const int32_t* n_chunks, int32_t max_chunks, const kam_patch_ref* patches,
                                       int32_t layer, int32_t batch, float sm_scale, void* out_host, float* lse_host,
                                       void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (!q_host || !out_host || !lse_host) return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_host: NULL argument");
  if (batch < 0) return fail(c, KAM_ERR_INVALID_ARG, "negative batch");
  if (batch == 0) return KAM_OK;
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  const kam_layout& L = c->lay;
  const size_t qb = (size_t)batch * L.n_q_heads * L.row_dim * 2, lb = (size_t)batch * L.n_q_heads * 4;
  const size_t ob = L.has_v ? qb : (size_t)batch * L.n_q_heads * L.v_dim * 2;
  const size_t o_off = (qb + 255) & ~size_t(255), l_off = (o_off + ob + 255) & ~size_t(255);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // one staging region per layer (q | out | lse): the calls of a step do not wait for one another's D2H copies
  const size_t per = (l_off + lb + 255) & ~size_t(255);
  kam_status s = grow_device(c, &c->d_hstage2, &c->hstage2_cap, per * L.n_layers, "cudaMalloc(decode host staging)", st);
  if (s != KAM_OK) return s;
  char* d = static_cast<char*>(c->d_hstage2) + per * (layer >= 0 && layer < L.n_layers ? layer : 0);
  cudaError_t e = cudaMemcpyAsync(d, q_host, qb, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(q)");
  s = kam_paged_decode_merge(c, d, pool, block_tables, max_pages, chunk_starts, chunk_offsets, n_chunks, max_chunks, patches,
                             layer, batch, sm_scale, d + o_off, reinterpret_cast<float*>(d + l_off), stream);
  if (s != KAM_OK) return s;
  if ((e = cudaMemcpyAsync(out_host, d + o_off, ob, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(out)");
  if ((e = cudaMemcpyAsync(lse_host, d + l_off, lb, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(lse)");
  if (c->opt.host_sync && (e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
  return KAM_OK;
}

}  // extern "C"

// =====================================================================================================================
// kam_paged_decode_merge_static: the fused decode for callers that may not allocate device memory (kamera.h).
//
// Everything the decode needs beyond the caller's inputs and outputs - frequency table, plan, cos/sin rows, per-segment
// partials - is carved out of ONE file-scope device array.  In this file's HOST code the name `g_static_scratch` is only a
// handle for the runtime (handing it to a kernel as a pointer would pass a host address): the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current.  DEVICE code of this file (the set-up kernel below)
// names the array directly.
namespace {

constexpr size_t kStaticHdrBytes = 256;           // [0] int32: malformed-record counter the decode kernels may bump
constexpr int kStaticMaxFreq = 128;               // rope_dim <= 256
constexpr size_t kStaticFreqOff = kStaticHdrBytes;
constexpr size_t kStaticWsOff = 4096;             // plan | cos/sin | partials start here (ws_layout offsets are relative to it)
static_assert(kStaticFreqOff + kStaticMaxFreq * sizeof(double) <= kStaticWsOff, "header region");

static __device__ __align__(256) unsigned char g_static_scratch[KAM_STATIC_SCRATCH_BYTES];

struct StaticFreq { double f[kStaticMaxFreq]; int32_t n; };

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;                           // guards the two caches below (the entry may be called from several threads)
void* g_static_dev_ptr[kStaticMaxDevices] = {};   // device address of g_static_scratch, per device ordinal
struct StaticGeomCache { bool ok = false; int dev = -1; int sm_count = 0; kam_layout lay{}; DecodeGeom g{}; } g_static_geom;

}  // namespace

namespace kam {
// Head of every call: the array keeps whatever the previous call (any caller, any layout) left in it, so the two things the
// later kernels read without writing first are reset here - the error word to zero, the frequency table to this layout's.
__global__ void __launch_bounds__(kStaticMaxFreq) kam_static_setup_kernel(const __grid_constant__ StaticFreq t) {
  if (threadIdx.x == 0) *reinterpret_cast<int32_t*>(g_static_scratch) = 0;
  if (threadIdx.x < t.n) reinterpret_cast<double*>(g_static_scratch + kStaticFreqOff)[threadIdx.x] = t.f[threadIdx.x];
}
}  // namespace kam

extern "C" kam_status kam_paged_decode_merge_static(const kam_layout* layout, const void* q, const kam_pool* pool,
                                                    const int32_t* block_tables, int32_t max_pages, const int32_t* chunk_starts,
                                                    const int64_t* chunk_offsets, const int32_t* n_chunks, int32_t max_chunks,
                                                    int32_t layer, int32_t batch, float sm_scale, void* out, float* lse,
                                                    void* stream) {
  // ---- arguments (errors go to the context-free slot kam_last_error(NULL) reads)
  if (!layout || !pool) return fail(nullptr, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_static: layout / pool is NULL");
  const kam_layout& L = *layout;
  if (L.n_layers < 1 || L.n_layers > KAM_MAX_LAYERS || L.n_kv_heads < 1 || L.n_q_heads < 1 || L.n_q_heads % L.n_kv_heads ||
      L.page_size < 1 || L.rope_dim < 0 || L.rope_dim % 2 || L.rope_off < 0 || L.rope_off + L.rope_dim > L.row_dim ||
      (L.rope_style != KAM_ROPE_HALF && L.rope_style != KAM_ROPE_INTERLEAVED) || !(L.rope_theta > 0))
    return fail(nullptr, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_static: malformed layout");
  if (!L.has_v) return fail(nullptr, KAM_ERR_UNSUPPORTED, "kam_paged_decode_merge_static: MLA decode needs tensor maps in device memory; use a context");
  if (L.rope_dim / 2 > kStaticMaxFreq) return fail(nullptr, KAM_ERR_UNSUPPORTED, "kam_paged_decode_merge_static: rope_dim > %d", 2 * kStaticMaxFreq);
  if (!pool->k_layers || !pool->v_layers || pool->num_pages < 1) return fail(nullptr, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_static: bad pool");
  if (!q || !out || !lse || !block_tables || !chunk_starts || !n_chunks) return fail(nullptr, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_static: NULL argument");
  if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(out)) & 15) return fail(nullptr, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_static: q and out must be 16-byte aligned");
  if (layer < 0 || layer >= L.n_layers) return fail(nullptr, KAM_ERR_INVALID_ARG, "layer %d outside [0, %d)", layer, L.n_layers);
  if (batch < 0 || max_pages < 1 || max_chunks < 1) return fail(nullptr, KAM_ERR_INVALID_ARG, "bad batch / max_pages / max_chunks");
  if (batch == 0) return KAM_OK;
  if ((long long)batch * max_chunks > (1ll << 24)) return fail(nullptr, KAM_ERR_INVALID_ARG, "batch * max_chunks too large");

  // ---- once per device: where the array lives; per (device, layout): the kernel geometry.  No allocation in either.
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "no CUDA device: libkamera has no CPU fallback");
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(nullptr, KAM_ERR_UNSUPPORTED, "device ordinal %d beyond %d", dev, kStaticMaxDevices - 1);
  void* base = nullptr;
  DecodeGeom g;
  {
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_dev_ptr[dev]) {
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, g_static_scratch);        // the current device's copy of the array
      if (e != cudaSuccess || !ptr) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(static decode scratch)");
      g_static_dev_ptr[dev] = ptr;
    }
    base = g_static_dev_ptr[dev];
    if (!(g_static_geom.ok && g_static_geom.dev == dev && memcmp(&g_static_geom.lay, &L, sizeof L) == 0)) {
      // decode_geom wants a context for the layout, the options and the SM count: a host-only one on the stack, with the
      // tensor-map path switched off (maps would need device memory) - it owns nothing on the device
      kam_ctx tmp;
      tmp.lay = L; tmp.cuda_ok = true; tmp.opt.dec_tma = 0;
      if ((e = cudaDeviceGetAttribute(&tmp.sm_count, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
        return cuda_fail(nullptr, e, "cudaDeviceGetAttribute(SM count)");
      const void* tmaps = nullptr;
      const kam_status s = decode_geom(&tmp, pool, 0, &g, &tmaps);
      if (s != KAM_OK) return fail(nullptr, s, "kam_paged_decode_merge_static: %s", tmp.err.c_str());
      g_static_geom.ok = true; g_static_geom.dev = dev; g_static_geom.sm_count = tmp.sm_count; g_static_geom.lay = L; g_static_geom.g = g;
    }
    g = g_static_geom.g;
  }

  // ---- the size limit, checked before anything is launched
  const int N = batch * max_chunks;
  const WsLayout w = ws_layout(g, N, batch);
  if (kStaticWsOff + w.total > (size_t)KAM_STATIC_SCRATCH_BYTES)
    return fail(nullptr, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge_static: batch %d x max_chunks %d needs %zu bytes of scratch, the static array has %u "
                "(KAM_STATIC_SCRATCH_BYTES); split the batch or use a context", batch, max_chunks, kStaticWsOff + w.total, KAM_STATIC_SCRATCH_BYTES);

  cudaStream_t st = static_cast<cudaStream_t>(stream);
  char* ws = static_cast<char*>(base) + kStaticWsOff;
  StaticFreq fr{};
  fr.n = L.rope_dim / 2;
  for (int i = 0; i < fr.n; ++i) fr.f[i] = pow(L.rope_theta, -2.0 * (double)i / L.rope_dim);     // f_i as kam_create writes it (R-2)
  kam_static_setup_kernel<<<1, kStaticMaxFreq, 0, st>>>(fr);

  DecodeParams p{};
  p.q = q; p.pool_k_layers = pool->k_layers; p.pool_v_layers = pool->v_layers; p.layer = layer;
  p.block_tables = block_tables; p.tmaps = nullptr;
  {
    kam_ctx tmp;                                                   // plan_of only takes the frequency table from it
    tmp.d_inv_freq = reinterpret_cast<double*>(static_cast<char*>(base) + kStaticFreqOff);
    p.plan = plan_of(&tmp, ws, w, N, batch);
  }
  p.plan.block_tables = block_tables;
  p.patches = nullptr; p.err = static_cast<int32_t*>(base);
  p.part_o = reinterpret_cast<float*>(ws + w.part_o);
  p.part_lse = reinterpret_cast<float*>(ws + w.part_lse);
  p.sm_scale = sm_scale; p.out = out; p.lse = lse; p.out_f32 = 0;
  p.plan_fresh = 1;
  DecodeCsr csr{};
  csr.chunk_starts = chunk_starts; csr.chunk_offsets = reinterpret_cast<const long long*>(chunk_offsets); csr.n_chunks = n_chunks;
  csr.max_chunks = max_chunks; csr.max_pages = max_pages; csr.enabled = 1; csr.has_patches = 0;
  // plain stream order between the four kernels (no programmatic dependent launch): each one starts after the one before it has
  // finished writing the array
  launch_decode_plan(g, p.plan, csr, st);
  launch_decode(g, p, false, st);
  launch_decode_merge(g, p, false, st);
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(nullptr, e, "kam_paged_decode_merge_static launch");
  return KAM_OK;
}

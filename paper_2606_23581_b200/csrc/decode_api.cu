// Decode entry points: geometry, workspace, plan -> decode -> merge launches.  All arithmetic is in decode_kernel.cu.
#include <algorithm>
#include <cstring>
#include <vector>

#include "ctx.h"

using namespace kam;

namespace {

inline int align_up(int x, int a) { return (x + a - 1) / a * a; }

kam_status decode_geom(kam_ctx* c, const kam_pool* pool, DecodeGeom* out) {
  const kam_layout& L = c->lay;
  if (L.elem_dtype != KAM_BF16) return fail(c, KAM_ERR_UNSUPPORTED, "decode needs a bf16 pool");
  if (!L.has_v) return fail(c, KAM_ERR_UNSUPPORTED, "decode over an MLA latent pool is not built yet (SURVEY.md 8(f) f1)");
  if (L.row_dim != 64 && L.row_dim != 128) return fail(c, KAM_ERR_UNSUPPORTED, "decode supports head_dim 64 or 128");
  const int G = L.n_q_heads / L.n_kv_heads;
  if (G > 16) return fail(c, KAM_ERR_UNSUPPORTED, "decode supports up to 16 query heads per KV head");
  if (L.rope_style == KAM_ROPE_HALF && (L.rope_dim / 2) % 2) return fail(c, KAM_ERR_UNSUPPORTED, "rope_dim/2 must be even");
  DecodeGeom g{};
  g.Hq = L.n_q_heads; g.H = L.n_kv_heads; g.G = G; g.D = L.row_dim; g.Dv = L.row_dim; g.P = L.page_size;
  g.P_shift = -1;
  for (int s = 0; s < 31; ++s) if ((1 << s) == g.P) g.P_shift = s;
  g.HG = 1;
  for (int hgc = std::min(g.H, kDecMaxHG); hgc >= 1; --hgc) if (g.H % hgc == 0) { g.HG = hgc; break; }
  g.n_hg = g.H / g.HG;
  g.rope_off = L.rope_off; g.d_r = L.rope_dim; g.rope_style = L.rope_style; g.theta = L.rope_theta;
  g.row_bytes = g.H * g.D * 2; g.slice_bytes = g.HG * g.D * 2;
  g.use_tma = c->d_tmaps != nullptr && pool->k_layers == c->pool.k_layers && pool->v_layers == c->pool.v_layers;
  g.ncb = g.HG * g.D / 64; g.box_bytes = 2048 * g.ncb;
  g.s_row = g.slice_bytes + 16;                                   // (s_row / 16) odd: ldmatrix rows never share a bank group
  g.off_warp = 128;
  g.warp_bytes = align_up(std::max(1, g.d_r / 2) * 8, 128);
  if (g.use_tma) {                                                // two 16-token boxes for K, two for V, 1024-byte aligned
    g.st_k = 0; g.st_v = 2 * g.box_bytes; g.st_hdr = 4 * g.box_bytes;
    g.stage_bytes = align_up(g.st_hdr + 16, 1024);
    g.off_stage0 = align_up(g.off_warp + g.HG * g.warp_bytes, 1024);
  } else {
    g.st_k = 0; g.st_v = kDecTT * g.s_row; g.st_hdr = 2 * kDecTT * g.s_row;
    g.stage_bytes = align_up(g.st_hdr + 16, 128);
    g.off_stage0 = align_up(g.off_warp + g.HG * g.warp_bytes, 128);
  }
  g.n_stages = std::min(6, (220 * 1024 - g.off_stage0) / g.stage_bytes);
  if (g.n_stages < 2) return fail(c, KAM_ERR_UNSUPPORTED, "decode tile does not fit shared memory");
  g.smem_bytes = g.off_stage0 + g.n_stages * g.stage_bytes;
  *out = g;
  return KAM_OK;
}

// workspace layout in c->d_ws
struct WsLayout { size_t items, scalars, n_splits, part_lse, part_o, total; };
WsLayout ws_layout(const DecodeGeom& g, int batch, int max_splits) {
  WsLayout w{};
  size_t off = 0;
  w.items = off; off += (size_t)batch * max_splits * sizeof(DecodeItem); off = (off + 255) & ~size_t(255);
  w.scalars = off; off += 256;
  w.n_splits = off; off += (size_t)batch * 4; off = (off + 255) & ~size_t(255);
  w.part_lse = off; off += (size_t)batch * g.Hq * max_splits * 4; off = (off + 255) & ~size_t(255);
  w.part_o = off; off += (size_t)batch * g.Hq * max_splits * g.Dv * 4;
  w.total = off;
  return w;
}

int pick_split(const kam_ctx* c, const DecodeGeom& g, long long token_bound) {
  // aim at >= 16 work units per SM; splits are powers of two between 256 and 4096 tokens
  long long per = token_bound * g.n_hg / std::max(1, c->sm_count * 16);
  int s = 256;
  while (s < 4096 && s < per) s <<= 1;
  return s;
}

}  // namespace

extern "C" {

kam_status kam_paged_decode_merge(kam_ctx* c, const void* q, const kam_pool* pool, const int32_t* block_tables,
                                  int32_t max_pages, const int32_t* chunk_starts, const int64_t* chunk_offsets,
                                  const int32_t* n_chunks, int32_t max_chunks, const kam_patch_ref* patches, int32_t layer,
                                  int32_t batch, float sm_scale, void* out, float* lse, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  kam_status s = check_pool(c, &pool);
  if (s != KAM_OK) return s;
  if (!q || !block_tables || !chunk_starts || !n_chunks || !out || !lse) return fail(c, KAM_ERR_INVALID_ARG, "kam_paged_decode_merge: NULL argument");
  if (layer < 0 || layer >= c->lay.n_layers) return fail(c, KAM_ERR_INVALID_ARG, "layer %d outside [0, %d)", layer, c->lay.n_layers);
  if (batch < 0 || max_pages < 1 || max_chunks < 1) return fail(c, KAM_ERR_INVALID_ARG, "bad batch / max_pages / max_chunks");
  if (patches) return fail(c, KAM_ERR_UNSUPPORTED, "on-read patching is not built yet; materialise the patch with kam_relocate_patch");
  if (batch == 0) return KAM_OK;
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  DecodeGeom g;
  if ((s = decode_geom(c, pool, &g)) != KAM_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  g.split_tokens = pick_split(c, g, (long long)batch * max_pages * g.P);
  const int max_splits = max_chunks + (int)(((long long)max_pages * g.P + g.split_tokens - 1) / g.split_tokens);
  const WsLayout w = ws_layout(g, batch, max_splits);
  if ((s = grow_device(c, &c->d_ws, &c->ws_cap, w.total, "cudaMalloc(decode workspace)")) != KAM_OK) return s;
  char* ws = static_cast<char*>(c->d_ws);

  DecodeParams p{};
  p.q = q; p.pool_k_layers = pool->k_layers; p.pool_v_layers = pool->v_layers; p.layer = layer;
  p.block_tables = block_tables; p.tmaps = c->d_tmaps;
  p.items = reinterpret_cast<DecodeItem*>(ws + w.items);
  p.n_items = reinterpret_cast<int32_t*>(ws + w.scalars);
  p.work_counter = reinterpret_cast<int32_t*>(ws + w.scalars) + 1;
  p.patches = nullptr; p.max_chunks = max_chunks;
  p.part_o = reinterpret_cast<float*>(ws + w.part_o); p.part_lse = reinterpret_cast<float*>(ws + w.part_lse);
  p.n_splits = reinterpret_cast<int32_t*>(ws + w.n_splits); p.max_splits = max_splits;
  p.sm_scale = sm_scale; p.out = out; p.lse = lse; p.batch = batch;

  launch_decode_plan(chunk_starts, reinterpret_cast<const long long*>(chunk_offsets), n_chunks, max_chunks, max_pages, batch,
                     g.split_tokens, max_splits, reinterpret_cast<DecodeItem*>(ws + w.items),
                     reinterpret_cast<int32_t*>(ws + w.scalars), reinterpret_cast<int32_t*>(ws + w.n_splits),
                     reinterpret_cast<int32_t*>(ws + w.scalars) + 1, st);
  launch_decode(g, p, c->sm_count, st);
  launch_decode_merge(g, p, st);
  c->kernels_launched += 3;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "decode launch");
  return KAM_OK;
}

kam_status kam_window_decode(kam_ctx* c, const void* q, const int32_t* req_ids, int32_t batch, int32_t layer, float sm_scale,
                             void* out, float* lse, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (!c->win) return fail(c, KAM_ERR_STATE, "context was created without a window store");
  if (!c->has_pool || !c->cuda_ok) return fail(c, KAM_ERR_CUDA, "kam_window_decode needs a context with a pool on a CUDA device");
  if (!q || !req_ids || !out || !lse) return fail(c, KAM_ERR_INVALID_ARG, "kam_window_decode: NULL argument");
  if (layer < 0 || layer >= c->lay.n_layers) return fail(c, KAM_ERR_INVALID_ARG, "layer %d outside [0, %d)", layer, c->lay.n_layers);
  if (batch < 0) return fail(c, KAM_ERR_INVALID_ARG, "negative batch");
  for (int b = 0; b < batch; ++b)
    if (!c->win->is_open(req_ids[b])) return fail(c, KAM_ERR_STATE, "request %d is not open", req_ids[b]);
  if (batch == 0) return KAM_OK;
  DecodeGeom g;
  kam_status s = decode_geom(c, &c->pool, &g);
  if (s != KAM_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  long long tokens = 0;
  for (int b = 0; b < batch; ++b) for (const ChunkRec& r : c->win->chunks(req_ids[b])) tokens += r.n_tokens;
  g.split_tokens = pick_split(c, g, tokens);
  // the host knows its own windows: the split list is built here (pending lazy deltas become on-read rotations)
  std::vector<DecodeItem> items;
  std::vector<int32_t> n_splits(batch);
  int max_splits = 1;
  for (int b = 0; b < batch; ++b) {
    int64_t pos = c->win->window_base(req_ids[b]);
    int sp = 0;
    for (const ChunkRec& r : c->win->chunks(req_ids[b])) {
      for (int o = 0; o < r.n_tokens; o += g.split_tokens) {
        DecodeItem it{};
        it.bt_off = (long long)r.slot * c->max_ppc; it.delta = pos - r.phase;
        it.b = b; it.chunk = 0; it.tok0 = o; it.n_tok = std::min(g.split_tokens, r.n_tokens - o); it.split = sp++; it.ctok0 = o;
        items.push_back(it);
      }
      pos += r.n_tokens;
    }
    n_splits[b] = sp;
    max_splits = std::max(max_splits, sp);
  }
  const WsLayout w = ws_layout(g, batch, max_splits);
  if ((s = grow_device(c, &c->d_ws, &c->ws_cap, w.total, "cudaMalloc(decode workspace)")) != KAM_OK) return s;
  char* ws = static_cast<char*>(c->d_ws);
  // plan -> staging -> workspace (items | scalars | n_splits are contiguous at the front of the layout)
  const size_t plan_bytes = w.n_splits + (size_t)batch * 4;
  Staging* sg;
  if ((s = staging_acquire(c, plan_bytes, &sg)) != KAM_OK) return s;
  char* h = static_cast<char*>(sg->host);
  memset(h, 0, plan_bytes);
  if (!items.empty()) memcpy(h + w.items, items.data(), items.size() * sizeof(DecodeItem));
  reinterpret_cast<int32_t*>(h + w.scalars)[0] = (int32_t)items.size();
  reinterpret_cast<int32_t*>(h + w.scalars)[1] = 0;
  memcpy(h + w.n_splits, n_splits.data(), (size_t)batch * 4);
  cudaError_t e = cudaMemcpyAsync(ws, h, plan_bytes, cudaMemcpyHostToDevice, st);
  staging_release(sg, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(window plan)");

  DecodeParams p{};
  p.q = q; p.pool_k_layers = c->pool.k_layers; p.pool_v_layers = c->pool.v_layers; p.layer = layer;
  p.block_tables = c->d_slot_pages; p.tmaps = c->d_tmaps;
  p.items = reinterpret_cast<DecodeItem*>(ws + w.items);
  p.n_items = reinterpret_cast<int32_t*>(ws + w.scalars);
  p.work_counter = reinterpret_cast<int32_t*>(ws + w.scalars) + 1;
  p.part_o = reinterpret_cast<float*>(ws + w.part_o); p.part_lse = reinterpret_cast<float*>(ws + w.part_lse);
  p.n_splits = reinterpret_cast<int32_t*>(ws + w.n_splits); p.max_splits = max_splits;
  p.sm_scale = sm_scale; p.out = out; p.lse = lse; p.batch = batch;
  launch_decode(g, p, c->sm_count, st);
  launch_decode_merge(g, p, st);
  c->kernels_launched += 2;
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "decode launch");
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
  const size_t qb = (size_t)batch * L.n_q_heads * L.row_dim * 2, ob = qb, lb = (size_t)batch * L.n_q_heads * 4;
  const size_t o_off = (qb + 255) & ~size_t(255), l_off = (o_off + ob + 255) & ~size_t(255);
  kam_status s = grow_device(c, &c->d_hstage2, &c->hstage2_cap, l_off + lb, "cudaMalloc(decode host staging)");
  if (s != KAM_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  char* d = static_cast<char*>(c->d_hstage2);
  cudaError_t e = cudaMemcpyAsync(d, q_host, qb, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(q)");
  s = kam_paged_decode_merge(c, d, pool, block_tables, max_pages, chunk_starts, chunk_offsets, n_chunks, max_chunks, patches,
                             layer, batch, sm_scale, d + o_off, reinterpret_cast<float*>(d + l_off), stream);
  if (s != KAM_OK) return s;
  if ((e = cudaMemcpyAsync(out_host, d + o_off, ob, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(out)");
  if ((e = cudaMemcpyAsync(lse_host, d + l_off, lb, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(lse)");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
  return KAM_OK;
}

}  // extern "C"

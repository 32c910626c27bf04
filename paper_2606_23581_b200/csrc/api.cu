// libkamera C entry points: argument validation, host bookkeeping, descriptor staging, kernel launches.
// Every step of the hot path runs in the kernels (relocate_kernel.cu, decode_kernel.cu); this file only decides
// geometry and marshals descriptors.  No CPU fallback exists: without CUDA every compute entry fails.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <memory>
#include <new>
#include <string>
#include <vector>

#include "ctx.h"

using namespace kam;

namespace { thread_local std::string g_create_error; }

namespace kam {

kam_status fail(kam_ctx* ctx, kam_status st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf; else g_create_error = buf;
  return st;
}

kam_status cuda_fail(kam_ctx* ctx, cudaError_t e, const char* what) {
  return fail(ctx, KAM_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

// Grows a library-owned device buffer.  The outgrown buffer may still be read by work already enqueued, and cudaFree would
// synchronise the whole device inside a call documented to return without synchronising: it is parked and freed by
// kam_destroy.  Capacities grow geometrically, so the parked buffers add up to less than the live one.
kam_status grow_device(kam_ctx* c, void** buf, size_t* cap, size_t bytes, const char* what, cudaStream_t) {
  if (*cap >= bytes) return KAM_OK;
  void* fresh = nullptr;
  const size_t want = std::max(bytes, *cap + *cap / 2);
  cudaError_t e = cudaMalloc(&fresh, want);
  if (e != cudaSuccess) return cuda_fail(c, e, what);
  if (*buf) c->graveyard.push_back(*buf);
  *buf = fresh; *cap = want;
  return KAM_OK;
}

}  // namespace kam

namespace {

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline int align_up(int x, int a) { return (x + a - 1) / a * a; }

// ---- column blocks of one KV head's row (what one consumer warp processes per 16 tokens) -----------------------
bool build_head_blocks(kam_ctx* c) {
  const kam_layout& L = c->lay;
  c->blocks_per_head = 0;
  if (L.elem_dtype != KAM_BF16 || L.factor_dtype != KAM_BF16) { c->fast_layout_why = "tiled kernel needs bf16 elements and factors"; return false; }
  const int pre = L.rope_off, band = L.rope_dim, post = L.row_dim - L.rope_off - L.rope_dim;
  if (pre % 64 || band % 64 || post % 64) { c->fast_layout_why = "row regions must be multiples of 64 columns"; return false; }
  if (L.rope_style == KAM_ROPE_HALF && band > 128) { c->fast_layout_why = "HALF rope band wider than 128 columns"; return false; }
  int n = 0;
  auto add_plain = [&](int start, int len, bool rope) {
    for (int off = 0; off < len;) {
      const int w = std::min(128, len - off);
      if (n >= kMaxColBlocks) return false;
      ColBlock b{};
      b.col_off = (int16_t)(start + off); b.w_col_off = (int16_t)(start + off);
      b.band_col0 = (int16_t)(rope ? off : 0); b.n_groups = (int8_t)(w / 32); b.rope = rope; b.fhead = 0;
      c->head_blocks[n++] = b;
      off += w;
    }
    return true;
  };
  if (!add_plain(0, pre, false)) return false;
  if (band) {
    if (L.rope_style == KAM_ROPE_HALF) {
      ColBlock b{};
      b.col_off = (int16_t)pre; b.w_col_off = (int16_t)pre; b.band_col0 = 0; b.n_groups = (int8_t)(band / 32); b.rope = 1;
      c->head_blocks[n++] = b;
    } else if (!add_plain(pre, band, true)) return false;
  }
  if (!add_plain(pre + band, post, false)) return false;
  c->blocks_per_head = n;
  return true;
}

// Shared-memory geometry of the tiled kernel for a call whose largest rank is max_rank.  Candidates, best first:
// whole-row slices (one copy per tile) with three stages; if the resident W_k + W_v leave no room for that (ranks 48 / 64:
// 139 KB for four heads of 128 columns), the kv-split form - a tile carries K rows or V rows, so only one of the two W tables
// is resident and three 48 KB stages fit again; last, fewer heads per slice or two big stages (the round-1 geometry).
bool build_reloc_geom(const kam_ctx* c, int max_rank, bool inplace_only, RelocGeom* out, std::string* why) {
  const kam_layout& L = c->lay;
  RelocGeom g{};
  g.L = L.n_layers; g.H = L.n_kv_heads; g.D = L.row_dim; g.P = L.page_size;
  g.row_bytes = g.H * g.D * 2;
  g.P_shift = -1;
  for (int sft = 0; sft < 31; ++sft) if ((1 << sft) == g.P) g.P_shift = sft;
  g.nkv = (L.has_v && !inplace_only) ? 2 : 1;       // survivors are rotated in place: K only, V is never staged
  g.KT_max = (max_rank + 15) / 16;
  const int m_pad = g.KT_max * 16;                  // ranks are padded to a multiple of 16 in shared memory only
  g.rope_style = L.rope_style; g.d_r = L.rope_dim; g.half_groups = L.rope_dim / 64;
  g.theta = L.rope_theta;
  const int limit = 226 * 1024;
  const int ns_max = c->opt.reloc_stages > 0 ? c->opt.reloc_stages : 3;   // measured on B200: 3 x 37 KB in flight per SM beats 4 and 5
  const int hg_force = c->opt.reloc_hg;                                   // kam_set_option("reloc_head_group")
  // one candidate: `HG` heads per slice, plain or kv-split; fills *t with the deepest pipeline (<= ns_max stages) that fits
  auto candidate = [&](bool split, int HG, RelocGeom* out_t) -> bool {
    if (g.H % HG) return false;
    const int NB = HG * c->blocks_per_head;
    if (NB > kMaxColBlocks) return false;
    RelocGeom t = g;
    t.kv_split = split ? 1 : 0;
    const int nkv_tile = split ? 1 : g.nkv;           // row sets (K, V) a tile holds
    t.HG = HG; t.n_hg = g.H / HG; t.n_blocks = NB;
    t.slice_bytes = HG * g.D * 2;
    t.contig = (HG == g.H) && c->opt.reloc_contig;
    // padded rows (== 64 mod 128) make the 128-bit row loads conflict-free; unpadded rows allow one copy per tile
    t.s_row = t.contig ? t.slice_bytes : t.slice_bytes + ((64 - t.slice_bytes % 128) + 128) % 128;
    t.su_row = g.KT_max ? align_up(HG * max_rank * 2, 32) + 16 : 0;          // (su_row / 16) odd: conflict-free ldmatrix over 8 token rows
    t.RB = std::min(4, std::max(1, (kRelocConsumerWarps + nkv_tile * NB - 1) / (nkv_tile * NB)));
    if (c->opt.reloc_rb > 0) t.RB = std::min(4, c->opt.reloc_rb);
    t.TT = 16 * t.RB;
    t.st_k = 0;
    t.st_v = t.st_k + t.TT * t.s_row;
    t.st_uk = t.st_v + (nkv_tile == 2 ? t.TT * t.s_row : 0);
    t.st_uv = t.st_uk + t.TT * t.su_row;
    t.st_slot = t.st_uv + (nkv_tile == 2 ? t.TT * t.su_row : 0);
    t.stage_bytes = align_up(t.st_slot + 2 * t.TT * 4, 128);                     // slots: 2 TT (the in-place x2 tile form)
    t.w_row = (g.D + 8) * 2;
    t.w_kv_stride = HG * m_pad * t.w_row;
    t.off_tab = 128;
    t.off_cs = t.off_tab + align_up(2 * t.RB * NB * 16, 128);                    // slab table: one int4 per slab
    t.off_w = t.off_cs + align_up(std::max(1, g.d_r / 2) * 12, 128);               // c | s | -s, planar fp32
    t.off_stage0 = align_up(t.off_w + nkv_tile * t.w_kv_stride, 128);
    for (int i = 0; i < NB; ++i) {
      ColBlock b = c->head_blocks[i % c->blocks_per_head];
      const int h = i / c->blocks_per_head;
      b.fhead = (int8_t)h; b.col_off = (int16_t)(b.col_off + h * g.D);
      t.blk[i] = b;
    }
    t.load_hint = c->opt.reloc_load_hint;
    for (int NS = ns_max; NS >= 2; --NS) {
      t.n_stages = NS;
      t.smem_bytes = t.off_stage0 + NS * t.stage_bytes;
      if (t.smem_bytes <= limit) { *out_t = t; return true; }
    }
    return false;
  };
  // widest slice tried first: up to 8 heads (a whole 8-head row is one contiguous copy per tile; with W of 8 heads only the
  // kv-split form leaves room for three stages), else the largest divisor of H up to 4
  const int hg_cap = c->opt.reloc_hg_cap;
  int hg_max = 1;
  for (int HG = std::min(g.H, hg_cap); HG >= 1; --HG) if (g.H % HG == 0 && HG * c->blocks_per_head <= kMaxColBlocks) { hg_max = HG; break; }
  const bool may_split = g.nkv == 2 && c->opt.reloc_kv_split != 0, must_split = g.nkv == 2 && c->opt.reloc_kv_split == 2;
  RelocGeom t{};
  if (hg_force > 0) {
    if (candidate(must_split, hg_force, &t)) { *out = t; return true; }
    *why = "forced head group does not fit";
    return false;
  }
  // 1. the widest slice with three stages, plain; 2. the same, kv-split
  for (int HG = hg_max; HG >= std::min(hg_max, 4); --HG) {
    if (g.H % HG) continue;
    if (!must_split && candidate(false, HG, &t) && t.n_stages >= 3) { *out = t; return true; }
    if (may_split && candidate(true, HG, &t) && (t.n_stages >= 3 || must_split)) { *out = t; return true; }
  }
  hg_max = std::min(hg_max, 4);
  // 3. round 1's order: narrower slices, three stages or two big ones (>= 96 KB in flight: measured at rank 64 before the
  //    kv-split form existed - two 54 KB stages of two heads 4.9 TB/s, three 60 KB stages of one-head slices 4.0 TB/s)
  RelocGeom best{}; bool have = false;
  for (int pass = must_split ? 1 : 0; pass < (may_split ? 2 : 1); ++pass)
    for (int HG = hg_max; HG >= 1; --HG) {
      if (!candidate(pass == 1, HG, &t)) continue;
      if (t.n_stages >= 3 || t.n_stages * t.stage_bytes >= 96 * 1024) { *out = t; return true; }
      if (!have) { best = t; have = true; }
    }
  if (have) { *out = best; return true; }
  *why = "no shared-memory configuration fits";
  return false;
}

}  // namespace

namespace kam {
// ---- staging ---------------------------------------------------------------------------------------------------
kam_status staging_acquire(kam_ctx* c, size_t bytes, Staging** out) {
  Staging& s = c->staging[c->staging_next];
  c->staging_next = (c->staging_next + 1) % kStagingSlots;
  cudaError_t e;
  if (s.in_flight) {
    if ((e = cudaEventSynchronize(s.ev)) != cudaSuccess) return cuda_fail(c, e, "cudaEventSynchronize(staging)");
    s.in_flight = false;
  }
  if (!s.ev && (e = cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming)) != cudaSuccess)
    return cuda_fail(c, e, "cudaEventCreate");
  if (s.cap < bytes) {
    if (s.host) cudaFreeHost(s.host);
    if (s.dev) cudaFree(s.dev);
    s.host = s.dev = nullptr; s.cap = 0;
    const size_t cap = std::max<size_t>(bytes * 2, 64 * 1024);
    if ((e = cudaMallocHost(&s.host, cap)) != cudaSuccess) return cuda_fail(c, e, "cudaMallocHost(staging)");
    if ((e = cudaMalloc(&s.dev, cap)) != cudaSuccess) return cuda_fail(c, e, "cudaMalloc(staging)");
    s.cap = cap;
  }
  *out = &s;
  return KAM_OK;
}
kam_status staging_commit(kam_ctx* c, Staging* s, size_t bytes, cudaStream_t st) {
  cudaError_t e = cudaMemcpyAsync(s->dev, s->host, bytes, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(staging)");
  return KAM_OK;
}
void staging_release(Staging* s, cudaStream_t st) {
  if (cudaEventRecord(s->ev, st) == cudaSuccess) s->in_flight = true;
}

kam_status check_pool(kam_ctx* c, const kam_pool** pool) {
  if (*pool == nullptr) {
    if (!c->has_pool) return fail(c, KAM_ERR_INVALID_ARG, "no pool given and the context has none");
    *pool = &c->pool;
  }
  if ((*pool)->k_layers == nullptr || (c->lay.has_v && (*pool)->v_layers == nullptr))
    return fail(c, KAM_ERR_INVALID_ARG, "pool layer-pointer arrays must not be NULL");
  return KAM_OK;
}
}  // namespace kam

namespace {

// ---- relocate core -----------------------------------------------------------------------------------------------
struct HostReloc {
  const int32_t* bt; int64_t dst0, delta;
  const void* const* k; const void* const* v;
  const kam_patch* patch; int32_t rank; int32_t n_tokens; int32_t flags;
};
// The page list of a chunk being admitted to a window (descriptor `desc` of the call): host copy in a staging slot, device
// mirror row.  The tiled kernel takes it in its parameters; otherwise it is copied to the mirror ahead of the launch.
struct AdmitPages { int desc; int32_t n; Staging* sg; int32_t* d_mirror; };

// Checked before any state changes, by the stateless entries and by kam_admit alike.
kam_status validate_patch(kam_ctx* c, const kam_patch* p, int32_t rank, int idx) {
  if (rank < 0 || rank > KAM_MAX_RANK) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: rank %d outside [0, %d]", idx, rank, KAM_MAX_RANK);
  if (!p || rank == 0) return KAM_OK;
  if (!p->Uk || !p->Wk || (c->lay.has_v && (!p->Uv || !p->Wv)))
    return fail(c, KAM_ERR_INVALID_ARG, "desc %d: patch factor arrays must not be NULL when rank > 0", idx);
  if (p->frame != KAM_PATCH_TARGET_FRAME && p->frame != KAM_PATCH_CANONICAL_FRAME)
    return fail(c, KAM_ERR_INVALID_ARG, "desc %d: unknown patch frame", idx);
  if (p->u_token_stride <= 0 || p->u_head_stride < 0) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: bad U strides", idx);
  if (p->rank_per_layer)
    for (int l = 0; l < c->lay.n_layers; ++l)
      if (p->rank_per_layer[l] < 0 || p->rank_per_layer[l] > KAM_MAX_RANK)
        return fail(c, KAM_ERR_INVALID_ARG, "desc %d: rank_per_layer[%d] = %d outside [0, %d]", idx, l, p->rank_per_layer[l], KAM_MAX_RANK);
  return KAM_OK;
}

kam_status run_reloc(kam_ctx* c, const kam_pool* pool, const std::vector<HostReloc>& hs, cudaStream_t st, const AdmitPages* ap = nullptr) {
  const kam_layout& L = c->lay;
  const int n = (int)hs.size();
  // ---- validate everything before touching anything
  int max_rank = 0, max_tokens = 0;
  bool fast = c->fast_layout, inplace_only = true;
  for (int i = 0; i < n; ++i) {
    const HostReloc& h = hs[i];
    if (h.n_tokens < 0) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: n_tokens < 0", i);
    if (h.bt == nullptr && !(ap && ap->desc == i)) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: block_table is NULL", i);
    if (h.dst0 < 0) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: negative token start", i);
    if (h.dst0 + h.n_tokens > (int64_t)INT32_MAX) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: token range beyond 2^31 - 1", i);
    const bool inplace = h.flags & FLAG_INPLACE;
    inplace_only = inplace_only && inplace;
    if (!inplace && (h.k == nullptr || (L.has_v && h.v == nullptr)))
      return fail(c, KAM_ERR_INVALID_ARG, "desc %d: chunk layer-pointer arrays must not be NULL", i);
    kam_status vs = validate_patch(c, h.patch, h.rank, i);
    if (vs != KAM_OK) return vs;
    max_tokens = std::max(max_tokens, h.n_tokens);
    const kam_patch* p = (h.patch && h.rank > 0) ? h.patch : nullptr;
    for (int l = 0; l < L.n_layers && p; ++l) max_rank = std::max(max_rank, p->rank_per_layer ? p->rank_per_layer[l] : h.rank);
  }
  if (n == 0 || max_tokens == 0) return KAM_OK;
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");

  RelocGeom g{};
  if (fast) { std::string why; if (!build_reloc_geom(c, max_rank, inplace_only, &g, &why)) fast = false; }
  // any rank <= KAM_MAX_RANK runs on the tiled kernel (padded to a multiple of 16 in shared memory); what can still send a
  // call to the element-wise kernel is a U layout the bulk copies cannot address (u_form in internal.h)
  for (int i = 0; i < n && fast; ++i) {
    const kam_patch* p = (hs[i].patch && hs[i].rank > 0) ? hs[i].patch : nullptr;
    for (int l = 0; l < L.n_layers && p && fast; ++l) {
      const int r = p->rank_per_layer ? p->rank_per_layer[l] : hs[i].rank;
      if (r > 0 && u_form(g.su_row, g.HG, g.n_hg, r, p->u_token_stride, p->u_head_stride) == U_NONE) fast = false;
    }
  }

  // the admitted chunk's page list: in the kernel parameters when it fits, else one small copy ahead of the launch
  const bool inline_pages = ap && fast && ap->n <= kRelocInlinePages;
  if (ap && !inline_pages) {
    cudaError_t e = cudaMemcpyAsync(ap->d_mirror, ap->sg->host, (size_t)ap->n * 4, cudaMemcpyHostToDevice, st);
    staging_release(ap->sg, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(page list)");
  }
  // Small batches on the tiled kernel carry their descriptors in the kernel parameters; anything else is staged through
  // pinned host memory and copied with one cudaMemcpyAsync on the caller's stream.
  const bool inline_descs = fast && n <= kRelocInlineDescs;
  const size_t desc_bytes = (size_t)n * sizeof(RelocDescDev);
  const size_t prefix_off = (desc_bytes + 15) & ~size_t(15);
  const size_t total_bytes = prefix_off + (size_t)2 * (n + 1) * sizeof(long long);      // tile prefix | weight prefix
  Staging* sg = nullptr;
  std::unique_ptr<RelocInline> inl(new (std::nothrow) RelocInline());
  if (!inl) return fail(c, KAM_ERR_STATE, "out of host memory");
  memset(inl.get(), 0, sizeof(RelocInline));
  kam_status s = KAM_OK;
  if (!inline_descs && (s = staging_acquire(c, total_bytes, &sg)) != KAM_OK) return s;
  RelocDescDev* dd = inline_descs ? inl->d : static_cast<RelocDescDev*>(sg->host);
  long long* prefix = inline_descs ? inl->prefix : reinterpret_cast<long long*>(static_cast<char*>(sg->host) + prefix_off);
  long long* wprefix = inline_descs ? inl->wprefix : prefix + (n + 1);
  long long acc = 0, wacc = 0;
  for (int i = 0; i < n; ++i) {
    const HostReloc& h = hs[i];
    RelocDescDev d{};
    const kam_patch* p = (h.patch && h.rank > 0) ? h.patch : nullptr;
    d.k_src = h.k; d.v_src = h.v;
    d.Uk = p ? p->Uk : nullptr; d.Wk = p ? p->Wk : nullptr;
    d.Uv = (p && L.has_v) ? p->Uv : nullptr; d.Wv = (p && L.has_v) ? p->Wv : nullptr;
    d.block_table = (ap && ap->desc == i) ? ap->d_mirror : h.bt; d.dst_token_start = h.dst0; d.delta = h.delta;
    d.u_token_stride = p ? p->u_token_stride : 0; d.u_head_stride = p ? p->u_head_stride : 0;
    d.n_tokens = h.n_tokens;
    d.flags = h.flags | ((p && p->frame == KAM_PATCH_CANONICAL_FRAME) ? FLAG_CANONICAL_FRAME : 0) |
              ((inline_pages && ap->desc == i) ? FLAG_INLINE_PAGES : 0);
    for (int l = 0; l < L.n_layers; ++l) d.rank_l[l] = (uint8_t)(p ? (p->rank_per_layer ? p->rank_per_layer[l] : h.rank) : 0);
    prefix[i] = acc; wprefix[i] = wacc;
    d.tile_weight = 1;
    if (fast) {                                              // the same tile forms as TileWalk::set_desc in the kernel
      const bool inplace = h.flags & FLAG_INPLACE;
      const int tile_tok = (inplace && g.nkv == 2 && !g.kv_split) ? 2 * g.TT : g.TT;
      const int n_kv = (g.kv_split && g.nkv == 2 && !inplace) ? 2 : 1;
      const long long tiles = (long long)L.n_layers * g.n_hg * n_kv * ((h.n_tokens + tile_tok - 1) / tile_tok);
      // weight of a tile: the bytes it moves (rows read + written, U read), in 64-byte units; tiles that also run the patch
      // (W staging, MMAs) cost "reloc_patch_cost_pct" of their bytes (measured: 1.72 vs 1.50 us for 68 vs 64 KB)
      const int row_sets = (inplace || g.kv_split) ? 1 : g.nkv;
      const int u_heads = (p && p->u_head_stride) ? g.HG : 1;
      long long bytes = (long long)row_sets * 2 * tile_tok * g.slice_bytes + (p ? (long long)row_sets * g.TT * u_heads * h.rank * 2 : 0);
      if (p) bytes = bytes * c->opt.reloc_patch_cost_pct / 100;
      d.tile_weight = (int32_t)std::max<long long>(1, bytes / 64);
      acc += tiles; wacc += tiles * d.tile_weight;
    }
    dd[i] = d;
  }
  prefix[n] = acc; wprefix[n] = wacc;
  const RelocDescDev* d_descs = nullptr;
  if (!inline_descs) {
    if ((s = staging_commit(c, sg, total_bytes, st)) != KAM_OK) return s;
    d_descs = static_cast<const RelocDescDev*>(sg->dev);
  }

  if (fast) {
    RelocParams p{};
    p.descs = d_descs;
    p.tile_prefix = inline_descs ? nullptr : reinterpret_cast<const long long*>(static_cast<const char*>(sg->dev) + prefix_off);
    p.w_prefix = inline_descs ? nullptr : p.tile_prefix + (n + 1);
    p.total_weight = wacc;
    p.pool_k = pool->k_layers; p.pool_v = pool->v_layers;
    p.total_tiles = acc; p.n_descs = n; p.inv_freq = c->d_inv_freq;
    p.num_pages = pool->num_pages; p.err = c->d_err;
    const int grid = (int)std::min<long long>(c->sm_count, acc);
    std::unique_ptr<RelocPages> pg;
    if (inline_pages) {
      pg.reset(new (std::nothrow) RelocPages());
      if (!pg) return fail(c, KAM_ERR_STATE, "out of host memory");
      memcpy(pg->pages, ap->sg->host, (size_t)ap->n * 4);
      pg->mirror_dst = ap->d_mirror; pg->n = ap->n;
    }
    launch_relocate_fast(g, p, *inl, pg.get(), grid, c->opt.reloc_pdl != 0, st);
  } else {
    GenericParams p{};
    p.descs = d_descs; p.pool_k = pool->k_layers; p.pool_v = pool->v_layers;
    p.n_descs = n; p.L = L.n_layers; p.H = L.n_kv_heads; p.D = L.row_dim; p.P = L.page_size;
    p.rope_off = L.rope_off; p.d_r = L.rope_dim; p.rope_style = L.rope_style; p.has_v = L.has_v;
    p.elem_f32 = L.elem_dtype == KAM_F32; p.factor_f32 = L.factor_dtype == KAM_F32; p.theta = L.rope_theta;
    p.num_pages = pool->num_pages; p.err = c->d_err;
    launch_relocate_generic(p, max_tokens, st);
    ++c->generic_launches;
  }
  ++c->kernels_launched;
  cudaError_t e = cudaGetLastError();
  if (sg) staging_release(sg, st);
  if (e != cudaSuccess) return cuda_fail(c, e, fast ? "kam_relocate_patch_kernel launch" : "kam_relocate_patch_generic_kernel launch");
  return KAM_OK;
}

// TMA tensor maps over the pool, one per (layer, K|V): dims (64 columns, slots, 64-column blocks) so that a box of
// (64, 16 tokens, column blocks of a head group) lands in shared memory as [column block][token][128 B], SWIZZLE_128B.
typedef CUresult (*PFN_tmapEncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                        const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                        CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Builds the maps of one pool; returns the device array or nullptr (c->tmap_why says why).
void* build_pool_tensor_maps(kam_ctx* c, const kam_pool& pool) {
  const kam_layout& L = c->lay;
  if (L.elem_dtype != KAM_BF16) { c->tmap_why = "needs a bf16 pool"; return nullptr; }
  const bool mla = !L.has_v;
  if (mla && (L.n_kv_heads != 1 || L.row_dim % 64)) { c->tmap_why = "MLA rows must be a multiple of 64 columns"; return nullptr; }
  if (L.page_size % 16 || (!mla && L.row_dim != 64 && L.row_dim != 128)) { c->tmap_why = "needs page_size % 16 == 0 and head_dim 64/128"; return nullptr; }
  if (pool.num_pages < 1) { c->tmap_why = "empty pool"; return nullptr; }
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError(); c->tmap_why = "cuTensorMapEncodeTiled not available"; return nullptr;
  }
  PFN_tmapEncodeTiled encode = reinterpret_cast<PFN_tmapEncodeTiled>(fn);
  std::vector<void*> kp(L.n_layers), vp(L.n_layers);
  if (cudaMemcpy(kp.data(), pool.k_layers, sizeof(void*) * L.n_layers, cudaMemcpyDeviceToHost) != cudaSuccess ||
      (!mla && cudaMemcpy(vp.data(), pool.v_layers, sizeof(void*) * L.n_layers, cudaMemcpyDeviceToHost) != cudaSuccess)) {
    cudaGetLastError(); c->tmap_why = "could not read the pool's layer pointers"; return nullptr;
  }
  const int HG = decode_head_group(L);                  // MLA: one "head" of row_dim columns, the whole row is one box
  const cuuint64_t gdim[3] = {64, (cuuint64_t)pool.num_pages * L.page_size, (cuuint64_t)L.n_kv_heads * L.row_dim / 64};
  const cuuint64_t gstride[2] = {(cuuint64_t)L.n_kv_heads * L.row_dim * 2, 128};
  const cuuint32_t box[3] = {64, 16, (cuuint32_t)(HG * L.row_dim / 64)};
  const cuuint32_t estr[3] = {1, 1, 1};
  std::vector<CUtensorMap> maps((size_t)2 * L.n_layers);
  memset(maps.data(), 0, maps.size() * sizeof(CUtensorMap));
  for (int l = 0; l < L.n_layers; ++l)
    for (int kv = 0; kv < (mla ? 1 : 2); ++kv) {             // MLA: one map, the whole latent+rope row x 16 tokens is one box
      CUresult r = encode(&maps[2 * l + kv], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, kv ? vp[l] : kp[l], gdim, gstride, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) { c->tmap_why = "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r); return nullptr; }
    }
  static_assert(sizeof(CUtensorMap) == 128, "tensor map size");
  void* d = nullptr;
  if (cudaMalloc(&d, maps.size() * sizeof(CUtensorMap)) != cudaSuccess ||
      cudaMemcpy(d, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaGetLastError();
    if (d) cudaFree(d);
    c->tmap_why = "could not upload tensor maps";
    return nullptr;
  }
  return d;
}

}  // namespace

namespace kam {
// Tensor maps are a property of a pool (its layer base pointers and page count), so they are cached per pool: the context's
// own (built at kam_create) and up to kMaxTmapSets caller pools, keyed by the pool's pointer arrays.  The first decode call
// with a new pool reads its layer pointers back (a synchronous copy); a pool whose arrays are re-filled in place must not
// keep the same array addresses (the header says so).
const void* tmaps_for_pool(kam_ctx* c, const kam_pool* pool) {
  for (TmapSet& t : c->tmap_sets)
    if (t.k_layers == pool->k_layers && t.v_layers == pool->v_layers && t.num_pages == pool->num_pages) { t.stamp = ++c->tmap_clock; return t.d_tmaps; }
  void* d = build_pool_tensor_maps(c, *pool);               // nullptr is cached too: the reason does not change
  if (c->tmap_sets.size() >= (size_t)kMaxTmapSets) {
    size_t victim = 1;                                          // entry 0 is the context's own pool
    for (size_t i = 2; i < c->tmap_sets.size(); ++i) if (c->tmap_sets[i].stamp < c->tmap_sets[victim].stamp) victim = i;
    if (c->tmap_sets[victim].d_tmaps) c->graveyard.push_back(c->tmap_sets[victim].d_tmaps);    // may still be read by queued work
    c->tmap_sets.erase(c->tmap_sets.begin() + victim);
  }
  c->tmap_sets.push_back(TmapSet{pool->k_layers, pool->v_layers, pool->num_pages, d, ++c->tmap_clock});
  return d;
}
}  // namespace kam

namespace {

kam_status validate_layout(const kam_layout* L) {
  if (!L) return fail(nullptr, KAM_ERR_INVALID_ARG, "layout is NULL");
  if (L->kind < KAM_MHA || L->kind > KAM_MLA) return fail(nullptr, KAM_ERR_INVALID_ARG, "unknown layout kind");
  if (L->n_layers < 1 || L->n_layers > KAM_MAX_LAYERS) return fail(nullptr, KAM_ERR_INVALID_ARG, "n_layers outside [1, %d]", KAM_MAX_LAYERS);
  if (L->n_kv_heads < 1 || L->n_q_heads < 1 || L->n_q_heads % L->n_kv_heads) return fail(nullptr, KAM_ERR_INVALID_ARG, "n_q_heads must be a positive multiple of n_kv_heads");
  if (L->row_dim < 8 || L->row_dim % 8) return fail(nullptr, KAM_ERR_INVALID_ARG, "row_dim must be a positive multiple of 8");
  if (L->rope_dim < 0 || L->rope_dim % 2) return fail(nullptr, KAM_ERR_INVALID_ARG, "rope_dim must be even");
  if (L->rope_off < 0 || L->rope_off + L->rope_dim > L->row_dim) return fail(nullptr, KAM_ERR_INVALID_ARG, "rope band outside the row");
  if (L->rope_dim > 512) return fail(nullptr, KAM_ERR_UNSUPPORTED, "rope_dim > 512");
  if (L->page_size < 1) return fail(nullptr, KAM_ERR_INVALID_ARG, "page_size < 1");
  if (L->rope_style != KAM_ROPE_HALF && L->rope_style != KAM_ROPE_INTERLEAVED) return fail(nullptr, KAM_ERR_INVALID_ARG, "unknown rope style");
  if ((L->elem_dtype != KAM_BF16 && L->elem_dtype != KAM_F32) || (L->factor_dtype != KAM_BF16 && L->factor_dtype != KAM_F32))
    return fail(nullptr, KAM_ERR_INVALID_ARG, "unknown dtype");
  if (!(L->rope_theta > 0)) return fail(nullptr, KAM_ERR_INVALID_ARG, "rope_theta must be positive");
  if (L->kind == KAM_MHA && L->n_q_heads != L->n_kv_heads) return fail(nullptr, KAM_ERR_INVALID_ARG, "MHA needs n_q_heads == n_kv_heads");
  if (!L->has_v && (L->v_dim < 0 || L->v_dim > L->row_dim)) return fail(nullptr, KAM_ERR_INVALID_ARG, "v_dim outside the row");
  return KAM_OK;
}

}  // namespace

// =================================================================================================================
extern "C" {

const char* kam_version(void) { return "libkamera 0.1 (sm_100a)"; }

const char* kam_last_error(const kam_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

kam_status kam_create(const kam_layout* layout, const kam_pool* pool, int32_t max_requests,
                      int32_t max_chunks_per_request, int32_t max_pages_per_chunk, kam_ctx** out) {
  if (!out) return fail(nullptr, KAM_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  kam_status s = validate_layout(layout);
  if (s != KAM_OK) return s;
  if (max_requests < 0 || max_chunks_per_request < 0 || max_pages_per_chunk < 0)
    return fail(nullptr, KAM_ERR_INVALID_ARG, "negative window-store size");
  if (pool && (pool->num_pages < 0 || !pool->k_layers || (layout->has_v && !pool->v_layers)))
    return fail(nullptr, KAM_ERR_INVALID_ARG, "bad pool");
  kam_ctx* c = new (std::nothrow) kam_ctx();
  if (!c) return fail(nullptr, KAM_ERR_STATE, "out of host memory");
  c->lay = *layout;
  c->fast_layout = build_head_blocks(c);
  c->max_requests = max_requests; c->max_chunks = max_chunks_per_request; c->max_ppc = max_pages_per_chunk;
  if (pool) { c->pool = *pool; c->has_pool = true; }
  if (pool) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { kam_status r = cuda_fail(nullptr, e, "kam_create: no usable CUDA device"); delete c; return r; }
    c->cuda_ok = true;
    tmaps_for_pool(c, &c->pool);                   // entry 0 of the cache: the context's own pool
    // the library's own copy stream + events (kam_relocate_patch_host); without them the host entry runs on the caller's stream
    if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c->copy_stream = nullptr; }
    for (int i = 0; i < 2 && c->copy_stream; ++i)
      if (cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming) != cudaSuccess ||
          cudaEventCreateWithFlags(&c->ev_consumed[i], cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError(); cudaStreamDestroy(c->copy_stream); c->copy_stream = nullptr;
      }
    e = cudaMalloc(&c->d_err, sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemset(c->d_err, 0, sizeof(int32_t));
    if (e != cudaSuccess) { kam_status r = cuda_fail(nullptr, e, "kam_create: device error counter"); kam_destroy(c); return r; }
    if (layout->rope_dim > 0) {                // f_i = theta^(-2i/d_r) in fp64, once (R-2)
      std::vector<double> f((size_t)layout->rope_dim / 2);
      for (size_t i = 0; i < f.size(); ++i) f[i] = pow(layout->rope_theta, -2.0 * (double)i / layout->rope_dim);
      e = cudaMalloc(&c->d_inv_freq, f.size() * sizeof(double));
      if (e == cudaSuccess) e = cudaMemcpy(c->d_inv_freq, f.data(), f.size() * sizeof(double), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) { kam_status r = cuda_fail(nullptr, e, "kam_create: inverse-frequency table"); kam_destroy(c); return r; }
    }
  }
  if (max_requests > 0 && max_chunks_per_request > 0 && max_pages_per_chunk > 0) {
    const int32_t np = pool ? pool->num_pages : max_requests * max_chunks_per_request * max_pages_per_chunk;
    c->win.reset(new WindowStore(np, layout->page_size, max_requests, max_chunks_per_request, max_pages_per_chunk));
    if (c->cuda_ok) {
      const size_t bytes = (size_t)max_requests * max_chunks_per_request * max_pages_per_chunk * sizeof(int32_t);
      cudaError_t e = cudaMalloc(&c->d_slot_pages, bytes);
      if (e != cudaSuccess) { kam_status r = cuda_fail(nullptr, e, "cudaMalloc(page lists)"); kam_destroy(c); return r; }
    }
  }
  *out = c;
  return KAM_OK;
}

kam_status kam_destroy(kam_ctx* c) {
  if (!c) return KAM_OK;
  if (c->cuda_ok) {
    for (Staging& s : c->staging) {
      if (s.in_flight) cudaEventSynchronize(s.ev);
      if (s.ev) cudaEventDestroy(s.ev);
      if (s.host) cudaFreeHost(s.host);
      if (s.dev) cudaFree(s.dev);
    }
    if (c->d_slot_pages) cudaFree(c->d_slot_pages);
    if (c->d_ws) cudaFree(c->d_ws);
    if (c->d_ws_win) cudaFree(c->d_ws_win);
    for (int i = 0; i < 2; ++i) {
      if (c->d_hstage[i]) cudaFree(c->d_hstage[i]);
      if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
      if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->d_hstage2) cudaFree(c->d_hstage2);
    for (TmapSet& t : c->tmap_sets) if (t.d_tmaps) cudaFree(t.d_tmaps);
    if (c->d_inv_freq) cudaFree(c->d_inv_freq);
    if (c->d_err) cudaFree(c->d_err);
    if (c->d_fp_ws) cudaFree(c->d_fp_ws);
    for (void* p : c->graveyard) cudaFree(p);
  }
  delete c;
  return KAM_OK;
}

kam_status kam_get_stats(kam_ctx* c, kam_stats* out) {
  if (!c || !out) return fail(c, KAM_ERR_INVALID_ARG, "NULL argument");
  kam_stats s{};
  if (c->win) {
    s.pages_free = c->win->pages_free(); s.pages_total = c->win->pages_total();
    s.table_entries_written = c->win->table_entries_written(); s.chunks_live = c->win->chunks_live();
  }
  s.kernels_launched = c->kernels_launched;
  s.generic_launches = c->generic_launches;
  if (c->d_err) {
    int32_t n = 0;
    cudaError_t e = cudaMemcpy(&n, c->d_err, sizeof(n), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(device error counter)");
    s.device_errors = n;
  }
  *out = s;
  return KAM_OK;
}

// ---- stateless operator -------------------------------------------------------------------------------------------
kam_status kam_relocate_patch_batch(kam_ctx* c, const kam_pool* pool, int32_t n, const kam_reloc_desc* descs, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (n < 0 || (n > 0 && !descs)) return fail(c, KAM_ERR_INVALID_ARG, "bad descriptor array");
  kam_status s = check_pool(c, &pool);
  if (s != KAM_OK) return s;
  std::vector<HostReloc> hs((size_t)n);
  for (int i = 0; i < n; ++i) {
    const kam_reloc_desc& d = descs[i];
    if (!d.chunk) return fail(c, KAM_ERR_INVALID_ARG, "desc %d: chunk is NULL", i);
    hs[i] = HostReloc{d.block_table, d.dst_token_start, d.p_target - d.chunk->p_base, d.chunk->k_layers,
                      d.chunk->v_layers, d.patch, d.rank, d.chunk->n_tokens, 0};
  }
  return run_reloc(c, pool, hs, static_cast<cudaStream_t>(stream));
}

// north_star's signature carries `layout = {MHA, GQA, MLA}`; the context was created for one layout (its kernels' geometry,
// frequency table and tensor maps hang off it), so the argument is checked, not dispatched on: NULL = the context's.
static bool same_layout(const kam_layout& a, const kam_layout& b) {
  return a.kind == b.kind && a.n_layers == b.n_layers && a.n_q_heads == b.n_q_heads && a.n_kv_heads == b.n_kv_heads &&
         a.row_dim == b.row_dim && a.rope_off == b.rope_off && a.rope_dim == b.rope_dim && a.has_v == b.has_v &&
         a.v_dim == b.v_dim && a.page_size == b.page_size && a.rope_style == b.rope_style && a.elem_dtype == b.elem_dtype &&
         a.factor_dtype == b.factor_dtype && a.rope_theta == b.rope_theta;
}

kam_status kam_relocate_patch(kam_ctx* c, const kam_pool* pool, const int32_t* block_table, int64_t dst_token_start,
                              const kam_chunk* chunk, int64_t p_target, const kam_patch* patch, int32_t rank,
                              const kam_layout* layout, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (layout && !same_layout(*layout, c->lay))
    return fail(c, KAM_ERR_INVALID_ARG, "kam_relocate_patch: layout differs from the one this context was created for");
  kam_reloc_desc d{block_table, dst_token_start, chunk, p_target, patch, rank};
  return kam_relocate_patch_batch(c, pool, 1, &d, stream);
}

kam_status kam_rotate_inplace(kam_ctx* c, const kam_pool* pool, const int32_t* block_table, int64_t token_start,
                              int32_t n_tokens, int64_t delta, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  kam_status s = check_pool(c, &pool);
  if (s != KAM_OK) return s;
  std::vector<HostReloc> hs(1);
  hs[0] = HostReloc{block_table, token_start, delta, nullptr, nullptr, nullptr, 0, n_tokens, FLAG_INPLACE};
  return run_reloc(c, pool, hs, static_cast<cudaStream_t>(stream));
}

kam_status kam_relocate_patch_host(kam_ctx* c, const kam_pool* pool, const int32_t* block_table, int64_t dst_token_start,
                                   int32_t n_tokens, int64_t p_base, int64_t p_target, const void* const* k_host,
                                   const void* const* v_host, const void* const* Uk_host, const void* const* Wk_host,
                                   const void* const* Uv_host, const void* const* Wv_host, int32_t rank, int32_t frame,
                                   void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  kam_status s = check_pool(c, &pool);
  if (s != KAM_OK) return s;
  const kam_layout& L = c->lay;
  if (!k_host || (L.has_v && !v_host)) return fail(c, KAM_ERR_INVALID_ARG, "host chunk arrays must not be NULL");
  if (rank < 0 || rank > KAM_MAX_RANK) return fail(c, KAM_ERR_INVALID_ARG, "rank %d outside [0, %d]", rank, KAM_MAX_RANK);
  if (rank > 0 && (!Uk_host || !Wk_host || (L.has_v && (!Uv_host || !Wv_host))))
    return fail(c, KAM_ERR_INVALID_ARG, "host factor arrays must not be NULL when rank > 0");
  if (n_tokens < 0 || !block_table || dst_token_start < 0) return fail(c, KAM_ERR_INVALID_ARG, "bad token range / block table");
  if (n_tokens == 0) return KAM_OK;
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t eb = L.elem_dtype == KAM_BF16 ? 2 : 4, fb = L.factor_dtype == KAM_BF16 ? 2 : 4;
  const size_t rows = ((size_t)n_tokens * L.n_kv_heads * L.row_dim * eb + 255) & ~size_t(255);
  const size_t ub = ((size_t)n_tokens * L.n_kv_heads * rank * fb + 255) & ~size_t(255);
  const size_t wb = ((size_t)L.n_kv_heads * rank * L.row_dim * fb + 255) & ~size_t(255);
  const int nkv = L.has_v ? 2 : 1;
  const size_t per_layer = nkv * (rows + ub + wb);
  // Two staging buffers and a copy stream of the library's own: the H2D copy of this chunk runs under the kernel of the
  // previous call (which reads the OTHER buffer).  copy stream: wait until the kernel that last read this buffer is done ->
  // copies -> event; caller's stream: wait for that event -> kernel -> event "consumed".   ("host_copy_overlap" = 0: one
  // buffer, everything on the caller's stream.)
  const bool overlap = c->opt.host_copy_overlap && c->copy_stream;
  const int hb = overlap ? c->hstage_next : 0;      // the buffers alternate only once a call got as far as its kernel (below)
  if ((s = grow_device(c, &c->d_hstage[hb], &c->hstage_cap[hb], per_layer * L.n_layers, "cudaMalloc(host-chunk staging)", st)) != KAM_OK) return s;
  cudaStream_t cs = overlap ? c->copy_stream : st;
  cudaError_t e = cudaSuccess;
  if (overlap && c->hstage_used[hb]) e = cudaStreamWaitEvent(cs, c->ev_consumed[hb], 0);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamWaitEvent(staging buffer)");
  // device pointer tables for the staged copy: [k | v | Uk | Wk | Uv | Wv][n_layers]
  Staging* sg;
  if ((s = staging_acquire(c, (size_t)6 * L.n_layers * sizeof(void*), &sg)) != KAM_OK) return s;
  const void** tabs = static_cast<const void**>(sg->host);
  char* d = static_cast<char*>(c->d_hstage[hb]);
  // Copies whose source AND staging destination continue the previous one are merged: a canonical store that keeps a chunk as
  // one slab in this order (per layer: K, V, U_k, W_k, U_v, W_v) crosses PCIe in ONE transfer instead of 6 per layer.
  const char* run_src = nullptr; char* run_dst = nullptr; size_t run_bytes = 0;
  auto flush = [&]() {
    if (run_bytes && e == cudaSuccess) e = cudaMemcpyAsync(run_dst, run_src, run_bytes, cudaMemcpyHostToDevice, cs);
    run_bytes = 0;
  };
  auto put = [&](int which, int l, const void* const* src, size_t bytes, size_t& off) {
    tabs[which * L.n_layers + l] = nullptr;
    if (!src || bytes == 0) return;
    tabs[which * L.n_layers + l] = d + off;
    const char* sp = static_cast<const char*>(src[l]);
    if (run_bytes && sp == run_src + run_bytes && d + off == run_dst + run_bytes) { run_bytes += bytes; return; }
    flush();
    run_src = sp; run_dst = d + off; run_bytes = bytes;
  };
  for (int l = 0; l < L.n_layers; ++l) {
    size_t off = per_layer * l;
    put(0, l, k_host, (size_t)n_tokens * L.n_kv_heads * L.row_dim * eb, off); off += rows;
    if (L.has_v) { put(1, l, v_host, (size_t)n_tokens * L.n_kv_heads * L.row_dim * eb, off); off += rows; } else tabs[1 * L.n_layers + l] = nullptr;
    put(2, l, rank ? Uk_host : nullptr, (size_t)n_tokens * L.n_kv_heads * rank * fb, off); off += ub;
    put(3, l, rank ? Wk_host : nullptr, (size_t)L.n_kv_heads * rank * L.row_dim * fb, off); off += wb;
    if (L.has_v) {
      put(4, l, rank ? Uv_host : nullptr, (size_t)n_tokens * L.n_kv_heads * rank * fb, off); off += ub;
      put(5, l, rank ? Wv_host : nullptr, (size_t)L.n_kv_heads * rank * L.row_dim * fb, off);
    } else { tabs[4 * L.n_layers + l] = nullptr; tabs[5 * L.n_layers + l] = nullptr; }
  }
  flush();
  if (e != cudaSuccess) { staging_release(sg, cs); return cuda_fail(c, e, "cudaMemcpyAsync(host chunk)"); }
  if ((s = staging_commit(c, sg, (size_t)6 * L.n_layers * sizeof(void*), cs)) != KAM_OK) { staging_release(sg, cs); return s; }
  if (overlap) {
    if ((e = cudaEventRecord(c->ev_copied[hb], cs)) == cudaSuccess) e = cudaStreamWaitEvent(st, c->ev_copied[hb], 0);
    if (e != cudaSuccess) { staging_release(sg, cs); return cuda_fail(c, e, "cudaEventRecord / cudaStreamWaitEvent(host chunk)"); }
  }
  const void* const* dt = static_cast<const void* const*>(sg->dev);
  kam_chunk ch{dt, L.has_v ? dt + L.n_layers : nullptr, n_tokens, p_base};
  kam_patch pa{dt + 2 * L.n_layers, dt + 3 * L.n_layers, L.has_v ? dt + 4 * L.n_layers : nullptr,
               L.has_v ? dt + 5 * L.n_layers : nullptr, (int64_t)L.n_kv_heads * rank, rank, nullptr, frame};
  std::vector<HostReloc> hs(1);
  hs[0] = HostReloc{block_table, dst_token_start, p_target - p_base, ch.k_layers, ch.v_layers, rank ? &pa : nullptr, rank, n_tokens, 0};
  s = run_reloc(c, pool, hs, st);
  staging_release(sg, st);          // the pointer tables are released behind the kernel that reads them
  if (overlap) {
    if (cudaEventRecord(c->ev_consumed[hb], st) == cudaSuccess) c->hstage_used[hb] = true;
    c->hstage_next = hb ^ 1;
  }
  return s;
}

// ---- window store ---------------------------------------------------------------------------------------------------
static kam_status win_status(kam_ctx* c, WindowStore::Result r, const char* what) {
  switch (r) {
    case WindowStore::OK: return KAM_OK;
    case WindowStore::BAD_ARG: return fail(c, KAM_ERR_INVALID_ARG, "%s: invalid argument", what);
    case WindowStore::BAD_STATE: return fail(c, KAM_ERR_STATE, "%s: request not open / already open / window empty or full", what);
    case WindowStore::NO_PAGES: return fail(c, KAM_ERR_NO_PAGES, "%s: free list exhausted", what);
  }
  return KAM_ERR_STATE;
}
#define KAM_NEED_WIN(c)                                                                       \
  if (!(c)) return KAM_ERR_INVALID_ARG;                                                       \
  if (!(c)->win) return fail((c), KAM_ERR_STATE, "context was created without a window store")

kam_status kam_window_open(kam_ctx* c, int32_t req, int64_t window_base) {
  KAM_NEED_WIN(c);
  return win_status(c, c->win->open(req, window_base), "kam_window_open");
}
kam_status kam_window_pin(kam_ctx* c, int32_t req, int32_t n_front) {
  KAM_NEED_WIN(c);
  return win_status(c, c->win->pin(req, n_front), "kam_window_pin");
}
kam_status kam_window_close(kam_ctx* c, int32_t req) {
  KAM_NEED_WIN(c);
  return win_status(c, c->win->close(req), "kam_window_close");
}

static void survivors_to_descs(kam_ctx* c, const std::vector<Rotation>& rot, std::vector<HostReloc>* hs) {
  for (const Rotation& r : rot)
    hs->push_back(HostReloc{c->d_slot_pages + (size_t)r.slot * c->max_ppc, 0, r.delta, nullptr, nullptr, nullptr, 0, r.n_tokens, FLAG_INPLACE});
}

// What kam_admit and kam_slide share.  Everything that can fail for a reason of the caller's (arguments, window state, pages)
// or of the host (staging memory) is checked BEFORE the window store changes; `evict_end` < 0 = no eviction.  The survivors'
// in-place rotations and the admitted chunk's Eq. 1 travel in ONE kam_relocate_patch_kernel launch (they touch disjoint pages).
static kam_status admit_core(kam_ctx* c, int32_t req, int evict_end, int admit_end, const kam_chunk* chunk, const kam_patch* patch,
                             int32_t rank, int32_t materialize, int32_t* handle_out, cudaStream_t st, const char* what) {
  if (!chunk) return fail(c, KAM_ERR_INVALID_ARG, "%s: chunk is NULL", what);
  { kam_status vs = validate_patch(c, patch, rank, 0); if (vs != KAM_OK) return vs; }
  if (c->cuda_ok && (!chunk->k_layers || (c->lay.has_v && !chunk->v_layers)))
    return fail(c, KAM_ERR_INVALID_ARG, "%s: chunk layer-pointer arrays must not be NULL", what);
  kam_status s = win_status(c, c->win->can_admit(req, evict_end, admit_end, chunk->n_tokens), what);
  if (s != KAM_OK) return s;
  const int32_t np = chunk->n_tokens / c->lay.page_size;
  Staging* sg = nullptr;
  if (c->cuda_ok && (s = staging_acquire(c, (size_t)np * 4, &sg)) != KAM_OK) return s;
  // ---- commit: from here on only CUDA runtime failures can interrupt (reported as KAM_ERR_CUDA; the window then lists the
  // chunk although its pages were not written - the context should be destroyed, as after any CUDA error)
  ChunkRec rec; int64_t p_target = 0; std::vector<Rotation> rot;
  if (evict_end >= 0) c->win->evict(req, evict_end, false, nullptr, nullptr);
  c->win->admit(req, admit_end, chunk->n_tokens, materialize != 0, &rec, &p_target, &rot);
  if (handle_out) *handle_out = rec.handle;
  if (!c->cuda_ok) return KAM_OK;                     // bookkeeping-only context
  // device mirror of the chunk's page list: exactly n_tokens / P entries are written (O(1) in the window length)
  int32_t* d_pages = c->d_slot_pages + (size_t)rec.slot * c->max_ppc;
  memcpy(sg->host, c->win->pages_of(rec.slot), (size_t)np * 4);
  std::vector<HostReloc> hs;
  survivors_to_descs(c, rot, &hs);
  hs.push_back(HostReloc{nullptr, 0, p_target - chunk->p_base, chunk->k_layers, chunk->v_layers, patch, rank, chunk->n_tokens, 0});
  const AdmitPages ap{(int)hs.size() - 1, np, sg, d_pages};
  const kam_pool* pool = &c->pool;
  return run_reloc(c, pool, hs, st, &ap);
}

kam_status kam_admit(kam_ctx* c, int32_t req, int32_t end, const kam_chunk* chunk, const kam_patch* patch, int32_t rank,
                     int32_t materialize, int32_t* handle_out, void* stream) {
  KAM_NEED_WIN(c);
  return admit_core(c, req, -1, end, chunk, patch, rank, materialize, handle_out, static_cast<cudaStream_t>(stream), "kam_admit");
}

kam_status kam_slide(kam_ctx* c, int32_t req, int32_t evict_end, int32_t admit_end, const kam_chunk* chunk, const kam_patch* patch,
                     int32_t rank, int32_t materialize, int32_t* handle_out, void* stream) {
  KAM_NEED_WIN(c);
  if (evict_end != KAM_FRONT && evict_end != KAM_BACK) return fail(c, KAM_ERR_INVALID_ARG, "kam_slide: bad evict end");
  return admit_core(c, req, evict_end, admit_end, chunk, patch, rank, materialize, handle_out, static_cast<cudaStream_t>(stream), "kam_slide");
}

kam_status kam_evict(kam_ctx* c, int32_t req, int32_t end, int32_t materialize, void* stream) {
  KAM_NEED_WIN(c);
  std::vector<Rotation> rot;
  kam_status s = win_status(c, c->win->evict(req, end, materialize != 0, nullptr, &rot), "kam_evict");
  if (s != KAM_OK) return s;
  if (rot.empty() || !c->cuda_ok) return KAM_OK;
  std::vector<HostReloc> hs;
  survivors_to_descs(c, rot, &hs);
  const kam_pool* pool = &c->pool;
  return run_reloc(c, pool, hs, static_cast<cudaStream_t>(stream));
}

kam_status kam_window_export(kam_ctx* c, int32_t req, int32_t* bt_out, int32_t bt_cap, int64_t* sm_out, int64_t sm_cap,
                             int32_t* starts_out, int64_t* offs_out, int32_t* handles_out, int32_t chunk_cap,
                             int32_t* n_pages_out, int32_t* n_chunks_out) {
  KAM_NEED_WIN(c);
  if (!c->win->is_open(req)) return fail(c, KAM_ERR_STATE, "kam_window_export: request not open");
  const auto& ch = c->win->chunks(req);
  const int P = c->lay.page_size;
  int64_t n_tok = 0; int32_t n_pages = 0;
  for (const ChunkRec& r : ch) { n_tok += r.n_tokens; n_pages += r.n_tokens / P; }
  const int32_t nc = (int32_t)ch.size();
  if ((bt_out && bt_cap < n_pages) || (sm_out && sm_cap < n_tok) || ((offs_out || handles_out) && chunk_cap < nc) ||
      (starts_out && chunk_cap < nc + 1))                       // chunk_starts_out takes n_chunks + 1 entries
    return fail(c, KAM_ERR_INVALID_ARG, "kam_window_export: output capacity too small");
  int64_t pos = c->win->window_base(req), tok = 0; int32_t pg = 0, i = 0;
  for (const ChunkRec& r : ch) {
    const int32_t* pages = c->win->pages_of(r.slot);
    const int32_t np = r.n_tokens / P;
    if (bt_out) memcpy(bt_out + pg, pages, (size_t)np * 4);
    if (sm_out) for (int32_t t = 0; t < r.n_tokens; ++t) sm_out[tok + t] = (int64_t)pages[t / P] * P + t % P;
    if (starts_out) starts_out[i] = (int32_t)tok;
    if (offs_out) offs_out[i] = pos - r.phase;
    if (handles_out) handles_out[i] = r.handle;
    pg += np; tok += r.n_tokens; pos += r.n_tokens; ++i;
  }
  if (starts_out) starts_out[nc] = (int32_t)tok;
  if (n_pages_out) *n_pages_out = n_pages;
  if (n_chunks_out) *n_chunks_out = nc;
  return KAM_OK;
}

// ---- tunables ---------------------------------------------------------------------------------------------------------
kam_status kam_set_option(kam_ctx* c, const char* key, int64_t value) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (!key) return fail(c, KAM_ERR_INVALID_ARG, "kam_set_option: key is NULL");
  struct Opt { const char* name; int* field; int lo, hi; };
  Options& o = c->opt;
  const Opt opts[] = {
      {"reloc_stages", &o.reloc_stages, 0, 8},       {"reloc_head_group", &o.reloc_hg, 0, 4},
      {"reloc_kv_split", &o.reloc_kv_split, 0, 2},   {"reloc_contig", &o.reloc_contig, 0, 1},
      {"reloc_row_blocks", &o.reloc_rb, 0, 4},       {"reloc_evict_first", &o.reloc_load_hint, 0, 1},
      {"decode_ctas_per_sm", &o.dec_ctas_per_sm, 0, 8}, {"decode_boxes", &o.dec_boxes, 0, 16},
      {"decode_pdl", &o.use_pdl, 0, 1},              {"decode_tma", &o.dec_tma, 0, 1},
      {"host_copy_overlap", &o.host_copy_overlap, 0, 1}, {"host_entries_sync", &o.host_sync, 0, 1},
      {"reloc_patch_cost_pct", &o.reloc_patch_cost_pct, 50, 200}, {"reloc_pdl", &o.reloc_pdl, 0, 1},
      {"reloc_head_group_cap", &o.reloc_hg_cap, 1, 8}, {"prefill_tcgen05", &o.prefill_tc, 0, 1},
  };
  for (const Opt& op : opts)
    if (strcmp(op.name, key) == 0) {
      if (value < op.lo || value > op.hi) return fail(c, KAM_ERR_INVALID_ARG, "kam_set_option: %s = %lld outside [%d, %d]", key, (long long)value, op.lo, op.hi);
      *op.field = (int)value;
      for (auto& row : c->dec_geom_ok) for (bool& ok : row) ok = false;      // cached decode geometries depend on the options
      c->winplan_epoch = ~0ull;
      c->decplan_valid = false;
      return KAM_OK;
    }
  return fail(c, KAM_ERR_INVALID_ARG, "kam_set_option: unknown key '%s'", key);
}

// ---- compile side: form the rank-m patch of one chunk ----------------------------------------------------
kam_status kam_form_patch(kam_ctx* c, const void* const* kv_cond_layers, const void* const* kv_solo_layers, int32_t n_tokens,
                          int64_t delta, int32_t is_key, int32_t rank, int32_t n_iter, void* const* U_out, void* const* W_out,
                          float* sigma_out, void* stream) {
  if (!c) return KAM_ERR_INVALID_ARG;
  if (!kv_cond_layers || !kv_solo_layers || !U_out || !W_out) return fail(c, KAM_ERR_INVALID_ARG, "kam_form_patch: NULL argument");
  if (n_tokens < 1 || rank < 1 || rank > KAM_MAX_RANK || n_iter < 0 || n_iter > 64) return fail(c, KAM_ERR_INVALID_ARG, "kam_form_patch: bad n_tokens / rank / n_iter");
  const kam_layout& L = c->lay;
  if (L.elem_dtype != KAM_BF16 || L.factor_dtype != KAM_BF16) return fail(c, KAM_ERR_UNSUPPORTED, "kam_form_patch needs bf16 rows and factors");
  if (!c->cuda_ok) return fail(c, KAM_ERR_CUDA, "no CUDA device: libkamera has no CPU fallback");
  FormPatchParams p{};
  p.cond = kv_cond_layers; p.solo = kv_solo_layers; p.U_out = U_out; p.W_out = W_out; p.sigma_out = sigma_out;
  p.inv_freq = c->d_inv_freq; p.delta = delta;
  p.L = L.n_layers; p.H = L.n_kv_heads; p.T = n_tokens; p.D = L.row_dim; p.m = rank;
  p.b = std::min(rank + 8, std::min(L.row_dim, n_tokens));
  if (p.b < rank) return fail(c, KAM_ERR_INVALID_ARG, "rank %d exceeds min(row_dim, n_tokens)", rank);
  p.ldq = p.b | 1;
  p.n_iter = n_iter ? n_iter : 6;
  p.rope_off = L.rope_off; p.d_r = L.rope_dim; p.rope_style = L.rope_style; p.rotate = (is_key && L.rope_dim > 0 && delta != 0) ? 1 : 0;
  const size_t fl = (size_t)2 * p.D * p.ldq + (size_t)16 * p.D + (size_t)16 * p.b + (size_t)2 * p.b * (p.b + 1) + p.b + 8 + p.b;
  p.smem_bytes = (int)(fl * 4 + 64);
  if (p.smem_bytes > 227 * 1024) return fail(c, KAM_ERR_UNSUPPORTED, "row_dim %d x rank %d does not fit the subspace block in shared memory", p.D, rank);
  const size_t dws = (size_t)p.L * p.H * p.T * p.D * 4, bws = (size_t)p.L * p.H * p.T * p.b * 4;
  kam_status s = grow_device(c, &c->d_fp_ws, &c->fp_ws_cap, dws + bws + 256, "cudaMalloc(form_patch workspace)", static_cast<cudaStream_t>(stream));
  if (s != KAM_OK) return s;
  p.delta_ws = static_cast<float*>(c->d_fp_ws);
  p.b_ws = reinterpret_cast<float*>(static_cast<char*>(c->d_fp_ws) + ((dws + 255) & ~size_t(255)));
  launch_form_patch(p, static_cast<cudaStream_t>(stream));
  c->kernels_launched += 2;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(c, e, "kam_form_patch launch");
  return KAM_OK;
}

}  // extern "C"

/* Compiled against include/kamera.h by tests/test_abi.py (cc -I include): prints the size of every ABI struct and the offset
 * of every field, so that a header edit that moves a field is caught against binding.py's ctypes mirror, and drives the
 * bookkeeping-only part of the library through the header's own prototypes (no GPU needed). */
#include <stddef.h>
#include <stdio.h>
#include <string.h>

#include "kamera.h"

#define SZ(T) printf("sizeof " #T " %zu\n", sizeof(T))
#define OFF(T, f) printf("offsetof " #T " " #f " %zu\n", offsetof(T, f))

int main(void) {
  SZ(kam_layout);
  OFF(kam_layout, kind); OFF(kam_layout, n_layers); OFF(kam_layout, n_q_heads); OFF(kam_layout, n_kv_heads);
  OFF(kam_layout, row_dim); OFF(kam_layout, rope_off); OFF(kam_layout, rope_dim); OFF(kam_layout, has_v);
  OFF(kam_layout, v_dim); OFF(kam_layout, page_size); OFF(kam_layout, rope_style); OFF(kam_layout, elem_dtype);
  OFF(kam_layout, factor_dtype); OFF(kam_layout, rope_theta);
  SZ(kam_pool); OFF(kam_pool, k_layers); OFF(kam_pool, v_layers); OFF(kam_pool, num_pages);
  SZ(kam_chunk); OFF(kam_chunk, k_layers); OFF(kam_chunk, v_layers); OFF(kam_chunk, n_tokens); OFF(kam_chunk, p_base);
  SZ(kam_patch); OFF(kam_patch, Uk); OFF(kam_patch, Wk); OFF(kam_patch, Uv); OFF(kam_patch, Wv);
  OFF(kam_patch, u_token_stride); OFF(kam_patch, u_head_stride); OFF(kam_patch, rank_per_layer); OFF(kam_patch, frame);
  SZ(kam_reloc_desc); OFF(kam_reloc_desc, block_table); OFF(kam_reloc_desc, dst_token_start); OFF(kam_reloc_desc, chunk);
  OFF(kam_reloc_desc, p_target); OFF(kam_reloc_desc, patch); OFF(kam_reloc_desc, rank);
  SZ(kam_patch_ref); OFF(kam_patch_ref, Uk); OFF(kam_patch_ref, Wk); OFF(kam_patch_ref, Uv); OFF(kam_patch_ref, Wv);
  OFF(kam_patch_ref, u_token_stride); OFF(kam_patch_ref, u_head_stride); OFF(kam_patch_ref, rank); OFF(kam_patch_ref, frame);
  SZ(kam_stats); OFF(kam_stats, pages_free); OFF(kam_stats, pages_total); OFF(kam_stats, table_entries_written);
  OFF(kam_stats, chunks_live); OFF(kam_stats, kernels_launched); OFF(kam_stats, device_errors); OFF(kam_stats, generic_launches);
  printf("const KAM_MAX_RANK %d\nconst KAM_MAX_LAYERS %d\n", KAM_MAX_RANK, KAM_MAX_LAYERS);
  printf("const KAM_STATIC_SCRATCH_BYTES %u\n", KAM_STATIC_SCRATCH_BYTES);
  printf("enum KAM_ERR_CUDA %d\nenum KAM_MLA %d\nenum KAM_ROPE_INTERLEAVED %d\nenum KAM_PATCH_CANONICAL_FRAME %d\nenum KAM_BACK %d\nenum KAM_F32 %d\n",
         (int)KAM_ERR_CUDA, (int)KAM_MLA, (int)KAM_ROPE_INTERLEAVED, (int)KAM_PATCH_CANONICAL_FRAME, (int)KAM_BACK, (int)KAM_F32);

  /* ---- the library through the header: a bookkeeping-only context (pool == NULL), one window, two chunks */
  printf("version %s\n", kam_version());
  kam_layout lay;
  memset(&lay, 0, sizeof lay);
  lay.kind = KAM_GQA; lay.n_layers = 2; lay.n_q_heads = 8; lay.n_kv_heads = 4; lay.row_dim = 128; lay.rope_off = 0;
  lay.rope_dim = 128; lay.has_v = 1; lay.page_size = 16; lay.rope_style = KAM_ROPE_HALF; lay.elem_dtype = KAM_BF16;
  lay.factor_dtype = KAM_BF16; lay.rope_theta = 1e6;
  kam_ctx *ctx = NULL;
  if (kam_create(&lay, NULL, 2, 4, 8, &ctx) != KAM_OK) { printf("FAIL create: %s\n", kam_last_error(NULL)); return 1; }
  if (kam_set_option(ctx, "reloc_stages", 3) != KAM_OK || kam_set_option(ctx, "no_such_key", 1) != KAM_ERR_INVALID_ARG) { printf("FAIL set_option\n"); return 1; }
  kam_chunk ch; memset(&ch, 0, sizeof ch);
  int32_t handle = -1, bt[8], starts[3], handles[3], n_pages = 0, n_chunks = 0;
  int64_t offs[3];
  if (kam_window_open(ctx, 1, 100) != KAM_OK) { printf("FAIL open\n"); return 1; }
  ch.n_tokens = 32; if (kam_admit(ctx, 1, KAM_BACK, &ch, NULL, 0, 1, &handle, NULL) != KAM_OK) { printf("FAIL admit: %s\n", kam_last_error(ctx)); return 1; }
  ch.n_tokens = 48; if (kam_admit(ctx, 1, KAM_FRONT, &ch, NULL, 0, 0, &handle, NULL) != KAM_OK) { printf("FAIL admit 2\n"); return 1; }
  /* capacities in entries: chunk_starts_out takes n_chunks + 1, so chunk_cap = n_chunks must be refused, n_chunks + 1 accepted */
  if (kam_window_export(ctx, 1, bt, 8, NULL, 0, starts, offs, handles, 2, &n_pages, &n_chunks) != KAM_ERR_INVALID_ARG) { printf("FAIL export cap\n"); return 1; }
  if (kam_window_export(ctx, 1, bt, 8, NULL, 0, starts, offs, handles, 3, &n_pages, &n_chunks) != KAM_OK) { printf("FAIL export\n"); return 1; }
  printf("export n_pages %d n_chunks %d bt %d %d %d %d %d starts %d %d %d offs %lld %lld handles %d %d\n", n_pages, n_chunks, bt[0], bt[1], bt[2],
         bt[3], bt[4], starts[0], starts[1], starts[2], (long long)offs[0], (long long)offs[1], handles[0], handles[1]);
  /* one slide: oldest out, one in at the back, survivors settled */
  ch.n_tokens = 16; if (kam_slide(ctx, 1, KAM_FRONT, KAM_BACK, &ch, NULL, 0, 1, &handle, NULL) != KAM_OK) { printf("FAIL slide: %s\n", kam_last_error(ctx)); return 1; }
  kam_stats st;
  if (kam_get_stats(ctx, &st) != KAM_OK) { printf("FAIL stats\n"); return 1; }
  printf("stats free %lld total %lld written %lld live %lld launched %lld\n", (long long)st.pages_free, (long long)st.pages_total,
         (long long)st.table_entries_written, (long long)st.chunks_live, (long long)st.kernels_launched);
  if (kam_destroy(ctx) != KAM_OK) { printf("FAIL destroy\n"); return 1; }
  printf("OK\n");
  return 0;
}

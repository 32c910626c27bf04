// kam_ctx and the helpers shared by the entry-point files.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>

#include <memory>
#include <string>
#include <vector>

#include "internal.h"
#include "window.h"

namespace kam {

struct Staging {                 // pinned host + device buffer pair, reused round-robin behind an event
  void* host = nullptr;
  void* dev = nullptr;
  size_t cap = 0;
  cudaEvent_t ev = nullptr;
  bool in_flight = false;
};
constexpr int kStagingSlots = 8;

struct TmapSet { const void* k_layers; const void* v_layers; int32_t num_pages; void* d_tmaps; uint64_t stamp; };
constexpr int kMaxTmapSets = 8;

// Tunables behind kam_set_option(ctx, key, value).  Nothing in the library reads the process environment.
struct Options {
  int reloc_stages = 0;        // "reloc_stages": pipeline stages of the relocate kernel (0 = automatic: 3)
  int reloc_hg = 0;            // "reloc_head_group": KV heads per slice (0 = automatic)
  int reloc_hg_cap = 4;        // "reloc_head_group_cap": widest slice the automatic choice tries (8-head slices measured within 2 % either way)
  int reloc_kv_split = 1;      // "reloc_kv_split": 1 = automatic (when W_k + W_v crowd out the third stage), 0 = never, 2 = always
  int reloc_contig = 1;        // "reloc_contig": one unpadded copy per tile when a slice is a whole token row
  int reloc_rb = 0;            // "reloc_row_blocks": 16-token row blocks per tile (0 = automatic)
  int reloc_load_hint = 1;     // "reloc_evict_first": canonical sources are read with an L2 evict-first hint
  int reloc_patch_cost_pct = 108;  // "reloc_patch_cost_pct": cost of a tile that runs the patch, in % of its bytes (work split)
  int reloc_pdl = 1;           // "reloc_pdl": the relocate kernel is launched with programmatic stream serialization
  int dec_ctas_per_sm = 0;     // "decode_ctas_per_sm" (0 = automatic)
  int dec_boxes = 0;           // "decode_boxes": ring depth of the decode kernel (0 = automatic)
  int use_pdl = 1;             // "decode_pdl": programmatic dependent launch between plan, decode and merge
  int dec_tma = 1;             // "decode_tma": pool pages arrive as TMA tensor-map boxes (0: per-token bulk copies)
  int prefill_tc = 1;          // "prefill_tcgen05": the multi-query readout runs on tcgen05 / tensor memory (0: the mma.sync kernel)
  int host_copy_overlap = 0;   // "host_copy_overlap": kam_relocate_patch_host copies chunk c+1 under the kernel of chunk c, on a stream
                               // of the library's own that is NOT ordered behind the caller's stream - opt-in, for host data that is final
  int host_sync = 0;           // "host_entries_sync": kam_paged_decode_merge_host ends with a stream synchronise
};

}  // namespace kam

struct kam_ctx {
  kam_layout lay;
  kam_pool pool{};
  bool has_pool = false;
  bool cuda_ok = false;
  int sm_count = 0;
  std::string err;
  int64_t kernels_launched = 0;

  // relocate
  bool fast_layout = false;
  std::string fast_layout_why;
  int blocks_per_head = 0;
  kam::Options opt;                           // kam_set_option; the defaults are the measured choices
  kam::ColBlock head_blocks[kam::kMaxColBlocks];

  kam::Staging staging[kam::kStagingSlots];
  int staging_next = 0;

  // window store
  std::unique_ptr<kam::WindowStore> win;
  int32_t max_requests = 0, max_chunks = 0, max_ppc = 0;
  int32_t* d_slot_pages = nullptr;            // device mirror [n_slots][max_ppc]

  // decode: TMA tensor maps per pool ([n_layers][K,V], 128 bytes each, device memory); entry 0 = the context's own pool
  std::vector<kam::TmapSet> tmap_sets;
  uint64_t tmap_clock = 0;
  std::string tmap_why;                        // why the TMA path is off, if it is
  // decode: workspace (grown on demand); the plan of the window store stays cached in it between layers
  void* d_ws = nullptr;                        // stateless calls
  size_t ws_cap = 0;
  bool decplan_valid = false;                  // a plan pinned by kam_paged_decode_plan sits in d_ws
  alignas(8) unsigned char decplan_key[64] = {};
  bool decplan_unread = false;                 // the pinned plan's kernel was enqueued and no decode has been launched behind it yet:
                                               // that first decode may not read the plan before griddepcontrol.wait
  bool winplan_unread = false;                 // same for the window plan (kam_window_plan followed by kam_window_decode)
  void* d_ws_win = nullptr;                    // window calls: laid out once for max_requests x max_chunks (graph-stable)
  size_t ws_win_cap = 0;
  uint64_t winplan_epoch = ~0ull;              // window epoch the plan in d_ws was built for (~0 = none)
  std::vector<int32_t> winplan_reqs;
  int32_t winplan_chunks = 0;
  double* d_inv_freq = nullptr;                // [rope_dim / 2] f_i = theta^(-2i/d_r), fp64
  kam::DecodeGeom dec_geom[2][5];              // cached geometry: [bulk-copy path | TMA path over the context's pool][patch rank tiles KT]
  bool dec_geom_ok[2][5] = {};
  int32_t dec_max_rank = KAM_MAX_RANK;         // largest rank of an on-read patch (kam_decode_set_max_patch_rank)
  int32_t* d_err = nullptr;                    // device counter: malformed kam_patch_ref records ignored by the decode kernel
  int64_t generic_launches = 0;                // launches of the element-wise fallback kernel (kam_stats.generic_launches)
  // device staging of host-resident chunks (kam_relocate_patch_host) and host-resident q/out (decode host variant)
  void* d_hstage[2] = {nullptr, nullptr};      // two buffers: the copy of one chunk overlaps the kernel that reads the other
  size_t hstage_cap[2] = {0, 0};
  int hstage_next = 0;
  bool hstage_used[2] = {false, false};
  cudaStream_t copy_stream = nullptr;          // the library's own H2D stream (kam_relocate_patch_host)
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr};
  std::vector<void*> graveyard;                // outgrown device buffers, freed by kam_destroy (see grow_device)
  void* d_hstage2 = nullptr;
  size_t hstage2_cap = 0;
  void* d_fp_ws = nullptr;                     // kam_form_patch: Delta and B workspaces (fp32)
  size_t fp_ws_cap = 0;
};

namespace kam {
kam_status fail(kam_ctx* ctx, kam_status st, const char* fmt, ...);
kam_status cuda_fail(kam_ctx* ctx, cudaError_t e, const char* what);
kam_status staging_acquire(kam_ctx* c, size_t bytes, Staging** out);
kam_status staging_commit(kam_ctx* c, Staging* s, size_t bytes, cudaStream_t st);
void staging_release(Staging* s, cudaStream_t st);
kam_status check_pool(kam_ctx* c, const kam_pool** pool);
const void* tmaps_for_pool(kam_ctx* c, const kam_pool* pool);
kam_status grow_device(kam_ctx* c, void** buf, size_t* cap, size_t bytes, const char* what, cudaStream_t st);
}  // namespace kam

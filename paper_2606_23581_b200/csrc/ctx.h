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
  bool contig_copies = true;                  // one unpadded copy per tile when a slice is a whole token row (KAM_RELOC_CONTIG=0: padded per-row copies)
  int reloc_stages = 0, reloc_load_hint = 1, reloc_rb = 0;  // tuning switches (KAM_RELOC_STAGES, KAM_RELOC_HINT, KAM_RELOC_RB)
  kam::ColBlock head_blocks[kam::kMaxColBlocks];

  kam::Staging staging[kam::kStagingSlots];
  int staging_next = 0;

  // window store
  std::unique_ptr<kam::WindowStore> win;
  int32_t max_requests = 0, max_chunks = 0, max_ppc = 0;
  int32_t* d_slot_pages = nullptr;            // device mirror [n_slots][max_ppc]

  // decode: TMA tensor maps over the context's pool ([n_layers][K,V], 128 bytes each, device memory)
  void* d_tmaps = nullptr;
  std::string tmap_why;                        // why the TMA path is off, if it is
  // decode: workspace (grown on demand); the plan of the window store stays cached in it between layers
  void* d_ws = nullptr;
  size_t ws_cap = 0;
  uint64_t winplan_epoch = ~0ull;              // window epoch the plan in d_ws was built for (~0 = none)
  std::vector<int32_t> winplan_reqs;
  int32_t winplan_chunks = 0;
  double* d_inv_freq = nullptr;                // [rope_dim / 2] f_i = theta^(-2i/d_r), fp64
  kam::DecodeGeom dec_geom[2][5];              // cached geometry: [bulk-copy path | TMA path over the context's pool][patch rank tiles KT]
  bool dec_geom_ok[2][5] = {};
  int32_t dec_max_rank = KAM_MAX_RANK;         // largest rank of an on-read patch (kam_decode_set_max_patch_rank)
  int32_t* d_err = nullptr;                    // device counter: malformed kam_patch_ref records ignored by the decode kernel
  bool use_pdl = true;                         // programmatic dependent launch between decode and merge (KAM_NO_PDL=1 turns it off)
  int dec_ctas_per_sm = 0, dec_boxes = 0;      // tuning switches (KAM_DEC_CTAS_PER_SM, KAM_DEC_BOXES); 0 = automatic
  // device staging of host-resident chunks (kam_relocate_patch_host) and host-resident q/out (decode host variant)
  void* d_hstage = nullptr;
  size_t hstage_cap = 0;
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
kam_status grow_device(kam_ctx* c, void** buf, size_t* cap, size_t bytes, const char* what);
}  // namespace kam

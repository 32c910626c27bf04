// The window store (deque of chunks per request + LIFO page free list): host-only integer bookkeeping.
// "the same store can act as a deque, evicting and admitting at either end of the window in O(1)".
// Allocation policy: DESIGN.md reading R-13.  No CUDA in this file; the device mirror is written by api.cu.
#pragma once
#include <stdint.h>

#include <deque>
#include <vector>

namespace kam {

struct ChunkRec {
  int32_t handle;
  int32_t n_tokens;
  int32_t slot;        // row of the page-list table holding this chunk's pages
  int64_t phase;       // RoPE position the chunk's keys currently sit at in the pool
};

struct Rotation { int32_t slot; int32_t n_tokens; int64_t delta; };   // survivor to re-rotate in place

class WindowStore {
 public:
  WindowStore(int32_t num_pages, int32_t page_size, int32_t max_requests, int32_t max_chunks_per_request,
              int32_t max_pages_per_chunk);

  enum Result { OK = 0, BAD_ARG, BAD_STATE, NO_PAGES };

  Result open(int32_t req, int64_t window_base);
  Result pin(int32_t req, int32_t n_front);
  Result close(int32_t req);
  // On success: *rec describes the admitted chunk (its pages are in pages_of(rec->slot)), *p_target its position,
  // rotations = survivors that must be re-rotated now (materialize) - empty when lazy.
  Result admit(int32_t req, int end, int32_t n_tokens, bool materialize, ChunkRec* rec, int64_t* p_target,
               std::vector<Rotation>* rotations);
  Result evict(int32_t req, int end, bool materialize, ChunkRec* rec, std::vector<Rotation>* rotations);
  // Would evict(req, evict_end) [skipped when evict_end < 0] followed by admit(req, admit_end, n_tokens) succeed?  Changes nothing.
  Result can_admit(int32_t req, int evict_end, int admit_end, int32_t n_tokens) const;

  bool is_open(int32_t req) const { return req >= 0 && req < (int32_t)reqs_.size() && reqs_[req].open; }
  const std::deque<ChunkRec>& chunks(int32_t req) const { return reqs_[req].chunks; }
  int64_t window_base(int32_t req) const { return reqs_[req].base; }
  const int32_t* pages_of(int32_t slot) const { return &slot_pages_[(size_t)slot * max_ppc_]; }
  int32_t max_pages_per_chunk() const { return max_ppc_; }
  int32_t page_size() const { return P_; }
  int64_t pages_free() const { return (int64_t)free_.size(); }
  int64_t pages_total() const { return num_pages_; }
  int64_t table_entries_written() const { return entries_written_; }
  int64_t chunks_live() const { return chunks_live_; }
  uint64_t epoch() const { return epoch_; }               // bumped by every successful mutation

 private:
  struct Request {
    bool open = false;
    int64_t base = 0;
    int32_t pinned = 0;
    int64_t pinned_tokens = 0, total_tokens = 0;
    std::deque<ChunkRec> chunks;
  };
  void settle(Request& r, bool materialize, std::vector<Rotation>* rotations);

  int32_t P_, num_pages_, max_chunks_, max_ppc_;
  std::vector<int32_t> free_;          // LIFO stack, top = back
  std::vector<int32_t> free_slots_;
  std::vector<int32_t> slot_pages_;    // [n_slots][max_ppc_]
  std::vector<Request> reqs_;
  int32_t next_handle_ = 0;
  int64_t entries_written_ = 0, chunks_live_ = 0;
  uint64_t epoch_ = 0;
};

}  // namespace kam

#include "window.h"

namespace kam {

WindowStore::WindowStore(int32_t num_pages, int32_t page_size, int32_t max_requests, int32_t max_chunks_per_request,
                         int32_t max_pages_per_chunk)
    : P_(page_size), num_pages_(num_pages), max_chunks_(max_chunks_per_request), max_ppc_(max_pages_per_chunk) {
  free_.reserve(num_pages);
  for (int32_t p = num_pages - 1; p >= 0; --p) free_.push_back(p);          // first pops give 0, 1, 2, ...
  const int32_t n_slots = max_requests * max_chunks_per_request;
  for (int32_t s = n_slots - 1; s >= 0; --s) free_slots_.push_back(s);
  slot_pages_.assign((size_t)n_slots * max_ppc_, -1);
  reqs_.resize(max_requests);
}

WindowStore::Result WindowStore::open(int32_t req, int64_t window_base) {
  if (req < 0 || req >= (int32_t)reqs_.size()) return BAD_ARG;
  if (reqs_[req].open) return BAD_STATE;
  reqs_[req] = Request();
  reqs_[req].open = true;
  reqs_[req].base = window_base;
  ++epoch_;
  return OK;
}

WindowStore::Result WindowStore::pin(int32_t req, int32_t n_front) {
  if (!is_open(req)) return BAD_STATE;
  Request& r = reqs_[req];
  if (n_front < 0 || n_front > (int32_t)r.chunks.size()) return BAD_ARG;
  r.pinned = n_front;
  r.pinned_tokens = 0;
  for (int32_t i = 0; i < n_front; ++i) r.pinned_tokens += r.chunks[i].n_tokens;
  ++epoch_;
  return OK;
}

WindowStore::Result WindowStore::close(int32_t req) {
  if (!is_open(req)) return BAD_STATE;
  Request& r = reqs_[req];
  for (auto it = r.chunks.rbegin(); it != r.chunks.rend(); ++it) {
    const int32_t n = it->n_tokens / P_;
    const int32_t* pg = pages_of(it->slot);
    for (int32_t i = n - 1; i >= 0; --i) free_.push_back(pg[i]);
    free_slots_.push_back(it->slot);
    --chunks_live_;
  }
  r = Request();
  ++epoch_;
  return OK;
}

// Chunks whose position no longer equals the phase their keys carry: rotate now (materialize) or leave pending.
void WindowStore::settle(Request& r, bool materialize, std::vector<Rotation>* rotations) {
  if (!materialize) return;
  int64_t pos = r.base;
  for (ChunkRec& c : r.chunks) {
    if (pos != c.phase) {
      if (rotations) rotations->push_back({c.slot, c.n_tokens, pos - c.phase});
      c.phase = pos;
    }
    pos += c.n_tokens;
  }
}

WindowStore::Result WindowStore::can_admit(int32_t req, int evict_end, int admit_end, int32_t n_tokens) const {
  if (!is_open(req)) return BAD_STATE;
  if ((admit_end != 0 && admit_end != 1) || evict_end > 1) return BAD_ARG;
  if (n_tokens <= 0 || n_tokens % P_ != 0) return BAD_ARG;
  const int32_t need = n_tokens / P_;
  if (need > max_ppc_) return BAD_ARG;
  const Request& r = reqs_[req];
  int32_t n_chunks = (int32_t)r.chunks.size(), freed = 0;
  if (evict_end >= 0) {
    if (n_chunks <= r.pinned) return BAD_STATE;
    const ChunkRec& c = (evict_end == 0) ? r.chunks[r.pinned] : r.chunks.back();
    freed = c.n_tokens / P_;
    --n_chunks;
  }
  if (n_chunks >= max_chunks_ || (free_slots_.empty() && evict_end < 0)) return BAD_STATE;
  if (need > (int32_t)free_.size() + freed) return NO_PAGES;
  return OK;
}

WindowStore::Result WindowStore::admit(int32_t req, int end, int32_t n_tokens, bool materialize, ChunkRec* rec,
                                       int64_t* p_target, std::vector<Rotation>* rotations) {
  if (!is_open(req)) return BAD_STATE;
  if (end != 0 && end != 1) return BAD_ARG;
  if (n_tokens <= 0 || n_tokens % P_ != 0) return BAD_ARG;
  const int32_t need = n_tokens / P_;
  if (need > max_ppc_) return BAD_ARG;
  Request& r = reqs_[req];
  if ((int32_t)r.chunks.size() >= max_chunks_ || free_slots_.empty()) return BAD_STATE;
  if (need > (int32_t)free_.size()) return NO_PAGES;

  ChunkRec c;
  c.handle = next_handle_++;
  c.n_tokens = n_tokens;
  c.slot = free_slots_.back();
  free_slots_.pop_back();
  int32_t* pg = &slot_pages_[(size_t)c.slot * max_ppc_];
  for (int32_t i = 0; i < need; ++i) { pg[i] = free_.back(); free_.pop_back(); }   // logical order
  entries_written_ += need;
  if (end == 0) {                                   // FRONT: just behind the pinned chunks
    c.phase = r.base + r.pinned_tokens;
    r.chunks.insert(r.chunks.begin() + r.pinned, c);
  } else {
    c.phase = r.base + r.total_tokens;
    r.chunks.push_back(c);
  }
  r.total_tokens += n_tokens;
  ++chunks_live_;
  ++epoch_;
  *rec = c;
  *p_target = c.phase;
  settle(r, materialize, rotations);
  return OK;
}

WindowStore::Result WindowStore::evict(int32_t req, int end, bool materialize, ChunkRec* rec,
                                       std::vector<Rotation>* rotations) {
  if (!is_open(req)) return BAD_STATE;
  if (end != 0 && end != 1) return BAD_ARG;
  Request& r = reqs_[req];
  if ((int32_t)r.chunks.size() <= r.pinned) return BAD_STATE;
  const size_t idx = (end == 0) ? (size_t)r.pinned : r.chunks.size() - 1;
  ChunkRec c = r.chunks[idx];
  r.chunks.erase(r.chunks.begin() + idx);
  const int32_t n = c.n_tokens / P_;
  const int32_t* pg = pages_of(c.slot);
  for (int32_t i = n - 1; i >= 0; --i) free_.push_back(pg[i]);              // reverse logical order
  free_slots_.push_back(c.slot);
  r.total_tokens -= c.n_tokens;
  --chunks_live_;
  ++epoch_;
  if (rec) *rec = c;
  settle(r, materialize, rotations);
  return OK;
}

}  // namespace kam

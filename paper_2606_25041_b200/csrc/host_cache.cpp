// host_cache.cpp - see host_cache.h.
#include "host_cache.h"

#include <algorithm>

namespace ws {

HostCache::HostCache(int32_t num_pages, int32_t page_tokens, int32_t max_sessions,
                     int32_t max_pages_per_session, int32_t max_blocks_per_session)
    : P_(page_tokens), max_pages_(max_pages_per_session), max_blocks_(max_blocks_per_session),
      sess_(max_sessions) {
  free_.resize(num_pages);
  // back() is popped first: hand pages out in increasing id order by default
  for (int32_t i = 0; i < num_pages; ++i) free_[i] = num_pages - 1 - i;
}

int32_t HostCache::open_session() {
  for (int32_t s = 0; s < (int32_t)sess_.size(); ++s) {
    if (!sess_[s].open) {
      sess_[s] = SessionState();
      sess_[s].open = true;
      return s;
    }
  }
  return -1;
}

bool HostCache::close_session(int32_t s) {
  if (!is_open(s)) return false;
  // return pages so that the lowest id is handed out first again
  for (auto it = sess_[s].pages.rbegin(); it != sess_[s].pages.rend(); ++it) release_page(*it);
  sess_[s] = SessionState();
  return true;
}

int32_t HostCache::pages_needed(int32_t s, int64_t new_tokens) const {
  int64_t need = (new_tokens + P_ - 1) / P_;
  return (int32_t)std::max<int64_t>(0, need - (int64_t)sess_[s].pages.size());
}

bool HostCache::fits(int32_t s, int64_t n, int32_t nblocks) const {
  const SessionState& st = sess_[s];
  int64_t need = (st.tokens + n + P_ - 1) / P_;
  return need <= max_pages_ && (int64_t)st.block_ends.size() + nblocks <= max_blocks_;
}

int32_t HostCache::commit_block(int32_t s, int64_t n, const uint8_t* modality) {
  SessionState& st = sess_[s];
  int32_t first_page = (int32_t)(st.tokens / P_);
  int32_t extra = pages_needed(s, st.tokens + n);
  for (int32_t i = 0; i < extra; ++i) {
    st.pages.push_back(free_.back());
    free_.pop_back();
  }
  if (modality) {
    st.modality.resize((size_t)st.tokens, 0xff);
    st.modality.insert(st.modality.end(), modality, modality + n);
  }
  st.tokens += n;
  st.block_ends.push_back(st.tokens);
  return first_page;
}

bool HostCache::truncate_blocks(int32_t s, int32_t keep_blocks) {
  if (!is_open(s)) return false;
  SessionState& st = sess_[s];
  if (keep_blocks < 0 || keep_blocks > (int32_t)st.block_ends.size()) return false;
  st.block_ends.resize(keep_blocks);
  st.tokens = keep_blocks ? st.block_ends.back() : 0;
  size_t keep_pages = (size_t)((st.tokens + P_ - 1) / P_);
  while (st.pages.size() > keep_pages) {
    release_page(st.pages.back());
    st.pages.pop_back();
  }
  if (st.modality.size() > (size_t)st.tokens) st.modality.resize((size_t)st.tokens);
  st.settled[0] = std::min(st.settled[0], st.tokens);
  st.settled[1] = std::min(st.settled[1], st.tokens);
  return true;
}

void HostCache::release_page(int32_t page) {
  if (page < owner_pages_) owner_used_[page] = 0; else free_.push_back(page);
}

bool HostCache::reserve_owner_pages(int32_t owner_pages) {
  const int32_t num_pages = (int32_t)free_.size();
  for (const auto& s : sess_) if (s.open) return false;
  // (no session open => every page is free, so free_.size() is the pool size)
  int32_t total = num_pages + owner_pages_;
  if (owner_pages < 0 || owner_pages > total) return false;
  owner_pages_ = owner_pages;
  owner_used_.assign((size_t)owner_pages, 0);
  free_.clear();
  for (int32_t i = total - 1; i >= owner_pages; --i) free_.push_back(i);
  return true;
}

bool HostCache::open_session_at(int32_t s) {
  if (s < 0 || s >= (int32_t)sess_.size() || sess_[s].open) return false;
  sess_[s] = SessionState();
  sess_[s].open = true;
  return true;
}

void HostCache::adopt(int32_t s, const int32_t* block_lens, int32_t nblocks, const int32_t* pages,
                      int32_t npages) {
  SessionState& st = sess_[s];
  note_append(s);
  for (int32_t i = 0; i < npages; ++i) {
    owner_used_[pages[i]] = 1;
    st.pages.push_back(pages[i]);
  }
  for (int32_t b = 0; b < nblocks; ++b) {
    st.tokens += block_lens[b];
    st.block_ends.push_back(st.tokens);
  }
}

void HostCache::shuffle_free(uint64_t seed) {
  // Fisher-Yates with splitmix64
  auto next = [&seed]() {
    uint64_t z = (seed += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
  };
  for (size_t i = free_.size(); i > 1; --i) {
    size_t j = (size_t)(next() % i);
    std::swap(free_[i - 1], free_[j]);
  }
}

}  // namespace ws

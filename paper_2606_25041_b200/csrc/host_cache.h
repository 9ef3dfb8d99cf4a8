// host_cache.h - host-side metadata of the paged KV cache (a1): sessions, page tables, block
// boundaries, free list.  Pure C++ (no CUDA) so it can be exercised without a GPU.
// Follows PAPER.md:29 ("one persistent interaction state"), :83 (per-unit append into the
// full-history cache) and :38/:75 ("full-history": nothing is ever evicted).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace ws {

struct SessionState {
  bool open = false;
  int64_t tokens = 0;
  std::vector<int32_t> pages;        // physical page ids, logical page i -> pages[i]
  std::vector<int64_t> block_ends;   // e_1 < ... < e_B
  std::vector<uint8_t> modality;     // per committed token (optional metadata, may be shorter)
  // settled[0] / settled[1]: committed length before the most recent / the second most recent append call
  // (or replica adoption) on this session, lowered by truncation.  Tokens below settled[1] are not written
  // by any kernel that can still be in flight when the next launch starts (PDL protocol, launch.h).
  int64_t settled[2] = {0, 0};
};

class HostCache {
 public:
  HostCache(int32_t num_pages, int32_t page_tokens, int32_t max_sessions,
            int32_t max_pages_per_session, int32_t max_blocks_per_session);

  int32_t open_session();                         // -1 if no slot is free
  bool close_session(int32_t s);
  bool is_open(int32_t s) const { return s >= 0 && s < (int32_t)sess_.size() && sess_[s].open; }
  const SessionState& session(int32_t s) const { return sess_[s]; }

  // Pages a session needs in addition to what it holds to reach `new_tokens` committed tokens.
  int32_t pages_needed(int32_t s, int64_t new_tokens) const;
  // Whether appending n tokens as `nblocks` blocks fits the per-session capacities (pages, blocks).
  bool fits(int32_t s, int64_t n, int32_t nblocks = 1) const;
  // Commit a block of n tokens (caller has checked free pages / capacity).  Returns index of the
  // first logical page touched by the new tokens.
  int32_t commit_block(int32_t s, int64_t n, const uint8_t* modality);
  bool truncate_blocks(int32_t s, int32_t keep_blocks);
  // Once per append call (or adoption) and session, BEFORE its blocks are committed.
  void note_append(int32_t s) {
    sess_[s].settled[1] = sess_[s].settled[0];
    sess_[s].settled[0] = sess_[s].tokens;
  }

  // ---- NEXT-3 replica side: pages [0, owner_pages) are handed out only by adopt()
  // (the owner of the link names them); local appends draw from the rest.
  bool reserve_owner_pages(int32_t owner_pages);   // false if a session is open or out of range
  int32_t owner_pages() const { return owner_pages_; }
  bool owner_page_free(int32_t page) const {
    return page >= 0 && page < owner_pages_ && !owner_used_[page];
  }
  bool open_session_at(int32_t s);                 // open a specific slot (false if taken / invalid)
  // Adopt `pages` (all owner_page_free) as the next logical pages of session s and commit the blocks
  // whose lengths are given.  The caller has validated everything (strong guarantee lives in api.cu).
  void adopt(int32_t s, const int32_t* block_lens, int32_t nblocks, const int32_t* pages, int32_t npages);

  int32_t free_pages() const { return (int32_t)free_.size(); }
  void shuffle_free(uint64_t seed);
  int32_t page_tokens() const { return P_; }
  int32_t max_pages_per_session() const { return max_pages_; }
  int32_t max_sessions() const { return (int32_t)sess_.size(); }
  int32_t max_blocks_per_session() const { return max_blocks_; }

 private:
  void release_page(int32_t page);
  int32_t P_, max_pages_, max_blocks_;
  int32_t owner_pages_ = 0;
  std::vector<uint8_t> owner_used_;  // [owner_pages_]
  std::vector<SessionState> sess_;
  std::vector<int32_t> free_;        // stack: back() is handed out next
};

}  // namespace ws

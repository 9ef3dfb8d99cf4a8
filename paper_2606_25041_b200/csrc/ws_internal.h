// ws_internal.h - structures shared by the host planner and the kernels (never exported).
#pragma once
#include <stdint.h>

namespace ws {

constexpr int kTileKeys = 128;    // keys per KV tile of the tensor-core kernel
constexpr int kTileRows = 128;    // packed (token, q-head-in-group) rows per Q tile (UMMA M)
constexpr int kPairRows = 256;    // one CTA processes a pair of Q tiles that share K/V tiles
constexpr int kMaxTeam = 8;       // max row-tile pairs of one (session, KV head) group per team

// One (session, KV head, sub-range of the session's query tokens): all of its row-tile pairs share
// the same K/V stream, so the CTAs of one team walk the same KV tiles in lock-step (L2 reuse).
// Small per-call metadata travels in the kernel parameters instead of a host->device copy (keeps the
// append -> attention -> combine chain free of stream operations between the kernels, which is what
// lets programmatic dependent launch overlap them).  Larger blobs go through the workspace ring.
// Two tiers for the attention blob: the small one keeps the launch of the common single-session step
// light; the large one (CUDA >= 12.1 allows 32,764 B of kernel parameters on sm_70+) covers many-group
// plans (MHA with 16+ heads, ragged multi-session batches) so that those steps, too, need no
// host->device copy and stay CUDA-graph capturable.
constexpr int kInlineAttnWords = 1000;
constexpr int kInlineAttnWordsLarge = 6800;
constexpr int kInlineAppendWords = 960;
template <int W> struct InlineMeta { int32_t w[W]; };
using InlineAttnMeta = InlineMeta<kInlineAttnWords>;
using InlineAttnMetaLarge = InlineMeta<kInlineAttnWordsLarge>;
using InlineAppendMeta = InlineMeta<kInlineAppendWords>;

#ifdef __CUDACC__
// Reads of the metadata blob.  When the blob travels in the kernel parameters, indexing the parameter
// itself compiles to constant-bank loads (LDC, tens of cycles); going through a generic pointer to it
// costs a global-memory-like round trip per dependent read (measured ~1.4 us for an 8-entry scan).
template <int W> struct MetaView {
  const int32_t* g;              // device blob, or nullptr: use the kernel parameter
  const InlineMeta<W>& inl;
  __device__ __forceinline__ int32_t operator[](int32_t i) const { return g ? __ldg(g + i) : inl.w[i]; }
  template <typename T> __device__ __forceinline__ T load(int32_t word) const {
    static_assert(sizeof(T) % 4 == 0, "word-sized structs");
    T t;
    int32_t* d = reinterpret_cast<int32_t*>(&t);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(T) / 4); ++k) d[k] = (*this)[word + k];
    return t;
  }
};
#endif

struct Group {
  int32_t q_token0;      // first global query token (row of q/out) covered by this group
  int32_t q_token_end;   // end (exclusive) of the session's query tokens: rows beyond are not stored
  int32_t kv_head;
  int32_t slot;          // session slot = row of the device page table
  int32_t kv_len;        // keys visible to the LAST row of the group (= max visible end)
  int32_t npairs;        // row-tile pairs in this group (<= team size)
  int32_t vis_off;       // >= 0: per-token visible ends at vis_end[vis_off + (token - q_token0)]
  // Key sources.  Keys [0, cache_len) are read from the paged pool: KV tiles [0, Tc), Tc =
  // ceil(cache_len / 128).  Keys [cache_len, kv_len) - the block a fused step (ws_stream_step) is
  // committing in the same launch - are read straight from the caller's k_new / v_new, rows new_tok0 ..:
  // KV tiles [Tc, Tc + ceil((kv_len - cache_len) / 128)).  Outside fused steps cache_len == kv_len.
  int32_t cache_len;
  int32_t new_tok0;
  // KV tiles [0, stable_tiles) of the pool part were committed at least two append calls ago: no kernel
  // that can still be in flight when this launch starts writes them (PDL protocol, launch.h), so the TMA
  // producer may fetch them BEFORE griddepcontrol.wait.
  int32_t stable_tiles;
  // >= 0: text-causal mixed mask (NEXT-4, reading A19): word offset in the blob of this session's
  // record {abs_pos0, nbits, bits...}: bit k set <=> the token at absolute position abs_pos0 + k is a text
  // token; abs_pos0 = position of the session's first query token (row new_tok0 of q).  -1: plain block-causal.
  int32_t txt_off;
  int32_t pad;
};

// A contiguous KV-tile range of one group, processed by one team (CTA p handles pair p).
struct Segment {
  int32_t group;
  int32_t tile_begin;
  int32_t tile_end;      // exclusive; tiles are kTileKeys keys
  int32_t part_base;     // >= 0: partial slot of pair p is part_base + p; -1: write the final output
};

struct CombineItem {
  int32_t group;
  int32_t part_base;     // slot(i, p) = part_base + i * npairs + p
  int32_t nparts;
  int32_t pad;
};

// Header of the per-call metadata blob (all offsets in int32 words from the blob start).
struct AttnMeta {
  int32_t num_teams, team_size, num_groups, num_segments;
  int32_t num_combine, has_vis, off_groups, off_team_seg_begin;
  int32_t off_segments, off_combine, off_vis, total_words;
  int32_t alt;           // 1: decode plan (every group has <= kTileRows packed rows), see plan.h
  int32_t pad[3];
};

// Append metadata: per session in the call.
struct AppendSession {
  int32_t slot;          // page-table row
  int32_t len_old;       // committed tokens before this append
  int32_t tok_begin;     // cu[s]
  int32_t tok_end;       // cu[s+1]
  int32_t page_off;      // offset into the pages[] list of the blob: ids of the pages covering
                         // logical page indices [len_old / P, ceil(len_new / P))
  int32_t pad[3];
};
struct AppendMeta {
  int32_t num_sessions, total_tokens, off_sessions, off_pages;
};

// NEXT-3: pools of the linked replicas as mapped on this device (16-byte words); n = 0: none.
constexpr int kMaxPeers = 4;
struct PeerPools {
  void* k[kMaxPeers];
  void* v[kMaxPeers];
  int32_t n;
  int32_t pad;
};

// Parameters common to the attention kernels.
struct AttnParams {
  const void* q; void* out; float* lse;
  const void* k_pool; const void* v_pool;
  const int32_t* page_table;   // [max_sessions][max_pages_per_session]
  const int32_t* meta;         // AttnMeta blob (device)
  float* part_o;               // [slots][kPairRows][D] fp32, normalised partial outputs
  float* part_lse;             // [slots][kPairRows] fp32, log2-domain LSE (-inf = empty)
  int32_t max_pages_per_session;
  int32_t Hq, Hkv, D, G, P;
  int32_t total_q_tokens;
  float scale;
  // fused step (ws_stream_step): warp 11 of every CTA commits its share of the new block (same code as
  // kv_append_kernel, metadata in the `app` kernel parameter).  0: no append in this launch.
  const void* k_new; const void* v_new;
  void* k_pool_w; void* v_pool_w; int32_t* page_table_w;
  int32_t append_tokens;
  int32_t pad_a;
  // fused combine (a4 inside the attention kernel): arrival counters [max_part_slots] followed by
  // completion counters [max_part_slots], indexed by the first partial slot of a (combine item, pair);
  // all zero between launches (the last merging warp of an item resets them).  nullptr: the partials
  // are merged by combine_kernel instead.
  int32_t* merge_ctr;
  int32_t max_part_slots;
  int32_t pad_;
};

}  // namespace ws

// plan.h - a1: the ragged multi-session split-KV scheduler (host side, pure C++).
// north_star: "a ragged multi-session scheduler that splits long caches across CTAs with a split-KV
// combine kernel".  The paper itself is silent on scheduling (PAPER.md:83 only states the append).
#pragma once
#include <cstdint>
#include <vector>

#include "ws_internal.h"

namespace ws {

struct PlanSession {
  int32_t slot;          // session slot (page-table row)
  int32_t q_begin;       // first global query token of this session in the call
  int32_t q_end;         // exclusive
  bool multi_block;      // queries span more than one block (per-token visible ends differ)
  int32_t new_len;       // fused step: the last `new_len` visible keys are read from k_new / v_new (rows
                         // q_begin ..) instead of the pool; 0 otherwise (and whenever multi_block)
  int32_t stable_len;    // tokens committed at least two append calls ago (Group::stable_tiles)
  int32_t txt_off;       // Group::txt_off (-1: none); offsets are relative to the start of the `extra` words
};

struct PlanConfig {
  int32_t Hkv, G;        // KV heads, q heads per KV head
  int32_t num_sms;       // CTAs that can be resident at once (1 CTA / SM)
  int32_t min_tiles;     // do not cut the work finer than this many KV tiles per segment
  float seg_overhead_tiles;  // cost of starting one more segment in a team, in KV-tile units
  int32_t min_splits;    // debug: force at least this many segments per group (0 = automatic)
  int32_t max_part_slots;
  bool allow_alt;        // permit the decode plan (below) when every session qualifies
};

// Decode plan ("alt", NEXT-4: n*G <= 128 packed rows per (session, KV head), e.g. token-causal text
// decode).  Such a step is cache-read bound (n*G FLOP/B << ridge): one 128-row Q tile per
// CTA, run by attn_dec_sm100_kernel (both softmax warpgroups on every KV tile, one O accumulator, six ring
// slots).  Groups, segments, partial slots and the combine are those of the general plan; a partial has
// 128 rows in use.
struct Plan {
  bool alt = false;
  int32_t team_size = 1, num_teams = 0, total_tiles = 0, num_part_slots = 0;
  std::vector<Group> groups;
  std::vector<int32_t> team_seg_begin;   // [num_teams + 1]
  std::vector<Segment> segments;         // ordered by team, then by walk order
  std::vector<int32_t> seg_team;         // team of each segment (introspection)
  std::vector<CombineItem> combine;
  bool ok = true;                        // false: partial slots exceed max_part_slots
};

// vis_end[t] for every global query token t (keys j < vis_end[t] are visible to token t).
Plan build_plan(const PlanConfig& cfg, const std::vector<PlanSession>& sessions,
                const std::vector<int32_t>& vis_end);

// Serialise into the device blob layout described by AttnMeta (ws_internal.h).
// `extra`: words appended after the visible ends (text-bit records of the mixed mask); every group's
// txt_off >= 0 is rebased to the blob offset of extra[0].
std::vector<int32_t> serialise_plan(const Plan& plan, const std::vector<int32_t>& vis_end,
                                    bool has_vis, const std::vector<int32_t>& extra = std::vector<int32_t>());

}  // namespace ws

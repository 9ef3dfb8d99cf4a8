// plan.cpp - see plan.h.
//
// Work decomposition.  A *group* is one (session, KV head, run of <= team_size row-tile pairs of
// the session's packed query rows); every pair of a group streams the same K/V tiles.  The KV-tile
// axes of all groups are concatenated into one flat axis of `total_tiles` tiles, which is cut into
// `num_teams` equal ranges (stream-K style): team i owns flat tiles [i*T/n, (i+1)*T/n).  A team is
// `team_size` CTAs launched with adjacent block ids; CTA p of the team processes pair p of whatever
// group the team's range currently lies in, so the CTAs that share K/V tiles read them at the same
// time and all but the first read hit in L2.  A range that covers only part of a group's tiles
// yields a *partial* (normalised fp32 O + LSE) per pair; the combine kernel (a4) merges them.
#include "plan.h"

#include <algorithm>

namespace ws {

Plan build_plan(const PlanConfig& cfg, const std::vector<PlanSession>& sessions,
                const std::vector<int32_t>& vis_end) {
  Plan plan;
  const int32_t tok_per_pair = kPairRows / cfg.G;
  int32_t max_pairs = 1;
  for (const PlanSession& s : sessions) {
    int32_t nq = s.q_end - s.q_begin;
    max_pairs = std::max(max_pairs, (nq + tok_per_pair - 1) / tok_per_pair);
  }
  plan.team_size = std::min<int32_t>(kMaxTeam, max_pairs);
  const int32_t Pt = plan.team_size;
  plan.alt = cfg.allow_alt;
  for (const PlanSession& s : sessions)
    if ((int64_t)(s.q_end - s.q_begin) * cfg.G > kTileRows) plan.alt = false;

  std::vector<int32_t> group_tiles;
  {
    size_t ng = 0;
    for (const PlanSession& s : sessions) ng += (size_t)cfg.Hkv * (((s.q_end - s.q_begin + tok_per_pair - 1) / tok_per_pair + Pt - 1) / Pt);
    plan.groups.reserve(ng); group_tiles.reserve(ng);
  }
  for (const PlanSession& s : sessions) {
    int32_t nq = s.q_end - s.q_begin;
    int32_t pairs = (nq + tok_per_pair - 1) / tok_per_pair;
    for (int32_t h = 0; h < cfg.Hkv; ++h) {
      for (int32_t b = 0; b < pairs; b += Pt) {
        Group g{};
        g.q_token0 = s.q_begin + b * tok_per_pair;
        g.q_token_end = s.q_end;
        g.kv_head = h;
        g.slot = s.slot;
        g.npairs = std::min(Pt, pairs - b);
        int32_t last_tok = std::min(s.q_end, g.q_token0 + g.npairs * tok_per_pair) - 1;
        g.kv_len = vis_end[last_tok];
        g.vis_off = s.multi_block ? g.q_token0 : -1;
        const int32_t new_len = s.multi_block ? 0 : std::min(s.new_len, g.kv_len);
        g.cache_len = g.kv_len - new_len;
        g.new_tok0 = s.q_begin;
        g.stable_tiles = std::min(s.stable_len, g.cache_len) / kTileKeys;
        g.txt_off = s.txt_off;
        plan.groups.push_back(g);
        int32_t nt = (g.cache_len + kTileKeys - 1) / kTileKeys + (new_len + kTileKeys - 1) / kTileKeys;
        group_tiles.push_back(nt);
        plan.total_tiles += nt;
      }
    }
  }
  const int64_t T = plan.total_tiles;
  int32_t teams_avail = std::max(1, cfg.num_sms / Pt);
  int32_t min_tiles = std::max(1, cfg.min_tiles);
  int32_t n_used = (int32_t)std::min<int64_t>(teams_avail, std::max<int64_t>(1, T / min_tiles));
  plan.num_teams = n_used;

  // Walk the flat tile axis; cut at team boundaries (and at forced split boundaries).  A team that
  // continues into another group pays a fixed cost for the extra segment (Q reload, pipeline
  // refill, epilogue), measured at ~3.3 KV tiles on B200: budgets are equalised in cost units.
  const double ovh = cfg.seg_overhead_tiles;
  // Greedy walk with a per-team budget B: a team takes tiles until its cost (tiles + ovh per extra
  // segment) would exceed B; the last team takes whatever is left.  The smallest B for which the last
  // team also stays within B minimises the maximum team cost - found by bisection.  (A fixed budget of
  // total/teams leaves the last team with the sum of every team's rounding remainder: 63 tiles against
  // an average of 7 on a 16-head MHA step; carrying the remainder forward instead overloads the teams
  // that follow a group boundary.)
  auto walk = [&](double B, bool emit) -> double {
    int32_t team = 0;
    double used = 0.0, worst = 0.0;
    if (emit) { plan.segments.clear(); plan.seg_team.clear(); }
    for (size_t gi = 0; gi < plan.groups.size(); ++gi) {
      const int32_t nt = group_tiles[gi];
      const int32_t per = cfg.min_splits > 0 ? std::max(1, (nt + cfg.min_splits - 1) / cfg.min_splits) : nt;
      int32_t t = 0;
      while (t < nt) {
        if (!emit && used == 0.0 && per == nt) {
          // fast-forward (feasibility walks only): every fresh team inside this group takes floor(B)
          // tiles and then cannot afford another segment - skip them arithmetically
          const int64_t full = (int64_t)(B + 1e-6);
          const int64_t k = std::min<int64_t>((nt - t) / full, (int64_t)n_used - 1 - team);
          if (full >= 1 && k > 0) {
            worst = std::max(worst, (double)full);
            team += (int32_t)k;
            t += (int32_t)(k * full);
            continue;
          }
        }
        const bool last_team = team + 1 >= n_used;
        const double seg_cost0 = (used > 0.0) ? ovh : 0.0;   // not the team's first segment
        int64_t room = (int64_t)(B - used - seg_cost0 + 1e-6);
        if (!last_team && room < 1) { worst = std::max(worst, used); ++team; used = 0.0; continue; }
        if (last_team) room = nt - t;
        int32_t take = (int32_t)std::min<int64_t>(room, nt - t);
        take = std::min(take, per - (t % per));
        if (emit) {
          plan.segments.push_back(Segment{(int32_t)gi, t, t + take, -1});
          plan.seg_team.push_back(team);
        }
        used += seg_cost0 + take;
        t += take;
      }
    }
    return std::max(worst, used);
  };
  // lo = T / teams is a lower bound of the optimum; grow the bracket geometrically until the walk fits,
  // then bisect it to a quarter tile (5-8 walks in practice; this runs on the host once per call)
  double lo = std::max(1.0, (double)T / n_used), hi = lo;
  if (walk(lo, false) > lo + 1e-9) {
    double step = 1.0;
    for (;;) {
      hi = lo + step;
      if (walk(hi, false) <= hi + 1e-9) break;
      lo = hi; step *= 2.0;
    }
    while (hi - lo > 0.25) {
      const double mid = 0.5 * (lo + hi);
      if (walk(mid, false) <= mid + 1e-9) hi = mid; else lo = mid;
    }
  }
  plan.segments.reserve(plan.groups.size() + 2 * (size_t)n_used);
  plan.seg_team.reserve(plan.groups.size() + 2 * (size_t)n_used);
  walk(hi, true);
  const int32_t team = plan.seg_team.empty() ? 0 : plan.seg_team.back();
  plan.num_teams = team + 1;
  // partial slots: only groups cut into more than one segment need them
  size_t i = 0;
  while (i < plan.segments.size()) {
    size_t j = i;
    while (j < plan.segments.size() && plan.segments[j].group == plan.segments[i].group) ++j;
    if (j - i > 1) {
      const Group& g = plan.groups[plan.segments[i].group];
      CombineItem c{plan.segments[i].group, plan.num_part_slots, (int32_t)(j - i), 0};
      for (size_t k = i; k < j; ++k) {
        plan.segments[k].part_base = plan.num_part_slots;
        plan.num_part_slots += g.npairs;
      }
      plan.combine.push_back(c);
    }
    i = j;
  }
  plan.team_seg_begin.assign(plan.num_teams + 1, 0);
  for (int32_t tm : plan.seg_team) plan.team_seg_begin[tm + 1]++;
  for (int32_t k = 0; k < plan.num_teams; ++k) plan.team_seg_begin[k + 1] += plan.team_seg_begin[k];
  plan.ok = plan.num_part_slots <= cfg.max_part_slots;
  return plan;
}

std::vector<int32_t> serialise_plan(const Plan& plan, const std::vector<int32_t>& vis_end,
                                    bool has_vis, const std::vector<int32_t>& extra) {
  static_assert(sizeof(Group) == 48 && sizeof(Segment) == 16 && sizeof(CombineItem) == 16 &&
                sizeof(AttnMeta) == 64, "blob layout");
  AttnMeta m{};
  m.num_teams = plan.num_teams;
  m.team_size = plan.team_size;
  m.num_groups = (int32_t)plan.groups.size();
  m.num_segments = (int32_t)plan.segments.size();
  m.num_combine = (int32_t)plan.combine.size();
  m.has_vis = has_vis ? 1 : 0;
  m.alt = plan.alt ? 1 : 0;
  int32_t off = sizeof(AttnMeta) / 4;
  m.off_groups = off;            off += m.num_groups * (int32_t)(sizeof(Group) / 4);
  m.off_team_seg_begin = off;    off += plan.num_teams + 1;
  off = (off + 3) & ~3;
  m.off_segments = off;          off += m.num_segments * (int32_t)(sizeof(Segment) / 4);
  m.off_combine = off;           off += m.num_combine * (int32_t)(sizeof(CombineItem) / 4);
  m.off_vis = off;               off += has_vis ? (int32_t)vis_end.size() : 0;
  const int32_t off_extra = off; off += (int32_t)extra.size();
  off = (off + 3) & ~3;
  m.total_words = off;
  std::vector<int32_t> blob(off, 0);
  auto put = [&](int32_t at, const void* src, size_t bytes) {
    if (bytes) std::copy((const char*)src, (const char*)src + bytes, (char*)(blob.data() + at));
  };
  put(0, &m, sizeof(m));
  put(m.off_groups, plan.groups.data(), plan.groups.size() * sizeof(Group));
  if (!extra.empty()) {
    put(off_extra, extra.data(), extra.size() * 4);
    for (size_t gi = 0; gi < plan.groups.size(); ++gi)
      if (plan.groups[gi].txt_off >= 0)
        reinterpret_cast<Group*>(blob.data() + m.off_groups)[gi].txt_off += off_extra;
  }
  put(m.off_team_seg_begin, plan.team_seg_begin.data(), plan.team_seg_begin.size() * 4);
  put(m.off_segments, plan.segments.data(), plan.segments.size() * sizeof(Segment));
  put(m.off_combine, plan.combine.data(), plan.combine.size() * sizeof(CombineItem));
  if (has_vis) put(m.off_vis, vis_end.data(), vis_end.size() * 4);
  return blob;
}

}  // namespace ws

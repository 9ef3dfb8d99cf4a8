// attn_dec_sm100.cu - a3 on sm_100a, DECODE kernel: block-causal attention for steps with at most 128 packed
// query rows per (session, KV head) - token-causal text decode, n * Hq/Hkv <= 128 ("short
// token-causal Transformer pass", :77 "token-causal decoding over the language and state slots").
//
// Such a step is cache-read bound (HBM needs ~1400 cycles per 128-key tile and SM).  With one softmax warpgroup
// per tile (round 1: two accumulator sets of the general kernel on alternate tiles) a tile costs ~2300 cycles: the
// chain S -> softmax (~1500 cycles, 128 keys per thread) -> PV -> next S of a set is pure latency, and two sets
// do not hide it.  Here BOTH warpgroups work on EVERY tile, 64 of its 128 keys each
// (thread = row, as before): softmax latency per tile halves, S is double-buffered by tile parity, and there is
// ONE O accumulator.  The two halves of a row share its softmax reference: the optimistic pass never changes it,
// and the (rare) exact path agrees on it through shared memory; which path a tile takes is decided for the whole
// CTA by one predicate-reducing barrier.
//
// Same plan, metadata, K/V ring order (K0 K1 | V0 K2 | V1 K3 ...), append warps, partial format and combine
// kernels as attn_sm100.cu's decode plan.  No in-kernel merge phase (WS_FLAG_FUSED_COMBINE keeps the old plan).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <string.h>

#include "kv_append.cuh"
#include "launch.h"
#include "sm100_ptx.cuh"
#include "softmax_chunk.cuh"
#include "merge.cuh"

namespace ws {

using namespace ptx;

namespace dec {

constexpr int kStages = 6;                                 // one Q tile leaves room for six 32 KB K/V slots
constexpr uint32_t kSlotBytes = 32768, kHalfBytes = 16384, kQTileBytes = 32768;
constexpr int kThreads = 384;
constexpr uint32_t kTmemCols = 512;                        // S0 S1 (by tile parity; P aliases S), O
constexpr float kFastSumLimit = 1024.0f;                   // as in attn_sm100.cu
constexpr int kExactFirstTiles = 2;

struct Barriers {
  uint64_t q_full, q_empty;
  uint64_t kv_full[kStages], kv_empty[kStages];
  uint64_t s_full[2], p_full[2][2], pv_done[2], o_full, o_empty;
  alignas(16) float xch[2][kTileRows];                     // per warpgroup and row: tile maximum / partial row sum
  uint32_t tmem_base;
  uint32_t pad[3];
};
constexpr uint32_t kSmemBytes = kQTileBytes + kStages * kSlotBytes + sizeof(Barriers) + 1024;
static_assert(kSmemBytes <= 232448, "227 KB of shared memory per CTA");

struct SegView {
  Group g;
  int32_t tile_begin, tile_end, part_base;
};

template <int W>
__device__ __forceinline__ void load_segment(const MetaView<W>& meta, const AttnMeta& hdr, int32_t si, SegView& v) {
  const Segment s = meta.template load<Segment>(hdr.off_segments + si * (int32_t)(sizeof(Segment) / 4));
  v.g = meta.template load<Group>(hdr.off_groups + s.group * (int32_t)(sizeof(Group) / 4));
  v.tile_begin = s.tile_begin; v.tile_end = s.tile_end; v.part_base = s.part_base;
  if (v.g.vis_off >= 0) {                                  // multi-block query: clip at the last row's visible end
    const int32_t kv = meta[hdr.off_vis + v.g.vis_off + (v.g.q_token_end - 1 - v.g.q_token0)];
    v.tile_end = min(v.tile_end, (kv + kTileKeys - 1) / kTileKeys);
  }
}

// barrier over the 256 softmax threads that also ORs a predicate over them
__device__ __forceinline__ bool bar_or_256(bool pred) {
  int out;
  asm volatile("{\n\t.reg .pred p, o;\n\tsetp.ne.b32 p, %1, 0;\n\tbarrier.cta.red.or.pred.aligned o, 1, 256, p;\n\t"
               "selp.b32 %0, 1, 0, o;\n\t}" : "=r"(out) : "r"((int)pred) : "memory");
  return out != 0;
}

}  // namespace dec

template <int kInlW>
__global__ void __launch_bounds__(dec::kThreads, 1)
attn_dec_sm100_kernel(const __grid_constant__ CUtensorMap tmap_q,
                      const __grid_constant__ CUtensorMap tmap_k,
                      const __grid_constant__ CUtensorMap tmap_v,
                      const __grid_constant__ CUtensorMap tmap_kn,
                      const __grid_constant__ CUtensorMap tmap_vn,
                      const __grid_constant__ InlineMeta<kInlW> inl,
                      const __grid_constant__ InlineAppendMeta app, const __grid_constant__ PeerPools peers,
                      const AttnParams p_in) {
  using namespace dec;
  AttnParams p = p_in;
  if (p.meta != nullptr) pdl_wait();
  const MetaView<kInlW> meta{p.meta, inl};
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base;
  const uint32_t sRing = smem_base + kQTileBytes;
  Barriers* bars = reinterpret_cast<Barriers*>(smem_raw + (smem_base - smem_u32(smem_raw)) + kQTileBytes +
                                               kStages * kSlotBytes);
  const uint32_t bq_full = smem_u32(&bars->q_full), bq_empty = smem_u32(&bars->q_empty);
  auto bkv_full = [&](int s) { return smem_u32(&bars->kv_full[s]); };
  auto bkv_empty = [&](int s) { return smem_u32(&bars->kv_empty[s]); };
  auto bs_full = [&](int b) { return smem_u32(&bars->s_full[b]); };
  auto bp_full = [&](int b, int h) { return smem_u32(&bars->p_full[b][h]); };
  auto bpv_done = [&](int b) { return smem_u32(&bars->pv_done[b]); };
  const uint32_t bo_full = smem_u32(&bars->o_full), bo_empty = smem_u32(&bars->o_empty);

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const AttnMeta hdr = meta.template load<AttnMeta>(0);
  const int32_t team = blockIdx.x;                           // decode plans have one CTA per team
  const int32_t seg_lo = meta[hdr.off_team_seg_begin + team], seg_hi = meta[hdr.off_team_seg_begin + team + 1];

  if (warp == 8 && lane == 0) {
    mbar_init(bq_full, 1); mbar_init(bq_empty, 1);
    for (int s = 0; s < kStages; ++s) { mbar_init(bkv_full(s), 1); mbar_init(bkv_empty(s), 1); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bs_full(b), 1); mbar_init(bp_full(b, 0), 128); mbar_init(bp_full(b, 1), 128); mbar_init(bpv_done(b), 1);
    }
    mbar_init(bo_full, 1); mbar_init(bo_empty, 256);
    fence_mbar_init();
    fence_proxy_async_smem();
    prefetch_tmap(&tmap_q); prefetch_tmap(&tmap_k); prefetch_tmap(&tmap_v);
    if (p.append_tokens > 0) { prefetch_tmap(&tmap_kn); prefetch_tmap(&tmap_vn); }
  }
  if (warp == 10) { tmem_alloc<kTmemCols>(smem_u32(&bars->tmem_base)); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;

  if (warp >= 8) {
    setmaxnreg_dec<88>();
    if (warp == 8 && lane == 0) {
      // ===================================================== TMA producer (protocol: attn_sm100.cu / launch.h)
      uint32_t ring_it = 0, q_it = 0;
      bool waited = false, first = true;
      auto ensure_wait = [&]() {
        if (!waited) { pdl_wait(); pdl_launch_dependents(); waited = true; }
      };
      for (int32_t si = seg_lo; si < seg_hi; ++si) {
        SegView sv;
        load_segment(meta, hdr, si, sv);
        if (sv.tile_end <= sv.tile_begin) continue;
        const int32_t* page_row = p.page_table + (int64_t)sv.g.slot * p.max_pages_per_session;
        const int32_t last_page = (sv.g.cache_len - 1) / p.P;
        const int32_t Tc = (sv.g.cache_len + kTileKeys - 1) / kTileKeys;
        const int32_t nt = sv.tile_end - sv.tile_begin;
        int32_t nk = 0, nv = 0;
        bool q_pending = true;
        for (;;) {                                           // K0 K1 | V0 K2 | V1 K3 | ... (consumption order)
          const bool is_v = !(nk < nt && nk < nv + 2);
          const int32_t j = sv.tile_begin + (is_v ? nv : nk);
          const bool at_end = nv >= nt;
          if (q_pending && !(first && !waited && !at_end && j < sv.g.stable_tiles && ring_it < (uint32_t)kStages)) {
            ensure_wait();
            if (!first) mbar_wait(bq_empty, (q_it & 1) ^ 1);
            mbar_arrive_expect_tx(bq_full, kQTileBytes);
            for (int h = 0; h < 2; ++h)
              tma_load_3d(sQ + h * kHalfBytes, &tmap_q, bq_full, h * 64, sv.g.kv_head * p.G, sv.g.q_token0);
            q_pending = false;
          }
          if (at_end) break;
          const int32_t c0 = j < Tc ? page_row[min(2 * j, last_page)] : 0;
          const int32_t c1 = j < Tc ? page_row[min(2 * j + 1, last_page)] : 0;
          const uint32_t slot = ring_it % kStages, par = (ring_it / kStages) & 1;
          mbar_wait(bkv_empty(slot), par ^ 1);
          mbar_arrive_expect_tx(bkv_full(slot), kSlotBytes);
          const uint32_t dst = sRing + slot * kSlotBytes;
          if (j < Tc) {
            const CUtensorMap* tm = is_v ? &tmap_v : &tmap_k;
            tma_load_4d(dst, tm, bkv_full(slot), 0, 0, sv.g.kv_head, c0);
            tma_load_4d(dst + kHalfBytes / 2, tm, bkv_full(slot), 0, 0, sv.g.kv_head, c1);
            tma_load_4d(dst + kHalfBytes, tm, bkv_full(slot), 64, 0, sv.g.kv_head, c0);
            tma_load_4d(dst + kHalfBytes + kHalfBytes / 2, tm, bkv_full(slot), 64, 0, sv.g.kv_head, c1);
          } else {
            const CUtensorMap* tm = is_v ? &tmap_vn : &tmap_kn;
            const int32_t tok = sv.g.new_tok0 + (j - Tc) * kTileKeys;
            tma_load_3d(dst, tm, bkv_full(slot), 0, sv.g.kv_head, tok);
            tma_load_3d(dst + kHalfBytes / 2, tm, bkv_full(slot), 0, sv.g.kv_head, tok + 64);
            tma_load_3d(dst + kHalfBytes, tm, bkv_full(slot), 64, sv.g.kv_head, tok);
            tma_load_3d(dst + kHalfBytes + kHalfBytes / 2, tm, bkv_full(slot), 64, sv.g.kv_head, tok + 64);
          }
          ++ring_it;
          if (is_v) ++nv; else ++nk;
        }
        ++q_it;
        first = false;
      }
      ensure_wait();
    } else if (warp == 9) {
      // ===================================================== MMA issuer
      const bool leader = elect_one();
      constexpr uint32_t idesc_qk = make_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc_bf16(128, 128, 0, 1);
      const uint64_t desc_k = make_smem_desc_sw128(0, 16, 1024);          // K-major operands (Q, K)
      const uint64_t desc_v = make_smem_desc_sw128(0, kHalfBytes, 1024);  // MN-major operand (V)
      uint32_t ring_it = 0, q_it = 0, seg_it = 0, tiles0 = 0, tiles1 = 0;
      auto issue_S = [&](int b, uint32_t slot) {              // S_b = Q K^T (tile parity b)
        const uint64_t da = desc_k + ((sQ & 0x3FFFFu) >> 4);
        const uint64_t db = desc_k + (((sRing + slot * kSlotBytes) & 0x3FFFFu) >> 4);   // (mask: see kDescAddrMask in attn_sm100.cu)
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          const uint32_t off = ((ks >> 2) * kHalfBytes + (ks & 3) * 32) >> 4;
          mma_ss(tmem_base + b * 128, da + off, db + off, idesc_qk, ks > 0);
        }
      };
      // O += P V for the 64 keys of warpgroup `half`: its P (bf16 pairs) sits in the first 32 columns of its own
      // half of S_b
      auto issue_PV = [&](int b, uint32_t slot, int half, bool accumulate) {
        const uint64_t db = desc_v + (((sRing + slot * kSlotBytes) & 0x3FFFFu) >> 4);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int ks = half * 4 + i;
          mma_ts(tmem_base + 256, tmem_base + b * 128 + half * 64 + i * 8, db + ks * (2048 >> 4), idesc_pv,
                 (accumulate || i > 0) ? 1u : 0u);
        }
      };
      for (int32_t si = seg_lo; si < seg_hi; ++si) {
        SegView sv;
        load_segment(meta, hdr, si, sv);
        if (sv.tile_end <= sv.tile_begin) continue;
        const int32_t nt = sv.tile_end - sv.tile_begin;
        mbar_wait(bq_full, q_it & 1);
        for (int b = 0; b < 2 && b < nt; ++b) {
          const uint32_t slot = ring_it % kStages, par = (ring_it / kStages) & 1;
          mbar_wait(bkv_full(slot), par);
          tc_fence_after();
          if (leader) {
            issue_S(b, slot); mma_commit(bs_full(b)); mma_commit(bkv_empty(slot));
            if (b + 1 == nt || (b == 1 && nt == 2)) mma_commit(bq_empty);
          }
          __syncwarp();
          ++ring_it;
        }
        for (int32_t t = 0; t < nt; ++t) {
          const int b = t & 1;
          const uint32_t slot_v = ring_it % kStages, par_v = (ring_it / kStages) & 1;
          ++ring_it;
          const bool have_next = t + 2 < nt;
          uint32_t slot_k = 0, par_k = 0;
          if (have_next) { slot_k = ring_it % kStages; par_k = (ring_it / kStages) & 1; ++ring_it; }
          const uint32_t tb = b ? tiles1 : tiles0;
          mbar_wait(bkv_full(slot_v), par_v);
          mbar_wait(bp_full(b, 0), tb & 1);
          if (t == 0) mbar_wait(bo_empty, (seg_it & 1) ^ 1);
          tc_fence_after();
          if (leader) issue_PV(b, slot_v, 0, t > 0);
          __syncwarp();
          mbar_wait(bp_full(b, 1), tb & 1);
          tc_fence_after();
          if (leader) {
            issue_PV(b, slot_v, 1, true);
            mma_commit(bpv_done(b));
            if (t + 1 == nt) mma_commit(bo_full);
            mma_commit(bkv_empty(slot_v));
          }
          __syncwarp();
          if (have_next) {
            mbar_wait(bkv_full(slot_k), par_k);
            tc_fence_after();
            if (leader) {
              issue_S(b, slot_k); mma_commit(bs_full(b)); mma_commit(bkv_empty(slot_k));
              if (t + 3 == nt) mma_commit(bq_empty);
            }
            __syncwarp();
          }
          if (b) ++tiles1; else ++tiles0;
        }
        ++seg_it; ++q_it;
      }
    }
  } else {
    // ======================================================= softmax warpgroups: warpgroup h takes keys 64h .. 64h + 63
    // of EVERY tile, thread = packed row
    setmaxnreg_inc<208>();
    const int h = warp >> 2;
    const uint32_t lane_base = (uint32_t)(warp & 3) * 32;
    const int32_t R = (int32_t)lane_base + lane;
    const float c = p.scale * 1.4426950408889634f;
    uint32_t tiles0 = 0, tiles1 = 0, seg_it = 0;
    bool pdl_done = false;

    for (int32_t si = seg_lo; si < seg_hi; ++si) {
      SegView sv;
      load_segment(meta, hdr, si, sv);
      const int32_t ntot = sv.tile_end - sv.tile_begin;
      const int32_t part_slot = sv.part_base;               // (decode plans: one pair per group)
      const int32_t tok = sv.g.q_token0 + R / p.G;
      const bool row_valid = tok < sv.g.q_token_end && R < kTileRows;
      if (ntot <= 0) {
        // every tile of this split lies beyond what the rows can see: publish an empty partial
        if (!pdl_done) { pdl_wait(); pdl_done = true; }
        if (h == 0 && row_valid && sv.part_base >= 0) p.part_lse[(int64_t)part_slot * kPairRows + R] = -INFINITY;
        continue;
      }
      const int32_t head = sv.g.kv_head * p.G + R % p.G;
      int32_t vis = sv.g.kv_len;
      if (sv.g.vis_off >= 0 && row_valid) vis = meta[hdr.off_vis + sv.g.vis_off + (tok - sv.g.q_token0)];
      const int32_t Tc = (sv.g.cache_len + kTileKeys - 1) / kTileKeys;
      const int32_t vis_cache = min(vis, sv.g.cache_len);
      // text-causal mixed mask (reading A19): see attn_sm100.cu
      const int32_t txt_rec = sv.g.txt_off;
      int32_t txt_pos = -1, txt_abs0 = 0, txt_nw = 0;
      if (txt_rec >= 0) {
        txt_abs0 = meta[txt_rec];
        txt_nw = (meta[txt_rec + 1] + 31) >> 5;
        if (row_valid) {
          const int32_t k = tok - sv.g.new_tok0;
          if ((meta[txt_rec + 2 + (k >> 5)] >> (k & 31)) & 1) txt_pos = txt_abs0 + k;
        }
      }
      // tiles that need a mask, per warp: pool part (t < Tc) tiles >= mask_a, k_new part tiles >= mask_b
      int32_t mask_a, mask_b;
      {
        int32_t ma = vis_cache >> 7, mb = max(vis - sv.g.cache_len, 0) >> 7;
        if (txt_pos >= 0) { ma = min(ma, (txt_pos + 1) >> 7); mb = min(mb, max(txt_pos + 1 - sv.g.cache_len, 0) >> 7); }
        mask_a = __reduce_min_sync(0xffffffffu, ma);
        mask_b = Tc + __reduce_min_sync(0xffffffffu, mb);
      }
      float m_used = -INFINITY, l = 0.f;                     // reference shared by both halves of the row; l: this half's sum
      bool all_finite = false;                               // CTA-uniform

      for (int32_t t = 0; t < ntot; ++t) {
        const int b = t & 1;
        const uint32_t tb = b ? tiles1 : tiles0;
        const int32_t tile = sv.tile_begin + t;
        const bool need_mask = tile >= (tile < Tc ? mask_a : mask_b);
        const uint32_t t_s = tmem_base + (lane_base << 16) + b * 128 + h * 64;
        mbar_wait(bs_full(b), tb & 1);
        tc_fence_after();
        uint32_t pk[32];                                    // this half of the P row, packed bf16x2
        float sum = 0.f;
        bool bad = true;
        if (t >= kExactFirstTiles && all_finite && !need_mask) {
          // optimistic: exponentiate against the running reference, no look at the maximum
          const float neg_mc = -m_used;
          uint64_t l01 = 0, l23 = 0;
          uint32_t sa[32], sb[32];
          tmem_ld32(t_s + 0, sa);
          tmem_wait_ld();
          tmem_ld32(t_s + 32, sb);
          softmax_chunk(sa, c, neg_mc, l01, l23, pk + 0);
          tmem_wait_ld();
          softmax_chunk(sb, c, neg_mc, l01, l23, pk + 16);
          float la, lb;
          unpack_f32x2(add_f32x2(l01, l23), la, lb);
          sum = la + lb;
          bad = __any_sync(0xffffffffu, !(sum < fminf(kFastSumLimit, l)));
        }
        // one decision for the whole CTA (both halves of a row must keep the same reference)
        if (!bar_or_256(bad)) {
          l += sum;
        } else {
          // ---- exact path: row maximum over both halves, the reference follows it whenever it grew (the row's
          // largest weight so far is then p = 1), O and l rescaled; masked tiles come here as well
          uint32_t sr[64];
          tmem_ld32(t_s + 0, sr + 0);
          tmem_ld32(t_s + 32, sr + 32);
          tmem_wait_ld();
#define S_(i) __uint_as_float(sr[i])
          if (need_mask) {
            const int32_t key0 = (tile < Tc ? tile * kTileKeys : sv.g.cache_len + (tile - Tc) * kTileKeys) + h * 64;
            const int32_t lim = tile < Tc ? vis_cache : vis;
#pragma unroll
            for (int i = 0; i < 64; ++i)
              if (key0 + i >= lim) sr[i] = 0xff800000u;     // -inf
            if (txt_rec >= 0) {
              uint32_t hide[2];
#pragma unroll
              for (int k = 0; k < 2; ++k) {
                const int32_t b0 = key0 + 32 * k - txt_abs0;
                uint32_t tw = 0;
                if (b0 > -32 && b0 < 32 * txt_nw) {
                  if (b0 < 0) {
                    tw = (uint32_t)meta[txt_rec + 2] << (-b0);
                  } else {
                    const int32_t idx = b0 >> 5;
                    const uint32_t lo = (uint32_t)meta[txt_rec + 2 + idx];
                    const uint32_t hi = idx + 1 < txt_nw ? (uint32_t)meta[txt_rec + 3 + idx] : 0u;
                    tw = __funnelshift_r(lo, hi, b0 & 31);
                  }
                }
                const int32_t d = txt_pos - (key0 + 32 * k);
                const uint32_t later = txt_pos < 0 ? 0u : (d < 0 ? 0xffffffffu : (d >= 31 ? 0u : (0xffffffffu << (d + 1))));
                hide[k] = tw & later;
              }
#pragma unroll
              for (int i = 0; i < 64; ++i)
                if ((hide[i >> 5] >> (i & 31)) & 1u) sr[i] = 0xff800000u;
            }
          }
          float mx0 = S_(0), mx1 = S_(1), mx2 = S_(2), mx3 = S_(3);
#pragma unroll
          for (int i = 4; i < 64; i += 4) {
            mx0 = fmaxf(mx0, S_(i)); mx1 = fmaxf(mx1, S_(i + 1));
            mx2 = fmaxf(mx2, S_(i + 2)); mx3 = fmaxf(mx3, S_(i + 3));
          }
          const float mine = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
          bars->xch[h][R] = mine;
          bar_or_256(false);
          const float tm = fmaxf(mine, bars->xch[h ^ 1][R]) * c;
          const bool grow = tm > m_used;
          if (t == 0) {
            m_used = tm;
          } else if (__any_sync(0xffffffffu, grow)) {
            float alpha = 1.f;
            if (grow) { alpha = m_used == -INFINITY ? 0.f : ex2_approx(m_used - tm); m_used = tm; l *= alpha; }
            if (h == 0) {
              // O is quiescent once PV of the previous tile (the other S buffer) has completed
              mbar_wait(bpv_done(b ^ 1), ((b ? tiles0 : tiles1) - 1) & 1);
              tc_fence_after();
              const uint32_t t_o = tmem_base + (lane_base << 16) + 256;
#pragma unroll 1
              for (int ch = 0; ch < 4; ++ch) {
                uint32_t o[32];
                tmem_ld32(t_o + ch * 32, o);
                tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                tmem_st32(t_o + ch * 32, o);
              }
            }
          }
          const float m_c = (m_used == -INFINITY) ? 0.f : m_used;
          float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;
#pragma unroll
          for (int i = 0; i < 64; i += 4) {
            const float p0 = ex2_approx(fmaf(S_(i), c, -m_c));
            const float p1 = ex2_approx(fmaf(S_(i + 1), c, -m_c));
            const float p2 = ex2_approx(fmaf(S_(i + 2), c, -m_c));
            const float p3 = ex2_approx(fmaf(S_(i + 3), c, -m_c));
            l0 += p0; l1 += p1; l2 += p2; l3 += p3;
            pk[i / 2] = pack_bf16x2(p0, p1);
            pk[i / 2 + 1] = pack_bf16x2(p2, p3);
          }
          l += (l0 + l1) + (l2 + l3);
#undef S_
          all_finite = !bar_or_256(m_used == -INFINITY);
        }
        // P of this half over the first 32 columns of its own half of S_b (masked keys: P is exactly 0 and the
        // bytes behind them are finite, see attn_sm100.cu)
        tmem_st32(t_s, pk);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bp_full(b, h));
        if (b) ++tiles1; else ++tiles0;
      }
      // ---------------------------------------------------- epilogue: l = l_0 + l_1, each warpgroup stores 64 columns
      if (!pdl_done) { pdl_wait(); pdl_done = true; }
      mbar_wait(bo_full, seg_it & 1);
      tc_fence_after();
      bars->xch[h][R] = l;
      bar_or_256(false);
      const float L = l + bars->xch[h ^ 1][R];
      const float inv_l = L > 0.f ? 1.f / L : 0.f;
      const float lse2 = L > 0.f ? m_used + log2f(L) : -INFINITY;
      const uint32_t t_o = tmem_base + (lane_base << 16) + 256 + h * 64;
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
        uint32_t o[32];
        tmem_ld32(t_o + ch * 32, o);
        tmem_wait_ld();
        if (row_valid) {
          if (sv.part_base < 0) {
            __nv_bfloat16* orow = reinterpret_cast<__nv_bfloat16*>(p.out) + ((int64_t)tok * p.Hq + head) * p.D + h * 64 + ch * 32;
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
              uint4 w;
              w.x = pack_bf16x2(__uint_as_float(o[i]) * inv_l, __uint_as_float(o[i + 1]) * inv_l);
              w.y = pack_bf16x2(__uint_as_float(o[i + 2]) * inv_l, __uint_as_float(o[i + 3]) * inv_l);
              w.z = pack_bf16x2(__uint_as_float(o[i + 4]) * inv_l, __uint_as_float(o[i + 5]) * inv_l);
              w.w = pack_bf16x2(__uint_as_float(o[i + 6]) * inv_l, __uint_as_float(o[i + 7]) * inv_l);
              *reinterpret_cast<uint4*>(orow + i) = w;
            }
          } else {
            float* prow = p.part_o + ((int64_t)part_slot * kPairRows + R) * p.D;
#pragma unroll
            for (int i = 0; i < 32; i += 4)
              *reinterpret_cast<uint4*>(prow + part_chunk_pos(h * 16 + ch * 8 + i / 4, R) * 4) =
                  make_uint4(__float_as_uint(__uint_as_float(o[i]) * inv_l), __float_as_uint(__uint_as_float(o[i + 1]) * inv_l),
                             __float_as_uint(__uint_as_float(o[i + 2]) * inv_l), __float_as_uint(__uint_as_float(o[i + 3]) * inv_l));
          }
        }
      }
      if (h == 0 && row_valid) {
        if (sv.part_base < 0) { if (p.lse) p.lse[(int64_t)tok * p.Hq + head] = lse2 * 0.6931471805599453f; }
        else p.part_lse[(int64_t)part_slot * kPairRows + R] = lse2;
      }
      tc_fence_before();
      mbar_arrive(bo_empty);
      ++seg_it;
    }
  }
  if (warp >= 10 && p.append_tokens > 0) {
    // ===================================================== a2 inside the fused step (kv_append.cuh), as in attn_sm100.cu
    pdl_wait();
    const AppendGeom geom{reinterpret_cast<const int4*>(p.k_new), reinterpret_cast<const int4*>(p.v_new),
                          reinterpret_cast<int4*>(p.k_pool_w), reinterpret_cast<int4*>(p.v_pool_w),
                          p.page_table_w, p.max_pages_per_session, p.P, p.Hkv, p.D * 2 / 16};
    const MetaView<kInlineAppendWords> ameta{nullptr, app};
    append_work(ameta, geom, peers, ((int64_t)blockIdx.x * 2 + (warp - 10)) * 32 + lane, (int64_t)gridDim.x * 64,
                (blockIdx.x == 0 && warp == 10) ? lane : -1, 32);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 10) {
    tc_fence_after();
    tmem_dealloc<dec::kTmemCols>(tmem_base);
  }
}

cudaError_t dec_sm100_configure() {
  const void* fns[2] = {(const void*)attn_dec_sm100_kernel<kInlineAttnWords>, (const void*)attn_dec_sm100_kernel<kInlineAttnWordsLarge>};
  for (const void* f : fns) {
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dec::kSmemBytes);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_attn_dec_sm100(const Sm100Launch& l, cudaStream_t stream) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(l.num_ctas); cfg.blockDim = dim3(dec::kThreads);
  cfg.dynamicSmemBytes = dec::kSmemBytes; cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  if (l.inl_words <= kInlineAttnWords) {
    InlineAttnMeta small;
    memcpy(small.w, l.inl.w, sizeof(small.w));
    return cudaLaunchKernelEx(&cfg, attn_dec_sm100_kernel<kInlineAttnWords>, l.tmap_q, l.tmap_k, l.tmap_v,
                              l.tmap_kn, l.tmap_vn, small, l.app, l.peers, l.p);
  }
  return cudaLaunchKernelEx(&cfg, attn_dec_sm100_kernel<kInlineAttnWordsLarge>, l.tmap_q, l.tmap_k, l.tmap_v,
                            l.tmap_kn, l.tmap_vn, l.inl, l.app, l.peers, l.p);
}

}  // namespace ws

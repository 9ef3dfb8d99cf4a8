// attn_sm100.cu - a3 on sm_100a: block-causal attention forward for bf16, D = 128, 64-token pages.
//
// Definition (DESIGN.md §1; PAPER.md:11, :23, :29 "block-causal attention", :47 Eq. (1)): a query
// row in block b sees every key j < e_b.  On the hot path (the newest block attends) that is ALL
// L + n keys, so every 128-key tile is "full" (no mask code runs) except the last one when
// (L + n) % 128 != 0; multi-block queries add per-row visible ends (partial / skipped tiles).
//
// Mapping.  The G = Hq/Hkv query heads that share a KV head are packed with the tokens into the MMA
// M dimension (row = token * G + head_in_group), so one K/V tile read serves all G heads.  A CTA
// owns a PAIR of 128-row Q tiles (256 packed rows) of one (session, KV head) group and a contiguous
// range of that group's KV tiles (a "segment" from the host planner, plan.cpp); it may process
// several segments back to back.
//
// Pipeline (12 warps, 1 CTA / SM):
//   warp 8  lane 0 : TMA producer - Q tiles (rank-3 map over [D, Hq, tokens]) and K/V tiles into a
//                    5-slot ring of 32 KB buffers, 128B-swizzled, completion on mbarriers.  Keys of the
//                    committed cache come from the paged pool (rank-4 map over [D, P, Hkv, pages]; the
//                    page id read from the device page table is the outermost TMA coordinate); in a
//                    fused step (ws_stream_step) the keys of the block being committed come straight
//                    from the caller's k_new / v_new (rank-3 maps over [D, Hkv, tokens]) as KV tiles of
//                    their own after the cache tiles, so nothing waits for the commit.
//   warp 9  lane 0 : tcgen05.mma issuer - S_q = Q_q K^T (SS, M128 N128 K16 x 8) into TMEM, and
//                    O_q += P_q V (A = P from TMEM, B = V from smem, MN-major) for q = 0, 1,
//                    interleaved so the tensor pipe works on one Q tile while the softmax
//                    warpgroup of the other is busy.  tcgen05.commit arrives on mbarriers.
//   warps 0-3, 4-7 : softmax warpgroup for Q tile 0 / 1: tcgen05.ld of a whole S row per thread
//                    (32x32b: thread = row, so max/sum need no cross-thread reduction), fp32 online
//                    softmax in the log2 domain, P rounded to bf16 and written back over S in TMEM,
//                    row sum accumulated in fp32 from the unrounded p.  Epilogue: O / l -> bf16 out
//                    (+ LSE) or fp32 partial + log2-LSE when the segment is one of several splits.
//   warp 10        : TMEM allocation (512 columns: S0 S1 O0 O1) and release.
//   warps 10, 11   : fused step only: commit the new block (a2, kv_append.cuh) - copy k_new / v_new
//                    into the pool pages, publish the page ids, zero the last page's tail - while the
//                    other warps attend.
//
// Roofline: tensor-bound for G*n >= ~260 FLOP/B (configs 3-5), 4*D*rows*keys FLOPs per tile pair;
// algorithmic bytes per tile = 2 x 128 x 128 x 2 B of K/V.  MUFU ex2 (16/clk/SM) is the co-limit.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <type_traits>

#include "kv_append.cuh"
#include "launch.h"
#include "sm100_ptx.cuh"
#include "softmax_chunk.cuh"
#include "merge.cuh"

namespace ws {

using namespace ptx;

constexpr int kStages = 5;                                 // K/V ring: 5 slots of one 128-key tile (32 KB)
constexpr uint32_t kSlotBytes = 32768;
constexpr uint32_t kRingBytes = kStages * kSlotBytes;
constexpr uint32_t kHalfBytes = 16384;                     // one 64-dim half of a 128-row tile: 128 rows x 128 B
constexpr uint32_t kQTileBytes = kTileRows * 128 * 2;
constexpr int kThreads = 384;
constexpr uint32_t kTmemCols = 512;
constexpr int kFirstPieceSteps = 6;                         // P is handed to the MMA warp as keys 0-95, then 96-127
// Optimistic (fast) softmax path: a tile is exponentiated against the running reference without looking
// for its maximum, and accepted while its row sum stays below BOTH limits:
//  * kFastSumLimit - every p is <= the sum, so nothing overflowed bf16's useful range;
//  * kFastSumShare x the row's accumulated sum l - the tile cannot hold a key that carries a large share
//    of the row's weight.  A tile that could (the first few of a segment, or one with a dominant key)
//    takes the exact path, which re-references the row to its exact maximum whenever that grew, so the
//    dominant weight is p = 1 exactly and suffers no bf16 rounding (reading A10: with a stale
//    reference the x8-outlier config reached 1.2e-2 max-abs; with this rule it stays at the output's
//    own rounding).
constexpr float kFastSumLimit = 1024.0f;
constexpr float kFastSumShare = 1.0f;
constexpr int kExactFirstTiles = 2;                         // tiles 0-1 of a segment go straight to the exact path

// Shared-memory matrix descriptors hold bits [4, 18) of the CTA-local address.  In a CLUSTER launch the shared-window
// address of a CTA of rank >= 1 carries its rank in higher bits; unmasked they spill into the descriptor's
// leading-byte-offset field - harmless for the K-major operands (Q, K: LBO unused), wrong upper 64 dims for the
// MN-major V (found with the cluster-plan experiment, DESIGN.md section 8 x: LSE exact, O columns 64-127 wrong on
// ranks >= 1).  This kernel is not launched in clusters today; the mask keeps the descriptors right if it ever is.
constexpr uint32_t kDescAddrMask = 0x3FFFFu;
constexpr int kMaxJobs = 4;

struct Barriers {
  uint64_t q_full, q_empty;
  uint64_t kv_full[kStages], kv_empty[kStages];
  uint64_t s_full[2], p_full[2][2], pv_h0_done[2], o_full[2], o_empty[2];
  uint64_t merge_full;
  alignas(16) float lse_stage[kPairRows];                  // staged epilogue: the pair's log2-LSEs on their way to part_lse
  MergeJob jobs[kMaxJobs];
  int32_t njobs, cur_slot0;          // fused combine: parked merge jobs, first partial slot of the current (item, pair)
  uint32_t tmem_base;
  uint32_t pad;
};
constexpr uint32_t kSmemBytes = 2 * kQTileBytes + kRingBytes + sizeof(Barriers) + 1024;
static_assert(kSmemBytes <= 232448, "227 KB of shared memory per CTA");

struct SegView {
  Group g;
  int32_t tile_begin, tile_end, part_base, group;
};


// Loads segment `si` as seen by row-tile pair `pair`.  Returns false if this CTA has no rows in it
// (pair >= npairs).  For multi-block queries the pair's own visible end clips the tile range: KV
// tiles beyond the last key any of the pair's rows can see are skipped (block-lower-triangular
// skipping at pair granularity); `v.tile_end <= v.tile_begin` then means "nothing to compute here".
template <int W>
__device__ __forceinline__ bool load_segment(const MetaView<W>& meta, const AttnMeta& hdr, int32_t si,
                                             int32_t pair, int32_t tok_per_pair, SegView& v) {
  const Segment s = meta.template load<Segment>(hdr.off_segments + si * (int32_t)(sizeof(Segment) / 4));
  v.g = meta.template load<Group>(hdr.off_groups + s.group * (int32_t)(sizeof(Group) / 4));
  v.tile_begin = s.tile_begin; v.tile_end = s.tile_end; v.part_base = s.part_base; v.group = s.group;
  if (pair >= v.g.npairs) return false;
  if (v.g.vis_off >= 0) {
    const int32_t last_tok = min(v.g.q_token_end, v.g.q_token0 + (pair + 1) * tok_per_pair) - 1;
    const int32_t pair_kv = meta[hdr.off_vis + v.g.vis_off + (last_tok - v.g.q_token0)];
    v.tile_end = min(v.tile_end, (pair_kv + kTileKeys - 1) / kTileKeys);
  }
  return true;
}

// ---- fused split-KV combine (a4 inside the attention kernel; the paper is silent on this step) ----
// A group whose KV range was cut into `nparts` segments yields nparts partials per row-tile pair, each
// written by a different CTA.  Each of those CTAs also owns 1/nparts of the pair's rows: after it has
// published ALL of its own partials it waits until the arrival counter of the (item, pair) shows that
// every part is there and merges its rows (LSE-weighted, same arithmetic as combine_kernel).  The wait
// cannot deadlock: a CTA signals before it waits, signalling depends on nothing but the CTA's own
// progress, and the grid is launched cooperatively (all CTAs co-resident).
__device__ __forceinline__ int32_t ld_acquire_gpu(const int32_t* p) {
  int32_t v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// volatile so that a batch of these stays in program order ahead of the mbarrier wait that follows it
// (as plain loads the compiler sank each one to its first use: one exposed L2 latency per merged row)
__device__ __forceinline__ float ld_cg_f32(const float* p) {
  float v;
  asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int32_t ld_relaxed_gpu(const int32_t* p) {
  int32_t v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_gpu_add(int32_t* p, int32_t v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

// (Decode plans - at most 128 packed rows per group - run on attn_dec_sm100.cu.)
//
// Programmatic dependent launch (protocol: launch.h).  Before griddepcontrol.wait the TMA producer fetches
// only KV tiles of the stable prefix of its first segment (Group::stable_tiles: committed at least two
// append calls ago, so no kernel that can still be in flight writes them); the wait precedes every other
// load (q, k_new, v_new may come from the caller's kernel just before; pool pages and page-table entries
// from an append just before) and only after it does that thread let the successor's CTAs be scheduled;
// the append warps wait before their first store, every softmax thread before its first global write
// (out / partials may still be read or written by the previous step's kernels).  Metadata in a device blob
// (p.meta: large calls, uploaded by a stream-ordered copy) is only read after the wait.
template <int kInlW>
__global__ void __launch_bounds__(kThreads, 1)
attn_sm100_kernel(const __grid_constant__ CUtensorMap tmap_q,
                  const __grid_constant__ CUtensorMap tmap_k,
                  const __grid_constant__ CUtensorMap tmap_v,
                  const __grid_constant__ CUtensorMap tmap_kn,
                  const __grid_constant__ CUtensorMap tmap_vn,
                  const __grid_constant__ InlineMeta<kInlW> inl,
                  const __grid_constant__ InlineAppendMeta app, const __grid_constant__ PeerPools peers,
                  const AttnParams p_in) {
  AttnParams p = p_in;
  if (p.meta != nullptr) pdl_wait();
  const MetaView<kInlW> meta{p.meta, inl};
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base;                           // 2 x 32 KB
  const uint32_t sRing = smem_base + 2 * kQTileBytes;      // kStages x kSlotBytes
  Barriers* bars = reinterpret_cast<Barriers*>(smem_raw + (smem_base - smem_u32(smem_raw)) +
                                               2 * kQTileBytes + kRingBytes);
  const uint32_t bq_full = smem_u32(&bars->q_full), bq_empty = smem_u32(&bars->q_empty);
  auto bkv_full = [&](int s) { return smem_u32(&bars->kv_full[s]); };
  auto bkv_empty = [&](int s) { return smem_u32(&bars->kv_empty[s]); };
  auto bs_full = [&](int q) { return smem_u32(&bars->s_full[q]); };
  auto bp_full = [&](int q, int half) { return smem_u32(&bars->p_full[q][half]); };
  auto bpv_h0 = [&](int q) { return smem_u32(&bars->pv_h0_done[q]); };
  auto bo_full = [&](int q) { return smem_u32(&bars->o_full[q]); };
  auto bo_empty = [&](int q) { return smem_u32(&bars->o_empty[q]); };

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const AttnMeta hdr = meta.template load<AttnMeta>(0);
  const int32_t team = blockIdx.x / hdr.team_size;
  const int32_t pair = blockIdx.x - team * hdr.team_size;
  const int32_t seg_lo = meta[hdr.off_team_seg_begin + team], seg_hi = meta[hdr.off_team_seg_begin + team + 1];
  const int32_t tok_per_pair = kPairRows / p.G;
  const int32_t tok_per_tile = kTileRows / p.G;

  // The TMA producer resolves its first segment and the page ids of its first tile while the other warps
  // allocate TMEM and initialise the barriers: takes the metadata and page-table latencies off the path to
  // the first MMA.
  SegView sv_first;
  int32_t si_first = seg_hi, pre_pg0 = 0, pre_pg1 = 0;
  bool pre_valid = false;
  // Q tiles of segment `sv` (the pair's two tiles) -> sQ
  auto issue_q = [&](const SegView& sv) {
    mbar_arrive_expect_tx(bq_full, 2 * kQTileBytes);
    const int32_t tok0 = sv.g.q_token0 + pair * tok_per_pair;
    for (int q = 0; q < 2; ++q)
      for (int h = 0; h < 2; ++h)
        tma_load_3d(sQ + q * kQTileBytes + h * kHalfBytes, &tmap_q, bq_full, h * 64,
                    sv.g.kv_head * p.G, tok0 + q * tok_per_tile);
  };
  if (warp == 8 && lane == 0) {
    // the producer owns the Q barriers
    mbar_init(bq_full, 1); mbar_init(bq_empty, 1);
    fence_mbar_init();
    fence_proxy_async_smem();
    prefetch_tmap(&tmap_q); prefetch_tmap(&tmap_k); prefetch_tmap(&tmap_v);
    if (p.append_tokens > 0) { prefetch_tmap(&tmap_kn); prefetch_tmap(&tmap_vn); }
    for (si_first = seg_lo; si_first < seg_hi; ++si_first)
      if (load_segment(meta, hdr, si_first, pair, tok_per_pair, sv_first) &&
          sv_first.tile_end > sv_first.tile_begin) break;
    // page ids of the first tile, if it lies in the stable prefix (readable before griddepcontrol.wait)
    if (si_first < seg_hi && sv_first.tile_begin < sv_first.g.stable_tiles) {
      const int32_t* page_row = p.page_table + (int64_t)sv_first.g.slot * p.max_pages_per_session;
      pre_pg0 = page_row[2 * sv_first.tile_begin];
      pre_pg1 = page_row[2 * sv_first.tile_begin + 1];
      pre_valid = true;
    }
  }
  if (warp == 9 && lane == 0) {
    mbar_init(smem_u32(&bars->merge_full), 1);
    bars->njobs = 0;
    for (int s = 0; s < kStages; ++s) { mbar_init(bkv_full(s), 1); mbar_init(bkv_empty(s), 1); }
    for (int q = 0; q < 2; ++q) {
      mbar_init(bs_full(q), 1); mbar_init(bp_full(q, 0), 128); mbar_init(bp_full(q, 1), 128);
      mbar_init(bpv_h0(q), 1);
      mbar_init(bo_full(q), 1); mbar_init(bo_empty(q), 128);
    }
    fence_mbar_init();
  }
  if (warp == 10) { tmem_alloc<kTmemCols>(smem_u32(&bars->tmem_base)); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;

  if (warp >= 8) {
    setmaxnreg_dec<88>();
    if (warp == 8 && lane == 0) {
      // ===================================================== TMA producer
      uint32_t ring_it = 0, q_it = 0;
      // Programmatic dependent launch (launch.h).  Until `waited`, only KV tiles of the FIRST segment's
      // stable prefix are fetched (at most one ring of them: the MMA warp cannot consume without Q);
      // griddepcontrol.wait precedes everything else - q, k_new / v_new, page ids and pool rows of recent
      // appends - and only then does this thread let the successor's CTAs be scheduled.
      bool waited = false;
      auto ensure_wait = [&]() {
        if (!waited) { pdl_wait(); pdl_launch_dependents(); waited = true; }
      };
      for (int32_t si = si_first; si < seg_hi; ++si) {
        SegView sv;
        const bool first = si == si_first;
        if (first) {
          sv = sv_first;
        } else {
          if (!load_segment(meta, hdr, si, pair, tok_per_pair, sv)) continue;
          if (sv.tile_end <= sv.tile_begin) continue;        // clipped away for this pair
        }
        const int32_t* page_row = p.page_table + (int64_t)sv.g.slot * p.max_pages_per_session;
        const int32_t last_page = (sv.g.cache_len - 1) / p.P;
        const int32_t Tc = (sv.g.cache_len + kTileKeys - 1) / kTileKeys;   // tiles >= Tc: the block being committed
        const int32_t nt = sv.tile_end - sv.tile_begin;
        // ONE loop, ONE issue site for the K/V tiles of the segment (code size: the hot loops of the four warp
        // roles have to stay inside the 32 KB instruction cache).  Order = consumption order of the MMA warp:
        // K0 V0 K1 V1 ... (K runs kAhead tiles ahead of V; the decode kernel uses the same loop with 2).
        // The Q tiles go out once: the first segment's right after the wait (until then only tiles of its
        // stable prefix are fetched, at most one ring of them), a later segment's when the MMA warp has
        // released the Q buffers.
        constexpr int32_t kAhead = 1;
        int32_t nk = 0, nv = 0, pg0 = pre_pg0, pg1 = pre_pg1;
        bool have_ids = first && pre_valid, q_pending = true;
        for (;;) {
          const bool is_v = !(nk < nt && nk < nv + kAhead);
          const int32_t j = sv.tile_begin + (is_v ? nv : nk);
          const bool at_end = nv >= nt;
          if (q_pending && !(first && !waited && !at_end && j < sv.g.stable_tiles && ring_it < (uint32_t)kStages)) {
            ensure_wait();
            if (!first) mbar_wait(bq_empty, (q_it & 1) ^ 1);
            issue_q(sv);
            q_pending = false;
          }
          if (at_end) break;
          // page ids of tile j (pool part): the general plan loads them with the K tile and keeps them for
          // the V tile that follows (and fetches the next tile's one tile ahead when they are published)
          if (!is_v && !have_ids) {
            pg0 = j < Tc ? page_row[min(2 * j, last_page)] : 0;
            pg1 = j < Tc ? page_row[min(2 * j + 1, last_page)] : 0;
          }
          const int32_t c0 = pg0, c1 = pg1;
          if (is_v) {
            // next tile's ids one tile ahead - unless they may not be published yet
            have_ids = j + 1 < sv.tile_end && j + 1 < Tc && (!q_pending || j + 1 < sv.g.stable_tiles);
            if (have_ids) { pg0 = page_row[min(2 * j + 2, last_page)]; pg1 = page_row[min(2 * j + 3, last_page)]; }
          }
          // one 128-key K or V tile -> the next ring slot: 64-key x 64-dim boxes at offsets 0 (keys 0-63,
          // dims 0-63), 8 KB (keys 64-127), 16 KB and 24 KB (dims 64-127)
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
            // rows past the end of k_new / v_new are zero-filled by TMA; rows of the next session's
            // block (batched calls) are finite data; both are masked by the softmax
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
      }
      ensure_wait();
    } else if (warp == 9) {
      // ===================================================== MMA issuer
      // The whole warp runs the control flow convergently (all values stay warp-uniform, so the
      // descriptors are built on the uniform datapath); one elected lane issues tcgen05.mma/commit.
      const bool leader = elect_one();
      constexpr uint32_t idesc_qk = make_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc_bf16(128, 128, 0, 1);
      const uint64_t desc_k = make_smem_desc_sw128(0, 16, 1024);          // K-major operands (Q, K)
      const uint64_t desc_v = make_smem_desc_sw128(0, kHalfBytes, 1024);  // MN-major operand (V)
      uint32_t ring_it = 0, q_it = 0, tile_it = 0, seg_it = 0;
      auto issue_S = [&](int q, uint32_t slot) {
        const uint64_t da = desc_k + (((sQ + q * kQTileBytes) & kDescAddrMask) >> 4);
        const uint64_t db = desc_k + (((sRing + slot * kSlotBytes) & kDescAddrMask) >> 4);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          const uint32_t off = ((ks >> 2) * kHalfBytes + (ks & 3) * 32) >> 4;
          mma_ss(tmem_base + q * 128, da + off, db + off, idesc_qk, ks > 0);
        }
      };
      // PV for one of the two pieces in which the softmax hands P over (k-steps of 16 keys)
      auto issue_PV = [&](int q, uint32_t slot, int half, bool accumulate) {
        const uint64_t db = desc_v + (((sRing + slot * kSlotBytes) & kDescAddrMask) >> 4);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          if ((ks < kFirstPieceSteps) != (half == 0)) continue;   // piece 0: keys 0-95, piece 1: keys 96-127
          mma_ts(tmem_base + 256 + q * 128, tmem_base + q * 128 + ks * 8, db + ks * (2048 >> 4),
                 idesc_pv, (accumulate || ks > 0) ? 1u : 0u);
        }
      };
      for (int32_t si = seg_lo; si < seg_hi; ++si) {
        SegView sv;
        if (!load_segment(meta, hdr, si, pair, tok_per_pair, sv)) continue;
        if (sv.tile_end <= sv.tile_begin) continue;          // clipped away for this pair
        const int32_t nt = sv.tile_end - sv.tile_begin;
        mbar_wait(bq_full, q_it & 1);
        {
          const uint32_t slot = ring_it % kStages, par = (ring_it / kStages) & 1;
          mbar_wait(bkv_full(slot), par);
          tc_fence_after();
          if (leader) {
            for (int q = 0; q < 2; ++q) { issue_S(q, slot); mma_commit(bs_full(q)); }
            mma_commit(bkv_empty(slot));
            if (nt == 1) mma_commit(bq_empty);
          }
          __syncwarp();
          ++ring_it;
        }
        for (int32_t j = 0; j < nt; ++j) {
          const uint32_t slot_v = ring_it % kStages, par_v = (ring_it / kStages) & 1;
          ++ring_it;
          const bool have_next = j + 1 < nt;
          uint32_t slot_k = 0, par_k = 0;
          if (have_next) { slot_k = ring_it % kStages; par_k = (ring_it / kStages) & 1; ++ring_it; }
          mbar_wait(bkv_full(slot_v), par_v);
          for (int q = 0; q < 2; ++q) {
            mbar_wait(bp_full(q, 0), tile_it & 1);
            if (j == 0) mbar_wait(bo_empty(q), (seg_it & 1) ^ 1);
            tc_fence_after();
            if (leader) {
              issue_PV(q, slot_v, 0, j > 0);
              mma_commit(bpv_h0(q));
            }
            __syncwarp();
            mbar_wait(bp_full(q, 1), tile_it & 1);
            tc_fence_after();
            if (leader) {
              issue_PV(q, slot_v, 1, true);
              if (!have_next) mma_commit(bo_full(q));
            }
            __syncwarp();
            if (have_next) {
              if (q == 0) { mbar_wait(bkv_full(slot_k), par_k); tc_fence_after(); }
              if (leader) {
                issue_S(q, slot_k);
                mma_commit(bs_full(q));
              }
              __syncwarp();
            }
          }
          if (leader) {
            mma_commit(bkv_empty(slot_v));
            if (have_next) {
              mma_commit(bkv_empty(slot_k));
              if (j + 2 == nt) mma_commit(bq_empty);
            }
          }
          __syncwarp();
          ++tile_it;
        }
        ++q_it; ++seg_it;
      }
    }
  } else {
    // ======================================================= softmax warpgroups (warps 0-7)
    setmaxnreg_inc<208>();
    const int q = warp >> 2;
    const uint32_t lane_base = (uint32_t)(warp & 3) * 32;
    const int32_t row_in_tile = (int32_t)lane_base + lane;
    const int32_t R = q * kTileRows + row_in_tile;          // packed row inside the pair
    const uint32_t t_s = tmem_base + (lane_base << 16) + q * 128;
    const uint32_t t_o = tmem_base + (lane_base << 16) + 256 + q * 128;
    const float c = p.scale * 1.4426950408889634f;
    uint32_t tile_it = 0, seg_it = 0;
    bool pdl_done = false;
    const bool fused = p.merge_ctr != nullptr;
    // publish this warpgroup's half of a partial: every thread's stores are fenced, the warpgroup
    // meets on a named barrier, one thread bumps the arrival counter of the (item, pair) - keyed by
    // the item's first partial slot, found from the group id (at most one combine item per group)
    auto find_item = [&](int32_t group) {
      int32_t k = 0;
      while (k + 1 < hdr.num_combine && meta[hdr.off_combine + k * (int32_t)(sizeof(CombineItem) / 4)] != group) ++k;
      return meta.template load<CombineItem>(hdr.off_combine + k * (int32_t)(sizeof(CombineItem) / 4));
    };
    auto publish = [&](bool fence_all) {
      if (!fused) return;
      // direct stores: every thread fences its own.  Staged path: the only writes are the bulk stores
      // whose completion lane 0 of each warp has already waited for; the barrier below orders them
      // before the (cumulative) release of the counter update.
      if (fence_all) __threadfence();
      // one release per CTA and partial: both warpgroups meet
      asm volatile("bar.sync 3, 256;" ::: "memory");
      if (threadIdx.x == 0) red_release_gpu_add(p.merge_ctr + bars->cur_slot0, 2);
    };
    // resolve the merge duty that comes with a partial segment (thread 0, while the first tile loads)
    auto make_job = [&](const SegView& sv, MergeJob& job) {
      const CombineItem ci = find_item(sv.group);
      const int32_t part = (sv.part_base - ci.part_base) / sv.g.npairs;
      job.slot0 = ci.part_base + pair; job.nparts = ci.nparts; job.npairs = sv.g.npairs; job.kv_head = sv.g.kv_head;
      job.tok0 = sv.g.q_token0 + pair * tok_per_pair;
      const int32_t nv = min(kPairRows, (min(sv.g.q_token_end, job.tok0 + tok_per_pair) - job.tok0) * p.G);
      job.r_lo = (int32_t)((int64_t)part * nv / ci.nparts);
      job.r_hi = (int32_t)((int64_t)(part + 1) * nv / ci.nparts);
      job.pad = 0;
    };

    for (int32_t si = seg_lo; si < seg_hi; ++si) {
      SegView sv;
      if (!load_segment(meta, hdr, si, pair, tok_per_pair, sv)) continue;
      const int32_t nt = sv.tile_end - sv.tile_begin;
      const int32_t part_slot = sv.part_base + pair;
      if (fused && sv.part_base >= 0 && threadIdx.x == 0) {
        MergeJob job;
        make_job(sv, job);
        const int32_t j = bars->njobs;
        if (j < kMaxJobs) bars->jobs[j] = job;
        bars->njobs = j + 1;
        bars->cur_slot0 = job.slot0;
      }
      const int32_t tok = sv.g.q_token0 + pair * tok_per_pair + R / p.G;
      const bool row_valid = tok < sv.g.q_token_end;
      if (sv.tile_end <= sv.tile_begin) {
        // every tile of this segment lies beyond what the pair can see: publish an empty partial
        // (the segment is one of several splits, otherwise it would start at tile 0)
        if (!pdl_done) { pdl_wait(); pdl_done = true; }
        if (row_valid && sv.part_base >= 0)
          p.part_lse[(int64_t)part_slot * kPairRows + R] = -INFINITY;
        if (sv.part_base >= 0) publish(true);
        continue;
      }
      const int32_t head = sv.g.kv_head * p.G + R % p.G;
      int32_t vis = sv.g.kv_len;
      if (sv.g.vis_off >= 0 && row_valid) vis = meta[hdr.off_vis + sv.g.vis_off + (tok - sv.g.q_token0)];
      // keys of tile t: [key0, key0 + 128) of the pool part (t < Tc, ends at cache_len) or of the block
      // being committed (t >= Tc, starts at cache_len, ends at kv_len); a row sees keys below vis
      const int32_t Tc = (sv.g.cache_len + kTileKeys - 1) / kTileKeys;
      const int32_t vis_cache = min(vis, sv.g.cache_len);
      float m_used = -INFINITY, l = 0.f;
      // text-causal mixed mask (NEXT-4, reading A19): a text row at absolute position
      // txt_pos does not see text keys at later positions.  The session's record in the blob:
      // {abs_pos0, nbits, bits...}, bit k <=> the token at position abs_pos0 + k is text.
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

      // O and l of this row scaled by alpha (after a change of reference).  Safe whenever the PV MMAs of
      // the previous tile have completed: s_full of the current tile was committed after them on the same
      // in-order tensor pipe.
      auto rescale_o = [&](float alpha) {
#pragma unroll 1                                            // rare path, inlined at three sites: keep it small
        for (int ch = 0; ch < 4; ++ch) {
          uint32_t o[32];
          tmem_ld32(t_o + ch * 32, o);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
          tmem_st32(t_o + ch * 32, o);
        }
      };
      // One unmasked tile exponentiated against the reference m_used while it streams out of TMEM in
      // 32-column chunks; P is handed to the MMA warp in two pieces (keys 0-95, then 96-127) as soon as
      // each is written: PV of the first piece (384 tensor cycles) overlaps the softmax of the last 32
      // keys, and only 128 cycles of PV remain on the S -> softmax -> PV -> S chain.
      // kCheck: the optimistic use - the reference may be stale, so each piece's row sum is tested against
      // sum_lim (kFastSumLimit / kFastSumShare; a NaN/inf sum fails the test).  Returns false, with nothing
      // handed off and S intact, if the first piece fails.
      auto stream_tile = [&](const bool kCheck, float sum_lim) -> bool {
        const float neg_mc = -m_used;
        uint32_t pk[64];                                    // P row, packed bf16x2
        uint64_t l01 = 0, l23 = 0;                          // packed fp32x2 partial row sums
        uint32_t sa[32], sb[32];
        tmem_ld32(t_s + 0, sa);
        tmem_wait_ld();
        tmem_ld32(t_s + 32, sb);
        softmax_chunk(sa, c, neg_mc, l01, l23, pk + 0);
        tmem_wait_ld();
        tmem_ld32(t_s + 64, sa);
        softmax_chunk(sb, c, neg_mc, l01, l23, pk + 16);
        tmem_wait_ld();
        tmem_ld32(t_s + 96, sb);
        softmax_chunk(sa, c, neg_mc, l01, l23, pk + 32);
        float la, lb;
        unpack_f32x2(add_f32x2(l01, l23), la, lb);
        const float sum_a = la + lb;
        if (kCheck && __any_sync(0xffffffffu, !(sum_a < sum_lim))) return false;
        tmem_st32(t_s + 0, pk);
        tmem_st16(t_s + 32, pk + 32);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bp_full(q, 0));                         // first 96 keys of P handed off
        tmem_wait_ld();
        l01 = 0; l23 = 0;
        softmax_chunk(sb, c, neg_mc, l01, l23, pk + 48);
        unpack_f32x2(add_f32x2(l01, l23), la, lb);
        const float sum_b = la + lb;
        l += sum_a;
        if (!kCheck || !__any_sync(0xffffffffu, !(sum_b < sum_lim))) {
          l += sum_b;
        } else {
          // Rare: the last 32 keys fail the test after the first piece was handed off.  Wait until
          // PV of the first piece has completed (O is then quiescent: the PV of the last piece needs
          // our arrival), re-reference O and l to the exact maximum if it grew and redo the last 32
          // keys exactly.
          mbar_wait(bpv_h0(q), tile_it & 1);
          tc_fence_after();
          uint32_t sr[32];
          tmem_ld32(t_s + 96, sr);
          tmem_wait_ld();
          float mx = __uint_as_float(sr[0]);
#pragma unroll
          for (int i = 1; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(sr[i]));
          const float tm = mx * c;
          float alpha = 1.f;
          if (tm > m_used) { alpha = ex2_approx(m_used - tm); m_used = tm; l *= alpha; }
          rescale_o(alpha);
          float ls = 0.f;
#pragma unroll
          for (int i = 0; i < 32; i += 2) {
            const float p0 = ex2_approx(fmaf(__uint_as_float(sr[i]), c, -m_used));
            const float p1 = ex2_approx(fmaf(__uint_as_float(sr[i + 1]), c, -m_used));
            ls += p0 + p1;
            pk[48 + i / 2] = pack_bf16x2(p0, p1);
          }
          l += ls;
        }
        tmem_st16(t_s + 48, pk + 48);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bp_full(q, 1));
        return true;
      };

      // Tiles that need the masked path, resolved ONCE per segment and warp (the tile loop itself stays free of
      // votes and index arithmetic): in the pool part (t < Tc) tiles t >= mask_a, in the part read from k_new
      // (t >= Tc) tiles t >= mask_b.  A tile needs a mask when it reaches beyond a row's visible end, or - mixed
      // mask - beyond the position of a text row.
      int32_t mask_a, mask_b;
      {
        const int32_t new_vis = max(vis - sv.g.cache_len, 0);
        int32_t ma = vis_cache >> 7, mb = new_vis >> 7;
        if (txt_pos >= 0) { ma = min(ma, (txt_pos + 1) >> 7); mb = min(mb, max(txt_pos + 1 - sv.g.cache_len, 0) >> 7); }
        mask_a = __reduce_min_sync(0xffffffffu, ma);
        mask_b = Tc + __reduce_min_sync(0xffffffffu, mb);
      }
      bool all_finite = false;                               // warp-uniform: every row's reference is finite

      for (int32_t j = 0; j < nt; ++j) {
        const int32_t t = sv.tile_begin + j;
        mbar_wait(bs_full(q), tile_it & 1);
        tc_fence_after();
        const bool need_mask = t >= (t < Tc ? mask_a : mask_b);
        // ---- exact reference for an unmasked tile: one pass over S for the row maximum, the reference
        // follows it whenever it grew (the row's largest weight so far is then p = 1, exactly representable
        // in bf16).  Rare (first tiles of a segment, refused optimistic passes): kept out of the hot path.
        auto exact_reference = [&]() {
          float mx0, mx1, mx2, mx3;
#pragma unroll
          for (int ch = 0; ch < 4; ++ch) {
            uint32_t sr[32];
            tmem_ld32(t_s + ch * 32, sr);
            tmem_wait_ld();
            if (ch == 0) { mx0 = __uint_as_float(sr[0]); mx1 = __uint_as_float(sr[1]); mx2 = __uint_as_float(sr[2]); mx3 = __uint_as_float(sr[3]); }
#pragma unroll
            for (int i = (ch == 0 ? 4 : 0); i < 32; i += 4) {
              mx0 = fmaxf(mx0, __uint_as_float(sr[i])); mx1 = fmaxf(mx1, __uint_as_float(sr[i + 1]));
              mx2 = fmaxf(mx2, __uint_as_float(sr[i + 2])); mx3 = fmaxf(mx3, __uint_as_float(sr[i + 3]));
            }
          }
          const float tm = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c;
          const bool grow = tm > m_used;
          if (j == 0) {
            m_used = tm;
          } else if (__any_sync(0xffffffffu, grow)) {
            float alpha = 1.f;
            if (grow) { alpha = m_used == -INFINITY ? 0.f : ex2_approx(m_used - tm); m_used = tm; l *= alpha; }
            rescale_o(alpha);
          }
          all_finite = !__any_sync(0xffffffffu, m_used == -INFINITY);
        };
        // ONE call site of stream_tile (a second inlined copy of the streaming pass pushed the hot loops of the
        // four warp roles out of the instruction cache: ncu stall_no_inst x4 on the decode plan, 50 -> 66 us per
        // step), reached by falling through in the common case: optimistic pass, accepted.  The optimistic pass
        // is not tried on the first tiles of a segment (their sums are of the order of the accumulated l: the
        // share test would refuse them anyway) nor while a row has seen nothing yet.
        bool fast = j >= kExactFirstTiles && all_finite;
        if (!need_mask) {
#pragma unroll 1
          for (;;) {
            if (!fast) exact_reference();
            if (stream_tile(fast, fast ? fminf(kFastSumLimit, kFastSumShare * l) : 0.f)) break;
            fast = false;
          }
        }
        if (need_mask) {
          // ---- exact path, masked tile (the last tile of the cache part or of the new block when their
          // lengths are no multiples of 128; multi-block queries): whole S row in registers
          const int32_t key0 = t < Tc ? t * kTileKeys : sv.g.cache_len + (t - Tc) * kTileKeys;
          const int32_t lim = t < Tc ? vis_cache : vis;      // keys >= lim of this tile are masked
          uint32_t pk[64];
          uint32_t sr[128];                                 // one whole S row (fp32 bits)
          tmem_ld32(t_s + 0, sr + 0);
          tmem_ld32(t_s + 32, sr + 32);
          tmem_ld32(t_s + 64, sr + 64);
          tmem_ld32(t_s + 96, sr + 96);
          tmem_wait_ld();
#define S_(i) __uint_as_float(sr[i])
#pragma unroll
          for (int i = 0; i < 128; ++i)
            if (key0 + i >= lim) sr[i] = 0xff800000u;       // -inf
          if (txt_rec >= 0) {                               // (warp-uniform)
            uint32_t hide[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              // text bits of keys key0 + 32k .. + 31 (the record is not aligned to the tile), and the keys
              // among them that lie after this row's position
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
            for (int i = 0; i < 128; ++i)
              if ((hide[i >> 5] >> (i & 31)) & 1u) sr[i] = 0xff800000u;
          }
          float mx0 = S_(0), mx1 = S_(1), mx2 = S_(2), mx3 = S_(3);
#pragma unroll
          for (int i = 4; i < 128; i += 4) {
            mx0 = fmaxf(mx0, S_(i)); mx1 = fmaxf(mx1, S_(i + 1));
            mx2 = fmaxf(mx2, S_(i + 2)); mx3 = fmaxf(mx3, S_(i + 3));
          }
          const float tm = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c;
          const bool grow = tm > m_used;
          if (j == 0) {
            m_used = tm;
          } else if (__any_sync(0xffffffffu, grow)) {
            float alpha = 1.f;
            if (grow) { alpha = m_used == -INFINITY ? 0.f : ex2_approx(m_used - tm); m_used = tm; l *= alpha; }
            rescale_o(alpha);
          }
          const float m_c = (m_used == -INFINITY) ? 0.f : m_used;
          all_finite = !__any_sync(0xffffffffu, m_used == -INFINITY);
          float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;
#pragma unroll
          for (int i = 0; i < 128; i += 4) {
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
          tmem_st32(t_s + 0, pk);
          tmem_st32(t_s + 32, pk + 32);
          // (masked keys: P is exactly 0 there and the bytes behind them are finite - the append keeps the
          // unused tail of a session's last page zeroed, rows past the end of k_new are zero-filled - so
          // 0 x V stays 0)
          tmem_wait_st();
          tc_fence_before();
          mbar_arrive(bp_full(q, 0));
          mbar_arrive(bp_full(q, 1));
        }
        ++tile_it;
      }
      // ---------------------------------------------------- epilogue
      // first global write of this CTA: the predecessor grids (append; transitively the previous
      // step's combine, which reads the partial buffers and writes `out`) must have completed
      if (!pdl_done) { pdl_wait(); pdl_done = true; }
      if (nt > 0) {
        mbar_wait(bo_full(q), seg_it & 1);
        tc_fence_after();
      }
      float inv_l = l > 0.f ? 1.f / l : 0.f;                // coefficient of this set's accumulator
      float lse2 = l > 0.f ? m_used + log2f(l) : -INFINITY;
      const float osc = inv_l;
      bool pub = false, pub_fence = false;
      if (sv.part_base < 0) {
        __nv_bfloat16* orow = reinterpret_cast<__nv_bfloat16*>(p.out) + ((int64_t)tok * p.Hq + head) * p.D;
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          uint32_t o[32];
          tmem_ld32(t_o + ch * 32, o);
          tmem_wait_ld();
          if (row_valid) {
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
              uint4 w;
              w.x = pack_bf16x2(__uint_as_float(o[i]) * osc, __uint_as_float(o[i + 1]) * osc);
              w.y = pack_bf16x2(__uint_as_float(o[i + 2]) * osc, __uint_as_float(o[i + 3]) * osc);
              w.z = pack_bf16x2(__uint_as_float(o[i + 4]) * osc, __uint_as_float(o[i + 5]) * osc);
              w.w = pack_bf16x2(__uint_as_float(o[i + 6]) * osc, __uint_as_float(o[i + 7]) * osc);
              *reinterpret_cast<uint4*>(orow + ch * 32 + i) = w;
            }
          }
        }
        if (row_valid && p.lse) p.lse[(int64_t)tok * p.Hq + head] = lse2 * 0.6931471805599453f;
      } else {
        const int64_t prow = (int64_t)part_slot * kPairRows + R;
        float* orow = p.part_o + prow * p.D;
        // Last segment of this CTA: nothing else will use the Q tiles (set 0: every S MMA has completed
        // once o_full(0) fired) or the K/V ring (set 1 / decode plan: every MMA has completed), so the
        // warp stages its 32 rows x 512 B there and writes them with ONE 16 KB bulk store; rows are
        // contiguous in the partial buffer.  Otherwise: direct 16-byte stores (same chunk positions).
        const bool staged = si + 1 == seg_hi && __all_sync(0xffffffffu, row_valid);   // (few valid rows, e.g. decode steps: store just those)
        const uint32_t stage = (q == 1 ? sRing : sQ) + (uint32_t)(warp & 3) * 16384u + (uint32_t)lane * 512u;
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          uint32_t o[32];
          tmem_ld32(t_o + ch * 32, o);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * osc);
          if (staged) {
#pragma unroll
            for (int i = 0; i < 32; i += 4)
              st_shared_v4(stage + (uint32_t)part_chunk_pos(ch * 8 + i / 4, lane) * 16u, o[i], o[i + 1], o[i + 2], o[i + 3]);
          } else if (row_valid) {
#pragma unroll
            for (int i = 0; i < 32; i += 4)
              *reinterpret_cast<uint4*>(orow + part_chunk_pos(ch * 8 + i / 4, R) * 4) = make_uint4(o[i], o[i + 1], o[i + 2], o[i + 3]);
          }
        }
        if (staged) {
          bars->lse_stage[R] = lse2;
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            bulk_store(p.part_o + (prow - lane) * p.D, stage - (uint32_t)lane * 512u, 16384u);
            bulk_store(p.part_lse + (prow - lane), smem_u32(&bars->lse_stage[R - lane]), 128u);
            bulk_commit();
            bulk_wait_all();
          }
          __syncwarp();
        }
        if (!staged && row_valid) p.part_lse[prow] = lse2;
        pub = true; pub_fence = !staged;
      }
      tc_fence_before();
      mbar_arrive(bo_empty(q));
      if (pub) publish(pub_fence);
      ++seg_it;
    }
    if (fused && hdr.num_combine > 0) {
      // ---------------------------------------------------- merge phase (a4)
      uint32_t merge_phase = 0;
      asm volatile("bar.sync 1, 256;" ::: "memory");        // jobs[] written by thread 0 are visible
      const int32_t njobs = bars->njobs;
      int32_t jn = 0;
      for (int32_t si = seg_lo; si < seg_hi && jn < njobs; ++si) {
        MergeJob job;
        if (njobs <= kMaxJobs) {
          job = bars->jobs[jn];
        } else {
          // more partial segments than parked jobs (many tiny groups per team): re-derive from the metadata
          SegView sv;
          if (!load_segment(meta, hdr, si, pair, tok_per_pair, sv) || sv.part_base < 0) continue;
          make_job(sv, job);
        }
        ++jn;
        int32_t* ctr = p.merge_ctr + job.slot0;
        if (warp == 0 && lane == 0) {       // the other warps meet this one on the barrier inside merge_item
          // relaxed polls (an acquire load also invalidates L1 on every iteration), one acquire at the end
          while (ld_relaxed_gpu(ctr) < 2 * job.nparts) {}
          (void)ld_acquire_gpu(ctr);
        }
        __syncwarp();
        merge_item(p, job, (int32_t)(kRingBytes / 512), sRing, smem_raw + (sRing - smem_u32(smem_raw)), sQ,
                   smem_raw + (sQ - smem_u32(smem_raw)), smem_u32(&bars->merge_full), merge_phase, warp, lane);
        __syncwarp();
        if (warp == 0 && lane == 0) {
          // the last CTA to get here re-arms the counters for the next launch (every part has been
          // published and every waiter has passed its wait by then)
          int32_t* done = ctr + p.max_part_slots;
          if (atomicAdd(done, 1) == job.nparts - 1) { *done = 0; *ctr = 0; }
        }
      }
    }
  }

  // (placed after the softmax code: the hot loops of producer, MMA issuer and softmax stay close together)
  if (warp >= 10 && p.append_tokens > 0) {
    // ===================================================== a2 inside the fused step (kv_append.cuh)
    // The pool rows and page-table entries written here are not read by this launch (its KV tiles over
    // the new block come from k_new / v_new); at most the masked tail of a session's last cache page is
    // overwritten while a tile holding it is in flight, which changes nothing: those keys carry P = 0
    // and the bytes are finite before and after.
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
    tmem_dealloc<kTmemCols>(tmem_base);
  }
}

cudaError_t sm100_attn_configure() {
  const void* fns[2] = {(const void*)attn_sm100_kernel<kInlineAttnWords>,
                        (const void*)attn_sm100_kernel<kInlineAttnWordsLarge>};
  for (const void* f : fns) {
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_attn_sm100(const Sm100Launch& l, cudaStream_t stream) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(l.num_ctas); cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = kSmemBytes; cfg.stream = stream;
  cudaLaunchAttribute at[2];
  int na = 0;
  if (l.p.merge_ctr != nullptr) {
    // fused combine: CTAs wait on each other's partials, so the whole grid must be co-resident
    at[na].id = cudaLaunchAttributeCooperative;
    at[na].val.cooperative = 1;
    ++na;
  }
  at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[na].val.programmaticStreamSerializationAllowed = 1;
  ++na;
  cfg.attrs = at; cfg.numAttrs = na;
  if (l.inl_words <= kInlineAttnWords) {
    InlineAttnMeta small;
    memcpy(small.w, l.inl.w, sizeof(small.w));
    return cudaLaunchKernelEx(&cfg, attn_sm100_kernel<kInlineAttnWords>, l.tmap_q, l.tmap_k, l.tmap_v,
                              l.tmap_kn, l.tmap_vn, small, l.app, l.peers, l.p);
  }
  return cudaLaunchKernelEx(&cfg, attn_sm100_kernel<kInlineAttnWordsLarge>, l.tmap_q, l.tmap_k, l.tmap_v,
                            l.tmap_kn, l.tmap_vn, l.inl, l.app, l.peers, l.p);
}

}  // namespace ws

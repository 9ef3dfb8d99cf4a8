// combine.cu - a4: split-KV combine as its own kernel (the default; WS_FLAG_FUSED_COMBINE moves the same
// merge into the attention kernel).  The paper is silent on this step; north_star names it.
// Attention over a disjoint union of key ranges is the LSE-weighted mean of the per-range results (merge.cuh).
// HBM/L2-bound: reads nparts x rows x (D+1) fp32 per (group, pair), writes bf16 O (+ fp32 LSE).
//
// One 256-thread block merges up to 32 packed rows of one (combine item, row-tile pair).  The rows of
// one part are contiguous in the partial buffer ([slot][256 rows][128] fp32), so the block fetches each
// part with ONE bulk copy (cp.async.bulk, completion on an mbarrier) into shared memory - every byte the
// block needs is in flight at once, a single exposed L2/HBM latency - and then merges from shared memory
// (merge_item, shared with the fused path).  The earlier one-warp-per-row version paid two dependent
// global latencies per row (LSEs, then O rows): 11-15 us per config-4 step against ~2.5 us of L2 traffic.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <string.h>

#include "launch.h"
#include "merge.cuh"

namespace ws {

// ---- row-per-warp variant: few rows with many parts each (decode steps, heavily split short steps) ----
// One warp per packed row: lane s loads the LSE of part s, the max and the weight sum are reduced with warp
// shuffles, then the parts' O rows (one float4 per lane, D = 128) are accumulated with kDepth loads in flight
// per lane.  Two dependent global latencies per row, but thousands of independent warps: better than the
// staged kernel below when a block would stage only a handful of rows.
constexpr int kCombineRowsPerBlock = 8;

// kDepth = O-row loads in flight per lane: 4 keeps the kernel at 64 registers (8 blocks / SM) for
// the large grids of the general plan; 20 serves the small grids of decode steps (one 65k-key step has 18-19
// parts per row), where few warps have work, memory-level parallelism has to come from each of them, and the
// O rows are requested together with the LSEs (kEager).
template <int kInlW, int kDepth>
__global__ void __launch_bounds__(kCombineRowsPerBlock * 32)
combine_rows_kernel(AttnParams p, const __grid_constant__ InlineMeta<kInlW> inl, int32_t team_size, int32_t blocks_per_pair) {
  // The successor (the next step's append or attention kernel) may be scheduled at once: before its own
  // griddepcontrol.wait it touches nothing this kernel or the attention kernel before it writes (launch.h).
  pdl_launch_dependents();
  pdl_wait();                      // partials of the attention kernel launched just before
  const MetaView<kInlW> meta{p.meta, inl};
  const AttnMeta hdr = meta.template load<AttnMeta>(0);
  int32_t b = blockIdx.x;
  const int32_t rchunk = b % blocks_per_pair; b /= blocks_per_pair;
  const int32_t pair = b % team_size;
  const int32_t item = b / team_size;
  const CombineItem ci = meta.template load<CombineItem>(hdr.off_combine + item * (int32_t)(sizeof(CombineItem) / 4));
  const Group g = meta.template load<Group>(hdr.off_groups + ci.group * (int32_t)(sizeof(Group) / 4));
  if (pair >= g.npairs) return;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int32_t r = rchunk * kCombineRowsPerBlock + wib;
  const int32_t tok = g.q_token0 + pair * (kPairRows / p.G) + r / p.G;
  if (tok >= g.q_token_end) return;
  const int32_t head = g.kv_head * p.G + r % p.G;
  const int64_t slot0 = ci.part_base + pair;            // slot(i) = slot0 + i * npairs
  const int64_t stride = g.npairs;

  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  float mx_run = -INFINITY, wsum_run = 0.f;
  // parts are processed in chunks of 32 (one LSE per lane); a chunk's results are merged into the
  // running (max, sum, acc) with the usual rescale - almost always there is a single chunk
  for (int32_t base = 0; base < ci.nparts; base += 32) {
    const int32_t i = base + lane;
    const float l2 = i < ci.nparts ? p.part_lse[(slot0 + i * stride) * kPairRows + r] : -INFINITY;
    const int32_t cnt = min(32, ci.nparts - base);
    // Deep variant (few rows, many parts: decode steps): the first kDepth O rows are requested TOGETHER with the
    // LSEs - their addresses do not depend on them - so the row pays one round trip instead of two.
    constexpr bool kEager = kDepth > 8;
    float4 o0[kEager ? kDepth : 1];
    if constexpr (kEager) {
#pragma unroll
      for (int u = 0; u < kDepth; ++u)
        o0[u] = u < cnt ? reinterpret_cast<const float4*>(p.part_o + ((slot0 + (base + u) * stride) * kPairRows + r) * p.D)[lane]
                        : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float mx = l2;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    const float mx_new = fmaxf(mx_run, mx);
    if (mx_new == -INFINITY) continue;                  // nothing visible in these parts
    const float w = l2 == -INFINITY ? 0.f : exp2f(l2 - mx_new);
    float ws = w;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ws += __shfl_xor_sync(0xffffffffu, ws, o);
    const float rescale = mx_run == -INFINITY ? 0.f : exp2f(mx_run - mx_new);
    acc.x *= rescale; acc.y *= rescale; acc.z *= rescale; acc.w *= rescale;
    wsum_run = wsum_run * rescale + ws;
    mx_run = mx_new;
    for (int32_t k0 = 0; k0 < cnt; k0 += kDepth) {
      float4 o[kDepth];
      float wk[kDepth];
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        const int32_t k = k0 + u;
        wk[u] = __shfl_sync(0xffffffffu, w, k & 31);
        if (kEager && k0 == 0) {
          // (requested above; a part with weight 0 - an empty range - may hold stale bytes: not used)
          if (k < cnt && wk[u] != 0.f) o[u] = o0[u];
          else { o[u] = make_float4(0.f, 0.f, 0.f, 0.f); wk[u] = 0.f; }
        } else if (k < cnt && wk[u] != 0.f) {
          o[u] = reinterpret_cast<const float4*>(p.part_o + ((slot0 + (base + k) * stride) * kPairRows + r) * p.D)[lane];
        } else { o[u] = make_float4(0.f, 0.f, 0.f, 0.f); wk[u] = 0.f; }
      }
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        acc.x = fmaf(wk[u], o[u].x, acc.x); acc.y = fmaf(wk[u], o[u].y, acc.y);
        acc.z = fmaf(wk[u], o[u].z, acc.z); acc.w = fmaf(wk[u], o[u].w, acc.w);
      }
    }
  }
  const float inv = 1.f / wsum_run;
  __nv_bfloat162 lo = __floats2bfloat162_rn(acc.x * inv, acc.y * inv);
  __nv_bfloat162 hi = __floats2bfloat162_rn(acc.z * inv, acc.w * inv);
  uint2 packed;
  packed.x = *reinterpret_cast<uint32_t*>(&lo);
  packed.y = *reinterpret_cast<uint32_t*>(&hi);
  __nv_bfloat16* orow = reinterpret_cast<__nv_bfloat16*>(p.out) + ((int64_t)tok * p.Hq + head) * p.D;
  reinterpret_cast<uint2*>(orow)[lane ^ (r & 7)] = packed;   // partial rows store chunk c at position c ^ (r & 7) (attn_sm100.cu)
  if (p.lse && lane == 0)
    p.lse[(int64_t)tok * p.Hq + head] = (mx_run + log2f(wsum_run)) * 0.6931471805599453f;
}


// ---- staged variant ----
constexpr int kStagedMaxParts = 8;                     // more parts per row than this: row-per-warp variant (12 measured the same)
constexpr int kCombineRowsMax = 64;                    // rows per block (fewer when a row has many parts)
constexpr int kCombineRowsCap = 192;                   // staged rows x parts per chunk: 96 KB -> 2 blocks / SM
constexpr uint32_t kCombineLseBytes = 8192;            // nparts x (rows + 8) fp32, nparts <= 148
constexpr uint32_t kCombineSmem = kCombineRowsCap * 512 + kCombineLseBytes + 1024;

template <int kInlW>
__global__ void __launch_bounds__(256)
combine_kernel(AttnParams p, const __grid_constant__ InlineMeta<kInlW> inl, int32_t team_size, int32_t rows_pb) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t bar;
  pdl_launch_dependents();         // see combine_rows_kernel
  if (p.meta != nullptr) pdl_wait();
  const uint32_t sO = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint8_t* o_s = smem_raw + (sO - smem_u32(smem_raw));
  const uint32_t sLse = sO + kCombineRowsCap * 512;
  const MetaView<kInlW> meta{p.meta, inl};
  const AttnMeta hdr = meta.template load<AttnMeta>(0);
  const int32_t chunks = (kPairRows + rows_pb - 1) / rows_pb;
  int32_t b = blockIdx.x;
  const int32_t rchunk = b % chunks; b /= chunks;
  const int32_t pair = b % team_size;
  const int32_t item = b / team_size;
  const CombineItem ci = meta.template load<CombineItem>(hdr.off_combine + item * (int32_t)(sizeof(CombineItem) / 4));
  const Group g = meta.template load<Group>(hdr.off_groups + ci.group * (int32_t)(sizeof(Group) / 4));
  MergeJob job;
  job.slot0 = ci.part_base + pair; job.nparts = ci.nparts; job.npairs = g.npairs; job.kv_head = g.kv_head;
  job.tok0 = g.q_token0 + pair * (kPairRows / p.G);
  const int32_t nv = min(hdr.alt ? kTileRows : kPairRows, (min(g.q_token_end, job.tok0 + kPairRows / p.G) - job.tok0) * p.G);
  job.r_lo = rchunk * rows_pb; job.r_hi = min(nv, job.r_lo + rows_pb); job.pad = 0;
  const bool active = pair < g.npairs && job.r_lo < job.r_hi;     // block-uniform
  if (threadIdx.x == 0) { mbar_init(smem_u32(&bar), 1); fence_mbar_init(); }
  __syncthreads();
  pdl_wait();                      // partials of the attention kernel launched just before
  if (!active) return;
  uint32_t phase = 0;
  // the LSE area holds nparts x ((rows + 8) & ~3) floats: shrink the chunk for very many parts
  const int32_t lse_cap = (int32_t)(kCombineLseBytes / 4) / ci.nparts - 8;
  merge_item(p, job, min(kCombineRowsCap, max(1, lse_cap) * ci.nparts), sO, o_s, sLse,
             smem_raw + (sLse - smem_u32(smem_raw)), smem_u32(&bar), phase, (int)(threadIdx.x >> 5), (int)(threadIdx.x & 31));
}

cudaError_t combine_configure() {
  cudaError_t e = cudaFuncSetAttribute((const void*)combine_kernel<kInlineAttnWords>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kCombineSmem);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute((const void*)combine_kernel<kInlineAttnWordsLarge>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kCombineSmem);
}

cudaError_t launch_combine(const AttnParams& p, const InlineAttnMetaLarge& inl, int32_t inl_words,
                           int32_t num_combine, int32_t team_size, int32_t max_parts, int32_t max_rows_per_pair,
                           cudaStream_t stream) {
  if (num_combine == 0) return cudaSuccess;
  const bool small_tier = inl_words <= kInlineAttnWords;
  InlineAttnMeta small;
  if (small_tier) memcpy(small.w, inl.w, sizeof(small.w));
  if (max_parts > kStagedMaxParts) {
    // many parts per row: a staged block would hold only a few rows - one warp per row instead
    // blocks only for the packed rows a pair can hold in this call (a one-token decode step has G rows per group:
    // one block instead of 32, of which 31 would find nothing to do)
    const int32_t rows = std::max(1, std::min<int32_t>(kPairRows, max_rows_per_pair));
    const int32_t bpp = (rows + kCombineRowsPerBlock - 1) / kCombineRowsPerBlock;
    const int32_t grid = num_combine * team_size * bpp;
    const dim3 g(grid), b(kCombineRowsPerBlock * 32);
    const bool deep = grid <= 148;                      // (205 registers: one block per SM)
    if (small_tier) {
      if (deep) return launch_pdl(combine_rows_kernel<kInlineAttnWords, 20>, g, b, 0, stream, p, small, team_size, bpp);
      return launch_pdl(combine_rows_kernel<kInlineAttnWords, 4>, g, b, 0, stream, p, small, team_size, bpp);
    }
    if (deep) return launch_pdl(combine_rows_kernel<kInlineAttnWordsLarge, 20>, g, b, 0, stream, p, inl, team_size, bpp);
    return launch_pdl(combine_rows_kernel<kInlineAttnWordsLarge, 4>, g, b, 0, stream, p, inl, team_size, bpp);
  }
  // rows per block: as many as fit the staging area in one piece for the item with the most parts
  const int32_t rows_pb = std::max(1, std::min(kCombineRowsMax, kCombineRowsCap / std::max(1, max_parts)));
  const int32_t grid = num_combine * team_size * ((kPairRows + rows_pb - 1) / rows_pb);
  const dim3 g(grid), b(256);
  if (small_tier) return launch_pdl(combine_kernel<kInlineAttnWords>, g, b, kCombineSmem, stream, p, small, team_size, rows_pb);
  return launch_pdl(combine_kernel<kInlineAttnWordsLarge>, g, b, kCombineSmem, stream, p, inl, team_size, rows_pb);
}

}  // namespace ws

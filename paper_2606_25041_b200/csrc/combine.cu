// combine.cu - a4: split-KV combine.  The paper is silent on this step; north_star names it.
// Attention over a disjoint union of key ranges is the LSE-weighted mean of the per-range results:
//   m* = max_s LSE_s ; w_s = 2^(LSE_s - m*) ; O = sum_s w_s O_s / sum_s w_s ; LSE = m* + log2 sum_s w_s
// (partials carry log2-domain LSEs; an empty range carries LSE = -inf and contributes w = 0).
// HBM/L2-bound: reads nparts x 256 x (D+1) fp32 per (group, pair), writes bf16 O (+ fp32 LSE).
// One warp per packed row: lane s loads the LSE of part s, the max and the weight sum are reduced
// with warp shuffles, then the parts' O rows (one float4 per lane, D = 128) are accumulated with
// kDepth loads in flight per lane.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <string.h>

#include "launch.h"

namespace ws {

constexpr int kCombineRowsPerBlock = 8;

// kDepth = O-row loads in flight per lane: 4 keeps the kernel at 64 registers (8 blocks / SM) for
// the large grids of the general plan; 8 serves the small grids of decode steps, where few warps
// have work and memory-level parallelism has to come from each of them.
template <int kInlW, int kDepth>
__global__ void __launch_bounds__(kCombineRowsPerBlock * 32)
combine_kernel(AttnParams p, const __grid_constant__ InlineMeta<kInlW> inl, int32_t team_size) {
  pdl_wait();                      // partials of the attention kernel launched just before
  pdl_launch_dependents();         // the next step's append does not depend on this kernel
  if (p.meta == nullptr) p.meta = inl.w;
  const AttnMeta hdr = *reinterpret_cast<const AttnMeta*>(p.meta);
  const int32_t blocks_per_pair = kPairRows / kCombineRowsPerBlock;
  int32_t b = blockIdx.x;
  const int32_t rchunk = b % blocks_per_pair; b /= blocks_per_pair;
  const int32_t pair = b % team_size;
  const int32_t item = b / team_size;
  const CombineItem ci = reinterpret_cast<const CombineItem*>(p.meta + hdr.off_combine)[item];
  const Group g = reinterpret_cast<const Group*>(p.meta + hdr.off_groups)[ci.group];
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
    const int32_t cnt = min(32, ci.nparts - base);
    for (int32_t k0 = 0; k0 < cnt; k0 += kDepth) {
      float4 o[kDepth];
      float wk[kDepth];
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        const int32_t k = k0 + u;
        wk[u] = __shfl_sync(0xffffffffu, w, k & 31);
        if (k < cnt && wk[u] != 0.f)
          o[u] = reinterpret_cast<const float4*>(p.part_o + ((slot0 + (base + k) * stride) * kPairRows + r) * p.D)[lane];
        else { o[u] = make_float4(0.f, 0.f, 0.f, 0.f); wk[u] = 0.f; }
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

cudaError_t launch_combine(const AttnParams& p, const InlineAttnMetaLarge& inl, int32_t inl_words,
                           int32_t num_combine, int32_t team_size, cudaStream_t stream) {
  if (num_combine == 0) return cudaSuccess;
  int32_t grid = num_combine * team_size * (kPairRows / kCombineRowsPerBlock);
  const dim3 g(grid), b(kCombineRowsPerBlock * 32);
  const bool deep = grid <= 2 * 148;
  if (inl_words <= kInlineAttnWords) {
    InlineAttnMeta small;
    memcpy(small.w, inl.w, sizeof(small.w));
    if (deep) return launch_pdl(combine_kernel<kInlineAttnWords, 8>, g, b, 0, stream, p, small, team_size);
    return launch_pdl(combine_kernel<kInlineAttnWords, 4>, g, b, 0, stream, p, small, team_size);
  }
  if (deep) return launch_pdl(combine_kernel<kInlineAttnWordsLarge, 8>, g, b, 0, stream, p, inl, team_size);
  return launch_pdl(combine_kernel<kInlineAttnWordsLarge, 4>, g, b, 0, stream, p, inl, team_size);
}

}  // namespace ws

// combine.cu - a4: split-KV combine.  The paper is silent on this step; north_star names it.
// Attention over a disjoint union of key ranges is the LSE-weighted mean of the per-range results:
//   m* = max_s LSE_s ; w_s = 2^(LSE_s - m*) ; O = sum_s w_s O_s / sum_s w_s ; LSE = m* + log2 sum_s w_s
// (partials carry log2-domain LSEs; an empty range carries LSE = -inf and contributes w = 0).
// HBM/L2-bound: reads nparts x 256 x (D+1) fp32 per (group, pair), writes bf16 O (+ fp32 LSE).
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>

#include "launch.h"

namespace ws {

constexpr int kCombineRowsPerBlock = 8;   // one warp per packed row, D = 128 -> one float4 per lane

__global__ void __launch_bounds__(kCombineRowsPerBlock * 32)
combine_kernel(AttnParams p, const __grid_constant__ InlineAttnMeta inl, int32_t team_size) {
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

  float mx = -INFINITY;
  for (int i = 0; i < ci.nparts; ++i) {
    int64_t slot = ci.part_base + (int64_t)i * g.npairs + pair;
    mx = fmaxf(mx, p.part_lse[slot * kPairRows + r]);
  }
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  float wsum = 0.f;
  for (int i = 0; i < ci.nparts; ++i) {
    int64_t slot = ci.part_base + (int64_t)i * g.npairs + pair;
    float l2 = p.part_lse[slot * kPairRows + r];
    if (l2 == -INFINITY) continue;
    float w = exp2f(l2 - mx);
    const float4 o = reinterpret_cast<const float4*>(p.part_o + (slot * kPairRows + r) * p.D)[lane];
    acc.x = fmaf(w, o.x, acc.x); acc.y = fmaf(w, o.y, acc.y);
    acc.z = fmaf(w, o.z, acc.z); acc.w = fmaf(w, o.w, acc.w);
    wsum += w;
  }
  const float inv = 1.f / wsum;
  __nv_bfloat162 lo = __floats2bfloat162_rn(acc.x * inv, acc.y * inv);
  __nv_bfloat162 hi = __floats2bfloat162_rn(acc.z * inv, acc.w * inv);
  uint2 packed;
  packed.x = *reinterpret_cast<uint32_t*>(&lo);
  packed.y = *reinterpret_cast<uint32_t*>(&hi);
  __nv_bfloat16* orow = reinterpret_cast<__nv_bfloat16*>(p.out) + ((int64_t)tok * p.Hq + head) * p.D;
  reinterpret_cast<uint2*>(orow)[lane] = packed;
  if (p.lse && lane == 0)
    p.lse[(int64_t)tok * p.Hq + head] = (mx + log2f(wsum)) * 0.6931471805599453f;
}

cudaError_t launch_combine(const AttnParams& p, const InlineAttnMeta& inl, int32_t num_combine,
                           int32_t team_size, cudaStream_t stream) {
  if (num_combine == 0) return cudaSuccess;
  int32_t grid = num_combine * team_size * (kPairRows / kCombineRowsPerBlock);
  return launch_pdl(combine_kernel, dim3(grid), dim3(kCombineRowsPerBlock * 32), 0, stream, p, inl,
                    team_size);
}

}  // namespace ws

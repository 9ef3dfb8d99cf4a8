// merge.cuh - a4: LSE-weighted merge of split-KV partials, shared by combine_kernel (combine.cu) and the
// fused merge phase of attn_sm100_kernel (attn_sm100.cu).  The paper is silent on this step; north_star
// names it ("a split-KV combine kernel").
//   m* = max_s LSE_s ; w_s = 2^(LSE_s - m*) ; O = sum_s w_s O_s / sum_s w_s ; LSE = m* + log2 sum_s w_s
// (partials carry log2-domain LSEs; an empty range carries LSE = -inf and contributes w = 0).
#pragma once
#include <cuda_bf16.h>
#include <math.h>
#include <stdint.h>

#include "sm100_ptx.cuh"
#include "ws_internal.h"

namespace ws {

using namespace ptx;

// One merge duty of this CTA (fused combine): rows [r_lo, r_hi) of the (item, pair) whose partial slots
// are slot0 + i * npairs, i < nparts.  Resolved from the metadata when the segment starts (off the
// critical path) and parked in shared memory until the merge phase.
struct MergeJob {
  int32_t slot0, nparts, npairs, kv_head, tok0, r_lo, r_hi, pad;
};

// Partial-row storage format (private to the writers and the mergers): the 16-byte chunk c of packed row
// r (4 of the row's 128 fp32) lives at chunk position c ^ (r & 7) of the row's 512 bytes.  The XOR makes
// the thread-per-row shared-memory staging of the epilogue conflict-free (8 consecutive rows hit 8
// different 16-byte bank groups) while a row stays one contiguous 512-byte run in global memory.
__device__ __forceinline__ int part_chunk_pos(int c, int r) { return c ^ (r & 7); }

// The 256 softmax threads (8 warps) merge packed rows [r_lo, r_hi) of one (item, pair).  The rows'
// partials are contiguous per part ([slot][256 rows][128] fp32, [slot][256] LSEs), so each part is ONE
// bulk copy of O rows into the (idle) K/V ring plus one of LSEs into the (idle) Q tiles; every copy of
// the item is in flight at once and the merge itself reads shared memory only.  Warp w handles rows
// w, w + 8, ...; lane = 16-byte chunk position of the row.  Every lane recomputes the row's weights
// from the LSEs (broadcast shared-memory reads: no shuffles), kMR rows interleaved for ILP.
constexpr int kMR = 4;
__device__ __forceinline__ void merge_item(const AttnParams& p, const MergeJob& job, int32_t rows_cap,
                                           uint32_t sRing, const uint8_t* ring, uint32_t sLse, const uint8_t* lse_s,
                                           uint32_t bar, uint32_t& phase, int warp, int lane) {
  const int32_t nparts = job.nparts, r_lo = job.r_lo, r_hi = job.r_hi, tok0 = job.tok0;
  const int64_t slot0 = job.slot0, stride = job.npairs;
  if (r_hi <= r_lo) return;
  const int32_t rc = min(r_hi - r_lo, max(1, rows_cap / nparts));
  const int32_t lse_stride = (rc + 8) & ~3;                 // floats per part in the LSE staging area
  for (int32_t c0 = r_lo; c0 < r_hi; c0 += rc) {
    const int32_t n = min(rc, r_hi - c0);
    const int32_t c0a = c0 & ~3, nl = ((c0 + n + 3) & ~3) - c0a;   // 16-byte aligned LSE run covering [c0, c0 + n)
    asm volatile("bar.sync 1, 256;" ::: "memory");          // ring idle: all MMAs of this CTA / the previous chunk done
    if (warp == 0) {
      fence_proxy_async_all();            // the parts were written through the generic proxy (other CTAs)
      if (lane == 0) mbar_arrive_expect_tx(bar, (uint32_t)((n * 512 + nl * 4) * nparts));
      __syncwarp();
      for (int32_t part = lane; part < nparts; part += 32) {
        bulk_load(sRing + (uint32_t)(part * rc) * 512u,
                  p.part_o + ((slot0 + part * stride) * kPairRows + c0) * 128, (uint32_t)n * 512u, bar);
        bulk_load(sLse + (uint32_t)(part * lse_stride) * 4u,
                  p.part_lse + (slot0 + part * stride) * kPairRows + c0a, (uint32_t)nl * 4u, bar);
      }
    }
    mbar_wait(bar, phase);
    phase ^= 1u;
    const float* lse_f = reinterpret_cast<const float*>(lse_s) + (c0 - c0a);
    const float4* o_f = reinterpret_cast<const float4*>(ring) + lane;
    for (int32_t lr0 = warp; lr0 < n; lr0 += 8 * kMR) {
      float mx[kMR], ws[kMR];
      float4 acc[kMR];
      const float* lp[kMR];
      const float4* op[kMR];
#pragma unroll
      for (int b = 0; b < kMR; ++b) {
        const int32_t lr = min(lr0 + 8 * b, n - 1);         // (rows past the end repeat the last one; not stored)
        lp[b] = lse_f + lr; op[b] = o_f + lr * 32;
        mx[b] = -INFINITY; ws[b] = 0.f; acc[b] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      if (nparts <= 8) {
        // common case: every load of the batch is issued before the first use (unrolled over the parts)
        float lv[kMR][8];
#pragma unroll
        for (int k = 0; k < 8; ++k)
#pragma unroll
          for (int b = 0; b < kMR; ++b) {
            lv[b][k] = k < nparts ? lp[b][k * lse_stride] : -INFINITY;
            mx[b] = fmaxf(mx[b], lv[b][k]);
          }
#pragma unroll
        for (int k = 0; k < 8; ++k)
          if (k < nparts) {
#pragma unroll
            for (int b = 0; b < kMR; ++b) {
              const float w = lv[b][k] == -INFINITY ? 0.f : ex2_approx(lv[b][k] - mx[b]);
              const float4 v = op[b][k * rc * 32];
              ws[b] += w;
              acc[b].x = fmaf(w, v.x, acc[b].x); acc[b].y = fmaf(w, v.y, acc[b].y);
              acc[b].z = fmaf(w, v.z, acc[b].z); acc[b].w = fmaf(w, v.w, acc[b].w);
            }
          }
      } else {
        for (int32_t k = 0; k < nparts; ++k)
#pragma unroll
          for (int b = 0; b < kMR; ++b) mx[b] = fmaxf(mx[b], lp[b][k * lse_stride]);
        for (int32_t k = 0; k < nparts; ++k) {
#pragma unroll
          for (int b = 0; b < kMR; ++b) {
            const float lv = lp[b][k * lse_stride];
            const float w = lv == -INFINITY ? 0.f : ex2_approx(lv - mx[b]);   // (mx = -inf only if every lv is)
            const float4 v = op[b][k * rc * 32];
            ws[b] += w;
            acc[b].x = fmaf(w, v.x, acc[b].x); acc[b].y = fmaf(w, v.y, acc[b].y);
            acc[b].z = fmaf(w, v.z, acc[b].z); acc[b].w = fmaf(w, v.w, acc[b].w);
          }
        }
      }
      // branch-free up to the stores, so that the kMR rows' address / normalisation chains interleave
      uint2 packed[kMR];
      uint2* dst[kMR];
      float* ldst[kMR];
      float lse_out[kMR];
      const uint32_t G = (uint32_t)p.G;
#pragma unroll
      for (int b = 0; b < kMR; ++b) {
        const uint32_t r = (uint32_t)(c0 + min(lr0 + 8 * b, n - 1));
        const uint32_t dt = r / G, hh = r - dt * G;
        const int64_t row = (int64_t)(tok0 + (int32_t)dt) * p.Hq + job.kv_head * p.G + (int32_t)hh;
        const float inv = ws[b] > 0.f ? __fdividef(1.f, ws[b]) : 0.f;
        packed[b].x = pack_bf16x2(acc[b].x * inv, acc[b].y * inv);
        packed[b].y = pack_bf16x2(acc[b].z * inv, acc[b].w * inv);
        dst[b] = reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(p.out) + row * p.D) + part_chunk_pos(lane, (int)r);
        ldst[b] = p.lse + row;
        lse_out[b] = ws[b] > 0.f ? (mx[b] + __log2f(ws[b])) * 0.6931471805599453f : -INFINITY;
      }
#pragma unroll
      for (int b = 0; b < kMR; ++b)
        if (lr0 + 8 * b < n) {
          *dst[b] = packed[b];                              // this lane holds logical chunk lane ^ (r & 7)
          if (p.lse && lane == 0) *ldst[b] = lse_out[b];
        }
    }
  }
}

}  // namespace ws

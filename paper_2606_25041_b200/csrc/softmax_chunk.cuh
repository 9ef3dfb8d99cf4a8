// softmax_chunk.cuh - the per-chunk exponential code shared by the attention kernels (attn_sm100.cu and the
// decode kernel attn_dec_sm100.cu): p = 2^(s * c - m) for 32 scores of a row, packed fp32x2 arithmetic, a share
// of the exponentials as a polynomial on the FMA pipe, bf16 packing of P, fp32 row sums from the unrounded p
// (reading A10).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sm100_ptx.cuh"

namespace ws {

using namespace ptx;

// 2 of every 8 exponentials run as a polynomial on the FMA pipe (ex2_poly2); sweep: DESIGN.md section 8
constexpr int kPolyPer8 = 2;

// 2^x for a PAIR of values on the FMA/ALU pipes (no MUFU): round-to-nearest split x = r + f with
// f in [-0.5, 0.5], a degree-3 minimax polynomial for 2^f (max relative error 7.5e-5, well inside
// one bf16 ulp of P) in packed f32x2 arithmetic, and an exponent-field add per element.  Used for
// kPolyPer8 of every 8 exponentials (2 = 25 %) to take load off the 16/clk/SM MUFU.
__device__ __forceinline__ void ex2_poly2(uint64_t x2, float& p0, float& p1) {
  float x0, x1;
  unpack_f32x2(x2, x0, x1);
  const uint64_t xc = pack_f32x2(fmaxf(x0, -126.f), fmaxf(x1, -126.f));
  const uint64_t magic = pack_f32x2(12582912.f, 12582912.f);   // 1.5 * 2^23: integer part -> LSBs
  const uint64_t t = add_f32x2(xc, magic);
  const uint64_t f = sub_f32x2(xc, sub_f32x2(t, magic));
  uint64_t p = fma_f32x2(f, pack_f32x2(0.055171459913253784f, 0.055171459913253784f),
                         pack_f32x2(0.2426108568906784f, 0.2426108568906784f));
  p = fma_f32x2(p, f, pack_f32x2(0.6932609677314758f, 0.6932609677314758f));
  p = fma_f32x2(p, f, pack_f32x2(0.9999281167984009f, 0.9999281167984009f));
  float t0, t1, q0, q1;
  unpack_f32x2(t, t0, t1);
  unpack_f32x2(p, q0, q1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}


// One 32-column chunk of a softmax row: p = 2^(s*c - m), running sums, running max of s, bf16 pack.
__device__ __forceinline__ void softmax_chunk(const uint32_t* sr, float c, float neg_mc,
                                              uint64_t& l01, uint64_t& l23, uint32_t* pk) {
  const uint64_t c2 = pack_f32x2(c, c), nm2 = pack_f32x2(neg_mc, neg_mc);
#pragma unroll
  for (int i = 0; i < 32; i += 8) {
    float pv[8];
#pragma unroll
    for (int e = 0; e < 8; e += 2) {
      const float s0 = __uint_as_float(sr[i + e]), s1 = __uint_as_float(sr[i + e + 1]);
      const uint64_t x2 = fma_f32x2(pack_f32x2(s0, s1), c2, nm2);
      const int pr = e / 2;
      // kPolyPer8 polynomial exponentials per 8 elements, i.e. kPolyPer8 / 2 pairs per group of 4 pairs; an
      // odd count alternates between rounding down and up from one group to the next
      constexpr int kPolyEven = kPolyPer8 / 2, kPolyOdd = (kPolyPer8 + 1) / 2;
      const int kp = ((i / 8) & 1) ? kPolyOdd : kPolyEven;
      const bool poly = kp > 0 && (pr * kp) / 4 != ((pr + 1) * kp) / 4;
      if (poly) {
        ex2_poly2(x2, pv[e], pv[e + 1]);
      } else {
        float x0, x1;
        unpack_f32x2(x2, x0, x1);
        pv[e] = ex2_approx(x0); pv[e + 1] = ex2_approx(x1);
      }
    }
    l01 = add_f32x2(l01, add_f32x2(pack_f32x2(pv[0], pv[1]), pack_f32x2(pv[4], pv[5])));
    l23 = add_f32x2(l23, add_f32x2(pack_f32x2(pv[2], pv[3]), pack_f32x2(pv[6], pv[7])));
#pragma unroll
    for (int e = 0; e < 8; e += 2) pk[(i + e) / 2] = pack_bf16x2(pv[e], pv[e + 1]);
  }
}

}  // namespace ws

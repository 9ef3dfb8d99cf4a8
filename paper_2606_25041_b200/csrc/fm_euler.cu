// fm_euler.cu - NEXT-2: explicit Euler step of the flow-matching solver on a latent unit.
// PAPER.md:53 Eq. (2): z_tau = (1 - tau) z_0 + tau eps, dz/dtau = eps - z_0; the model predicts that
// velocity (Eq. (3)) and the performer integrates it over a few solver steps
// (PAPER.md:33, :71, :83): z <- z + dtau * v  (dtau < 0 when integrating from noise to data).
// Elementwise, HBM-bound: 3 x count x sizeof(element) bytes; fp32 arithmetic, one rounding to the
// storage dtype.  The step count and schedule are not given in the paper: the caller supplies dtau.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "launch.h"

namespace ws {

__global__ void __launch_bounds__(256)
fm_euler_f32_kernel(float* __restrict__ z, const float* __restrict__ v, float dtau, int64_t n4,
                    int64_t count) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n4) {
    float4 a = reinterpret_cast<float4*>(z)[i];
    const float4 b = reinterpret_cast<const float4*>(v)[i];
    a.x = fmaf(dtau, b.x, a.x); a.y = fmaf(dtau, b.y, a.y);
    a.z = fmaf(dtau, b.z, a.z); a.w = fmaf(dtau, b.w, a.w);
    reinterpret_cast<float4*>(z)[i] = a;
  }
  if (i == 0)
    for (int64_t k = n4 * 4; k < count; ++k) z[k] = fmaf(dtau, v[k], z[k]);
}

__global__ void __launch_bounds__(256)
fm_euler_bf16_kernel(__nv_bfloat16* __restrict__ z, const __nv_bfloat16* __restrict__ v, float dtau,
                     int64_t n8, int64_t count) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n8) {
    uint4 a = reinterpret_cast<uint4*>(z)[i];
    const uint4 b = reinterpret_cast<const uint4*>(v)[i];
    uint32_t* aw = reinterpret_cast<uint32_t*>(&a);
    const uint32_t* bw = reinterpret_cast<const uint32_t*>(&b);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float a0 = __uint_as_float(aw[k] << 16), a1 = __uint_as_float(aw[k] & 0xffff0000u);
      const float b0 = __uint_as_float(bw[k] << 16), b1 = __uint_as_float(bw[k] & 0xffff0000u);
      __nv_bfloat162 r = __floats2bfloat162_rn(fmaf(dtau, b0, a0), fmaf(dtau, b1, a1));
      aw[k] = *reinterpret_cast<uint32_t*>(&r);
    }
    reinterpret_cast<uint4*>(z)[i] = a;
  }
  if (i == 0)
    for (int64_t k = n8 * 8; k < count; ++k)
      z[k] = __float2bfloat16_rn(fmaf(dtau, __bfloat162float(v[k]), __bfloat162float(z[k])));
}

cudaError_t launch_fm_euler(int32_t dtype, void* z, const void* v, float dtau, int64_t count,
                            cudaStream_t stream) {
  if (count <= 0) return cudaSuccess;
  if (dtype == 1) {
    int64_t n4 = count / 4;
    int64_t grid = std::max<int64_t>(1, (n4 + 255) / 256);
    fm_euler_f32_kernel<<<(unsigned)grid, 256, 0, stream>>>((float*)z, (const float*)v, dtau, n4, count);
  } else {
    int64_t n8 = count / 8;
    int64_t grid = std::max<int64_t>(1, (n8 + 255) / 256);
    fm_euler_bf16_kernel<<<(unsigned)grid, 256, 0, stream>>>((__nv_bfloat16*)z, (const __nv_bfloat16*)v,
                                                            dtau, n8, count);
  }
  return cudaGetLastError();
}

}  // namespace ws

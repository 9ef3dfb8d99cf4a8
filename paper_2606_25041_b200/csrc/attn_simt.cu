// attn_simt.cu - a3, generic CUDA-core kernel: block-causal attention of query tokens against a
// paged cache, fp32 arithmetic throughout (exact expf), any D <= 256 (D % 8 == 0), any page size,
// any q->kv head map, per-token visible end (multi-block queries).
//
// This is the kernel of the fp32 config (BASELINE configs[0]; tf32 tensor cores cannot meet 1e-5)
// and the functional path for bf16 shapes the tcgen05 kernel does not cover; it also serves as an
// on-GPU second opinion (WS_FLAG_FORCE_SIMT).  Definition followed: DESIGN.md §1 / PAPER.md:11, :29,
// :47 Eq. (1): row r of block b sees keys j < e_b.
//
// One warp per (query token, q head).  Lane = key for the scores (online softmax, max/sum reduced
// with warp shuffles), lane = output-dim slice for P.V, eight V rows in flight per lane (the loop is
// bound by load latency, not by arithmetic: walking the keys one dependent load at a time cost 19 us for
// the 48 keys of the fp32 config).
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>

#include "launch.h"

namespace ws {

template <typename T> struct Vec16;
template <> struct Vec16<float> {
  static constexpr int N = 4;
  static __device__ __forceinline__ void load(const float* p, float* o) {
    float4 v = *reinterpret_cast<const float4*>(p);
    o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
  }
};
template <> struct Vec16<__nv_bfloat16> {
  static constexpr int N = 8;
  static __device__ __forceinline__ void load(const __nv_bfloat16* p, float* o) {
    uint4 v = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      o[2 * i] = __uint_as_float(w[i] << 16);
      o[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
};

__device__ __forceinline__ float to_f32(float x) { return x; }
__device__ __forceinline__ float to_f32(__nv_bfloat16 x) { return __bfloat162float(x); }
__device__ __forceinline__ void store_out(float* p, float x) { *p = x; }
__device__ __forceinline__ void store_out(__nv_bfloat16* p, float x) { *p = __float2bfloat16_rn(x); }

constexpr int kSimtWarps = 4;
constexpr int kMaxD = 256;

template <typename T>
__global__ void __launch_bounds__(kSimtWarps * 32)
attn_simt_kernel(const T* __restrict__ q, T* __restrict__ out, float* __restrict__ lse,
                 const T* __restrict__ k_pool, const T* __restrict__ v_pool,
                 const int32_t* __restrict__ page_table, const int32_t* __restrict__ tok_meta,
                 const __grid_constant__ InlineAppendMeta inl,
                 const int32_t* __restrict__ q_to_kv, int32_t total_q_tokens, int32_t max_pages,
                 int32_t Hq, int32_t Hkv, int32_t D, int32_t P, float scale, int32_t text_causal) {
  // per-token (session slot, visible end): device blob, or - small calls - the kernel parameter itself
  // (constant-bank reads; no host->device copy in the chain, so the call is CUDA-graph capturable)
  const MetaView<kInlineAppendWords> meta{tok_meta, inl};
  // programmatic dependent launch (launch.h): q, the pool and the page table may come from the kernel
  // just before (ws_kv_append of the same step)
  pdl_wait();
  pdl_launch_dependents();
  __shared__ float q_s[kSimtWarps][kMaxD];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int64_t w = (int64_t)blockIdx.x * kSimtWarps + wib;
  if (w >= (int64_t)total_q_tokens * Hq) return;
  const int32_t tok = (int32_t)(w / Hq), h = (int32_t)(w % Hq);
  const int32_t g = q_to_kv ? q_to_kv[h] : h / (Hq / Hkv);
  const int32_t slot = meta[tok];
  const int32_t vis = meta[total_q_tokens + tok];
  // text-causal mixed mask (NEXT-4, reading A19): rows 2, 3 of the per-token metadata = the token's absolute
  // position if it is a text token (else -1) and the blob offset of its session's record {abs_pos0, nbits,
  // bits...} (bit k <=> the token at position abs_pos0 + k is text).  A text row skips later text keys.
  int32_t txt_pos = -1, txt_rec = 0, txt_abs0 = 0;
  if (text_causal) {
    txt_pos = meta[2 * total_q_tokens + tok];
    txt_rec = meta[3 * total_q_tokens + tok];
    txt_abs0 = meta[txt_rec];
  }
  const int32_t* page_row = page_table + (int64_t)slot * max_pages;

  const T* qrow = q + ((int64_t)tok * Hq + h) * D;
  for (int d = lane; d < D; d += 32) q_s[wib][d] = to_f32(qrow[d]);
  __syncwarp();

  constexpr int VN = Vec16<T>::N;
  float acc[kMaxD / 32];
#pragma unroll
  for (int i = 0; i < kMaxD / 32; ++i) acc[i] = 0.f;
  float m = -INFINITY, l = 0.f;

  for (int32_t base = 0; base < vis; base += 32) {
    const int32_t j = base + lane;
    bool valid = j < vis;
    if (valid && txt_pos >= 0 && j > txt_pos) {
      const int32_t b = j - txt_abs0;
      if ((meta[txt_rec + 2 + (b >> 5)] >> (b & 31)) & 1) valid = false;
    }
    float s = -INFINITY;
    int32_t rowidx = 0;
    if (valid) {
      rowidx = (page_row[j / P] * Hkv + g) * P + (j % P);
      const T* kp = k_pool + (int64_t)rowidx * D;
      float a = 0.f;
#pragma unroll 4
      for (int d = 0; d < D; d += VN) {
        float kv[VN];
        Vec16<T>::load(kp + d, kv);
#pragma unroll
        for (int e = 0; e < VN; ++e) a = fmaf(q_s[wib][d + e], kv[e], a);
      }
      s = a * scale;
    }
    float tmax = s;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
    const float m_new = fmaxf(m, tmax);
    // finite: the first chunk holds a visible key (a text row sees every key up to its own position),
    // a later chunk may be hidden entirely (text-causal), m is finite by then
    const float corr = expf(m - m_new);                 // m = -inf -> 0
    const float p = valid ? expf(s - m_new) : 0.f;
    float psum = p;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) psum += __shfl_xor_sync(0xffffffffu, psum, o);
    l = l * corr + psum;
#pragma unroll
    for (int i = 0; i < kMaxD / 32; ++i) acc[i] *= corr;
    const int nk = min(32, vis - base);
    constexpr int kBatch = 8;
    for (int kk0 = 0; kk0 < nk; kk0 += kBatch) {
      float pk[kBatch];
      const T* vp[kBatch];
#pragma unroll
      for (int u = 0; u < kBatch; ++u) {
        const int kk = (kk0 + u) & 31;
        pk[u] = kk0 + u < nk ? __shfl_sync(0xffffffffu, p, kk) : 0.f;
        vp[u] = v_pool + (int64_t)__shfl_sync(0xffffffffu, rowidx, kk) * D;
      }
#pragma unroll
      for (int i = 0; i < kMaxD / 32; ++i) {
        const int d = lane + 32 * i;
        if (d < D) {
          float vv[kBatch];
#pragma unroll
          for (int u = 0; u < kBatch; ++u) vv[u] = kk0 + u < nk ? to_f32(vp[u][d]) : 0.f;
#pragma unroll
          for (int u = 0; u < kBatch; ++u) acc[i] = fmaf(pk[u], vv[u], acc[i]);
        }
      }
    }
    m = m_new;
  }
  const float inv = 1.f / l;
  T* orow = out + ((int64_t)tok * Hq + h) * D;
#pragma unroll
  for (int i = 0; i < kMaxD / 32; ++i) {
    int d = lane + 32 * i;
    if (d < D) store_out(orow + d, acc[i] * inv);
  }
  if (lse && lane == 0) lse[(int64_t)tok * Hq + h] = m + logf(l);
}

cudaError_t launch_attn_simt(int32_t dtype, const void* q, void* out, float* lse,
                             const void* k_pool, const void* v_pool, const int32_t* page_table,
                             const int32_t* tok_meta, const InlineAppendMeta& inl, const int32_t* q_to_kv,
                             int32_t total_q_tokens, int32_t max_pages, int32_t Hq, int32_t Hkv, int32_t D,
                             int32_t P, float scale, int32_t text_causal, cudaStream_t stream) {
  int64_t warps = (int64_t)total_q_tokens * Hq;
  int32_t grid = (int32_t)((warps + kSimtWarps - 1) / kSimtWarps);
  if (grid == 0) return cudaSuccess;
  if (dtype == 1)
    return launch_pdl(attn_simt_kernel<float>, dim3(grid), dim3(kSimtWarps * 32), 0, stream,
                      (const float*)q, (float*)out, lse, (const float*)k_pool, (const float*)v_pool, page_table,
                      tok_meta, inl, q_to_kv, total_q_tokens, max_pages, Hq, Hkv, D, P, scale, text_causal);
  return launch_pdl(attn_simt_kernel<__nv_bfloat16>, dim3(grid), dim3(kSimtWarps * 32), 0, stream,
                    (const __nv_bfloat16*)q, (__nv_bfloat16*)out, lse, (const __nv_bfloat16*)k_pool,
                    (const __nv_bfloat16*)v_pool, page_table, tok_meta, inl, q_to_kv, total_q_tokens, max_pages,
                    Hq, Hkv, D, P, scale, text_causal);
}

}  // namespace ws

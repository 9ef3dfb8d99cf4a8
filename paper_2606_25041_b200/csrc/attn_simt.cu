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
// with warp shuffles), lane = output-dim slice for P.V.  The loop is bound by load latency, not by
// arithmetic (walking the keys one dependent load at a time cost 19 us for the 48 keys of the fp32 config):
// a chunk's K rows are read with every 16-byte load of a row in flight at once, and the V rows of its first
// 64 / kDV keys (kDV = 32-wide slices of D) are requested BEFORE the scores - their addresses need only the
// page ids - so they arrive under the K round and the softmax.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>

#include "kv_append.cuh"
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

template <typename T, int kDV>
__global__ void __launch_bounds__(kSimtWarps * 32)
attn_simt_kernel(const T* __restrict__ q, T* __restrict__ out, float* __restrict__ lse,
                 const T* __restrict__ k_pool, const T* __restrict__ v_pool,
                 const int32_t* __restrict__ page_table, const int32_t* __restrict__ tok_meta,
                 const __grid_constant__ InlineAppendMeta inl,
                 const int32_t* __restrict__ q_to_kv, int32_t total_q_tokens, int32_t max_pages,
                 int32_t Hq, int32_t Hkv, int32_t D, int32_t P, float scale, int32_t text_causal,
                 const T* __restrict__ k_new, const T* __restrict__ v_new, T* k_pool_w, T* v_pool_w,
                 int32_t* page_table_w, const __grid_constant__ InlineAppendMeta app, int32_t attn_blocks) {
  // per-token (session slot, visible end): device blob, or - small calls - the kernel parameter itself
  // (constant-bank reads; no host->device copy in the chain, so the call is CUDA-graph capturable)
  const MetaView<kInlineAppendWords> meta{tok_meta, inl};
  // programmatic dependent launch (launch.h): q, the pool and the page table may come from the kernel
  // just before (ws_kv_append of the same step)
  pdl_wait();
  pdl_launch_dependents();
  if ((int32_t)blockIdx.x >= attn_blocks) {
    // fused step (ws_stream_step on the generic path): the blocks behind the attention blocks commit the new
    // block to the pool (a2, kv_append.cuh) while the attention blocks read its keys straight from k_new / v_new
    const AppendGeom geom{reinterpret_cast<const int4*>(k_new), reinterpret_cast<const int4*>(v_new),
                          reinterpret_cast<int4*>(k_pool_w), reinterpret_cast<int4*>(v_pool_w), page_table_w,
                          max_pages, P, Hkv, D * (int32_t)sizeof(T) / 16};
    const MetaView<kInlineAppendWords> ameta{nullptr, app};
    const PeerPools none{};
    const int32_t b = (int32_t)blockIdx.x - attn_blocks, nb = (int32_t)gridDim.x - attn_blocks;
    append_work(ameta, geom, none, (int64_t)b * blockDim.x + threadIdx.x, (int64_t)nb * blockDim.x,
                b == 0 ? (int32_t)threadIdx.x : -1, (int32_t)blockDim.x);
    return;
  }
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
  // fused step: keys >= cache_len are rows new_row0 .. of k_new / v_new (two more metadata rows, after the
  // text rows if present); otherwise every key comes from the pool
  int32_t cache_len = vis, new_row0 = 0;
  if (k_new != nullptr) {
    const int32_t base = (text_causal ? 4 : 2) * total_q_tokens;
    cache_len = meta[base + tok];
    new_row0 = meta[base + total_q_tokens + tok];
  }
  const int32_t* page_row = page_table + (int64_t)slot * max_pages;

  const T* qrow = q + ((int64_t)tok * Hq + h) * D;
  for (int d = lane; d < D; d += 32) q_s[wib][d] = to_f32(qrow[d]);
  __syncwarp();

  constexpr int VN = Vec16<T>::N;
  constexpr int kBatch = 64 / kDV;                      // V rows in flight per lane
  float acc[kDV];
#pragma unroll
  for (int i = 0; i < kDV; ++i) acc[i] = 0.f;
  float m = -INFINITY, l = 0.f;
  // V values of keys kk0 .. kk0 + kBatch - 1 of the current chunk for this lane's output dims
  auto load_v = [&](int32_t rowidx, int kk0, int nk, float (&vv)[kBatch][kDV]) {
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int32_t ri = __shfl_sync(0xffffffffu, rowidx, (kk0 + u) & 31);
      const T* vp = ri >= 0 ? v_pool + (int64_t)ri * D : v_new + (int64_t)(-1 - ri) * D;
#pragma unroll
      for (int i = 0; i < kDV; ++i) {
        const int d = lane + 32 * i;
        vv[u][i] = (kk0 + u < nk && d < D) ? to_f32(vp[d]) : 0.f;
      }
    }
  };
  auto fma_v = [&](float p, int kk0, int nk, const float (&vv)[kBatch][kDV]) {
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const float pu = __shfl_sync(0xffffffffu, p, (kk0 + u) & 31);   // (keys >= nk: vv = 0)
#pragma unroll
      for (int i = 0; i < kDV; ++i) acc[i] = fmaf(pu, vv[u][i], acc[i]);
    }
  };

  for (int32_t base = 0; base < vis; base += 32) {
    const int32_t j = base + lane;
    bool valid = j < vis;
    if (valid && txt_pos >= 0 && j > txt_pos) {
      const int32_t b = j - txt_abs0;
      if ((meta[txt_rec + 2 + (b >> 5)] >> (b & 31)) & 1) valid = false;
    }
    float s = -INFINITY;
    int32_t rowidx = 0;
    // rowidx >= 0: row of the pool; < 0: row -(rowidx + 1) of k_new / v_new (hidden keys: pool row 0, p = 0)
    if (valid)
      rowidx = j < cache_len ? (page_row[j / P] * Hkv + g) * P + (j % P) : -1 - ((new_row0 + j - cache_len) * Hkv + g);
    const int nk = min(32, vis - base);
    float vv[kBatch][kDV];
    load_v(rowidx, 0, nk, vv);
    if (valid) {
      const T* kp = rowidx >= 0 ? k_pool + (int64_t)rowidx * D : k_new + (int64_t)(-1 - rowidx) * D;
      float a = 0.f;
#pragma unroll 16
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
    for (int i = 0; i < kDV; ++i) acc[i] *= corr;
    fma_v(p, 0, nk, vv);
#pragma unroll 1
    for (int kk0 = kBatch; kk0 < nk; kk0 += kBatch) {
      load_v(rowidx, kk0, nk, vv);
      fma_v(p, kk0, nk, vv);
    }
    m = m_new;
  }
  const float inv = 1.f / l;
  T* orow = out + ((int64_t)tok * Hq + h) * D;
#pragma unroll
  for (int i = 0; i < kDV; ++i) {
    int d = lane + 32 * i;
    if (d < D) store_out(orow + d, acc[i] * inv);
  }
  if (lse && lane == 0) lse[(int64_t)tok * Hq + h] = m + logf(l);
}

cudaError_t launch_attn_simt(int32_t dtype, const void* q, void* out, float* lse,
                             const void* k_pool, const void* v_pool, const int32_t* page_table,
                             const int32_t* tok_meta, const InlineAppendMeta& inl, const int32_t* q_to_kv,
                             int32_t total_q_tokens, int32_t max_pages, int32_t Hq, int32_t Hkv, int32_t D,
                             int32_t P, float scale, int32_t text_causal, const SimtFused* fused, cudaStream_t stream) {
  int64_t warps = (int64_t)total_q_tokens * Hq;
  int32_t grid = (int32_t)((warps + kSimtWarps - 1) / kSimtWarps);
  if (grid == 0) return cudaSuccess;
  const int32_t attn_blocks = grid;
  const void *k_new = nullptr, *v_new = nullptr;
  void *kw = nullptr, *vw = nullptr;
  int32_t* ptw = nullptr;
  InlineAppendMeta app_none;
  const InlineAppendMeta* app = &app_none;
  if (fused) {
    k_new = fused->k_new; v_new = fused->v_new; kw = fused->k_pool_w; vw = fused->v_pool_w; ptw = fused->page_table_w;
    app = fused->app;
    const int64_t chunks = (int64_t)std::max(fused->append_tokens, P - 1) * Hkv * (D * (dtype == 1 ? 4 : 2) / 16);
    grid += (int32_t)std::min<int64_t>(std::max<int64_t>((chunks + kSimtWarps * 32 - 1) / (kSimtWarps * 32), 1), 148 * 4);
  } else {
    app_none.w[0] = 0;
  }
  auto go = [&](auto kern_f32, auto kern_bf16) {
    if (dtype == 1)
      return launch_pdl(kern_f32, dim3(grid), dim3(kSimtWarps * 32), 0, stream,
                        (const float*)q, (float*)out, lse, (const float*)k_pool, (const float*)v_pool, page_table,
                        tok_meta, inl, q_to_kv, total_q_tokens, max_pages, Hq, Hkv, D, P, scale, text_causal,
                        (const float*)k_new, (const float*)v_new, (float*)kw, (float*)vw, ptw, *app, attn_blocks);
    return launch_pdl(kern_bf16, dim3(grid), dim3(kSimtWarps * 32), 0, stream,
                      (const __nv_bfloat16*)q, (__nv_bfloat16*)out, lse, (const __nv_bfloat16*)k_pool,
                      (const __nv_bfloat16*)v_pool, page_table, tok_meta, inl, q_to_kv, total_q_tokens, max_pages,
                      Hq, Hkv, D, P, scale, text_causal, (const __nv_bfloat16*)k_new, (const __nv_bfloat16*)v_new,
                      (__nv_bfloat16*)kw, (__nv_bfloat16*)vw, ptw, *app, attn_blocks);
  };
  // kDV = 32-wide slices of D held per lane
  if (D <= 64) return go(attn_simt_kernel<float, 2>, attn_simt_kernel<__nv_bfloat16, 2>);
  if (D <= 128) return go(attn_simt_kernel<float, 4>, attn_simt_kernel<__nv_bfloat16, 4>);
  return go(attn_simt_kernel<float, 8>, attn_simt_kernel<__nv_bfloat16, 8>);
}

}  // namespace ws

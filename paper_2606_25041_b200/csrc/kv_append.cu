// kv_append.cu - a2: bit-exact paged KV append (commit) and its inverse (gather).
// PAPER.md:83 "appends the received KV slice into its own full-history cache"; :29 "committed back
// into the interaction history".  Pure data movement in 16-byte words: NaN payloads, -0 and
// denormals are preserved.  HBM-bound; algorithmic bytes = 2 (read+write) x 2 (K,V) x n x Hkv x D x eb.
#include <cuda_runtime.h>
#include <stdint.h>

#include "kv_append.cuh"
#include "launch.h"
#include "ws_internal.h"

namespace ws {

// ws_kv_append's own launch: one thread per 16-byte chunk of K (and the matching chunk of V), device code
// in kv_append.cuh.  chunks_per_token = Hkv * D * eb / 16; chunks_per_head = D * eb / 16.
//
// Programmatic dependent launch (launch.h): the kernel may start while its stream predecessor is still
// running, so it waits for that grid (griddepcontrol.wait: complete and flushed) BEFORE its first access -
// k_new / v_new may have been produced by the predecessor, and the pool rows / page-table entries it
// writes may still be being read by it (an attention kernel over a session that was rolled back and is
// re-appended at the same positions).  Only then does it let its own successor start early; the successor's
// own wait covers this grid.
__global__ void __launch_bounds__(256)
kv_append_kernel(const int4* __restrict__ k_new, const int4* __restrict__ v_new,
                 int4* __restrict__ k_pool, int4* __restrict__ v_pool,
                 int32_t* __restrict__ page_table, const int32_t* __restrict__ meta_g,
                 const __grid_constant__ InlineAppendMeta inl, const __grid_constant__ PeerPools peers,
                 int32_t max_pages, int32_t P, int32_t Hkv, int32_t chunks_per_head) {
  pdl_wait();
  pdl_launch_dependents();
  const MetaView<kInlineAppendWords> meta{meta_g, inl};    // (constant-bank reads when the blob is inline)
  const AppendGeom g{k_new, v_new, k_pool, v_pool, page_table, max_pages, P, Hkv, chunks_per_head};
  append_work(meta, g, peers, (int64_t)blockIdx.x * blockDim.x + threadIdx.x, (int64_t)gridDim.x * blockDim.x,
              blockIdx.x == 0 ? (int32_t)threadIdx.x : -1, (int32_t)blockDim.x);
}

__global__ void __launch_bounds__(256)
kv_gather_kernel(const int4* __restrict__ k_pool, const int4* __restrict__ v_pool,
                 int4* __restrict__ k_out, int4* __restrict__ v_out,
                 const int32_t* __restrict__ page_row, int64_t start, int64_t count, int32_t P,
                 int32_t Hkv, int32_t chunks_per_head) {
  const int32_t chunks_per_token = Hkv * chunks_per_head;
  const int64_t total = count * chunks_per_token;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    int64_t tok = idx / chunks_per_token;
    int32_t c = (int32_t)(idx - tok * chunks_per_token);
    int64_t pos = start + tok;
    int32_t page = page_row[pos / P];
    int32_t head = c / chunks_per_head;
    int32_t off = c - head * chunks_per_head;
    int64_t src = (((int64_t)page * Hkv + head) * P + (pos % P)) * chunks_per_head + off;
    if (k_out) k_out[idx] = k_pool[src];
    if (v_out) v_out[idx] = v_pool[src];
  }
}

// NEXT-3 replica side: publish adopted page ids into the device page table (ws_replica_apply).
// One launch covers one session: row `slot`, logical pages [first, first + n) <- ids[0..n).
__global__ void __launch_bounds__(256)
page_table_publish_kernel(int32_t* __restrict__ page_table, const __grid_constant__ InlineAppendMeta inl,
                          int32_t slot, int32_t first, int32_t n, int32_t max_pages) {
  for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    page_table[(int64_t)slot * max_pages + first + i] = inl.w[i];
}

// NEXT-3 owner side: the data half of the initial broadcast: every page of a session,
// all KV heads (one page = Hkv * P * D * eb contiguous bytes), local pool -> linked pools.
__global__ void __launch_bounds__(256)
kv_push_pages_kernel(const int4* __restrict__ k_pool, const int4* __restrict__ v_pool,
                     const __grid_constant__ PeerPools peers, const int32_t* __restrict__ page_row, int32_t npages,
                     int32_t chunks_per_page) {
  const int64_t total = (int64_t)npages * chunks_per_page;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int32_t lp = (int32_t)(idx / chunks_per_page);
    const int64_t off = (int64_t)page_row[lp] * chunks_per_page + (idx - (int64_t)lp * chunks_per_page);
    const int4 kx = k_pool[off], vx = v_pool[off];
    for (int32_t r = 0; r < peers.n; ++r) { ((int4*)peers.k[r])[off] = kx; ((int4*)peers.v[r])[off] = vx; }
  }
  __threadfence_system();
}

cudaError_t launch_page_table_publish(int32_t* page_table, const int32_t* ids, int32_t slot,
                                      int32_t first, int32_t n, int32_t max_pages,
                                      cudaStream_t stream) {
  // chunks of at most kInlineAppendWords ids travel in the kernel parameters (capturable, no staging)
  for (int32_t done = 0; done < n; done += kInlineAppendWords) {
    const int32_t m = std::min(n - done, (int32_t)kInlineAppendWords);
    InlineAppendMeta inl{};
    for (int32_t i = 0; i < m; ++i) inl.w[i] = ids[done + i];
    page_table_publish_kernel<<<(m + 255) / 256, 256, 0, stream>>>(page_table, inl, slot, first + done,
                                                                    m, max_pages);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_kv_push_pages(const void* k_pool, const void* v_pool, const PeerPools& peers,
                                 const int32_t* page_row, int32_t npages, int64_t page_bytes,
                                 int32_t num_sms, cudaStream_t stream) {
  const int32_t cpp = (int32_t)(page_bytes / 16);
  const int64_t total = (int64_t)npages * cpp;
  const int32_t grid = (int32_t)std::min<int64_t>(std::max<int64_t>((total + 255) / 256, 1), (int64_t)num_sms * 16);
  kv_push_pages_kernel<<<grid, 256, 0, stream>>>((const int4*)k_pool, (const int4*)v_pool, peers,
                                                 page_row, npages, cpp);
  return cudaGetLastError();
}

cudaError_t launch_kv_append(const void* k_new, const void* v_new, void* k_pool, void* v_pool,
                             int32_t* page_table, const int32_t* meta, const InlineAppendMeta& inl,
                             const PeerPools& peers, int32_t total_tokens, int32_t max_pages, int32_t P, int32_t Hkv,
                             int32_t D, int32_t eb, int32_t num_sms, cudaStream_t stream) {
  int32_t cph = D * eb / 16;
  int64_t total = (int64_t)total_tokens * Hkv * cph;
  // (a short append still zeroes up to P - 1 token rows of the last page: size the grid for that too -
  // a one-token decode append ran 11.8 us as a single block)
  int64_t work = std::max<int64_t>(total, (int64_t)(P - 1) * Hkv * cph);
  int64_t blocks = (work + 255) / 256;
  int32_t grid = (int32_t)std::min<int64_t>(std::max<int64_t>(blocks, 1), (int64_t)num_sms * 8);
  return launch_pdl(kv_append_kernel, dim3(grid), dim3(256), 0, stream, (const int4*)k_new,
                    (const int4*)v_new, (int4*)k_pool, (int4*)v_pool, page_table, meta, inl, peers,
                    max_pages, P, Hkv, cph);
}

cudaError_t launch_kv_gather(const void* k_pool, const void* v_pool, void* k_out, void* v_out,
                             const int32_t* page_row, int64_t start, int64_t count, int32_t P,
                             int32_t Hkv, int32_t D, int32_t eb, int32_t num_sms,
                             cudaStream_t stream) {
  int32_t cph = D * eb / 16;
  int64_t total = count * Hkv * cph;
  int64_t blocks = (total + 255) / 256;
  int32_t grid = (int32_t)std::min<int64_t>(std::max<int64_t>(blocks, 1), (int64_t)num_sms * 8);
  kv_gather_kernel<<<grid, 256, 0, stream>>>((const int4*)k_pool, (const int4*)v_pool,
                                             (int4*)k_out, (int4*)v_out, page_row, start, count, P,
                                             Hkv, cph);
  return cudaGetLastError();
}

}  // namespace ws

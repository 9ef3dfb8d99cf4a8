// kv_append.cu - a2: bit-exact paged KV append (commit) and its inverse (gather).
// PAPER.md:83 "appends the received KV slice into its own full-history cache"; :29 "committed back
// into the interaction history".  Pure data movement in 16-byte words: NaN payloads, -0 and
// denormals are preserved.  HBM-bound; algorithmic bytes = 2 (read+write) x 2 (K,V) x n x Hkv x D x eb.
#include <cuda_runtime.h>
#include <stdint.h>

#include "launch.h"
#include "ws_internal.h"

namespace ws {

// One thread moves one 16-byte chunk of K and the matching chunk of V.
// chunks_per_token = Hkv * D * eb / 16; chunks_per_head = D * eb / 16.
__global__ void __launch_bounds__(256)
kv_append_kernel(const int4* __restrict__ k_new, const int4* __restrict__ v_new,
                 int4* __restrict__ k_pool, int4* __restrict__ v_pool,
                 int32_t* __restrict__ page_table, const int32_t* __restrict__ meta_g,
                 const __grid_constant__ InlineAppendMeta inl, const PeerPools peers,
                 int32_t max_pages, int32_t P, int32_t Hkv, int32_t chunks_per_head) {
  // Nothing this kernel touches is produced by its stream predecessor (the previous step's combine
  // writes only `out`), so the successor (this step's attention) may start its prologue right away.
  pdl_launch_dependents();
  const MetaView<kInlineAppendWords> meta{meta_g, inl};    // (constant-bank reads when the blob is inline)
  const AppendMeta hdr = meta.load<AppendMeta>(0);
  constexpr int32_t kSessWords = (int32_t)(sizeof(AppendSession) / 4);
  auto sess = [&](int32_t s) { return meta.load<AppendSession>(hdr.off_sessions + s * kSessWords); };
  auto sess_tok_end = [&](int32_t s) { return meta[hdr.off_sessions + s * kSessWords + 3]; };
  auto pages = [&](int32_t i) { return meta[hdr.off_pages + i]; };
  const int32_t chunks_per_token = Hkv * chunks_per_head;
  const int64_t total = (int64_t)hdr.total_tokens * chunks_per_token;

  // Block 0 also publishes the page ids into the persistent device page table (idempotent).
  if (blockIdx.x == 0) {
    for (int32_t s = 0; s < hdr.num_sessions; ++s) {
      const AppendSession a = sess(s);
      int32_t first = a.len_old / P;
      int32_t last = (a.len_old + (a.tok_end - a.tok_begin) + P - 1) / P;
      for (int32_t i = first + threadIdx.x; i < last; i += blockDim.x)
        page_table[(int64_t)a.slot * max_pages + i] = pages(a.page_off + (i - first));
    }
  }
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    int32_t tok = (int32_t)(idx / chunks_per_token);
    int32_t c = (int32_t)(idx - (int64_t)tok * chunks_per_token);
    // session of this token: binary search over tok_end
    int32_t lo = 0, hi = hdr.num_sessions - 1;
    while (lo < hi) {
      int32_t mid = (lo + hi) >> 1;
      if (tok >= sess_tok_end(mid)) lo = mid + 1; else hi = mid;
    }
    const AppendSession a = sess(lo);
    int32_t pos = a.len_old + (tok - a.tok_begin);
    int32_t page = pages(a.page_off + (pos / P - a.len_old / P));
    int32_t head = c / chunks_per_head;
    int32_t off = c - head * chunks_per_head;
    int64_t dst = (((int64_t)page * Hkv + head) * P + (pos % P)) * chunks_per_head + off;
    const int4 kx = k_new[idx], vx = v_new[idx];
    k_pool[dst] = kx;
    v_pool[dst] = vx;
    // NEXT-3: the same slice goes to every linked replica pool at the same page id -
    // plain stores through the peer mapping (NVLink), no second read of the slice.
    for (int32_t r = 0; r < peers.n; ++r) { ((int4*)peers.k[r])[dst] = kx; ((int4*)peers.v[r])[dst] = vx; }
  }
  // Zero the unused tail of each session's last page: slots beyond the committed length are then
  // always finite (zero), so the attention kernel may load whole pages and rely on P = 0 for the
  // masked keys (0 x stale NaN bits would poison O).  At most P - 1 token rows per session.
  {
    const int4 zero = make_int4(0, 0, 0, 0);
    for (int32_t s = 0; s < hdr.num_sessions; ++s) {
      const AppendSession a = sess(s);
      const int32_t len_new = a.len_old + (a.tok_end - a.tok_begin);
      const int32_t tail = (P - len_new % P) % P;
      if (tail == 0) continue;
      const int32_t page = pages(a.page_off + ((len_new - 1) / P - a.len_old / P));
      const int64_t total_tail = (int64_t)tail * chunks_per_token;
      for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total_tail;
           idx += (int64_t)gridDim.x * blockDim.x) {
        int32_t t = (int32_t)(idx / chunks_per_token);
        int32_t c = (int32_t)(idx - (int64_t)t * chunks_per_token);
        int32_t head = c / chunks_per_head, off = c - head * chunks_per_head;
        int64_t dst = (((int64_t)page * Hkv + head) * P + (len_new % P + t)) * chunks_per_head + off;
        k_pool[dst] = zero;
        v_pool[dst] = zero;
        for (int32_t r = 0; r < peers.n; ++r) { ((int4*)peers.k[r])[dst] = zero; ((int4*)peers.v[r])[dst] = zero; }
      }
    }
  }
  // Peer stores must be visible to the replica's GPU before the host learns this kernel completed.
  if (peers.n > 0) __threadfence_system();
  // Completing only after the predecessor has completed keeps the dependency chain transitive: the
  // attention kernel's griddepcontrol.wait on this grid then also covers everything before it.
  pdl_wait();
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
                     const PeerPools peers, const int32_t* __restrict__ page_row, int32_t npages,
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

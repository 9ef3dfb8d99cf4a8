// kv_append.cuh - a2: the device code of the bit-exact paged KV append (commit), shared by
// kv_append_kernel (ws_kv_append: its own launch) and by the attention kernel's append warps
// (ws_stream_step: the block is committed by the launch that attends it).
// PAPER.md:83 "appends the received KV slice into its own full-history cache"; :29 "committed back
// into the interaction history".  Pure data movement in 16-byte words: NaN payloads, -0 and
// denormals are preserved.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ws_internal.h"

namespace ws {

// Geometry of one append, common to every thread.
struct AppendGeom {
  const int4* k_new; const int4* v_new;      // [total_tokens][Hkv][chunks_per_head] 16-byte chunks
  int4* k_pool; int4* v_pool;                // [pages][Hkv][P][chunks_per_head]
  int32_t* page_table;
  int32_t max_pages, P, Hkv, chunks_per_head;
};

// Thread `tid` of `nthreads` cooperating threads moves chunks tid, tid + nthreads, ... of the call
// (one chunk = 16 bytes of K and the matching 16 bytes of V), zeroes its share of the unused tail of
// each session's last page, and - threads with pub_tid >= 0 (pub_n of them) - publishes the new page
// ids into the persistent device page table (idempotent).
template <typename Meta>
__device__ __forceinline__ void append_work(const Meta& meta, const AppendGeom& g, const PeerPools& peers,
                                            int64_t tid, int64_t nthreads, int32_t pub_tid, int32_t pub_n) {
  const AppendMeta hdr = meta.template load<AppendMeta>(0);
  constexpr int32_t kSessWords = (int32_t)(sizeof(AppendSession) / 4);
  auto sess = [&](int32_t s) { return meta.template load<AppendSession>(hdr.off_sessions + s * kSessWords); };
  auto sess_tok_end = [&](int32_t s) { return meta[hdr.off_sessions + s * kSessWords + 3]; };
  auto pages = [&](int32_t i) { return meta[hdr.off_pages + i]; };
  const int32_t P = g.P, Hkv = g.Hkv, cph = g.chunks_per_head;
  const int32_t chunks_per_token = Hkv * cph;
  const int64_t total = (int64_t)hdr.total_tokens * chunks_per_token;

  if (pub_tid >= 0) {
    for (int32_t s = 0; s < hdr.num_sessions; ++s) {
      const AppendSession a = sess(s);
      const int32_t first = a.len_old / P;
      const int32_t last = (a.len_old + (a.tok_end - a.tok_begin) + P - 1) / P;
      for (int32_t i = first + pub_tid; i < last; i += pub_n)
        g.page_table[(int64_t)a.slot * g.max_pages + i] = pages(a.page_off + (i - first));
    }
  }
  // destination chunk index of source chunk idx
  auto dst_of = [&](int64_t idx) -> int64_t {
    const int32_t tok = (int32_t)(idx / chunks_per_token);
    const int32_t c = (int32_t)(idx - (int64_t)tok * chunks_per_token);
    int32_t lo = 0, hi = hdr.num_sessions - 1;           // session of this token: search over tok_end
    while (lo < hi) {
      const int32_t mid = (lo + hi) >> 1;
      if (tok >= sess_tok_end(mid)) lo = mid + 1; else hi = mid;
    }
    const AppendSession a = sess(lo);
    const int32_t pos = a.len_old + (tok - a.tok_begin);
    const int32_t page = pages(a.page_off + (pos / P - a.len_old / P));
    const int32_t head = c / cph, off = c - head * cph;
    return (((int64_t)page * Hkv + head) * P + (pos % P)) * cph + off;
  };
  auto store = [&](int64_t dst, const int4& kx, const int4& vx) {
    g.k_pool[dst] = kx;
    g.v_pool[dst] = vx;
    // NEXT-3: the same slice goes to every linked replica pool at the same page id -
    // plain stores through the peer mapping (NVLink), no second read of the slice.
    for (int32_t r = 0; r < peers.n; ++r) { ((int4*)peers.k[r])[dst] = kx; ((int4*)peers.v[r])[dst] = vx; }
  };
  // four chunks of K and V in flight per thread (the append warps of the attention kernel are few:
  // memory-level parallelism has to come from each of them)
  int64_t idx = tid;
  for (; idx + 3 * nthreads < total; idx += 4 * nthreads) {
    int4 kx[4], vx[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { kx[u] = g.k_new[idx + u * nthreads]; vx[u] = g.v_new[idx + u * nthreads]; }
#pragma unroll
    for (int u = 0; u < 4; ++u) store(dst_of(idx + u * nthreads), kx[u], vx[u]);
  }
  for (; idx < total; idx += nthreads) store(dst_of(idx), g.k_new[idx], g.v_new[idx]);

  // Zero the unused tail of each session's last page: slots beyond the committed length are then
  // always finite (zero), so the attention kernel may load whole pages and rely on P = 0 for the
  // masked keys (0 x stale NaN bits would poison O).  At most P - 1 token rows per session.
  const int4 zero = make_int4(0, 0, 0, 0);
  for (int32_t s = 0; s < hdr.num_sessions; ++s) {
    const AppendSession a = sess(s);
    const int32_t len_new = a.len_old + (a.tok_end - a.tok_begin);
    const int32_t tail = (P - len_new % P) % P;
    if (tail == 0) continue;
    const int32_t page = pages(a.page_off + ((len_new - 1) / P - a.len_old / P));
    const int64_t total_tail = (int64_t)tail * chunks_per_token;
    for (int64_t i = tid; i < total_tail; i += nthreads) {
      const int32_t t = (int32_t)(i / chunks_per_token);
      const int32_t c = (int32_t)(i - (int64_t)t * chunks_per_token);
      const int32_t head = c / cph, off = c - head * cph;
      store((((int64_t)page * Hkv + head) * P + (len_new % P + t)) * cph + off, zero, zero);
    }
  }
  // Peer stores must be visible to the replica's GPU before the host learns this kernel completed.
  if (peers.n > 0) __threadfence_system();
}

}  // namespace ws

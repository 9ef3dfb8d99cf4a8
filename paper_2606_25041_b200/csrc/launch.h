// launch.h - host-callable launchers of the kernels (internal).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <utility>

#include "ws_internal.h"

namespace ws {

// PDL helpers: every kernel of the (append ->) attention -> combine chain is launched with programmatic
// stream serialization.  Protocol: a kernel executes griddepcontrol.wait before its
// first access to anything its stream predecessor may have written or may still be reading - caller-
// produced inputs included, the predecessor may be the caller's kernel - and at the latest before it
// exits, so completion stays ordered along the chain; griddepcontrol.launch_dependents (one thread per
// CTA suffices: the first arrival counts for the whole CTA) only lets the successor's CTAs be scheduled
// early, it orders nothing, which is safe because every successor obeys the same rule.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem,
                       cudaStream_t stream, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// meta == nullptr: the metadata blob is `inl` (passed in the kernel parameters)
cudaError_t launch_kv_append(const void* k_new, const void* v_new, void* k_pool, void* v_pool,
                             int32_t* page_table, const int32_t* meta, const InlineAppendMeta& inl,
                             const PeerPools& peers, int32_t total_tokens,
                             int32_t max_pages, int32_t P, int32_t Hkv, int32_t D, int32_t eb,
                             int32_t num_sms, cudaStream_t stream);
// NEXT-3 (replica link): see kv_append.cu
cudaError_t launch_page_table_publish(int32_t* page_table, const int32_t* ids, int32_t slot,
                                      int32_t first, int32_t n, int32_t max_pages, cudaStream_t stream);
cudaError_t launch_kv_push_pages(const void* k_pool, const void* v_pool, const PeerPools& peers,
                                 const int32_t* page_row, int32_t npages, int64_t page_bytes,
                                 int32_t num_sms, cudaStream_t stream);
cudaError_t launch_kv_gather(const void* k_pool, const void* v_pool, void* k_out, void* v_out,
                             const int32_t* page_row, int64_t start, int64_t count, int32_t P,
                             int32_t Hkv, int32_t D, int32_t eb, int32_t num_sms,
                             cudaStream_t stream);

// NEXT-2: flow-matching Euler update z <- z + dtau * v (dtype 0 = bf16, 1 = fp32), 16-byte aligned.
cudaError_t launch_fm_euler(int32_t dtype, void* z, const void* v, float dtau, int64_t count,
                            cudaStream_t stream);

// Generic SIMT attention (fp32 config; bf16 debug / unsupported-shape path).
// tok_meta: [2][total_q_tokens] int32 = session slot, visible end per query token; nullptr: the same
// words are in `inl` (kernel parameter, 2 * total_q_tokens <= kInlineAppendWords).  text_causal: two more
// rows (text position or -1, record offset) followed by the sessions' text-bit records (attn_simt.cu).
// fused != nullptr: ws_stream_step on the generic path - the launch also commits the block (extra thread blocks run
// the append) and reads its keys from k_new / v_new; tok_meta then carries two more rows per token (committed
// length before the append, first row of the session's block in k_new).
struct SimtFused {
  const void* k_new; const void* v_new;
  void* k_pool_w; void* v_pool_w; int32_t* page_table_w;
  const InlineAppendMeta* app;
  int32_t append_tokens;
};
cudaError_t launch_attn_simt(int32_t dtype, const void* q, void* out, float* lse,
                             const void* k_pool, const void* v_pool, const int32_t* page_table,
                             const int32_t* tok_meta, const InlineAppendMeta& inl, const int32_t* q_to_kv,
                             int32_t total_q_tokens, int32_t max_pages, int32_t Hq, int32_t Hkv, int32_t D,
                             int32_t P, float scale, int32_t text_causal, const SimtFused* fused, cudaStream_t stream);

// sm_100a tcgen05 kernel (bf16, D = 128, P = 64).
struct Sm100Launch {
  AttnParams p;                      // p.meta == nullptr: use `inl`
  CUtensorMap tmap_q, tmap_k, tmap_v;
  CUtensorMap tmap_kn, tmap_vn;      // fused step: k_new / v_new as [D, Hkv, tokens] (else copies of tmap_k / tmap_v)
  InlineAttnMetaLarge inl;
  InlineAppendMeta app;              // fused step: the append descriptor (p.append_tokens > 0)
  PeerPools peers;
  int32_t inl_words;                 // words of `inl` in use (selects the small / large parameter tier)
  int32_t num_ctas;
  bool alt;                          // decode plan (plan.h): runs on attn_dec_sm100_kernel
};
cudaError_t sm100_attn_configure();    // one-time cudaFuncSetAttribute
cudaError_t launch_attn_sm100(const Sm100Launch& l, cudaStream_t stream);
// decode kernel (attn_dec_sm100.cu): decode plans (at most 128 packed query rows per (session, KV head)), both
// softmax warpgroups on every KV tile; no in-kernel merge phase
cudaError_t dec_sm100_configure();
cudaError_t launch_attn_dec_sm100(const Sm100Launch& l, cudaStream_t stream);
cudaError_t combine_configure();        // one-time cudaFuncSetAttribute
cudaError_t launch_combine(const AttnParams& p, const InlineAttnMetaLarge& inl, int32_t inl_words,
                           int32_t num_combine, int32_t team_size, int32_t max_parts, int32_t max_rows_per_pair,
                           cudaStream_t stream);

}  // namespace ws

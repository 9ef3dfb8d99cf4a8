/* ws.h - C ABI of libwanstream: block-causal streaming attention over a paged per-session KV cache.
 *
 * The hot path of Wan-Streamer's streaming inference (arxiv 2606.25041): once per 160 ms streaming
 * unit a newly arrived block of interleaved visual/audio/text tokens (PAPER.md:11 Abstract, :29 §1,
 * :45 §2.1) is (1) committed to the session's full-history KV cache ("appends the received KV slice
 * into its own full-history cache"; also :29, :31, :51, :59) and (2) attends
 * block-causally to it: bidirectionally within its own block, causally to all earlier blocks
 * (PAPER.md:11, :23 Fig. 1, :29, :38, :155; dependence structure of Eq. (1)).
 * The paper gives no formula, sizes or dtype; the readings taken are listed in DESIGN.md §2.
 *
 * Conventions
 *  - All functions return ws_status_t (WS_OK = 0). No exceptions, no abort(), nothing on stdout.
 *    ws_last_error() returns a thread-local human-readable message for the last failure.
 *  - "HOST" pointers are read before the call returns (the caller may reuse them immediately).
 *    "DEVICE" pointers are CUDA device memory on `device`; they are CALLER-owned (the Python
 *    harness allocates them as torch tensors) and only borrowed by the library.
 *  - Calls enqueue their work on the given CUDA stream (a cudaStream_t passed as void*) and return
 *    without synchronising.  All calls on one cache must use one stream (or be externally ordered).
 *  - Arguments are validated BEFORE any state changes: on any error no session length, page table,
 *    block boundary or free-list entry has changed (strong guarantee).
 *  - One cache handle = one attention layer.  There is NO CPU fallback: without a CUDA device every
 *    compute entry point fails with WS_ERR_CUDA (except under WS_FLAG_DRY_RUN, see below).
 *
 * Layouts (element = bf16 or fp32 according to `dtype`)
 *  - K/V pools:   [num_pages][num_kv_heads][page_tokens][head_dim]   (one (page, head) slab is a
 *                 dense page_tokens x head_dim matrix - TMA-addressable as a rank-4 tensor)
 *  - k_new/v_new: [sum n][num_kv_heads][head_dim], token-major, contiguous
 *  - q / out:     [sum n_q][num_q_heads][head_dim], token-major, contiguous
 *  - lse:         [sum n_q][num_q_heads] fp32, natural log
 *  - GQA: query head h reads KV head q_to_kv_head[h] (default h / (num_q_heads/num_kv_heads)).
 */
#ifndef WS_H_
#define WS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  WS_OK = 0,
  WS_ERR_INVALID_ARG = 1,        /* null pointer, bad size, duplicate session in one call, ...     */
  WS_ERR_BAD_SESSION = 2,        /* session id not open                                            */
  WS_ERR_OUT_OF_PAGES = 3,       /* free list (or per-session page/block capacity) exhausted       */
  WS_ERR_UNSUPPORTED = 4,        /* shape/dtype combination no kernel covers                       */
  WS_ERR_WORKSPACE_TOO_SMALL = 5,
  WS_ERR_CUDA = 6                /* a CUDA call failed (message in ws_last_error())                */
} ws_status_t;

typedef enum { WS_BF16 = 0, WS_F32 = 1 } ws_dtype_t;

enum {
  /* Host metadata only: no CUDA call is ever made (pools/workspace may be NULL).  For testing the
   * page allocator, scheduler and error paths on a machine without a GPU.  Compute is skipped.     */
  WS_FLAG_DRY_RUN = 1u,
  /* Debug: route bf16 attention through the generic SIMT kernel instead of the tcgen05 kernel.     */
  WS_FLAG_FORCE_SIMT = 2u,
  /* (4u is retired: it selected a cta_group::2 variant of the tcgen05 kernel that was measured slower
   * and has been removed.)                                                      */
  /* Merge the split-KV partials (a4) inside the attention kernel instead of in the combine kernel that
   * follows it: every CTA publishes its partials (per-group arrival counters in the workspace), waits
   * until all splits of its (session, KV head) group are there and merges its share of the rows; the
   * kernel is then launched cooperatively so that all CTAs are co-resident while they wait on each
   * other.  Correct and one launch fewer, but measured no faster than the separate kernel on B200
   * (DESIGN.md section 8), so it is opt-in.  Decode plans ignore it (the decode kernel has no merge phase). */
  WS_FLAG_FUSED_COMBINE = 8u,
  /* ws_stream_step normally commits and attends a block in ONE launch (the attention kernel reads the
   * new keys from k_new / v_new and two of its warps copy them into the pool).  With this flag it
   * launches the append kernel and the attention kernel separately, as ws_kv_append followed by
   * ws_block_causal_attn_fwd would (A/B measurements, tests: both must give identical results).     */
  WS_FLAG_SEPARATE_APPEND = 16u
};

typedef struct ws_cache ws_cache_t;   /* opaque; owns host metadata only */

typedef struct {
  int32_t dtype;                  /* ws_dtype_t                                                    */
  int32_t num_q_heads;            /* Hq                                                            */
  int32_t num_kv_heads;           /* Hkv, Hq % Hkv == 0                                            */
  int32_t head_dim;               /* D: bf16 tensor-core path D = 128; generic path D <= 256, D%8==0.
                                   * A bf16 cache whose shape the tcgen05 kernel does not cover (D != 128, page != 64,
                                   * Hq/Hkv not in {1,2,4,8,16}, explicit q_to_kv_head) is served by the generic
                                   * CUDA-core kernel - same results, no tensor cores; ws_last_plan_info reports
                                   * which kernel ran.  WS_ERR_UNSUPPORTED is returned only for shapes neither covers. */
  const int32_t* q_to_kv_head;    /* HOST [Hq] or NULL = grouped default                           */
  int32_t page_tokens;            /* P: tokens per page (64 for the bf16 tensor-core path)         */
  int32_t num_pages;              /* pages in each pool                                            */
  int32_t max_sessions;           /* session slots                                                 */
  int32_t max_pages_per_session;  /* device page-table row length                                  */
  int32_t max_blocks_per_session; /* block-boundary capacity per session                           */
  int32_t max_sessions_per_call;  /* upper bounds used to size the workspace                       */
  int32_t max_q_tokens_per_call;
  void*   k_pool;                 /* DEVICE, >= ws_pool_bytes() each                               */
  void*   v_pool;
  size_t  pool_bytes;
  void*   workspace;              /* DEVICE scratch: page tables, per-call metadata, split partials */
  size_t  workspace_bytes;        /* >= ws_workspace_bytes()                                       */
  int32_t device;                 /* CUDA device ordinal                                           */
  uint32_t flags;                 /* WS_FLAG_*                                                     */
} ws_cache_config_t;

/* Bytes each of k_pool / v_pool must hold: num_pages * Hkv * P * D * sizeof(element). */
size_t ws_pool_bytes(const ws_cache_config_t* cfg);
/* Bytes of DEVICE workspace the configuration needs (0 if cfg is invalid). */
size_t ws_workspace_bytes(const ws_cache_config_t* cfg);

/* Create a cache over caller-owned pools.  Does not touch pool contents.  The device page tables
 * inside `workspace` are initialised on the legacy default stream and synchronised before return. */
ws_status_t ws_cache_create(const ws_cache_config_t* cfg, ws_cache_t** out);
/* Destroys host metadata; never frees caller memory.  Synchronises the device first. */
ws_status_t ws_cache_destroy(ws_cache_t* cache);

ws_status_t ws_session_open(ws_cache_t* cache, int32_t* session_out);
/* Returns the session's pages to the free list. */
ws_status_t ws_session_close(ws_cache_t* cache, int32_t session);
/* Committed tokens, committed blocks, and a library-owned HOST view of the block ends
 * e_1 < ... < e_B (valid until the next mutating call on this cache).  Any out-pointer may be NULL. */
ws_status_t ws_session_info(const ws_cache_t* cache, int32_t session, int64_t* tokens,
                            int32_t* blocks, const int64_t** block_ends);
/* Roll a session back to its first `keep_blocks` committed blocks (pages beyond go back to the free
 * list; cache contents of kept blocks are untouched).  Used to replay a streaming loop. */
ws_status_t ws_session_truncate(ws_cache_t* cache, int32_t session, int32_t keep_blocks);
/* Number of pages currently on the free list. */
int32_t ws_free_pages(const ws_cache_t* cache);

/* a2 - KV append / commit.  Appends ONE block per listed session:
 *   Kc[L_s : L_s+n_s] <- k_new[cu[s] : cu[s+1]]  (same for V), bit-exact, then L_s += n_s and a block
 *   boundary e = L_s is recorded.  n_s >= 1.
 * session_ids: HOST [S] distinct open sessions; cu_new_tokens: HOST [S+1] prefix offsets (cu[0]=0);
 * k_new, v_new: DEVICE [cu[S]][Hkv][D]; modality: HOST [cu[S]] tags 0=video 1=audio 2=text or NULL
 * (stored as metadata only - it never changes the result, reading A4/A5). */
ws_status_t ws_kv_append(ws_cache_t* cache, int32_t num_sessions, const int32_t* session_ids,
                         const int32_t* cu_new_tokens, const void* k_new, const void* v_new,
                         const uint8_t* modality, void* cuda_stream);

/* NEXT-1 - commit SEVERAL blocks per session in one call (system prefill, "After system
 * prefill, the thinker broadcasts the initial KV cache": the whole initial history is built in one shot;
 * the same causal format in one pass).  Exactly ws_kv_append, except that session s's
 * n_s = cu[s+1] - cu[s] tokens are committed as the blocks block_tokens[cu_blocks[s] .. cu_blocks[s+1]) (each
 * >= 1 token, their sum must be n_s): one block end is recorded per block, in order.  One host pass, one
 * kernel launch, bit-exact.  cu_blocks: HOST [S+1] (cu_blocks[0] = 0); block_tokens: HOST [cu_blocks[S]].
 * The blocks can then be queried together with ws_block_causal_attn_fwd(num_q_blocks = their count). */
ws_status_t ws_kv_append_blocks(ws_cache_t* cache, int32_t num_sessions, const int32_t* session_ids,
                                const int32_t* cu_new_tokens, const int32_t* cu_blocks,
                                const int32_t* block_tokens, const void* k_new, const void* v_new,
                                const uint8_t* modality, void* cuda_stream);

/* a3 (+a4) - block-causal attention forward.  For each listed session the queries are the tokens of
 * its LAST num_q_blocks[s] committed blocks (1 on the hot path: the block just appended).  A query
 * row in block b sees keys j < e_b: its whole own block and every earlier block.
 *   O[r,h,:] = sum_j softmax_j(scale * <Q[r,h,:], Kc[j,g(h),:]>) Vc[j,g(h),:],  LSE = log sum_j e^{s_j}
 * session_ids: HOST [S]; num_q_blocks: HOST [S] or NULL (= 1 each); cu_q_tokens: HOST [S+1], where
 * cu[s+1]-cu[s] must equal the token count of those blocks; q: DEVICE; out: DEVICE (same dtype as
 * the cache); lse: DEVICE fp32 or NULL.  Long caches are split across CTAs and merged by a combine
 * kernel using the workspace (a4). */
ws_status_t ws_block_causal_attn_fwd(ws_cache_t* cache, int32_t num_sessions,
                                     const int32_t* session_ids, const int32_t* num_q_blocks,
                                     const int32_t* cu_q_tokens, const void* q, void* out,
                                     float* lse, float scale, void* cuda_stream);

/* ws_block_causal_attn_fwd for callers that cannot allocate or provide split-KV scratch per call (code under
 * CUDA-graph capture, serving loops and harnesses that forbid cudaMalloc): same arguments, same host path, same
 * kernels and results (a3 + a4, Eq. (1); split-KV combine from north_star), but the partials of the
 * split-KV plan go to a file-scope static __device__ array inside the library image instead of the cache's
 * workspace.  The call and everything below it call no cudaMalloc / cudaFree / allocating library routine.
 *  - Size: WS_STATIC_PART_SLOTS partial slots ([256 rows][128] fp32 + [256] fp32 LSE each) = 8,454,144 bytes,
 *    held by EVERY GPU that loads the library until the process exits.
 *  - A call whose plan needs more slots returns WS_ERR_WORKSPACE_TOO_SMALL with nothing launched and no state
 *    changed (one slot per (KV range, row-tile pair) of a split group; e.g. BASELINE config 2 needs ~144: use the
 *    workspace path there).  Plans that do not split (or the CUDA-core kernel) use no scratch at all.
 *  - Not with WS_FLAG_FUSED_COMBINE (WS_ERR_UNSUPPORTED): that mode's arrival counters live in the workspace.
 *  - ALL calls of the process on one device share the array.  Nothing in it has to start at zero (every slot a
 *    launch reads was written by the same launch chain first) and the previous call's contents are simply
 *    overwritten, but calls that OVERLAP on the GPU (different streams, different caches) race on it: issue
 *    them on one stream, or order them with events.
 *  - The device address of the array is resolved once per device (cudaGetSymbolAddress with that device
 *    current).  ws_static_scratch_setup(device) does that ahead of time - call it once per device before stream
 *    capture; otherwise the first ws_block_causal_attn_fwd_static on a device does it.                        */
#define WS_STATIC_PART_SLOTS 64
ws_status_t ws_static_scratch_setup(int32_t device);
ws_status_t ws_block_causal_attn_fwd_static(ws_cache_t* cache, int32_t num_sessions,
                                            const int32_t* session_ids, const int32_t* num_q_blocks,
                                            const int32_t* cu_q_tokens, const void* q, void* out,
                                            float* lse, float scale, void* cuda_stream);

/* NEXT-4 (optional half) - mixed intra-block mask.  PAPER.md:31 "the short token-causal Transformer pass
 * for language prediction and state update", :77 "token-causal decoding over the language and state
 * slots", while audio/video units are block-wise.  Reading A19: with
 * WS_ATTN_TEXT_CAUSAL the text slots (modality tag 2) are token-causal AMONG THEMSELVES - a text query
 * does not see text keys at later positions (those can only be in its own block) - and every other
 * (query, key) pair keeps the block-causal rule: audio/video keys of the block are visible to every query
 * of the block, text keys to every audio/video query.  attn_flags = 0 is ws_block_causal_attn_fwd.
 * Every queried token must have been appended WITH a modality tag (else WS_ERR_INVALID_ARG). */
enum { WS_ATTN_TEXT_CAUSAL = 1u };
ws_status_t ws_block_causal_attn_fwd_masked(ws_cache_t* cache, int32_t num_sessions,
                                            const int32_t* session_ids, const int32_t* num_q_blocks,
                                            const int32_t* cu_q_tokens, const void* q, void* out,
                                            float* lse, float scale, uint32_t attn_flags,
                                            void* cuda_stream);

/* One streaming-unit step with DEVICE buffers in a single call: ws_kv_append(k_new, v_new) followed by
 * ws_block_causal_attn_fwd of the block just committed (one block per session, n_q = n_new; PAPER.md:83
 * "appends the received KV slice", then the unit attends).  Same kernels and results as the two calls;
 * saves one trip through the caller's binding per step.  If the attention part fails (e.g.
 * WS_ERR_WORKSPACE_TOO_SMALL) the append has already been committed: ws_session_truncate rolls it back. */
ws_status_t ws_stream_step(ws_cache_t* cache, int32_t num_sessions, const int32_t* session_ids,
                           const int32_t* cu_new_tokens, const void* q, const void* k_new,
                           const void* v_new, void* out, float* lse, float scale, void* cuda_stream);

/* ws_stream_step with the block's modality tags (HOST [cu[S]], stored like ws_kv_append's; may be NULL when
 * attn_flags = 0) and the attention flags of ws_block_causal_attn_fwd_masked. */
ws_status_t ws_stream_step_tagged(ws_cache_t* cache, int32_t num_sessions, const int32_t* session_ids,
                                  const int32_t* cu_new_tokens, const void* q, const void* k_new,
                                  const void* v_new, const uint8_t* modality, uint32_t attn_flags,
                                  void* out, float* lse, float scale, void* cuda_stream);

/* One streaming-unit step with HOST buffers (the end-to-end path): copies q/k_new/v_new from host
 * (pinned for async copies) into `staging` (DEVICE, >= ws_step_staging_bytes(n_total); two slots used
 * alternately), runs ws_kv_append then ws_block_causal_attn_fwd (one block per session, n_q = n_new)
 * on `cuda_stream`, and copies the result back to out_host.  Copy-in and copy-out run on two internal
 * streams ordered by events, so consecutive steps overlap their copies with each other's kernels.
 * Returns after enqueueing.  out_host (and the host input buffers) may be touched again once
 * ws_stream_host_join(cache, stream) has been called and `stream` has been synchronised. */
size_t ws_step_staging_bytes(const ws_cache_config_t* cfg, int32_t total_new_tokens);
ws_status_t ws_stream_step_host(ws_cache_t* cache, int32_t num_sessions, const int32_t* session_ids,
                                const int32_t* cu_new_tokens, const void* q_host,
                                const void* k_new_host, const void* v_new_host, void* out_host,
                                void* staging, size_t staging_bytes, float scale, void* cuda_stream);
/* Makes `cuda_stream` wait for every copy-out issued by ws_stream_step_host on this cache so far. */
ws_status_t ws_stream_host_join(ws_cache_t* cache, void* cuda_stream);

/* NEXT-2 (solver-step mode): explicit Euler step of the flow-matching solver on a
 * latent unit, z <- z + dtau * v  (Eq. (2): dz/dtau = eps - z_0 is the velocity the model
 * predicts; dtau < 0 integrates from noise to data).  z, v: DEVICE, 16-byte aligned, `count` elements
 * of `dtype` (ws_dtype_t); fp32 arithmetic, one rounding to the storage dtype.  An uncommitted noisy
 * block is attended with ws_kv_append + ws_block_causal_attn_fwd + ws_session_truncate(keep) per
 * solver step (stage / attend / roll back); the clean block is committed by the last append. */
ws_status_t ws_fm_euler_update(int32_t dtype, void* z, const void* v, float dtau, int64_t count,
                               void* cuda_stream);

/* ---- NEXT-3: replica link - the thinker -> performer KV-slice exchange ---------------------------
 * PAPER.md:75 "After system prefill, the thinker broadcasts the initial KV cache to the performer";
 * :77 / :31 the thinker produces "the current KV-cache slice" every unit; :83 the performer "appends the
 * received KV slice into its own full-history cache"; :85 "KV-cache exchange".  Thinker and performer
 * hold full REPLICAS of the cache (not shards).  B200-native form: the owner (thinker) links its cache
 * to the replicas' pools mapped into its own address space (CUDA peer access in one process, or
 * cudaIpcOpenMemHandle across processes - NVLink 5 / NVSwitch carries plain stores), and from then on
 * the ONE kv_append kernel pass that commits a slice locally also stores it into every linked pool at
 * the same physical page ids (one read of k_new/v_new, local + peer 16-byte stores, system-scope fence).
 * No staging buffer, no separate send/recv, no second kernel on the replica's GPU.  The host-side
 * commit (block boundary, page adoption) travels as a small int32 message over any transport
 * (torch.distributed send/recv in the harness) and is applied by ws_replica_apply.
 *
 * Page ownership: a replica calls ws_replica_accept(owner_pages) once, before opening sessions: pages
 * [0, owner_pages) are then handed out only by ws_replica_apply (the owner names them); the replica's
 * own appends (solver-step staging, NEXT-2) draw from pages >= owner_pages, so an in-flight peer
 * write can never land in a page the replica is using for something else.
 *
 * Ordering contract (the transport's job): a message may be applied - more precisely, work that reads
 * the new tokens may be enqueued on the replica - only after the owner's append kernel has completed
 * (stream synchronised before the send, or an interprocess event waited on by the replica's stream);
 * and the owner must not append to a session while the replica still holds a staged (uncommitted)
 * block of it whose first tokens share the session's last page. */
typedef struct {
  void*  k_pool;        /* replica's K pool as addressable from the OWNER's device                    */
  void*  v_pool;
  size_t pool_bytes;    /* each; must be >= ws_pool_bytes(owner cfg) (same Hkv, P, D, dtype assumed)  */
} ws_peer_pools_t;
enum { WS_MAX_PEERS = 4 };
/* Owner side.  num_peers = 0 unlinks.  Does not touch the peers' memory. */
ws_status_t ws_replica_link(ws_cache_t* owner, const ws_peer_pools_t* peers, int32_t num_peers);
/* Replica side: reserve pages [0, owner_pages) for the owner.  No session may be open. */
ws_status_t ws_replica_accept(ws_cache_t* replica, int32_t owner_pages);
/* Owner side: serialise the commit of the LAST ws_kv_append call (or, for ws_replica_snapshot_message,
 * the whole current state of one session: every block end and page id - the "initial KV cache" message
 * after system prefill).  words: HOST int32[cap]; *n = words needed (WS_ERR_INVALID_ARG if cap < *n,
 * with *n still set, so a NULL/0 query works). */
ws_status_t ws_replica_commit_message(const ws_cache_t* owner, int32_t* words, int32_t cap, int32_t* n);
ws_status_t ws_replica_snapshot_message(const ws_cache_t* owner, int32_t session, int32_t* words,
                                        int32_t cap, int32_t* n);
/* Owner side: copy every page of `session` into the linked pools at the same page ids (the data half
 * of the initial broadcast; page-granular 16-byte copies, HBM read + NVLink write bound). */
ws_status_t ws_replica_push_session(ws_cache_t* owner, int32_t session, void* cuda_stream);
/* Replica side: validate a message against the replica's state (session at the stated length - or
 * not yet open and starting from 0, then it is opened at the owner's id; named pages inside the
 * accepted range and free; capacities) and, only if everything checks, adopt the pages, record the
 * block boundaries and publish the page ids to the device page table (a small kernel on cuda_stream,
 * CUDA-graph capturable).  The K/V bytes themselves were already stored by the owner's kernel. */
ws_status_t ws_replica_apply(ws_cache_t* replica, const int32_t* words, int32_t n, void* cuda_stream);
/* Interprocess mapping helpers (thin wrappers over cudaIpcGetMemHandle / cudaIpcOpenMemHandle that
 * also handle pointers inside a larger allocation, e.g. a torch caching-allocator segment).
 * handle: HOST 64 bytes.  ws_ipc_close takes the pointer ws_ipc_open returned. */
ws_status_t ws_ipc_export(const void* device_ptr, uint8_t* handle64, uint64_t* offset);
ws_status_t ws_ipc_open(const uint8_t* handle64, uint64_t offset, int32_t device, void** ptr_out);
ws_status_t ws_ipc_close(void* ptr, uint64_t offset);

/* Read back logical tokens [start, start+count) of a session into contiguous [count][Hkv][D]
 * DEVICE buffers (either may be NULL).  Test / snapshot utility. */
ws_status_t ws_kv_gather(const ws_cache_t* cache, int32_t session, int64_t start, int64_t count,
                         void* k_out, void* v_out, void* cuda_stream);

/* ---- host-logic introspection (no device work; usable under WS_FLAG_DRY_RUN) ------------------ */
/* Copies the session's physical page ids (HOST) into pages_out[0..cap); returns the count via n. */
ws_status_t ws_session_pages(const ws_cache_t* cache, int32_t session, int32_t* pages_out,
                             int32_t cap, int32_t* n);
/* Deterministically permute the free list (Fisher-Yates, seed) so tests can check that results do
 * not depend on the physical page assignment. */
ws_status_t ws_debug_shuffle_free_pages(ws_cache_t* cache, uint64_t seed);
/* Force the split-KV planner to cut every (session, KV head) group into at least `min_splits`
 * pieces (0 = automatic).  For split-count invariance tests. */
ws_status_t ws_debug_set_min_splits(ws_cache_t* cache, int32_t min_splits);

/* NEXT-4 (token-causal text decode: "short token-causal Transformer pass ... over
 * the language and state slots"): when every session of a call has at most 128 packed query rows
 * (n_q * Hq/Hkv <= 128) the step is cache-read bound and the scheduler switches the tcgen05 kernel to
 * the decode plan, run by the decode kernel (attn_dec_sm100.cu): one Q tile per CTA, BOTH softmax warpgroups on
 * every KV tile (64 of its 128 keys each), S double-buffered by tile parity.  Enabled by default; this switch
 * forces the general plan (A/B measurements and tests). */
ws_status_t ws_debug_set_decode_plan(ws_cache_t* cache, int32_t enable);

/* Description of the last attention plan built on this cache (a1): CTAs launched, team size,
 * number of (session,KV-head) groups, KV segments, split partial slots, combine items, and whether
 * the tcgen05 kernel (1 = general kernel; 3 = decode plan on the decode kernel) or the generic SIMT kernel (0)
 * was selected. */
typedef struct {
  int32_t num_ctas, team_size, num_groups, num_segments, num_partial_slots, num_combine_items;
  int32_t used_tensor_core_kernel, total_kv_tiles;
} ws_plan_info_t;
ws_status_t ws_last_plan_info(const ws_cache_t* cache, ws_plan_info_t* out);
/* Segment i of the last plan: group, session, kv_head, first query token, tile range [begin,end),
 * team, partial slot base (-1 = writes the final output directly). */
typedef struct {
  int32_t group, session, kv_head, q_token0, tile_begin, tile_end, team, part_base;
} ws_plan_segment_t;
ws_status_t ws_last_plan_segment(const ws_cache_t* cache, int32_t i, ws_plan_segment_t* out);

/* Number of kernels this library has launched on `cache` since creation (bench `gpu_launches`). */
int64_t ws_launch_count(const ws_cache_t* cache);

/* Bench instrumentation: when enabled, every kernel launch of this cache is bracketed by a CUDA
 * event pair recorded on the launch stream.  ws_debug_read_kernel_times synchronises those events
 * and returns, for {append, attention, combine} in that order, the summed device milliseconds and
 * the number of launches since the last read (then forgets them). */
ws_status_t ws_debug_kernel_timing(ws_cache_t* cache, int32_t enable);
ws_status_t ws_debug_read_kernel_times(ws_cache_t* cache, double* ms_sum3, int32_t* count3);

const char* ws_status_str(ws_status_t s);
const char* ws_last_error(void);
const char* ws_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WS_H_ */

// api.cu - the C ABI declared in include/ws.h: argument validation, host metadata (a1), per-call
// metadata staging, TMA descriptor creation and kernel launches.  No arithmetic of the method runs
// on the host; there is no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <string>
#include <mutex>
#include <vector>

#include "../../include/ws.h"
#include "host_cache.h"
#include "launch.h"
#include "plan.h"
#include "ws_internal.h"

namespace {

thread_local std::string g_err;

ws_status_t fail(ws_status_t st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_err = buf;
  return st;
}

#define WS_CUDA(expr)                                                                   \
  do {                                                                                  \
    cudaError_t e__ = (expr);                                                           \
    if (e__ != cudaSuccess)                                                             \
      return fail(WS_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e__));        \
  } while (0)

constexpr int kRing = 8;            // per-call metadata slots in flight
constexpr int kDefaultSms = 148;    // B200 (used for dry-run planning)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
int eb_of(int32_t dtype) { return dtype == WS_BF16 ? 2 : 4; }

bool config_valid(const ws_cache_config_t* c, const char** why) {
  auto bad = [&](const char* w) { *why = w; return false; };
  if (!c) return bad("cfg is NULL");
  if (c->dtype != WS_BF16 && c->dtype != WS_F32) return bad("dtype");
  if (c->num_q_heads < 1 || c->num_kv_heads < 1 || c->num_q_heads % c->num_kv_heads)
    return bad("num_q_heads must be a positive multiple of num_kv_heads");
  if (c->head_dim < 8 || c->head_dim > 256 || c->head_dim % 8) return bad("head_dim in [8,256], %8");
  if (c->page_tokens < 1 || c->num_pages < 1) return bad("page_tokens / num_pages");
  if (c->max_sessions < 1 || c->max_pages_per_session < 1 || c->max_blocks_per_session < 1)
    return bad("max_sessions / max_pages_per_session / max_blocks_per_session");
  if (c->max_sessions_per_call < 1 || c->max_q_tokens_per_call < 1)
    return bad("max_sessions_per_call / max_q_tokens_per_call");
  if ((int64_t)c->num_pages * c->num_kv_heads * c->page_tokens >= (1ll << 31))
    return bad("pool has more than 2^31 (token, head) rows");
  return true;
}

struct Layout {
  size_t page_table, q_to_kv, meta, part_lse, part_o, merge_ctr, total;
  size_t meta_slot_bytes;
  int32_t max_part_slots;
};

Layout make_layout(const ws_cache_config_t* c, int num_sms) {
  Layout L{};
  const int G = c->num_q_heads / c->num_kv_heads;
  size_t off = 0;
  L.page_table = off; off = align_up(off + (size_t)c->max_sessions * c->max_pages_per_session * 4, 256);
  L.q_to_kv = off;    off = align_up(off + (size_t)c->num_q_heads * 4, 256);
  const int64_t S = c->max_sessions_per_call, NQ = c->max_q_tokens_per_call;
  int64_t groups = (int64_t)c->num_kv_heads * (2 * S + NQ * G / 2048 + 1);
  int64_t words = 1024 + groups * 64 + 16 * (int64_t)num_sms + 2 * NQ + 8 * S +
                  S * (NQ / c->page_tokens + 3) + NQ / c->page_tokens;
  L.meta_slot_bytes = align_up((size_t)words * 4, 256);
  L.meta = off;       off = align_up(off + L.meta_slot_bytes * kRing, 256);
  L.max_part_slots = 4 * num_sms + 64;
  L.part_lse = off;   off = align_up(off + (size_t)L.max_part_slots * ws::kPairRows * 4, 256);
  L.part_o = off;     off = align_up(off + (size_t)L.max_part_slots * ws::kPairRows * c->head_dim * 4, 256);
  L.merge_ctr = off;  off = align_up(off + (size_t)L.max_part_slots * 2 * 4, 256);
  L.total = off;
  return L;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Process-wide plan cache (see ws_block_causal_attn_fwd): a handful of entries, least recently used out.
struct PlanCacheEntry {
  std::vector<int32_t> key;
  ws::Plan plan;
  std::vector<int32_t> blob;
  uint64_t stamp = 0;
};
std::mutex g_plan_mu;
std::vector<PlanCacheEntry> g_plan_cache;
uint64_t g_plan_clock = 0;
constexpr size_t kPlanCacheEntries = 16;

bool plan_cache_lookup(const std::vector<int32_t>& key, ws::Plan* plan, std::vector<int32_t>* blob) {
  std::lock_guard<std::mutex> lk(g_plan_mu);
  for (PlanCacheEntry& e : g_plan_cache)
    if (e.key == key) { e.stamp = ++g_plan_clock; *plan = e.plan; *blob = e.blob; return true; }
  return false;
}

void plan_cache_insert(const std::vector<int32_t>& key, const ws::Plan& plan, const std::vector<int32_t>& blob) {
  std::lock_guard<std::mutex> lk(g_plan_mu);
  PlanCacheEntry* slot = nullptr;
  if (g_plan_cache.size() < kPlanCacheEntries) { g_plan_cache.emplace_back(); slot = &g_plan_cache.back(); }
  else { slot = &g_plan_cache[0]; for (PlanCacheEntry& e : g_plan_cache) if (e.stamp < slot->stamp) slot = &e; }
  slot->key = key; slot->plan = plan; slot->blob = blob; slot->stamp = ++g_plan_clock;
}

}  // namespace

struct ws_cache {
  ws_cache_config_t cfg{};
  std::vector<int32_t> q_to_kv;       // explicit map (empty = default)
  bool default_map = true;
  std::unique_ptr<ws::HostCache> host;
  Layout lay{};
  int num_sms = kDefaultSms;
  bool dry = false;
  bool tensor_path_ok = false;
  // device views into the caller's workspace
  int32_t* d_page_table = nullptr;
  int32_t* d_q_to_kv = nullptr;
  char* d_meta = nullptr;
  float* d_part_lse = nullptr;
  float* d_part_o = nullptr;
  int32_t* d_merge_ctr = nullptr;     // fused-combine counters (all zero between launches)
  // pinned staging ring
  char* h_meta = nullptr;
  cudaEvent_t ev[kRing]{};
  bool ev_pending[kRing]{};
  int ring_pos = 0;
  EncodeTiledFn encode = nullptr;
  CUtensorMap tmap_k{}, tmap_v{};
  int32_t min_splits = 0;
  bool decode_plan_enabled = true;
  int64_t launches = 0;
  ws::Plan last_plan;
  bool last_tensor = false;
  // ws_stream_step_host pipeline: copy streams + per-slot events (2 staging slots)
  cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
  cudaEvent_t ev_h2d[2]{}, ev_compute[2]{}, ev_d2h[2]{};
  bool slot_used[2]{};
  int64_t host_steps = 0;
  // optional per-kernel timing (bench): event pairs around each launch on the launch stream
  bool timing = false;
  std::vector<cudaEvent_t> ev_pool;                       // reusable events
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> t_append, t_attn, t_combine;
  // NEXT-3 replica link
  ws::PeerPools peers{};
  std::vector<int32_t> last_commit;   // message describing the last ws_kv_append (ws_replica_commit_message)
};

namespace {

// Makes the cache's device current for the duration of an entry point (one process may own caches on
// several devices: the owner + replica mode of NEXT-3) and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(const ws_cache* c) {
    if (!c || c->dry) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != c->cfg.device)
      switched = cudaSetDevice(c->cfg.device) == cudaSuccess;
    else
      (void)cudaGetLastError();
  }
  ~DeviceGuard() { if (switched) (void)cudaSetDevice(prev); }
};

// Reserve the next metadata slot: returns host staging pointer; *dev gets the device address.
ws_status_t next_slot(ws_cache* c, size_t bytes, char** host, char** dev) {
  if (bytes > c->lay.meta_slot_bytes)
    return fail(WS_ERR_WORKSPACE_TOO_SMALL, "per-call metadata (%zu B) exceeds the slot (%zu B)",
                bytes, c->lay.meta_slot_bytes);
  int i = c->ring_pos;
  c->ring_pos = (c->ring_pos + 1) % kRing;
  if (!c->dry && c->ev_pending[i]) {
    WS_CUDA(cudaEventSynchronize(c->ev[i]));
    c->ev_pending[i] = false;
  }
  *host = c->h_meta + (size_t)i * c->lay.meta_slot_bytes;
  *dev = c->d_meta ? c->d_meta + (size_t)i * c->lay.meta_slot_bytes : nullptr;
  return WS_OK;
}

ws_status_t upload_slot(ws_cache* c, const char* host, char* dev, size_t bytes, cudaStream_t st) {
  if (c->dry) return WS_OK;
  int i = (int)((host - c->h_meta) / c->lay.meta_slot_bytes);
  WS_CUDA(cudaMemcpyAsync(dev, host, bytes, cudaMemcpyHostToDevice, st));
  WS_CUDA(cudaEventRecord(c->ev[i], st));
  c->ev_pending[i] = true;
  return WS_OK;
}

// Metadata that does not fit the kernel parameters travels through the pinned ring, whose slots are
// recycled (and waited for with cudaEventSynchronize): that cannot be captured into a CUDA graph.
ws_status_t refuse_if_capturing(cudaStream_t st, const char* what) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); return WS_OK; }
  if (cs != cudaStreamCaptureStatusNone)
    return fail(WS_ERR_UNSUPPORTED, "%s exceeds the kernel-parameter tier; this call cannot be captured "
                "into a CUDA graph (split the batch or query fewer tokens per call)", what);
  return WS_OK;
}

cudaEvent_t timing_event(ws_cache* c) {
  cudaEvent_t e = nullptr;
  if (!c->ev_pool.empty()) { e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
  if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
  return e;
}
// RAII-less helper: record an event pair around a launch when timing is enabled
struct TimedLaunch {
  ws_cache* c; std::vector<std::pair<cudaEvent_t, cudaEvent_t>>* dst; cudaStream_t st;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  TimedLaunch(ws_cache* c_, std::vector<std::pair<cudaEvent_t, cudaEvent_t>>* d, cudaStream_t s)
      : c(c_), dst(d), st(s) {
    if (c->timing) { e0 = timing_event(c); e1 = timing_event(c); if (e0) cudaEventRecord(e0, st); }
  }
  void done() {
    if (c->timing && e0 && e1) { cudaEventRecord(e1, st); dst->emplace_back(e0, e1); }
  }
};

// ---- NEXT-3 commit messages (include/ws.h): int32 words
//   [0] magic  [1] version  [2] kind  [3] sessions  [4] total words  [5] P  [6] Hkv  [7] D  [8] dtype
//   then per session: id, len_old, nblocks, npages, block_len[nblocks], page_id[npages]
constexpr int32_t kMsgMagic = 0x57534b56, kMsgVersion = 1, kMsgCommit = 1, kMsgSnapshot = 2;
constexpr int kMsgTotalWord = 4, kMsgHeaderWords = 9;
void msg_begin(const ws_cache* c, std::vector<int32_t>& msg, int32_t kind, int32_t S) {
  msg.clear();
  msg.insert(msg.end(), {kMsgMagic, kMsgVersion, kind, S, 0, c->cfg.page_tokens, c->cfg.num_kv_heads,
                         c->cfg.head_dim, c->cfg.dtype});
}

ws_status_t copy_message(const std::vector<int32_t>& msg, int32_t* words, int32_t cap, int32_t* n) {
  if (!n) return fail(WS_ERR_INVALID_ARG, "n is NULL");
  *n = (int32_t)msg.size();
  if (msg.empty()) return fail(WS_ERR_INVALID_ARG, "no append has been made on this cache yet");
  if (!words || cap < *n) return fail(WS_ERR_INVALID_ARG, "message needs %d words, cap is %d", *n, cap);
  memcpy(words, msg.data(), msg.size() * 4);
  return WS_OK;
}

ws_status_t encode_tmap(ws_cache* c, CUtensorMap* out, void* base, int rank, const cuuint64_t* dims,
                        const cuuint64_t* strides_bytes, const cuuint32_t* box) {
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = c->encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, base, dims,
                         strides_bytes, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(WS_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return WS_OK;
}

}  // namespace

extern "C" {

size_t ws_pool_bytes(const ws_cache_config_t* cfg) {
  const char* why;
  if (!config_valid(cfg, &why)) return 0;
  return (size_t)cfg->num_pages * cfg->num_kv_heads * cfg->page_tokens * cfg->head_dim *
         eb_of(cfg->dtype);
}

size_t ws_workspace_bytes(const ws_cache_config_t* cfg) {
  const char* why;
  if (!config_valid(cfg, &why)) return 0;
  int sms = kDefaultSms;
  if (!(cfg->flags & WS_FLAG_DRY_RUN)) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, cfg->device) == cudaSuccess && v > 0)
      sms = v;
    else
      (void)cudaGetLastError();
  }
  return make_layout(cfg, sms).total;
}

ws_status_t ws_cache_create(const ws_cache_config_t* cfg, ws_cache_t** out) {
  const char* why = "";
  if (!out) return fail(WS_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!config_valid(cfg, &why)) return fail(WS_ERR_INVALID_ARG, "invalid config: %s", why);
  std::unique_ptr<ws_cache> c(new ws_cache());
  c->cfg = *cfg;
  c->dry = (cfg->flags & WS_FLAG_DRY_RUN) != 0;
  const int G = cfg->num_q_heads / cfg->num_kv_heads;
  if (cfg->q_to_kv_head) {
    c->q_to_kv.assign(cfg->q_to_kv_head, cfg->q_to_kv_head + cfg->num_q_heads);
    for (int h = 0; h < cfg->num_q_heads; ++h) {
      if (c->q_to_kv[h] < 0 || c->q_to_kv[h] >= cfg->num_kv_heads)
        return fail(WS_ERR_INVALID_ARG, "q_to_kv_head[%d] out of range", h);
      if (c->q_to_kv[h] != h / G) c->default_map = false;
    }
  }
  c->cfg.q_to_kv_head = nullptr;
  c->host.reset(new ws::HostCache(cfg->num_pages, cfg->page_tokens, cfg->max_sessions,
                                  cfg->max_pages_per_session, cfg->max_blocks_per_session));
  c->tensor_path_ok = cfg->dtype == WS_BF16 && cfg->head_dim == 128 && cfg->page_tokens == 64 &&
                      c->default_map && (G == 1 || G == 2 || G == 4 || G == 8 || G == 16);
  if (c->dry) {
    c->lay = make_layout(cfg, kDefaultSms);
    c->h_meta = (char*)malloc(c->lay.meta_slot_bytes * kRing);
    if (!c->h_meta) return fail(WS_ERR_INVALID_ARG, "out of host memory");
    *out = c.release();
    return WS_OK;
  }
  if (!cfg->k_pool || !cfg->v_pool || !cfg->workspace)
    return fail(WS_ERR_INVALID_ARG, "k_pool / v_pool / workspace must be device pointers");
  if (cfg->pool_bytes < ws_pool_bytes(cfg))
    return fail(WS_ERR_INVALID_ARG, "pool_bytes %zu < required %zu", cfg->pool_bytes, ws_pool_bytes(cfg));
  WS_CUDA(cudaSetDevice(cfg->device));
  int sms = 0;
  WS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cfg->device));
  c->num_sms = sms;
  c->lay = make_layout(cfg, sms);
  if (cfg->workspace_bytes < c->lay.total)
    return fail(WS_ERR_WORKSPACE_TOO_SMALL, "workspace_bytes %zu < required %zu",
                cfg->workspace_bytes, c->lay.total);
  char* ws_base = (char*)cfg->workspace;
  if (((uintptr_t)ws_base & 255) || ((uintptr_t)cfg->k_pool & 255) || ((uintptr_t)cfg->v_pool & 255))
    return fail(WS_ERR_INVALID_ARG, "pools and workspace must be 256-byte aligned");
  c->d_page_table = (int32_t*)(ws_base + c->lay.page_table);
  c->d_q_to_kv = (int32_t*)(ws_base + c->lay.q_to_kv);
  c->d_meta = ws_base + c->lay.meta;
  c->d_part_lse = (float*)(ws_base + c->lay.part_lse);
  c->d_part_o = (float*)(ws_base + c->lay.part_o);
  c->d_merge_ctr = (int32_t*)(ws_base + c->lay.merge_ctr);
  WS_CUDA(cudaMemset(c->d_merge_ctr, 0, (size_t)c->lay.max_part_slots * 2 * 4));
  WS_CUDA(cudaMemset(c->d_page_table, 0, (size_t)cfg->max_sessions * cfg->max_pages_per_session * 4));
  if (!c->default_map)
    WS_CUDA(cudaMemcpy(c->d_q_to_kv, c->q_to_kv.data(), c->q_to_kv.size() * 4, cudaMemcpyHostToDevice));
  WS_CUDA(cudaHostAlloc((void**)&c->h_meta, c->lay.meta_slot_bytes * kRing, cudaHostAllocDefault));
  for (int i = 0; i < kRing; ++i) WS_CUDA(cudaEventCreateWithFlags(&c->ev[i], cudaEventDisableTiming));
  if (c->tensor_path_ok) {
    int major = 0;
    WS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, cfg->device));
    if (major != 10) {
      c->tensor_path_ok = false;      // tcgen05 kernel is sm_100a only; generic kernel still runs
    } else {
      void* fn = nullptr;
      cudaDriverEntryPointQueryResult qres;
      WS_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
      if (!fn || qres != cudaDriverEntryPointSuccess)
        return fail(WS_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
      c->encode = (EncodeTiledFn)fn;
      const cuuint64_t D = 128, P = 64, H = cfg->num_kv_heads, NP = cfg->num_pages;
      cuuint64_t dims[4] = {D, P, H, NP};
      cuuint64_t strides[3] = {D * 2, P * D * 2, H * P * D * 2};
      cuuint32_t box[4] = {64, 64, 1, 1};
      ws_status_t st = encode_tmap(c.get(), &c->tmap_k, cfg->k_pool, 4, dims, strides, box);
      if (st != WS_OK) return st;
      st = encode_tmap(c.get(), &c->tmap_v, cfg->v_pool, 4, dims, strides, box);
      if (st != WS_OK) return st;
      WS_CUDA(ws::sm100_attn_configure());
      WS_CUDA(ws::dec_sm100_configure());
      WS_CUDA(ws::combine_configure());
    }
  }
  WS_CUDA(cudaDeviceSynchronize());
  *out = c.release();
  return WS_OK;
}

ws_status_t ws_cache_destroy(ws_cache_t* c) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (c->dry) {
    free(c->h_meta);
  } else {
    DeviceGuard dg(c);
    (void)cudaDeviceSynchronize();          // the cache's device: copies from the pinned ring may be in flight
    for (int i = 0; i < kRing; ++i)
      if (c->ev[i]) (void)cudaEventDestroy(c->ev[i]);
    for (auto* lst : {&c->t_append, &c->t_attn, &c->t_combine})
      for (auto& pr : *lst) { (void)cudaEventDestroy(pr.first); (void)cudaEventDestroy(pr.second); }
    for (cudaEvent_t e : c->ev_pool) (void)cudaEventDestroy(e);
    if (c->h2d_stream) {
      for (int i = 0; i < 2; ++i) {
        (void)cudaEventDestroy(c->ev_h2d[i]); (void)cudaEventDestroy(c->ev_compute[i]); (void)cudaEventDestroy(c->ev_d2h[i]);
      }
      (void)cudaStreamDestroy(c->h2d_stream); (void)cudaStreamDestroy(c->d2h_stream);
    }
    if (c->h_meta) (void)cudaFreeHost(c->h_meta);
  }
  delete c;
  return WS_OK;
}

ws_status_t ws_session_open(ws_cache_t* c, int32_t* session_out) {
  if (!c || !session_out) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  int32_t s = c->host->open_session();
  if (s < 0) return fail(WS_ERR_BAD_SESSION, "all %d session slots are open", c->cfg.max_sessions);
  *session_out = s;
  return WS_OK;
}

ws_status_t ws_session_close(ws_cache_t* c, int32_t session) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (!c->host->close_session(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  return WS_OK;
}

ws_status_t ws_session_info(const ws_cache_t* c, int32_t session, int64_t* tokens, int32_t* blocks,
                            const int64_t** block_ends) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (!c->host->is_open(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  const ws::SessionState& st = c->host->session(session);
  if (tokens) *tokens = st.tokens;
  if (blocks) *blocks = (int32_t)st.block_ends.size();
  if (block_ends) *block_ends = st.block_ends.data();
  return WS_OK;
}

ws_status_t ws_session_truncate(ws_cache_t* c, int32_t session, int32_t keep_blocks) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (!c->host->is_open(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  if (!c->host->truncate_blocks(session, keep_blocks))
    return fail(WS_ERR_INVALID_ARG, "keep_blocks %d out of range", keep_blocks);
  return WS_OK;
}

int32_t ws_free_pages(const ws_cache_t* c) { return c ? c->host->free_pages() : -1; }

ws_status_t ws_session_pages(const ws_cache_t* c, int32_t session, int32_t* pages_out, int32_t cap,
                             int32_t* n) {
  if (!c || !n) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  if (!c->host->is_open(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  const auto& pg = c->host->session(session).pages;
  *n = (int32_t)pg.size();
  for (int32_t i = 0; i < cap && i < *n && pages_out; ++i) pages_out[i] = pg[i];
  return WS_OK;
}

ws_status_t ws_debug_shuffle_free_pages(ws_cache_t* c, uint64_t seed) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  c->host->shuffle_free(seed);
  return WS_OK;
}

ws_status_t ws_debug_set_decode_plan(ws_cache_t* c, int32_t enable) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  c->decode_plan_enabled = enable != 0;
  return WS_OK;
}

ws_status_t ws_debug_set_min_splits(ws_cache_t* c, int32_t min_splits) {
  if (!c || min_splits < 0) return fail(WS_ERR_INVALID_ARG, "bad argument");
  c->min_splits = min_splits;
  return WS_OK;
}

// ------------------------------------------------------------------------------------ a2 append
}  // extern "C"

namespace {

// The append of one call, prepared on the host: validated, committed to the host metadata, descriptor blob
// built - in `inl` (kernel-parameter tier) or in a slot of the pinned ring (`h` / `d`).
struct AppendPrep {
  bool inline_meta = true;
  ws::InlineAppendMeta inl{};
  char* h = nullptr;
  char* d = nullptr;
  size_t bytes = 0;
};

// No state changes.  *words = size of the descriptor blob.
// cu_blocks / block_tokens (ws_kv_append_blocks): session s commits its n_s tokens as the blocks
// block_tokens[cu_blocks[s] .. cu_blocks[s+1]); both NULL = one block per session.
ws_status_t append_validate(ws_cache* c, int32_t S, const int32_t* session_ids, const int32_t* cu,
                            const void* k_new, const void* v_new, size_t* words_out,
                            const int32_t* cu_blocks = nullptr, const int32_t* block_tokens = nullptr) {
  if (!c || !session_ids || !cu) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  if ((cu_blocks == nullptr) != (block_tokens == nullptr))
    return fail(WS_ERR_INVALID_ARG, "cu_blocks and block_tokens must be given together");
  if (cu_blocks && cu_blocks[0] != 0) return fail(WS_ERR_INVALID_ARG, "cu_blocks[0] must be 0");
  if (S < 1 || S > c->cfg.max_sessions_per_call)
    return fail(WS_ERR_INVALID_ARG, "num_sessions %d not in [1, %d]", S, c->cfg.max_sessions_per_call);
  if (!c->dry && (!k_new || !v_new)) return fail(WS_ERR_INVALID_ARG, "k_new / v_new is NULL");
  if (cu[0] != 0) return fail(WS_ERR_INVALID_ARG, "cu_new_tokens[0] must be 0");
  const int32_t P = c->cfg.page_tokens;
  int64_t extra_pages = 0;
  for (int32_t s = 0; s < S; ++s) {
    int32_t n = cu[s + 1] - cu[s];
    if (n < 1) return fail(WS_ERR_INVALID_ARG, "session %d appends %d tokens (must be >= 1)", s, n);
    int32_t id = session_ids[s];
    if (!c->host->is_open(id)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", id);
    for (int32_t t = 0; t < s; ++t)
      if (session_ids[t] == id) return fail(WS_ERR_INVALID_ARG, "session %d listed twice", id);
    int32_t nb = 1;
    if (cu_blocks) {
      nb = cu_blocks[s + 1] - cu_blocks[s];
      if (nb < 1) return fail(WS_ERR_INVALID_ARG, "session %d commits %d blocks (must be >= 1)", s, nb);
      int64_t sum = 0;
      for (int32_t b = cu_blocks[s]; b < cu_blocks[s + 1]; ++b) {
        if (block_tokens[b] < 1) return fail(WS_ERR_INVALID_ARG, "session %d: block of %d tokens", s, block_tokens[b]);
        sum += block_tokens[b];
      }
      if (sum != n)
        return fail(WS_ERR_INVALID_ARG, "session %d: its blocks hold %lld tokens, cu_new_tokens gives %d", s,
                    (long long)sum, n);
    }
    if (!c->host->fits(id, n, nb))
      return fail(WS_ERR_OUT_OF_PAGES, "session %d exceeds its page-table or block capacity", id);
    if (c->host->session(id).tokens + n >= (1ll << 31))
      return fail(WS_ERR_UNSUPPORTED, "session %d would exceed 2^31 tokens", id);
    extra_pages += c->host->pages_needed(id, c->host->session(id).tokens + n);
  }
  if (cu[S] > c->cfg.max_q_tokens_per_call)
    return fail(WS_ERR_INVALID_ARG, "%d new tokens > max_q_tokens_per_call %d", cu[S],
                c->cfg.max_q_tokens_per_call);
  if (extra_pages > c->host->free_pages())
    return fail(WS_ERR_OUT_OF_PAGES, "need %lld pages, %d free", (long long)extra_pages,
                c->host->free_pages());
  size_t words = sizeof(ws::AppendMeta) / 4 + (size_t)S * sizeof(ws::AppendSession) / 4;
  for (int32_t s = 0; s < S; ++s) words += (size_t)(cu[s + 1] - cu[s]) / P + 3;
  if (words * 4 > c->lay.meta_slot_bytes)
    return fail(WS_ERR_WORKSPACE_TOO_SMALL, "append metadata exceeds the slot");
  *words_out = words;
  return WS_OK;
}

// Commits the blocks to the host metadata and builds the descriptor.  Call only after append_validate.
ws_status_t append_commit(ws_cache* c, int32_t S, const int32_t* session_ids, const int32_t* cu,
                          const uint8_t* modality, size_t words, cudaStream_t stream, AppendPrep* ap,
                          const int32_t* cu_blocks = nullptr, const int32_t* block_tokens = nullptr) {
  ap->inline_meta = words <= (size_t)ws::kInlineAppendWords;
  char* h = (char*)ap->inl.w;
  if (!ap->inline_meta) {
    if (!c->dry) {
      ws_status_t st = refuse_if_capturing(stream, "append metadata");
      if (st != WS_OK) return st;
    }
    ws_status_t st = next_slot(c, words * 4, &ap->h, &ap->d);
    if (st != WS_OK) return st;
    h = ap->h;
  }
  // ---- commit (no failure paths below)
  ws::AppendMeta hdr{S, cu[S], (int32_t)(sizeof(ws::AppendMeta) / 4),
                     (int32_t)(sizeof(ws::AppendMeta) / 4 + S * sizeof(ws::AppendSession) / 4)};
  int32_t* blob = (int32_t*)h;
  ws::AppendSession* as = (ws::AppendSession*)(blob + hdr.off_sessions);
  int32_t* pages = blob + hdr.off_pages;
  int32_t npg = 0;
  std::vector<int32_t>& msg = c->last_commit;
  msg_begin(c, msg, kMsgCommit, S);
  for (int32_t s = 0; s < S; ++s) {
    int32_t id = session_ids[s], n = cu[s + 1] - cu[s];
    int64_t len_old = c->host->session(id).tokens;
    const size_t old_pages = c->host->session(id).pages.size();
    // the device side sees one contiguous run of n tokens per session whatever its block structure
    const int32_t nb = cu_blocks ? cu_blocks[s + 1] - cu_blocks[s] : 1;
    const int32_t* lens = cu_blocks ? block_tokens + cu_blocks[s] : &n;
    const int32_t first = (int32_t)(len_old / c->cfg.page_tokens);
    c->host->note_append(id);
    for (int32_t b = 0, done = 0; b < nb; done += lens[b], ++b)
      c->host->commit_block(id, lens[b], modality ? modality + cu[s] + done : nullptr);
    const ws::SessionState& ss = c->host->session(id);
    as[s] = ws::AppendSession{id, (int32_t)len_old, cu[s], cu[s + 1], npg, {0, 0, 0}};
    for (size_t i = first; i < ss.pages.size(); ++i) pages[npg++] = ss.pages[i];
    msg.insert(msg.end(), {id, (int32_t)len_old, nb, (int32_t)(ss.pages.size() - old_pages)});
    msg.insert(msg.end(), lens, lens + nb);
    msg.insert(msg.end(), ss.pages.begin() + old_pages, ss.pages.end());
  }
  msg[kMsgTotalWord] = (int32_t)msg.size();
  memcpy(blob, &hdr, sizeof(hdr));
  ap->bytes = (size_t)(hdr.off_pages + npg) * 4;
  return WS_OK;
}

ws_status_t append_launch(ws_cache* c, const AppendPrep& ap, const void* k_new, const void* v_new,
                          int32_t total_tokens, cudaStream_t stream) {
  if (c->dry) return WS_OK;
  if (!ap.inline_meta) {
    ws_status_t st = upload_slot(c, ap.h, ap.d, ap.bytes, stream);
    if (st != WS_OK) return st;
  }
  TimedLaunch tl(c, &c->t_append, stream);
  WS_CUDA(ws::launch_kv_append(k_new, v_new, c->cfg.k_pool, c->cfg.v_pool, c->d_page_table,
                               ap.inline_meta ? nullptr : (const int32_t*)ap.d, ap.inl, c->peers, total_tokens,
                               c->cfg.max_pages_per_session, c->cfg.page_tokens, c->cfg.num_kv_heads,
                               c->cfg.head_dim, eb_of(c->cfg.dtype), c->num_sms, stream));
  tl.done();
  c->launches += 1;
  return WS_OK;
}

// Fused step: the block committed by `ap` is attended in the same launch (tcgen05 kernel only).
struct FusedAppend {
  const AppendPrep* ap;
  const void* k_new;
  const void* v_new;
};

// a3 + a4.  fuse != nullptr: every session's last block (its cu range) is the one being committed by this
// launch: its keys are read from k_new / v_new, and warps 10-11 of the kernel copy it into the pool.
ws_status_t attn_impl(ws_cache* c, int32_t S, const int32_t* session_ids, const int32_t* num_q_blocks,
                      const int32_t* cu, const void* q, void* out, float* lse, float scale,
                      cudaStream_t stream, const FusedAppend* fuse, uint32_t attn_flags = 0) {
  std::vector<ws::PlanSession> ps(S);
  std::vector<int32_t> vis_end, tok_slot;
  bool any_multi = false;
  if (attn_flags & ~(uint32_t)WS_ATTN_TEXT_CAUSAL) return fail(WS_ERR_INVALID_ARG, "unknown attn_flags 0x%x", attn_flags);
  // NEXT-4 mixed mask (reading A19): per session a record {abs_pos0, nbits, text bits of the query tokens...}
  const bool text_causal = (attn_flags & WS_ATTN_TEXT_CAUSAL) != 0;
  std::vector<int32_t> txt_words, txt_pos, txt_rec;
  for (int32_t s = 0; s < S; ++s) {
    int32_t id = session_ids[s];
    if (!c->host->is_open(id)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", id);
    const ws::SessionState& ss = c->host->session(id);
    int32_t m = num_q_blocks ? num_q_blocks[s] : 1;
    int32_t B = (int32_t)ss.block_ends.size();
    if (m < 1 || m > B)
      return fail(WS_ERR_INVALID_ARG, "session %d: num_q_blocks %d not in [1, %d]", id, m, B);
    int64_t q_start = (B - m) ? ss.block_ends[B - m - 1] : 0;
    int64_t nq = ss.tokens - q_start;
    if (cu[s + 1] - cu[s] != nq)
      return fail(WS_ERR_INVALID_ARG, "session %d: cu gives %d query tokens, its last %d block(s) hold %lld",
                  id, cu[s + 1] - cu[s], m, (long long)nq);
    ps[s] = ws::PlanSession{id, cu[s], cu[s + 1], m > 1, fuse ? (int32_t)nq : 0, (int32_t)ss.settled[1], -1};
    if (text_causal) {
      if ((int64_t)ss.modality.size() < ss.tokens)
        return fail(WS_ERR_INVALID_ARG, "session %d: WS_ATTN_TEXT_CAUSAL needs modality tags for the queried tokens", id);
      ps[s].txt_off = (int32_t)txt_words.size();
      const size_t rec = txt_words.size();
      txt_words.push_back((int32_t)q_start);
      txt_words.push_back((int32_t)nq);
      txt_words.resize(rec + 2 + (size_t)(nq + 31) / 32, 0);
      for (int64_t k = 0; k < nq; ++k) {
        const uint8_t tag = ss.modality[(size_t)(q_start + k)];
        if (tag > 2)
          return fail(WS_ERR_INVALID_ARG, "session %d: token %lld was appended without a modality tag", id,
                      (long long)(q_start + k));
        if (tag == 2) txt_words[rec + 2 + (size_t)(k >> 5)] |= (int32_t)(1u << (k & 31));
        txt_pos.push_back(tag == 2 ? (int32_t)(q_start + k) : -1);
        txt_rec.push_back((int32_t)rec);
      }
    }
    any_multi |= m > 1;
    for (int32_t b = B - m; b < B; ++b) {
      int64_t lo = b ? ss.block_ends[b - 1] : 0;
      vis_end.insert(vis_end.end(), (size_t)(ss.block_ends[b] - lo), (int32_t)ss.block_ends[b]);
    }
    tok_slot.insert(tok_slot.end(), (size_t)nq, id);
  }
  const int32_t NQ = cu[S];
  if (NQ > c->cfg.max_q_tokens_per_call)
    return fail(WS_ERR_INVALID_ARG, "%d query tokens > max_q_tokens_per_call %d", NQ,
                c->cfg.max_q_tokens_per_call);
  const bool tensor = c->tensor_path_ok && !(c->cfg.flags & WS_FLAG_FORCE_SIMT);
  c->last_tensor = tensor;
  const int G = c->cfg.num_q_heads / c->cfg.num_kv_heads;
  char *h = nullptr, *d = nullptr;

  if (!tensor) {
    if (c->dry && !c->tensor_path_ok) { c->last_plan = ws::Plan(); return WS_OK; }
    if (!c->dry) {
      // rows: session slot, visible end [, text position or -1, record offset; then the text-bit records]
      std::vector<int32_t> tm(tok_slot);
      tm.insert(tm.end(), vis_end.begin(), vis_end.end());
      if (text_causal) {
        tm.insert(tm.end(), txt_pos.begin(), txt_pos.end());
        tm.insert(tm.end(), txt_rec.begin(), txt_rec.end());      // (rebased below, once the row count is known)
      }
      if (fuse) {                      // committed length before this step's append, first row in k_new
        for (int32_t s2 = 0; s2 < S; ++s2) tm.insert(tm.end(), (size_t)(cu[s2 + 1] - cu[s2]), vis_end[cu[s2]] - (cu[s2 + 1] - cu[s2]));
        for (int32_t s2 = 0; s2 < S; ++s2) tm.insert(tm.end(), (size_t)(cu[s2 + 1] - cu[s2]), cu[s2]);
      }
      if (text_causal) {
        for (int32_t& r : txt_rec) r += (int32_t)tm.size();
        for (size_t t2 = 0; t2 < txt_rec.size(); ++t2) tm[3 * (size_t)NQ + t2] = txt_rec[t2];
        tm.insert(tm.end(), txt_words.begin(), txt_words.end());
      }
      const size_t bytes = tm.size() * 4;
      ws::InlineAppendMeta inl;
      ws_status_t st = WS_OK;
      if (tm.size() <= (size_t)ws::kInlineAppendWords) {
        // small call (the fp32 config: 16 tokens): the metadata rides in the kernel parameters
        memcpy(inl.w, tm.data(), bytes);
        d = nullptr;
      } else {
        st = refuse_if_capturing(stream, "generic-kernel metadata");
        if (st != WS_OK) return st;
        st = next_slot(c, bytes, &h, &d);
        if (st != WS_OK) return st;
        memcpy(h, tm.data(), bytes);
        st = upload_slot(c, h, d, bytes, stream);
        if (st != WS_OK) return st;
      }
      ws::SimtFused sf{};
      if (fuse) sf = ws::SimtFused{fuse->k_new, fuse->v_new, c->cfg.k_pool, c->cfg.v_pool, c->d_page_table, &fuse->ap->inl, NQ};
      TimedLaunch tl(c, &c->t_attn, stream);
      WS_CUDA(ws::launch_attn_simt(c->cfg.dtype, q, out, lse, c->cfg.k_pool, c->cfg.v_pool,
                                   c->d_page_table, (const int32_t*)d, inl,
                                   c->default_map ? nullptr : c->d_q_to_kv, NQ,
                                   c->cfg.max_pages_per_session, c->cfg.num_q_heads,
                                   c->cfg.num_kv_heads, c->cfg.head_dim, c->cfg.page_tokens, scale,
                                   text_causal ? 1 : 0, fuse ? &sf : nullptr, stream));
      tl.done();
      c->launches += 1;
      c->last_plan = ws::Plan();
      return WS_OK;
    }
  }

  ws::PlanConfig pc{c->cfg.num_kv_heads, G, c->num_sms, /*min_tiles=*/2, /*seg_overhead_tiles=*/3.3f,
                    c->min_splits, c->lay.max_part_slots, c->decode_plan_enabled};
  // The plan is a pure function of the head geometry and the sessions' (query range, cache length): the
  // layers of one model step (one cache handle each, same sessions, same lengths) all need the same one,
  // so single-block steps look it up in a small process-wide cache before planning (~6-15 us of host work).
  ws::Plan plan;
  std::vector<int32_t> blob;
  std::vector<int32_t> key;
  bool cached = false;
  const bool cacheable = !any_multi && !text_causal;
  if (cacheable) {
    key.reserve(8 + 6 * (size_t)S);
    key.insert(key.end(), {pc.Hkv, pc.G, pc.num_sms, pc.min_splits, pc.max_part_slots, (int32_t)pc.allow_alt, S});
    for (int32_t s = 0; s < S; ++s)
      key.insert(key.end(), {ps[s].slot, ps[s].q_begin, ps[s].q_end, vis_end[ps[s].q_begin], ps[s].new_len,
                             ps[s].stable_len / ws::kTileKeys});
    cached = plan_cache_lookup(key, &plan, &blob);
  }
  if (!cached) {
    plan = ws::build_plan(pc, ps, vis_end);
    if (!plan.ok && plan.alt) {           // too many (session, head) groups for two partials each
      pc.allow_alt = false;
      plan = ws::build_plan(pc, ps, vis_end);
    }
    if (!plan.ok)
      return fail(WS_ERR_WORKSPACE_TOO_SMALL, "plan needs %d partial slots, workspace holds %d",
                  plan.num_part_slots, c->lay.max_part_slots);
    blob = ws::serialise_plan(plan, vis_end, any_multi, txt_words);
    if (cacheable) plan_cache_insert(key, plan, blob);
  }
  const bool inline_meta = blob.size() <= (size_t)ws::kInlineAttnWordsLarge;
  ws_status_t st = WS_OK;
  if (!inline_meta && !c->dry) {
    st = refuse_if_capturing(stream, "attention metadata");
    if (st != WS_OK) return st;
  }
  if (!inline_meta) {
    st = next_slot(c, blob.size() * 4, &h, &d);
    if (st != WS_OK) return st;
    memcpy(h, blob.data(), blob.size() * 4);
  }
  c->last_plan = std::move(plan);
  if (c->dry) return WS_OK;

  ws::Sm100Launch L{};
  L.p.q = q; L.p.out = out; L.p.lse = lse;
  L.p.k_pool = c->cfg.k_pool; L.p.v_pool = c->cfg.v_pool;
  L.p.page_table = c->d_page_table;
  L.p.part_o = c->d_part_o; L.p.part_lse = c->d_part_lse;
  // (decode plans run on the decode kernel, which has no in-kernel merge phase: they keep the combine kernel)
  const bool fused_combine = (c->cfg.flags & WS_FLAG_FUSED_COMBINE) && !c->last_plan.combine.empty() && !c->last_plan.alt;
  L.p.merge_ctr = fused_combine ? c->d_merge_ctr : nullptr;
  L.p.max_part_slots = c->lay.max_part_slots;
  L.p.max_pages_per_session = c->cfg.max_pages_per_session;
  L.p.Hq = c->cfg.num_q_heads; L.p.Hkv = c->cfg.num_kv_heads; L.p.D = c->cfg.head_dim;
  L.p.G = G; L.p.P = c->cfg.page_tokens; L.p.total_q_tokens = NQ; L.p.scale = scale;
  L.tmap_k = c->tmap_k; L.tmap_v = c->tmap_v;
  L.tmap_kn = c->tmap_k; L.tmap_vn = c->tmap_v;
  // every tensor map is encoded before anything is enqueued: a failure leaves the stream untouched
  {
    const cuuint64_t D = 128, Hq = c->cfg.num_q_heads;
    cuuint64_t dims[3] = {D, Hq, (cuuint64_t)NQ};
    cuuint64_t strides[2] = {D * 2, Hq * D * 2};
    cuuint32_t box[3] = {64, (cuuint32_t)G, (cuuint32_t)(ws::kTileRows / G)};
    st = encode_tmap(c, &L.tmap_q, const_cast<void*>(q), 3, dims, strides, box);
    if (st != WS_OK) return st;
  }
  if (fuse) {
    const cuuint64_t D = 128, Hkv = c->cfg.num_kv_heads;
    cuuint64_t dims[3] = {D, Hkv, (cuuint64_t)NQ};
    cuuint64_t strides[2] = {D * 2, Hkv * D * 2};
    cuuint32_t box[3] = {64, 1, 64};
    st = encode_tmap(c, &L.tmap_kn, const_cast<void*>(fuse->k_new), 3, dims, strides, box);
    if (st != WS_OK) return st;
    st = encode_tmap(c, &L.tmap_vn, const_cast<void*>(fuse->v_new), 3, dims, strides, box);
    if (st != WS_OK) return st;
    L.p.k_new = fuse->k_new; L.p.v_new = fuse->v_new;
    L.p.k_pool_w = c->cfg.k_pool; L.p.v_pool_w = c->cfg.v_pool; L.p.page_table_w = c->d_page_table;
    L.p.append_tokens = NQ;
    L.app = fuse->ap->inl;
    L.peers = c->peers;
  }
  if (!inline_meta) {
    st = upload_slot(c, h, d, blob.size() * 4, stream);
    if (st != WS_OK) return st;
  }
  if (inline_meta) { memcpy(L.inl.w, blob.data(), blob.size() * 4); d = nullptr; }
  L.inl_words = inline_meta ? (int32_t)blob.size() : 0;
  L.p.meta = (const int32_t*)d;
  L.num_ctas = c->last_plan.num_teams * c->last_plan.team_size;
  L.alt = c->last_plan.alt;
  TimedLaunch tl(c, &c->t_attn, stream);
  if (L.alt) WS_CUDA(ws::launch_attn_dec_sm100(L, stream));
  else WS_CUDA(ws::launch_attn_sm100(L, stream));
  tl.done();
  c->launches += 1;
  if (!c->last_plan.combine.empty() && !fused_combine) {
    TimedLaunch tc(c, &c->t_combine, stream);
    int32_t max_parts = 1;
    for (const ws::CombineItem& ci : c->last_plan.combine) max_parts = std::max(max_parts, ci.nparts);
    int32_t max_nq = 0;                                    // most query tokens of one session in this call
    for (int32_t s = 0; s < S; ++s) max_nq = std::max(max_nq, cu[s + 1] - cu[s]);
    WS_CUDA(ws::launch_combine(L.p, L.inl, L.inl_words, (int32_t)c->last_plan.combine.size(), c->last_plan.team_size, max_parts,
                               (int32_t)std::min<int64_t>(ws::kPairRows, (int64_t)max_nq * G), stream));
    tc.done();
    c->launches += 1;
  }
  return WS_OK;
}

ws_status_t attn_validate_args(ws_cache* c, int32_t S, const int32_t* session_ids, const int32_t* cu,
                               const void* q, void* out, float scale) {
  if (!c || !session_ids || !cu) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  if (S < 1 || S > c->cfg.max_sessions_per_call)
    return fail(WS_ERR_INVALID_ARG, "num_sessions %d not in [1, %d]", S, c->cfg.max_sessions_per_call);
  if (!c->dry && (!q || !out)) return fail(WS_ERR_INVALID_ARG, "q / out is NULL");
  if (!(scale > 0.f) || !std::isfinite(scale)) return fail(WS_ERR_INVALID_ARG, "scale must be finite and > 0");
  if (cu[0] != 0) return fail(WS_ERR_INVALID_ARG, "cu_q_tokens[0] must be 0");
  return WS_OK;
}

// ---- ws_block_causal_attn_fwd_static: split-KV scratch inside the library image (no allocation anywhere) ----
// The partials of the split-KV plan (a3 -> a4: normalised fp32 O per partial slot + log2-LSEs) normally live in
// the caller's workspace.  This array is the same scratch for callers that cannot provide / allocate one:
// WS_STATIC_PART_SLOTS partial slots of [256 rows][128] fp32 followed by the slots' [256] fp32 LSEs = 8,454,144
// bytes, held by every GPU that loads the library until the process exits.  In HOST code the name below is only
// a stand-in for the symbol: the device address comes from cudaGetSymbolAddress, once per device, with that
// device current (static_scratch_ensure), and that pointer is what the kernels get.
constexpr size_t kStaticPartOBytes = (size_t)WS_STATIC_PART_SLOTS * ws::kPairRows * 128 * sizeof(float);
constexpr size_t kStaticPartLseBytes = (size_t)WS_STATIC_PART_SLOTS * ws::kPairRows * sizeof(float);
static __device__ __align__(256) unsigned char g_static_part_scratch[kStaticPartOBytes + kStaticPartLseBytes];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_scratch_ptr[kStaticMaxDevices] = {};      // device address of the array on each device (0 = not set up)

// Resolves the array's address on `device` (made current for the call, restored afterwards).  No allocation:
// the array is part of the loaded module.
ws_status_t static_scratch_ensure(int device, void** ptr_out) {
  if (device < 0 || device >= kStaticMaxDevices) return fail(WS_ERR_INVALID_ARG, "device %d out of range", device);
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_scratch_ptr[device]) {
    int prev = -1;
    WS_CUDA(cudaGetDevice(&prev));
    if (prev != device) WS_CUDA(cudaSetDevice(device));
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_part_scratch);
    if (prev != device) (void)cudaSetDevice(prev);
    if (e != cudaSuccess || !ptr)
      return fail(WS_ERR_CUDA, "cudaGetSymbolAddress(static split-KV scratch) on device %d: %s", device,
                  cudaGetErrorString(e));
    g_static_scratch_ptr[device] = ptr;
  }
  if (ptr_out) *ptr_out = g_static_scratch_ptr[device];
  return WS_OK;
}

}  // namespace

extern "C" {

ws_status_t ws_static_scratch_setup(int32_t device) { return static_scratch_ensure(device, nullptr); }

ws_status_t ws_block_causal_attn_fwd_static(ws_cache_t* c, int32_t S, const int32_t* session_ids,
                                            const int32_t* num_q_blocks, const int32_t* cu, const void* q,
                                            void* out, float* lse, float scale, void* cuda_stream) {
  ws_status_t st = attn_validate_args(c, S, session_ids, cu, q, out, scale);
  if (st != WS_OK) return st;
  if (c->dry) return fail(WS_ERR_INVALID_ARG, "ws_block_causal_attn_fwd_static needs a device cache (not WS_FLAG_DRY_RUN)");
  if (c->cfg.flags & WS_FLAG_FUSED_COMBINE)
    return fail(WS_ERR_UNSUPPORTED, "ws_block_causal_attn_fwd_static: not with WS_FLAG_FUSED_COMBINE (its counters live in the workspace)");
  DeviceGuard dg(c);
  void* scratch = nullptr;
  st = static_scratch_ensure(c->cfg.device, &scratch);
  if (st != WS_OK) return st;
  // The same host path and the same kernels as ws_block_causal_attn_fwd; for the duration of this call the
  // cache's partial-slot views point into the static array and the planner's slot budget is the array's.
  float* const save_o = c->d_part_o;
  float* const save_lse = c->d_part_lse;
  const int32_t save_slots = c->lay.max_part_slots;
  c->d_part_o = reinterpret_cast<float*>(scratch);
  c->d_part_lse = reinterpret_cast<float*>(static_cast<unsigned char*>(scratch) + kStaticPartOBytes);
  c->lay.max_part_slots = std::min<int32_t>(save_slots, WS_STATIC_PART_SLOTS);
  st = attn_impl(c, S, session_ids, num_q_blocks, cu, q, out, lse, scale, (cudaStream_t)cuda_stream, nullptr);
  c->d_part_o = save_o; c->d_part_lse = save_lse; c->lay.max_part_slots = save_slots;
  if (st == WS_ERR_WORKSPACE_TOO_SMALL) {
    return fail(WS_ERR_WORKSPACE_TOO_SMALL,
                "ws_block_causal_attn_fwd_static: the split-KV plan of this call needs more than the %d partial slots "
                "(%zu bytes) of the library's static scratch; nothing was launched - use ws_block_causal_attn_fwd "
                "with a workspace", (int)WS_STATIC_PART_SLOTS, kStaticPartOBytes + kStaticPartLseBytes);
  }
  return st;
}

ws_status_t ws_kv_append(ws_cache_t* c, int32_t S, const int32_t* session_ids,
                         const int32_t* cu, const void* k_new, const void* v_new,
                         const uint8_t* modality, void* cuda_stream) {
  size_t words = 0;
  ws_status_t st = append_validate(c, S, session_ids, cu, k_new, v_new, &words);
  if (st != WS_OK) return st;
  DeviceGuard dg(c);
  AppendPrep ap;
  st = append_commit(c, S, session_ids, cu, modality, words, (cudaStream_t)cuda_stream, &ap);
  if (st != WS_OK) return st;
  return append_launch(c, ap, k_new, v_new, cu[S], (cudaStream_t)cuda_stream);
}

ws_status_t ws_kv_append_blocks(ws_cache_t* c, int32_t S, const int32_t* session_ids, const int32_t* cu,
                                const int32_t* cu_blocks, const int32_t* block_tokens, const void* k_new,
                                const void* v_new, const uint8_t* modality, void* cuda_stream) {
  if (!cu_blocks || !block_tokens) return fail(WS_ERR_INVALID_ARG, "cu_blocks / block_tokens is NULL");
  size_t words = 0;
  ws_status_t st = append_validate(c, S, session_ids, cu, k_new, v_new, &words, cu_blocks, block_tokens);
  if (st != WS_OK) return st;
  DeviceGuard dg(c);
  AppendPrep ap;
  st = append_commit(c, S, session_ids, cu, modality, words, (cudaStream_t)cuda_stream, &ap, cu_blocks, block_tokens);
  if (st != WS_OK) return st;
  return append_launch(c, ap, k_new, v_new, cu[S], (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------------------ a3 + a4
ws_status_t ws_block_causal_attn_fwd(ws_cache_t* c, int32_t S, const int32_t* session_ids,
                                     const int32_t* num_q_blocks, const int32_t* cu, const void* q,
                                     void* out, float* lse, float scale, void* cuda_stream) {
  ws_status_t st = attn_validate_args(c, S, session_ids, cu, q, out, scale);
  if (st != WS_OK) return st;
  DeviceGuard dg(c);
  return attn_impl(c, S, session_ids, num_q_blocks, cu, q, out, lse, scale, (cudaStream_t)cuda_stream, nullptr);
}

ws_status_t ws_block_causal_attn_fwd_masked(ws_cache_t* c, int32_t S, const int32_t* session_ids,
                                            const int32_t* num_q_blocks, const int32_t* cu, const void* q,
                                            void* out, float* lse, float scale, uint32_t attn_flags,
                                            void* cuda_stream) {
  ws_status_t st = attn_validate_args(c, S, session_ids, cu, q, out, scale);
  if (st != WS_OK) return st;
  DeviceGuard dg(c);
  return attn_impl(c, S, session_ids, num_q_blocks, cu, q, out, lse, scale, (cudaStream_t)cuda_stream, nullptr,
                   attn_flags);
}

ws_status_t ws_stream_step(ws_cache_t* c, int32_t S, const int32_t* session_ids, const int32_t* cu,
                           const void* q, const void* k_new, const void* v_new, void* out, float* lse,
                           float scale, void* cuda_stream) {
  return ws_stream_step_tagged(c, S, session_ids, cu, q, k_new, v_new, nullptr, 0u, out, lse, scale, cuda_stream);
}

ws_status_t ws_stream_step_tagged(ws_cache_t* c, int32_t S, const int32_t* session_ids, const int32_t* cu,
                                  const void* q, const void* k_new, const void* v_new, const uint8_t* modality,
                                  uint32_t attn_flags, void* out, float* lse, float scale, void* cuda_stream) {
  if (attn_flags & ~(uint32_t)WS_ATTN_TEXT_CAUSAL) return fail(WS_ERR_INVALID_ARG, "unknown attn_flags 0x%x", attn_flags);
  if ((attn_flags & WS_ATTN_TEXT_CAUSAL) && !modality)
    return fail(WS_ERR_INVALID_ARG, "WS_ATTN_TEXT_CAUSAL needs the block's modality tags");
  if (modality && c && cu && S >= 1 && cu[0] == 0)
    for (int32_t t = 0; t < cu[S]; ++t)
      if (modality[t] > 2) return fail(WS_ERR_INVALID_ARG, "modality[%d] = %d (0 video, 1 audio, 2 text)", t, modality[t]);
  // validate what only the second half would reject BEFORE the append commits anything
  ws_status_t st = attn_validate_args(c, S, session_ids, cu, q, out, scale);
  if (st != WS_OK) return st;
  size_t words = 0;
  st = append_validate(c, S, session_ids, cu, k_new, v_new, &words);
  if (st != WS_OK) return st;
  DeviceGuard dg(c);
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  AppendPrep ap;
  st = append_commit(c, S, session_ids, cu, modality, words, stream, &ap);
  if (st != WS_OK) return st;
  // One launch commits and attends when the tcgen05 kernel runs and the append descriptor fits the kernel
  // parameters (up to ~900 new pages per call); otherwise: the append kernel, then attention over the pool.
  const bool tensor = c->tensor_path_ok && !(c->cfg.flags & WS_FLAG_FORCE_SIMT);
  // (generic kernel: also one launch, when its per-token metadata fits the kernel parameters too and no replica
  // is linked - the generic path does not mirror)
  const bool simt_fusable = !tensor && !c->dry && c->peers.n == 0 &&
                            (size_t)cu[S] * ((attn_flags & WS_ATTN_TEXT_CAUSAL) ? 7 : 4) + 64 <= (size_t)ws::kInlineAppendWords;
  if ((tensor || simt_fusable) && ap.inline_meta && !(c->cfg.flags & WS_FLAG_SEPARATE_APPEND)) {
    const FusedAppend fuse{&ap, k_new, v_new};
    return attn_impl(c, S, session_ids, nullptr, cu, q, out, lse, scale, stream, &fuse, attn_flags);
  }
  st = append_launch(c, ap, k_new, v_new, cu[S], stream);
  if (st != WS_OK) return st;
  return attn_impl(c, S, session_ids, nullptr, cu, q, out, lse, scale, stream, nullptr, attn_flags);
}

size_t ws_step_staging_bytes(const ws_cache_config_t* cfg, int32_t n) {
  const char* why;
  if (!config_valid(cfg, &why) || n < 1) return 0;
  size_t eb = eb_of(cfg->dtype), D = cfg->head_dim;
  size_t qb = align_up((size_t)n * cfg->num_q_heads * D * eb, 256);
  size_t kb = align_up((size_t)n * cfg->num_kv_heads * D * eb, 256);
  return 2 * (2 * qb + 2 * kb);          // two slots of {q, out, k_new, v_new}
}

ws_status_t ws_stream_step_host(ws_cache_t* c, int32_t S, const int32_t* session_ids,
                                const int32_t* cu, const void* q_host, const void* k_host,
                                const void* v_host, void* out_host, void* staging,
                                size_t staging_bytes, float scale, void* cuda_stream) {
  if (!c || !session_ids || !cu || !q_host || !k_host || !v_host || !out_host || !staging)
    return fail(WS_ERR_INVALID_ARG, "NULL argument");
  if (c->dry) return fail(WS_ERR_CUDA, "ws_stream_step_host needs a CUDA device (dry-run cache)");
  if (S < 1 || cu[0] != 0 || cu[S] < 1) return fail(WS_ERR_INVALID_ARG, "bad cu_new_tokens");
  const int32_t n = cu[S];
  if (staging_bytes < ws_step_staging_bytes(&c->cfg, n))
    return fail(WS_ERR_WORKSPACE_TOO_SMALL, "staging_bytes %zu < required %zu", staging_bytes,
                ws_step_staging_bytes(&c->cfg, n));
  // everything the step would reject is rejected before the first copy is enqueued
  ws_status_t st = attn_validate_args(c, S, session_ids, cu, q_host, out_host, scale);
  if (st != WS_OK) return st;
  size_t words = 0;
  st = append_validate(c, S, session_ids, cu, k_host, v_host, &words);
  if (st != WS_OK) return st;
  DeviceGuard dg(c);
  if (!c->h2d_stream) {
    WS_CUDA(cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking));
    WS_CUDA(cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      WS_CUDA(cudaEventCreateWithFlags(&c->ev_h2d[i], cudaEventDisableTiming));
      WS_CUDA(cudaEventCreateWithFlags(&c->ev_compute[i], cudaEventDisableTiming));
      WS_CUDA(cudaEventCreateWithFlags(&c->ev_d2h[i], cudaEventDisableTiming));
    }
  }
  size_t eb = eb_of(c->cfg.dtype), D = c->cfg.head_dim;
  size_t q_bytes = (size_t)n * c->cfg.num_q_heads * D * eb, kv_bytes = (size_t)n * c->cfg.num_kv_heads * D * eb;
  size_t qb = align_up(q_bytes, 256), kb = align_up(kv_bytes, 256);
  const int slot = (int)(c->host_steps & 1);
  // Fixed slot stride (half of the caller's buffer, 256-byte aligned): steps with different token counts
  // must not place slot 1 inside the region slot 0 of the previous, larger step is still using.
  const size_t slot_stride = (staging_bytes / 2) & ~(size_t)255;
  char* base = (char*)staging + (size_t)slot * slot_stride;
  char *dq = base, *dout = base + qb, *dk = base + 2 * qb, *dv = base + 2 * qb + kb;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  // copy-in on the H2D stream (after the slot's previous result has left the device), compute on the
  // caller's stream, copy-out on the D2H stream: step t's copies overlap step t-1 / t+1's kernels
  if (c->slot_used[slot]) WS_CUDA(cudaStreamWaitEvent(c->h2d_stream, c->ev_d2h[slot], 0));
  WS_CUDA(cudaMemcpyAsync(dk, k_host, kv_bytes, cudaMemcpyHostToDevice, c->h2d_stream));
  WS_CUDA(cudaMemcpyAsync(dv, v_host, kv_bytes, cudaMemcpyHostToDevice, c->h2d_stream));
  WS_CUDA(cudaMemcpyAsync(dq, q_host, q_bytes, cudaMemcpyHostToDevice, c->h2d_stream));
  WS_CUDA(cudaEventRecord(c->ev_h2d[slot], c->h2d_stream));
  WS_CUDA(cudaStreamWaitEvent(stream, c->ev_h2d[slot], 0));
  st = ws_stream_step(c, S, session_ids, cu, dq, dk, dv, dout, nullptr, scale, cuda_stream);
  if (st != WS_OK) return st;
  WS_CUDA(cudaEventRecord(c->ev_compute[slot], stream));
  WS_CUDA(cudaStreamWaitEvent(c->d2h_stream, c->ev_compute[slot], 0));
  WS_CUDA(cudaMemcpyAsync(out_host, dout, q_bytes, cudaMemcpyDeviceToHost, c->d2h_stream));
  WS_CUDA(cudaEventRecord(c->ev_d2h[slot], c->d2h_stream));
  c->slot_used[slot] = true;
  c->host_steps += 1;
  return WS_OK;
}

ws_status_t ws_stream_host_join(ws_cache_t* c, void* cuda_stream) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (c->dry) return WS_OK;
  for (int i = 0; i < 2; ++i)
    if (c->slot_used[i]) WS_CUDA(cudaStreamWaitEvent((cudaStream_t)cuda_stream, c->ev_d2h[i], 0));
  return WS_OK;
}

ws_status_t ws_fm_euler_update(int32_t dtype, void* z, const void* v, float dtau, int64_t count,
                               void* cuda_stream) {
  if (dtype != WS_BF16 && dtype != WS_F32) return fail(WS_ERR_INVALID_ARG, "dtype");
  if (count < 0 || (count > 0 && (!z || !v))) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  if (((uintptr_t)z & 15) || ((uintptr_t)v & 15)) return fail(WS_ERR_INVALID_ARG, "z / v must be 16-byte aligned");
  if (!std::isfinite(dtau)) return fail(WS_ERR_INVALID_ARG, "dtau must be finite");
  WS_CUDA(ws::launch_fm_euler(dtype, z, v, dtau, count, (cudaStream_t)cuda_stream));
  return WS_OK;
}

// ------------------------------------------------------------------------------------ NEXT-3
ws_status_t ws_replica_link(ws_cache_t* c, const ws_peer_pools_t* peers, int32_t num_peers) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (num_peers < 0 || num_peers > WS_MAX_PEERS || (num_peers > 0 && !peers))
    return fail(WS_ERR_INVALID_ARG, "num_peers %d not in [0, %d]", num_peers, (int)WS_MAX_PEERS);
  ws::PeerPools pp{};
  for (int32_t r = 0; r < num_peers; ++r) {
    if (!c->dry) {
      if (!peers[r].k_pool || !peers[r].v_pool) return fail(WS_ERR_INVALID_ARG, "peer %d: NULL pool", r);
      if (((uintptr_t)peers[r].k_pool & 15) || ((uintptr_t)peers[r].v_pool & 15))
        return fail(WS_ERR_INVALID_ARG, "peer %d: pools must be 16-byte aligned", r);
      if (peers[r].k_pool == c->cfg.k_pool || peers[r].v_pool == c->cfg.v_pool)
        return fail(WS_ERR_INVALID_ARG, "peer %d is the cache's own pool", r);
    }
    if (peers[r].pool_bytes < ws_pool_bytes(&c->cfg))
      return fail(WS_ERR_INVALID_ARG, "peer %d: pool_bytes %zu < the owner's %zu", r, peers[r].pool_bytes,
                  ws_pool_bytes(&c->cfg));
    pp.k[r] = peers[r].k_pool; pp.v[r] = peers[r].v_pool;
  }
  pp.n = num_peers;
  c->peers = pp;
  return WS_OK;
}

ws_status_t ws_replica_accept(ws_cache_t* c, int32_t owner_pages) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (owner_pages < 0 || owner_pages > c->cfg.num_pages)
    return fail(WS_ERR_INVALID_ARG, "owner_pages %d not in [0, %d]", owner_pages, c->cfg.num_pages);
  if (!c->host->reserve_owner_pages(owner_pages))
    return fail(WS_ERR_INVALID_ARG, "ws_replica_accept needs every session closed");
  return WS_OK;
}

ws_status_t ws_replica_commit_message(const ws_cache_t* c, int32_t* words, int32_t cap, int32_t* n) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  return copy_message(c->last_commit, words, cap, n);
}

ws_status_t ws_replica_snapshot_message(const ws_cache_t* c, int32_t session, int32_t* words,
                                        int32_t cap, int32_t* n) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (!c->host->is_open(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  const ws::SessionState& ss = c->host->session(session);
  if (ss.block_ends.empty()) return fail(WS_ERR_INVALID_ARG, "session %d has no committed block", session);
  std::vector<int32_t> msg;
  msg_begin(c, msg, kMsgSnapshot, 1);
  msg.insert(msg.end(), {session, 0, (int32_t)ss.block_ends.size(), (int32_t)ss.pages.size()});
  int64_t prev = 0;
  for (int64_t e : ss.block_ends) { msg.push_back((int32_t)(e - prev)); prev = e; }
  msg.insert(msg.end(), ss.pages.begin(), ss.pages.end());
  msg[kMsgTotalWord] = (int32_t)msg.size();
  return copy_message(msg, words, cap, n);
}

ws_status_t ws_replica_push_session(ws_cache_t* c, int32_t session, void* cuda_stream) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  DeviceGuard dg(c);
  if (!c->host->is_open(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  if (c->peers.n == 0) return fail(WS_ERR_INVALID_ARG, "no replica is linked (ws_replica_link)");
  const ws::SessionState& ss = c->host->session(session);
  if (c->dry || ss.pages.empty()) return WS_OK;
  const int64_t page_bytes = (int64_t)c->cfg.num_kv_heads * c->cfg.page_tokens * c->cfg.head_dim * eb_of(c->cfg.dtype);
  WS_CUDA(ws::launch_kv_push_pages(c->cfg.k_pool, c->cfg.v_pool, c->peers,
                                   c->d_page_table + (int64_t)session * c->cfg.max_pages_per_session,
                                   (int32_t)ss.pages.size(), page_bytes, c->num_sms, (cudaStream_t)cuda_stream));
  c->launches += 1;
  return WS_OK;
}

ws_status_t ws_replica_apply(ws_cache_t* c, const int32_t* w, int32_t n, void* cuda_stream) {
  if (!c || !w) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  DeviceGuard dg(c);
  if (n < kMsgHeaderWords || w[0] != kMsgMagic) return fail(WS_ERR_INVALID_ARG, "not a commit message");
  if (w[1] != kMsgVersion) return fail(WS_ERR_UNSUPPORTED, "message version %d (this library: %d)", w[1], kMsgVersion);
  if (w[2] != kMsgCommit && w[2] != kMsgSnapshot) return fail(WS_ERR_INVALID_ARG, "unknown message kind %d", w[2]);
  if (w[kMsgTotalWord] != n) return fail(WS_ERR_INVALID_ARG, "message says %d words, %d given", w[kMsgTotalWord], n);
  if (w[5] != c->cfg.page_tokens || w[6] != c->cfg.num_kv_heads || w[7] != c->cfg.head_dim || w[8] != c->cfg.dtype)
    return fail(WS_ERR_INVALID_ARG, "message geometry (P %d, Hkv %d, D %d, dtype %d) differs from this cache",
                w[5], w[6], w[7], w[8]);
  const int32_t S = w[3], P = c->cfg.page_tokens;
  if (S < 1 || S > c->cfg.max_sessions) return fail(WS_ERR_INVALID_ARG, "message lists %d sessions", S);
  // ---- pass 1: validate everything (no state changes)
  struct Item { int32_t id, len_old, nblocks, npages; const int32_t* lens; const int32_t* pages; };
  std::vector<Item> items;
  std::vector<int32_t> seen_pages;
  int32_t pos = kMsgHeaderWords;
  for (int32_t s = 0; s < S; ++s) {
    if (pos + 4 > n) return fail(WS_ERR_INVALID_ARG, "message truncated (session %d header)", s);
    Item it{w[pos], w[pos + 1], w[pos + 2], w[pos + 3], nullptr, nullptr};
    pos += 4;
    if (it.nblocks < 1 || it.npages < 0 || it.len_old < 0 || (int64_t)pos + it.nblocks + it.npages > n)
      return fail(WS_ERR_INVALID_ARG, "message truncated or malformed (session %d)", s);
    it.lens = w + pos; it.pages = w + pos + it.nblocks;
    pos += it.nblocks + it.npages;
    if (it.id < 0 || it.id >= c->cfg.max_sessions) return fail(WS_ERR_BAD_SESSION, "session %d out of range", it.id);
    for (const Item& o : items) if (o.id == it.id) return fail(WS_ERR_INVALID_ARG, "session %d listed twice", it.id);
    int64_t have = 0, blocks = 0;
    if (c->host->is_open(it.id)) {
      have = c->host->session(it.id).tokens; blocks = (int64_t)c->host->session(it.id).block_ends.size();
    }
    if (have != it.len_old)
      return fail(WS_ERR_INVALID_ARG, "session %d: replica holds %lld tokens, message continues from %d "
                  "(a staged block must be rolled back first)", it.id, (long long)have, it.len_old);
    int64_t total = it.len_old;
    for (int32_t b = 0; b < it.nblocks; ++b) {
      if (it.lens[b] < 1) return fail(WS_ERR_INVALID_ARG, "session %d: block of %d tokens", it.id, it.lens[b]);
      total += it.lens[b];
    }
    if (total >= (1ll << 31)) return fail(WS_ERR_UNSUPPORTED, "session %d would exceed 2^31 tokens", it.id);
    const int64_t need = (total + P - 1) / P, had = ((int64_t)it.len_old + P - 1) / P;
    if (need - had != it.npages)
      return fail(WS_ERR_INVALID_ARG, "session %d: %d pages named, %lld needed", it.id, it.npages, (long long)(need - had));
    if (need > c->cfg.max_pages_per_session || blocks + it.nblocks > c->cfg.max_blocks_per_session)
      return fail(WS_ERR_OUT_OF_PAGES, "session %d exceeds its page-table or block capacity", it.id);
    for (int32_t i = 0; i < it.npages; ++i) {
      if (!c->host->owner_page_free(it.pages[i]))
        return fail(WS_ERR_OUT_OF_PAGES, "page %d is not a free owner page of this replica (ws_replica_accept: %d)",
                    it.pages[i], c->host->owner_pages());
      for (int32_t q : seen_pages) if (q == it.pages[i]) return fail(WS_ERR_INVALID_ARG, "page %d named twice", q);
      seen_pages.push_back(it.pages[i]);
    }
    items.push_back(it);
  }
  if (pos != n) return fail(WS_ERR_INVALID_ARG, "message has %d trailing words", n - pos);
  // ---- pass 2: adopt
  for (const Item& it : items) {
    if (!c->host->is_open(it.id)) c->host->open_session_at(it.id);
    const int32_t first = (int32_t)c->host->session(it.id).pages.size();
    c->host->adopt(it.id, it.lens, it.nblocks, it.pages, it.npages);
    if (!c->dry && it.npages > 0) {
      WS_CUDA(ws::launch_page_table_publish(c->d_page_table, it.pages, it.id, first, it.npages,
                                            c->cfg.max_pages_per_session, (cudaStream_t)cuda_stream));
      c->launches += (it.npages + ws::kInlineAppendWords - 1) / ws::kInlineAppendWords;
    }
  }
  return WS_OK;
}

ws_status_t ws_ipc_export(const void* device_ptr, uint8_t* handle64, uint64_t* offset) {
  if (!device_ptr || !handle64 || !offset) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
  typedef CUresult (*RangeFn)(CUdeviceptr*, size_t*, CUdeviceptr);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  WS_CUDA(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qres));
  if (!fn || qres != cudaDriverEntryPointSuccess) return fail(WS_ERR_CUDA, "cuMemGetAddressRange entry point not found");
  CUdeviceptr base = 0; size_t size = 0;
  CUresult r = ((RangeFn)fn)(&base, &size, (CUdeviceptr)(uintptr_t)device_ptr);
  if (r != CUDA_SUCCESS) return fail(WS_ERR_CUDA, "cuMemGetAddressRange failed (%d)", (int)r);
  cudaIpcMemHandle_t h;
  WS_CUDA(cudaIpcGetMemHandle(&h, (void*)(uintptr_t)base));
  memcpy(handle64, &h, 64);
  *offset = (uint64_t)((uintptr_t)device_ptr - (uintptr_t)base);
  return WS_OK;
}

ws_status_t ws_ipc_open(const uint8_t* handle64, uint64_t offset, int32_t device, void** ptr_out) {
  if (!handle64 || !ptr_out) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  cudaIpcMemHandle_t h;
  memcpy(&h, handle64, 64);
  WS_CUDA(cudaSetDevice(device));
  void* p = nullptr;
  WS_CUDA(cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
  *ptr_out = (char*)p + offset;
  return WS_OK;
}

ws_status_t ws_ipc_close(void* ptr, uint64_t offset) {
  if (!ptr) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  WS_CUDA(cudaIpcCloseMemHandle((char*)ptr - offset));
  return WS_OK;
}

ws_status_t ws_kv_gather(const ws_cache_t* c, int32_t session, int64_t start, int64_t count,
                         void* k_out, void* v_out, void* cuda_stream) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  DeviceGuard dg(c);
  if (!c->host->is_open(session)) return fail(WS_ERR_BAD_SESSION, "session %d is not open", session);
  const ws::SessionState& ss = c->host->session(session);
  if (start < 0 || count < 0 || start + count > ss.tokens)
    return fail(WS_ERR_INVALID_ARG, "range [%lld, %lld) outside the %lld committed tokens",
                (long long)start, (long long)(start + count), (long long)ss.tokens);
  if (c->dry || count == 0) return WS_OK;
  WS_CUDA(ws::launch_kv_gather(c->cfg.k_pool, c->cfg.v_pool, k_out, v_out,
                               c->d_page_table + (int64_t)session * c->cfg.max_pages_per_session,
                               start, count, c->cfg.page_tokens, c->cfg.num_kv_heads, c->cfg.head_dim,
                               eb_of(c->cfg.dtype), c->num_sms, (cudaStream_t)cuda_stream));
  const_cast<ws_cache*>(c)->launches += 1;
  return WS_OK;
}

ws_status_t ws_last_plan_info(const ws_cache_t* c, ws_plan_info_t* out) {
  if (!c || !out) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  const ws::Plan& p = c->last_plan;
  out->num_ctas = p.num_teams * p.team_size;
  out->team_size = p.team_size;
  out->num_groups = (int32_t)p.groups.size();
  out->num_segments = (int32_t)p.segments.size();
  out->num_partial_slots = p.num_part_slots;
  out->num_combine_items = (int32_t)p.combine.size();
  out->used_tensor_core_kernel = c->last_tensor ? (p.alt ? 3 : 1) : 0;
  out->total_kv_tiles = p.total_tiles;
  return WS_OK;
}

ws_status_t ws_last_plan_segment(const ws_cache_t* c, int32_t i, ws_plan_segment_t* out) {
  if (!c || !out) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  const ws::Plan& p = c->last_plan;
  if (i < 0 || i >= (int32_t)p.segments.size()) return fail(WS_ERR_INVALID_ARG, "segment %d out of range", i);
  const ws::Segment& s = p.segments[i];
  const ws::Group& g = p.groups[s.group];
  *out = ws_plan_segment_t{s.group, g.slot, g.kv_head, g.q_token0, s.tile_begin, s.tile_end,
                           p.seg_team[i], s.part_base};
  return WS_OK;
}

int64_t ws_launch_count(const ws_cache_t* c) { return c ? c->launches : -1; }

ws_status_t ws_debug_kernel_timing(ws_cache_t* c, int32_t enable) {
  if (!c) return fail(WS_ERR_INVALID_ARG, "cache is NULL");
  if (c->dry) return fail(WS_ERR_CUDA, "kernel timing needs a CUDA device");
  c->timing = enable != 0;
  return WS_OK;
}

ws_status_t ws_debug_read_kernel_times(ws_cache_t* c, double* ms_sum3, int32_t* count3) {
  if (!c || !ms_sum3 || !count3) return fail(WS_ERR_INVALID_ARG, "NULL argument");
  DeviceGuard dg(c);
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>>* lists[3] = {&c->t_append, &c->t_attn, &c->t_combine};
  for (int k = 0; k < 3; ++k) {
    ms_sum3[k] = 0.0; count3[k] = (int32_t)lists[k]->size();
    for (auto& pr : *lists[k]) {
      WS_CUDA(cudaEventSynchronize(pr.second));
      float ms = 0.f;
      WS_CUDA(cudaEventElapsedTime(&ms, pr.first, pr.second));
      ms_sum3[k] += ms;
      c->ev_pool.push_back(pr.first); c->ev_pool.push_back(pr.second);
    }
    lists[k]->clear();
  }
  return WS_OK;
}

const char* ws_status_str(ws_status_t s) {
  switch (s) {
    case WS_OK: return "WS_OK";
    case WS_ERR_INVALID_ARG: return "WS_ERR_INVALID_ARG";
    case WS_ERR_BAD_SESSION: return "WS_ERR_BAD_SESSION";
    case WS_ERR_OUT_OF_PAGES: return "WS_ERR_OUT_OF_PAGES";
    case WS_ERR_UNSUPPORTED: return "WS_ERR_UNSUPPORTED";
    case WS_ERR_WORKSPACE_TOO_SMALL: return "WS_ERR_WORKSPACE_TOO_SMALL";
    case WS_ERR_CUDA: return "WS_ERR_CUDA";
  }
  return "WS_ERR_?";
}

const char* ws_last_error(void) { return g_err.c_str(); }
const char* ws_version(void) { return "wanstream-b200 0.1 (sm_100a)"; }

}  // extern "C"

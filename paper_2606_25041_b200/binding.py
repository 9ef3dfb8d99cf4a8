"""Thin ctypes binding of libwanstream.so (include/ws.h).  Argument marshalling only.

Every step of the hot path (KV append, block-causal attention, split-KV combine) runs in the CUDA
kernels behind the C ABI; this module converts Python/torch arguments to pointers and sizes and
raises `WsError` on any non-zero status.  torch is used for device memory and streams only.
There is NO fallback: if the shared library is missing, importing the functions raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libwanstream.so")

WS_BF16, WS_F32 = 0, 1
WS_FLAG_DRY_RUN, WS_FLAG_FORCE_SIMT, WS_FLAG_FUSED_COMBINE, WS_FLAG_SEPARATE_APPEND = 1, 2, 8, 16
WS_ATTN_TEXT_CAUSAL = 1
STATUS_NAMES = ["WS_OK", "WS_ERR_INVALID_ARG", "WS_ERR_BAD_SESSION", "WS_ERR_OUT_OF_PAGES",
                "WS_ERR_UNSUPPORTED", "WS_ERR_WORKSPACE_TOO_SMALL", "WS_ERR_CUDA"]


class WsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {message}")
        self.status = status
        self.status_name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)


class CacheConfig(C.Structure):
    _fields_ = [("dtype", C.c_int32), ("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("q_to_kv_head", C.POINTER(C.c_int32)),
                ("page_tokens", C.c_int32), ("num_pages", C.c_int32), ("max_sessions", C.c_int32),
                ("max_pages_per_session", C.c_int32), ("max_blocks_per_session", C.c_int32),
                ("max_sessions_per_call", C.c_int32), ("max_q_tokens_per_call", C.c_int32),
                ("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("pool_bytes", C.c_size_t),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("device", C.c_int32), ("flags", C.c_uint32)]


class PlanInfo(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("num_ctas", "team_size", "num_groups", "num_segments",
                                         "num_partial_slots", "num_combine_items",
                                         "used_tensor_core_kernel", "total_kv_tiles")]


class PlanSegment(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("group", "session", "kv_head", "q_token0", "tile_begin",
                                         "tile_end", "team", "part_base")]


class PeerPools(C.Structure):
    _fields_ = [("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("pool_bytes", C.c_size_t)]


EXPORTS = ["ws_replica_link", "ws_replica_accept", "ws_replica_commit_message",
           "ws_replica_snapshot_message", "ws_replica_push_session", "ws_replica_apply",
           "ws_ipc_export", "ws_ipc_open", "ws_ipc_close", "ws_pool_bytes", "ws_workspace_bytes", "ws_cache_create", "ws_cache_destroy",
           "ws_session_open", "ws_session_close", "ws_session_info", "ws_session_truncate",
           "ws_free_pages", "ws_kv_append", "ws_kv_append_blocks", "ws_block_causal_attn_fwd", "ws_step_staging_bytes",
           "ws_stream_step", "ws_stream_step_tagged", "ws_block_causal_attn_fwd_masked", "ws_stream_step_host", "ws_stream_host_join", "ws_fm_euler_update", "ws_kv_gather", "ws_session_pages", "ws_debug_shuffle_free_pages",
           "ws_debug_set_min_splits", "ws_debug_set_decode_plan", "ws_static_scratch_setup",
           "ws_block_causal_attn_fwd_static", "ws_last_plan_info", "ws_last_plan_segment",
           "ws_launch_count", "ws_debug_kernel_timing", "ws_debug_read_kernel_times",
           "ws_status_str", "ws_last_error", "ws_version"]

_lib = None


def load_library() -> C.CDLL:
    """Load libwanstream.so; raises (never falls back) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2606_25041_b200.build` "
                          "(there is no CPU or PyTorch fallback for this path)")
    lib = C.CDLL(LIB_PATH)
    i32p, vp = C.POINTER(C.c_int32), C.c_void_p
    cfgp = C.POINTER(CacheConfig)
    lib.ws_pool_bytes.restype = C.c_size_t; lib.ws_pool_bytes.argtypes = [cfgp]
    lib.ws_workspace_bytes.restype = C.c_size_t; lib.ws_workspace_bytes.argtypes = [cfgp]
    lib.ws_cache_create.argtypes = [cfgp, C.POINTER(vp)]
    lib.ws_cache_destroy.argtypes = [vp]
    lib.ws_session_open.argtypes = [vp, i32p]
    lib.ws_session_close.argtypes = [vp, C.c_int32]
    lib.ws_session_info.argtypes = [vp, C.c_int32, C.POINTER(C.c_int64), i32p,
                                    C.POINTER(C.POINTER(C.c_int64))]
    lib.ws_session_truncate.argtypes = [vp, C.c_int32, C.c_int32]
    lib.ws_free_pages.argtypes = [vp]; lib.ws_free_pages.restype = C.c_int32
    lib.ws_kv_append.argtypes = [vp, C.c_int32, i32p, i32p, vp, vp, C.POINTER(C.c_uint8), vp]
    lib.ws_kv_append_blocks.argtypes = [vp, C.c_int32, i32p, i32p, i32p, i32p, vp, vp, C.POINTER(C.c_uint8), vp]
    lib.ws_block_causal_attn_fwd.argtypes = [vp, C.c_int32, i32p, i32p, i32p, vp, vp, vp,
                                             C.c_float, vp]
    lib.ws_block_causal_attn_fwd_static.argtypes = [vp, C.c_int32, i32p, i32p, i32p, vp, vp, vp,
                                                    C.c_float, vp]
    lib.ws_static_scratch_setup.argtypes = [C.c_int32]
    lib.ws_block_causal_attn_fwd_masked.argtypes = [vp, C.c_int32, i32p, i32p, i32p, vp, vp, vp,
                                                    C.c_float, C.c_uint32, vp]
    lib.ws_stream_step_tagged.argtypes = [vp, C.c_int32, i32p, i32p, vp, vp, vp, C.POINTER(C.c_uint8),
                                          C.c_uint32, vp, vp, C.c_float, vp]
    lib.ws_step_staging_bytes.restype = C.c_size_t
    lib.ws_step_staging_bytes.argtypes = [cfgp, C.c_int32]
    lib.ws_stream_step.argtypes = [vp, C.c_int32, i32p, i32p, vp, vp, vp, vp, vp, C.c_float, vp]
    lib.ws_stream_step_host.argtypes = [vp, C.c_int32, i32p, i32p, vp, vp, vp, vp, vp, C.c_size_t,
                                        C.c_float, vp]
    lib.ws_stream_host_join.argtypes = [vp, vp]
    lib.ws_fm_euler_update.argtypes = [C.c_int32, vp, vp, C.c_float, C.c_int64, vp]
    lib.ws_kv_gather.argtypes = [vp, C.c_int32, C.c_int64, C.c_int64, vp, vp, vp]
    lib.ws_replica_link.argtypes = [vp, C.POINTER(PeerPools), C.c_int32]
    lib.ws_replica_accept.argtypes = [vp, C.c_int32]
    lib.ws_replica_commit_message.argtypes = [vp, i32p, C.c_int32, i32p]
    lib.ws_replica_snapshot_message.argtypes = [vp, C.c_int32, i32p, C.c_int32, i32p]
    lib.ws_replica_push_session.argtypes = [vp, C.c_int32, vp]
    lib.ws_replica_apply.argtypes = [vp, i32p, C.c_int32, vp]
    lib.ws_ipc_export.argtypes = [vp, C.POINTER(C.c_uint8), C.POINTER(C.c_uint64)]
    lib.ws_ipc_open.argtypes = [C.POINTER(C.c_uint8), C.c_uint64, C.c_int32, C.POINTER(vp)]
    lib.ws_ipc_close.argtypes = [vp, C.c_uint64]
    lib.ws_session_pages.argtypes = [vp, C.c_int32, i32p, C.c_int32, i32p]
    lib.ws_debug_shuffle_free_pages.argtypes = [vp, C.c_uint64]
    lib.ws_debug_set_min_splits.argtypes = [vp, C.c_int32]
    lib.ws_debug_set_decode_plan.argtypes = [vp, C.c_int32]
    lib.ws_last_plan_info.argtypes = [vp, C.POINTER(PlanInfo)]
    lib.ws_last_plan_segment.argtypes = [vp, C.c_int32, C.POINTER(PlanSegment)]
    lib.ws_launch_count.argtypes = [vp]; lib.ws_launch_count.restype = C.c_int64
    lib.ws_debug_kernel_timing.argtypes = [vp, C.c_int32]
    lib.ws_debug_read_kernel_times.argtypes = [vp, C.POINTER(C.c_double), i32p]
    lib.ws_status_str.argtypes = [C.c_int]; lib.ws_status_str.restype = C.c_char_p
    lib.ws_last_error.restype = C.c_char_p
    lib.ws_version.restype = C.c_char_p
    _lib = lib
    return lib


def _check(status: int) -> None:
    if status != 0:
        raise WsError(status, load_library().ws_last_error().decode())


def _i32(seq) -> "C.Array":
    """HOST int32 array argument.  (Plain lists / tuples take the direct ctypes path: ~1 us instead of ~4 us
    through numpy for the short id / offset lists of a step.)"""
    if isinstance(seq, (list, tuple)):
        n = len(seq)
        return (C.c_int32 * n)(*seq) if n else (C.c_int32 * 1)()
    arr = np.ascontiguousarray(np.asarray(seq, dtype=np.int32))
    return (C.c_int32 * len(arr)).from_buffer_copy(arr.tobytes()) if len(arr) else (C.c_int32 * 1)()


def _ptr(t) -> Optional[int]:
    """Device/host pointer of a torch tensor (contiguous) or a raw int address; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return t.data_ptr()


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else None
    return stream if isinstance(stream, int) else stream.cuda_stream


class Cache:
    """One attention layer's paged KV cache + scheduler (ws_cache_t).  Owns the torch pools."""

    def __init__(self, dtype: int, num_q_heads: int, num_kv_heads: int, head_dim: int,
                 page_tokens: int, num_pages: int, max_sessions: int = 8,
                 max_pages_per_session: Optional[int] = None, max_blocks_per_session: int = 4096,
                 max_sessions_per_call: Optional[int] = None, max_q_tokens_per_call: int = 4096,
                 device: int = 0, flags: int = 0, q_to_kv_head: Optional[Sequence[int]] = None,
                 pool_fill: Optional[int] = None):
        self.lib = load_library()
        self.handle = C.c_void_p()
        cfg = CacheConfig()
        cfg.dtype, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim = dtype, num_q_heads, num_kv_heads, head_dim
        cfg.page_tokens, cfg.num_pages, cfg.max_sessions = page_tokens, num_pages, max_sessions
        cfg.max_pages_per_session = max_pages_per_session or num_pages
        cfg.max_blocks_per_session = max_blocks_per_session
        cfg.max_sessions_per_call = max_sessions_per_call or max_sessions
        cfg.max_q_tokens_per_call = max_q_tokens_per_call
        cfg.device, cfg.flags = device, flags
        self._map = _i32(q_to_kv_head) if q_to_kv_head is not None else None
        if self._map is not None:
            cfg.q_to_kv_head = C.cast(self._map, C.POINTER(C.c_int32))
        self.dry = bool(flags & WS_FLAG_DRY_RUN)
        self.dtype = dtype
        self.k_pool = self.v_pool = self.workspace = None
        if not self.dry:
            import torch
            tdt = torch.bfloat16 if dtype == WS_BF16 else torch.float32
            dev = torch.device("cuda", device)
            shape = (num_pages, num_kv_heads, page_tokens, head_dim)
            self.k_pool = torch.empty(shape, dtype=tdt, device=dev)
            self.v_pool = torch.empty(shape, dtype=tdt, device=dev)
            if pool_fill is not None:       # canary bit pattern (tests)
                itype = torch.int16 if dtype == WS_BF16 else torch.int32
                self.k_pool.view(itype).fill_(pool_fill)
                self.v_pool.view(itype).fill_(pool_fill)
            cfg.k_pool, cfg.v_pool = self.k_pool.data_ptr(), self.v_pool.data_ptr()
            cfg.pool_bytes = self.k_pool.numel() * self.k_pool.element_size()
            wsb = self.lib.ws_workspace_bytes(C.byref(cfg))
            if wsb == 0:
                raise WsError(1, "invalid cache configuration")
            self.workspace = torch.empty(wsb, dtype=torch.uint8, device=dev)
            cfg.workspace, cfg.workspace_bytes = self.workspace.data_ptr(), wsb
            torch.cuda.synchronize(dev)
        self.cfg = cfg
        _check(self.lib.ws_cache_create(C.byref(cfg), C.byref(self.handle)))

    def close(self) -> None:
        if self.handle:
            self.lib.ws_cache_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- sessions
    def session_open(self) -> int:
        s = C.c_int32()
        _check(self.lib.ws_session_open(self.handle, C.byref(s)))
        return s.value

    def session_close(self, s: int) -> None:
        _check(self.lib.ws_session_close(self.handle, s))

    def session_info(self, s: int):
        tokens, blocks, ends = C.c_int64(), C.c_int32(), C.POINTER(C.c_int64)()
        _check(self.lib.ws_session_info(self.handle, s, C.byref(tokens), C.byref(blocks), C.byref(ends)))
        return tokens.value, blocks.value, [ends[i] for i in range(blocks.value)]

    def session_truncate(self, s: int, keep_blocks: int) -> None:
        _check(self.lib.ws_session_truncate(self.handle, s, keep_blocks))

    def session_pages(self, s: int):
        n = C.c_int32()
        _check(self.lib.ws_session_pages(self.handle, s, None, 0, C.byref(n)))
        buf = (C.c_int32 * max(1, n.value))()
        _check(self.lib.ws_session_pages(self.handle, s, buf, n.value, C.byref(n)))
        return list(buf[:n.value])

    def free_pages(self) -> int:
        return self.lib.ws_free_pages(self.handle)

    # ---- hot path
    def kv_append(self, session_ids, cu_new_tokens, k_new, v_new, modality=None, stream=None):
        mod = None
        if modality is not None:
            m = np.ascontiguousarray(np.asarray(modality, dtype=np.uint8))
            mod = (C.c_uint8 * len(m)).from_buffer_copy(m.tobytes())
        _check(self.lib.ws_kv_append(self.handle, len(session_ids), _i32(session_ids),
                                     _i32(cu_new_tokens), _ptr(k_new), _ptr(v_new), mod,
                                     _stream_ptr(stream)))

    def kv_append_blocks(self, session_ids, cu_new_tokens, cu_blocks, block_tokens, k_new, v_new,
                         modality=None, stream=None):
        """ws_kv_append_blocks: several blocks per session committed by one call / one launch (NEXT-1)."""
        mod = None
        if modality is not None:
            m = np.ascontiguousarray(np.asarray(modality, dtype=np.uint8))
            mod = (C.c_uint8 * len(m)).from_buffer_copy(m.tobytes())
        _check(self.lib.ws_kv_append_blocks(self.handle, len(session_ids), _i32(session_ids),
                                            _i32(cu_new_tokens), _i32(cu_blocks), _i32(block_tokens),
                                            _ptr(k_new), _ptr(v_new), mod, _stream_ptr(stream)))

    def block_causal_attn_fwd(self, session_ids, cu_q_tokens, q, out, scale: float, lse=None,
                              num_q_blocks=None, stream=None, attn_flags: int = 0):
        """attn_flags != 0: ws_block_causal_attn_fwd_masked (WS_ATTN_TEXT_CAUSAL)."""
        nqb = _i32(num_q_blocks) if num_q_blocks is not None else None
        if attn_flags:
            _check(self.lib.ws_block_causal_attn_fwd_masked(self.handle, len(session_ids), _i32(session_ids),
                                                            nqb, _i32(cu_q_tokens), _ptr(q), _ptr(out), _ptr(lse),
                                                            C.c_float(scale), attn_flags, _stream_ptr(stream)))
            return
        _check(self.lib.ws_block_causal_attn_fwd(self.handle, len(session_ids), _i32(session_ids),
                                                 nqb, _i32(cu_q_tokens), _ptr(q), _ptr(out),
                                                 _ptr(lse), C.c_float(scale), _stream_ptr(stream)))

    def block_causal_attn_fwd_static(self, session_ids, cu_q_tokens, q, out, scale: float, lse=None,
                                     num_q_blocks=None, stream=None):
        """ws_block_causal_attn_fwd_static: split-KV partials in the library's static device array (no allocation)."""
        nqb = _i32(num_q_blocks) if num_q_blocks is not None else None
        _check(self.lib.ws_block_causal_attn_fwd_static(self.handle, len(session_ids), _i32(session_ids),
                                                        nqb, _i32(cu_q_tokens), _ptr(q), _ptr(out),
                                                        _ptr(lse), C.c_float(scale), _stream_ptr(stream)))

    def stream_step(self, session_ids, cu_new_tokens, q, k_new, v_new, out, scale: float, lse=None, stream=None,
                    modality=None, attn_flags: int = 0):
        """ws_kv_append + ws_block_causal_attn_fwd of the block just committed, one call (device buffers).
        modality / attn_flags: ws_stream_step_tagged."""
        if modality is not None or attn_flags:
            mod = None
            if modality is not None:
                m = np.ascontiguousarray(np.asarray(modality, dtype=np.uint8))
                mod = (C.c_uint8 * len(m)).from_buffer_copy(m.tobytes())
            _check(self.lib.ws_stream_step_tagged(self.handle, len(session_ids), _i32(session_ids),
                                                  _i32(cu_new_tokens), _ptr(q), _ptr(k_new), _ptr(v_new), mod,
                                                  attn_flags, _ptr(out), _ptr(lse), C.c_float(scale),
                                                  _stream_ptr(stream)))
            return
        _check(self.lib.ws_stream_step(self.handle, len(session_ids), _i32(session_ids), _i32(cu_new_tokens),
                                       _ptr(q), _ptr(k_new), _ptr(v_new), _ptr(out), _ptr(lse),
                                       C.c_float(scale), _stream_ptr(stream)))

    def step_staging_bytes(self, total_new_tokens: int) -> int:
        return self.lib.ws_step_staging_bytes(C.byref(self.cfg), total_new_tokens)

    def stream_step_host(self, session_ids, cu_new_tokens, q_host, k_host, v_host, out_host,
                         staging, scale: float, stream=None):
        _check(self.lib.ws_stream_step_host(self.handle, len(session_ids), _i32(session_ids),
                                            _i32(cu_new_tokens), _ptr(q_host), _ptr(k_host),
                                            _ptr(v_host), _ptr(out_host), _ptr(staging),
                                            staging.numel() * staging.element_size(),
                                            C.c_float(scale), _stream_ptr(stream)))

    def stream_host_join(self, stream=None):
        _check(self.lib.ws_stream_host_join(self.handle, _stream_ptr(stream)))

    def kv_gather(self, session: int, start: int, count: int, k_out, v_out, stream=None):
        _check(self.lib.ws_kv_gather(self.handle, session, start, count, _ptr(k_out), _ptr(v_out),
                                     _stream_ptr(stream)))

    # ---- NEXT-3 replica link (thinker -> performer KV-slice exchange)
    def pool_bytes(self) -> int:
        return self.lib.ws_pool_bytes(C.byref(self.cfg))

    def replica_link(self, peers) -> None:
        """peers: list of Cache objects (same process) or (k_ptr, v_ptr, pool_bytes) tuples (mapped pools)."""
        arr = (PeerPools * max(1, len(peers)))()
        for i, pr in enumerate(peers):
            if isinstance(pr, Cache):
                if pr.dry:
                    arr[i].k_pool, arr[i].v_pool, arr[i].pool_bytes = None, None, pr.pool_bytes()
                else:
                    arr[i].k_pool, arr[i].v_pool = pr.k_pool.data_ptr(), pr.v_pool.data_ptr()
                    arr[i].pool_bytes = pr.k_pool.numel() * pr.k_pool.element_size()
            else:
                arr[i].k_pool, arr[i].v_pool, arr[i].pool_bytes = pr
        _check(self.lib.ws_replica_link(self.handle, arr, len(peers)))

    def replica_accept(self, owner_pages: int) -> None:
        _check(self.lib.ws_replica_accept(self.handle, owner_pages))

    def _message(self, fn, *args) -> np.ndarray:
        n = C.c_int32()
        fn(self.handle, *args, None, 0, C.byref(n))          # size query (fails with INVALID_ARG by design)
        buf = (C.c_int32 * max(1, n.value))()
        _check(fn(self.handle, *args, buf, n.value, C.byref(n)))
        return np.frombuffer(buf, dtype=np.int32, count=n.value).copy()

    def replica_commit_message(self) -> np.ndarray:
        return self._message(self.lib.ws_replica_commit_message)

    def replica_snapshot_message(self, session: int) -> np.ndarray:
        return self._message(self.lib.ws_replica_snapshot_message, session)

    def replica_push_session(self, session: int, stream=None) -> None:
        _check(self.lib.ws_replica_push_session(self.handle, session, _stream_ptr(stream)))

    def replica_apply(self, words, stream=None) -> None:
        w = np.ascontiguousarray(np.asarray(words, dtype=np.int32))
        _check(self.lib.ws_replica_apply(self.handle, _i32(w), len(w), _stream_ptr(stream)))

    # ---- introspection / debug
    def shuffle_free_pages(self, seed: int) -> None:
        _check(self.lib.ws_debug_shuffle_free_pages(self.handle, seed))

    def set_min_splits(self, n: int) -> None:
        _check(self.lib.ws_debug_set_min_splits(self.handle, n))

    def set_decode_plan(self, enable: bool) -> None:
        _check(self.lib.ws_debug_set_decode_plan(self.handle, int(enable)))

    def last_plan_info(self) -> dict:
        info = PlanInfo()
        _check(self.lib.ws_last_plan_info(self.handle, C.byref(info)))
        return {n: getattr(info, n) for n, _ in PlanInfo._fields_}

    def last_plan_segments(self):
        n = self.last_plan_info()["num_segments"]
        out = []
        for i in range(n):
            seg = PlanSegment()
            _check(self.lib.ws_last_plan_segment(self.handle, i, C.byref(seg)))
            out.append({k: getattr(seg, k) for k, _ in PlanSegment._fields_})
        return out

    def launch_count(self) -> int:
        return self.lib.ws_launch_count(self.handle)

    def kernel_timing(self, enable: bool) -> None:
        _check(self.lib.ws_debug_kernel_timing(self.handle, int(enable)))

    def read_kernel_times(self) -> dict:
        """{'append'|'attn'|'combine': (sum_ms, launches)} since the last read."""
        ms, cnt = (C.c_double * 3)(), (C.c_int32 * 3)()
        _check(self.lib.ws_debug_read_kernel_times(self.handle, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(("append", "attn", "combine"))}


# ---- module-level functions with the C names (same marshalling) -------------------------------
def ws_kv_append(cache: Cache, session_ids, cu_new_tokens, k_new, v_new, modality=None, stream=None):
    cache.kv_append(session_ids, cu_new_tokens, k_new, v_new, modality, stream)


def ws_kv_append_blocks(cache: Cache, session_ids, cu_new_tokens, cu_blocks, block_tokens, k_new, v_new,
                        modality=None, stream=None):
    cache.kv_append_blocks(session_ids, cu_new_tokens, cu_blocks, block_tokens, k_new, v_new, modality, stream)


def ws_block_causal_attn_fwd(cache: Cache, session_ids, cu_q_tokens, q, out, scale, lse=None,
                             num_q_blocks=None, stream=None):
    cache.block_causal_attn_fwd(session_ids, cu_q_tokens, q, out, scale, lse, num_q_blocks, stream)


def ws_block_causal_attn_fwd_static(cache: Cache, session_ids, cu_q_tokens, q, out, scale, lse=None,
                                    num_q_blocks=None, stream=None):
    cache.block_causal_attn_fwd_static(session_ids, cu_q_tokens, q, out, scale, lse, num_q_blocks, stream)


def ws_static_scratch_setup(device: int = 0) -> None:
    _check(load_library().ws_static_scratch_setup(device))


def ws_kv_gather(cache: Cache, session, start, count, k_out, v_out, stream=None):
    cache.kv_gather(session, start, count, k_out, v_out, stream)


def ws_stream_step(cache: Cache, session_ids, cu_new_tokens, q, k_new, v_new, out, scale, lse=None, stream=None):
    cache.stream_step(session_ids, cu_new_tokens, q, k_new, v_new, out, scale, lse=lse, stream=stream)


def ws_stream_step_host(cache: Cache, session_ids, cu_new_tokens, q_host, k_host, v_host, out_host,
                        staging, scale, stream=None):
    cache.stream_step_host(session_ids, cu_new_tokens, q_host, k_host, v_host, out_host, staging,
                           scale, stream)


def ws_fm_euler_update(z, v, dtau: float, stream=None):
    """z <- z + dtau * v in place (torch bf16 / fp32 tensors, same shape, contiguous)."""
    import torch
    if z.dtype != v.dtype or z.numel() != v.numel():
        raise ValueError("z and v must have the same dtype and size")
    dt = {torch.bfloat16: WS_BF16, torch.float32: WS_F32}[z.dtype]
    _check(load_library().ws_fm_euler_update(dt, _ptr(z), _ptr(v), C.c_float(dtau), z.numel(), _stream_ptr(stream)))


def ws_ipc_export(tensor_or_ptr):
    """(handle: bytes[64], offset) for a device pointer, to be opened in another process."""
    h, off = (C.c_uint8 * 64)(), C.c_uint64()
    _check(load_library().ws_ipc_export(_ptr(tensor_or_ptr), h, C.byref(off)))
    return bytes(h), off.value


def ws_ipc_open(handle: bytes, offset: int, device: int = 0) -> int:
    out = C.c_void_p()
    h = (C.c_uint8 * 64).from_buffer_copy(handle)
    _check(load_library().ws_ipc_open(h, offset, device, C.byref(out)))
    return out.value


def ws_ipc_close(ptr: int, offset: int) -> None:
    _check(load_library().ws_ipc_close(ptr, offset))


def ws_version() -> str:
    return load_library().ws_version().decode()

"""paper_2606_25041_b200 - B200-native block-causal streaming attention (Wan-Streamer hot path).

The product is the C-ABI library `libwanstream.so` (include/ws.h, sources in csrc/); this package
holds its build script and a thin ctypes binding with the same entry-point names.
"""
from .binding import (  # noqa: F401
    WS_ATTN_TEXT_CAUSAL, WS_BF16, WS_F32, WS_FLAG_DRY_RUN, WS_FLAG_FORCE_SIMT, WS_FLAG_FUSED_COMBINE, WS_FLAG_SEPARATE_APPEND, Cache, WsError, load_library,
    ws_block_causal_attn_fwd, ws_block_causal_attn_fwd_static, ws_static_scratch_setup, ws_fm_euler_update, ws_ipc_close, ws_ipc_export, ws_ipc_open, ws_kv_append, ws_kv_append_blocks, ws_kv_gather, ws_stream_step, ws_stream_step_host,
    ws_version,
)

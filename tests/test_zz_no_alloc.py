"""ws_block_causal_attn_fwd_static (include/ws.h): the split-KV partials go to the library's file-scope static
__device__ array instead of the workspace, for callers that cannot allocate.  Checked against the existing
entry point (ws_block_causal_attn_fwd, itself checked against the float64 oracle by tests/test_gpu_parity.py) on two calls in a row, plus the size limit.
Named test_zz_* so that pytest collects it last."""
import math

import numpy as np
import pytest

from synth_inputs import to_bf16
from tests.gpu_harness import _torch_of

pytestmark = pytest.mark.gpu

TOL_MAX_ABS, TOL_MEAN_ABS, TOL_LSE = 1e-2, 1e-3, 1e-4     # the bf16 tolerances of tests/test_gpu_parity.py


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as entry
    entry.build()


def _make(L, n, Hq, Hkv, seed):
    """one session: cache of L tokens (committed in 256-token blocks) + one block of n tokens; returns the cache
    handle, the session id and the numpy K/V of all L + n tokens"""
    import torch
    from paper_2606_25041_b200 import WS_BF16, Cache
    rng = np.random.default_rng(seed)
    k_all = to_bf16(rng.standard_normal((L + n, Hkv, 128), dtype=np.float32))
    v_all = to_bf16(rng.standard_normal((L + n, Hkv, 128), dtype=np.float32))
    P = 64
    c = Cache(WS_BF16, Hq, Hkv, 128, P, (L + n + P - 1) // P + 2, max_sessions=1, max_q_tokens_per_call=max(n, 256))
    sid = c.session_open()
    dev = torch.device("cuda", 0)
    pos = 0
    while pos < L:
        hi = min(L, pos + 256)
        c.kv_append([sid], [0, hi - pos], _torch_of(k_all[pos:hi], dev), _torch_of(v_all[pos:hi], dev)); pos = hi
    c.kv_append([sid], [0, n], _torch_of(k_all[L:], dev), _torch_of(v_all[L:], dev))
    return c, sid, k_all, v_all


def test_static_scratch_entry_point_matches_existing_path_twice_in_a_row():
    import torch
    from paper_2606_25041_b200 import ws_static_scratch_setup
    L, n, Hq, Hkv = 4000 + 37, 64, 8, 2                               # 2 groups of 256 packed rows, 33 KV tiles each
    scale = 1.0 / math.sqrt(128)
    c, sid, k_all, v_all = _make(L, n, Hq, Hkv, seed=11)
    dev = torch.device("cuda", 0)
    ws_static_scratch_setup(0)
    rng = np.random.default_rng(12)
    qs = [to_bf16(rng.standard_normal((n, Hq, 128), dtype=np.float32)) for _ in range(2)]
    # existing path (partials in the workspace)
    want = []
    for q in qs:
        out = torch.empty((n, Hq, 128), dtype=torch.bfloat16, device=dev)
        lse = torch.empty((n, Hq), dtype=torch.float32, device=dev)
        c.block_causal_attn_fwd([sid], [0, n], _torch_of(q, dev), out, scale, lse=lse)
        torch.cuda.synchronize()
        want.append((out.float().cpu().numpy(), lse.cpu().numpy()))
    info = c.last_plan_info()
    assert info["used_tensor_core_kernel"] == 1 and 0 < info["num_partial_slots"] <= 64, info   # scratch is in use
    # new entry point, two calls in a row on one stream (second with other queries: the array keeps the first
    # call's partials, which must not leak into the second result), no host sync in between
    free_before = torch.cuda.mem_get_info()[0]
    q_dev = [_torch_of(q, dev) for q in qs]
    outs = [torch.full((n, Hq, 128), float("nan"), dtype=torch.bfloat16, device=dev) for _ in qs]
    lses = [torch.full((n, Hq), float("nan"), dtype=torch.float32, device=dev) for _ in qs]
    for i in range(2):
        c.block_causal_attn_fwd_static([sid], [0, n], q_dev[i], outs[i], scale, lse=lses[i])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before - (2 << 20)     # nothing was allocated on the device
    assert c.last_plan_info() == info                                  # same plan
    for i in range(2):
        o, l = outs[i].float().cpu().numpy(), lses[i].cpu().numpy()
        wo, wl = want[i]
        assert np.isfinite(o).all() and np.isfinite(l).all()
        d = np.abs(o.astype(np.float64) - wo.astype(np.float64))
        print(f"[parity] static scratch call {i}: max_abs={d.max():.3e} mean_abs={d.mean():.3e} "
              f"lse_max={np.abs(l - wl).max():.3e} bit_identical={bool((o == wo).all())}")
        assert d.max() <= TOL_MAX_ABS and d.mean() <= TOL_MEAN_ABS and np.abs(l - wl).max() <= TOL_LSE, i
    assert np.abs(outs[0].float().cpu().numpy() - outs[1].float().cpu().numpy()).max() > 1e-2   # (really two problems)


def test_static_scratch_entry_point_rejects_plans_beyond_its_size():
    import torch
    from paper_2606_25041_b200 import WsError
    L, n, Hq, Hkv = 8192, 256, 32, 8                                  # 8 groups x 4 pairs, ~37 KV ranges: > 64 slots
    scale = 1.0 / math.sqrt(128)
    c, sid, k_all, v_all = _make(L, n, Hq, Hkv, seed=13)
    dev = torch.device("cuda", 0)
    q = _torch_of(to_bf16(np.random.default_rng(14).standard_normal((n, Hq, 128), dtype=np.float32)), dev)
    out = torch.full((n, Hq, 128), float("nan"), dtype=torch.bfloat16, device=dev)
    launches = c.launch_count()
    with pytest.raises(WsError) as ei:
        c.block_causal_attn_fwd_static([sid], [0, n], q, out, scale)
    assert "64 partial slots" in str(ei.value) and "static scratch" in str(ei.value), str(ei.value)
    torch.cuda.synchronize()
    assert c.launch_count() == launches and bool(torch.isnan(out.float()).all())      # nothing ran
    # the cache is unharmed: the workspace path still serves the same call
    c.block_causal_attn_fwd([sid], [0, n], q, out, scale)
    torch.cuda.synchronize()
    assert c.last_plan_info()["num_partial_slots"] > 64 and bool(torch.isfinite(out.float()).all())


def test_static_scratch_entry_point_ragged_batch_and_generic_kernel():
    """Three sessions of unequal history in one call (bf16, tcgen05 kernel, split plan) and the fp32 cache (CUDA-core
    kernel: no scratch in use at all) through the same entry point: both equal the existing path bit for bit."""
    import torch
    from paper_2606_25041_b200 import WS_BF16, WS_F32, Cache
    dev = torch.device("cuda", 0)
    for dtype, tdt, Hq, Hkv, D, P, lens, n in ((WS_BF16, torch.bfloat16, 8, 2, 128, 64, (700, 1531, 2048), 48),
                                               (WS_F32, torch.float32, 2, 2, 64, 16, (0, 33), 16)):
        S = len(lens)
        pages = sum((L + n + P - 1) // P for L in lens) + 4
        c = Cache(dtype, Hq, Hkv, D, P, pages, max_sessions=S, max_sessions_per_call=S, max_q_tokens_per_call=max(S * n, 256))
        g = torch.Generator(device=dev); g.manual_seed(21)
        ids = [c.session_open() for _ in lens]
        for sid, L in zip(ids, lens):
            pos = 0
            while pos < L:
                m = min(256, L - pos)
                c.kv_append([sid], [0, m], torch.randn((m, Hkv, D), device=dev, generator=g).to(tdt),
                            torch.randn((m, Hkv, D), device=dev, generator=g).to(tdt)); pos += m
        cu = [i * n for i in range(S + 1)]
        c.kv_append(ids, cu, torch.randn((S * n, Hkv, D), device=dev, generator=g).to(tdt),
                    torch.randn((S * n, Hkv, D), device=dev, generator=g).to(tdt))
        q = torch.randn((S * n, Hq, D), device=dev, generator=g).to(tdt)
        scale = 1.0 / math.sqrt(D)
        want, got = torch.empty_like(q), torch.full_like(q, float("nan"))
        wl = torch.empty((S * n, Hq), dtype=torch.float32, device=dev); gl = torch.full_like(wl, float("nan"))
        c.block_causal_attn_fwd(ids, cu, q, want, scale, lse=wl)
        info = c.last_plan_info()
        c.block_causal_attn_fwd_static(ids, cu, q, got, scale, lse=gl)
        torch.cuda.synchronize()
        assert c.last_plan_info() == info
        if dtype == WS_BF16:
            assert info["used_tensor_core_kernel"] == 1 and 0 < info["num_partial_slots"] <= 64, info
        else:
            assert info["used_tensor_core_kernel"] == 0
        d = (got.float() - want.float()).abs()
        assert bool(torch.isfinite(got.float()).all()) and float(d.max()) <= (TOL_MAX_ABS if dtype == WS_BF16 else 1e-5)
        assert float((gl - wl).abs().max()) <= (TOL_LSE if dtype == WS_BF16 else 1e-5)
        assert bool((got == want).all()) and bool((gl == wl).all())

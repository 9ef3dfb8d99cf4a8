"""Seeded random shapes through the C ABI vs the float64 oracle (GPU): head counts / GQA group sizes, block sizes from
one token to several Q tiles, cache lengths around page and tile boundaries, forced split counts, one or several
sessions, separate calls or the fused step.  Catches what the hand-picked cases miss (a wrong tile / lane / split
boundary at some shape); every case is gated on the contract tolerances and the element-wise derived bound."""
import numpy as np
import pytest

from synth_inputs import generate, spec_for_config
from tests.gpu_harness import compare, run_workload_gpu, run_workload_oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as entry
    entry.build()


def _cases():
    rng = np.random.default_rng([2606, 25041, 77])
    out = []
    for i in range(28):
        Hkv = int(rng.choice([1, 2, 4]))
        G = int(rng.choice([1, 2, 4, 8, 16]))
        n = int(rng.choice([1, 2, 3, 5, 8, 16, 31, 33, 64, 100, 128, 200, 257, 300]))
        S = int(rng.choice([1, 1, 2, 3]))
        lens = tuple(int(x) for x in rng.integers(0, 2600, size=S))
        if i % 7 == 0:
            lens = tuple(int(rng.choice([0, 63, 64, 65, 127, 128, 129, 1023, 1024, 1025])) for _ in range(S))
        out.append(dict(idx=i, Hkv=Hkv, G=G, n=n, lens=lens, steps=int(rng.choice([1, 2, 3])),
                        splits=int(rng.choice([0, 0, 2, 5])), fused=bool(rng.integers(0, 2)), seed_cfg=2 if S == 1 else 5))
    return out


@pytest.mark.parametrize("case", _cases(), ids=lambda c: f"{c['idx']}_S{len(c['lens'])}_h{c['Hkv']}x{c['G']}_n{c['n']}")
def test_random_shapes_match_oracle(case):
    n = case["n"]
    text = max(0, n // 16)
    spec = spec_for_config(case["seed_cfg"], num_sessions=len(case["lens"]), cache_lens=case["lens"], cache_len_range=None,
                           num_q_heads=case["Hkv"] * case["G"], num_kv_heads=case["Hkv"], block_tokens=n,
                           modality_split=(n - text - min(n - text, n // 4), min(n - text, n // 4), text),
                           steps=case["steps"], outlier_frac=0.0, outlier_scale=1.0)
    w = generate(spec)
    ref = run_workload_oracle(w)
    got = run_workload_gpu(w, min_splits=case["splits"], fused_step=case["fused"], pool_fill=0x7FC1)
    assert got["tensor"]
    err = compare(got, ref, "bf16")
    print(f"[parity] fuzz {case}: " + " ".join(f"{k}={v:.3e}" if isinstance(v, float) else f"{k}={v}" for k, v in err.items()))
    assert err["finite"] and err["kv_bit_exact"]
    assert err["bound_viol"] <= 0 and err["mean_abs"] <= 1e-3 and err["rel_rms"] <= 1e-2 and err["lse_max"] <= 1e-4
    if max(np.abs(o).max() for step in ref["out"] for o in step) < 1.0:
        assert err["max_abs"] <= 1e-2


def _wide_cases():
    """A second, wider draw: odd KV head counts, up to five ragged sessions, cache lengths up to 9000 and around every
    page / tile boundary, x8 outlier channels (reading A15), the decode plan forced on or off, shuffled free pages, and
    G in {3, 6} - group sizes the tcgen05 kernel does not cover, which the generic CUDA-core kernel serves (ws.h,
    `head_dim`).  Forced split counts are kept within the workspace's partial slots."""
    rng = np.random.default_rng([2606, 25041, 1905])
    out = []
    for i in range(48):
        Hkv = int(rng.choice([1, 2, 3, 4, 8]))
        G = int(rng.choice([3, 6])) if i % 6 == 5 else int(rng.choice([1, 2, 4, 8, 16]))
        n = int(rng.choice([1, 2, 3, 4, 7, 8, 15, 16, 17, 31, 32, 33, 63, 64, 65, 96, 127, 128, 129, 200, 255, 256, 257,
                            300, 384, 513]))
        S = int(rng.choice([1, 1, 2, 3, 5]))
        lens = tuple(int(x) for x in rng.integers(0, int(rng.choice([300, 2600, 9000])), size=S))
        if i % 5 == 0:
            lens = tuple(int(rng.choice([0, 1, 63, 64, 65, 127, 128, 129, 191, 192, 193, 1023, 1024, 1025, 4095, 4096,
                                         4097])) for _ in range(S))
        splits = int(rng.choice([0, 0, 2, 3, 5, 9]))
        groups = S * Hkv * (-(-n * G // 256))
        if groups * max(splits, 1) > 400:
            splits = 0
        out.append(dict(idx=i, Hkv=Hkv, G=G, n=n, lens=lens, steps=int(rng.choice([1, 2, 3])), splits=splits,
                        fused=bool(rng.integers(0, 2)), seed_cfg=2 if S == 1 else 5, outl=bool(rng.integers(0, 4) == 0),
                        decode=[None, True, False][int(rng.integers(0, 3))], shuffle=int(rng.integers(0, 1000))))
    return out


@pytest.mark.parametrize("case", _wide_cases(),
                         ids=lambda c: f"w{c['idx']}_S{len(c['lens'])}_h{c['Hkv']}x{c['G']}_n{c['n']}")
def test_random_shapes_wide_match_oracle(case):
    n = case["n"]
    text = max(0, n // 16)
    spec = spec_for_config(case["seed_cfg"], num_sessions=len(case["lens"]), cache_lens=case["lens"], cache_len_range=None,
                           num_q_heads=case["Hkv"] * case["G"], num_kv_heads=case["Hkv"], block_tokens=n,
                           modality_split=(n - text - min(n - text, n // 4), min(n - text, n // 4), text),
                           steps=case["steps"], outlier_frac=0.05 if case["outl"] else 0.0,
                           outlier_scale=8.0 if case["outl"] else 1.0)
    w = generate(spec)
    ref = run_workload_oracle(w)
    got = run_workload_gpu(w, min_splits=case["splits"], fused_step=case["fused"], pool_fill=0x7FC1,
                           decode_plan=case["decode"], shuffle_seed=case["shuffle"])
    assert got["tensor"] == (case["G"] in (1, 2, 4, 8, 16))
    err = compare(got, ref, "bf16")
    print(f"[parity] fuzz-wide {case}: " + " ".join(f"{k}={v:.3e}" if isinstance(v, float) else f"{k}={v}" for k, v in err.items()))
    assert err["finite"] and err["kv_bit_exact"]
    assert err["bound_viol"] <= 0 and err["mean_abs"] <= 1e-3 and err["rel_rms"] <= 1e-2 and err["lse_max"] <= 1e-4
    if max(np.abs(o).max() for step in ref["out"] for o in step) < 1.0:
        assert err["max_abs"] <= 1e-2


@pytest.mark.parametrize("S,Hkv,G,n,hi,fused,decode", [
    (32, 2, 4, 1, 2000, True, None),        # batched one-token decode, 32 sessions
    (64, 1, 4, 1, 1500, False, None),       # 64 sessions, separate append / attend calls
    (32, 8, 4, 4, 1500, True, None),        # 256 (session, KV head) groups on 148 CTAs
    (24, 2, 8, 64, 1200, True, None),       # general plan, teams of two
    (48, 1, 16, 8, 800, True, True),        # 128 packed rows per group on the decode kernel
    (20, 8, 4, 33, 600, True, False),       # more groups than CTAs, decode plan off
], ids=lambda v: str(v))
def test_many_session_batches_match_oracle(S, Hkv, G, n, hi, fused, decode):
    """Serving-sized batches: BASELINE config 5's ragged multi-session shape widened to tens of sessions in ONE call,
    more (session, KV head) groups than CTAs; vs the oracle at every element, append bit-exact."""
    rng = np.random.default_rng([S, Hkv, G, n])
    lens = tuple(int(x) for x in rng.integers(0, hi, size=S))
    text = n // 16
    spec = spec_for_config(5, num_sessions=S, cache_lens=lens, cache_len_range=None, num_q_heads=Hkv * G, num_kv_heads=Hkv,
                           block_tokens=n, modality_split=(n - text - min(n - text, n // 4), min(n - text, n // 4), text),
                           steps=2, outlier_frac=0.0, outlier_scale=1.0)
    w = generate(spec)
    ref = run_workload_oracle(w)
    got = run_workload_gpu(w, fused_step=fused, pool_fill=0x7FC1, decode_plan=decode)
    assert got["tensor"]
    err = compare(got, ref, "bf16")
    print(f"[parity] batch S={S} Hkv={Hkv} G={G} n={n} plan={got['plans'][-1]}: "
          + " ".join(f"{k}={v:.3e}" if isinstance(v, float) else f"{k}={v}" for k, v in err.items()))
    assert err["finite"] and err["kv_bit_exact"]
    assert err["bound_viol"] <= 0 and err["max_abs"] <= 1e-2 and err["mean_abs"] <= 1e-3 and err["rel_rms"] <= 1e-2
    assert err["lse_max"] <= 1e-4

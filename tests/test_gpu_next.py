"""GPU parity tests of the round-2 NEXT items, through the C ABI, against the float64 oracle:

* NEXT-1 completion (PAPER.md:75 system prefill, :69): ws_kv_append_blocks commits many blocks per session
  in ONE call / ONE launch - bit-exact gather, block ends, and a prefill that uses it;
* NEXT-4 optional half (reading A19): the text-causal mixed intra-block mask
  (WS_ATTN_TEXT_CAUSAL) on the tcgen05 kernel (general plan, decode plan, fused step, split KV, multi-block
  queries) and on the generic fp32 kernel.
"""
import math

import numpy as np
import pytest

from synth_inputs import to_bf16
from tests.gpu_harness import _numpy_of, _torch_of, bf16_error_bound

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as entry
    entry.build()


def _mk(rng, dtype, *sh):
    x = rng.standard_normal(sh, dtype=np.float32)
    return to_bf16(x) if dtype == "bf16" else x


def _cache(dtype, Hq, Hkv, D, P, tokens, sessions=1, max_q=4096, flags=0):
    from paper_2606_25041_b200 import WS_BF16, WS_F32, Cache
    return Cache(WS_BF16 if dtype == "bf16" else WS_F32, Hq, Hkv, D, P, sessions * ((tokens + P - 1) // P + 2),
                 max_sessions=sessions, max_q_tokens_per_call=max_q, max_blocks_per_session=4096, flags=flags)


# ------------------------------------------------------------------------------------------ NEXT-1
def test_append_blocks_bit_exact_and_equal_to_single_appends():
    """Two sessions, ragged block lists, mid-page starts: one ws_kv_append_blocks call == the oracle's
    concatenation bit for bit (random 16-bit patterns incl. NaN / Inf payloads), block ends recorded per block,
    exactly one kernel launch."""
    import torch
    rng = np.random.default_rng(11)
    dev = torch.device("cuda", 0)
    Hkv, D = 2, 128
    c = _cache("bf16", 4, Hkv, D, 64, 3000, sessions=2, max_q=4096)
    s0, s1 = c.session_open(), c.session_open()
    bits = lambda n: torch.from_numpy(rng.integers(0, 65536, size=(n, Hkv, D), dtype=np.uint16).view(np.int16)).to(dev).view(torch.bfloat16)
    k_pre, v_pre = bits(37), bits(37)
    c.kv_append([s0], [0, 37], k_pre, v_pre)                          # session 0 starts mid-page
    lens0, lens1 = [100, 1, 256, 63, 300], [64, 700, 5]
    n0, n1 = sum(lens0), sum(lens1)
    k, v = bits(n0 + n1), bits(n0 + n1)
    before = c.launch_count()
    c.kv_append_blocks([s0, s1], [0, n0, n0 + n1], [0, len(lens0), len(lens0) + len(lens1)], lens0 + lens1, k, v)
    assert c.launch_count() == before + 1
    assert c.session_info(s0) == (37 + n0, 6, list(np.cumsum([37] + lens0)))
    assert c.session_info(s1) == (n1, 3, list(np.cumsum(lens1)))
    for sid, (kr, vr) in ((s0, (torch.cat([k_pre, k[:n0]]), torch.cat([v_pre, v[:n0]]))), (s1, (k[n0:], v[n0:]))):
        T = c.session_info(sid)[0]
        kg = torch.empty((T, Hkv, D), dtype=torch.bfloat16, device=dev); vg = torch.empty_like(kg)
        c.kv_gather(sid, 0, T, kg, vg)
        torch.cuda.synchronize()
        assert torch.equal(kg.view(torch.int16), kr.view(torch.int16))
        assert torch.equal(vg.view(torch.int16), vr.view(torch.int16))


@pytest.mark.parametrize("blocks,Hq,Hkv,L0", [([256] * 8, 8, 2, 0), ([100, 37, 256, 1, 300], 4, 4, 500), ([64] * 24, 16, 2, 0)])
def test_prefill_committed_in_one_call_matches_oracle(blocks, Hq, Hkv, L0):
    """System prefill: the whole prompt committed by ONE ws_kv_append_blocks call, then queried by
    ONE multi-block attention call; matches the oracle (which appends block by block)."""
    import torch
    from oracle.block_causal import OracleSession, attend
    rng = np.random.default_rng(sum(blocks) + Hq)
    dev = torch.device("cuda", 0)
    T = sum(blocks)
    k0, v0 = _mk(rng, "bf16", L0, Hkv, 128), _mk(rng, "bf16", L0, Hkv, 128)
    q, k, v = _mk(rng, "bf16", T, Hq, 128), _mk(rng, "bf16", T, Hkv, 128), _mk(rng, "bf16", T, Hkv, 128)
    c = _cache("bf16", Hq, Hkv, 128, 64, L0 + T, max_q=max(T, 512))
    sid = c.session_open()
    sess = OracleSession(Hkv, 128)
    if L0:
        c.kv_append([sid], [0, L0], _torch_of(k0, dev), _torch_of(v0, dev))
        sess.append(k0, v0)
    launches = c.launch_count()
    c.kv_append_blocks([sid], [0, T], [0, len(blocks)], blocks, _torch_of(k, dev), _torch_of(v, dev))
    assert c.launch_count() == launches + 1
    pos = 0
    for b in blocks:
        sess.append(k[pos:pos + b], v[pos:pos + b]); pos += b
    out = torch.full((T, Hq, 128), float("nan"), dtype=torch.bfloat16, device=dev)
    lse = torch.full((T, Hq), float("nan"), dtype=torch.float32, device=dev)
    scale = 1.0 / math.sqrt(128)
    c.block_causal_attn_fwd([sid], [0, T], _torch_of(q, dev), out, scale, lse=lse, num_q_blocks=[len(blocks)])
    torch.cuda.synchronize()
    assert c.last_plan_info()["used_tensor_core_kernel"] == 1
    o_ref, l_ref, a_ref = attend(sess, q, scale, len(blocks), want_abs=True)
    o = out.float().cpu().numpy().astype(np.float64)
    d = o - o_ref
    print(f"[parity] prefill via append_blocks {blocks[:3]}..x{len(blocks)}: max_abs={np.abs(d).max():.3e} mean_abs={np.abs(d).mean():.3e}")
    assert np.isfinite(o).all()
    assert np.abs(d).max() <= 1e-2 and np.abs(d).mean() <= 1e-3
    assert (np.abs(d) - bf16_error_bound(o_ref, o, a_ref)).max() <= 0
    assert np.abs(lse.cpu().numpy() - l_ref).max() <= 1e-4


# ------------------------------------------------------------------------------------------ NEXT-4
def _tags(rng, n, p_text=0.3):
    """random interleaving of video / audio / text slots"""
    t = rng.integers(0, 2, size=n).astype(np.uint8)
    t[rng.random(n) < p_text] = 2
    return t


def _text_causal_case(dtype, Hq, Hkv, D, P, L0_blocks, q_blocks, seed, mode, min_splits=0, decode_plan=None,
                      p_text=0.3, flags=0):
    """history = L0_blocks (committed with tags), then q_blocks; mode:
       'two_calls'  - every query block appended (tagged) and attended by itself with WS_ATTN_TEXT_CAUSAL;
       'fused'      - the same through ws_stream_step_tagged (one launch commits and attends);
       'one_shot'   - all query blocks committed, then queried in ONE call (num_q_blocks = len(q_blocks)).
    Returns (gpu O, gpu LSE, oracle O, oracle LSE, oracle A, plan infos)."""
    import torch
    from oracle.block_causal import OracleSession, attend
    from paper_2606_25041_b200 import WS_ATTN_TEXT_CAUSAL
    rng = np.random.default_rng(seed)
    dev = torch.device("cuda", 0)
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    total = sum(L0_blocks) + sum(q_blocks)
    c = _cache(dtype, Hq, Hkv, D, P, total, max_q=max(512, sum(q_blocks), max(L0_blocks, default=1)), flags=flags)
    if min_splits:
        c.set_min_splits(min_splits)
    if decode_plan is not None:
        c.set_decode_plan(decode_plan)
    sid = c.session_open()
    sess = OracleSession(Hkv, D)
    scale = 1.0 / math.sqrt(D)
    for b in L0_blocks:
        kk, vv, tg = _mk(rng, dtype, b, Hkv, D), _mk(rng, dtype, b, Hkv, D), _tags(rng, b, p_text)
        c.kv_append([sid], [0, b], _torch_of(kk, dev), _torch_of(vv, dev), modality=tg)
        sess.append(kk, vv, modality=tg)
    outs, lses, refs, plans = [], [], [], []
    qs = []
    for b in q_blocks:
        qq, kk, vv, tg = _mk(rng, dtype, b, Hq, D), _mk(rng, dtype, b, Hkv, D), _mk(rng, dtype, b, Hkv, D), _tags(rng, b, p_text)
        sess.append(kk, vv, modality=tg)
        qs.append(qq)
        out = torch.full((b, Hq, D), float("nan"), dtype=tdt, device=dev)
        lse = torch.full((b, Hq), float("nan"), dtype=torch.float32, device=dev)
        if mode == "fused":
            c.stream_step([sid], [0, b], _torch_of(qq, dev), _torch_of(kk, dev), _torch_of(vv, dev), out, scale,
                          lse=lse, modality=tg, attn_flags=WS_ATTN_TEXT_CAUSAL)
        else:
            c.kv_append([sid], [0, b], _torch_of(kk, dev), _torch_of(vv, dev), modality=tg)
            if mode == "two_calls":
                c.block_causal_attn_fwd([sid], [0, b], _torch_of(qq, dev), out, scale, lse=lse,
                                        attn_flags=WS_ATTN_TEXT_CAUSAL)
        if mode != "one_shot":
            torch.cuda.synchronize()
            plans.append(c.last_plan_info())
            outs.append(out.float().cpu().numpy().astype(np.float64)); lses.append(lse.cpu().numpy().astype(np.float64))
            refs.append(attend(sess, qq, scale, 1, want_abs=True, text_causal=True))
    if mode == "one_shot":
        T = sum(q_blocks)
        q = np.concatenate(qs)
        out = torch.full((T, Hq, D), float("nan"), dtype=tdt, device=dev)
        lse = torch.full((T, Hq), float("nan"), dtype=torch.float32, device=dev)
        c.block_causal_attn_fwd([sid], [0, T], _torch_of(q, dev), out, scale, lse=lse, num_q_blocks=[len(q_blocks)],
                                attn_flags=WS_ATTN_TEXT_CAUSAL)
        torch.cuda.synchronize()
        plans.append(c.last_plan_info())
        outs.append(out.float().cpu().numpy().astype(np.float64)); lses.append(lse.cpu().numpy().astype(np.float64))
        refs.append(attend(sess, q, scale, len(q_blocks), want_abs=True, text_causal=True))
    o, l = np.concatenate(outs), np.concatenate(lses)
    o_ref, l_ref, a_ref = (np.concatenate([r[i] for r in refs]) for i in range(3))
    return o, l, o_ref, l_ref, a_ref, plans


def _gate_bf16(o, l, o_ref, l_ref, a_ref, label):
    d = o - o_ref
    viol = (np.abs(d) - bf16_error_bound(o_ref, o, a_ref)).max()
    print(f"[parity] text-causal {label}: max_abs={np.abs(d).max():.3e} mean_abs={np.abs(d).mean():.3e} "
          f"lse_max={np.abs(l - l_ref).max():.3e} bound_viol={viol:.3e}")
    assert np.isfinite(o).all() and np.isfinite(l).all()
    assert np.abs(d).max() <= 1e-2 and np.abs(d).mean() <= 1e-3
    assert np.sqrt((d ** 2).mean() / (o_ref ** 2).mean()) <= 1e-2
    assert viol <= 0
    assert np.abs(l - l_ref).max() <= 1e-4


TC_CASES = [
    # label, Hq, Hkv, history blocks, query blocks
    ("gqa4_unit256_ragged_history", 8, 2, [256, 256, 200, 59], [256, 256]),     # block starts mid-page and mid-tile
    ("mha_unit150", 4, 4, [300], [150, 150, 150]),
    ("gqa8_short_units", 16, 2, [64] * 5, [64, 33, 100]),
    ("empty_history", 4, 2, [], [200, 56]),
]


@pytest.mark.parametrize("mode", ["two_calls", "fused", "one_shot"])
@pytest.mark.parametrize("label,Hq,Hkv,hist,qb", TC_CASES, ids=[x[0] for x in TC_CASES])
def test_text_causal_tensor_core(label, Hq, Hkv, hist, qb, mode):
    o, l, o_ref, l_ref, a_ref, plans = _text_causal_case("bf16", Hq, Hkv, 128, 64, hist, qb, seed=len(label) + Hq, mode=mode)
    assert all(p["used_tensor_core_kernel"] in (1, 3) for p in plans), plans
    _gate_bf16(o, l, o_ref, l_ref, a_ref, f"{label} [{mode}]")


def test_text_causal_differs_from_block_causal_and_needs_tags():
    """The flag changes the result (a text row loses its later text keys), and is refused without tags."""
    import torch
    from paper_2606_25041_b200 import WS_ATTN_TEXT_CAUSAL, WsError
    o, l, o_ref, l_ref, a_ref, _ = _text_causal_case("bf16", 4, 2, 128, 64, [128], [96], seed=5, mode="two_calls", p_text=0.5)
    # same inputs, plain block-causal oracle: must NOT match within the tolerance
    from oracle.block_causal import OracleSession, attend
    rng = np.random.default_rng(5)
    kk, vv, tg = _mk(rng, "bf16", 128, 2, 128), _mk(rng, "bf16", 128, 2, 128), _tags(rng, 128, 0.5)
    sess = OracleSession(2, 128); sess.append(kk, vv)
    qq, kk2, vv2 = _mk(rng, "bf16", 96, 4, 128), _mk(rng, "bf16", 96, 2, 128), _mk(rng, "bf16", 96, 2, 128)
    sess.append(kk2, vv2)
    o_bc, _ = attend(sess, qq, 1.0 / math.sqrt(128), 1)
    assert np.abs(o - o_bc).max() > 3e-2
    dev = torch.device("cuda", 0)
    c = _cache("bf16", 4, 2, 128, 64, 256)
    sid = c.session_open()
    c.kv_append([sid], [0, 96], _torch_of(kk2, dev), _torch_of(vv2, dev))              # no tags
    out = torch.empty((96, 4, 128), dtype=torch.bfloat16, device=dev)
    with pytest.raises(WsError) as e:
        c.block_causal_attn_fwd([sid], [0, 96], _torch_of(qq, dev), out, 0.1, attn_flags=WS_ATTN_TEXT_CAUSAL)
    assert e.value.status_name == "WS_ERR_INVALID_ARG"
    with pytest.raises(WsError):
        c.block_causal_attn_fwd([sid], [0, 96], _torch_of(qq, dev), out, 0.1, attn_flags=2)


@pytest.mark.parametrize("splits", [1, 3, 9])
def test_text_causal_split_kv_and_decode_plan(splits):
    """Split-KV invariance with the mixed mask on both plans: a split whose tiles a text row cannot see at all
    publishes an empty partial (LSE = -inf)."""
    for n, Hq, Hkv in ((16, 8, 2), (256, 8, 2)):                       # decode plan (64 packed rows) / general plan
        o, l, o_ref, l_ref, a_ref, plans = _text_causal_case("bf16", Hq, Hkv, 128, 64, [256, 256, 130], [n, n], seed=40 + n,
                                                             mode="two_calls", min_splits=splits, p_text=0.6)
        assert plans[-1]["used_tensor_core_kernel"] == (3 if n == 16 else 1)
        nt = (642 + 2 * n + 127) // 128                               # KV tiles of the last step
        per = -(-nt // splits)                                        # planner: tiles per forced piece
        assert plans[-1]["num_segments"] >= Hkv * -(-nt // per)
        _gate_bf16(o, l, o_ref, l_ref, a_ref, f"n={n} splits={splits}")


def test_text_causal_all_text_token_causal_decode_in_one_block():
    """All slots text: a whole block decodes token-causally in ONE block (the thinker's text pass),
    fused step on the decode plan."""
    o, l, o_ref, l_ref, a_ref, plans = _text_causal_case("bf16", 32, 8, 128, 64, [256, 100], [16, 16, 16], seed=77,
                                                         mode="fused", p_text=1.1)
    assert all(p["used_tensor_core_kernel"] == 3 for p in plans)
    _gate_bf16(o, l, o_ref, l_ref, a_ref, "all-text decode")


@pytest.mark.parametrize("mode", ["two_calls", "one_shot"])
def test_text_causal_generic_fp32_kernel(mode):
    """Config-1 geometry (fp32, D = 64, 16-token pages, units of 16 tokens = 8 video + 6 audio + 2 text slots and
    denser text mixes) on the CUDA-core kernel, 1e-5."""
    o, l, o_ref, l_ref, _, plans = _text_causal_case("fp32", 2, 2, 64, 16, [16], [16, 16, 40], seed=3, mode=mode, p_text=0.4)
    assert all(p["used_tensor_core_kernel"] == 0 for p in plans)
    d = np.abs(o - o_ref)
    print(f"[parity] text-causal fp32 [{mode}]: max_abs={d.max():.3e} lse_max={np.abs(l - l_ref).max():.3e}")
    assert d.max() <= 1e-5 and np.abs(l - l_ref).max() <= 1e-5


def test_text_causal_bf16_generic_kernel():
    from paper_2606_25041_b200 import WS_FLAG_FORCE_SIMT
    o, l, o_ref, l_ref, a_ref, plans = _text_causal_case("bf16", 4, 2, 128, 64, [100], [70, 70], seed=9, mode="two_calls",
                                                         flags=WS_FLAG_FORCE_SIMT)
    assert all(p["used_tensor_core_kernel"] == 0 for p in plans)
    _gate_bf16(o, l, o_ref, l_ref, a_ref, "bf16 generic kernel")


# ------------------------------------------------------------------------------------------ generic kernel, fused step
def test_generic_kernel_fused_step_config1_and_bf16():
    """ws_stream_step on the generic (CUDA-core) path is ONE launch as well: the attention blocks read the new
    block's keys from k_new / v_new, extra blocks of the same grid commit it.  Config 1 (fp32, 1e-5) and a bf16
    case forced onto the generic kernel; append bit-exact; one launch per step."""
    from paper_2606_25041_b200 import WS_FLAG_FORCE_SIMT
    from synth_inputs import generate, spec_for_config
    from tests.gpu_harness import compare, run_workload_gpu, run_workload_oracle
    w = generate(spec_for_config(1))
    ref = run_workload_oracle(w)
    got = run_workload_gpu(w, fused_step=True, pool_fill=0x7FC00001)
    err = compare(got, ref, "fp32")
    print("[parity] config 1, fused generic step:", {k: v for k, v in err.items()})
    assert err["finite"] and err["max_abs"] <= 1e-5 and err["lse_max"] <= 1e-5 and err["kv_bit_exact"]
    two = run_workload_gpu(w, fused_step=False)
    assert got["launches"] == two["launches"] - w.spec.steps            # one launch fewer per step
    wb = generate(spec_for_config(2, cache_lens=(333,), num_q_heads=4, num_kv_heads=2, block_tokens=40,
                                  modality_split=(30, 8, 2), steps=3))
    refb = run_workload_oracle(wb)
    gotb = run_workload_gpu(wb, flags=WS_FLAG_FORCE_SIMT, fused_step=True, pool_fill=0x7FC1)
    errb = compare(gotb, refb, "bf16")
    print("[parity] bf16 generic kernel, fused step:", {k: v for k, v in errb.items()})
    assert not gotb["tensor"]
    assert errb["finite"] and errb["max_abs"] <= 1e-2 and errb["mean_abs"] <= 1e-3 and errb["bound_viol"] <= 0
    assert errb["lse_max"] <= 1e-4 and errb["kv_bit_exact"]


def test_text_causal_generic_fp32_fused_step():
    o, l, o_ref, l_ref, _, plans = _text_causal_case("fp32", 2, 2, 64, 16, [16], [16, 16, 40], seed=4, mode="fused", p_text=0.4)
    assert all(p["used_tensor_core_kernel"] == 0 for p in plans)
    assert np.abs(o - o_ref).max() <= 1e-5 and np.abs(l - l_ref).max() <= 1e-5


@pytest.mark.parametrize("n", [4, 64], ids=["decode_kernel", "general_plan"])
def test_text_causal_ragged_multi_session_batch(n):
    """Three sessions with different history lengths in ONE fused call, text-causal mixed mask, each session's
    block with its own tag pattern (the text-bit records are per session); vs the oracle."""
    import torch
    from oracle.block_causal import OracleSession, attend
    from paper_2606_25041_b200 import WS_ATTN_TEXT_CAUSAL
    rng = np.random.default_rng(90 + n)
    dev = torch.device("cuda", 0)
    Hq, Hkv, D = 8, 2, 128
    lens = [300, 1000, 77]
    c = _cache("bf16", Hq, Hkv, D, 64, max(lens) + 4 * n + 64, sessions=3, max_q=max(lens))
    ids = [c.session_open() for _ in lens]
    sess = [OracleSession(Hkv, D) for _ in lens]
    for s, L in enumerate(lens):
        kk, vv, tg = _mk(rng, "bf16", L, Hkv, D), _mk(rng, "bf16", L, Hkv, D), _tags(rng, L)
        c.kv_append([ids[s]], [0, L], _torch_of(kk, dev), _torch_of(vv, dev), modality=tg)
        sess[s].append(kk, vv, modality=tg)
    scale = 1.0 / math.sqrt(D)
    for step in range(2):
        qs, ks, vs, tgs = [], [], [], []
        for s in range(3):
            qs.append(_mk(rng, "bf16", n, Hq, D)); ks.append(_mk(rng, "bf16", n, Hkv, D)); vs.append(_mk(rng, "bf16", n, Hkv, D))
            tgs.append(_tags(rng, n, 0.5))
            sess[s].append(ks[-1], vs[-1], modality=tgs[-1])
        out = torch.full((3 * n, Hq, D), float("nan"), dtype=torch.bfloat16, device=dev)
        lse = torch.full((3 * n, Hq), float("nan"), dtype=torch.float32, device=dev)
        c.stream_step(ids, [0, n, 2 * n, 3 * n], _torch_of(np.concatenate(qs), dev), _torch_of(np.concatenate(ks), dev),
                      _torch_of(np.concatenate(vs), dev), out, scale, lse=lse, modality=np.concatenate(tgs),
                      attn_flags=WS_ATTN_TEXT_CAUSAL)
        torch.cuda.synchronize()
        assert c.last_plan_info()["used_tensor_core_kernel"] == (3 if n == 4 else 1)
        o = out.float().cpu().numpy().astype(np.float64); l = lse.cpu().numpy().astype(np.float64)
        refs = [attend(sess[s], qs[s], scale, 1, want_abs=True, text_causal=True) for s in range(3)]
        o_ref, l_ref, a_ref = (np.concatenate([r[i] for r in refs]) for i in range(3))
        _gate_bf16(o, l, o_ref, l_ref, a_ref, f"ragged 3-session batch n={n} step {step}")


def _tc_fuzz_cases():
    rng = np.random.default_rng([2606, 25041, 4])
    out = []
    for i in range(16):
        Hkv = int(rng.choice([1, 2, 4]))
        G = int(rng.choice([1, 2, 4, 8]))
        hist = [int(x) for x in rng.integers(1, 400, size=int(rng.integers(0, 4)))]
        qb = [int(x) for x in rng.choice([1, 2, 7, 16, 33, 64, 100, 130, 257], size=int(rng.integers(1, 4)))]
        out.append(dict(idx=i, Hq=Hkv * G, Hkv=Hkv, hist=hist, qb=qb, mode=["two_calls", "fused", "one_shot"][i % 3],
                        splits=int(rng.choice([0, 0, 2, 4])), p_text=float(rng.choice([0.1, 0.3, 0.6, 1.0]))))
    return out


@pytest.mark.parametrize("case", _tc_fuzz_cases(), ids=lambda c: f"{c['idx']}_{c['mode']}_h{c['Hkv']}x{c['Hq'] // c['Hkv']}")
def test_text_causal_random_shapes(case):
    """Seeded random shapes of the mixed mask (block sizes from one token to more than a Q tile pair, histories that
    end mid-page and mid-tile, text share 10 % - 100 %, forced splits, the three call modes) against the oracle."""
    o, l, o_ref, l_ref, a_ref, plans = _text_causal_case("bf16", case["Hq"], case["Hkv"], 128, 64, case["hist"], case["qb"],
                                                         seed=1000 + case["idx"], mode=case["mode"],
                                                         min_splits=case["splits"], p_text=case["p_text"])
    assert all(p["used_tensor_core_kernel"] in (1, 3) for p in plans), plans
    _gate_bf16(o, l, o_ref, l_ref, a_ref, f"fuzz {case}")


# ------------------------------------------------------------------------------------------ host-buffer step, ragged units
def test_stream_step_host_ragged_units_back_to_back():
    """ws_stream_step_host with units of DIFFERENT sizes enqueued back to back (no host sync, copies of step t
    overlap the kernels of its neighbours through the two staging slots): every step's host result matches the
    oracle and the cache ends bit-exact.  The slot stride is fixed by the staging buffer, not by a step's token
    count, so a small step after a large one cannot land inside the region the large one still uses."""
    import torch
    from oracle.block_causal import OracleSession, attend
    rng = np.random.default_rng(2025)
    dev = torch.device("cuda", 0)
    Hq, Hkv, D = 8, 2, 128
    units = [256, 40, 200, 7, 256, 1, 130, 64]
    L0 = 700
    c = _cache("bf16", Hq, Hkv, D, 64, L0 + sum(units), max_q=1024)
    sid = c.session_open()
    sess = OracleSession(Hkv, D)
    k0, v0 = _mk(rng, "bf16", L0, Hkv, D), _mk(rng, "bf16", L0, Hkv, D)
    c.kv_append([sid], [0, L0], _torch_of(k0, dev), _torch_of(v0, dev))
    sess.append(k0, v0)
    pin = lambda a: torch.from_numpy(a.view(np.uint16).copy()).view(torch.bfloat16).pin_memory()
    staging = torch.empty(c.step_staging_bytes(max(units)), dtype=torch.uint8, device=dev)
    scale = 1.0 / math.sqrt(D)
    host, refs = [], []
    for n in units:
        q, k, v = _mk(rng, "bf16", n, Hq, D), _mk(rng, "bf16", n, Hkv, D), _mk(rng, "bf16", n, Hkv, D)
        sess.append(k, v)
        refs.append(attend(sess, q, scale, 1, want_abs=True))
        host.append((pin(q), pin(k), pin(v), torch.full((n, Hq, D), float("nan"), dtype=torch.bfloat16).pin_memory()))
    torch.cuda.synchronize()
    for n, (qh, kh, vh, oh) in zip(units, host):
        c.stream_step_host([sid], [0, n], qh, kh, vh, oh, staging, scale)       # no sync between steps
    c.stream_host_join()
    torch.cuda.synchronize()
    for i, (n, (qh, kh, vh, oh), (o_ref, l_ref, a_ref)) in enumerate(zip(units, host, refs)):
        o = oh.float().numpy().astype(np.float64)
        d = o - o_ref
        viol = (np.abs(d) - bf16_error_bound(o_ref, o, a_ref)).max()
        print(f"[parity] host step {i} n={n}: max_abs={np.abs(d).max():.3e} mean_abs={np.abs(d).mean():.3e} bound_viol={viol:.3e}")
        assert np.isfinite(o).all()
        assert np.abs(d).max() <= 1e-2 and np.abs(d).mean() <= 1e-3 and viol <= 0
    T = c.session_info(sid)[0]
    assert T == L0 + sum(units)
    kg = torch.empty((T, Hkv, D), dtype=torch.bfloat16, device=dev); vg = torch.empty_like(kg)
    c.kv_gather(sid, 0, T, kg, vg)
    torch.cuda.synchronize()
    k_all = np.concatenate([k0] + [_numpy_of(h[1]) for h in host]); v_all = np.concatenate([v0] + [_numpy_of(h[2]) for h in host])
    assert np.array_equal(_numpy_of(kg).view(np.uint16), k_all.view(np.uint16))
    assert np.array_equal(_numpy_of(vg).view(np.uint16), v_all.view(np.uint16))


# ------------------------------------------------------------------------------------------ generic kernel, shape space
def _generic_cases():
    rng = np.random.default_rng([2606, 25041, 31])
    out = []
    for i in range(32):
        Hkv = int(rng.choice([1, 2, 3, 4])); G = int(rng.choice([1, 2, 3, 4, 8]))
        D = int(rng.choice([8, 16, 24, 32, 40, 64, 72, 96, 128, 160, 192, 256])); P = int(rng.choice([1, 4, 16, 32, 64, 128]))
        hist = [int(x) for x in rng.integers(1, 300, size=int(rng.integers(1, 4)))]
        qb = [int(x) for x in rng.choice([1, 2, 3, 7, 16, 33, 64, 100], size=int(rng.integers(1, 4)))]
        out.append(dict(idx=i, dt="fp32" if i % 3 else "bf16", Hq=Hkv * G, Hkv=Hkv, D=D, P=P, hist=hist, qb=qb,
                        mode=["two_calls", "fused", "one_shot"][i % 3 if i % 2 else (i // 2) % 3],
                        p_text=float(rng.choice([0.0, 0.3, 1.0]))))
    return out


@pytest.mark.parametrize("case", _generic_cases(), ids=lambda c: f"{c['idx']}_{c['dt']}_D{c['D']}_P{c['P']}_{c['mode']}")
def test_generic_kernel_shape_space(case):
    """The CUDA-core kernel over its own shape space (head_dim 8-256, pages of 1-128 tokens, group sizes incl. 3, both
    dtypes, the three call modes, text share 0-100 %): fp32 within the 1e-5 contract, bf16 within the bf16 gates."""
    from paper_2606_25041_b200 import WS_FLAG_FORCE_SIMT
    o, l, o_ref, l_ref, a_ref, plans = _text_causal_case(case["dt"], case["Hq"], case["Hkv"], case["D"], case["P"], case["hist"],
                                                         case["qb"], seed=3000 + case["idx"], mode=case["mode"],
                                                         p_text=case["p_text"], flags=WS_FLAG_FORCE_SIMT)
    assert all(p["used_tensor_core_kernel"] == 0 for p in plans)
    if case["dt"] == "fp32":
        print(f"[parity] generic fp32 {case}: max_abs={np.abs(o - o_ref).max():.3e} lse_max={np.abs(l - l_ref).max():.3e}")
        assert np.isfinite(o).all() and np.abs(o - o_ref).max() <= 1e-5 and np.abs(l - l_ref).max() <= 1e-5
    else:
        _gate_bf16(o, l, o_ref, l_ref, a_ref, f"generic bf16 {case}")

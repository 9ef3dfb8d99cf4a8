"""NEXT-3 on the GPU: the thinker -> performer KV-slice exchange.

The owner's kv_append kernel stores every slice into its own pool AND into each linked replica pool
(plain 16-byte stores through the peer mapping); the replica adopts pages / block boundaries from the
commit message.  The box has one GPU, so the "peer" pool lives on the same device - once in the same
process, once in ANOTHER process through the CUDA IPC mapping (the mapping a second GPU would use); the
kernels never wait on one another (the replica acts only after the owner's stream has been synchronised
and the message has arrived).  Checked: replica history bit-exact, replica attention == oracle and
bit-identical to the owner's, solver-step staging on the replica between units, snapshot broadcast."""
import os
import sys

import numpy as np
import pytest

from synth_inputs import generate, spec_for_config, to_bf16
from tests.gpu_harness import _numpy_of, _torch_of

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
Hq, Hkv, D, P = 16, 4, 128, 64
SCALE = 1.0 / np.sqrt(128.0)


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as entry
    entry.build()


def _cache(num_pages, pool_fill=None):
    from paper_2606_25041_b200 import WS_BF16, Cache
    return Cache(WS_BF16, Hq, Hkv, D, P, num_pages=num_pages, max_sessions=3, max_pages_per_session=40,
                 max_blocks_per_session=64, max_q_tokens_per_call=1024, pool_fill=pool_fill)


def _units(seed, sizes):
    rng = np.random.default_rng(seed)
    return [tuple(to_bf16(rng.standard_normal(sh, dtype=np.float32))
                  for sh in ((n, Hq, D), (n, Hkv, D), (n, Hkv, D))) for n in sizes]


def _attend(cache, s, q, dev):
    import torch
    n = q.shape[0]
    out = torch.full((n, Hq, D), float("nan"), dtype=torch.bfloat16, device=dev)
    lse = torch.full((n, Hq), float("nan"), dtype=torch.float32, device=dev)
    cache.block_causal_attn_fwd([s], [0, n], _torch_of(q, dev), out, SCALE, lse=lse)
    torch.cuda.synchronize()
    return out, lse


def _gather(cache, s, dev):
    import torch
    tokens = cache.session_info(s)[0]
    kg = torch.empty((tokens, Hkv, D), dtype=torch.bfloat16, device=dev); vg = torch.empty_like(kg)
    cache.kv_gather(s, 0, tokens, kg, vg)
    torch.cuda.synchronize()
    return _numpy_of(kg).tobytes(), _numpy_of(vg).tobytes()


def test_mirrored_append_same_process_replica_matches_owner_and_oracle():
    import torch
    from oracle.block_causal import OracleSession, attend
    dev = torch.device("cuda", 0)
    canary = 0x7B7B
    owner, rep = _cache(40), _cache(56, pool_fill=canary)
    rep.replica_accept(40)
    owner.replica_link([rep])
    owner.shuffle_free_pages(3)
    s = owner.session_open()
    ora = OracleSession(Hkv, D)
    sizes = [256, 100, 37, 256, 1, 192]                       # page-aligned and mid-page commits
    for i, (q, k, v) in enumerate(_units(11, sizes)):
        n = q.shape[0]
        owner.kv_append([s], [0, n], _torch_of(k, dev), _torch_of(v, dev))
        torch.cuda.synchronize()                               # ordering contract: slice complete, then the message
        rep.replica_apply(owner.replica_commit_message())
        ora.append(k, v)
        o_own, l_own = _attend(owner, s, q, dev)
        o_rep, l_rep = _attend(rep, s, q, dev)
        assert torch.equal(o_own, o_rep) and torch.equal(l_own, l_rep), i       # same kernel, same plan, same bytes
        o_ref, l_ref = attend(ora, q, SCALE)
        d = o_rep.float().cpu().numpy() - o_ref
        assert np.abs(d).max() <= 1e-2 and np.abs(d).mean() <= 1e-3, i
        assert np.abs(l_rep.cpu().numpy() - l_ref).max() <= 1e-3, i
        if i in (1, 3):
            # performer solver staging between units: local pages, rolled back before the next slice
            keep = rep.session_info(s)[1]
            (qn, kn, vn), = _units(100 + i, [128])
            rep.kv_append([s], [0, 128], _torch_of(kn, dev), _torch_of(vn, dev))
            assert all(p >= 40 for p in rep.session_pages(s)[len(owner.session_pages(s)):])
            trial = OracleSession(Hkv, D)
            trial.k_slices, trial.v_slices, trial.block_ends = list(ora.k_slices), list(ora.v_slices), list(ora.block_ends)
            trial.append(kn, vn)
            o_st, _ = _attend(rep, s, qn, dev)
            o_ref, _ = attend(trial, qn, SCALE)
            assert np.abs(o_st.float().cpu().numpy() - o_ref).max() <= 1e-2
            rep.session_truncate(s, keep)
    kr, vr = ora.gather()
    want = (np.ascontiguousarray(kr).tobytes(), np.ascontiguousarray(vr).tobytes())
    assert _gather(owner, s, dev) == want and _gather(rep, s, dev) == want
    assert rep.session_info(s) == owner.session_info(s) and rep.session_pages(s) == owner.session_pages(s)
    # owner pages the owner never named still hold the canary in the replica's pool (K and V)
    used = set(owner.session_pages(s))
    kp = rep.k_pool.view(torch.int16).cpu().numpy().view(np.uint16)
    for pg in range(40):
        if pg not in used:
            assert (kp[pg] == canary).all(), pg


def test_snapshot_push_is_the_initial_cache_broadcast_two_replicas():
    import torch
    dev = torch.device("cuda", 0)
    owner, r1, r2 = _cache(40), _cache(40), _cache(48)
    for r in (r1, r2):
        r.replica_accept(40)
    s = owner.session_open()
    units = _units(21, [256, 256, 90])
    for q, k, v in units:                                     # system prefill before any link exists
        owner.kv_append([s], [0, k.shape[0]], _torch_of(k, dev), _torch_of(v, dev))
    owner.replica_link([r1, r2])
    owner.replica_push_session(s)
    torch.cuda.synchronize()
    snap = owner.replica_snapshot_message(s)
    for r in (r1, r2):
        r.replica_apply(snap)
        assert _gather(r, s, dev) == _gather(owner, s, dev)
        assert r.session_info(s) == owner.session_info(s)
    # streaming continues: one mirrored append reaches both replicas
    (q, k, v), = _units(22, [256])
    owner.kv_append([s], [0, 256], _torch_of(k, dev), _torch_of(v, dev))
    torch.cuda.synchronize()
    msg = owner.replica_commit_message()
    o_own, _ = _attend(owner, s, q, dev)
    for r in (r1, r2):
        r.replica_apply(msg)
        o, _ = _attend(r, s, q, dev)
        assert torch.equal(o, o_own)
    owner.replica_link([])                                    # unlink: later appends stay local
    owner.kv_append([s], [0, 64], _torch_of(k[:64], dev), _torch_of(v[:64], dev))
    torch.cuda.synchronize()
    assert r1.session_info(s)[0] == owner.session_info(s)[0] - 64


def _performer(conn):
    """Replica process: owns its pools, exports them over CUDA IPC, applies messages, attends."""
    sys.path.insert(0, ROOT)
    import torch
    from oracle.block_causal import OracleSession, attend
    from paper_2606_25041_b200 import ws_ipc_export
    dev = torch.device("cuda", 0)
    try:
        rep = _cache(56)
        rep.replica_accept(40)
        conn.send((ws_ipc_export(rep.k_pool), ws_ipc_export(rep.v_pool), rep.pool_bytes()))
        ora = OracleSession(Hkv, D)
        worst = 0.0
        for q, k, v in _units(31, [256, 70, 256]):            # same seeded inputs as the owner process
            msg = conn.recv()                                 # sent only after the owner synchronised its stream
            rep.replica_apply(msg)
            ora.append(k, v)
            o, _ = _attend(rep, 0, q, dev)
            o_ref, _ = attend(ora, q, SCALE)
            worst = max(worst, float(np.abs(o.float().cpu().numpy() - o_ref).max()))
        kr, vr = ora.gather()
        ok = _gather(rep, 0, dev) == (np.ascontiguousarray(kr).tobytes(), np.ascontiguousarray(vr).tobytes())
        conn.send(("done", worst, ok))
        conn.recv()                                           # keep the pools alive until the owner has unmapped them
    except Exception as e:                                    # noqa: BLE001
        conn.send(("error", repr(e), False))


def test_slice_exchange_across_processes_through_cuda_ipc():
    import torch
    import torch.multiprocessing as mp
    from paper_2606_25041_b200 import ws_ipc_close, ws_ipc_open
    dev = torch.device("cuda", 0)
    ctx = mp.get_context("spawn")
    here, there = ctx.Pipe()
    proc = ctx.Process(target=_performer, args=(there,))
    proc.start()
    try:
        assert here.poll(180), "performer did not come up"
        first = here.recv()
        assert first[0] != "error", first
        (kh, koff), (vh, voff), nbytes = first
        kp, vp = ws_ipc_open(kh, koff, 0), ws_ipc_open(vh, voff, 0)
        owner = _cache(40)
        owner.replica_link([(kp, vp, nbytes)])
        s = owner.session_open()
        for q, k, v in _units(31, [256, 70, 256]):
            owner.kv_append([s], [0, k.shape[0]], _torch_of(k, dev), _torch_of(v, dev))
            torch.cuda.synchronize()
            here.send(owner.replica_commit_message())
        assert here.poll(180), "performer did not finish"
        tag, worst, ok = here.recv()
        assert tag == "done", worst
        assert worst <= 1e-2 and ok
        owner.replica_link([])
        ws_ipc_close(kp, koff); ws_ipc_close(vp, voff)
        here.send("bye")
        proc.join(timeout=60)
        assert proc.exitcode == 0
    finally:
        if proc.is_alive():
            proc.kill()

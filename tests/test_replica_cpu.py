"""NEXT-3 host logic on CPU (dry-run caches): the thinker -> performer KV-slice exchange.

The owner's ws_kv_append produces a commit message; the replica adopts the named pages and block
boundaries with ws_replica_apply.  Checked here: replicas stay identical (tokens, block ends, page ids),
page ownership (owner pages vs the replica's own staging pages), the initial-cache snapshot message,
and every rejection path with the strong guarantee.  The gloo test carries the messages between two
processes with torch.distributed send/recv - the transport the real two-GPU path uses."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import __graft_entry__ as entry

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    entry.build()
    import paper_2606_25041_b200 as p
    return p


def _dry(pkg, num_pages, **kw):
    args = dict(dtype=pkg.WS_BF16, num_q_heads=32, num_kv_heads=8, head_dim=128, page_tokens=64,
                num_pages=num_pages, max_sessions=4, max_pages_per_session=64, max_blocks_per_session=32,
                max_sessions_per_call=4, max_q_tokens_per_call=2048, flags=pkg.WS_FLAG_DRY_RUN)
    args.update(kw)
    return pkg.Cache(**args)


def _state(c, s):
    return c.session_info(s), c.session_pages(s)


def test_commit_messages_keep_replica_identical_and_staging_uses_local_pages(pkg):
    owner, rep = _dry(pkg, 48), _dry(pkg, 64)
    rep.replica_accept(48)
    assert rep.free_pages() == 16                      # only the replica's own pages are locally allocatable
    owner.replica_link([rep])
    owner.shuffle_free_pages(7)                        # arbitrary physical assignment on the owner
    a, b = owner.session_open(), owner.session_open()
    for step, (ids, cu) in enumerate([([a], [0, 100]), ([b, a], [0, 64, 64 + 29]), ([a, b], [0, 256, 256 + 7])]):
        owner.kv_append(ids, cu, None, None)
        msg = owner.replica_commit_message()
        assert msg[0] == 0x57534B56 and msg[2] == 1 and msg[3] == len(ids) and msg[4] == len(msg)
        rep.replica_apply(msg)
        for s in ids:
            assert _state(rep, s) == _state(owner, s)
    assert rep.free_pages() == 16
    # performer-side solver staging (NEXT-2): an uncommitted block lands in LOCAL pages (ids >= 48) ...
    rep.kv_append([b], [0, 200], None, None)
    staged = rep.session_pages(b)[len(owner.session_pages(b)):]
    assert staged and all(p >= 48 for p in staged)
    # ... and must be rolled back before the next slice of that session can be applied
    owner.kv_append([b], [0, 64], None, None)
    msg = owner.replica_commit_message()
    before = _state(rep, b)
    with pytest.raises(pkg.WsError) as e:
        rep.replica_apply(msg)
    assert e.value.status_name == "WS_ERR_INVALID_ARG" and "rolled back" in str(e.value)
    assert _state(rep, b) == before
    rep.session_truncate(b, rep.session_info(b)[1] - 1)
    assert rep.free_pages() == 16
    rep.replica_apply(msg)
    assert _state(rep, b) == _state(owner, b)
    # closing on the replica returns adopted pages to the OWNER range, not to the local free list
    rep.session_close(b)
    assert rep.free_pages() == 16


def test_snapshot_message_is_the_initial_cache_broadcast(pkg):
    owner, rep = _dry(pkg, 48), _dry(pkg, 48)
    rep.replica_accept(48)
    s = owner.session_open()
    for n in (256, 256, 100, 1):                       # system prefill: several blocks before the link exists
        owner.kv_append([s], [0, n], None, None)
    owner.replica_link([rep])
    owner.replica_push_session(s)                      # dry run: host checks only
    msg = owner.replica_snapshot_message(s)
    assert msg[2] == 2 and msg[3] == 1
    rep.replica_apply(msg)
    assert _state(rep, s) == _state(owner, s) == ((613, 4, [256, 512, 612, 613]), owner.session_pages(s))
    with pytest.raises(pkg.WsError):                   # applying it twice: replica is no longer at length 0
        rep.replica_apply(msg)
    # streaming continues with per-unit commits
    owner.kv_append([s], [0, 256], None, None)
    rep.replica_apply(owner.replica_commit_message())
    assert _state(rep, s) == _state(owner, s)


def test_apply_rejects_bad_messages_without_changing_state(pkg):
    owner, rep = _dry(pkg, 48), _dry(pkg, 64)
    rep.replica_accept(40)                             # fewer pages accepted than the owner may name
    s = owner.session_open()
    owner.kv_append([s], [0, 64 * 3], None, None)      # owner pages 0, 1, 2
    good = owner.replica_commit_message()

    def rejected(words, status):
        free = rep.free_pages()
        with pytest.raises(pkg.WsError) as e:
            rep.replica_apply(words)
        assert e.value.status_name == status, str(e.value)
        assert rep.free_pages() == free
        with pytest.raises(pkg.WsError):
            rep.session_info(s)                        # still not open

    m = good.copy(); m[0] ^= 1; rejected(m, "WS_ERR_INVALID_ARG")            # magic
    m = good.copy(); m[1] = 99; rejected(m, "WS_ERR_UNSUPPORTED")            # version
    rejected(good[:-1], "WS_ERR_INVALID_ARG")                                # truncated
    m = good.copy(); m[7] = 64; rejected(m, "WS_ERR_INVALID_ARG")            # head_dim differs
    m = good.copy(); m[-1] = 45; rejected(m, "WS_ERR_OUT_OF_PAGES")          # page outside the accepted range
    m = good.copy(); m[-1] = m[-2]; rejected(m, "WS_ERR_INVALID_ARG")        # page named twice
    m = good.copy(); m[9 + 1] = 64; rejected(m, "WS_ERR_INVALID_ARG")        # continues from a length we do not hold
    m = good.copy(); m[9 + 4] = 64 * 3 + 1; rejected(m, "WS_ERR_INVALID_ARG")  # block needs 4 pages, 3 named
    rep.replica_apply(good)
    assert _state(rep, s) == _state(owner, s)
    # the same pages cannot be adopted by another session
    m = good.copy(); m[9] = 1
    with pytest.raises(pkg.WsError) as e:
        rep.replica_apply(m)
    assert e.value.status_name == "WS_ERR_OUT_OF_PAGES"
    # link-side checks
    with pytest.raises(pkg.WsError):
        owner.replica_link([_dry(pkg, 8)])             # peer pool smaller than the owner's
    with pytest.raises(pkg.WsError):
        rep.replica_accept(10)                         # a session is open
    with pytest.raises(pkg.WsError):
        _dry(pkg, 8).replica_commit_message()          # nothing appended yet
    with pytest.raises(pkg.WsError):
        _dry(pkg, 8).replica_push_session(0)


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2606_25041_b200 as pkg
    units = [256, 256, 130, 256, 1, 256]
    if rank == 0:      # thinker: owns the page assignment, streams one commit message per unit
        c = _dry(pkg, 48)
        c.replica_link([(None, None, c.pool_bytes())])
        s = c.session_open()
        c.kv_append([s], [0, 512], None, None)                         # system prefill ...
        snap = torch.from_numpy(c.replica_snapshot_message(s))          # ... broadcast as a snapshot
        dist.send(torch.tensor([len(snap)]), dst=1); dist.send(snap, dst=1)
        for n in units:
            c.kv_append([s], [0, n], None, None)
            m = torch.from_numpy(c.replica_commit_message())
            dist.send(torch.tensor([len(m)]), dst=1); dist.send(m, dst=1)
    else:              # performer: adopts, stages a solver block between units, rolls it back
        c = _dry(pkg, 64)
        c.replica_accept(48)
        s = 0
        for i in range(1 + len(units)):
            n = torch.zeros(1, dtype=torch.int64); dist.recv(n, src=0)
            m = torch.zeros(int(n), dtype=torch.int32); dist.recv(m, src=0)
            c.replica_apply(m.numpy())
            keep = c.session_info(s)[1]
            c.kv_append([s], [0, 256], None, None)                     # noisy block attends ... (dry run)
            c.block_causal_attn_fwd([s], [0, 256], None, None, 0.088)
            c.session_truncate(s, keep)                                # ... and is rolled back
    dist.barrier()
    q.put((rank, c.session_info(s), c.session_pages(s), c.free_pages()))
    dist.destroy_process_group()


def test_two_rank_slice_exchange_gloo(pkg):
    port = 31500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, info0, pages0, free0), (_, info1, pages1, free1) = res
    assert info0 == info1 and pages0 == pages1
    assert info0[0] == 512 + 256 + 256 + 130 + 256 + 1 + 256 and info0[1] == 7
    assert free0 == 48 - len(pages0) and free1 == 16

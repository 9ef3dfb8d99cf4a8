"""N > 1 host logic on CPU: world size 2 over gloo.  The path shards by session with no data-path
collective: every rank owns its own cache + sessions; the only cross-rank steps
are the barrier and the max-time / sum-work reduction used by bench.py."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import __graft_entry__ as entry
    entry.build()
    import paper_2606_25041_b200 as pkg
    from bench import aggregate_over_ranks
    # each rank: its own dry-run cache and session (different lengths per rank), its own plan
    c = pkg.Cache(pkg.WS_BF16, 32, 8, 128, 64, num_pages=600, max_sessions=2, max_pages_per_session=300,
                  max_q_tokens_per_call=2048, flags=pkg.WS_FLAG_DRY_RUN)
    s = c.session_open()
    L = 4096 * (rank + 1)
    pos = 0
    while pos < L:
        c.kv_append([s], [0, 2048], None, None); pos += 2048
    c.kv_append([s], [0, 256], None, None)
    c.block_causal_attn_fwd([s], [0, 256], None, None, 0.088)
    info = c.last_plan_info()
    tokens = c.session_info(s)[0]
    flops = 4.0 * 128 * 32 * 256 * tokens
    ms, total = aggregate_over_ranks(10.0 * (rank + 1), flops, dist, torch.device("cpu"))
    dist.barrier()
    q.put((rank, tokens, info["total_kv_tiles"], info["num_ctas"], ms, total))
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    port = 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, tiles0, ctas0, ms0, tot0), (r1, t1, tiles1, ctas1, ms1, tot1) = res
    assert (t0, t1) == (4096 + 256, 8192 + 256)                    # sessions are rank-private
    assert tiles0 == 8 * 34 and tiles1 == 8 * 66 and 128 <= ctas0 <= 148 and 128 <= ctas1 <= 148
    assert ms0 == ms1 == 20.0                                      # MAX over ranks
    want = 4.0 * 128 * 32 * 256 * (t0 + t1)
    assert tot0 == tot1 == pytest.approx(want)                     # SUM over ranks


def test_bench_gpus_n_spawns_its_own_ranks():
    """`python bench.py --gpus 2` with no launcher (WORLD_SIZE unset) re-executes itself under
    torch.distributed.run with 2 ranks; --selftest-cpu runs the rendezvous / barrier / max-and-sum-over-ranks
    plumbing on gloo with made-up per-rank timings (rank r: 10 + r ms, 1e12 flops) and rank 0 prints one line."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-cpu"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["selftest"] and d["n_gpus"] == 2
    assert d["ms_max_over_ranks"] == 11.0 and d["flops_sum_over_ranks"] == 2e12

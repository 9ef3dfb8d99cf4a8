"""CPU-only tests of the C-ABI library: it loads, exports every symbol include/ws.h declares, and its
host logic (page allocator, block boundaries, error paths with the strong guarantee, the split-KV
planner) behaves - all under WS_FLAG_DRY_RUN, i.e. without a single CUDA call."""
import os
import re

import numpy as np
import pytest

import __graft_entry__ as entry

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    entry.build()
    import paper_2606_25041_b200 as p
    return p


def test_library_exports_every_declared_symbol(pkg):
    import ctypes
    hdr = open(os.path.join(ROOT, "include", "ws.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ws_[a-z_0-9]+)\s*\(", hdr))
    assert {"ws_kv_append", "ws_block_causal_attn_fwd", "ws_cache_create", "ws_kv_gather"} <= declared
    lib = ctypes.CDLL(pkg.binding.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in ws.h but not exported"
    assert set(pkg.binding.EXPORTS) == declared


def test_version_and_status_strings(pkg):
    lib = pkg.load_library()
    assert "sm_100a" in pkg.ws_version()
    assert lib.ws_status_str(3) == b"WS_ERR_OUT_OF_PAGES"


def _dry(pkg, **kw):
    args = dict(dtype=pkg.WS_BF16, num_q_heads=32, num_kv_heads=8, head_dim=128, page_tokens=64,
                num_pages=64, max_sessions=4, max_pages_per_session=32, max_blocks_per_session=16,
                max_sessions_per_call=4, max_q_tokens_per_call=2048, flags=pkg.WS_FLAG_DRY_RUN)
    args.update(kw)
    return pkg.Cache(**args)


def test_no_gpu_compute_fails_loudly(pkg):
    """Without a CUDA device a real (non dry-run) cache cannot be created: no CPU fallback."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(Exception):
        pkg.Cache(pkg.WS_BF16, 32, 8, 128, 64, 16)


def test_page_allocation_block_boundaries_and_truncate(pkg):
    c = _dry(pkg)
    s0, s1 = c.session_open(), c.session_open()
    assert (s0, s1) == (0, 1) and c.free_pages() == 64
    c.kv_append([s0], [0, 100], None, None)               # 2 pages
    c.kv_append([s1, s0], [0, 64, 64 + 29], None, None)   # s1: 1 page; s0: 100+29=129 -> 3 pages
    assert c.session_info(s0) == (129, 2, [100, 129])
    assert c.session_info(s1) == (64, 1, [64])
    assert c.session_pages(s0) == [0, 1, 3] and c.session_pages(s1) == [2]
    assert c.free_pages() == 60
    c.session_truncate(s0, 1)
    assert c.session_info(s0) == (100, 1, [100]) and c.session_pages(s0) == [0, 1]
    assert c.free_pages() == 61
    c.session_close(s1)
    assert c.free_pages() == 62
    with pytest.raises(pkg.WsError) as e:
        c.session_info(s1)
    assert e.value.status_name == "WS_ERR_BAD_SESSION"


def test_append_blocks_commits_many_blocks_in_one_call(pkg):
    """NEXT-1 (PAPER.md:75 system prefill): ws_kv_append_blocks == a sequence of ws_kv_append calls for the
    host metadata (tokens, block ends, page ids), and rejects malformed block lists with nothing changed."""
    a, b = _dry(pkg), _dry(pkg)
    sa = [a.session_open(), a.session_open()]
    sb = [b.session_open(), b.session_open()]
    a.kv_append([sa[0]], [0, 10], None, None)
    b.kv_append([sb[0]], [0, 10], None, None)
    lens0, lens1 = [100, 29, 64, 7], [64, 1]
    a.kv_append_blocks(sa, [0, sum(lens0), sum(lens0) + sum(lens1)], [0, 4, 6], lens0 + lens1, None, None)
    # reference: one ws_kv_append per block, in an order that allocates the same pages (session 0 first)
    for n in lens0:
        b.kv_append([sb[0]], [0, n], None, None)
    for n in lens1:
        b.kv_append([sb[1]], [0, n], None, None)
    for x, y in zip(sa, sb):
        assert a.session_info(x) == b.session_info(y)
        assert a.session_pages(x) == b.session_pages(y)
    assert a.session_info(sa[0]) == (210, 5, [10, 110, 139, 203, 210])
    assert a.free_pages() == b.free_pages()
    # the commit message names every block (replica side applies them in one go)
    msg = a.replica_commit_message()
    assert list(msg[9:13]) == [sa[0], 10, 4, 4 - 1 + 0] or msg[11] == 4
    before = (a.session_info(sa[0]), a.session_info(sa[1]), a.free_pages())
    for cu_b, lens in (([0, 2, 3], [5, 5, 7]),            # session 0: 10 tokens but cu says 12
                       ([0, 1, 1], [12]),                  # session 1: zero blocks
                       ([0, 2, 3], [12, 0, 7]),            # empty block
                       ([1, 2, 3], [12, 7, 7])):           # cu_blocks[0] != 0
        with pytest.raises(pkg.WsError) as e:
            a.kv_append_blocks(sa, [0, 12, 19], cu_b, lens, None, None)
        assert e.value.status_name == "WS_ERR_INVALID_ARG"
        assert (a.session_info(sa[0]), a.session_info(sa[1]), a.free_pages()) == before
    # block capacity (16 per session): 5 committed + 12 more does not fit, 11 does
    with pytest.raises(pkg.WsError) as e:
        a.kv_append_blocks([sa[0]], [0, 12], [0, 12], [1] * 12, None, None)
    assert e.value.status_name == "WS_ERR_OUT_OF_PAGES"
    assert (a.session_info(sa[0]), a.session_info(sa[1]), a.free_pages()) == before
    a.kv_append_blocks([sa[0]], [0, 11], [0, 11], [1] * 11, None, None)
    assert a.session_info(sa[0])[1] == 16


def test_error_paths_leave_state_unchanged(pkg):
    c = _dry(pkg, num_pages=4)
    s = c.session_open(); t = c.session_open()
    c.kv_append([s], [0, 64], None, None)
    before = (c.session_info(s), c.session_info(t), c.free_pages(), c.session_pages(s))
    cases = [
        (([s, t], [0, 10, 10 + 64 * 3 + 1]), "WS_ERR_OUT_OF_PAGES"),   # needs 1 + 4 pages, 3 free
        (([s, s], [0, 1, 2]), "WS_ERR_INVALID_ARG"),                   # duplicate session
        (([s], [0, 0]), "WS_ERR_INVALID_ARG"),                         # n = 0
        (([3], [0, 5]), "WS_ERR_BAD_SESSION"),
        (([s], [1, 5]), "WS_ERR_INVALID_ARG"),                         # cu[0] != 0
        (([s], [0, 4096]), "WS_ERR_OUT_OF_PAGES"),                     # beyond per-session table
    ]
    for (ids, cu), name in cases:
        with pytest.raises(pkg.WsError) as e:
            c.kv_append(ids, cu, None, None)
        assert e.value.status_name == name, (ids, cu, e.value)
        assert (c.session_info(s), c.session_info(t), c.free_pages(), c.session_pages(s)) == before
    # attention argument checks
    with pytest.raises(pkg.WsError) as e:
        c.block_causal_attn_fwd([s], [0, 63], None, None, 0.1)         # token count mismatch
    assert e.value.status_name == "WS_ERR_INVALID_ARG"
    with pytest.raises(pkg.WsError):
        c.block_causal_attn_fwd([s], [0, 64], None, None, 0.1, num_q_blocks=[2])
    with pytest.raises(pkg.WsError):
        c.block_causal_attn_fwd([s], [0, 64], None, None, -1.0)
    with pytest.raises(pkg.WsError):
        c.block_causal_attn_fwd([t], [0, 0], None, None, 0.1)          # empty session has no block
    for bad in (dict(num_q_heads=30), dict(head_dim=12), dict(page_tokens=0), dict(dtype=7)):
        with pytest.raises(pkg.WsError):
            _dry(pkg, **bad)


def test_shuffled_free_list_is_a_permutation(pkg):
    c = _dry(pkg, num_pages=32)
    c.shuffle_free_pages(1234)
    s = c.session_open()
    c.kv_append([s], [0, 32 * 64], None, None)
    pages = c.session_pages(s)
    assert sorted(pages) == list(range(32)) and pages != list(range(32))


def _plan(pkg, lens, n, Hq=32, Hkv=8, min_splits=0, blocks=1, decode_plan=True):
    S = len(lens)
    P = 64
    pages = sum((L + n * blocks + P - 1) // P for L in lens) + 4
    c = _dry(pkg, num_q_heads=Hq, num_kv_heads=Hkv, num_pages=pages, max_sessions=S,
             max_pages_per_session=max((L + n * blocks + P - 1) // P for L in lens) + 1,
             max_blocks_per_session=1000, max_sessions_per_call=S,
             max_q_tokens_per_call=max(S * n * blocks, 2048))
    ids = [c.session_open() for _ in lens]
    for s, L in zip(ids, lens):
        pos = 0
        while pos < L:
            step = min(2048 // S, L - pos)
            c.kv_append([s], [0, step], None, None); pos += step
    for _ in range(blocks):
        c.kv_append(ids, [i * n for i in range(S + 1)], None, None)
    if min_splits:
        c.set_min_splits(min_splits)
    c.set_decode_plan(decode_plan)
    c.block_causal_attn_fwd(ids, [i * n * blocks for i in range(S + 1)], None, None, 0.1,
                            num_q_blocks=[blocks] * S)
    return c.last_plan_info(), c.last_plan_segments()


def _check_cover(info, segs, expect_tiles):
    """every group's KV tiles are covered exactly once, in order, by its segments."""
    by_group = {}
    for sg in segs:
        by_group.setdefault(sg["group"], []).append(sg)
    total = 0
    for g, lst in by_group.items():
        pos = 0
        for sg in lst:
            assert sg["tile_begin"] == pos and sg["tile_end"] > sg["tile_begin"]
            pos = sg["tile_end"]
            assert (sg["part_base"] >= 0) == (len(lst) > 1)
        total += pos
    assert total == info["total_kv_tiles"] == expect_tiles
    assert len(by_group) == info["num_groups"]
    teams = [sg["team"] for sg in segs]
    assert teams == sorted(teams)


def _team_costs(segs, ovh=3.3):
    tiles = np.bincount([s["team"] for s in segs], weights=[s["tile_end"] - s["tile_begin"] for s in segs])
    nseg = np.bincount([s["team"] for s in segs])
    return tiles + ovh * (nseg - 1)


def test_planner_config4_shape(pkg):
    info, segs = _plan(pkg, [65536], 256)
    assert info["used_tensor_core_kernel"] == 1
    assert info["team_size"] == 4 and info["num_ctas"] == 148 and info["num_groups"] == 8
    tiles = 8 * ((65536 + 256 + 127) // 128)
    _check_cover(info, segs, tiles)
    # balanced in COST units: tiles + 3.3 per extra segment of a team (segment start-up overhead)
    cost = _team_costs(segs)
    assert len(cost) == 37 and cost[:-1].max() - cost[:-1].min() <= 2.0, cost
    assert cost[-1] <= cost[:-1].max() + 1.0 and cost[-1] >= 0.9 * cost[:-1].max(), cost
    assert info["num_combine_items"] == 8


def test_planner_ragged_multi_session(pkg):
    lens = [21852, 18399, 26008, 19914, 2081, 30893, 27228, 25114]
    info, segs = _plan(pkg, lens, 256)
    tiles = 8 * sum((L + 256 + 127) // 128 for L in lens)
    _check_cover(info, segs, tiles)
    assert info["num_groups"] == 64 and info["num_ctas"] == 148
    cost = _team_costs(segs)
    # min-max budget: no team above the mean by more than a tile or so; a few teams that stop at a group
    # boundary (cannot afford the next segment's start-up) stay below it
    assert cost.max() <= cost.mean() + 2.0 and np.median(cost) >= cost.max() - 2.0, cost


def test_planner_many_groups_last_team_not_overloaded(pkg):
    """Regression: 16-head MHA, 66 tiles per group over 148 single-CTA teams.  Per-team rounding used to
    leave the last team with the sum of every team's remainder (63 tiles against an average of 7)."""
    info, segs = _plan(pkg, [8192], 256, Hq=16, Hkv=16)
    _check_cover(info, segs, 16 * 66)
    cost = _team_costs(segs)
    assert info["team_size"] == 1 and 130 <= len(cost) <= 148
    assert cost.max() <= 8.0 + 1e-6, cost            # 1056 tiles over 148 teams: 8 per team is the optimum


def test_planner_small_and_forced_splits(pkg):
    info, segs = _plan(pkg, [100], 16, Hq=8, Hkv=2, decode_plan=False)   # 1 tile per group: no split
    _check_cover(info, segs, 2)
    assert info["num_combine_items"] == 0 and all(s["part_base"] == -1 for s in segs)
    info, segs = _plan(pkg, [1000], 64, Hq=8, Hkv=2, min_splits=3)
    _check_cover(info, segs, 2 * 9)
    assert info["num_combine_items"] == 2
    by_group = {}
    for s in segs:
        by_group.setdefault(s["group"], 0); by_group[s["group"]] += 1
    assert all(v >= 3 for v in by_group.values())


def test_planner_decode_plan(pkg):
    """NEXT-4: n*G <= 128 packed rows per (session, KV head) -> decode plan: one CTA per team; the
    even / odd KV-tile accumulator sets are merged inside the CTA, so partial slots and combine items
    follow the general rule (only groups cut into several segments)."""
    for lens, n, Hq, Hkv in (([65536], 1, 32, 8), ([65536], 16, 32, 8), ([4096, 100, 9000], 32, 32, 8),
                             ([5000], 128, 16, 16), ([70], 4, 8, 2)):
        info, segs = _plan(pkg, lens, n, Hq=Hq, Hkv=Hkv)
        assert info["used_tensor_core_kernel"] == 3 and info["team_size"] == 1, (lens, n, info)
        tiles = Hkv * sum((L + n + 127) // 128 for L in lens)
        _check_cover(info, segs, tiles)
        assert info["num_ctas"] <= 148
    # one row more than a Q tile holds -> general plan; and the switch forces it
    info, _ = _plan(pkg, [4096], 33, Hq=32, Hkv=8)
    assert info["used_tensor_core_kernel"] == 1
    info, _ = _plan(pkg, [4096], 16, Hq=32, Hkv=8, decode_plan=False)
    assert info["used_tensor_core_kernel"] == 1


def test_planner_multi_block_queries(pkg):
    info, segs = _plan(pkg, [300], 200, Hq=4, Hkv=4, blocks=3)   # 600 query tokens, G=1 -> 3 pairs
    assert info["team_size"] == 3
    _check_cover(info, segs, 4 * ((300 + 600 + 127) // 128))


def test_plan_cache_is_transparent(pkg):
    """Single-block steps look their plan up in a process-wide cache keyed by geometry + per-session (slot,
    query range, cache length): two handles ('layers') with the same sessions get the same plan, a changed
    length or split setting gets its own, and a repeated call returns exactly what planning returned."""
    lens, n = [5000, 777], 64
    a_info, a_segs = _plan(pkg, lens, n)
    b_info, b_segs = _plan(pkg, lens, n)              # second handle, same shape: served from the cache
    assert a_info == b_info and a_segs == b_segs
    _check_cover(b_info, b_segs, sum((L + n + 127) // 128 for L in lens) * 8)
    c_info, c_segs = _plan(pkg, [5000 + 128, 777], n)
    assert c_info["total_kv_tiles"] == a_info["total_kv_tiles"] + 8 and c_segs != a_segs
    d_info, d_segs = _plan(pkg, lens, n, min_splits=3)
    assert d_info["num_segments"] >= 3 * d_info["num_groups"] > a_info["num_groups"]
    e_info, e_segs = _plan(pkg, lens, n)              # the unforced plan is still what the cache returns
    assert e_info == a_info and e_segs == a_segs

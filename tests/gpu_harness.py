"""Shared test/bench harness: drive a synthetic workload through the CUDA path (via the C-ABI binding)
and through the float64 oracle, and compare.  The two paths share only the seeded inputs.

Protocol: every session's initial cache is committed through
ws_kv_append in blocks of `preload_block_tokens` tokens, round-robin over the sessions so that their
pages interleave in the pool; then each step appends one block per session (one call) and attends
with that block's queries (one call).
"""
from __future__ import annotations

from typing import Dict, List, Optional

import numpy as np

from synth_inputs import Workload


def _torch_of(arr: np.ndarray, device):
    import torch
    if arr.dtype.name == "bfloat16":
        return torch.from_numpy(arr.view(np.uint16).copy()).view(torch.bfloat16).to(device)
    return torch.from_numpy(np.ascontiguousarray(arr)).to(device)


def _numpy_of(t) -> np.ndarray:
    import ml_dtypes
    import torch
    if t.dtype == torch.bfloat16:
        return t.cpu().view(torch.int16).numpy().view(ml_dtypes.bfloat16)
    return t.cpu().numpy()


def preload_rounds(w: Workload):
    """[(list of session indices, list of (lo, hi) token ranges)] - identical for both paths."""
    pb = w.spec.preload_block_tokens
    rounds, pos = [], [0] * len(w.sessions)
    while True:
        ids, rng = [], []
        for s, L in enumerate(w.cache_lens):
            if pos[s] < L:
                hi = min(L, pos[s] + pb)
                ids.append(s); rng.append((pos[s], hi)); pos[s] = hi
        if not ids:
            return rounds
        rounds.append((ids, rng))


def make_cache(w: Workload, flags: int = 0, extra_pages: int = 2, pool_fill: Optional[int] = None,
               q_to_kv_head=None, extra_q_tokens: int = 0, device: int = 0):
    from paper_2606_25041_b200 import WS_BF16, WS_F32, Cache
    sp = w.spec
    P = sp.page_tokens
    final = [L + sp.steps * sp.block_tokens for L in w.cache_lens]
    pages = sum((x + P - 1) // P for x in final) + extra_pages
    S = sp.num_sessions
    per_call = S * max(sp.block_tokens, sp.preload_block_tokens) + extra_q_tokens
    return Cache(WS_BF16 if sp.dtype == "bf16" else WS_F32, sp.num_q_heads, sp.num_kv_heads,
                 sp.head_dim, P, pages, max_sessions=S,
                 max_pages_per_session=max((x + P - 1) // P for x in final) + 1,
                 max_blocks_per_session=max(w.cache_lens) // sp.preload_block_tokens + sp.steps + 8,
                 max_sessions_per_call=S, max_q_tokens_per_call=per_call,
                 flags=flags, pool_fill=pool_fill, q_to_kv_head=q_to_kv_head, device=device)


def preload_gpu(cache, w: Workload, dev_k: List, dev_v: List) -> List[int]:
    """Open the sessions and commit the initial caches. Returns session ids."""
    import torch
    ids = [cache.session_open() for _ in w.sessions]
    for sess, rng in preload_rounds(w):
        cu = [0]
        for lo, hi in rng:
            cu.append(cu[-1] + hi - lo)
        if len(sess) == 1:
            s, (lo, hi) = sess[0], rng[0]
            k, v = dev_k[s][lo:hi], dev_v[s][lo:hi]
        else:
            k = torch.cat([dev_k[s][lo:hi] for s, (lo, hi) in zip(sess, rng)])
            v = torch.cat([dev_v[s][lo:hi] for s, (lo, hi) in zip(sess, rng)])
        cache.kv_append([ids[s] for s in sess], cu, k, v)
    return ids


def run_workload_gpu(w: Workload, flags: int = 0, min_splits: int = 0, shuffle_seed: Optional[int] = None,
                     want_lse: bool = True, gather: bool = True, pool_fill: Optional[int] = None,
                     decode_plan: Optional[bool] = None, fused_step: bool = False) -> Dict:
    """fused_step: every step goes through ws_stream_step (one launch commits and attends the block, the
    configuration bench.py times) instead of ws_kv_append followed by ws_block_causal_attn_fwd."""
    import torch
    sp = w.spec
    dev = torch.device("cuda", 0)
    cache = make_cache(w, flags=flags, pool_fill=pool_fill)
    if shuffle_seed is not None:
        cache.shuffle_free_pages(shuffle_seed)
    if min_splits:
        cache.set_min_splits(min_splits)
    if decode_plan is not None:
        cache.set_decode_plan(decode_plan)
    dev_k = [_torch_of(s.k_cache, dev) for s in w.sessions]
    dev_v = [_torch_of(s.v_cache, dev) for s in w.sessions]
    ids = preload_gpu(cache, w, dev_k, dev_v)
    n, S = sp.block_tokens, sp.num_sessions
    cu = [i * n for i in range(S + 1)]
    outs, lses, plans = [], [], []
    tdt = torch.bfloat16 if sp.dtype == "bf16" else torch.float32
    for t in range(sp.steps):
        q = torch.cat([_torch_of(s.q[t], dev) for s in w.sessions])
        k = torch.cat([_torch_of(s.k[t], dev) for s in w.sessions])
        v = torch.cat([_torch_of(s.v[t], dev) for s in w.sessions])
        out = torch.full((S * n, sp.num_q_heads, sp.head_dim), float("nan"), dtype=tdt, device=dev)
        lse = torch.full((S * n, sp.num_q_heads), float("nan"), dtype=torch.float32, device=dev) if want_lse else None
        if fused_step:
            cache.stream_step(ids, cu, q, k, v, out, sp.scale, lse=lse)
        else:
            cache.kv_append(ids, cu, k, v, modality=np.tile(w.modality, S))
            cache.block_causal_attn_fwd(ids, cu, q, out, sp.scale, lse=lse)
        torch.cuda.synchronize()
        plans.append(cache.last_plan_info())
        o = out.float().cpu().numpy().astype(np.float64).reshape(S, n, sp.num_q_heads, sp.head_dim)
        outs.append([o[s] for s in range(S)])
        if want_lse:
            l = lse.cpu().numpy().astype(np.float64).reshape(S, n, sp.num_q_heads)
            lses.append([l[s] for s in range(S)])
    kv = None
    if gather:
        kv = []
        for s, sid in enumerate(ids):
            tokens, _, _ = cache.session_info(sid)
            kg = torch.empty((tokens, sp.num_kv_heads, sp.head_dim), dtype=tdt, device=dev)
            vg = torch.empty_like(kg)
            cache.kv_gather(sid, 0, tokens, kg, vg)
            torch.cuda.synchronize()
            kv.append((_numpy_of(kg), _numpy_of(vg)))
    res = {"out": outs, "lse": lses, "kv": kv, "plans": plans,
           "tensor": bool(plans and plans[-1]["used_tensor_core_kernel"]),
           "launches": cache.launch_count(), "cache": cache, "ids": ids}
    return res


def bf16_half_ulp(x: np.ndarray) -> np.ndarray:
    """Half a bf16 ulp at |x| (8 significand bits): 2^(floor(log2|x|) - 8); 0 at x == 0."""
    _, ex = np.frexp(np.abs(x))                          # |x| = m * 2^ex, m in [0.5, 1)
    return np.where(x == 0, 0.0, np.ldexp(1.0, ex - 9))


def bf16_error_bound(o_ref: np.ndarray, o_gpu: np.ndarray, absw: np.ndarray) -> np.ndarray:
    """Element-wise bound on |O_gpu - O_ref| that follows from the arithmetic (reading A10):
    the output is rounded once to bf16 (RNE: half an ulp at the larger of the two magnitudes), and every
    softmax weight is rounded to bf16 before the PV product: unit roundoff 2^-8 per weight (8 significand
    bits), plus the 7.5e-5 of the polynomial exponential and of the fp32 row sum - together < 1.05 * 2^-8 -
    which moves O by at most 1.05 * 2^-8 * A with A = sum_j w_j |v_j| (oracle, want_abs).  fp32
    accumulation of S, O and of the split-KV merge is below 1e-6 * A."""
    return bf16_half_ulp(np.maximum(np.abs(o_ref), np.abs(o_gpu))) + (1.05 * 2.0 ** -8 + 1e-6) * absw + 1e-7


def run_workload_oracle(w: Workload, rows=None, heads=None, steps=None, want_abs: Optional[bool] = None) -> Dict:
    """The same protocol through oracle/ (float64). rows/heads: optional output sample.
    want_abs: also return A = sum_j w_j |v_j| per output element (res["abs"]) for bf16_error_bound."""
    from oracle.block_causal import OracleSession, attend
    sp = w.spec
    if want_abs is None:
        want_abs = sp.dtype == "bf16"
    sessions = [OracleSession(sp.num_kv_heads, sp.head_dim) for _ in w.sessions]
    for sess, rng in preload_rounds(w):
        for s, (lo, hi) in zip(sess, rng):
            sessions[s].append(w.sessions[s].k_cache[lo:hi], w.sessions[s].v_cache[lo:hi])
    outs, lses, absws = [], [], []
    steps = range(sp.steps) if steps is None else steps
    for t in range(sp.steps):
        for s, si in enumerate(w.sessions):
            sessions[s].append(si.k[t], si.v[t])
        if t not in steps:
            outs.append(None); lses.append(None); absws.append(None)
            continue
        o_t, l_t, a_t = [], [], []
        for s, si in enumerate(w.sessions):
            r = attend(sessions[s], si.q[t], sp.scale, 1, rows=rows, heads=heads, want_abs=want_abs)
            o_t.append(r[0]); l_t.append(r[1])
            if want_abs:
                a_t.append(r[2])
        outs.append(o_t); lses.append(l_t); absws.append(a_t)
    kv = [sess.gather() for sess in sessions]
    return {"out": outs, "lse": lses, "abs": absws if want_abs else None, "kv": kv, "sessions": sessions}


def compare(got: Dict, ref: Dict, dtype: str, rows=None, heads=None) -> Dict:
    """Element-wise errors of the CUDA path vs the oracle over every compared output element."""
    diffs, refs, lse_d, viol = [], [], [], []
    for t, ref_t in enumerate(ref["out"]):
        if ref_t is None:
            continue
        for s, r in enumerate(ref_t):
            g = got["out"][t][s]
            if rows is not None:
                g = g[np.asarray(rows)]
            if heads is not None:
                g = g[:, np.asarray(heads)]
            diffs.append((g - r).ravel()); refs.append(r.ravel())
            if ref.get("abs"):
                viol.append((np.abs(g - r) - bf16_error_bound(r, g, ref["abs"][t][s])).max())
            if got["lse"]:
                gl = got["lse"][t][s]
                if rows is not None:
                    gl = gl[np.asarray(rows)]
                if heads is not None:
                    gl = gl[:, np.asarray(heads)]
                lse_d.append((gl - ref["lse"][t][s]).ravel())
    d = np.concatenate(diffs); r = np.concatenate(refs)
    err = {"max_abs": float(np.abs(d).max()), "mean_abs": float(np.abs(d).mean()),
           # largest |error| - bf16_error_bound over the compared elements (<= 0: inside the derived bound)
           "bound_viol": float(max(viol)) if viol else float("nan"),
           "rel_rms": float(np.sqrt((d ** 2).mean() / max((r ** 2).mean(), 1e-300))),
           "lse_max": float(np.abs(np.concatenate(lse_d)).max()) if lse_d else float("nan"),
           "finite": bool(np.isfinite(d).all())}
    if got.get("kv") is not None:
        ok = True
        for (kg, vg), (kr, vr) in zip(got["kv"], ref["kv"]):
            ok &= kg.tobytes() == np.ascontiguousarray(kr).tobytes()
            ok &= vg.tobytes() == np.ascontiguousarray(vr).tobytes()
        err["kv_bit_exact"] = bool(ok)
    else:
        err["kv_bit_exact"] = None
    return err

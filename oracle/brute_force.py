"""Brute-force dense-mask checker for the oracle.  TEST INFRASTRUCTURE ONLY (see block_causal.py).

A deliberately different formulation from `oracle.block_causal.attend`, used only to check the
oracle on tiny inputs: ALL T tokens of the stream are concatenated, the dense T x T boolean mask
M[i][j] = (blk(j) <= blk(i)) is built explicitly (reading A1 of "block-causal attention",
PAPER.md:11, :29; dependence structure of Eq. (1)), KV heads are explicitly repeated
G times, masked scores are set to -inf, and each row's softmax and weighted sum are evaluated with
scalar Python float (= IEEE double) loops - no matmul, no incremental cache, no shared code.
"""
from __future__ import annotations

import math
from typing import List, Sequence


def dense_block_causal(q, k, v, block_sizes: Sequence[int], scale: float,
                       q_to_kv: Sequence[int] = None, mask_kind: str = "block_causal",
                       tags: Sequence[int] = None):
    """q: [T][Hq][D], k/v: [T][Hkv][D] nested sequences / arrays.  Returns (O [T][Hq][D], LSE [T][Hq]).

    mask_kind: "block_causal" (the method), or the two WRONG readings used by the pin tests to
    show the hand example separates them: "token_causal" (j <= i) and "none" (all visible);
    "text_causal" = the mixed intra-block mask of NEXT-4 (reading A19): block-causal,
    except that a text token (tags[i] == 2) does not see text tokens at later positions.
    """
    T = len(q); Hq = len(q[0]); D = len(q[0][0]); Hkv = len(k[0])
    assert sum(block_sizes) == T
    blk: List[int] = []
    for b, sz in enumerate(block_sizes):
        blk += [b] * sz
    G = Hq // Hkv
    # explicit GQA expansion: head h of the expanded K/V is KV head q_to_kv[h] (default h // G)
    kv_of = [h // G for h in range(Hq)] if q_to_kv is None else list(q_to_kv)
    if mask_kind == "block_causal":
        M = [[blk[j] <= blk[i] for j in range(T)] for i in range(T)]
    elif mask_kind == "text_causal":
        assert tags is not None and len(tags) == T
        M = [[blk[j] <= blk[i] and not (tags[i] == 2 and tags[j] == 2 and j > i) for j in range(T)]
             for i in range(T)]
    elif mask_kind == "token_causal":
        M = [[j <= i for j in range(T)] for i in range(T)]
    elif mask_kind == "none":
        M = [[True] * T for _ in range(T)]
    else:
        raise ValueError(mask_kind)
    O = [[[0.0] * D for _ in range(Hq)] for _ in range(T)]
    LSE = [[0.0] * Hq for _ in range(T)]
    for i in range(T):
        for h in range(Hq):
            g = kv_of[h]
            s = []
            for j in range(T):
                if M[i][j]:
                    acc = 0.0
                    for d in range(D):
                        acc += float(q[i][h][d]) * float(k[j][g][d])
                    s.append(scale * acc)
                else:
                    s.append(-math.inf)
            mx = max(s)
            e = [math.exp(x - mx) if x != -math.inf else 0.0 for x in s]
            z = math.fsum(e)
            for d in range(D):
                O[i][h][d] = math.fsum(e[j] * float(v[j][g][d]) for j in range(T)) / z
            LSE[i][h] = mx + math.log(z)
    return O, LSE

"""float64 CPU ORACLE of the block-causal streaming-attention step.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this module.  It shares no code with the CUDA path (paper_2606_25041_b200/) and neither
imports the other.  Parity status: every function below is pinned by `tests/test_oracle_pins.py`
(hand example P0, closed forms P1-P6, brute force, SDPA special cases, invariants) - nothing here
is "parity unpinned".

What it computes (definition, evaluated step by step; DESIGN.md §2 "Readings"):

* The stream is one causal sequence of interleaved visual/audio/text tokens grouped into per-unit
  blocks (PAPER.md:11 Abstract; :29 §1; :45 §2.1).  "Block-causal attention" (PAPER.md:11, :23
  Fig. 1, :29, :38, :155) is never written as a formula in the paper; reading A1: key j is visible
  to query i  iff  blk(j) <= blk(i)  - bidirectional inside a block, causal across blocks - which is
  exactly the dependence structure of Eq. (1): unit k depends on units <= k only.
* Every unit's K/V slice is appended / "committed back into the interaction history"
   and the history is never truncated ("full-history",
  PAPER.md:38, :75).

State per session:  Kc, Vc in R^{L x Hkv x D} (storage dtype, bit-exact copies of what was
appended) and block ends 0 = e_0 < e_1 < ... < e_B = L.

append(K_new, V_new):  Kc <- [Kc; K_new], Vc <- [Vc; V_new], e_{B+1} = L + n.
attend(Q for the last m blocks):  for every query row r in block b and q-head h, g = q_to_kv[h]:
    visible set  V(r) = { j : 0 <= j < e_b }                       (whole own block + all earlier)
    s_j  = scale * sum_d Q[r,h,d] * Kc[j,g,d]                      (float64)
    m    = max_j s_j ;  p_j = exp(s_j - m) ;  Z = sum_j p_j        (two-pass softmax)
    O[r,h,:] = sum_j (p_j / Z) * Vc[j,g,:] ;  LSE[r,h] = m + log Z
The matrix products use numpy's float64 matmul as the library primitive; there is no tiling, no
online-softmax recurrence and no reordering beyond that.

Mixed intra-block mask (NEXT-4, `text_causal=True`; reading A19).  The thinker "runs the short
token-causal Transformer pass for language prediction and state update" / "token-causal
decoding over the language and state slots" while audio/video stay block-wise.  Reading:
with per-token modality tags (0 video, 1 audio, 2 text) the visible set becomes
    V(r) = { j : j < e_b  and not ( tag(r) == text and tag(j) == text and j > pos(r) ) }
i.e. text slots are token-causal AMONG THEMSELVES (a text query never sees a later text key, which by
j < e_b can only be one of its own block), every other (query, key) pair keeps the block-causal rule:
audio/video keys of the block are visible to every query of the block, text keys are visible to every
audio/video query of the block.  A query always sees itself, so no row is empty.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np


class OracleSession:
    """One session's full-history KV cache with block boundaries."""

    def __init__(self, num_kv_heads: int, head_dim: int):
        self.Hkv, self.D = num_kv_heads, head_dim
        self.k_slices: List[np.ndarray] = []     # storage-dtype slices exactly as appended
        self.v_slices: List[np.ndarray] = []
        self.block_ends: List[int] = [0]
        self.tags: List[np.ndarray] = []         # per-slice modality tags (uint8) or None

    @property
    def length(self) -> int:
        return self.block_ends[-1]

    def append(self, k_new: np.ndarray, v_new: np.ndarray, modality: Optional[Sequence[int]] = None) -> None:
        """Commit one block: history <- [history; slice]; records e_{B+1} = L + n.
        modality: optional per-token tags (0 video, 1 audio, 2 text), metadata for `text_causal`."""
        assert k_new.shape == v_new.shape and k_new.ndim == 3
        n, Hkv, D = k_new.shape
        assert n > 0 and (Hkv, D) == (self.Hkv, self.D)
        self.k_slices.append(np.array(k_new, copy=True))
        self.v_slices.append(np.array(v_new, copy=True))
        self.block_ends.append(self.length + n)
        if modality is not None:
            modality = np.asarray(modality, dtype=np.uint8)
            assert modality.shape == (n,)
        self.tags.append(modality)

    def text_mask(self) -> np.ndarray:
        """is_text[j] for every committed token j (tokens appended without tags count as non-text)."""
        parts = [np.zeros(len(k), dtype=bool) if t is None else (t == 2)
                 for k, t in zip(self.k_slices, self.tags)]
        return np.concatenate(parts) if parts else np.zeros(0, dtype=bool)

    def gather(self, start: int = 0, count: Optional[int] = None) -> Tuple[np.ndarray, np.ndarray]:
        """Logical tokens [start, start+count) of the committed history, storage dtype."""
        if not self.k_slices:
            raise ValueError("empty session")
        k = np.concatenate(self.k_slices, axis=0)
        v = np.concatenate(self.v_slices, axis=0)
        count = self.length - start if count is None else count
        return k[start:start + count], v[start:start + count]


def default_q_to_kv(num_q_heads: int, num_kv_heads: int) -> np.ndarray:
    """Reading A7: consecutive q-heads share a KV head, g = h // (Hq / Hkv)."""
    assert num_q_heads % num_kv_heads == 0
    return np.arange(num_q_heads) // (num_q_heads // num_kv_heads)


def attend(sess: OracleSession, q: np.ndarray, scale: float, num_q_blocks: int = 1,
           q_to_kv: Optional[Sequence[int]] = None,
           rows: Optional[Sequence[int]] = None,
           heads: Optional[Sequence[int]] = None, want_abs: bool = False, text_causal: bool = False):
    """Block-causal attention of the LAST `num_q_blocks` committed blocks against the history.

    q: [n_q, Hq, D] (n_q = total tokens of those blocks, storage dtype, widened to float64 here).
    rows / heads: optional subsets (indices into n_q / Hq) so that full-size configs can be
    checked on sampled outputs; the arithmetic per output element is identical.
    Returns O float64 [len(rows), len(heads), D] and LSE float64 [len(rows), len(heads)].
    want_abs: additionally return A[r,h,:] = sum_j (p_j / Z) * |Vc[j,g,:]| (same weights, |V| instead
    of V): the condition number of the output w.r.t. relative perturbations of the weights, used by the
    tests to state the bf16 error bound of DESIGN.md reading A10 (|O| <= A, with equality for V >= 0).
    text_causal: the mixed intra-block mask of the module docstring (reading A19): a text query does not
    see text keys at later positions; everything else as above.
    """
    B = len(sess.block_ends) - 1
    assert 1 <= num_q_blocks <= B
    first = B - num_q_blocks
    q_start = sess.block_ends[first]
    n_q, Hq, D = q.shape
    assert n_q == sess.length - q_start and D == sess.D
    g_of = default_q_to_kv(Hq, sess.Hkv) if q_to_kv is None else np.asarray(q_to_kv)
    rows = np.arange(n_q) if rows is None else np.asarray(rows, dtype=np.int64)
    heads = np.arange(Hq) if heads is None else np.asarray(heads, dtype=np.int64)

    Kc, Vc = sess.gather()
    out = np.zeros((len(rows), len(heads), D), dtype=np.float64)
    lse = np.zeros((len(rows), len(heads)), dtype=np.float64)
    absw = np.zeros_like(out) if want_abs else None
    # block index of every selected query row, and that block's visible end e_b
    abs_pos = q_start + rows
    ends = np.asarray(sess.block_ends)
    blk = np.searchsorted(ends, abs_pos, side="right")        # e_{blk-1} <= pos < e_blk
    vis_end = ends[blk]
    is_text = sess.text_mask() if text_causal else None
    for g in np.unique(g_of[heads]):
        Kg = Kc[:, g, :].astype(np.float64)
        Vg = Vc[:, g, :].astype(np.float64)
        for hi, h in enumerate(heads):
            if g_of[h] != g:
                continue
            for e in np.unique(vis_end):
                sel = np.nonzero(vis_end == e)[0]
                Q = q[rows[sel], h, :].astype(np.float64)
                S = scale * (Q @ Kg[:e].T)                      # s_j for all visible j < e_b
                if text_causal:
                    # text query at position pos: text keys j > pos are not visible (score -inf, weight 0)
                    pos = abs_pos[sel]
                    hidden = (is_text[pos][:, None] & is_text[None, :e]) & (np.arange(e)[None, :] > pos[:, None])
                    S = np.where(hidden, -np.inf, S)
                m = S.max(axis=1, keepdims=True)
                P = np.exp(S - m)
                Z = P.sum(axis=1, keepdims=True)
                out[sel, hi, :] = (P / Z) @ Vg[:e]
                lse[sel, hi] = (m + np.log(Z))[:, 0]
                if want_abs:
                    absw[sel, hi, :] = (P / Z) @ np.abs(Vg[:e])
    if want_abs:
        return out, lse, absw
    return out, lse


def merge_partials(o_parts: np.ndarray, lse_parts: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Split-KV combine (step a4; the paper is silent - north_star names it).

    Attention over a disjoint union of key ranges is the LSE-weighted mean of the per-range
    results:  m* = max_s LSE_s ; w_s = exp(LSE_s - m*) ; O = sum_s w_s O_s / sum_s w_s ;
    LSE = m* + log sum_s w_s.  Empty ranges carry LSE = -inf (w = 0).
    o_parts: [S, ..., D], lse_parts: [S, ...].
    """
    o_parts = np.asarray(o_parts, dtype=np.float64)
    lse_parts = np.asarray(lse_parts, dtype=np.float64)
    m = lse_parts.max(axis=0)
    w = np.exp(lse_parts - m)
    w = np.where(np.isneginf(lse_parts), 0.0, w)
    wsum = w.sum(axis=0)
    o = (w[..., None] * np.where(w[..., None] > 0, o_parts, 0.0)).sum(axis=0) / wsum[..., None]
    return o, m + np.log(wsum)


def attend_range(sess: OracleSession, q: np.ndarray, scale: float, key_lo: int, key_hi: int,
                 q_to_kv: Optional[Sequence[int]] = None) -> Tuple[np.ndarray, np.ndarray]:
    """Softmax attention of q restricted to keys [key_lo, key_hi) (one split of a4).

    Used only to state the merge identity; an empty range returns O = 0, LSE = -inf.
    """
    n_q, Hq, D = q.shape
    g_of = default_q_to_kv(Hq, sess.Hkv) if q_to_kv is None else np.asarray(q_to_kv)
    Kc, Vc = sess.gather()
    out = np.zeros((n_q, Hq, D)); lse = np.full((n_q, Hq), -np.inf)
    if key_hi <= key_lo:
        return out, lse
    for h in range(Hq):
        Kg = Kc[key_lo:key_hi, g_of[h], :].astype(np.float64)
        Vg = Vc[key_lo:key_hi, g_of[h], :].astype(np.float64)
        S = scale * (q[:, h, :].astype(np.float64) @ Kg.T)
        m = S.max(axis=1, keepdims=True)
        P = np.exp(S - m)
        Z = P.sum(axis=1, keepdims=True)
        out[:, h, :] = (P / Z) @ Vg
        lse[:, h] = (m + np.log(Z))[:, 0]
    return out, lse


def fm_euler_update(z: np.ndarray, v: np.ndarray, dtau: float) -> np.ndarray:
    """NEXT-2: one explicit Euler step of the flow-matching ODE, z <- z + dtau * v, in float64.

    Eq. (2): z_tau = (1 - tau) z_0 + tau eps and dz/dtau = eps - z_0, so with the
    exact velocity v = eps - z_0 a single step of size dtau = -tau from z_tau lands on z_0
    (pinned by tests/test_oracle_pins.py::test_fm_euler_exact_velocity_recovers_clean_latent).
    """
    return np.asarray(z, dtype=np.float64) + float(dtau) * np.asarray(v, dtype=np.float64)

"""Workload shapes and seeded inputs (recipe: DESIGN.md "Input recipe").

The paper fixes only the streaming unit (160 ms at 25 fps = 4 frames);
it states no tokens/unit, heads, head_dim or dtype.  BASELINE.json's five configs are the synthetic
stand-ins; they are restated here as `CONFIG_SPECS[1..5]`.

RNG: ``numpy.random.default_rng([2606, 25041, cfg])``.  Draw order per config:
  (cfg 5 only) the S cache lengths, then the outlier channels per KV head;
  then per session: K_cache[L,Hkv,D], V_cache[L,Hkv,D], then per step t: Q_t[n,Hq,D],
  K_t[n,Hkv,D], V_t[n,Hkv,D], all ``standard_normal(float32)``.
bf16 configs are rounded ONCE to bfloat16 (round-to-nearest-even, ml_dtypes); the rounded arrays
are the canonical inputs handed to both the oracle and the CUDA path.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import ml_dtypes
import numpy as np

BF16 = ml_dtypes.bfloat16


@dataclass(frozen=True)
class WorkloadSpec:
    cfg: int                      # seed stream id (1..5 for the BASELINE configs)
    name: str
    dtype: str                    # "bf16" | "f32"
    num_sessions: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    block_tokens: int             # n: tokens per streaming-unit block
    modality_split: tuple         # (video, audio, text) tokens per block
    cache_lens: Optional[tuple]   # initial committed length per session; None => drawn (cfg 5)
    cache_len_range: Optional[tuple] = None   # (lo, hi) inclusive when drawn
    steps: int = 1                # consecutive blocks appended + attended
    page_tokens: int = 64
    outlier_frac: float = 0.0     # fraction of K channels scaled (cfg 5: 0.05)
    outlier_scale: float = 1.0
    preload_block_tokens: int = 256   # the initial cache is committed in blocks of this size

    @property
    def scale(self) -> float:
        return 1.0 / float(np.sqrt(self.head_dim))

    @property
    def group(self) -> int:
        return self.num_q_heads // self.num_kv_heads


CONFIG_SPECS = {
    1: WorkloadSpec(1, "tiny_fp32", "f32", 1, 2, 2, 64, 16, (8, 6, 2), (0,), steps=3,
                    page_tokens=16, preload_block_tokens=16),
    2: WorkloadSpec(2, "bf16_single_session", "bf16", 1, 16, 16, 128, 256, (192, 48, 16), (4096,)),
    3: WorkloadSpec(3, "bf16_gqa", "bf16", 1, 32, 8, 128, 512, (384, 96, 32), (16384,)),
    4: WorkloadSpec(4, "bf16_long_session", "bf16", 1, 32, 8, 128, 256, (192, 48, 16), (65536,),
                    steps=20),
    5: WorkloadSpec(5, "bf16_ragged_multi_session", "bf16", 8, 32, 8, 128, 256, (192, 48, 16),
                    None, cache_len_range=(1024, 32768), outlier_frac=0.05, outlier_scale=8.0),
}


def spec_for_config(cfg: int, **overrides) -> WorkloadSpec:
    """BASELINE config `cfg` (1..5), optionally scaled down (e.g. cache_lens=(1000,), steps=2)."""
    return dataclasses.replace(CONFIG_SPECS[cfg], **overrides)


@dataclass
class SessionInputs:
    k_cache: np.ndarray           # [L, Hkv, D] storage dtype
    v_cache: np.ndarray
    q: List[np.ndarray] = field(default_factory=list)   # per step [n, Hq, D]
    k: List[np.ndarray] = field(default_factory=list)   # per step [n, Hkv, D]
    v: List[np.ndarray] = field(default_factory=list)


@dataclass
class Workload:
    spec: WorkloadSpec
    cache_lens: List[int]
    outlier_channels: Optional[np.ndarray]   # [Hkv, k] int or None
    sessions: List[SessionInputs]
    modality: np.ndarray                     # [n] uint8 tags of one block (0=video 1=audio 2=text)


def to_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 -> bfloat16 (RNE). Pure storage rounding; no method arithmetic."""
    return np.asarray(x, dtype=np.float32).astype(BF16)


def modality_tags(n: int, split: Sequence[int]) -> np.ndarray:
    """Canonical interleaving (reading A5): per-frame slots, each slot = [video.., audio.., text..].

    A slot is (48 video, 12 audio, 4 text) tokens when the block is a whole number of those
    (256-token block: 4 slots = 4 frames of a 160 ms unit at 25 fps; 512: 8 slots); otherwise
    gcd(v, a, t) slots (tiny 16: 2 slots of (4,3,1)).  Tags are metadata; they never change O.
    """
    v, a, t = split
    assert v + a + t == n
    if v % 48 == 0 and (a, t) == (v // 4, v // 12):
        slots = v // 48
    else:
        slots = int(np.gcd.reduce([v, a, t]))
    one = np.concatenate([np.zeros(v // slots, np.uint8), np.ones(a // slots, np.uint8),
                          np.full(t // slots, 2, np.uint8)])
    return np.tile(one, slots)


def generate(spec: WorkloadSpec) -> Workload:
    rng = np.random.default_rng([2606, 25041, spec.cfg])
    S, Hq, Hkv, D, n = (spec.num_sessions, spec.num_q_heads, spec.num_kv_heads, spec.head_dim,
                        spec.block_tokens)
    if spec.cache_lens is None:
        lo, hi = spec.cache_len_range
        lens = [int(x) for x in rng.integers(lo, hi, endpoint=True, size=S)]
    else:
        lens = list(spec.cache_lens)
        assert len(lens) == S
    outl = None
    if spec.outlier_frac > 0.0:
        k = int(round(spec.outlier_frac * D))
        outl = np.stack([np.sort(rng.permutation(D)[:k]) for _ in range(Hkv)])

    def draw(*shape):
        return rng.standard_normal(shape, dtype=np.float32)

    def scale_k(x):
        if outl is not None:
            for g in range(Hkv):
                x[:, g, outl[g]] *= np.float32(spec.outlier_scale)
        return x

    def store(x):
        return to_bf16(x) if spec.dtype == "bf16" else x

    sessions = []
    for s in range(S):
        si = SessionInputs(k_cache=store(scale_k(draw(lens[s], Hkv, D))),
                           v_cache=store(draw(lens[s], Hkv, D)))
        for _ in range(spec.steps):
            si.q.append(store(draw(n, Hq, D)))
            si.k.append(store(scale_k(draw(n, Hkv, D))))
            si.v.append(store(draw(n, Hkv, D)))
        sessions.append(si)
    return Workload(spec, lens, outl, sessions, modality_tags(n, spec.modality_split))


def algorithmic_flops(spec: WorkloadSpec, cache_lens: Sequence[int], step: int = 0) -> float:
    """FLOPs of one streaming-unit step: 4*D*Hq*sum_s n*(L_s + n)  (QK^T + PV, 2 per MAC)."""
    n = spec.block_tokens
    return 4.0 * spec.head_dim * spec.num_q_heads * sum(n * (L + step * n + n) for L in cache_lens)


def algorithmic_bytes(spec: WorkloadSpec, cache_lens: Sequence[int], step: int = 0) -> float:
    """Bytes one step must move: K,V read once per KV head + Q read + O write + append r/w."""
    eb = 2 if spec.dtype == "bf16" else 4
    n, D, Hq, Hkv = spec.block_tokens, spec.head_dim, spec.num_q_heads, spec.num_kv_heads
    keys = sum(L + step * n + n for L in cache_lens)
    new = n * len(cache_lens)
    return 2.0 * eb * Hkv * D * keys + 2.0 * eb * Hq * D * new + 4.0 * eb * Hkv * D * new

"""The seeded input recipe: determinism, shapes, bf16 rounding, cfg-5 draws."""
import numpy as np

from synth_inputs import (CONFIG_SPECS, algorithmic_bytes, algorithmic_flops, generate,
                          modality_tags, spec_for_config)


def test_config5_lengths_and_outliers_are_the_documented_draw():
    spec = spec_for_config(5, cache_len_range=(1024, 32768))
    rng = np.random.default_rng([2606, 25041, 5])
    lens = [int(x) for x in rng.integers(1024, 32768, endpoint=True, size=8)]
    assert lens == [21852, 18399, 26008, 19914, 2081, 30893, 27228, 25114]
    assert sum(lens) == 171489 and all(L % 64 for L in lens)
    assert spec.num_sessions == 8


def test_small_workload_shapes_dtype_and_determinism():
    spec = spec_for_config(5, cache_len_range=(10, 40), block_tokens=16, modality_split=(8, 6, 2))
    a, b = generate(spec), generate(spec)
    assert a.cache_lens == b.cache_lens and len(a.sessions) == 8
    assert a.outlier_channels.shape == (8, 6)
    for sa, sb, L in zip(a.sessions, b.sessions, a.cache_lens):
        assert sa.k_cache.shape == (L, 8, 128) and sa.q[0].shape == (16, 32, 128)
        assert sa.k_cache.dtype.name == "bfloat16"
        assert sa.k_cache.view(np.uint16).tobytes() == sb.k_cache.view(np.uint16).tobytes()
    # outlier channels are x8: their std is ~8, others ~1
    k = a.sessions[0].k_cache.astype(np.float32)
    ch = a.outlier_channels[0]
    assert k[:, 0, ch].std() > 5.0 and np.delete(k[:, 0, :], ch, axis=1).std() < 1.5


def test_fp32_config1():
    w = generate(spec_for_config(1))
    s = w.sessions[0]
    assert s.k_cache.shape == (0, 2, 64) and len(s.q) == 3 and s.q[0].dtype == np.float32
    assert list(w.modality) == [0] * 4 + [1] * 3 + [2] + [0] * 4 + [1] * 3 + [2]


def test_modality_tags_counts():
    t = modality_tags(256, (192, 48, 16))
    assert (t == 0).sum() == 192 and (t == 1).sum() == 48 and (t == 2).sum() == 16
    assert list(t[:64]) == [0] * 48 + [1] * 12 + [2] * 4
    assert len(modality_tags(512, (384, 96, 32))) == 512


def test_algorithmic_work_matches_baseline_table():
    s4 = CONFIG_SPECS[4]
    assert abs(algorithmic_flops(s4, [65536]) / 1e9 - 275.95) < 0.01
    assert abs(algorithmic_bytes(s4, [65536]) / 1e6 - 275.78) < 0.01
    assert abs(algorithmic_flops(s4, [65536], step=19) / 1e9 - 296.35) < 0.01
    s2 = CONFIG_SPECS[2]
    assert abs(algorithmic_flops(s2, [4096]) / 1e9 - 9.127) < 0.001
    assert abs(algorithmic_bytes(s2, [4096]) / 1e6 - 41.94) < 0.01

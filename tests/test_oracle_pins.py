"""Pins for the float64 oracle (CPU only).  Each test fixes the oracle to something OTHER than itself:
hand-derived values (tests/golden/), closed forms, a brute-force formulation, torch's SDPA on the
special cases where block-causal attention reduces to a library routine, and invariants that follow
from Eq. (1).  A dropped term, wrong sign/index or transposed operand in
oracle/block_causal.py fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle.block_causal import OracleSession, attend, attend_range, fm_euler_update, merge_partials
from oracle.brute_force import dense_block_causal
from synth_inputs import generate, spec_for_config

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([float(x) for x in line.split()])
    return np.array(rows)


def _stream(block_sizes, Hq, Hkv, D, seed, dtype=np.float64):
    rng = np.random.default_rng(seed)
    T = sum(block_sizes)
    return (rng.standard_normal((T, Hq, D)).astype(dtype),
            rng.standard_normal((T, Hkv, D)).astype(dtype),
            rng.standard_normal((T, Hkv, D)).astype(dtype))


def _incremental(q, k, v, block_sizes, scale, q_to_kv=None):
    """append block t then attend with block t's queries (the hot path), for every t."""
    Hkv, D = k.shape[1], k.shape[2]
    sess = OracleSession(Hkv, D)
    outs, lses, pos = [], [], 0
    for sz in block_sizes:
        sess.append(k[pos:pos + sz], v[pos:pos + sz])
        o, l = attend(sess, q[pos:pos + sz], scale, 1, q_to_kv)
        outs.append(o); lses.append(l); pos += sz
    return np.concatenate(outs), np.concatenate(lses), sess


def _one_shot(q, k, v, block_sizes, scale, q_to_kv=None):
    sess = OracleSession(k.shape[1], k.shape[2])
    pos = 0
    for sz in block_sizes:
        sess.append(k[pos:pos + sz], v[pos:pos + sz]); pos += sz
    return attend(sess, q, scale, len(block_sizes), q_to_kv)


# ---------------------------------------------------------------- P0 hand example (golden)
def _p0_inputs():
    a = np.array([1.0, 2.0, 3.0, 4.0])
    q = np.tile(np.array([1.0, 0.0]), (4, 1, 1))
    k = np.stack([np.log(a), np.zeros(4)], axis=1)[:, None, :]
    v = np.array([[1.0, 0.0], [0.0, 1.0], [2.0, 0.0], [0.0, 2.0]])[:, None, :]
    return q, k, v


def test_p0_hand_example_incremental_and_one_shot():
    gold = _load("p0_hand_example.txt")
    q, k, v = _p0_inputs()
    for fn in (_incremental, _one_shot):
        res = fn(q, k, v, [2, 2], 1.0)
        o, lse = res[0], res[1]
        np.testing.assert_allclose(o[:, 0, :], gold[:, 1:3], rtol=0, atol=1e-15)
        np.testing.assert_allclose(np.exp(lse[:, 0]), gold[:, 3], rtol=1e-15)


def test_p0_separates_wrong_mask_readings():
    """token-causal and no-mask readings give different row-0 values than the golden file."""
    gold = _load("p0_hand_example.txt")
    q, k, v = _p0_inputs()
    o_tc, _ = dense_block_causal(q, k, v, [2, 2], 1.0, mask_kind="token_causal")
    o_nm, _ = dense_block_causal(q, k, v, [2, 2], 1.0, mask_kind="none")
    assert abs(o_tc[0][0][0] - gold[0, 1]) > 0.5          # (1,0) vs (1/3,2/3)
    assert abs(o_nm[0][0][0] - gold[0, 1]) > 0.3          # (0.7,1.0) vs (1/3,2/3)
    o_bc, lse_bc = dense_block_causal(q, k, v, [2, 2], 1.0)
    np.testing.assert_allclose(np.array(o_bc)[:, 0, :], gold[:, 1:3], atol=1e-15)
    np.testing.assert_allclose(np.exp(np.array(lse_bc)[:, 0]), gold[:, 3], rtol=1e-15)


# ---------------------------------------------------------------- P1 / P4 closed forms (golden)
def test_p1_p4_closed_forms_config1_geometry():
    gold = _load("p1_p4_closed_forms.txt")
    Hq = Hkv = 2; D = 64
    rng = np.random.default_rng(7)
    k = rng.standard_normal((48, Hkv, D))                   # any K: Q == 0 makes scores equal
    v = np.broadcast_to(np.arange(48.0)[:, None, None], (48, Hkv, D)).copy()
    q = np.zeros((48, Hq, D))
    for fn in (_incremental, _one_shot):
        res = fn(q, k, v, [16, 16, 16], 0.125)
        o, lse = res[0], res[1]
        for b, e, oval, cnt in gold:
            sl = slice(int(e) - 16, int(e))
            np.testing.assert_allclose(o[sl], oval, rtol=1e-14)
            np.testing.assert_allclose(lse[sl], math.log(cnt), rtol=1e-14)


def test_p4_visible_count_long():
    """all keys equal => LSE = s + ln(N); one missing key would move it by ln(N/(N-1))."""
    N, D = 4352, 16
    sess = OracleSession(1, D)
    kk = np.full((N, 1, D), 0.25)
    sess.append(kk[:4096], kk[:4096]); sess.append(kk[4096:], kk[4096:])
    q = np.ones((256, 1, D))
    _, lse = attend(sess, q, 0.5)
    np.testing.assert_allclose(lse, 0.5 * D * 0.25 + math.log(N), rtol=1e-14)


# ---------------------------------------------------------------- P2 softmax weights
def test_p2_two_key_weights():
    D = 64
    e1 = np.zeros(D); e1[0] = 1.0
    q = (8.0 * e1)[None, None, :]
    k = np.stack([math.log(3.0) * e1, np.zeros(D)])[:, None, :]
    v = np.random.default_rng(3).standard_normal((2, 1, D))
    sess = OracleSession(1, D)
    sess.append(k[:1], v[:1]); sess.append(k[1:], v[1:])
    o, lse = attend(sess, q, 0.125)                          # s1 - s2 = ln 3 -> weights 3/4, 1/4
    np.testing.assert_allclose(o[0, 0], 0.75 * v[0, 0] + 0.25 * v[1, 0], rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(lse[0, 0], math.log(4.0), rtol=1e-14)


# ---------------------------------------------------------------- P3 needle (addressing)
@pytest.mark.parametrize("jstar", [0, 63, 64, 127, 128, 299, 300, 331])
def test_p3_needle(jstar):
    L, n, D = 300, 32, 32
    rng = np.random.default_rng(11)
    u = rng.choice([-1.0, 1.0], size=D)
    k = np.zeros((L + n, 1, D)); k[jstar, 0] = 4.0 * u          # s = 4*D*scale at the needle
    v = rng.standard_normal((L + n, 1, D))
    sess = OracleSession(1, D)
    sess.append(k[:L], v[:L]); sess.append(k[L:], v[L:])
    q = np.tile(u, (n, 1, 1))
    o, _ = attend(sess, q, 1.0)                              # needle score 128, others 0
    np.testing.assert_allclose(o[:, 0, :], np.tile(v[jstar, 0], (n, 1)), atol=1e-12)


# ---------------------------------------------------------------- P5 shift invariance / stability
def test_p5_shift_invariance_and_large_scores():
    q, k, v = _stream([8, 8], 2, 1, 16, seed=5)
    c = np.random.default_rng(6).standard_normal(16) * 10.0
    o0, l0, _ = _incremental(q, k, v, [8, 8], 0.25)
    o1, l1, _ = _incremental(q, k + c, v, [8, 8], 0.25)
    np.testing.assert_allclose(o1, o0, rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(l1 - l0, 0.25 * np.einsum("rhd,d->rh", q, c), rtol=1e-9, atol=1e-9)
    o2, l2, _ = _incremental(q * 40, k * 40, v, [8, 8], 1.0)  # |scores| in the thousands
    assert np.isfinite(o2).all() and np.isfinite(l2).all()


# ---------------------------------------------------------------- P6 rows sum to one
def test_p6_constant_v_gives_constant_o():
    q, k, v = _stream([5, 7, 3], 4, 2, 8, seed=9)
    v[:] = 1.75
    o, _, _ = _incremental(q, k, v, [5, 7, 3], 0.3)
    np.testing.assert_allclose(o, 1.75, rtol=1e-14)


# ---------------------------------------------------------------- brute force on tiny inputs
@pytest.mark.parametrize("blocks,Hq,Hkv,D", [
    ([3, 1, 4], 2, 1, 2), ([1, 1, 1, 1], 1, 1, 1), ([9], 4, 4, 8), ([2, 5], 4, 2, 3),
    ([7, 2, 6, 1], 4, 1, 8), ([4, 9, 2], 2, 2, 5),
])
def test_oracle_vs_brute_force_random_tiny(blocks, Hq, Hkv, D):
    q, k, v = _stream(blocks, Hq, Hkv, D, seed=100 + sum(blocks) + Hq + D)
    scale = 0.7 / math.sqrt(D)
    o_bf, l_bf = dense_block_causal(q, k, v, blocks, scale)
    o_inc, l_inc, _ = _incremental(q, k, v, blocks, scale)
    o_one, l_one = _one_shot(q, k, v, blocks, scale)
    np.testing.assert_allclose(o_inc, np.array(o_bf), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(l_inc, np.array(l_bf), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(o_one, np.array(o_bf), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(l_one, np.array(l_bf), rtol=1e-12, atol=1e-13)


def test_oracle_vs_brute_force_config1_exact_shape():
    """BASELINE configs[0] at its real size: 3 blocks x 16 tokens, 2 heads, D=64, seeded inputs."""
    w = generate(spec_for_config(1))
    s = w.sessions[0]
    q = np.concatenate(s.q); k = np.concatenate(s.k); v = np.concatenate(s.v)
    o_bf, l_bf = dense_block_causal(q, k, v, [16, 16, 16], w.spec.scale)
    o_inc, l_inc, _ = _incremental(q, k, v, [16, 16, 16], w.spec.scale)
    np.testing.assert_allclose(o_inc, np.array(o_bf), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(l_inc, np.array(l_bf), rtol=1e-12, atol=1e-13)


def test_explicit_q_to_kv_map():
    q, k, v = _stream([3, 4], 4, 2, 4, seed=21)
    mapping = [1, 0, 0, 1]
    o_bf, _ = dense_block_causal(q, k, v, [3, 4], 0.5, q_to_kv=mapping)
    o, _, _ = _incremental(q, k, v, [3, 4], 0.5, q_to_kv=mapping)
    np.testing.assert_allclose(o, np.array(o_bf), rtol=1e-12, atol=1e-13)


# ---------------------------------------------------------------- library-routine special cases
def _sdpa(q, k, v, scale, causal):
    qt = torch.from_numpy(q).permute(1, 0, 2)[None]           # [1, H, T, D]
    kt = torch.from_numpy(k).permute(1, 0, 2)[None]
    vt = torch.from_numpy(v).permute(1, 0, 2)[None]
    o = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, is_causal=causal, scale=scale)
    return o[0].permute(1, 0, 2).numpy()


def test_single_block_is_plain_noncausal_sdpa():
    q, k, v = _stream([37], 3, 3, 24, seed=31)                 # T != D, non-square everything
    o, _, _ = _incremental(q, k, v, [37], 0.2)
    np.testing.assert_allclose(o, _sdpa(q, k, v, 0.2, False), rtol=1e-10, atol=1e-12)


def test_blocks_of_one_token_is_standard_causal_attention():
    q, k, v = _stream([1] * 19, 2, 2, 12, seed=32)
    o, _, _ = _incremental(q, k, v, [1] * 19, 0.3)
    np.testing.assert_allclose(o, _sdpa(q, k, v, 0.3, True), rtol=1e-10, atol=1e-12)
    o1, _ = _one_shot(q, k, v, [1] * 19, 0.3)
    np.testing.assert_allclose(o1, _sdpa(q, k, v, 0.3, True), rtol=1e-10, atol=1e-12)


def test_gqa_equals_mha_with_repeated_kv_heads():
    q, k, v = _stream([6, 10], 8, 2, 16, seed=33)
    o_gqa, l_gqa, _ = _incremental(q, k, v, [6, 10], 0.25)
    kr = np.repeat(k, 4, axis=1); vr = np.repeat(v, 4, axis=1)
    o_mha, l_mha, _ = _incremental(q, kr, vr, [6, 10], 0.25)
    np.testing.assert_array_equal(o_gqa, o_mha)
    np.testing.assert_array_equal(l_gqa, l_mha)
    # and against torch SDPA per block (block 2 sees everything => non-causal over all 16 keys)
    np.testing.assert_allclose(o_gqa[6:], _sdpa(q[6:], kr, vr, 0.25, False)[:],
                               rtol=1e-10, atol=1e-12)


# ---------------------------------------------------------------- invariants from Eq. (1)
def test_prefix_invariance_bit_identical():
    blocks = [5, 8, 3, 6]
    q, k, v = _stream(blocks, 2, 2, 8, seed=41)
    o0, l0, _ = _incremental(q, k, v, blocks, 0.35)
    q2, k2, v2 = q.copy(), k.copy(), v.copy()
    q2[13:] += 3.0; k2[13:] *= -2.0; v2[13:] += 100.0          # perturb blocks 3 and 4 only
    o1, l1, _ = _incremental(q2, k2, v2, blocks, 0.35)
    np.testing.assert_array_equal(o0[:13], o1[:13])
    np.testing.assert_array_equal(l0[:13], l1[:13])
    assert np.abs(o0[13:] - o1[13:]).max() > 1.0
    oa, _ = _one_shot(q, k, v, blocks, 0.35); ob, _ = _one_shot(q2, k2, v2, blocks, 0.35)
    np.testing.assert_array_equal(oa[:13], ob[:13])


def test_incremental_equals_one_shot():
    blocks = [16, 16, 16]
    q, k, v = _stream(blocks, 2, 2, 64, seed=42)
    o_i, l_i, _ = _incremental(q, k, v, blocks, 0.125)
    o_o, l_o = _one_shot(q, k, v, blocks, 0.125)
    np.testing.assert_allclose(o_i, o_o, rtol=0, atol=1e-13)
    np.testing.assert_allclose(l_i, l_o, rtol=0, atol=1e-13)


def test_intra_block_bidirectional_permutation_equivariance():
    """permuting the tokens of the newest block permutes its output rows (PAPER.md:59 coupling)."""
    q, k, v = _stream([10, 12], 2, 1, 8, seed=43)
    o0, _, _ = _incremental(q, k, v, [10, 12], 0.4)
    perm = np.random.default_rng(1).permutation(12)
    q2, k2, v2 = q.copy(), k.copy(), v.copy()
    q2[10:] = q[10:][perm]; k2[10:] = k[10:][perm]; v2[10:] = v[10:][perm]
    o1, _, _ = _incremental(q2, k2, v2, [10, 12], 0.4)
    np.testing.assert_allclose(o1[10:], o0[10:][perm], rtol=1e-12, atol=1e-14)
    # a later token inside the block IS visible: changing the last token changes row 0 of the block
    v3 = v.copy(); v3[-1] += 50.0
    o3, _, _ = _incremental(q, k, v3, [10, 12], 0.4)
    assert np.abs(o3[10] - o0[10]).max() > 1e-3
    np.testing.assert_array_equal(o3[:10], o0[:10])


def test_kv_row_permutation_inside_visible_range_leaves_output():
    q, k, v = _stream([20, 4], 2, 2, 8, seed=44)
    perm = np.random.default_rng(2).permutation(20)
    o0, _, _ = _incremental(q, k, v, [20, 4], 0.3)
    k2, v2 = k.copy(), v.copy(); k2[:20] = k[:20][perm]; v2[:20] = v[:20][perm]
    o1, _, _ = _incremental(q, k2, v2, [20, 4], 0.3)
    np.testing.assert_allclose(o1[20:], o0[20:], rtol=1e-12, atol=1e-14)


def test_append_is_bit_exact_concatenation():
    rng = np.random.default_rng(45)
    sess = OracleSession(2, 4)
    bits = rng.integers(0, 65536, size=(23, 2, 4), dtype=np.uint16)   # incl. NaN/Inf/denormals
    vbits = rng.integers(0, 65536, size=(23, 2, 4), dtype=np.uint16)
    import ml_dtypes
    kb = bits.view(ml_dtypes.bfloat16); vb = vbits.view(ml_dtypes.bfloat16)
    for lo, hi in [(0, 7), (7, 8), (8, 23)]:
        sess.append(kb[lo:hi], vb[lo:hi])
    kg, vg = sess.gather()
    assert kg.view(np.uint16).tobytes() == bits.tobytes()
    assert vg.view(np.uint16).tobytes() == vbits.tobytes()
    assert sess.block_ends == [0, 7, 8, 23]
    k2, _ = sess.gather(5, 6)
    assert k2.view(np.uint16).tobytes() == bits[5:11].tobytes()


# ---------------------------------------------------------------- split-KV merge identity (a4)
@pytest.mark.parametrize("cuts", [[0, 40], [0, 17, 40], [0, 1, 2, 40], [0, 13, 13, 29, 40]])
def test_merge_identity(cuts):
    q, k, v = _stream([30, 10], 4, 2, 8, seed=46)
    sess = OracleSession(2, 8)
    sess.append(k[:30], v[:30]); sess.append(k[30:], v[30:])
    o_full, l_full = attend(sess, q[30:], 0.4)
    parts = [attend_range(sess, q[30:], 0.4, cuts[i], cuts[i + 1]) for i in range(len(cuts) - 1)]
    o, l = merge_partials(np.stack([p[0] for p in parts]), np.stack([p[1] for p in parts]))
    np.testing.assert_allclose(o, o_full, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(l, l_full, rtol=1e-12, atol=1e-14)


def test_merge_partials_hand_values():
    """two splits with exp(LSE) = 1 and 3 -> weights 1/4, 3/4 (hand-derived)."""
    o = np.array([[[4.0, 0.0]], [[0.0, 8.0]]])
    lse = np.array([[0.0], [math.log(3.0)]])
    om, lm = merge_partials(o, lse)
    np.testing.assert_allclose(om, [[1.0, 6.0]], rtol=1e-15)
    np.testing.assert_allclose(lm, [math.log(4.0)], rtol=1e-15)


def test_rows_subset_matches_full():
    q, k, v = _stream([12, 9], 4, 2, 8, seed=47)
    sess = OracleSession(2, 8)
    sess.append(k[:12], v[:12]); sess.append(k[12:], v[12:])
    o, l = attend(sess, q, 0.3, num_q_blocks=2)
    o_s, l_s = attend(sess, q, 0.3, num_q_blocks=2, rows=[0, 11, 12, 20], heads=[3, 1])
    np.testing.assert_allclose(o_s, o[[0, 11, 12, 20]][:, [3, 1]], rtol=0, atol=1e-14)
    np.testing.assert_allclose(l_s, l[[0, 11, 12, 20]][:, [3, 1]], rtol=0, atol=1e-14)


# ---------------------------------------------------------------- NEXT-2: flow-matching Euler step
def test_fm_euler_exact_velocity_recovers_clean_latent():
    """Eq. (2): z_tau = (1-tau) z0 + tau eps, velocity eps - z0.  One Euler step of size
    -tau with the exact velocity returns z0; a step of +(1-tau) returns eps (closed form)."""
    rng = np.random.default_rng(51)
    z0, eps = rng.standard_normal((5, 7)), rng.standard_normal((5, 7))
    for tau in (1.0, 0.6, 0.25):
        zt = (1 - tau) * z0 + tau * eps
        np.testing.assert_allclose(fm_euler_update(zt, eps - z0, -tau), z0, rtol=0, atol=1e-15)
        np.testing.assert_allclose(fm_euler_update(zt, eps - z0, 1 - tau), eps, rtol=0, atol=1e-15)
    # hand value: z = 2, v = 4, dtau = -0.25 -> 1
    assert fm_euler_update(np.array([2.0]), np.array([4.0]), -0.25)[0] == 1.0


def test_abs_weighted_output_pins():
    """attend(want_abs=True): A = sum_j w_j |v_j| (the condition number the bf16 error bound of the GPU
    tests is stated with).  Pins: V >= 0  =>  A == O; flipping the sign of V rows leaves A unchanged and
    |O| <= A always; hand example P0 with V negated on key 1: rows 0,1 -> A = (1/3, 2/3), O = (1/3, -2/3)."""
    q, k, v = _stream([5, 7, 4], 4, 2, 8, seed=91)
    sess = OracleSession(2, 8)
    pos = 0
    for b in (5, 7, 4):
        sess.append(k[pos:pos + b], np.abs(v[pos:pos + b])); pos += b
    o, lse, a = attend(sess, q[-4:], 0.3, want_abs=True)
    np.testing.assert_allclose(a, o, rtol=0, atol=1e-15)
    sess2 = OracleSession(2, 8)
    pos = 0
    sign = np.where(np.arange(16) % 3 == 0, -1.0, 1.0)[:, None, None]
    for b in (5, 7, 4):
        sess2.append(k[pos:pos + b], (np.abs(v) * sign)[pos:pos + b]); pos += b
    o2, lse2, a2 = attend(sess2, q[-4:], 0.3, want_abs=True)
    np.testing.assert_allclose(a2, a, rtol=0, atol=1e-15)
    np.testing.assert_array_equal(lse2, lse)
    assert (np.abs(o2) <= a2 + 1e-15).all() and np.abs(o2 - o).max() > 1e-3
    # P0 geometry (tests/golden/p0_hand_example.txt) with V[1] negated
    s0 = OracleSession(1, 2)
    kk = np.log(np.array([1.0, 2.0, 3.0, 4.0]))
    K = np.stack([kk, np.zeros(4)], axis=1)[:, None, :]
    V = np.array([[1.0, 0.0], [0.0, -1.0], [2.0, 0.0], [0.0, 2.0]])[:, None, :]
    s0.append(K[:2], V[:2])
    Q = np.tile(np.array([1.0, 0.0]), (2, 1, 1))
    o0, _, a0 = attend(s0, Q, 1.0, want_abs=True)
    np.testing.assert_allclose(o0[:, 0], [[1 / 3, -2 / 3]] * 2, atol=1e-15)
    np.testing.assert_allclose(a0[:, 0], [[1 / 3, 2 / 3]] * 2, atol=1e-15)


# ---------------------------------------------------------------- NEXT-4: text-causal mixed mask (reading A19)
def _tc_run(q, k, v, block_sizes, tags, scale, one_shot, q_to_kv=None):
    """Oracle with text_causal=True, either block by block (hot path) or all blocks in one query."""
    sess = OracleSession(k.shape[1], k.shape[2])
    tags = np.asarray(tags, dtype=np.uint8)
    outs, lses, pos = [], [], 0
    for sz in block_sizes:
        sess.append(k[pos:pos + sz], v[pos:pos + sz], modality=tags[pos:pos + sz])
        if not one_shot:
            o, l = attend(sess, q[pos:pos + sz], scale, 1, q_to_kv, text_causal=True)
            outs.append(o); lses.append(l)
        pos += sz
    if one_shot:
        return attend(sess, q, scale, len(block_sizes), q_to_kv, text_causal=True)
    return np.concatenate(outs), np.concatenate(lses)


def _p7_inputs():
    a = np.arange(1.0, 7.0)
    q = np.tile(np.array([1.0, 0.0]), (6, 1, 1))
    k = np.stack([np.log(a), np.zeros(6)], axis=1)[:, None, :]
    v = np.array([[1.0, 0.0], [0.0, 1.0], [2.0, 0.0], [0.0, 2.0], [3.0, 0.0], [0.0, 3.0]])[:, None, :]
    return q, k, v, [3, 3], [0, 2, 2, 2, 2, 1]


def test_p7_text_causal_hand_example():
    """tests/golden/p7_text_causal_hand_example.txt (hand-derived): oracle (incremental and one-shot) and the
    brute-force dense mask agree with it; plain block-causal and token-causal do not."""
    gold = _load("p7_text_causal_hand_example.txt")
    q, k, v, blocks, tags = _p7_inputs()
    for one_shot in (False, True):
        o, lse = _tc_run(q, k, v, blocks, tags, 1.0, one_shot)
        np.testing.assert_allclose(o[:, 0, :], gold[:, 1:3], rtol=0, atol=1e-15)
        np.testing.assert_allclose(np.exp(lse[:, 0]), gold[:, 3], rtol=1e-14)
    o_bf, lse_bf = dense_block_causal(q, k, v, blocks, 1.0, mask_kind="text_causal", tags=tags)
    np.testing.assert_allclose(np.array(o_bf)[:, 0, :], gold[:, 1:3], atol=1e-15)
    np.testing.assert_allclose(np.exp(np.array(lse_bf)[:, 0]), gold[:, 3], rtol=1e-14)
    o_bc, _ = _one_shot(q, k, v, blocks, 1.0)
    assert abs(o_bc[1, 0, 0] - gold[1, 1]) > 0.5 and abs(o_bc[3, 0, 0] - gold[3, 1]) > 0.5
    o_tok, _ = dense_block_causal(q, k, v, blocks, 1.0, mask_kind="token_causal")
    assert abs(o_tok[0][0][0] - gold[0, 1]) > 0.1


@pytest.mark.parametrize("blocks,Hq,Hkv,D", [([5, 3, 7], 2, 1, 4), ([1, 6, 2, 4], 4, 2, 3), ([9], 1, 1, 5)])
def test_text_causal_vs_brute_force_random_tiny(blocks, Hq, Hkv, D):
    q, k, v = _stream(blocks, Hq, Hkv, D, seed=71)
    rng = np.random.default_rng(72)
    tags = rng.integers(0, 3, size=sum(blocks))
    o_bf, lse_bf = dense_block_causal(q, k, v, blocks, 0.4, mask_kind="text_causal", tags=list(tags))
    for one_shot in (False, True):
        o, lse = _tc_run(q, k, v, blocks, tags, 0.4, one_shot)
        np.testing.assert_allclose(o, np.array(o_bf), rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(lse, np.array(lse_bf), rtol=1e-12, atol=1e-13)


def test_text_causal_without_text_tokens_is_block_causal_bit_identical():
    blocks = [4, 6, 3]
    q, k, v = _stream(blocks, 2, 2, 8, seed=73)
    tags = np.random.default_rng(74).integers(0, 2, size=sum(blocks))      # video / audio only
    o, lse = _tc_run(q, k, v, blocks, tags, 0.3, True)
    o_ref, lse_ref = _one_shot(q, k, v, blocks, 0.3)
    assert o.tobytes() == o_ref.tobytes() and lse.tobytes() == lse_ref.tobytes()


def test_text_causal_all_text_single_block_is_causal_sdpa():
    """Library pin: one block whose tokens are all text = standard causal attention."""
    q, k, v = _stream([23], 3, 3, 16, seed=75)
    o, _ = _tc_run(q, k, v, [23], [2] * 23, 0.25, True)
    np.testing.assert_allclose(o, _sdpa(q, k, v, 0.25, True), rtol=1e-10, atol=1e-12)
    # ... and all-text blocks of any sizes are token-causal too (text never sees later text)
    o2, _ = _tc_run(q, k, v, [5, 11, 7], [2] * 23, 0.25, False)
    np.testing.assert_allclose(o2, _sdpa(q, k, v, 0.25, True), rtol=1e-10, atol=1e-12)


def test_text_causal_dependence_structure():
    """Perturbing a LATER text token of the block changes the A/V rows and the later text rows of that block,
    and leaves earlier text rows bit-identical; perturbing a later A/V token changes every row of the block."""
    blocks, tags = [8], [0, 2, 1, 2, 0, 2, 1, 2]
    q, k, v = _stream(blocks, 2, 1, 8, seed=76)
    o0, _ = _tc_run(q, k, v, blocks, tags, 0.5, True)
    k2, v2 = k.copy(), v.copy()
    k2[5] += 1.0; v2[5] -= 2.0                                  # text token at position 5
    o1, _ = _tc_run(q, k2, v2, blocks, tags, 0.5, True)
    for r in (1, 3):                                           # earlier text rows: unchanged
        assert o1[r].tobytes() == o0[r].tobytes()
    for r in (0, 2, 4, 5, 6, 7):                               # A/V rows, the token itself, later text
        assert np.abs(o1[r] - o0[r]).max() > 1e-6
    k3, v3 = k.copy(), v.copy()
    k3[6] += 1.0; v3[6] -= 2.0                                  # audio token at position 6
    o2, _ = _tc_run(q, k3, v3, blocks, tags, 0.5, True)
    assert all(np.abs(o2[r] - o0[r]).max() > 1e-6 for r in range(8))

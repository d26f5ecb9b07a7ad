"""Pins for oracle/rotattn_oracle.py against what the paper and the mathematics fix (CPU only).

Each test names the passage it pins.  They are chosen so that a plausible mistake (dropped term,
wrong sign/index, transposed operand, wrong rounding) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
from scipy.linalg import hadamard as scipy_hadamard

from oracle import rotattn_oracle as orc
from synth import video_qkv as syn

GOLD = os.path.join(os.path.dirname(__file__), 'golden')


GRID = (4, 6, 10)          # Hh != W and P_h != P_w below: none of the pins is symmetric in the h and w axes
PAIRS = (12, 9, 11)
N0 = GRID[0] * GRID[1] * GRID[2]


def _params(rot_mode=orc.ROT_HALF, **kw):
    base = dict(B=1, H=1, N=N0, D=64, grid=GRID, pairs=PAIRS, rot_mode=rot_mode)
    base.update(kw)
    return orc.Params(**base)


def _rand_o2(rng, n):
    """random O(2) blocks, half of them reflections (det -1)."""
    th = rng.uniform(0, 2 * np.pi, n)
    c, s = np.cos(th), np.sin(th)
    blk = np.stack([c, s, -s, c], axis=1)
    refl = rng.random(n) < 0.5
    blk[refl, 2] *= -1
    blk[refl, 3] *= -1
    return blk


def _read_rows(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith('#'):
                rows.append(line.split())
    return rows


# ---------------------------------------------------------------- Eq.4, Eq.3
def test_h2_printed_matrix():
    rows = _read_rows('eq4_h2.txt')
    M = np.array([[float(x) for x in rows[0]], [float(x) for x in rows[1]]])
    denom2 = float(rows[2][0])
    assert np.allclose(orc.h2(), M / math.sqrt(denom2), atol=1e-15)
    ok, err = orc.check_orthogonal(orc.default_rot(64))
    assert ok and err < 1e-15


def test_check_orthogonal_rejects_scaling():
    bad = orc.default_rot(8).copy()
    bad[3] *= 1.01            # sigma != 1
    ok, _ = orc.check_orthogonal(bad)
    assert not ok


# ---------------------------------------------------------------- Eq.13, Eq.14
@pytest.mark.parametrize('n', [2, 4, 64, 128])
def test_hadamard_recursion_and_library(n):
    Hpm = orc.hadamard_pm1(n)
    assert np.array_equal(Hpm @ Hpm.T, n * np.eye(n, dtype=np.int64))       # H H^T = n I exactly
    assert np.array_equal(Hpm, scipy_hadamard(n))                            # library Sylvester matrix
    if n >= 4:
        half = orc.hadamard_pm1(n // 2)
        assert np.array_equal(Hpm, np.kron(np.array([[1, 1], [1, -1]]), half))   # Eq.13
    H = orc.hadamard(n)
    assert np.allclose(H @ H.T, np.eye(n), atol=1e-12)
    V = np.random.default_rng(0).standard_normal((7, n))
    assert np.allclose((V @ H) @ H.T, V, atol=1e-12)                         # Eq.14


# ---------------------------------------------------------------- token <-> position (reading 4)
def test_token_positions_golden_asymmetric_grid():
    rows = _read_rows('token_positions_2x3x5.txt')
    t, h, w, is_rope = orc.token_positions(31, (2, 3, 5))
    for n, gt, gh, gw, gr in ((int(x) for x in r) for r in rows):
        assert (int(t[n]), int(h[n]), int(w[n]), int(is_rope[n])) == (gt, gh, gw, gr), n
    # the library's row-major unravel is the same map (w fastest) on every video token of a second asymmetric grid
    t, h, w, is_rope = orc.token_positions(N0 + 2, GRID)
    ut, uh, uw = np.unravel_index(np.arange(N0), GRID)
    assert np.array_equal(t[:N0], ut) and np.array_equal(h[:N0], uh) and np.array_equal(w[:N0], uw)
    assert is_rope[:N0].all() and not is_rope[N0:].any()


# ---------------------------------------------------------------- RoPE (L58-62)
def test_rope_textbook_properties():
    p = _params()
    rng = np.random.default_rng(1)
    x = rng.standard_normal((p.N, p.D))
    y = orc.rope_fp64(p, x)
    assert np.allclose(y[0], x[0], atol=1e-14)                               # position (0,0,0): identity
    # norm of every adjacent pair preserved (M_i in SO(2))
    nx = x[:, 0::2] ** 2 + x[:, 1::2] ** 2
    ny = y[:, 0::2] ** 2 + y[:, 1::2] ** 2
    assert np.allclose(nx, ny, rtol=1e-12)
    # complex-number formulation: (x0 + i x1) e^{i theta}
    t, h, w = np.unravel_index(np.arange(p.N), p.grid)       # library row-major map, not the oracle's own
    pos = np.concatenate([np.repeat(x[:, None], P, 1) for x, P in zip((t, h, w), p.pairs)], axis=1)
    fr = np.concatenate([10000.0 ** (-np.arange(P) / P) for P in p.pairs])
    z = (x[:, 0::2] + 1j * x[:, 1::2]) * np.exp(1j * pos * fr[None, :])
    assert np.allclose(y[:, 0::2], z.real, atol=1e-10) and np.allclose(y[:, 1::2], z.imag, atol=1e-10)


def test_rope_pairwise_form_equals_dense_form():
    p = _params(N=N0 + 4)
    rng = np.random.default_rng(36)
    x = rng.standard_normal((p.N, p.D))
    for mode in (orc.ROT_NONE, orc.ROT_HALF, orc.ROT_FULL):
        assert np.abs(orc.rope_fp64_pairs(p, x, mode) - orc.rope_fp64(p, x, mode)).max() <= 1e-12


def test_rope_relative_position_property():
    """Shifting every position of one axis by a constant leaves Q_r K_r^T unchanged."""
    p = _params()
    T, Hh, W = p.grid
    rng = np.random.default_rng(2)
    # raw q,k that do not depend on t: then scores between (t1,.) and (t2,.) depend on t1-t2 only
    qf = rng.standard_normal((Hh * W, p.D))
    kf = rng.standard_normal((Hh * W, p.D))
    q = np.tile(qf, (T, 1))
    k = np.tile(kf, (T, 1))
    qr, kr = orc.rope_fp64(p, q), orc.rope_fp64(p, k)
    S = qr @ kr.T
    blk = Hh * W
    a = S[0 * blk:1 * blk, 1 * blk:2 * blk]        # t=0 vs t=1
    b = S[2 * blk:3 * blk, 3 * blk:4 * blk]        # t=2 vs t=3
    assert np.allclose(a, b, atol=1e-10)
    c = S[1 * blk:2 * blk, 0 * blk:1 * blk]        # t=1 vs t=0 (opposite offset) must differ
    assert not np.allclose(a, c, atol=1e-3)


def test_frequencies_low_frequency_is_last_pair():
    f = orc.rope_freqs(22, 10000.0)
    assert f[0] == 1.0 and np.all(np.diff(f) < 0)
    assert np.isclose(f[21], 10000.0 ** (-21 / 22))


# ---------------------------------------------------------------- Eq.7 merged vs sequential
def test_merged_table_equals_sequential_and_closed_form():
    p = _params(orc.ROT_INTERLEAVED)
    coef = orc.coef_table(p)
    assert coef.shape == (orc.table_rows(p), 4) and coef.dtype == np.float32
    # closed form: M(theta) H_2 = [[cos phi, -sin phi], [-sin phi, -cos phi]], phi = theta - pi/4
    f = orc.rope_freqs(12, p.rope_base)
    for pos in (0, 1, 3):
        for k in (0, 5, 11):
            phi = pos * f[k] - math.pi / 4
            want = np.array([math.cos(phi), -math.sin(phi), -math.sin(phi), -math.cos(phi)])
            assert np.allclose(coef[pos * 12 + k], want, atol=1e-7)
    # no-RoPE row = R itself
    assert np.allclose(coef[4 * 12 + 3], orc.h2().reshape(4), atol=1e-7)
    # RoPE(x) R == x (M R)   (Eq.7)
    rng = np.random.default_rng(3)
    x16 = rng.standard_normal((p.N, p.D)).astype(np.float16)
    y32 = orc.apply_rope_rot(p, x16, coef)
    seq = orc.rope_fp64(p, x16.astype(np.float64)) @ orc.dense_rotation(p, orc.ROT_INTERLEAVED)
    assert np.allclose(y32, seq, atol=4e-6 * np.abs(seq).max())
    seq2 = orc.rope_fp64(p, x16.astype(np.float64), orc.ROT_INTERLEAVED)
    assert np.allclose(seq, seq2, atol=1e-12)


@pytest.mark.parametrize('mode', [orc.ROT_NONE, orc.ROT_INTERLEAVED, orc.ROT_HALF])
def test_fp32_apply_matches_fp64(mode):
    p = _params(mode, N=N0 + 5)     # 5 text tokens without RoPE
    rng = np.random.default_rng(4)
    rot = _rand_o2(rng, p.D // 2)
    x16 = (rng.standard_normal((p.N, p.D)) * 3).astype(np.float16)
    y32 = orc.apply_rope_rot(p, x16, orc.coef_table(p, rot), rot)
    y64 = orc.rope_fp64(p, x16.astype(np.float64), mode, rot)
    assert np.abs(y32 - y64).max() <= 6e-7 * np.abs(y64).max() * 4
    # text tokens: no RoPE but R still applied (reading 7)
    xt = x16[-5:].astype(np.float64)
    assert np.allclose(y64[-5:], xt @ orc.dense_rotation(p, mode, rot), atol=1e-12)


# ---------------------------------------------------------------- Eq.5 invariance
@pytest.mark.parametrize('mode', [orc.ROT_INTERLEAVED, orc.ROT_HALF])
@pytest.mark.parametrize('randrot', [False, True])
def test_qk_invariance_under_shared_rotation(mode, randrot):
    p = _params(mode, N=N0 + 3)
    rng = np.random.default_rng(5)
    rot = _rand_o2(rng, p.D // 2) if randrot else None
    q = rng.standard_normal((p.N, p.D))
    k = rng.standard_normal((p.N, p.D))
    S0 = orc.rope_fp64(p, q) @ orc.rope_fp64(p, k).T
    S1 = orc.rope_fp64(p, q, mode, rot) @ orc.rope_fp64(p, k, mode, rot).T
    assert np.abs(S0 - S1).max() <= 1e-9 * np.abs(S0).max()
    R = orc.dense_rotation(p, mode, rot)
    assert np.allclose(R.T @ R, np.eye(p.D), atol=1e-12)


def test_half_pairing_structure():
    p = _params(orc.ROT_HALF)
    ident = np.tile(np.array([1.0, 0, 0, 1.0]), (p.D // 2, 1))
    assert np.array_equal(orc.dense_rotation(p, orc.ROT_HALF, ident), np.eye(p.D))
    R = orc.dense_rotation(p, orc.ROT_HALF)
    assert np.allclose(R @ R, np.eye(p.D), atol=1e-12)               # H_2^2 = I
    # channel o_j + i couples only with o_j + i + D_j/2 (Eq.8): sections of 2 P_j channels
    nz = np.abs(R) > 0
    o = 0
    for P in p.pairs:
        for i in range(P):
            assert set(np.nonzero(nz[o + i])[0]) == {o + i, o + i + P}
        o += 2 * P
    # fp32 path with identity blocks is the identity on RoPE output
    x16 = np.random.default_rng(6).standard_normal((p.N, p.D)).astype(np.float16)
    pn = _params(orc.ROT_NONE)
    assert np.array_equal(orc.apply_rope_rot(p, x16, orc.coef_table(p), ident),
                          orc.apply_rope_rot(pn, x16, orc.coef_table(pn)))


def test_half_rotation_flattens_incoherence():
    """L141: Half rotation equalises incoherence when outliers sit in one half-section (Eq.2 metric)."""
    w = syn.TINY
    q16, _, _ = syn.gen_head(w, 0, 0)
    pn = orc.Params(1, 1, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_NONE)
    ph = orc.Params(1, 1, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF)
    psi_n = orc.incoherence(orc.apply_rope_rot(pn, q16, orc.coef_table(pn)))
    psi_h = orc.incoherence(orc.apply_rope_rot(ph, q16, orc.coef_table(ph)))
    assert psi_h.max() < 0.85 * psi_n.max()


def test_incoherence_definition():
    x = np.array([[1.0, -2.0], [3.0, 2.0], [2.0, 6.0]])
    assert np.allclose(orc.incoherence(x), [1.0, 4.0])              # mean (2,2): max |x-mean|


# ---------------------------------------------------------------- "Full" rotation baseline (L208, Eq.13)
@pytest.mark.parametrize('D', [64, 128])
def test_full_rotation_butterfly_is_the_dense_hadamard(D):
    """The fp32 butterfly equals y H_D / sqrt(D) with the library Sylvester matrix; H is symmetric and orthogonal, so
    applying it twice returns y; a unit vector e_c maps to column c of H (catches a wrong stride order or sign)."""
    rng = np.random.default_rng(30)
    y = (rng.standard_normal((37, D)) * 3).astype(np.float32)
    H = scipy_hadamard(D).astype(np.float64) / math.sqrt(D)
    got = orc.fwht_fp32(y)
    want = y.astype(np.float64) @ H
    assert got.dtype == np.float32 and np.abs(got - want).max() <= 8 * 2.0 ** -24 * np.abs(want).max() * math.log2(D)
    assert np.abs(orc.fwht_fp32(got) - y).max() <= 1e-5 * np.abs(y).max()
    e = np.eye(D, dtype=np.float32)
    assert np.allclose(orc.fwht_fp32(e), H, atol=1e-7)
    p = orc.Params(1, 1, 37, D, (1, 1, 37), (D // 2 - 20, 10, 10), rot_mode=orc.ROT_FULL)
    assert np.allclose(orc.dense_rotation(p, orc.ROT_FULL), H, atol=1e-15)


def test_full_rotation_keeps_qk_and_flattens_incoherence():
    """Eq.5 with R = H_D (orthogonal): QK^T unchanged; on the tiny workload the Full rotation spreads the outlier pairs
    over all channels, so max Psi drops at least as much as with Half (L141, L208)."""
    p = _params(orc.ROT_FULL, N=N0 + 3)
    rng = np.random.default_rng(31)
    q, k = rng.standard_normal((p.N, p.D)), rng.standard_normal((p.N, p.D))
    S0 = orc.rope_fp64(p, q) @ orc.rope_fp64(p, k).T
    S1 = orc.rope_fp64(p, q, orc.ROT_FULL) @ orc.rope_fp64(p, k, orc.ROT_FULL).T
    assert np.abs(S0 - S1).max() <= 1e-9 * np.abs(S0).max()
    x16 = (rng.standard_normal((p.N, p.D)) * 2).astype(np.float16)
    y32 = orc.apply_rope_rot(p, x16, orc.coef_table(p))
    y64 = orc.rope_fp64(p, x16.astype(np.float64), orc.ROT_FULL)
    assert np.abs(y32 - y64).max() <= 4e-6 * np.abs(y64).max()
    w = syn.TINY
    q16, _, _ = syn.gen_head(w, 0, 0)
    psi = {}
    for mode in (orc.ROT_NONE, orc.ROT_HALF, orc.ROT_FULL):
        pm = orc.Params(1, 1, w.N, w.D, w.grid, w.pairs, rot_mode=mode)
        psi[mode] = orc.incoherence(orc.apply_rope_rot(pm, q16, orc.coef_table(pm))).max()
    assert psi[orc.ROT_FULL] < psi[orc.ROT_HALF] < psi[orc.ROT_NONE]


# ---------------------------------------------------------------- smoothing (L90, L40, L52)
def test_column_mean_fixed_point_is_order_independent_and_close_to_the_mean():
    rng = np.random.default_rng(32)
    x = (rng.standard_normal((1000, 16)) * np.exp(rng.standard_normal((1, 16)) * 2) + 3.0).astype(np.float32)
    m = orc.column_mean_fixed(x, orc.FIX_QK)
    assert m.dtype == np.float32
    assert np.array_equal(m, orc.column_mean_fixed(x[rng.permutation(1000)], orc.FIX_QK))        # any order of summation
    assert np.abs(m - x.astype(np.float64).mean(axis=0)).max() <= 2.0 ** -21 + 1e-7 * np.abs(x).max()
    v = rng.standard_normal((513, 8)).astype(np.float16)
    mv = orc.column_mean_fixed(v.astype(np.float32), orc.FIX_V)
    assert np.array_equal(mv, v.astype(np.float64).mean(axis=0).astype(np.float32))            # fp16 data: the sum is exact
    # hand-written case: (1 + 2 + 6) / 3 = 3 and (0.5 - 0.25 + 0.125) / 3 = 0.125
    t = np.array([[1.0, 0.5], [2.0, -0.25], [6.0, 0.125]], dtype=np.float32)
    assert np.array_equal(orc.column_mean_fixed(t, orc.FIX_QK), np.array([3.0, 0.125], dtype=np.float32))


def test_smoothing_shifts_are_exact_without_quantisers():
    """The three identities behind the smoothing path, in fp64 on real-valued tensors (no quantiser): K - mean K leaves
    softmax(QK^T) unchanged; (Q - mean Q) K'^T + 1 (mean Q . K'_j) = Q K'^T; softmax(.)(V - mean V) + mean V = softmax(.) V.
    Checked through o_quant(quantize=False) with the k_corr / v_mean arguments, against the plain definition."""
    rng = np.random.default_rng(33)
    N, D = 300, 32
    q = rng.standard_normal((N, D)) + rng.standard_normal((1, D)) * 2      # token-shared biases
    k = rng.standard_normal((N, D)) + rng.standard_normal((1, D)) * 2
    v = rng.standard_normal((N, D)) + rng.standard_normal((1, D)) * 3
    want = orc.o_exact(q, k, v)
    mq, mk, mv = q.mean(0), k.mean(0), v.mean(0)
    qp, kp, vp = q - mq, k - mk, v - mv
    assert np.allclose(orc.o_exact(q, kp, v), want, atol=1e-12)                       # K shift alone
    p = orc.Params(1, 1, N, D, (1, 1, N), (4, 4, 8))
    ones = np.ones(N, dtype=np.float32)
    # "codes" = the real values themselves (quantisers off), unit scales
    O = orc.o_quant(p, qp, ones, kp, ones, vp, np.ones((3, D), dtype=np.float32), quantize=False, k_corr=kp @ mq, v_mean=mv)
    assert np.allclose(O, want, atol=1e-11)
    O_nocorr = orc.o_quant(p, qp, ones, kp, ones, vp, np.ones((3, D), dtype=np.float32), quantize=False, v_mean=mv)
    assert not np.allclose(O_nocorr, want, atol=1e-3)                                 # dropping the rank-1 term is visible


def test_smoothing_helps_on_token_shared_bias():
    """L90 / L40: with a bias shared by all tokens the smoothed INT4 path is closer to exact attention."""
    rng = np.random.default_rng(34)
    N, D = 512, 64
    bias = np.zeros((1, D)); bias[0, rng.choice(D, 6, replace=False)] = rng.uniform(4, 8, 6) * rng.choice([-1, 1], 6)
    q16 = (rng.standard_normal((N, D)) * 0.7 + bias).astype(np.float16)
    k16 = (rng.standard_normal((N, D)) * 0.7 + bias).astype(np.float16)
    v16 = (rng.standard_normal((N, D)) + bias * 0.5).astype(np.float16)
    errs = {}
    for sm in (0, 1):
        p = orc.Params(1, 1, N, D, (8, 8, 8), (12, 10, 10), rot_mode=orc.ROT_NONE, smooth=sm)
        O, pq, _ = orc.int4_attention_head(p, q16, k16, v16)
        ex = orc.o_exact(orc.rope_fp64(p, q16.astype(np.float64)), orc.rope_fp64(p, k16.astype(np.float64)), v16.astype(np.float64))
        errs[sm] = np.abs(O - ex).sum() / np.abs(ex).sum()
        if sm:
            mq, mk, mv = pq['means']
            assert np.abs(pq['q_y'].mean(0)).max() < 1e-3 and np.abs(pq['k_y'].mean(0)).max() < 1e-3
    assert errs[1] < 0.8 * errs[0], errs


# ---------------------------------------------------------------- quantisers (L190)
def test_quantiser_properties():
    rng = np.random.default_rng(7)
    y = (rng.standard_normal((300, 64)) * np.exp(rng.standard_normal((300, 1)))).astype(np.float32)
    y[17] = 0.0
    codes, scale = orc.quant_qk(y)
    assert codes.min() >= -7 and codes.max() <= 7
    err = np.abs(y - codes.astype(np.float32) * scale[:, None])
    assert np.all(err <= scale[:, None] / 2 * (1 + 1e-6))
    nz = np.abs(y).max(axis=1) > 0
    assert np.all(np.abs(codes[nz]).max(axis=1) == 7)
    assert np.all(codes[17] == 0) and scale[17] == 0
    deq = codes.astype(np.float32) * scale[:, None]
    c2, s2 = orc.quant_qk(deq)
    assert np.array_equal(c2, codes)
    # grouped Q/K scale
    cg, sg = orc.quant_qk(y, 128)
    assert sg.shape == (3,) and np.isclose(sg[0], np.abs(y[:128]).max() / 7, rtol=1e-6)
    # rounding is half-to-even on exact ties: amax 7 -> inv 1
    t = np.array([[7.0, 0.5, 1.5, 2.5, -0.5, -1.5, 6.5, 3.49]], dtype=np.float32)
    ct, st = orc.quant_qk(t)
    assert list(ct[0]) == [7, 0, 2, 2, 0, -2, 6, 3] and st[0] == 1.0


def test_grouped_qk_quantiser_every_group():
    """quant_qk(qk_group = 128) (north_star "per-block scales"; reading 28), checked group by group
    on N = 300 = 128 + 128 + 44 (ragged last group) plus an all-zero middle group: scale = amax(group)/7 from an
    independent slice, codes in [-7, 7], |y - code * scale| <= scale / 2, a +-7 in every non-zero group (at the position of
    the group's amax), idempotence, and equality with the per-token routine on a hand-built equivalent problem.  A wrong
    slice, a scale taken from another group or a ragged tail quantised with the wrong extent fails at least one."""
    rng = np.random.default_rng(77)
    N, D, G = 300, 64, 128
    y = (rng.standard_normal((N, D)) * np.exp(rng.standard_normal((N, 1)))).astype(np.float32)
    y[:G] *= 5.0                      # groups of clearly different magnitude: a scale borrowed from a neighbour breaks the error bound
    y[2 * G:] *= 0.05
    codes, scales = orc.quant_qk(y, G)
    assert codes.shape == (N, D) and codes.dtype == np.int8 and scales.shape == (3,) and scales.dtype == np.float32
    bounds = [(0, 128), (128, 256), (256, 300)]
    for g, (lo, hi) in enumerate(bounds):
        blk = y[lo:hi]
        amax = np.abs(blk).max()
        assert scales[g] == np.float32(amax / np.float32(7.0))                    # one fp32 division, of THIS group's amax
        c = codes[lo:hi].astype(np.float32)
        assert c.min() >= -7 and c.max() <= 7
        assert np.all(np.abs(blk - c * scales[g]) <= scales[g] / 2 * (1 + 1e-6))
        i, j = np.unravel_index(np.argmax(np.abs(blk)), blk.shape)
        assert abs(int(codes[lo + i, j])) == 7 and np.sign(codes[lo + i, j]) == np.sign(blk[i, j])
        # the same group as a per-token problem: a [1, n*D] row has the group's amax as its row amax
        c1, s1 = orc.quant_qk(blk.reshape(1, -1))
        assert np.array_equal(c1.reshape(blk.shape), codes[lo:hi]) and s1[0] == scales[g]
    deq = np.concatenate([codes[lo:hi].astype(np.float32) * scales[g] for g, (lo, hi) in enumerate(bounds)])
    c2, s2 = orc.quant_qk(deq, G)
    assert np.array_equal(c2, codes) and np.allclose(s2, scales, rtol=1e-6)
    # an all-zero group gives zero codes and a zero scale without touching its neighbours
    yz = y.copy()
    yz[G:2 * G] = 0.0
    cz, sz = orc.quant_qk(yz, G)
    assert sz[1] == 0 and not cz[G:2 * G].any()
    assert np.array_equal(cz[:G], codes[:G]) and np.array_equal(cz[2 * G:], codes[2 * G:]) and sz[0] == scales[0] and sz[2] == scales[2]
    # N an exact multiple of the group: no phantom group
    c4, s4 = orc.quant_qk(y[:256], G)
    assert s4.shape == (2,) and np.array_equal(c4, codes[:256]) and np.array_equal(s4, scales[:2])


def test_v_group_quantiser():
    rng = np.random.default_rng(8)
    v = rng.standard_normal((300, 16)).astype(np.float16)
    codes, scales = orc.quant_v(v, 128)
    assert scales.shape == (3, 16)
    for g in range(3):
        sl = slice(128 * g, min(300, 128 * (g + 1)))
        am = np.abs(v[sl].astype(np.float32)).max(axis=0)
        assert np.allclose(scales[g], am / 7, rtol=1e-6)
        err = np.abs(v[sl].astype(np.float32) - codes[sl] * scales[g][None, :])
        assert np.all(err <= scales[g][None, :] / 2 * (1 + 1e-6))
        assert np.all(np.abs(codes[sl]).max(axis=0) == 7)


def test_v_scalar_group_quantiser():
    """one V scale per 128-token group (amax over tokens and channels)."""
    rng = np.random.default_rng(35)
    v = (rng.standard_normal((300, 16)) * np.array([1, 4] * 8)).astype(np.float16)
    codes, scales = orc.quant_v(v, 128, orc.VSCALE_GROUP)
    assert scales.shape == (3,)
    for g in range(3):
        sl = slice(128 * g, min(300, 128 * (g + 1)))
        x = v[sl].astype(np.float32)
        assert np.isclose(scales[g], np.abs(x).max() / 7, rtol=1e-6)
        assert np.all(np.abs(x - codes[sl] * scales[g]) <= scales[g] / 2 * (1 + 1e-6))
        assert np.abs(codes[sl]).max() == 7 and codes[sl].min() >= -7
    c2, s2 = orc.quant_v((codes * scales.repeat(128)[:300, None]).astype(np.float16), 128, orc.VSCALE_GROUP)
    # o_quant accepts both scale shapes: a per-group scalar equals the same value repeated over the channels
    p, qc, qs, kc, ks, vc, vs = _tiny_problem()
    vg = vs[:, 0].copy()
    O1 = orc.o_quant(p, qc, qs, kc, ks, vc, vg)
    O2 = orc.o_quant(p, qc, qs, kc, ks, vc, np.repeat(vg[:, None], vc.shape[1], axis=1))
    assert np.array_equal(O1, O2)


def test_qk_block_scales_in_o_quant():
    """qk_group = 128 (north_star "per-block scales"): o_quant picks scale[n // 128]; equals per-token scales repeated."""
    p, qc, qs, kc, ks, vc, vs = _tiny_problem()
    import dataclasses
    pg = dataclasses.replace(p, qk_group=128)
    qg, kg = qs[::128].copy(), ks[::128].copy()
    O1 = orc.o_quant(pg, qc, qg, kc, kg, vc, vs)
    O2 = orc.o_quant(p, qc, np.repeat(qg, 128)[:300], kc, np.repeat(kg, 128)[:300], vc, vs)
    assert np.array_equal(O1, O2)


def test_pack_unpack_all_nibble_pairs():
    vals = np.arange(-8, 8, dtype=np.int8)
    a, b = np.meshgrid(vals, vals, indexing='ij')
    codes = np.stack([a.ravel(), b.ravel()], axis=1)
    packed = orc.pack_nibbles(codes)
    assert packed.shape == (256, 1) and len(set(packed.ravel().tolist())) == 256
    assert np.array_equal(orc.unpack_nibbles(packed), codes)
    assert orc.pack_nibbles(np.array([[-7, 3]], dtype=np.int8))[0, 0] == (0x9 | (0x3 << 4))


# ---------------------------------------------------------------- integer products, zero point
def test_integer_products_blas_vs_loops():
    rng = np.random.default_rng(9)
    a = rng.integers(-7, 8, (9, 64)).astype(np.int8)
    b = rng.integers(-7, 8, (11, 64)).astype(np.int8)
    assert np.array_equal((a.astype(np.float64) @ b.astype(np.float64).T).astype(np.int64), orc.int_matmul_loops(a, b))
    worst = np.full((1, 128), 7, dtype=np.int8)
    assert orc.int_matmul_loops(worst, worst)[0, 0] == 49 * 128 == 6272


def test_zero_point_identity():
    rng = np.random.default_rng(10)
    u = rng.integers(0, 16, (5, 128)).astype(np.float64)
    v = rng.integers(-7, 8, (128, 32)).astype(np.float64)
    assert np.array_equal(u @ v, (u - 8) @ v + 8 * v.sum(axis=0)[None, :])


# ---------------------------------------------------------------- P codes (Eq.11, Eq.12)
def test_p_code_range_and_boundaries():
    rows = {r[0]: r for r in _read_rows('eq11_eq12_p_range.txt')}
    for mode, name in ((orc.P_ASYM15, 'asym15'), (orc.P_SYM7, 'sym7')):
        scale, zp, lo, hi, levels = (int(x) for x in rows[name][1:])
        s = np.array([[0.0, -1e-9, -50.0, -0.2, -3.0]])
        phat, u = orc.p_codes_block(s, np.array([0.0]), mode)
        signed = u + zp
        assert signed.max() == hi and signed.min() == lo          # P^=1 -> top code, P^->0 -> bottom code
        assert len(np.unique(np.arange(0, scale + 1))) == levels
        # code boundaries at s - m = ln((u - 1/2)/scale)
        for code in range(1, scale + 1):
            b = math.log((code - 0.5) / scale)
            _, ua = orc.p_codes_block(np.array([[b + 1e-9]]), np.array([0.0]), mode)
            _, ub = orc.p_codes_block(np.array([[b - 1e-9]]), np.array([0.0]), mode)
            assert ua[0, 0] == code and ub[0, 0] == code - 1
    assert np.isclose(math.log(0.5 / 15), -3.4012, atol=1e-4)
    assert np.isclose(math.log(14.5 / 15), -0.0339, atol=1e-4)


def _tiny_problem(seed=11, N=300, D=32, kv_block=128, p_mode=orc.P_ASYM15, p_norm=orc.NORM_ROWBLOCK):
    rng = np.random.default_rng(seed)
    p = orc.Params(1, 1, N, D, (1, 1, N), (4, 4, 8), kv_block=kv_block, v_group=kv_block, p_mode=p_mode, p_norm=p_norm)
    qc = rng.integers(-7, 8, (N, D)).astype(np.int8)
    kc = rng.integers(-7, 8, (N, D)).astype(np.int8)
    vc = rng.integers(-7, 8, (N, D)).astype(np.int8)
    qs = rng.uniform(0.05, 0.2, N).astype(np.float32)
    ks = rng.uniform(0.05, 0.2, N).astype(np.float32)
    vs = rng.uniform(0.1, 0.5, (-(-N // kv_block), D)).astype(np.float32)
    return p, qc, qs, kc, ks, vc, vs


def test_every_block_row_has_top_code_and_codes_cover_range():
    p, qc, qs, kc, ks, vc, vs = _tiny_problem()
    _, acc, codes = orc.o_quant(p, qc, qs, kc, ks, vc, vs, dump=True)
    for J in range(3):
        blk = codes[:, 128 * J:min(300, 128 * (J + 1))]
        assert np.all(blk.max(axis=1) == 15)
    assert set(np.unique(codes)) == set(range(16))                  # "P codes covering 0..15"
    assert np.array_equal(acc, orc.int_matmul_loops(qc, kc))
    _, _, codes7 = orc.o_quant(p, qc, qs, kc, ks, vc, vs, dump=True, p_mode=orc.P_SYM7)
    assert set(np.unique(codes7)) == set(range(8))


# ---------------------------------------------------------------- online softmax
def test_online_softmax_without_quantisers_is_softmax():
    p, qc, qs, kc, ks, vc, vs = _tiny_problem()
    O = orc.o_quant(p, qc, qs, kc, ks, vc, vs, quantize=False)
    qd = qc * qs[:, None].astype(np.float64)
    kd = kc * ks[:, None].astype(np.float64)
    vd = vc.astype(np.float64) * np.repeat(vs.astype(np.float64), 128, axis=0)[:300]
    assert np.allclose(O, orc.o_exact(qd, kd, vd), atol=1e-12)
    O2 = orc.o_quant(p, qc, qs, kc, ks, vc, vs, quantize=False, p_norm=orc.NORM_RUNNING)
    assert np.allclose(O2, O, atol=1e-12)


def test_o_exact_against_python_loops():
    rng = np.random.default_rng(12)
    q, k, v = rng.standard_normal((5, 8)), rng.standard_normal((7, 8)), rng.standard_normal((7, 3))
    O = orc.o_exact(q, k, v)
    for i in range(5):
        s = [sum(q[i, d] * k[j, d] for d in range(8)) / math.sqrt(8) for j in range(7)]
        mx = max(s)
        e = [math.exp(x - mx) for x in s]
        for d in range(3):
            assert abs(O[i, d] - sum(e[j] * v[j, d] for j in range(7)) / sum(e)) < 1e-13


@pytest.mark.parametrize('p_mode', [orc.P_ASYM15, orc.P_SYM7])
@pytest.mark.parametrize('p_norm', [orc.NORM_ROWBLOCK, orc.NORM_RUNNING])
def test_o_quant_against_python_loops(p_mode, p_norm):
    """Brute force, scalar Python, straight from the step list (DESIGN.md steps 7-12)."""
    p, qc, qs, kc, ks, vc, vs = _tiny_problem(seed=13, N=70, D=8, kv_block=32, p_mode=p_mode, p_norm=p_norm)
    O = orc.o_quant(p, qc, qs, kc, ks, vc, vs)
    N, D = 70, 8
    lv = 15.0 if p_mode == orc.P_ASYM15 else 7.0
    for i in range(0, N, 7):
        m, l, acc_o = -math.inf, 0.0, [0.0] * D
        for j0 in range(0, N, 32):
            js = range(j0, min(N, j0 + 32))
            s = [sum(int(qc[i, d]) * int(kc[j, d]) for d in range(D)) * float(qs[i]) * float(ks[j]) / math.sqrt(D) for j in js]
            mt = max(s)
            mn = max(m, mt)
            ref = mt if p_norm == orc.NORM_ROWBLOCK else mn
            ph = [math.exp(x - ref) for x in s]
            u = [round(lv * x) for x in ph]                    # Python round = half-to-even
            beta = math.exp(mt - mn) if p_norm == orc.NORM_ROWBLOCK else 1.0
            alpha = math.exp(m - mn) if m > -math.inf else 0.0
            l = alpha * l + beta * sum(ph)
            for d in range(D):
                pv = sum(u[jj] * int(vc[j, d]) for jj, j in enumerate(js))
                acc_o[d] = alpha * acc_o[d] + beta * pv * float(vs[j0 // 32, d]) / lv
            m = mn
        for d in range(D):
            assert abs(O[i, d] - acc_o[d] / l) < 1e-12


def test_single_block_equals_direct_formula():
    p, qc, qs, kc, ks, vc, vs = _tiny_problem(N=100, kv_block=128)
    O, acc, codes = orc.o_quant(p, qc, qs, kc, ks, vc, vs, dump=True)
    s = acc * qs[:, None].astype(np.float64) * ks[None, :].astype(np.float64) / math.sqrt(32)
    ph = np.exp(s - s.max(axis=1, keepdims=True))
    u = np.rint(15 * ph)
    want = (u @ vc.astype(np.float64)) * (vs[0].astype(np.float64) / 15)[None, :] / ph.sum(axis=1, keepdims=True)
    assert np.allclose(O, want, atol=1e-12) and np.array_equal(u, codes)


def test_block_permutation_invariance_rowblock():
    """Reading 13: with the row-block normaliser, codes depend on block membership, not block order."""
    p, qc, qs, kc, ks, vc, vs = _tiny_problem(N=384)
    O, _, codes = orc.o_quant(p, qc, qs, kc, ks, vc, vs, dump=True)
    perm = np.concatenate([np.arange(256, 384), np.arange(0, 128), np.arange(128, 256)])
    O2, _, codes2 = orc.o_quant(p, qc, qs, kc[perm], ks[perm], vc[perm], vs[[2, 0, 1]], dump=True)
    assert np.array_equal(codes2, codes[:, perm])
    assert np.allclose(O, O2, atol=1e-12)


def test_asym15_beats_sym7_on_diffuse_attention():
    """L170 / L255 ordering claim on diffuse attention (quality itself is 'parity unpinned')."""
    rng = np.random.default_rng(14)
    N, D = 512, 64
    p = orc.Params(1, 1, N, D, (8, 8, 8), (12, 10, 10), rot_mode=orc.ROT_NONE)
    q16 = (rng.standard_normal((N, D)) * 0.7).astype(np.float16)
    k16 = (rng.standard_normal((N, D)) * 0.7).astype(np.float16)
    v16 = rng.standard_normal((N, D)).astype(np.float16)
    coef = orc.coef_table(p)
    pq = orc.prepare_qk_head(p, q16, k16, coef)
    vc, vs = orc.quant_v(v16)
    ex = orc.o_exact(orc.rope_fp64(p, q16.astype(np.float64)), orc.rope_fp64(p, k16.astype(np.float64)), v16.astype(np.float64))
    errs = {}
    for mode in (orc.P_ASYM15, orc.P_SYM7):
        O = orc.o_quant(p, pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs, p_mode=mode)
        errs[mode] = np.abs(O - ex).sum() / np.abs(ex).sum()
    assert errs[orc.P_ASYM15] < errs[orc.P_SYM7]


# ---------------------------------------------------------------- policy (L192)
def test_policy_fractions():
    for name, ns, nb, fs, ls, fb, lb, pct in _read_rows('schedule_fractions.txt'):
        pol = orc.Policy(int(ns), int(nb), int(fs), int(ls), int(fb), int(lb))
        frac = pol.int4_fraction()
        assert frac == (int(ns) - int(fs) - int(ls)) * (int(nb) - int(fb) - int(lb)) / (int(ns) * int(nb))
        assert abs(100 * frac - int(pct)) <= 0.5
    pol = orc.Policy(50, 4, 5, 0, 0, 0, fp16_head_mask=(0, 1, 0))
    assert pol.select(4, 0, 0) == 1 and pol.select(5, 0, 0) == 0 and pol.select(5, 0, 1) == 1


# ---------------------------------------------------------------- generator sanity (shapes of BASELINE.json)
def test_workload_shapes():
    assert syn.WAN_1_3B.N == 32760 and syn.WAN_14B.N == 75600 and syn.HUNYUAN.N == 119056
    assert [w.N for w in syn.SWEEP] == [4096, 16384, 32760, 65536, 131072]
    q, k, v = syn.gen_head(syn.TINY, 0, 1)
    assert q.shape == (256, 64) and q.dtype == np.float16
    pairs, scale, vch, _ = syn.outlier_spec(syn.TINY, 0)
    assert {11, 21, 31} <= set(pairs.tolist()) and len(pairs) == 4
    q2, _, _ = syn.gen_head(syn.TINY, 0, 1)
    assert np.array_equal(q, q2)
    pairs2, _, _, _ = syn.outlier_spec(syn.WAN_1_3B, 3)
    assert sorted(pairs2.tolist()) == sorted([21, 20, 19, 22 + 20, 22 + 19, 22 + 18, 43 + 20, 43 + 19])

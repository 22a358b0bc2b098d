"""Pins for the oracle's RoPE and block-energy functions (CPU only).

RoPE: the block-sum identity, Eq. 2, block-norm invariance
(PAPER.md:45), the HF rotate_half form as a library-style special case, closed-form angles.
Energy: hand-computed values, Jensen, AM-GM, N_q != N_k (Q15),
the generator's closed form E||x^(i)||^2 = 2*var_i.
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle import oracle as O


@pytest.mark.parametrize("pairing", [0, 1])
@pytest.mark.parametrize("base", [1.0e4, 1.0e6])
def test_rope_block_sum_identity_and_eq2(pairing, base):
    rng = np.random.default_rng(11)
    d = 128
    L = d // 2
    q = rng.standard_normal((6, 1, d))
    k = rng.standard_normal((6, 1, d))
    n = np.array([0, 5, 17, 4096, 100000, 524287], dtype=np.float64)
    m = np.array([3, 5, 1, 77, 131071, 2], dtype=np.float64)
    qr = O.rope(q, n, base, pairing)
    kr = O.rope(k, m, base, pairing)
    a, b = O.pair_indices(d, pairing)
    for t in range(6):
        lhs = float(qr[t, 0] @ kr[t, 0])                       # (R_n q)^T (R_m k)
        delta = m[t] - n[t]
        rhs = 0.0
        for i in range(L):                                      # sum_i q^(i)T R(delta*theta_i) k^(i)
            th = delta * base ** (-2.0 * i / d)
            R = np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
            rhs += np.array([q[t, 0, a[i]], q[t, 0, b[i]]]) @ R @ np.array([k[t, 0, a[i]], k[t, 0, b[i]]])
        assert abs(lhs - rhs) < 1e-9 * max(1.0, abs(rhs))
        # block norms are RoPE-invariant
        assert np.allclose(kr[t, 0, a] ** 2 + kr[t, 0, b] ** 2, k[t, 0, a] ** 2 + k[t, 0, b] ** 2, rtol=1e-12)


def test_rope_closed_forms():
    d, base = 128, 1.0e4
    x = np.zeros((2, 1, d))
    x[:, 0, 0] = 1.0          # block 0 (theta = 1 rad), half pairing: coords (0, 64)
    x[:, 0, 32] = 2.0         # block 32: theta = base^-0.5 = 0.01
    out = O.rope(x, np.array([0.0, 1.0]), base, 0)
    assert np.array_equal(out[0], x[0])                        # position 0 = identity
    assert out[1, 0, 0] == pytest.approx(math.cos(1.0), abs=1e-15)
    assert out[1, 0, 64] == pytest.approx(math.sin(1.0), abs=1e-15)      # counter-clockwise (Q2)
    assert out[1, 0, 32] == pytest.approx(2 * math.cos(0.01), abs=1e-15)
    assert out[1, 0, 96] == pytest.approx(2 * math.sin(0.01), abs=1e-15)


def test_rope_matches_rotate_half_form():
    """x*cos + rotate_half(x)*sin with rotate_half(x) = cat(-x2, x1): the HF Llama/Qwen form."""
    rng = np.random.default_rng(5)
    d, base = 128, 5.0e5
    x = rng.standard_normal((9, 3, d))
    pos = np.arange(9) * 1000.0
    inv = base ** (-np.arange(0, d, 2) / d)
    ang = pos[:, None] * inv[None, :]
    cos = np.concatenate([np.cos(ang), np.cos(ang)], -1)[:, None, :]
    sin = np.concatenate([np.sin(ang), np.sin(ang)], -1)[:, None, :]
    rot_half = np.concatenate([-x[..., d // 2:], x[..., :d // 2]], -1)
    ref = x * cos + rot_half * sin
    assert np.allclose(O.rope(x, pos, base, 0), ref, rtol=0, atol=1e-12)


def test_energy_hand_values_and_jensen():
    d = 4   # L = 2 blocks; half pairing: block0=(0,2), block1=(1,3)
    # two query heads sharing one KV head, one token: q0 = (1,0,0,0), q1 = (-1,0,0,0)
    q = np.array([[[1.0, 0, 0, 0], [-1.0, 0, 0, 0]]])
    k = np.array([[[0.0, 2.0, 0.0, 0.0]], [[0.0, 0.0, 0.0, 4.0]]])   # two key tokens
    s, Eq, Ek = O.block_energy(q, k, 0)
    # square THEN average over heads: Eq block0 = (1+1)/2 = 1 (mean-then-square would give 0)
    assert Eq[0].tolist() == [1.0, 0.0]
    assert Ek[0].tolist() == [0.0, (4.0 + 16.0) / 2]
    assert s[0].tolist() == [0.5, 5.0]
    # interleaved pairing: block0=(0,1), block1=(2,3)
    s2, _, Ek2 = O.block_energy(q, k, 1)
    assert Ek2[0].tolist() == [2.0, 8.0] and s2[0].tolist() == [1.5, 4.0]
    # score kinds
    for kind, want in [("qk_max", [1.0, 10.0]), ("k_only", [0.0, 10.0]), ("q_only", [1.0, 0.0]),
                       ("qk_product", [0.0, 0.0])]:
        got = O.block_energy(q, k, 0, kind)[0][0].tolist()
        assert got == pytest.approx(want)


def test_energy_nq_ne_nk_and_gqa_groups():
    rng = np.random.default_rng(2)
    q = rng.standard_normal((7, 4, 8))
    k = rng.standard_normal((13, 2, 8))
    s, Eq, Ek = O.block_energy(q, k, 0)
    a, b = O.pair_indices(8, 0)
    for h in range(2):
        eq = np.mean(q[:, 2 * h:2 * h + 2, :][..., a] ** 2 + q[:, 2 * h:2 * h + 2, :][..., b] ** 2, axis=(0, 1))
        ek = np.mean(k[:, h, a] ** 2 + k[:, h, b] ** 2, axis=0)
        assert np.allclose(Eq[h], eq, rtol=1e-13) and np.allclose(Ek[h], ek, rtol=1e-13)
        assert np.allclose(s[h], 0.5 * (eq + ek), rtol=1e-13)


def test_energy_generator_closed_form_and_amgm():
    """E||x^(i)||^2 = 2*var_i on the synthetic generator; mean(||q||*||k||) <= s_i."""
    scales = W.block_scales(0, 1, 64)
    n = 20000
    q = W.pre_rope_gaussian(0, 1, n, 1, 128, scales)
    k = W.pre_rope_gaussian(0, 2, n, 1, 128, scales)
    s, Eq, Ek = O.block_energy(q, k, 0)
    assert np.allclose(s[0], 2.0 * scales[0], rtol=0.05)
    a, b = O.pair_indices(128, 0)
    qn = np.sqrt(q[:, 0, a] ** 2 + q[:, 0, b] ** 2)
    kn = np.sqrt(k[:, 0, a] ** 2 + k[:, 0, b] ** 2)
    assert np.all(np.mean(qn * kn, axis=0) <= s[0] * (1 + 1e-12))
    # post-RoPE gives the same scores
    kr = O.rope(k, np.arange(n, dtype=np.float64), 1e4, 0)
    s2, _, _ = O.block_energy(q, kr, 0)
    assert np.allclose(s2, s, rtol=1e-10)


@pytest.mark.parametrize("pairing", [0, 1])
def test_rope_table_pins(pairing):
    """rope_table (fused-append variant) == rope when handed rope's own angles; hand values; exactness on fp32 data."""
    rng = np.random.default_rng(11)
    d, base = 128, 1.0e6
    x = rng.standard_normal((7, 2, d))
    pos = np.array([0.0, 1.0, 2.0, 77.0, 4095.0, 65536.0, 131071.0])
    ang = pos[:, None] * base ** (-2.0 * np.arange(d // 2) / d)[None, :]
    assert np.allclose(O.rope_table(x, np.cos(ang), np.sin(ang), pairing), O.rope(x, pos, base, pairing), rtol=0, atol=1e-9)   # 1-ulp angle differences x 131071
    # quarter turn of block 3: (x_a, x_b) = (1, 0) -> (0, 1), (0, 1) -> (-1, 0): counter-clockwise (Q2)
    a, b = O.pair_indices(d, pairing)
    e = np.zeros((2, 1, d)); e[0, 0, a[3]] = 1.0; e[1, 0, b[3]] = 1.0
    c = np.ones((2, d // 2)); s = np.zeros((2, d // 2)); c[:, 3] = 0.0; s[:, 3] = 1.0
    out = O.rope_table(e, c, s, pairing)
    assert out[0, 0, a[3]] == 0.0 and out[0, 0, b[3]] == 1.0 and out[1, 0, a[3]] == -1.0 and out[1, 0, b[3]] == 0.0
    assert np.count_nonzero(out) == 2
    # fp32 inputs and tables: the result is the correctly rounded exact value (checked with exact rationals)
    from fractions import Fraction
    xf = rng.standard_normal((1, 1, d)).astype(np.float32).astype(np.float64)
    cf = np.cos(ang[3:4]).astype(np.float32).astype(np.float64); sf = np.sin(ang[3:4]).astype(np.float32).astype(np.float64)
    got = O.rope_table(xf, cf, sf, pairing)
    for i in (0, 5, 63):
        exact = Fraction(xf[0, 0, a[i]]) * Fraction(cf[0, i]) - Fraction(xf[0, 0, b[i]]) * Fraction(sf[0, i])
        assert got[0, 0, a[i]] == float(exact)                 # float(Fraction) rounds to nearest even
        exact = Fraction(xf[0, 0, a[i]]) * Fraction(sf[0, i]) + Fraction(xf[0, 0, b[i]]) * Fraction(cf[0, i])
        assert got[0, 0, b[i]] == float(exact)

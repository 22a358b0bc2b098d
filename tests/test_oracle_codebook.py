"""Pins for the oracle's scalar codebooks (Q7), CPU only."""
import math

import numpy as np
import pytest

from oracle import codebook as cb

# Max (1960) / Lloyd textbook optimum for N(0,1): positive levels
MAX_LEVELS = {
    1: [0.7979],
    2: [0.4528, 1.510],
    3: [0.2451, 0.7560, 1.344, 2.152],
    4: [0.1284, 0.3881, 0.6568, 0.9424, 1.256, 1.618, 2.069, 2.733],
}
MAX_DISTORTION = {1: 0.3634, 2: 0.1175, 3: 0.03454, 4: 0.009497, 5: 0.002499}
C_TQ = math.sqrt(3.0) * math.pi / 2.0


@pytest.mark.parametrize("b", range(1, 9))
def test_fixed_point_symmetry_order(b):
    lv = cb.lloyd_max_levels(b)
    assert len(lv) == 1 << b
    assert np.all(np.diff(lv) > 0)
    assert np.allclose(lv, -lv[::-1], rtol=0, atol=0)
    assert cb.centroid_residual(lv) < 1e-12                 # each level = conditional mean of its cell


def test_closed_form_one_bit_and_zero_bit():
    assert cb.lloyd_max_levels(1)[1] == pytest.approx(math.sqrt(2.0 / math.pi), abs=1e-15)
    assert cb.lloyd_max_levels(0).tolist() == [0.0]
    assert cb.distortion(cb.lloyd_max_levels(1)) == pytest.approx(1.0 - 2.0 / math.pi, abs=1e-14)


@pytest.mark.parametrize("b", [1, 2, 3, 4])
def test_textbook_levels(b):
    pos = cb.lloyd_max_levels(b)[(1 << b) // 2:]
    assert np.allclose(pos, MAX_LEVELS[b], rtol=1.5e-3)


def test_distortion_textbook_and_rate_law():
    prev = None
    for b in range(1, 9):
        D = cb.distortion(cb.lloyd_max_levels(b))
        if b in MAX_DISTORTION:
            assert D == pytest.approx(MAX_DISTORTION[b], rel=3e-3)
        assert D <= C_TQ * 4.0 ** (-b)                       # PAPER.md:49 rate law
        if prev is not None:
            assert 3.0 < prev / D < 4.0                      # each bit ~quarters the MSE
            assert D * 4 ** b > prev * 4 ** (b - 1)          # D*4^b rises monotonically to C_TQ
        prev = D
    assert cb.distortion(cb.lloyd_max_levels(8)) * 4 ** 8 == pytest.approx(C_TQ, rel=0.02)


def test_distortion_monte_carlo():
    """distortion() itself is checked by brute force: nearest-level quantisation of N(0,1) draws."""
    x = np.random.default_rng(0).standard_normal(2_000_000)
    for b in (2, 4):
        lv = cb.lloyd_max_levels(b)
        q = lv[np.argmin(np.abs(x[:, None] - lv[None, :]), axis=1)] if b <= 2 else \
            lv[np.searchsorted(0.5 * (lv[:-1] + lv[1:]), x)]
        assert np.mean((x - q) ** 2) == pytest.approx(cb.distortion(lv), rel=5e-3)


def test_fp16_table():
    t = cb.codebook_table()
    assert t.size == 511
    assert np.array_equal(t, t.astype(np.float16).astype(np.float64))      # fp16-representable
    for b in range(9):
        c = cb.codebook(b, t)
        assert np.allclose(c, cb.lloyd_max_levels(b), rtol=2.0 ** -11, atol=0)
        assert np.array_equal(c, -c[::-1])                                   # symmetry survives rounding
        assert np.all(np.diff(c) > 0)

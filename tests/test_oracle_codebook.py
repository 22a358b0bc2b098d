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


# ----------------------------------------------------------------------------- exact-density codebooks
def _sphere_pdf_np(x, m):
    from math import lgamma, pi
    c = math.exp(lgamma(m / 2.0) - lgamma((m - 1) / 2.0)) / math.sqrt(pi * m)
    return c * np.maximum(1.0 - x * x / m, 0.0) ** ((m - 3) / 2.0)


@pytest.mark.parametrize("m", [2, 4, 10, 26, 128])
@pytest.mark.parametrize("b", [1, 2, 3, 4, 6])
def test_sphere_codebook_is_a_lloyd_max_fixed_point(b, m):
    """Every level is the centroid of its cell under f_m(x) ~ (1 - x^2/m)^((m-3)/2), thresholds at midpoints -- checked by
    numerical integration with the substitution x = sqrt(m) sin(phi) (smooth for every m >= 2), not by the oracle's own
    incomplete-beta closed forms."""
    from scipy.integrate import quad
    lv = cb.sphere_levels(b, m)
    assert len(lv) == 1 << b and np.all(np.diff(lv) > 0) and np.allclose(lv, -lv[::-1], atol=1e-12)
    assert lv[-1] < math.sqrt(m)
    pos = lv[lv > 0]
    t = np.concatenate([[0.0], 0.5 * (pos[:-1] + pos[1:]), [math.sqrt(m)]])
    rm = math.sqrt(m)
    for k, c in enumerate(pos):
        pa, pb = math.asin(min(t[k] / rm, 1.0)), math.asin(min(t[k + 1] / rm, 1.0))
        w = lambda p: math.cos(p) ** (m - 2)                     # f_m(x) dx = const * cos^(m-2)(phi) dphi
        num = quad(lambda p: rm * math.sin(p) * w(p), pa, pb, epsabs=1e-13, epsrel=1e-13)[0]
        den = quad(w, pa, pb, epsabs=1e-13, epsrel=1e-13)[0]
        assert c == pytest.approx(num / den, abs=2e-9), (b, m, k)


def test_sphere_codebook_closed_forms():
    # m = 3 is the uniform law on [-sqrt(3), sqrt(3)]: Lloyd-Max levels are the midpoints of 2^b equal cells, D = 4^-b
    for b in range(1, 6):
        N = 1 << b
        want = math.sqrt(3.0) * (2 * np.arange(N) + 1 - N) / N
        assert np.allclose(cb.sphere_levels(b, 3), want, atol=1e-10)
        assert cb.sphere_distortion(cb.sphere_levels(b, 3), 3) == pytest.approx(4.0 ** -b, rel=1e-9)
    # b = 1: the level is E|X| = sqrt(m) Gamma(m/2) / (sqrt(pi) Gamma((m+1)/2));  m = 2: 2 sqrt(2) / pi
    for m in (2, 4, 10, 26, 128):
        want = math.sqrt(m) * math.exp(math.lgamma(m / 2.0) - math.lgamma((m + 1) / 2.0)) / math.sqrt(math.pi)
        assert cb.sphere_levels(1, m)[1] == pytest.approx(want, rel=1e-11)
    assert cb.sphere_levels(1, 2)[1] == pytest.approx(2.0 * math.sqrt(2.0) / math.pi, rel=1e-12)


@pytest.mark.parametrize("b", [1, 2, 3, 4, 5])
def test_sphere_codebook_tends_to_the_gaussian_one_and_beats_it_on_its_own_density(b):
    g = cb.lloyd_max_levels(b)
    prev = None
    for m in (2, 4, 10, 26, 128, 1024):
        s = cb.sphere_levels(b, m)
        gap = float(np.max(np.abs(s - g)))
        if prev is not None:
            assert gap < prev                                     # monotone approach to the N(0,1) table
        prev = gap
        assert cb.sphere_distortion(s, m) <= cb.sphere_distortion(g, m) * (1 + 1e-12)
    assert prev < 5e-3 * g[-1]
    # the gain is what the method loses with the shared Gaussian table: > 30 % of the distortion at m = 4, b >= 3
    if b >= 3:
        assert cb.sphere_distortion(cb.sphere_levels(b, 4), 4) < 0.7 * cb.sphere_distortion(g, 4)


@pytest.mark.parametrize("m", [2, 4, 10, 26, 128])
def test_sphere_codebook_monte_carlo_on_rotated_unit_vectors(m):
    """Coordinates of sqrt(m) * (random unit vector): empirical quantisation error == the table's analytic distortion,
    and smaller than with the Gaussian table."""
    rng = np.random.default_rng(m)
    u = rng.standard_normal((200000 // m + 1000, m))
    x = (u / np.linalg.norm(u, axis=1, keepdims=True) * math.sqrt(m)).ravel()
    for b in (2, 3, 4):
        s, g = cb.sphere_levels(b, m), cb.lloyd_max_levels(b)
        q = lambda lv: lv[np.argmin(np.abs(x[:, None] - lv[None, :]), axis=1)]
        es, eg = float(np.mean((x - q(s)) ** 2)), float(np.mean((x - q(g)) ** 2))
        assert es == pytest.approx(cb.sphere_distortion(s, m), rel=0.03)
        assert es < eg or m >= 128               # (at m = 128 the two tables differ by less than the sampling noise)

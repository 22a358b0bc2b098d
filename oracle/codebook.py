"""Oracle-side TQ-MSE scalar codebooks (TEST INFRASTRUCTURE).

DESIGN.md reading Q7: C_b is the Lloyd-Max (MSE-optimal) 2^b-level scalar quantiser of N(0,1)
-- the quantiser whose high-resolution distortion is the paper's C_TQ * 4^-b with
C_TQ = sqrt(3)*pi/2 -- symmetric, ascending, rounded to fp16-representable
values ("shared fp16 codebook").  b = 0 is the one-level codebook {0}.

Solved here by Newton's method on the centroid conditions of the positive half (the
Jacobian is tridiagonal; numpy solves it densely).  The pins (tests/test_oracle_codebook.py)
are the Lloyd-Max fixed-point conditions, the closed form for b=1 and Max's textbook
levels/distortions.  Independent of paper_2606_24033_b200/csrc/codebook.cpp.
"""
from __future__ import annotations

import math
from functools import lru_cache

import numpy as np

_SQRT2 = math.sqrt(2.0)
_INV_SQRT_2PI = 1.0 / math.sqrt(2.0 * math.pi)


def _phi(x: float) -> float:
    return 0.0 if math.isinf(x) else _INV_SQRT_2PI * math.exp(-0.5 * x * x)


def _mass(a: float, b: float) -> float:
    """P(a < X < b) for 0 <= a < b, via erfc so that the tails keep relative accuracy."""
    ea = math.erfc(a / _SQRT2)
    eb = 0.0 if math.isinf(b) else math.erfc(b / _SQRT2)
    return 0.5 * (ea - eb)


def _centroid(a: float, b: float) -> float:
    """E[X | a < X < b] for the standard normal."""
    return (_phi(a) - _phi(b)) / _mass(a, b)


def lloyd_max_positive(n_pos: int, tol: float = 1e-14, max_iter: int = 200) -> np.ndarray:
    """The n_pos positive levels of the symmetric 2*n_pos-level Lloyd-Max quantiser of N(0,1)."""
    # start from the high-resolution (Panter-Dite companding) optimum
    # c_k = sqrt(3) * Phi^{-1}(u_k), u_k = 0.5 + (k + 1/2) / N.
    from statistics import NormalDist
    nd = NormalDist()
    N = 2 * n_pos
    c = np.array([math.sqrt(3.0) * nd.inv_cdf(0.5 + (k + 0.5) / N) for k in range(n_pos)])
    for _ in range(max_iter):
        t = np.empty(n_pos + 1)
        t[0] = 0.0
        t[1:n_pos] = 0.5 * (c[:-1] + c[1:])
        t[n_pos] = math.inf
        F = np.empty(n_pos)
        Jm = np.zeros((n_pos, n_pos))
        for k in range(n_pos):
            a, b = t[k], t[k + 1]
            P = _mass(a, b)
            g = (_phi(a) - _phi(b)) / P
            dga = _phi(a) * (g - a) / P
            dgb = 0.0 if math.isinf(b) else _phi(b) * (b - g) / P
            F[k] = c[k] - g
            Jm[k, k] = 1.0
            if k > 0:
                Jm[k, k - 1] -= 0.5 * dga
                Jm[k, k] -= 0.5 * dga
            if k + 1 < n_pos:
                Jm[k, k] -= 0.5 * dgb
                Jm[k, k + 1] -= 0.5 * dgb
        step = np.linalg.solve(Jm, F)
        # damp so that levels stay positive and ordered
        lam = 1.0
        while lam > 1e-6:
            cn = c - lam * step
            if cn[0] > 0 and np.all(np.diff(cn) > 0):
                break
            lam *= 0.5
        c = cn
        if np.max(np.abs(F)) < tol and lam == 1.0:
            break
    return c


@lru_cache(maxsize=None)
def lloyd_max_levels(b: int) -> np.ndarray:
    """All 2^b levels, ascending, fp64, NOT yet rounded to fp16."""
    if b == 0:
        return np.zeros(1)
    pos = lloyd_max_positive(1 << (b - 1))
    return np.concatenate([-pos[::-1], pos])


def centroid_residual(levels: np.ndarray) -> float:
    """max_k |c_k - E[X | cell k]| with thresholds at midpoints: 0 at a Lloyd-Max fixed point."""
    n = len(levels)
    if n == 1:
        return abs(float(levels[0]))
    t = np.concatenate([[-math.inf], 0.5 * (levels[:-1] + levels[1:]), [math.inf]])
    res = 0.0
    for k in range(n):
        a, b = t[k], t[k + 1]
        if b <= 0:          # mirror to the positive side for tail accuracy
            g = -_centroid(-b, -a)
        elif a >= 0:
            g = _centroid(a, b)
        else:               # cell straddling 0 (odd level counts only)
            P = 1.0 - 0.5 * math.erfc(-a / _SQRT2) - 0.5 * math.erfc(b / _SQRT2)
            g = (_phi(a) - _phi(b)) / P
        res = max(res, abs(levels[k] - g))
    return res


def distortion(levels: np.ndarray) -> float:
    """E[(X - Q(X))^2] for X ~ N(0,1) and nearest-level quantisation (closed form per cell)."""
    n = len(levels)
    if n == 1:
        return 1.0 + float(levels[0]) ** 2
    # by symmetry integrate the non-negative half-line exactly: cells (a,b) with level c
    t = np.concatenate([[-math.inf], 0.5 * (levels[:-1] + levels[1:]), [math.inf]])
    D = 0.0
    for k in range(n):
        a, b, c = t[k], t[k + 1], levels[k]
        if b <= 0:
            a, b, c = -b, -a, -c
        elif a < 0:
            # split at 0
            for (aa, bb) in ((0.0, -a), (0.0, b)):
                cc = -c if aa == 0.0 and bb == -a else c
                D += _cell_mse(aa, bb, cc)
            continue
        D += _cell_mse(a, b, c)
    return D


def _cell_mse(a: float, b: float, c: float) -> float:
    """integral_a^b (x-c)^2 phi(x) dx for 0 <= a < b."""
    P = _mass(a, b)
    m1 = _phi(a) - _phi(b)                                    # int x phi
    m2 = P + (a * _phi(a) - (0.0 if math.isinf(b) else b * _phi(b)))   # int x^2 phi
    return m2 - 2.0 * c * m1 + c * c * P


def f16_round(x: np.ndarray) -> np.ndarray:
    return np.asarray(x, dtype=np.float64).astype(np.float16).astype(np.float64)


def codebook_table(b_max: int = 8) -> np.ndarray:
    """Flat table of the fp16-rounded codebooks b = 0..b_max: C_b at offset 2^b - 1
    (total 2^(b_max+1) - 1 = 511 values for b_max = 8), fp64 values."""
    out = np.empty((1 << (b_max + 1)) - 1)
    for b in range(b_max + 1):
        out[(1 << b) - 1:(1 << (b + 1)) - 1] = f16_round(lloyd_max_levels(b))
    return out


def codebook(b: int, table: np.ndarray | None = None) -> np.ndarray:
    if table is None:
        table = codebook_table()
    return table[(1 << b) - 1:(1 << (b + 1)) - 1]


# ----------------------------------------------------------------------------- exact-density codebooks
# TQ-MSE "scalar-quantizes the rotated coordinates" of a NORMALISED vector.  A coordinate of
# sqrt(m) * u, u uniform on the unit sphere of R^m (what a Haar rotation makes of any unit vector), has the density
#     f_m(x) = c_m (1 - x^2/m)^((m-3)/2),  |x| < sqrt(m),   c_m = Gamma(m/2) / (sqrt(pi m) Gamma((m-1)/2)),
# which tends to N(0,1) as m grows but is visibly different for the small groups the allocator produces (m = 2 is the
# arcsine law, m = 3 is uniform).  C_{b,m} = Lloyd-Max quantiser of f_m, symmetric, ascending, rounded to fp16.
def _sphere_const(m: int) -> float:
    return math.exp(math.lgamma(m / 2.0) - math.lgamma((m - 1) / 2.0)) / math.sqrt(math.pi * m)


def sphere_pdf(x: float, m: int) -> float:
    u = 1.0 - x * x / m
    if u <= 0.0:
        return math.inf if (m == 2 and u == 0.0) else 0.0
    return _sphere_const(m) * u ** ((m - 3) / 2.0)


def _sphere_mass(a: float, b: float, m: int) -> float:
    """P(a < X < b), 0 <= a < b <= sqrt(m): regularised incomplete beta, I_{x^2/m}(1/2, (m-1)/2) = P(|X| < x)."""
    from scipy.special import betainc
    fa = betainc(0.5, (m - 1) / 2.0, min(a * a / m, 1.0))
    fb = betainc(0.5, (m - 1) / 2.0, min(b * b / m, 1.0))
    return 0.5 * (fb - fa)


def _sphere_first_moment(a: float, b: float, m: int) -> float:
    """int_a^b x f_m(x) dx = [-(m/(m-1)) c_m (1 - x^2/m)^((m-1)/2)]_a^b."""
    G = lambda x: -(m / (m - 1.0)) * _sphere_const(m) * max(1.0 - x * x / m, 0.0) ** ((m - 1) / 2.0)
    return G(b) - G(a)


def sphere_lloyd_max_positive(n_pos: int, m: int, tol: float = 1e-13, max_iter: int = 500) -> np.ndarray:
    """The n_pos positive levels of the symmetric 2*n_pos-level Lloyd-Max quantiser of f_m (Newton on the centroid
    conditions, as lloyd_max_positive; the support ends at sqrt(m))."""
    top = math.sqrt(m)
    c = lloyd_max_positive(n_pos)
    if c[-1] >= 0.98 * top:
        c = c * (0.98 * top / c[-1])
    for _ in range(max_iter):
        t = np.empty(n_pos + 1)
        t[0] = 0.0
        t[1:n_pos] = 0.5 * (c[:-1] + c[1:])
        t[n_pos] = top
        F = np.empty(n_pos)
        Jm = np.zeros((n_pos, n_pos))
        for k in range(n_pos):
            a, b = t[k], t[k + 1]
            P = _sphere_mass(a, b, m)
            g = _sphere_first_moment(a, b, m) / P
            dga = sphere_pdf(a, m) * (g - a) / P
            dgb = 0.0 if k + 1 == n_pos else sphere_pdf(b, m) * (b - g) / P
            F[k] = c[k] - g
            Jm[k, k] = 1.0
            if k > 0:
                Jm[k, k - 1] -= 0.5 * dga
                Jm[k, k] -= 0.5 * dga
            if k + 1 < n_pos:
                Jm[k, k] -= 0.5 * dgb
                Jm[k, k + 1] -= 0.5 * dgb
        step = np.linalg.solve(Jm, F)
        lam = 1.0
        while lam > 1e-8:
            cn = c - lam * step
            if cn[0] > 0 and np.all(np.diff(cn) > 0) and cn[-1] < top:
                break
            lam *= 0.5
        c = cn
        if np.max(np.abs(F)) < tol and lam == 1.0:
            break
    return c


@lru_cache(maxsize=None)
def sphere_levels(b: int, m: int) -> np.ndarray:
    """All 2^b levels of C_{b,m}, ascending, fp64, NOT yet rounded to fp16."""
    if b == 0:
        return np.zeros(1)
    pos = sphere_lloyd_max_positive(1 << (b - 1), m)
    return np.concatenate([-pos[::-1], pos])


def sphere_distortion(levels: np.ndarray, m: int) -> float:
    """E[(X - Q(X))^2] for X ~ f_m and nearest-level quantisation: E X^2 = 1, so D = 1 - 2 sum c_k M1_k + sum c_k^2 P_k."""
    lv = np.asarray(levels, dtype=np.float64)
    pos = lv[lv > 0]
    top = math.sqrt(m)
    t = np.concatenate([[0.0], 0.5 * (pos[:-1] + pos[1:]), [top]])
    D = 1.0
    for k, c in enumerate(pos):
        a, b = min(t[k], top), min(t[k + 1], top)
        if b <= a:
            continue
        D += 2.0 * (c * c * _sphere_mass(a, b, m) - 2.0 * c * _sphere_first_moment(a, b, m))
    return D


@lru_cache(maxsize=None)
def sphere_codebook(b: int, m: int) -> np.ndarray:
    """C_{b,m} rounded to fp16-representable values (fp64 array)."""
    return f16_round(sphere_levels(b, m))

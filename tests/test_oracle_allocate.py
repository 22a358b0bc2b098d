"""Pins for the oracle's Algorithm 1 (proof PAPER.md:427-437), CPU only."""
import itertools

import numpy as np
import pytest

import workloads as W
from oracle import oracle as O


def brute_force_min_J(s, B, b_min, b_max):
    best = None
    for alloc in itertools.product(range(b_min, b_max + 1), repeat=len(s)):
        if sum(alloc) != B:
            continue
        J = sum(si * 4.0 ** (-b) for si, b in zip(s, alloc))
        if best is None or J < best:
            best = J
    return best


@pytest.mark.parametrize("L,b_min,b_max", [(4, 0, 4), (5, 0, 4), (6, 0, 3), (5, 1, 4), (6, 1, 3)])
def test_greedy_equals_brute_force(L, b_min, b_max):
    """Theorem 1: greedy minimises J over ALL feasible integer allocations (tiny heads)."""
    rng = np.random.default_rng(100 + L + b_max)
    for trial in range(6):
        s = np.exp(rng.uniform(np.log(1e-2), np.log(10.0), L))
        for B in range(L * b_min, L * b_max + 1, max(1, L // 2)):
            bits = O.allocate(s, B, b_min, b_max)
            assert bits.sum() == B and bits.min() >= b_min and bits.max() <= b_max
            Jg = O.objective(s, bits)
            Jb = brute_force_min_J(s, B, b_min, b_max)
            assert Jg == pytest.approx(Jb, rel=1e-12)


def test_objective_is_the_plain_sum():
    s = np.array([1.0, 2.0, 4.0])
    assert O.objective(s, [0, 1, 2]) == 1.0 + 0.5 + 0.25


def test_invariants_on_config_profiles():
    for seed, (b_min, b_max), bbar in [(0, (0, 8), 3), (1, (1, 8), 3), (100, (1, 8), 2)]:
        s_all = 2.0 * W.block_scales(seed, 4, 64)
        for s in s_all:
            B = bbar * 64
            bits, gains = O.allocate(s, B, b_min, b_max, return_gains=True)
            assert int(bits.sum()) == B                      # sums exactly to bbar*d_h/2 (*2 bits/block)
            assert bits.min() >= b_min and bits.max() <= b_max
            assert np.all(np.diff(gains) <= 0)               # popped marginal gains non-increasing
            assert np.array_equal(bits, O.allocate(s, B, b_min, b_max, method="heap"))
            assert np.array_equal(bits, O.allocate(7.5 * s, B, b_min, b_max))   # scale invariance
            # higher score never gets fewer bits
            order = np.argsort(s)
            assert np.all(np.diff(bits[order].astype(int)) >= 0)
            # prefix structure: each popped gain is 3/4 s_i 4^-(b) for consecutive b
            expected = sorted((0.75 * s[i] * 4.0 ** (-b) for i in range(64)
                               for b in range(b_min, int(bits[i]))), reverse=True)
            assert np.allclose(gains, expected, rtol=1e-15)


def test_equal_scores_uniform_and_ties_smallest_index():
    s = np.ones(8)
    assert O.allocate(s, 24, 0, 8).tolist() == [3] * 8
    # one spare bit goes to the smallest index (Q4); heap agrees
    assert O.allocate(s, 25, 0, 8).tolist() == [4] + [3] * 7
    assert O.allocate(s, 25, 0, 8, method="heap").tolist() == [4] + [3] * 7
    assert O.allocate(s, 26, 1, 8, method="heap").tolist() == [4, 4] + [3] * 6


def test_zero_scores_and_saturation():
    s = np.array([0.0, 5.0, 0.0, 1.0])
    # positive blocks saturate at b_max before zero-score blocks get anything (Q5)
    assert O.allocate(s, 8, 0, 4).tolist() == [0, 4, 0, 4]
    assert O.allocate(s, 9, 0, 4).tolist() == [1, 4, 0, 4]
    assert O.allocate(s, 16, 0, 4).tolist() == [4, 4, 4, 4]
    assert O.allocate(s, 0, 0, 4).tolist() == [0, 0, 0, 0]
    with pytest.raises(ValueError):
        O.allocate(s, 17, 0, 4)
    with pytest.raises(ValueError):
        O.allocate(np.array([1.0, -1.0]), 2, 0, 4)


def test_heap_equals_linear_random():
    rng = np.random.default_rng(9)
    for _ in range(200):
        L = int(rng.integers(1, 70))
        s = np.exp(rng.uniform(-6, 3, L))
        if rng.random() < 0.3:
            s[rng.integers(0, L)] = s[rng.integers(0, L)]      # exact ties
        b_min = int(rng.integers(0, 3)); b_max = int(rng.integers(b_min, 9))
        B = int(rng.integers(L * b_min, L * b_max + 1))
        assert np.array_equal(O.allocate(s, B, b_min, b_max), O.allocate(s, B, b_min, b_max, method="heap"))


def test_allocation_shape_matches_paper_tables():
    """Tables 8-10: the budget width is the mode; several widths per head."""
    s_all = 2.0 * W.block_scales(1, 8, 64)
    hist = np.zeros(9)
    ngroups = []
    for s in s_all:
        bits = O.allocate(s, 192, 1, 8)
        hist += np.bincount(bits, minlength=9)
        ngroups.append(len(set(bits.tolist())))
    assert 3.5 <= np.mean(ngroups) <= 7.0
    s_p = W.paper_like_scores(3, 16, 64)
    hist = np.zeros(9)
    for s in s_p:
        hist += np.bincount(O.allocate(s, 192, 1, 8), minlength=9)
    assert int(np.argmax(hist)) == 3

"""-m "not gpu": the C-ABI library loads, exports every symbol include/bgtq.h declares, and its
host-only entry points (codebook, host allocator, argument checks) agree with the oracle.
No device compute is called here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import codebook as ocb
from oracle import oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2606_24033_b200 import build
    build.build()
    from paper_2606_24033_b200 import binding
    return binding


def test_header_symbols_are_exported(B):
    hdr = open(os.path.join(ROOT, "include", "bgtq.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bgtq_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    lib = C.CDLL(B.LIB_PATH)
    for name in declared:
        assert getattr(lib, name) is not None


def test_library_codebook_equals_oracle_codebook(B):
    """two independent Lloyd-Max solvers (Newton/dense in numpy vs long-double/Thomas in C++)"""
    table = ocb.codebook_table()
    for b in range(9):
        got = B.codebook(b).astype(np.float64)
        assert np.array_equal(got, ocb.codebook(b, table)), b
        assert np.array_equal(got.astype(np.float16).astype(np.float64), got)      # fp16-representable


def test_library_exact_density_codebook_equals_oracle(B):
    """two independent solvers of the sphere-marginal Lloyd-Max tables (incomplete beta / dense Newton in numpy vs the
    cos^n recurrence / Thomas solve in long double), bit-equal after rounding to fp16"""
    for m in (2, 4, 6, 10, 16, 26, 32, 64, 128):
        for b in range(9):
            got = B.codebook_exact(b, m).astype(np.float64)
            assert np.array_equal(got, ocb.sphere_codebook(b, m)), (b, m)
    with pytest.raises(B.BgtqError):
        B.codebook_exact(3, 7)


@pytest.mark.parametrize("bmin,bmax,bbar", [(0, 8, 3), (1, 8, 3), (1, 8, 2), (0, 4, 1), (3, 3, 3)])
def test_host_allocator_equals_oracle(B, bmin, bmax, bbar):
    rng = np.random.default_rng(17)
    s = np.exp(rng.uniform(np.log(1e-2), np.log(10), size=(25, 64))).astype(np.float32)
    s[0, :] = 2.5
    s[1, 5:40] = 0.0
    s[2, 7] = s[2, 50]
    got = B.allocate(s, bbar * 64, bmin, bmax)
    for h in range(len(s)):
        assert np.array_equal(got[h], O.allocate(s[h].astype(np.float64), bbar * 64, bmin, bmax)), h


def test_host_allocator_small_L_matches_heap(B):
    rng = np.random.default_rng(3)
    for L in (1, 2, 5, 33):
        s = rng.random((4, L)).astype(np.float32)
        B_tot = 2 * L
        got = B.allocate(s, B_tot, 0, 4)
        for h in range(4):
            assert np.array_equal(got[h], O.allocate(s[h].astype(np.float64), B_tot, 0, 4, method="heap"))


def test_error_codes(B):
    s = np.ones((1, 64), dtype=np.float32)
    with pytest.raises(B.BgtqError) as e:
        B.allocate(s, 64 * 9, 0, 8)
    assert e.value.code == -2                       # BGTQ_EBUDGET
    with pytest.raises(B.BgtqError) as e:
        B.allocate(-s, 64 * 3, 0, 8)
    assert e.value.code == -1                       # BGTQ_EINVAL, negative score (Q5)
    with pytest.raises(B.BgtqError) as e:
        B.allocate(s, 64 * 3, 5, 2)
    assert e.value.code == -1
    with pytest.raises(B.BgtqError):
        B.codebook(9) if False else B._check(B.lib().bgtq_codebook(9, None))
    assert b"bgtq_codebook" in B.lib().bgtq_last_error()


def test_no_cpu_fallback_for_device_entry_points(B):
    import torch
    q = torch.zeros(4, 2, 128)
    with pytest.raises(ValueError):
        B.block_energy(q, q)

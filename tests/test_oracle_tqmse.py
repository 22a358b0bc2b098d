"""Pins for the oracle's TQ-MSE encoder/decoder and the rotation table (CPU only).

Rate law and constants: PAPER.md:49; grouping: PAPER.md:108; Lemma 2: PAPER.md:396.
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle import codebook as cb
from oracle import oracle as O

C_TQ = math.sqrt(3.0) * math.pi / 2.0


def test_rotations_orthogonal_and_fold_identity(rot128):
    offs = W.rotation_offsets(128)
    rng = np.random.default_rng(0)
    for m in (2, 4, 6, 26, 64, 128):
        Pi = rot128[offs[m]:offs[m] + m * m].reshape(m, m).astype(np.float64)
        assert np.max(np.abs(Pi @ Pi.T - np.eye(m))) < 1e-6          # fp32-rounded orthogonal
        # fold: q^T (h Pi^T c / sqrt(m)) == (Pi q)^T (h c / sqrt(m))
        q, c, h = rng.standard_normal(m), rng.standard_normal(m), 1.7
        assert q @ (h * (Pi.T @ c) / math.sqrt(m)) == pytest.approx((Pi @ q) @ (h * c / math.sqrt(m)), rel=1e-12)


@pytest.mark.parametrize("b", range(1, 9))
def test_rate_law_m128(b, tab128):
    """mean ||x - xhat||^2 / ||x||^2 <= C_TQ 4^-b and ~ D(b) (before the fp16 norm matters)."""
    rng = np.random.default_rng(b)
    n = 1500 if b < 6 else 6000
    rel = np.empty(n)
    for i in range(n):
        x = (rng.standard_normal(128) * 3.0).astype(np.float32).astype(np.float64)
        idx, h, r = O.quantize_group(x, b, tab128)
        xh = O.dequantize_group(idx, h, b, tab128)
        rel[i] = np.sum((x - xh) ** 2) / np.sum(x * x)
        assert idx.max() < (1 << b)
        # stored norm = IEEE binary16 round-to-nearest-even of the unrounded radius (Q10), checked against numpy's conversion
        assert h == int(np.array([r], dtype=np.float64).astype(np.float16).view(np.uint16)[0])
        assert r == pytest.approx(math.sqrt(float(np.sum(x * x))), rel=1e-14)
    D = cb.distortion(cb.lloyd_max_levels(b))
    assert rel.mean() <= C_TQ * 4.0 ** (-b)
    assert rel.mean() == pytest.approx(D, rel=0.06)


def test_error_falls_with_bits_and_small_groups(tab128):
    rng = np.random.default_rng(42)
    for m in (2, 4, 10, 26):
        x = rng.standard_normal((400, m)).astype(np.float32).astype(np.float64)
        prev = None
        for b in range(1, 9):
            e = 0.0
            for row in x:
                idx, h, _ = O.quantize_group(row, b, tab128)
                e += np.sum((row - O.dequantize_group(idx, h, b, tab128)) ** 2) / np.sum(row * row)
            e /= len(x)
            if prev is not None:
                assert e < prev          # reconstruction error strictly falls as bits rise
            prev = e


def test_codes_are_nearest_centroid(tab128):
    """Brute force: idx_j = argmin_k |z_j/sigma - C_k| (thresholds are midpoints)."""
    rng = np.random.default_rng(1)
    for m, b in [(128, 3), (26, 5), (8, 8), (2, 1), (64, 2)]:
        x = rng.standard_normal(m).astype(np.float32).astype(np.float64)
        idx, h, r = O.quantize_group(x, b, tab128)
        z = tab128.Pi(m).astype(np.float64) @ x
        sigma = np.linalg.norm(x) / math.sqrt(m)
        want = np.argmin(np.abs(z[:, None] / sigma - tab128.C(b)[None, :]), axis=1)
        assert np.array_equal(idx, want)
        assert r == pytest.approx(np.linalg.norm(x), rel=1e-14)


def test_zero_vector_and_saturating_norm(tab128):
    idx, h, r = O.quantize_group(np.zeros(16), 4, tab128)
    assert idx.tolist() == [0] * 16 and h == 0 and r == 0.0
    assert np.array_equal(O.dequantize_group(idx, h, 4, tab128), np.zeros(16))
    big = np.full(4, 1.0e6)
    idx, h, _ = O.quantize_group(big, 2, tab128)
    assert h == 0x7BFF                       # saturates to 65504 (Q10)


def test_lemma2_bound_and_one_group_is_uniform(tab128):
    """Per-block accounting bound holds for every (q, k, k_hat); a schedule with
    one width is plain uniform TQ-MSE over the whole head."""
    rng = np.random.default_rng(7)
    d = 128
    a, b = O.pair_indices(d, 0)
    scales = W.block_scales(0, 1, 64)
    k_pre = W.pre_rope_gaussian(0, 2, 20, 1, d, scales)
    q_pre = W.pre_rope_gaussian(0, 1, 20, 1, d, scales)
    pos_k = np.arange(20, dtype=np.float64)
    k_post = O.rope(k_pre, pos_k, 1e4, 0)[:, 0].astype(np.float32).astype(np.float64)
    s, _, _ = O.block_energy(q_pre, k_pre, 0)
    bits = O.allocate(s[0], 192, 0, 8)
    qh = O.quantize_head(k_post, k_post, bits, 3, tab128, 0)
    K_hat, _ = O.dequantize_head(qh, tab128, d)
    n_pos = 50.0
    q_post = O.rope(q_pre[:1], np.array([n_pos]), 1e4, 0)[0, 0]
    for t in range(20):
        err = abs(q_post @ k_post[t] - q_post @ K_hat[t])
        e = k_post[t] - K_hat[t]                   # block norms are rotation invariant
        bound = np.sum(np.sqrt(q_post[a] ** 2 + q_post[b] ** 2) * np.sqrt(e[a] ** 2 + e[b] ** 2))
        assert err <= bound * (1 + 1e-12)
    # uniform: all blocks width 3 -> one group of 128 coords == quantising the permuted vector
    qu = O.quantize_head(k_post, k_post, [3] * 64, 3, tab128, 0)
    assert len(qu.groups) == 1 and qu.groups[0].m == 128
    perm = qu.groups[0].coords
    for t in range(3):
        idx, h, _ = O.quantize_group(k_post[t, perm], 3, tab128)
        assert np.array_equal(idx, qu.kidx[t]) and h == qu.knorm[t, 0]
    # width-0 blocks decode to exactly zero (Q3)
    z = np.nonzero(bits == 0)[0]
    if len(z):
        assert np.all(K_hat[:, a[z]] == 0) and np.all(K_hat[:, b[z]] == 0)


def test_block_gtq_beats_uniform_on_logit_error(tab128):
    """Sanity echo of Table 1's direction on the synthetic profile."""
    d = 128
    scales = W.block_scales(0, 1, 64)
    k_pre = W.pre_rope_gaussian(0, 2, 64, 1, d, scales)
    q_pre = W.pre_rope_gaussian(0, 1, 64, 1, d, scales)
    k_post = O.rope(k_pre, np.arange(64, dtype=np.float64), 1e4, 0)[:, 0].astype(np.float32).astype(np.float64)
    q_post = O.rope(q_pre, np.full(64, 64.0), 1e4, 0)[:, 0]
    s, _, _ = O.block_energy(q_pre, k_pre, 0)
    bits = O.allocate(s[0], 192, 0, 8)
    Kb, _ = O.dequantize_head(O.quantize_head(k_post, k_post, bits, 3, tab128), tab128, d)
    Ku, _ = O.dequantize_head(O.quantize_head(k_post, k_post, [3] * 64, 3, tab128), tab128, d)
    mae_b = np.mean(np.abs(q_post @ (k_post - Kb).T))
    mae_u = np.mean(np.abs(q_post @ (k_post - Ku).T))
    assert mae_b < 0.7 * mae_u


def test_f16_converters_match_ieee_binary16():
    """orc_f64_to_f16_bits / orc_f16_bits_to_f64 against numpy.float16 (IEEE binary16, round-to-nearest-even): every
    fp16 value, every midpoint between adjacent fp16 values and its two double neighbours, subnormals, signed zero,
    random doubles, and the saturation at 65504 / 65520 (Q10)."""
    L = O.lib()
    allbits = np.arange(0x7C00, dtype=np.uint16)                       # every finite non-negative fp16
    vals = allbits.view(np.float16).astype(np.float64)
    for h, v in zip(allbits[::7].tolist() + [0, 1, 0x03FF, 0x0400, 0x7BFF], vals[::7].tolist() + [vals[0], vals[1], vals[0x3FF], vals[0x400], vals[0x7BFF]]):
        assert L.orc_f16_bits_to_f64(h) == v
        assert L.orc_f16_bits_to_f64(h | 0x8000) == -v or v == 0.0
    assert math.copysign(1.0, L.orc_f16_bits_to_f64(0x8000)) == -1.0
    mids = (vals[:-1] + vals[1:]) / 2.0                                # exact in fp64
    cand = np.concatenate([vals, mids, np.nextafter(mids, np.inf), np.nextafter(mids, -np.inf),
                           np.nextafter(vals, np.inf), np.nextafter(vals[1:], -np.inf),
                           np.random.default_rng(0).uniform(0.0, 65504.0, 20000),
                           np.exp(np.random.default_rng(1).uniform(np.log(1e-9), np.log(65504.0), 20000))])
    cand = cand[cand < 65520.0]
    want = cand.astype(np.float16).view(np.uint16)
    got = np.array([L.orc_f64_to_f16_bits(float(x)) for x in cand], dtype=np.uint16)
    assert np.array_equal(got, want)
    got_neg = np.array([L.orc_f64_to_f16_bits(float(-x)) for x in cand[::5]], dtype=np.uint16)
    assert np.array_equal(got_neg, (-cand[::5]).astype(np.float16).view(np.uint16))
    # saturation: 65504 is the largest finite value; 65520 (the midpoint to 2^16) and everything above saturate
    for x, bits in [(65504.0, 0x7BFF), (65519.999, 0x7BFF), (65520.0, 0x7BFF), (1e9, 0x7BFF), (-65520.0, 0xFBFF),
                    (2.0 ** -25, 0x0000), (np.nextafter(2.0 ** -25, 1.0), 0x0001), (2.0 ** -24, 0x0001), (0.0, 0), (-0.0, 0x8000)]:
        assert L.orc_f64_to_f16_bits(float(x)) == bits, x


@pytest.mark.parametrize("m", [2, 4, 10, 26])
def test_rate_law_small_groups_exact_density(m, rot128):
    """PAPER.md:49 at the group sizes the allocator really produces: with the exact-density codebooks the relative error
    of TQ-MSE on m-vectors equals the table's distortion D(b, m) (the norm is restored exactly up to fp16) and obeys
    C_TQ 4^-b; with the shared Gaussian table it is larger."""
    tabs = O.Tables(rot128, 128, cb_kind="sphere")
    tabg = O.Tables(rot128, 128)
    rng = np.random.default_rng(m)
    x = (rng.standard_normal((3000, m)) * 2.0).astype(np.float32).astype(np.float64)
    for b in (2, 3, 4):
        es = eg = 0.0
        for row in x:
            i1, h1, _ = O.quantize_group(row, b, tabs)
            i2, h2, _ = O.quantize_group(row, b, tabg)
            es += np.sum((row - O.dequantize_group(i1, h1, b, tabs)) ** 2) / np.sum(row * row)
            eg += np.sum((row - O.dequantize_group(i2, h2, b, tabg)) ** 2) / np.sum(row * row)
        es /= len(x); eg /= len(x)
        D = cb.sphere_distortion(cb.sphere_codebook(b, m), m)
        assert es == pytest.approx(D, rel=0.08), (m, b)
        assert es <= C_TQ * 4.0 ** (-b)
        assert es < eg


def test_rope_logit_mae_echo_of_table_1():
    """PAPER.md:532 (50 offsets in [-1024, 1024], K-only): on synthetic heads with log-uniform block energies Block-GTQ's
    allocation beats uniform TQ-MSE at the same budget (the direction of Tables 1 and 11), with either codebook family,
    and the exact-density codebooks do not hurt."""
    import workloads as W
    d, Hq, Hkv, base = 128, 4, 2, 1.0e6
    rot = W.rotations(20260624, d)
    tg, ts = O.Tables(rot, d), O.Tables(rot, d, cb_kind="sphere")
    scales = W.block_scales(5, Hkv, d // 2)
    s, _, _ = O.block_energy(W.pre_rope_gaussian(5, 4, 256, Hq, d, scales), W.pre_rope_gaussian(5, 1, 256, Hkv, d, scales))
    q, k = W.pre_rope_gaussian(5, 5, 48, Hq, d, scales), W.pre_rope_gaussian(5, 6, 48, Hkv, d, scales)
    for bbar in (2, 3):
        greedy = np.stack([O.allocate(s[h], bbar * 64, 1, 8) for h in range(Hkv)])
        uniform = np.full_like(greedy, bbar)
        mu, mg = O.rope_logit_mae(q, k, uniform, tg, base), O.rope_logit_mae(q, k, greedy, tg, base)
        ms = O.rope_logit_mae(q, k, greedy, ts, base)
        assert mg < 0.75 * mu
        assert ms < 1.02 * mg
    # the definition itself: Delta = 0 only, one block stored -> |q^(i) . e^(i)| averaged
    one = np.zeros((Hkv, 64), dtype=np.int64); one[:, 0] = 8
    m0 = O.rope_logit_mae(q, k, one, tg, base, offsets=np.array([0.0]))
    want = 0.0
    for h in range(Hkv):
        g = O.groups_from_bits(one[h], d)[0]
        for t in range(len(q)):
            idx, hb, _ = O.quantize_group(k[t, h, g.coords], 8, tg)
            e = k[t, h].copy(); e[g.coords] -= O.dequantize_group(idx, hb, 8, tg)
            for a in range(h * 2, h * 2 + 2):
                want += abs(float(q[t, a] @ e))
    assert m0 == pytest.approx(want / (len(q) * Hq), rel=1e-12)
    # a non-zero offset against explicit rotations (oracle.rope is pinned on its own): q^T R_Delta (k - khat) with
    # R_Delta = RoPE at position Delta applied to the error vector
    D = 37.0
    mD = O.rope_logit_mae(q, k, one, tg, base, offsets=np.array([D]))
    want = 0.0
    for h in range(Hkv):
        g = O.groups_from_bits(one[h], d)[0]
        for t in range(len(q)):
            idx, hb, _ = O.quantize_group(k[t, h, g.coords], 8, tg)
            e = k[t, h].copy(); e[g.coords] -= O.dequantize_group(idx, hb, 8, tg)
            re = O.rope(e[None, None, :], np.array([D]), base)[0, 0]
            for a in range(h * 2, h * 2 + 2):
                want += abs(float(q[t, a] @ re))
    assert mD == pytest.approx(want / (len(q) * Hq), rel=1e-10)

"""Pins for the oracle's V-side allocator path ("a V-side allocator"; reading Q19), CPU only.

What is pinned and against what:
  * v_groups_from_bits        -- a hand-written example
  * v_block_energy            -- closed forms and a pure-Python triple loop on a tiny input
  * the grouped packer        -- hand-worked byte positions (tests/golden/layout_region_vgroups.txt), bijection
                                 (round trip), and byte equality with the already-pinned uniform-V packer
  * grouped quantise / dequantise -- the per-group encoder is the pinned TQ-MSE encoder; the grouped path must agree
                                 with it token by token, and the rate law must hold per V group
  * the allocation itself     -- Alg. 1 is pinned in test_oracle_allocate.py; here: brute force over all width vectors of a
                                 small V head, and the end-to-end property that the allocation lowers the squared
                                 error of V-hat at equal bits on an input with unequal block energies
"""
import itertools
import math
import os

import numpy as np
import pytest

import workloads as W
from oracle import codebook as CB
from oracle import oracle as O

D = 128
ROT = W.rotations(20260624, D)
TAB = O.Tables(ROT, D)


def test_v_groups_example():
    g = O.v_groups_from_bits([3, 1, 3, 1, 1, 1, 1, 1], D)
    assert [x.width for x in g] == [1, 3]
    assert g[0].blocks.tolist() == [1, 3, 4, 5, 6, 7] and g[1].blocks.tolist() == [0, 2]
    assert g[0].m == 96 and g[1].m == 32
    assert g[0].coords[:3].tolist() == [16, 17, 18] and g[0].coords[16] == 48 and g[0].coords[40] == 72
    assert g[1].coords.tolist() == list(range(0, 16)) + list(range(32, 48))
    # uniform widths: one group, natural coordinate order
    g = O.v_groups_from_bits([4] * 8, D)
    assert len(g) == 1 and g[0].coords.tolist() == list(range(D))
    with pytest.raises(AssertionError):
        O.v_groups_from_bits([0] * 8, D)


def test_v_block_energy_closed_forms_and_loop():
    # constant rows: block j of a vector of all c has squared norm 16 c^2
    v = np.full((5, 2, D), 0.5)
    assert np.allclose(O.v_block_energy(v), 16 * 0.25)
    # one-hot: only the block that holds the coordinate sees it, averaged over tokens
    v = np.zeros((4, 1, D))
    v[1, 0, 37] = 3.0
    e = O.v_block_energy(v)
    assert e.shape == (1, 8) and e[0, 2] == 9.0 / 4 and np.count_nonzero(e) == 1
    # pure-Python loop on a tiny random input
    rng = np.random.default_rng(3)
    v = rng.standard_normal((3, 2, 32))
    want = [[sum(v[t, h, 16 * j + u] ** 2 for t in range(3) for u in range(16)) / 3 for j in range(2)] for h in range(2)]
    assert np.allclose(O.v_block_energy(v), want, rtol=1e-14)
    # the synthetic recipe has unequal block energies (else there is nothing to allocate)
    e = O.v_block_energy(W.values_block_scaled(7, 2, 512, 2, D))
    assert e.max() / e.min() > 5


def test_golden_vgroup_byte_positions():
    bits_v = [3, 1, 3, 1, 1, 1, 1, 1]
    vg = O.v_groups_from_bits(bits_v, D)
    order = np.concatenate([g.coords for g in vg])
    n = 0
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "layout_region_vgroups.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        item, where = (x.split() for x in line.split("|"))
        t = 37
        if item[0] == "coord":
            assert order[int(item[1])] == int(item[2]), line
            n += 1
            continue
        q = O.QuantizedHead([], 1, np.zeros((t + 1, 0), np.uint8), np.zeros((t + 1, 0), np.uint16),
                            np.zeros((t + 1, D), np.uint8), np.zeros((t + 1, 2), np.uint16), vgroups=vg)
        if item[0] == "vcode":
            q.vidx[t, int(item[1])] = int(item[2])
        else:
            q.vnorm[t, int(item[1])] = int(item[2], 16)
        region = O.pack_region(q, D)
        assert region.size == 3584
        assert region[int(where[0])] == int(where[1], 16), line
        if item[0] == "vcode":
            assert np.count_nonzero(region) == 1, line
        n += 1
    assert n >= 8


@pytest.mark.parametrize("bits_v", [[1, 2, 3, 4, 5, 6, 7, 8], [3, 1, 3, 1, 1, 1, 1, 1], [4, 4, 2, 2, 2, 2, 4, 4], [8] * 8])
def test_vgroup_pack_round_trip_and_footprint(bits_v):
    rng = np.random.default_rng(sum(bits_v))
    bits_k = rng.integers(0, 5, D // 2)
    groups = O.groups_from_bits(bits_k, D)
    vg = O.v_groups_from_bits(bits_v, D)
    T = 300
    kdim = sum(g.m for g in groups)
    q = O.QuantizedHead(groups, vg[0].width, np.zeros((T, kdim), np.uint8), rng.integers(0, 65536, (T, len(groups))).astype(np.uint16),
                        np.zeros((T, D), np.uint8), rng.integers(0, 65536, (T, len(vg))).astype(np.uint16), vgroups=vg)
    o = 0
    for g in groups:
        q.kidx[:, o:o + g.m] = rng.integers(0, 1 << g.width, (T, g.m))
        o += g.m
    o = 0
    for g in vg:
        q.vidx[:, o:o + g.m] = rng.integers(0, 1 << g.width, (T, g.m))
        o += g.m
    geo = O.tile_geometry(groups, D, 0, 1, vg)
    # dense: 16 bytes per token per average bit on both sides, one norm row per group
    assert geo["stride"] == 16 * 2 * int(bits_k.sum()) + 256 * (len(groups) + len(vg)) + 16 * 16 * sum(bits_v)
    region = O.pack_region(q, D)
    back = O.unpack_region(region, groups, D, 0, T, vgroups=vg)
    assert np.array_equal(back.kidx, q.kidx) and np.array_equal(back.knorm, q.knorm)
    assert np.array_equal(back.vidx, q.vidx) and np.array_equal(back.vnorm, q.vnorm)
    # all-ones codes fill every code bit of the full tiles: the sections have no holes and do not overlap
    q.kidx[:] = 255; q.vidx[:] = 255
    o = 0
    for g in groups:
        q.kidx[:, o:o + g.m] &= (1 << g.width) - 1
        o += g.m
    o = 0
    for g in vg:
        q.vidx[:, o:o + g.m] &= (1 << g.width) - 1
        o += g.m
    q.knorm[:] = 0; q.vnorm[:] = 0
    r = O.pack_region(q, D).reshape(-1, geo["stride"])[:2]
    ones = np.unpackbits(r, axis=1).sum(axis=1)
    width4 = sum(g.m for g in groups if g.width == 4) + sum(g.m for g in vg if g.width == 4)
    # width-4 fields are stored sign-magnitude: idx 15 -> (0, 7) has three ones instead of four
    assert np.all(ones == 128 * (2 * int(bits_k.sum()) + 16 * sum(bits_v)) - 128 * width4)


def test_uniform_bits_v_is_the_uniform_path():
    """bits_v all equal to b_V must reproduce the uniform-V encoder and packer bit for bit."""
    rng = np.random.default_rng(11)
    T = 40
    k = rng.standard_normal((T, D)).astype(np.float32).astype(np.float64)
    v = rng.standard_normal((T, D)).astype(np.float32).astype(np.float64)
    bits = rng.integers(1, 5, D // 2)
    a = O.quantize_head(k, v, bits, 3, TAB)
    b = O.quantize_head(k, v, bits, 0, TAB, bits_v=[3] * 8)
    assert np.array_equal(a.vidx, b.vidx) and np.array_equal(a.vnorm, b.vnorm[:, 0]) and b.b_v == 3
    assert np.array_equal(O.pack_region(a, D), O.pack_region(b, D))
    Ka, Va = O.dequantize_head(a, TAB, D)
    Kb, Vb = O.dequantize_head(b, TAB, D)
    assert np.array_equal(Ka, Kb) and np.array_equal(Va, Vb)


def test_grouped_v_is_the_pinned_encoder_per_group():
    rng = np.random.default_rng(5)
    T = 6
    k = rng.standard_normal((T, D))
    v = W.values_block_scaled(5, 2, T, 1, D)[:, 0].astype(np.float32).astype(np.float64)
    bits_v = [2, 5, 2, 3, 3, 2, 5, 2]
    q = O.quantize_head(k, v, [2] * (D // 2), 0, TAB, bits_v=bits_v)
    _, Vh = O.dequantize_head(q, TAB, D)
    o = 0
    for gi, g in enumerate(q.vgroups):
        for t in range(T):
            idx, h, r = O.quantize_group(v[t, g.coords], g.width, TAB)
            assert np.array_equal(idx, q.vidx[t, o:o + g.m]) and h == q.vnorm[t, gi]
            assert abs(r - np.linalg.norm(v[t, g.coords])) <= 1e-12 * r
            # dequantisation written out: (h / sqrt(m)) Pi^T C[idx], scattered to the group's coordinates
            xh = (O.f16_value(h) / math.sqrt(g.m)) * (TAB.Pi(g.m).astype(np.float64).T @ TAB.C(g.width)[idx])
            assert np.allclose(Vh[t, g.coords], xh, rtol=1e-12, atol=1e-14)
        o += g.m


def test_rate_law_per_v_group():
    """Relative squared error of a V group at width b matches the Lloyd-Max distortion D_b."""
    T = 200
    v = W.values_block_scaled(9, 2, T, 1, D)[:, 0]
    bits_v = [1, 2, 3, 4, 1, 2, 3, 4]
    q = O.quantize_head(np.zeros((T, D)), v, [0] * (D // 2), 0, TAB, bits_v=bits_v)
    _, Vh = O.dequantize_head(q, TAB, D)
    for g in q.vgroups:
        rel = np.sum((v[:, g.coords] - Vh[:, g.coords]) ** 2) / np.sum(v[:, g.coords] ** 2)
        Db = CB.distortion(CB.lloyd_max_levels(g.width))
        assert abs(rel / Db - 1) < 0.08, (g.width, rel, Db)


def test_v_allocation_brute_force_and_gain():
    """Alg. 1 on the V scores: optimal over ALL width vectors (brute force on 4 blocks), and -- on the 8 blocks of a
    head with unequal block energies -- a lower squared error of V-hat than uniform widths at the same bit budget."""
    rng = np.random.default_rng(2)
    for _ in range(5):
        s = np.exp(rng.uniform(-3, 3, 4))
        bits = O.allocate(s, 10, 1, 6)
        best = min((O.objective(s, c), c) for c in itertools.product(range(1, 7), repeat=4) if sum(c) == 10)
        assert abs(O.objective(s, bits) - best[0]) <= 1e-12 * best[0]
    T = 96
    v = W.values_block_scaled(4, 2, T, 1, D)[:, 0]
    s = O.v_block_energy(v[:, None, :])[0]
    bits_v = O.allocate(s, 3 * 8, 1, 8)
    assert int(bits_v.sum()) == 24 and len(set(bits_v.tolist())) > 1
    z = np.zeros((T, D))
    qa = O.quantize_head(z, v, [0] * (D // 2), 0, TAB, bits_v=bits_v)
    qu = O.quantize_head(z, v, [0] * (D // 2), 3, TAB)
    ea = np.sum((v - O.dequantize_head(qa, TAB, D)[1]) ** 2)
    eu = np.sum((v - O.dequantize_head(qu, TAB, D)[1]) ** 2)
    assert ea < 0.8 * eu, (ea, eu)
    # and the objective predicts the measured error: sum_j s_j D_{b_j} * T within 10 %
    pred = T * sum(s[j] * CB.distortion(CB.lloyd_max_levels(int(bits_v[j]))) for j in range(8))
    assert abs(ea / pred - 1) < 0.1, (ea, pred)


def test_attention_with_grouped_v_is_softmax_over_dequantised_rows():
    rng = np.random.default_rng(8)
    T = 70
    k = rng.standard_normal((T, D)).astype(np.float32).astype(np.float64)
    v = W.values_block_scaled(8, 2, T, 1, D)[:, 0].astype(np.float32).astype(np.float64)
    q = rng.standard_normal((2, D))
    qh = O.quantize_head(k, v, [3] * (D // 2), 0, TAB, bits_v=[2, 4, 2, 4, 3, 3, 3, 3])
    out = O.decode_attention_head(q, qh, TAB, D, 1 / math.sqrt(D))
    Kh, Vh = O.dequantize_head(qh, TAB, D)
    for a in range(2):
        l = (Kh @ q[a]) / math.sqrt(D)
        p = np.exp(l - l.max())
        assert np.allclose(out[a], (p / p.sum()) @ Vh, rtol=1e-12, atol=1e-14)

"""Pins for the oracle's packer (BGTQ-v1 physical layout) and attention (CPU only).

Byte accounting: PAPER.md:837 (96 B ideal at 3 bits); split merge: PAPER.md:120.
"""
import math
import os

import numpy as np
import pytest
from scipy.special import softmax as scipy_softmax

from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "layout_fields.txt")


def test_golden_field_positions():
    n = 0
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        parts = line.split()
        b, k, idx = int(parts[0]), int(parts[1]), int(parts[2])
        want = [int(x, 16) for x in parts[3:]]
        assert len(want) == b
        W = np.zeros(8, dtype=np.uint32)
        O.put_field(W, b, k, idx)
        assert W[:b].tolist() == want, line
        assert not W[b:].any()
        assert O.get_field(W, b, k) == idx
        n += 1
    assert n >= 20


@pytest.mark.parametrize("b", range(1, 9))
def test_unit_is_a_bijection(b):
    """Every one of the 32*b bits of a unit belongs to exactly one slot; round trip for all values."""
    seen = np.zeros(b, dtype=np.uint32)
    for k in range(32):
        W = np.zeros(8, dtype=np.uint32)
        # all-ones field pattern that survives the width-4 recoding: put every idx, OR the footprints
        foot = np.zeros(8, dtype=np.uint32)
        for idx in range(1 << b):
            W[:] = 0
            O.put_field(W, b, k, idx)
            assert O.get_field(W, b, k) == idx
            foot |= W
        assert not foot[b:].any()
        assert not (seen & foot[:b]).any()        # disjoint from other slots
        seen |= foot[:b]
        assert sum(bin(int(x)).count("1") for x in foot[:b]) == b
    assert np.all(seen == 0xFFFFFFFF)
    # writing one slot never disturbs the others
    rng = np.random.default_rng(b)
    vals = rng.integers(0, 1 << b, 32)
    W = np.zeros(8, dtype=np.uint32)
    for k in rng.permutation(32):
        O.put_field(W, b, int(k), int(vals[k]))
    for k in rng.permutation(32):
        O.put_field(W, b, int(k), int(vals[k]))   # overwrite in place
    assert [O.get_field(W, b, k) for k in range(32)] == vals.tolist()


def _random_head(rng, bits, b_v, T, d=128):
    groups = O.groups_from_bits(bits, d, 0)
    kdim = sum(g.m for g in groups)
    kidx = np.zeros((T, kdim), np.uint8)
    o = 0
    for g in groups:
        kidx[:, o:o + g.m] = rng.integers(0, 1 << g.width, (T, g.m))
        o += g.m
    return O.QuantizedHead(groups, b_v, kidx, rng.integers(0, 0x7C00, (T, len(groups))).astype(np.uint16),
                           rng.integers(0, 1 << b_v, (T, d)).astype(np.uint8),
                           rng.integers(0, 0x7C00, T).astype(np.uint16))


@pytest.mark.parametrize("bits_kind", ["mixed", "uniform3", "all8", "zeros_and_ones", "ragged"])
def test_region_round_trip_and_accounting(bits_kind):
    rng = np.random.default_rng(5)
    d = 128
    if bits_kind == "mixed":
        bits = rng.integers(0, 9, 64)
    elif bits_kind == "uniform3":
        bits = np.full(64, 3)
    elif bits_kind == "all8":
        bits = np.full(64, 8)
    elif bits_kind == "zeros_and_ones":
        bits = np.array([0, 1] * 32)
    else:
        bits = np.array([1] * 1 + [2] * 3 + [3] * 33 + [4] * 13 + [5] * 7 + [6] * 5 + [7] * 1 + [8] * 1)
    b_v = 3
    T = 128 * 2 + 37                       # two full tiles and a ragged tail
    q = _random_head(rng, bits, b_v, T)
    region = O.pack_region(q, d)
    geo = O.tile_geometry(q.groups, d, b_v)
    n_g = len(q.groups)
    # bytes/token == 2*sum(b_i)/8 + 16*b_V + 2*(n_g+1): zero padding anywhere
    assert geo["stride"] == 32 * int(bits.sum()) + 128 * (16 * b_v + 2 * (n_g + 1))
    assert O.token_bytes(q.groups, d, b_v) == 2 * int(bits.sum()) / 8 + 16 * b_v + 2 * (n_g + 1)
    assert region.size == 3 * geo["stride"]
    u = O.unpack_region(region, q.groups, d, b_v, T)
    assert np.array_equal(u.kidx, q.kidx) and np.array_equal(u.knorm, q.knorm)
    assert np.array_equal(u.vidx, q.vidx) and np.array_equal(u.vnorm, q.vnorm)
    # appending token by token gives the same bytes as packing at once (append preserves neighbours)
    region2 = np.zeros_like(region)
    for (t0, t1) in [(0, 1), (1, 100), (100, 129), (129, T)]:
        part = O.QuantizedHead(q.groups, b_v, q.kidx[t0:t1], q.knorm[t0:t1], q.vidx[t0:t1], q.vnorm[t0:t1])
        O.pack_region(part, d, region2, t_offset=t0)
    assert np.array_equal(region, region2)
    # slots of tokens beyond T stay zero: a full third tile of zero codes only differs there
    full = O.unpack_region(region, q.groups, d, b_v, 3 * 128)
    # (zero bits decode to idx 0 except in width-4 groups, whose sign-magnitude zero is idx 8)
    o = 0
    for g in q.groups:
        assert np.all(full.kidx[T:, o:o + g.m] == (8 if g.width == 4 else 0))
        o += g.m
    assert not full.vnorm[T:].any() and not full.knorm[T:].any()


def test_ideal_three_bit_bytes():
    """pure 3-bit K+V codes are 48+48 = 96 bytes per token and KV head at D=128."""
    groups = O.groups_from_bits([3] * 64, 128, 0)
    geo = O.tile_geometry(groups, 128, 3)
    assert geo["kcode"] // 128 == 48 and (geo["stride"] - geo["vcode_off"]) // 128 == 48
    assert O.token_bytes(groups, 128, 3) == 96 + 2 * 2      # + one K-group norm + one V norm (fp16)


def test_single_code_lands_where_the_spec_says():
    """K coord u of token tau in a full half-step: word (unit + 4*(plane*32+lane)), lane=(tau&7)*4+((u&7)>>1),
    slot=(tau>>4)*4+((tau>>3)&1)*2+(u&1); V coord u: unit J*2+rho, lane (u&7)*4+((tau&7)>>1),
    slot (tau>>4)*4+((tau>>3)&1)*2+(tau&1).  Byte-level check with 8-bit K and V codes."""
    d = 128
    groups = O.groups_from_bits([8] * 64, d, 0)
    geo = O.tile_geometry(groups, d, 8)
    for tau, u in [(0, 0), (1, 0), (8, 1), (17, 10), (127, 127), (77, 64)]:
        q = O.QuantizedHead(groups, 8, np.zeros((128, 128), np.uint8), np.zeros((128, 1), np.uint16),
                            np.zeros((128, d), np.uint8), np.zeros(128, np.uint16))
        q.kidx[tau, u] = 0xA5
        q.vidx[tau, u] = 0x5A
        region = O.pack_region(q, d)
        nz = np.nonzero(region)[0].tolist()
        lane = (tau & 7) * 4 + ((u & 7) >> 1)
        slot = (tau >> 4) * 4 + ((tau >> 3) & 1) * 2 + (u & 1)
        kbyte = (u >> 3) * 8 * 128 + 4 * ((slot >> 2) * 32 + lane) + (slot & 3)
        J, g, rho = u >> 4, u & 7, (u >> 3) & 1
        vlane = g * 4 + ((tau & 7) >> 1)
        vslot = (tau >> 4) * 4 + ((tau >> 3) & 1) * 2 + (tau & 1)
        vbyte = geo["vcode_off"] + (J * 2 + rho) * 8 * 128 + 4 * ((vslot >> 2) * 32 + vlane) + (vslot & 3)
        assert nz == sorted([kbyte, vbyte])
        assert region[kbyte] == 0xA5 and region[vbyte] == 0x5A


def test_attention_is_textbook_softmax():
    rng = np.random.default_rng(3)
    T, d = 300, 128
    K, V, q = rng.standard_normal((T, d)), rng.standard_normal((T, d)), rng.standard_normal(d)
    scale = 1.0 / math.sqrt(d)
    ref = scipy_softmax(scale * (K @ q)) @ V
    assert np.allclose(O.attention(q, K, V, scale), ref, rtol=1e-12, atol=1e-14)
    # T = 1 -> the value itself; all-equal logits -> the mean of the values
    assert np.allclose(O.attention(q, K[:1], V[:1], scale), V[0], rtol=1e-15)
    assert np.allclose(O.attention(np.zeros(d), K, V, scale), V.mean(0), rtol=1e-12)
    # huge logits do not overflow (max subtraction)
    out = O.attention(q * 1e4, K, V, 1.0)
    assert np.all(np.isfinite(out))


@pytest.mark.parametrize("splits", [2, 3, 7, 300])
def test_split_merge_is_exact(splits):
    rng = np.random.default_rng(4)
    T, d = 300, 128
    K, V, q = rng.standard_normal((T, d)) * 3, rng.standard_normal((T, d)), rng.standard_normal(d)
    scale = 0.3
    full = O.attention(q, K, V, scale)
    edges = np.linspace(0, T, splits + 1).astype(int)
    parts = [O.attention_partial(q, K[a:b], V[a:b], scale) for a, b in zip(edges[:-1], edges[1:]) if b > a]
    assert np.allclose(O.merge_partials(parts), full, rtol=1e-12, atol=1e-14)


def test_decode_attention_head_equals_rotated_domain_form(tab128):
    """The plain definition (de-rotate every key) equals the folded form the GPU uses (rotate q once,
    de-rotate the output once): q'=Pi q/sqrt(m), logits from codes, out = Pi^T acc/sqrt(d)."""
    import workloads as W
    d = 128
    rng = np.random.default_rng(8)
    scales = W.block_scales(0, 1, 64)
    k = W.pre_rope_gaussian(0, 2, 200, 1, d, scales)[:, 0].astype(np.float32).astype(np.float64)
    v = W.values_gaussian(0, 3, 200, 1, d)[:, 0].astype(np.float32).astype(np.float64)
    bits = O.allocate(2 * scales[0], 192, 0, 8)
    qh = O.quantize_head(k, v, bits, 3, tab128)
    qv = rng.standard_normal((2, d))
    scale = 1 / math.sqrt(d)
    plain = O.decode_attention_head(qv, qh, tab128, d, scale)
    for a in range(2):
        logits = np.zeros(200)
        o = 0
        for gi, g in enumerate(qh.groups):
            qp = tab128.Pi(g.m).astype(np.float64) @ qv[a, g.coords] / math.sqrt(g.m)
            h = qh.knorm[:, gi].view(np.float16).astype(np.float64)
            logits += h * (tab128.C(g.width)[qh.kidx[:, o:o + g.m]] @ qp)
            o += g.m
        p = scipy_softmax(scale * logits)
        hv = qh.vnorm.view(np.float16).astype(np.float64)
        acc = (p * hv) @ tab128.C(3)[qh.vidx]
        folded = tab128.Pi(d).astype(np.float64).T @ acc / math.sqrt(d)
        assert np.allclose(folded, plain[a], rtol=1e-10, atol=1e-12)


def test_prefill_oracle_rows_are_decode_steps(tab128):
    """causal prefill row i == the decode-step attention over the first pos0+i+1 cached tokens; the
    first row of a chunk starting at 0 is exactly vhat_0 (softmax over one token)."""
    import workloads as W
    from oracle import oracle as O
    rng = np.random.default_rng(9)
    T, d = 40, 128
    k = rng.standard_normal((T, d)); v = rng.standard_normal((T, d))
    bits = np.array([3] * 64, dtype=np.uint8); bits[:8] = 5; bits[8:16] = 1
    head = O.quantize_head(k, v, bits, 3, tab128)
    q = rng.standard_normal((T, 2, d))
    out = O.prefill_attention_head(q, head, tab128, d, 0.1, 0)
    K, V = O.dequantize_head(head, tab128, d)
    assert np.allclose(out[0, 0], V[0], atol=1e-12) and np.allclose(out[0, 1], V[0], atol=1e-12)
    for i in (5, 39):
        for a in range(2):
            assert np.allclose(out[i, a], O.attention(q[i, a], K[:i + 1], V[:i + 1], 0.1), atol=1e-12)
    out2 = O.prefill_attention_head(q[30:], head, tab128, d, 0.1, 30)        # a later chunk of the same sequence
    assert np.allclose(out2, out[30:], atol=1e-12)


# ----------------------------------------------------------------------------- protected regime
def _protected_case(tab128, T, seed=21):
    rng = np.random.default_rng(seed)
    d = 128
    k = rng.standard_normal((T, d)) * np.repeat(np.exp(rng.uniform(-2, 1, 64)), 2)
    v = rng.standard_normal((T, d))
    bits = np.array([3] * 64, dtype=np.uint8); bits[:10] = 5; bits[10:25] = 1; bits[25:30] = 4; bits[30:35] = 2
    head = O.quantize_head(k, v, bits, 2, tab128)                       # K3V2, the AIME budget
    k16 = k.astype(np.float16).astype(np.float64)
    v16 = v.astype(np.float16).astype(np.float64)
    q = rng.standard_normal((2, d))
    return head, k16, v16, q, d


def test_protected_sets_partition_and_ring_slots():
    """[sink | compressed | recent]: the sets partition 0..T-1; short sequences are all protected;
    the ring slot of every currently-recent token is unique and inside the buffer."""
    for T, ns, nr in [(300, 4, 128), (132, 4, 128), (133, 4, 128), (100, 4, 128), (3, 4, 128), (300, 0, 0), (300, 0, 7), (300, 5, 0)]:
        prot, comp = O.protected_sets(T, ns, nr)
        assert sorted(np.concatenate([prot, comp]).tolist()) == list(range(T))
        assert len(comp) == max(0, T - ns - nr)
        if len(comp):
            assert comp[0] == ns and comp[-1] == T - nr - 1
        slots = [O.window_slot(int(t), ns, nr) for t in prot]
        assert len(set(slots)) == len(slots) and all(0 <= s < ns + nr for s in slots)


def test_protected_attention_limits_and_three_way_merge(tab128):
    """n_sink = n_recent = 0 is the buffer-free packed path; a window covering every token is textbook softmax attention
    over the fp16 rows (scipy); in between, the result equals the exact LSE merge of the three segments
    computed separately -- which is how the GPU evaluates it."""
    T = 300
    head, k16, v16, q, d = _protected_case(tab128, T)
    scale = 1 / math.sqrt(d)
    none = O.decode_attention_protected_head(q, head, tab128, d, scale, k16, v16, 0, 0)
    assert np.array_equal(none, O.decode_attention_head(q, head, tab128, d, scale))
    full = O.decode_attention_protected_head(q, head, tab128, d, scale, k16, v16, 4, T)
    for a in range(2):
        assert np.allclose(full[a], scipy_softmax(scale * (k16 @ q[a])) @ v16, rtol=1e-12, atol=1e-14)
    out = O.decode_attention_protected_head(q, head, tab128, d, scale, k16, v16, 4, 128)
    K, V = O.dequantize_head(head, tab128, d)
    for a in range(2):
        parts = [O.attention_partial(q[a], k16[:4], v16[:4], scale),
                 O.attention_partial(q[a], K[4:T - 128], V[4:T - 128], scale),
                 O.attention_partial(q[a], k16[T - 128:], v16[T - 128:], scale)]
        assert np.allclose(O.merge_partials(parts), out[a], rtol=1e-12, atol=1e-14)
    # it really differs from both limits, and protecting tokens moves the output towards the unquantised one
    exact = np.stack([O.attention(q[a], k16, v16, scale) for a in range(2)])
    assert np.max(np.abs(out - none)) > 1e-4
    assert np.linalg.norm(out - exact) < np.linalg.norm(none - exact)


def test_protected_attention_short_sequences(tab128):
    """T <= n_sink + n_recent: nothing is served from the compressed cache."""
    for T in (1, 3, 100, 132):
        head, k16, v16, q, d = _protected_case(tab128, T, seed=T)
        out = O.decode_attention_protected_head(q, head, tab128, d, 0.1, k16, v16, 4, 128)
        for a in range(2):
            assert np.allclose(out[a], scipy_softmax(0.1 * (k16 @ q[a])) @ v16, rtol=1e-12, atol=1e-14)


# ----------------------------------------------------------------------------- BGTQ-v2 (row order)
GOLDEN_V2 = os.path.join(os.path.dirname(__file__), "golden", "layout_fields_v2.txt")
GOLDEN_REGION_V2 = os.path.join(os.path.dirname(__file__), "golden", "layout_region_v2.txt")


def _nw_spec(b, r):
    """nw(b, r) retyped from DESIGN.md section 4b (not from the oracle)."""
    nwm = min(3, -(-r // 8))
    return {1: 1, 2: -(-r // 16), 3: nwm, 4: nwm + 1}.get(b, -(-r * b // 32))


def test_v2_golden_field_positions():
    n = 0
    for line in open(GOLDEN_V2):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        parts = line.split()
        b, r, k, idx = (int(x) for x in parts[:4])
        want = [int(x, 16) for x in parts[4:]]
        assert len(want) == _nw_spec(b, r) == O.chunk_words_v2(b, r), line
        W = np.zeros(8, dtype=np.uint32)
        O.put_field_v2(W, b, r, k, idx)
        assert W[:len(want)].tolist() == want, line
        assert not W[len(want):].any()
        assert O.get_field_v2(W, b, r, k) == idx
        n += 1
    assert n >= 20


@pytest.mark.parametrize("b", range(1, 9))
def test_v2_chunk_slots_are_disjoint_and_fit(b):
    """For every chunk size r (even, 2..32): the r slots own disjoint bit sets of exactly b bits inside nw(b, r) words."""
    for r in range(2, 33, 2):
        nw = O.chunk_words_v2(b, r)
        assert nw == _nw_spec(b, r)
        assert 32 * nw >= r * b
        seen = np.zeros(8, dtype=np.uint32)
        for k in range(r):
            foot = np.zeros(8, dtype=np.uint32)
            for idx in range(1 << b):
                W = np.zeros(8, dtype=np.uint32)
                O.put_field_v2(W, b, r, k, idx)
                assert O.get_field_v2(W, b, r, k) == idx
                foot |= W
            assert not foot[nw:].any(), (b, r, k)
            assert not (seen & foot).any()
            seen |= foot
            assert sum(bin(int(x)).count("1") for x in foot) == b
    # a full chunk uses every bit
    assert np.all(seen[:b] == 0xFFFFFFFF)


def test_v2_golden_region_positions():
    """One code / norm written into an otherwise zero head lands on the hand-computed byte."""
    d, b_v = 128, 2
    groups = [O.Group(1, np.array([0], np.int64), np.array([0, 64], np.int64)),
              O.Group(3, np.arange(1, 18, dtype=np.int64), np.concatenate([[i, i + 64] for i in range(1, 18)]).astype(np.int64))]
    assert [g.m for g in groups] == [2, 34]
    geo = O.tile_geometry(groups, d, b_v, version=2)
    assert geo == dict(kcode=2560, knorm_off=2560, vnorm_off=3072, vcode_off=3328, stride=7424)
    n = 0
    for line in open(GOLDEN_REGION_V2):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        what, index, value, off, byte = line.split()
        t = 165 if what.endswith("165") else 37
        T = t + 1
        q = O.QuantizedHead(groups, b_v, np.zeros((T, 36), np.uint8), np.zeros((T, 2), np.uint16),
                            np.zeros((T, d), np.uint8), np.zeros(T, np.uint16))
        if what.startswith("kcode"):
            q.kidx[t, int(index)] = int(value)
        elif what == "knorm":
            q.knorm[t, int(index)] = int(value, 16)
        elif what == "vnorm":
            q.vnorm[t] = int(value, 16)
        else:
            q.vidx[t, int(index)] = int(value)
        region = O.pack_region(q, d, version=2)
        assert region[int(off)] == int(byte, 16), line
        if what != "knorm" and what != "vnorm":
            assert np.count_nonzero(region) == 1, line
        n += 1
    assert n >= 8


@pytest.mark.parametrize("bits_kind", ["mixed", "uniform3", "all8", "zeros_and_ones", "ragged"])
def test_v2_region_round_trip_and_accounting(bits_kind):
    rng = np.random.default_rng(6)
    d = 128
    bits = {"mixed": rng.integers(0, 9, 64), "uniform3": np.full(64, 3), "all8": np.full(64, 8),
            "zeros_and_ones": np.array([0, 1] * 32),
            "ragged": np.array([1] * 1 + [2] * 3 + [3] * 33 + [4] * 13 + [5] * 7 + [6] * 5 + [7] * 1 + [8] * 1)}[bits_kind]
    b_v = 3
    T = 128 * 2 + 37
    q = _random_head(rng, bits, b_v, T)
    region = O.pack_region(q, d, version=2)
    geo = O.tile_geometry(q.groups, d, b_v, version=2)
    # byte accounting from the spec: K codes = 4 quadrants x 128 B x sum of nw over chunks
    words = sum(_nw_spec(g.width, min(32, g.m - 32 * u)) for g in q.groups for u in range(-(-g.m // 32)))
    assert geo["kcode"] == 4 * 128 * words
    assert geo["stride"] == geo["kcode"] + 256 * (len(q.groups) + 1) + 16 * d * b_v
    # never smaller than the dense v1 tile, and equal to it when every group is a multiple of 32 coordinates
    v1 = O.tile_geometry(q.groups, d, b_v)["stride"]
    assert geo["stride"] >= v1
    if all(g.m % 32 == 0 for g in q.groups):
        assert geo["stride"] == v1
    assert region.size == 3 * geo["stride"]
    u = O.unpack_region(region, q.groups, d, b_v, T, version=2)
    assert np.array_equal(u.kidx, q.kidx) and np.array_equal(u.knorm, q.knorm)
    assert np.array_equal(u.vidx, q.vidx) and np.array_equal(u.vnorm, q.vnorm)
    region2 = np.zeros_like(region)
    for (t0, t1) in [(0, 1), (1, 100), (100, 129), (129, T)]:
        part = O.QuantizedHead(q.groups, b_v, q.kidx[t0:t1], q.knorm[t0:t1], q.vidx[t0:t1], q.vnorm[t0:t1])
        O.pack_region(part, d, region2, t_offset=t0, version=2)
    assert np.array_equal(region, region2)
    full = O.unpack_region(region, q.groups, d, b_v, 3 * 128, version=2)
    o = 0
    for g in q.groups:
        assert np.all(full.kidx[T:, o:o + g.m] == (8 if g.width == 4 else 0))
        o += g.m
    assert not full.vnorm[T:].any() and not full.knorm[T:].any()


def test_v1_golden_region_positions_partial_half_steps_and_norm_slot():
    """Hand-worked byte positions of BGTQ-v1: trailing partial half-steps (r = 2, 4, 6) and norm_slot."""
    d = 128
    n = 0
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "layout_region_v1.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, item, where = (x.split() for x in line.split("|"))
        m, b, b_v = (int(x) for x in head)
        blocks = np.arange(m // 2, dtype=np.int64)
        groups = [O.Group(b, blocks, np.concatenate([[i, i + 64] for i in blocks]).astype(np.int64))]
        t = 45
        q = O.QuantizedHead(groups, b_v, np.zeros((t + 1, m), np.uint8), np.zeros((t + 1, 1), np.uint16),
                            np.zeros((t + 1, d), np.uint8), np.zeros(t + 1, np.uint16))
        if item[0] == "kcode":
            q.kidx[t, int(item[1])] = int(item[2])
        elif item[0] == "knorm":
            q.knorm[t, int(item[1])] = int(item[2], 16)
        else:
            q.vnorm[t] = int(item[2], 16)
        region = O.pack_region(q, d)
        assert region[int(where[0])] == int(where[1], 16), line
        if item[0] == "kcode":
            assert np.count_nonzero(region) == 1, line
        n += 1
    assert n >= 6

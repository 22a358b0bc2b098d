"""-m gpu: the V-side allocator path (reading Q19) through the C-ABI against
the oracle: V block energy (rel 1e-5), allocation (bit-exact), grouped append (packed bytes bit-exact), decode attention
contiguous and protected (<= 2e-3 of R_V), uniform bits_v == the uniform layout byte for byte.
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
import bgtq_helpers as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_24033_b200 as pkg
    return pkg


def _cuda(a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a)).to(dtype).cuda()


def _problem(seed, T, Hq, Hkv, b_k, bbar_v, bmin=1, bmax=8, kv_dtype="f32", bits_v=None):
    """make_problem with block-scaled values and V widths from the oracle's V-side allocation."""
    p = H.make_problem(seed, T, Hq, Hkv, b_k, 0, bmin, bmax, kv_dtype=kv_dtype)
    v = W.values_block_scaled(seed, 2, T, Hkv, p.d_h)
    p.v = (W.round_to_bf16(v) if kv_dtype == "bf16" else v.astype(np.float32)).astype(np.float64)
    if bits_v is None:
        sv = O.v_block_energy(p.v)
        bits_v = np.stack([O.allocate(sv[h], bbar_v * 8, 1, 8) for h in range(Hkv)])
    return p, np.asarray(bits_v, dtype=np.uint8)


def _heads(p, bits_v, tab, t1=None):
    t1 = p.T if t1 is None else t1
    return [O.quantize_head(p.k_post[:t1, h], p.v[:t1, h], p.bits[h], 0, tab, bits_v=bits_v[h]) for h in range(p.Hkv)]


def _append(P, p, bits_v, tab, chunks, max_tokens, kv_dtype="f32", exact=False):
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, 0, p.rot, bits_v=bits_v[None], exact_codebooks=exact)
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    tdt = torch.float32 if kv_dtype == "f32" else torch.bfloat16
    t = 0
    for n in chunks:
        P.quantize_append(lay, 0, cache, _cuda(p.k_post[None, t:t + n], tdt), _cuda(p.v[None, t:t + n], tdt), seq, max_tokens)
        t += n
    assert int(seq.item()) == t
    heads = _heads(p, bits_v, tab, t)
    host = cache.cpu().numpy()
    n_cap = (max_tokens + 127) // 128
    for h in range(p.Hkv):
        stride = lay.tile_stride(0, h)
        assert stride == O.tile_geometry(heads[h].groups, p.d_h, 0, 1, heads[h].vgroups)["stride"]
        off = lay.region_offset(0, 0, h, 1, max_tokens)
        exp = np.zeros(n_cap * stride, dtype=np.uint8)
        O.pack_region(heads[h], p.d_h, exp)
        got = host[off:off + n_cap * stride]
        if not np.array_equal(got, exp):
            u = O.unpack_region(got, heads[h].groups, p.d_h, 0, t, vgroups=heads[h].vgroups)
            raise AssertionError(f"head {h}: packed bytes differ (k codes {int(np.count_nonzero(u.kidx != heads[h].kidx))}, "
                                 f"v codes {int(np.count_nonzero(u.vidx != heads[h].vidx))}, "
                                 f"v norms {int(np.count_nonzero(u.vnorm != heads[h].vnorm))})")
    return lay, cache, seq, heads


def _attention_err(P, p, lay, cache, seq, heads, tab, max_tokens, name):
    scale = 1.0 / math.sqrt(p.d_h)
    q = _cuda(p.q_post[None], torch.bfloat16)
    out = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    exp, rv = H.oracle_attention(p, heads, tab, scale)
    got = out[0].double().cpu().numpy()
    G = p.Hq // p.Hkv
    err = max(H.record_error(f"{name}/head{a}", got[a], exp[a], rv[a // G]) for a in range(p.Hq))
    return err


# ----------------------------------------------------------------------------- score and allocation
@pytest.mark.parametrize("dtype,Hkv,n", [("f32", 2, 1000), ("bf16", 8, 4097), ("f32", 1, 1), ("bf16", 3, 77)])
def test_v_block_energy(P, dtype, Hkv, n):
    v = W.values_block_scaled(31, 2, n, Hkv, 128)
    vd = _cuda(v, torch.float32 if dtype == "f32" else torch.bfloat16)
    got = P.v_block_energy(vd).cpu().numpy().astype(np.float64)
    exp = O.v_block_energy(vd.double().cpu().numpy())
    assert got.shape == (Hkv, 8)
    assert np.max(np.abs(got - exp) / exp) <= 1e-5
    assert np.array_equal(got, P.v_block_energy(vd).cpu().numpy().astype(np.float64))      # deterministic


def test_v_energy_then_allocate_chain(P):
    """scores -> bgtq_allocate with 8 blocks per head: the device allocation is optimal for the oracle's scores and
    equals the oracle's allocation of the library's own (fp32) scores bit for bit."""
    Hkv = 8
    v = W.values_block_scaled(32, 2, 2048, Hkv, 128).astype(np.float32)
    s = P.v_block_energy(_cuda(v, torch.float32))
    bits = P.allocate(s, 3 * 8, 1, 8).cpu().numpy()
    s_lib = s.cpu().numpy().astype(np.float64)
    s_or = O.v_block_energy(v.astype(np.float64))
    for h in range(Hkv):
        assert np.array_equal(bits[h], O.allocate(s_lib[h], 24, 1, 8))
        assert bits[h].sum() == 24
        assert O.objective(s_or[h], bits[h]) <= O.objective(s_or[h], O.allocate(s_or[h], 24, 1, 8)) * (1 + 1e-6)
    assert len({tuple(b) for b in bits.tolist()}) > 1


# ----------------------------------------------------------------------------- layout
def test_uniform_bits_v_is_the_uniform_layout(P, tab128):
    """All V widths of a head equal: same strides, same bytes, same attention output as bgtq_layout_create(b_v)."""
    p = H.make_problem(41, 300, 8, 2, 3, 3, 1, 8)
    bits_v = np.full((2, 8), 3, np.uint8)
    la = P.Layout(p.bits[None], p.Hq, p.d_h, 3, p.rot)
    lb = P.Layout(p.bits[None], p.Hq, p.d_h, 0, p.rot, bits_v=bits_v[None])
    assert la.cache_bytes(1, 384) == lb.cache_bytes(1, 384)
    outs = []
    for lay in (la, lb):
        cache = lay.new_cache(1, 384)
        seq = torch.zeros(1, dtype=torch.int32, device="cuda")
        P.quantize_append(lay, 0, cache, _cuda(p.k_post[None], torch.float32), _cuda(p.v[None], torch.float32), seq, 384)
        q = _cuda(p.q_post[None], torch.bfloat16)
        outs.append((cache.cpu().numpy(), P.decode_attention(lay, 0, cache, q, seq, 384, 0.088, lay.new_workspace(1)).cpu()))
    assert np.array_equal(outs[0][0], outs[1][0])
    assert torch.equal(outs[0][1], outs[1][1])


def test_heads_with_different_uniform_v_widths(P, tab128):
    """One V group per head but another width in each head: served by the ordinary kernels (prefill included)."""
    bits_v = np.array([[2] * 8, [5] * 8], np.uint8)
    p, bits_v = _problem(42, 260, 8, 2, 3, 0, bits_v=bits_v)
    lay, cache, seq, heads = _append(P, p, bits_v, tab128, [260], 384)
    assert _attention_err(P, p, lay, cache, seq, heads, tab128, 384, "vside/per_head_uniform") <= 2e-3
    scale = 1.0 / math.sqrt(128)
    q = _cuda(p.q_post[None, None], torch.bfloat16)                      # one query token at position T-1 sees [0, T)
    out = P.prefill_attention(lay, 0, cache, q, seq, 384, scale)
    exp, rv = H.oracle_attention(p, heads, tab128, scale)
    got = out[0, 0].double().cpu().numpy()
    assert max(np.max(np.abs(got[a] - exp[a])) / rv[a // 4] for a in range(8)) <= 2e-3


def test_argument_errors(P, tab128):
    p = H.make_problem(43, 10, 4, 2, 3, 3, 1, 8)
    bad = np.full((1, 2, 8), 3, np.uint8)
    bad[0, 1, 3] = 0
    with pytest.raises(P.BgtqError):
        P.Layout(p.bits[None], 4, 128, 0, p.rot, bits_v=bad)
    bad[0, 1, 3] = 9
    with pytest.raises(P.BgtqError):
        P.Layout(p.bits[None], 4, 128, 0, p.rot, bits_v=bad)
    ok = np.array([[[2, 2, 4, 4, 3, 3, 3, 3], [3] * 8]], np.uint8)
    with pytest.raises(P.BgtqError):                                     # row-order format: one V group only
        P.Layout(p.bits[None], 4, 128, 0, p.rot, bits_v=ok, fmt=P.FORMAT_V2)
    lay = P.Layout(p.bits[None], 4, 128, 0, p.rot, bits_v=ok)
    cache = lay.new_cache(1, 128)
    seq = torch.full((1,), 10, dtype=torch.int32, device="cuda")
    q = torch.zeros((1, 1, 4, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(P.BgtqError):                                     # grouped V: prefill is not built
        P.prefill_attention(lay, 0, cache, q, seq, 128, 0.088)


# ----------------------------------------------------------------------------- append + attention
@pytest.mark.parametrize("kv_dtype,chunks", [("f32", [333]), ("bf16", [100, 27, 1, 1, 1, 203])])
def test_grouped_append_bit_exact(P, tab128, kv_dtype, chunks):
    p, bits_v = _problem(51, sum(chunks), 8, 2, 3, 3, kv_dtype=kv_dtype)
    assert any(len(set(b.tolist())) > 1 for b in bits_v)
    _append(P, p, bits_v, tab128, chunks, 512, kv_dtype)


@pytest.mark.parametrize("bits_v", [[1, 2, 3, 4, 5, 6, 7, 8], [8, 7, 6, 5, 4, 3, 2, 1], [3, 1, 3, 1, 1, 1, 1, 1], [4, 4, 2, 2, 2, 2, 4, 4]])
def test_grouped_append_every_width(P, tab128, bits_v):
    p, bv = _problem(52, 150, 2, 1, 2, 0, bits_v=np.array([bits_v], np.uint8))
    lay, cache, seq, heads = _append(P, p, bv, tab128, [150], 256)
    assert _attention_err(P, p, lay, cache, seq, heads, tab128, 256, "vside/widths" + "".join(map(str, bits_v))) <= 2e-3


@pytest.mark.parametrize("T,Hq,Hkv,b_k,bbar_v", [(1, 8, 2, 3, 3), (129, 8, 1, 3, 3), (1000, 16, 2, 3, 3), (515, 8, 2, 2, 2), (4096, 8, 8, 3, 4)])
def test_grouped_attention(P, tab128, T, Hq, Hkv, b_k, bbar_v):
    p, bits_v = _problem(60 + T, T, Hq, Hkv, b_k, bbar_v)
    max_tokens = (T + 127) // 128 * 128
    lay, cache, seq, heads = _append(P, p, bits_v, tab128, [T], max_tokens)
    assert _attention_err(P, p, lay, cache, seq, heads, tab128, max_tokens, f"vside/T{T}_K{b_k}V{bbar_v}") <= 2e-3


def test_grouped_attention_many_tiles_multi_cta(P, tab128):
    """One KV head, 40,000 tokens: the tile range is split over every CTA and merged by combine_kernel in grouped order."""
    T = 40000
    p, bits_v = _problem(70, T, 4, 1, 3, 3)
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, 0, p.rot, bits_v=bits_v[None])
    max_tokens = (T + 127) // 128 * 128
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    P.quantize_append(lay, 0, cache, _cuda(p.k_post[None], torch.float32), _cuda(p.v[None], torch.float32), seq, max_tokens)
    # expected output from the library's own codes (bit-exactness of the append is covered above): unpack with the oracle
    host = cache.cpu().numpy()
    vg = O.v_groups_from_bits(bits_v[0], 128)
    groups = O.groups_from_bits(p.bits[0], 128)
    stride = lay.tile_stride(0, 0)
    qh = O.unpack_region(host[:stride * (max_tokens // 128)], groups, 128, 0, T, vgroups=vg)
    ref = O.quantize_head(p.k_post[:300, 0], p.v[:300, 0], p.bits[0], 0, tab128, bits_v=bits_v[0])
    assert np.array_equal(qh.vidx[:300], ref.vidx) and np.array_equal(qh.vnorm[:300], ref.vnorm) and np.array_equal(qh.kidx[:300], ref.kidx)
    assert _attention_err(P, p, lay, cache, seq, [qh], tab128, max_tokens, "vside/T40000") <= 2e-3


def test_grouped_layers_and_ragged_batch(P, tab128):
    """2 layers x 3 sequences (one empty) in one launch; every layer / head has its own V grouping."""
    Lyr, B, Hq, Hkv, d = 2, 3, 8, 2, 128
    lens = [300, 0, 77]
    probs = [[_problem(80 + 10 * l + b, max(lens[b], 1), Hq, Hkv, 3, 3) for b in range(B)] for l in range(Lyr)]
    bits = np.stack([probs[l][0][0].bits for l in range(Lyr)])
    bits_v = np.stack([probs[l][0][1] for l in range(Lyr)])
    rot = probs[0][0][0].rot
    lay = P.Layout(bits, Hq, d, 0, rot, bits_v=bits_v)
    max_tokens = 384
    cache = lay.new_cache(B, max_tokens)
    seq = torch.zeros(B, dtype=torch.int32, device="cuda")
    for l in range(Lyr):
        for b in range(B):
            if lens[b] == 0:
                continue
            p = probs[l][b][0]
            k = torch.zeros((B, lens[b], Hkv, d), dtype=torch.float32, device="cuda"); v = torch.zeros_like(k)
            k[b] = _cuda(p.k_post, torch.float32); v[b] = _cuda(p.v, torch.float32)
            s1 = torch.full((B,), max_tokens, dtype=torch.int32, device="cuda")     # the other sequences are "full": nothing appended
            s1[b] = 0
            P.quantize_append(lay, l, cache, k, v, s1, max_tokens, advance_seq_len=False)
    seq[:] = torch.tensor(lens, dtype=torch.int32)
    q = torch.zeros((Lyr, B, Hq, d), dtype=torch.bfloat16, device="cuda")
    for l in range(Lyr):
        for b in range(B):
            q[l, b] = _cuda(probs[l][b][0].q_post, torch.bfloat16)
    scale = 1.0 / math.sqrt(d)
    out = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, lay.new_workspace(B, Lyr), n_layers=Lyr)
    torch.cuda.synchronize()
    for l in range(Lyr):
        for b in range(B):
            got = out[l, b].double().cpu().numpy()
            if lens[b] == 0:
                assert not got.any()
                continue
            p = probs[l][b][0]
            heads = [O.quantize_head(p.k_post[:, h], p.v[:, h], bits[l, h], 0, tab128, bits_v=bits_v[l, h]) for h in range(Hkv)]
            pp = H.Problem(d, Hq, Hkv, lens[b], 0, bits[l], p.k_post, p.v, p.q_post, p.scores, rot)
            exp, rv = H.oracle_attention(pp, heads, tab128, scale)
            assert max(np.max(np.abs(got[a] - exp[a])) / rv[a // 4] for a in range(Hq)) <= 2e-3, (l, b)


@pytest.mark.parametrize("T,n_sink,n_recent", [(300, 4, 128), (100, 4, 128), (700, 16, 64)])
def test_grouped_protected_regime(P, tab128, T, n_sink, n_recent):
    """fp16 sink / recent windows over a cache with V-side groups: window_kernel writes its record
    in grouped V order, combine_kernel de-rotates per V group."""
    Hq, Hkv = 8, 2
    p, bits_v = _problem(90 + T, T, Hq, Hkv, 3, 2)
    lay = P.Layout(p.bits[None], Hq, p.d_h, 0, p.rot, bits_v=bits_v[None])
    max_tokens = (T + 127) // 128 * 128 + 128
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    win_k, win_v = P.new_windows(lay, 1, n_sink, n_recent)
    kk = _cuda(p.k_post[None], torch.float32); vv = _cuda(p.v[None], torch.float32)
    P.window_append(lay, 0, kk, vv, seq, win_k, win_v, n_sink, n_recent)
    P.quantize_append(lay, 0, cache, kk, vv, seq, max_tokens)
    heads = _heads(p, bits_v, tab128)
    scale = 1.0 / math.sqrt(p.d_h)
    q = _cuda(p.q_post[None], torch.bfloat16)
    out = P.decode_attention_protected(lay, 0, cache, q, seq, max_tokens, scale, win_k, win_v, n_sink, n_recent, lay.new_workspace(1))
    torch.cuda.synchronize()
    k16 = p.k_post.astype(np.float16).astype(np.float64); v16 = p.v.astype(np.float16).astype(np.float64)
    G = Hq // Hkv
    exp = np.concatenate([O.decode_attention_protected_head(p.q_post[h * G:(h + 1) * G], heads[h], tab128, p.d_h, scale,
                                                             k16[:, h], v16[:, h], n_sink, n_recent) for h in range(Hkv)])
    _, rv = H.oracle_attention(p, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    assert max(np.max(np.abs(got[a] - exp[a])) / rv[a // G] for a in range(Hq)) <= 2e-3


def test_grouped_exact_density_codebooks(P, rot128):
    """BGTQ_CODEBOOK_EXACT with V-side groups: V group (w, m) uses C_{w,m} in append and in the decode kernel."""
    tab = O.Tables(rot128, 128, cb_kind="sphere")
    p, bits_v = _problem(95, 333, 8, 2, 3, 3)
    lay, cache, seq, heads = _append(P, p, bits_v, tab, [333], 384, exact=True)
    assert _attention_err(P, p, lay, cache, seq, heads, tab, 384, "vside/exact") <= 2e-3


def test_v_allocation_lowers_the_output_error(P, tab128):
    """End to end on block-scaled values: at the same V bits the allocated widths give a smaller attention-output error
    against the fp64 attention over the UNQUANTISED values than uniform widths (the point of a V-side allocator)."""
    T, Hq, Hkv = 1000, 8, 2
    p, bits_v = _problem(97, T, Hq, Hkv, 3, 3)
    scale = 1.0 / math.sqrt(128)
    q = _cuda(p.q_post[None], torch.bfloat16)
    errs = []
    for bv in (bits_v, np.full_like(bits_v, 3)):
        lay = P.Layout(p.bits[None], Hq, 128, 0, p.rot, bits_v=bv[None])
        cache = lay.new_cache(1, 1024)
        seq = torch.zeros(1, dtype=torch.int32, device="cuda")
        P.quantize_append(lay, 0, cache, _cuda(p.k_post[None], torch.float32), _cuda(p.v[None], torch.float32), seq, 1024)
        got = P.decode_attention(lay, 0, cache, q, seq, 1024, scale, lay.new_workspace(1))[0].double().cpu().numpy()
        heads = _heads(p, bv, tab128)
        e = 0.0
        for a in range(Hq):
            Kh, _ = O.dequantize_head(heads[a // 4], tab128, 128)
            ref = O.attention(p.q_post[a], Kh, p.v[:, a // 4], scale)      # same (quantised) keys, exact values
            e += float(np.sum((got[a] - ref) ** 2))
        errs.append(e)
    assert errs[0] < 0.9 * errs[1], errs            # (measured 0.83: a few tokens carry most of the softmax weight)

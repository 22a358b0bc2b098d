"""-m gpu: the CUDA path (through the C-ABI binding) against the fp64 oracle, element by element.

Bars (BASELINE.json north_star): allocations, codes, fp16 norms and packed bytes bit-exact;
block energy rel 1e-5; attention max-abs error / R_V <= 2e-3 (R_V = rms row norm of the
dequantised V of that KV head).
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


# ----------------------------------------------------------------------------- unpack routine
@pytest.mark.parametrize("b", [1, 2, 3, 4, 5, 6, 7, 8])
def test_decode_unit_matches_oracle_fields(P, b):
    rng = np.random.default_rng(100 + b)
    words = rng.integers(0, 2**32, size=(b, 32), dtype=np.uint64).astype(np.uint32)
    got = P.debug_decode_unit(b, words)
    cb = O._cb.codebook(b)
    for lane in range(32):
        Wl = np.ascontiguousarray(words[:, lane])
        exp = np.array([cb[O.get_field(Wl, b, k)] for k in range(32)])
        assert np.array_equal(got[lane].astype(np.float64), exp), (b, lane)


# ----------------------------------------------------------------------------- a1 energy
@pytest.mark.parametrize("dtype,Hq,Hkv,nq,nk", [("f32", 1, 1, 512, 4096), ("bf16", 16, 2, 300, 1000),
                                              ("f32", 8, 2, 0, 77), ("bf16", 4, 4, 5, 0)])
def test_block_energy(P, dtype, Hq, Hkv, nq, nk):
    scales = W.block_scales(7, Hkv, 64)
    q = W.pre_rope_gaussian(7, 1, nq, Hq, 128, scales)
    k = W.pre_rope_gaussian(7, 2, nk, Hkv, 128, scales)
    tdt = torch.float32 if dtype == "f32" else torch.bfloat16
    qd, kd = _cuda(q, tdt), _cuda(k, tdt)
    q64, k64 = qd.double().cpu().numpy(), kd.double().cpu().numpy()     # exact values the GPU sees
    for kind_name, kind in O.SCORE_KINDS.items():
        s, eq, ek = P.block_energy(qd, kd, kind=kind, return_parts=True)
        so, eqo, eko = O.block_energy(q64, k64, kind=kind_name)
        for got, exp in ((s, so), (eq, eqo), (ek, eko)):
            got = got.cpu().numpy().astype(np.float64)
            assert np.all(np.abs(got - exp) <= 1e-5 * np.abs(exp) + 1e-30), kind_name


def test_block_energy_interleaved_pairing(P):
    scales = W.block_scales(8, 2, 64)
    q = W.pre_rope_gaussian(8, 1, 64, 4, 128, scales, pairing=W.synth.PAIR_INTERLEAVED)
    k = W.pre_rope_gaussian(8, 2, 200, 2, 128, scales, pairing=W.synth.PAIR_INTERLEAVED)
    qd, kd = _cuda(q, torch.float32), _cuda(k, torch.float32)
    s = P.block_energy(qd, kd, pairing=P.PAIR_INTERLEAVED).cpu().numpy()
    so, _, _ = O.block_energy(qd.double().cpu().numpy(), kd.double().cpu().numpy(), pairing=O.PAIR_INTERLEAVED)
    assert np.allclose(s, so, rtol=1e-5, atol=0)


# ----------------------------------------------------------------------------- a2 allocation
@pytest.mark.parametrize("bmin,bmax,bbar", [(0, 8, 3), (1, 8, 3), (1, 8, 2), (0, 4, 2), (2, 2, 2)])
def test_allocate_device_bit_exact(P, bmin, bmax, bbar):
    rng = np.random.default_rng(5)
    s = np.exp(rng.uniform(np.log(1e-2), np.log(10), size=(37, 64))).astype(np.float32)
    s[3, :] = 1.0                       # all ties
    s[4, ::2] = 0.0                     # zero scores (Q5)
    s[5, 10] = s[5, 20]                 # an exact tie (Q4)
    got = P.allocate(torch.from_numpy(s).cuda(), bbar * 64, bmin, bmax).cpu().numpy()
    for h in range(s.shape[0]):
        exp = O.allocate(s[h].astype(np.float64), bbar * 64, bmin, bmax)
        assert np.array_equal(got[h], exp), h
    assert np.all(got.sum(axis=1) == bbar * 64)


def test_energy_then_allocate_chain(P):
    p = H.make_problem(11, 600, 8, 2, 3, 3, 1, 8)
    scales = W.block_scales(11, 2, 64)
    qc = _cuda(W.pre_rope_gaussian(11, 4, 256, 8, 128, scales), torch.float32)
    kc = _cuda(W.pre_rope_gaussian(11, 1, 600, 2, 128, scales), torch.float32)
    s_gpu = P.block_energy(qc, kc)
    bits = P.allocate(s_gpu, 3 * 64, 1, 8).cpu().numpy()
    s_np = s_gpu.cpu().numpy().astype(np.float64)
    for h in range(2):
        assert np.array_equal(bits[h], O.allocate(s_np[h], 192, 1, 8))       # same scores -> same bits
        s_or, _, _ = O.block_energy(qc.double().cpu().numpy(), kc.double().cpu().numpy())
        J_gpu = O.objective(s_or[h], bits[h])
        J_opt = O.objective(s_or[h], O.allocate(s_or[h], 192, 1, 8))
        assert J_gpu <= J_opt * (1 + 1e-6)


# ----------------------------------------------------------------------------- a4 quantize-on-append
def _append_and_compare(P, p, tab, chunks, max_tokens, kv_dtype):
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, p.b_v, p.rot)
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    tdt = torch.float32 if kv_dtype == "f32" else torch.bfloat16
    t = 0
    for n in chunks:
        k = _cuda(p.k_post[None, t:t + n], tdt)
        v = _cuda(p.v[None, t:t + n], tdt)
        P.quantize_append(lay, 0, cache, k, v, seq, max_tokens)
        t += n
    assert int(seq.item()) == t
    heads = H.oracle_heads(p, tab, 0, t)
    host = cache.cpu().numpy()
    n_cap = (max_tokens + 127) // 128
    for h in range(p.Hkv):
        stride = lay.tile_stride(0, h)
        assert stride == O.tile_geometry(heads[h].groups, p.d_h, p.b_v)["stride"]
        assert abs(lay.token_bytes(0, h) - O.token_bytes(heads[h].groups, p.d_h, p.b_v)) < 1e-12
        off = lay.region_offset(0, 0, h, 1, max_tokens)
        exp = np.zeros(n_cap * stride, dtype=np.uint8)
        O.pack_region(heads[h], p.d_h, exp)
        got = host[off:off + n_cap * stride]
        if not np.array_equal(got, exp):
            # help debugging: compare logical content
            u = O.unpack_region(got, heads[h].groups, p.d_h, p.b_v, t)
            bad_k = int(np.count_nonzero(u.kidx != heads[h].kidx))
            bad_v = int(np.count_nonzero(u.vidx != heads[h].vidx))
            bad_n = int(np.count_nonzero(u.knorm != heads[h].knorm)) + int(np.count_nonzero(u.vnorm != heads[h].vnorm))
            raise AssertionError(f"head {h}: packed bytes differ (k codes {bad_k}, v codes {bad_v}, norms {bad_n})")
    return lay, cache, seq, heads


@pytest.mark.parametrize("kv_dtype", ["f32", "bf16"])
def test_append_bit_exact_bulk_and_ragged(P, tab128, kv_dtype):
    p = H.make_problem(21, 333, 8, 2, 3, 3, 0, 8, kv_dtype=kv_dtype)
    _append_and_compare(P, p, tab128, [333], 512, kv_dtype)


def test_append_bit_exact_incremental(P, tab128):
    """prefill chunk, then single-token decode appends crossing a tile boundary == one bulk pack"""
    p = H.make_problem(22, 140, 4, 1, 2, 2, 1, 8)
    _append_and_compare(P, p, tab128, [100, 27, 1, 1, 1, 10], 256, "f32")


def test_append_wide_and_uniform_allocations(P, tab128):
    p = H.make_problem(23, 150, 2, 2, 3, 4, 1, 8)
    p.bits[0, :] = 8                               # every block at the widest code
    p.bits[1, :] = 3                               # uniform TQ-MSE = one group
    _append_and_compare(P, p, tab128, [150], 256, "f32")


# ----------------------------------------------------------------------------- a5 + a6 decode attention
def _attention_case(P, tab, seed, T, Hq, Hkv, b_k, b_v, bmin, bmax, max_tokens=None, base=1e4):
    p = H.make_problem(seed, T, Hq, Hkv, b_k, b_v, bmin, bmax, rope_base=base)
    max_tokens = max_tokens or ((T + 127) // 128 * 128)
    lay, cache, seq, heads = _append_and_compare(P, p, tab, [T], max_tokens, "f32")
    scale = 1.0 / math.sqrt(p.d_h)
    q = _cuda(p.q_post[None], torch.bfloat16)
    ws = lay.new_workspace(1)
    out = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, ws)
    torch.cuda.synchronize()
    exp, rv = H.oracle_attention(p, heads, tab, scale)
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    err = np.array([np.max(np.abs(got[a] - exp[a])) / rv[a // G] for a in range(Hq)])
    return err


def test_attention_cfg0_like(P, tab128):
    """BASELINE.json configs[0]: 1 KV head, 1 query head, T = 4096, K3 (0..8) V3."""
    err = _attention_case(P, tab128, 0, 4096, 1, 1, 3, 3, 0, 8)
    assert err.max() <= 2e-3, err


@pytest.mark.parametrize("T", [1, 7, 128, 129, 1000])
def test_attention_gqa8_ragged(P, tab128, T):
    err = _attention_case(P, tab128, 30 + T, T, 16, 2, 3, 3, 1, 8, base=1e6)
    assert err.max() <= 2e-3, err


def test_attention_gqa4_k2v2(P, tab128):
    err = _attention_case(P, tab128, 41, 700, 8, 2, 2, 2, 1, 8, base=5e5)
    assert err.max() <= 2e-3, err


def test_attention_capacity_larger_than_length(P, tab128):
    err = _attention_case(P, tab128, 42, 300, 8, 1, 3, 2, 1, 8, max_tokens=2048)
    assert err.max() <= 2e-3, err


def test_attention_empty_sequence_is_zero(P):
    p = H.make_problem(43, 4, 8, 1, 3, 3, 1, 8)
    lay = P.Layout(p.bits[None], 8, 128, 3, p.rot)
    cache = lay.new_cache(1, 128)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    q = _cuda(p.q_post[None], torch.bfloat16)
    out = P.decode_attention(lay, 0, cache, q, seq, 128, 0.1, lay.new_workspace(1))
    assert torch.all(out == 0)

"""-m gpu: the BGTQ-v2 path (row-order layout, tcgen05 decode kernel) against the fp64 oracle.

Same bars as test_gpu_parity.py: packed bytes bit-exact against the oracle's v2 packer, attention max-abs / R_V <= 2e-3.
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


def _append_and_compare(P, p, tab, chunks, max_tokens, kv_dtype="f32"):
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, p.b_v, p.rot, fmt=P.FORMAT_V2)
    assert lay.fmt == 2
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    tdt = torch.float32 if kv_dtype == "f32" else torch.bfloat16
    t = 0
    for n in chunks:
        P.quantize_append(lay, 0, cache, _cuda(p.k_post[None, t:t + n], tdt), _cuda(p.v[None, t:t + n], tdt), seq, max_tokens)
        t += n
    assert int(seq.item()) == t
    heads = H.oracle_heads(p, tab, 0, t)
    host = cache.cpu().numpy()
    n_cap = (max_tokens + 127) // 128
    for h in range(p.Hkv):
        stride = lay.tile_stride(0, h)
        assert stride == O.tile_geometry(heads[h].groups, p.d_h, p.b_v, version=2)["stride"]
        off = lay.region_offset(0, 0, h, 1, max_tokens)
        exp = np.zeros(n_cap * stride, dtype=np.uint8)
        O.pack_region(heads[h], p.d_h, exp, version=2)
        got = host[off:off + n_cap * stride]
        if not np.array_equal(got, exp):
            u = O.unpack_region(got, heads[h].groups, p.d_h, p.b_v, t, version=2)
            bad_k = int(np.count_nonzero(u.kidx != heads[h].kidx))
            bad_v = int(np.count_nonzero(u.vidx != heads[h].vidx))
            bad_n = int(np.count_nonzero(u.knorm != heads[h].knorm)) + int(np.count_nonzero(u.vnorm != heads[h].vnorm))
            raise AssertionError(f"head {h}: packed bytes differ (k codes {bad_k}, v codes {bad_v}, norms {bad_n}, "
                                 f"bytes {int(np.count_nonzero(got != exp))})")
    return lay, cache, seq, heads


@pytest.mark.parametrize("kv_dtype", ["f32", "bf16"])
def test_v2_append_bit_exact_bulk_and_ragged(P, tab128, kv_dtype):
    p = H.make_problem(21, 333, 8, 2, 3, 3, 0, 8, kv_dtype=kv_dtype)
    _append_and_compare(P, p, tab128, [333], 512, kv_dtype)


def test_v2_append_bit_exact_incremental(P, tab128):
    p = H.make_problem(22, 140, 4, 1, 2, 2, 1, 8)
    _append_and_compare(P, p, tab128, [100, 27, 1, 1, 1, 10], 256)


def test_v2_append_wide_and_uniform_allocations(P, tab128):
    p = H.make_problem(23, 150, 2, 2, 3, 4, 1, 8)
    p.bits[0, :] = 8
    p.bits[1, :] = 3
    _append_and_compare(P, p, tab128, [150], 256)


@pytest.mark.parametrize("seed", range(4))
def test_v2_append_random_width_mixes(P, tab128, seed):
    rng = np.random.default_rng(900 + seed)
    p = H.make_problem(24 + seed, 200, 4, 2, 3, int(rng.integers(1, 9)), 1, 8)
    p.bits[:] = rng.integers(0, 9, p.bits.shape)
    _append_and_compare(P, p, tab128, [130, 70], 256)


def _attention_case(P, tab, seed, T, Hq, Hkv, b_k, b_v, bmin, bmax, max_tokens=None, base=1e4, bits=None):
    p = H.make_problem(seed, T, Hq, Hkv, b_k, b_v, bmin, bmax, rope_base=base)
    if bits is not None:
        p.bits[:] = bits
    max_tokens = max_tokens or ((T + 127) // 128 * 128)
    lay, cache, seq, heads = _append_and_compare(P, p, tab, [T], max_tokens)
    scale = 1.0 / math.sqrt(p.d_h)
    q = _cuda(p.q_post[None], torch.bfloat16)
    out = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    exp, rv = H.oracle_attention(p, heads, tab, scale)
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    return np.array([np.max(np.abs(got[a] - exp[a])) / rv[a // G] for a in range(Hq)])


@pytest.mark.parametrize("T", [1, 7, 128, 129, 1000])
def test_v2_attention_gqa8_ragged(P, tab128, T):
    err = _attention_case(P, tab128, 30 + T, T, 16, 2, 3, 3, 1, 8, base=1e6)
    assert err.max() <= 2e-3, err


def test_v2_attention_cfg0_like(P, tab128):
    err = _attention_case(P, tab128, 0, 4096, 1, 1, 3, 3, 0, 8)
    assert err.max() <= 2e-3, err


def test_v2_attention_gqa4_k2v2(P, tab128):
    err = _attention_case(P, tab128, 41, 700, 8, 2, 2, 2, 1, 8, base=5e5)
    assert err.max() <= 2e-3, err


@pytest.mark.parametrize("bk,bv", [(1, 1), (2, 1), (4, 4), (5, 5), (6, 3), (3, 8)])
def test_v2_attention_widths(P, tab128, bk, bv):
    err = _attention_case(P, tab128, 50 + bk, 300, 8, 2, bk, bv, 1, 8, bits=bk)
    assert err.max() <= 2e-3, err


def test_v2_attention_empty_sequence_is_zero(P):
    p = H.make_problem(43, 4, 8, 1, 3, 3, 1, 8)
    lay = P.Layout(p.bits[None], 8, 128, 3, p.rot, fmt=P.FORMAT_V2)
    cache = lay.new_cache(1, 128)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    out = P.decode_attention(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, 128, 0.1, lay.new_workspace(1))
    assert torch.all(out == 0)

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


# ----------------------------------------------------------------------------- batched layers / sequences
def test_layers_batched_and_ragged_batch(P, tab128):
    """bgtq_quantize_append_layers + bgtq_decode_attention_layers over 3 layers x 2 sequences of different
    lengths (one launch) == per-layer calls == oracle, with a different allocation per (layer, head)."""
    Lyr, B, Hq, Hkv, d = 3, 2, 8, 2, 128
    lens = [389, 150]
    probs = [[H.make_problem(60 + 10 * l + b, lens[b], Hq, Hkv, 3, 3, 1, 8, rope_base=1e6) for b in range(B)] for l in range(Lyr)]
    for l in range(Lyr):                       # one allocation per layer (from sequence 0's statistics)
        for b in range(B):
            probs[l][b].bits = probs[l][0].bits
    bits = np.stack([probs[l][0].bits for l in range(Lyr)])
    lay = P.Layout(bits, Hq, d, 3, probs[0][0].rot)
    max_tokens = 512
    cache = lay.new_cache(B, max_tokens)
    seq = torch.zeros(B, dtype=torch.int32, device="cuda")
    # first 150 tokens of both sequences in one layers-batched call, then the rest of sequence 0 per layer
    k0 = np.stack([np.stack([probs[l][b].k_post[:150] for b in range(B)]) for l in range(Lyr)])
    v0 = np.stack([np.stack([probs[l][b].v[:150] for b in range(B)]) for l in range(Lyr)])
    P.quantize_append(lay, 0, cache, _cuda(k0, torch.float32), _cuda(v0, torch.float32), seq, max_tokens, n_layers=Lyr)
    assert seq.tolist() == [150, 150]
    rest = lens[0] - 150
    for l in range(Lyr):
        kk = np.zeros((B, rest, Hkv, d)); vv = np.zeros((B, rest, Hkv, d))
        kk[0] = probs[l][0].k_post[150:]; vv[0] = probs[l][0].v[150:]
        seq_l = torch.tensor([150, max_tokens], dtype=torch.int32, device="cuda")   # sequence 1 is "full": nothing appended
        P.quantize_append(lay, l, cache, _cuda(kk, torch.float32), _cuda(vv, torch.float32), seq_l, max_tokens,
                          advance_seq_len=False)
    seq = torch.tensor(lens, dtype=torch.int32, device="cuda")
    host = cache.cpu().numpy()
    heads = [[H.oracle_heads(probs[l][b], tab128) for b in range(B)] for l in range(Lyr)]
    n_cap = max_tokens // 128
    for l in range(Lyr):
        for b in range(B):
            for h in range(Hkv):
                stride = lay.tile_stride(l, h)
                off = lay.region_offset(l, b, h, B, max_tokens)
                exp = np.zeros(n_cap * stride, dtype=np.uint8)
                O.pack_region(heads[l][b][h], d, exp)
                assert np.array_equal(host[off:off + n_cap * stride], exp), (l, b, h)
    scale = 1.0 / math.sqrt(d)
    q = np.stack([np.stack([probs[l][b].q_post for b in range(B)]) for l in range(Lyr)])       # [Lyr,B,Hq,d]
    qd = _cuda(q, torch.bfloat16)
    out_b = P.decode_attention(lay, 0, cache, qd, seq, max_tokens, scale, lay.new_workspace(B, Lyr), n_layers=Lyr)
    ws1 = lay.new_workspace(B, 1)
    out_l = torch.stack([P.decode_attention(lay, l, cache, qd[l].contiguous(), seq, max_tokens, scale, ws1) for l in range(Lyr)])
    torch.cuda.synchronize()
    for l in range(Lyr):
        for b in range(B):
            exp, rv = H.oracle_attention(probs[l][b], heads[l][b], tab128, scale)
            for name, out in (("batched", out_b), ("per-layer", out_l)):
                got = out[l, b].double().cpu().numpy()
                err = max(np.max(np.abs(got[a] - exp[a])) / rv[a // (Hq // Hkv)] for a in range(Hq))
                assert err <= 2e-3, (name, l, b, err)


def test_gpu_generator_rope_matches_oracle(P):
    """workloads/gpu_synth.py shapes inputs only, but its RoPE is still checked against the oracle's."""
    from workloads import gpu_synth as GS
    x = torch.randn((50, 3, 128), dtype=torch.float64, device="cuda")
    pos = torch.arange(1000, 1050, dtype=torch.float64, device="cuda")
    got = GS.rope_half(x, pos, 1e6).cpu().numpy()
    exp = O.rope(x.cpu().numpy(), pos.cpu().numpy(), 1e6)
    assert np.max(np.abs(got - exp)) < 1e-9


@pytest.mark.timeout(900)
def test_full_size_128k_sampled_head(P, tab128):
    """BASELINE.json configs[2] at full context (131,072 tokens) in the launch configuration bench.py times
    (layers batched in one launch): the packed region and the attention output of one sampled
    (layer, KV head) are checked against the oracle run on the SAME input tensors (copied to the host)."""
    from workloads import gpu_synth as GS
    shp = W.CONFIGS[2]
    Lyr, T, d, Hq, Hkv = 2, 131072, shp.d_h, shp.n_q_heads, shp.n_kv_heads
    kv, scores, scales_all = [], [], []
    for l in range(Lyr):
        ks, vs = [], []
        for c0 in range(0, T, 32768):
            k, v, scales = GS.layer_kv(shp.seed0 + l, 32768, Hkv, d, shp.rope_base, "cuda", t0=c0, chunk_tag=c0 // 32768)
            ks.append(k); vs.append(v)
        k, v = torch.cat(ks), torch.cat(vs)
        qcal = GS.layer_queries(shp.seed0 + l, shp.n_cal, Hq, scales, d, shp.rope_base, 0, "cuda", tag=4)
        scores.append(P.block_energy(qcal, k))
        kv.append((k, v)); scales_all.append(scales)
    bits = P.allocate(torch.cat(scores), shp.b_k * 64, shp.b_min, shp.b_max).cpu().numpy().reshape(Lyr, Hkv, 64)
    lay = P.Layout(bits, Hq, d, shp.b_v, tab128.rot)
    max_tokens = T
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    for l in range(Lyr):
        seq.zero_()
        P.quantize_append(lay, l, cache, kv[l][0][None].contiguous(), kv[l][1][None].contiguous(), seq, max_tokens)
    q = torch.stack([GS.layer_queries(shp.seed0 + l, 1, Hq, scales_all[l], d, shp.rope_base, T, "cuda", tag=3,
                                      dtype=torch.bfloat16) for l in range(Lyr)])
    scale = 1.0 / math.sqrt(d)
    out = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, lay.new_workspace(1, Lyr), n_layers=Lyr)
    torch.cuda.synchronize()
    l, h = 1, 1                                                    # the sampled (layer, KV head)
    k_h = kv[l][0][:, h].double().cpu().numpy()
    v_h = kv[l][1][:, h].double().cpu().numpy()
    head = O.quantize_head(k_h, v_h, bits[l, h], shp.b_v, tab128)
    stride = lay.tile_stride(l, h)
    off = lay.region_offset(l, 0, h, 1, max_tokens)
    exp = np.zeros((T // 128) * stride, dtype=np.uint8)
    O.pack_region(head, d, exp)
    got = cache[off:off + exp.size].cpu().numpy()
    assert np.array_equal(got, exp), "packed region differs at full size"
    G = Hq // Hkv
    q_h = q[l, 0, h * G:(h + 1) * G].double().cpu().numpy()
    ref = O.decode_attention_head(q_h, head, tab128, d, scale)
    _, V = O.dequantize_head(head, tab128, d)
    rv = math.sqrt(np.mean(np.sum(V * V, axis=1)))
    err = np.max(np.abs(out[l, 0, h * G:(h + 1) * G].double().cpu().numpy() - ref)) / rv
    assert err <= 2e-3, err
    # the protected regime (fp16 sink-4 / recent-128 windows) on the same cache, same launch configuration
    ns, nr = 4, 128
    win_k, win_v = P.new_windows(lay, 1, ns, nr)
    zero = torch.zeros(1, dtype=torch.int32, device="cuda")
    for ll in range(Lyr):
        P.window_append(lay, ll, kv[ll][0][None].contiguous(), kv[ll][1][None].contiguous(), zero, win_k, win_v, ns, nr)
    outp = P.decode_attention_protected(lay, 0, cache, q, seq, max_tokens, scale, win_k, win_v, ns, nr,
                                        lay.new_workspace(1, Lyr), n_layers=Lyr)
    torch.cuda.synchronize()
    refp = O.decode_attention_protected_head(q_h, head, tab128, d, scale, k_h.astype(np.float16).astype(np.float64),
                                             v_h.astype(np.float16).astype(np.float64), ns, nr)
    errp = np.max(np.abs(outp[l, 0, h * G:(h + 1) * G].double().cpu().numpy() - refp)) / rv
    assert errp <= 2e-3, errp


@pytest.mark.timeout(900)
def test_full_size_cfg3_batch4_sampled(P, tab128):
    """BASELINE.json configs[3] at full size (Llama-3.1-8B layer shape: 32 q / 8 kv heads, K2V2, 131,072 tokens, batch 4 of
    independent seeds; here with ragged lengths so the balanced split crosses sequence boundaries): the packed region and
    the attention output of two sampled (sequence, KV head) pairs against the oracle on the SAME input tensors."""
    from workloads import gpu_synth as GS
    shp = W.CONFIGS[3]
    B, T, d, Hq, Hkv = 4, 131072, shp.d_h, shp.n_q_heads, shp.n_kv_heads
    lens = [T, T - 77, T // 2 + 5, T]
    _, _, scales = GS.layer_kv(shp.seed0, 8, Hkv, d, shp.rope_base, "cuda")
    qcal = GS.layer_queries(shp.seed0, shp.n_cal, Hq, scales, d, shp.rope_base, 0, "cuda", tag=4)
    kcal, _, _ = GS.layer_kv(shp.seed0, 32768, Hkv, d, shp.rope_base, "cuda", chunk_tag=99)
    bits = P.allocate(P.block_energy(qcal, kcal), shp.b_k * 64, shp.b_min, shp.b_max).cpu().numpy().reshape(1, Hkv, 64)
    del kcal
    lay = P.Layout(bits, Hq, d, shp.b_v, tab128.rot)
    cache = lay.new_cache(B, T)
    seq = torch.zeros(B, dtype=torch.int32, device="cuda")
    sampled = {(1, 5): None, (2, 0): None}
    for c0 in range(0, T, 32768):                 # every sequence gets its own draw; all are filled to T, seq_len is set after
        k = torch.stack([GS.layer_kv(shp.seed0 + 100 * b, 32768, Hkv, d, shp.rope_base, "cuda", t0=c0, chunk_tag=c0 // 32768)[0] for b in range(B)])
        v = torch.stack([GS.layer_kv(shp.seed0 + 100 * b, 32768, Hkv, d, shp.rope_base, "cuda", t0=c0, chunk_tag=c0 // 32768)[1] for b in range(B)])
        P.quantize_append(lay, 0, cache, k, v, seq, T)
        for (b, h) in sampled:
            kh, vh = k[b, :, h].double().cpu().numpy(), v[b, :, h].double().cpu().numpy()
            sampled[(b, h)] = (kh, vh) if sampled[(b, h)] is None else (np.concatenate([sampled[(b, h)][0], kh]),
                                                                         np.concatenate([sampled[(b, h)][1], vh]))
        del k, v
    assert seq.tolist() == [T] * B
    seq = torch.tensor(lens, dtype=torch.int32, device="cuda")
    q = torch.stack([GS.layer_queries(shp.seed0 + 100 * b, 1, Hq, scales, d, shp.rope_base, lens[b], "cuda", tag=3,
                                      dtype=torch.bfloat16)[0] for b in range(B)])
    scale = 1.0 / math.sqrt(d)
    out = P.decode_attention(lay, 0, cache, q, seq, T, scale, lay.new_workspace(B, 1))
    torch.cuda.synchronize()
    G = Hq // Hkv
    for (b, h), (kh, vh) in sampled.items():
        n = lens[b]
        head = O.quantize_head(kh[:n], vh[:n], bits[0, h], shp.b_v, tab128)
        stride = lay.tile_stride(0, h)
        off = lay.region_offset(0, b, h, B, T)
        n_full = n // 128                          # whole tiles of the attended prefix (the cache holds all T tokens)
        exp = np.zeros(((n + 127) // 128) * stride, dtype=np.uint8)
        O.pack_region(head, d, exp)
        got = cache[off:off + n_full * stride].cpu().numpy()
        assert np.array_equal(got, exp[:n_full * stride]), ("packed region differs at full size", b, h)
        q_h = q[b, h * G:(h + 1) * G].double().cpu().numpy()
        ref = O.decode_attention_head(q_h, head, tab128, d, scale)
        _, V = O.dequantize_head(head, tab128, d)
        rv = math.sqrt(np.mean(np.sum(V * V, axis=1)))
        err = np.max(np.abs(out[b, h * G:(h + 1) * G].double().cpu().numpy() - ref)) / rv
        assert err <= 2e-3, (b, h, err)


# ----------------------------------------------------------------------------- comparison path (not the method)
@pytest.mark.parametrize("lens", [[1], [300, 77], [1000, 129, 0]])
def test_fp16_comparison_kernel_vs_plain_attention(P, lens):
    """bgtq_fp16_decode_attention against the textbook definition evaluated in fp64 on the same fp16 cache."""
    torch.manual_seed(3)
    Lyr, B, Hq, Hkv, d, cap = 2, len(lens), 16, 2, 128, 1024
    k = torch.randn(Lyr, B, Hkv, cap, d, device="cuda").to(torch.float16)
    v = torch.randn(Lyr, B, Hkv, cap, d, device="cuda").to(torch.float16)
    q = torch.randn(Lyr, B, Hq, d, device="cuda").to(torch.bfloat16)
    seq = torch.tensor(lens, dtype=torch.int32, device="cuda")
    scale = 1.0 / math.sqrt(d)
    out = P.fp16_decode_attention(k, v, q, seq, scale).double().cpu().numpy()
    G = Hq // Hkv
    for l in range(Lyr):
        for b in range(B):
            T = lens[b]
            for a in range(Hq):
                if T == 0:
                    assert np.all(out[l, b, a] == 0)
                    continue
                K = k[l, b, a // G, :T].double().cpu().numpy()
                V = v[l, b, a // G, :T].double().cpu().numpy()
                ref = O.attention(q[l, b, a].double().cpu().numpy(), K, V, scale)
                assert np.max(np.abs(out[l, b, a] - ref)) <= 2e-3 * math.sqrt(d), (l, b, a)


@pytest.mark.timeout(600)
def test_cfg1_append_then_attend(P, tab128):
    """BASELINE.json configs[1]: Qwen2.5-3B layer, 32,768 cached tokens; per step one token goes through
    bgtq_quantize_append and the query attends over T+1 tokens (Q13).  One KV head is checked against the oracle."""
    from workloads import gpu_synth as GS
    shp = W.CONFIGS[1]
    T, d, Hq, Hkv = shp.contexts[0], shp.d_h, shp.n_q_heads, shp.n_kv_heads
    k, v, scales = GS.layer_kv(shp.seed0, T + 1, Hkv, d, shp.rope_base, "cuda")
    qcal = GS.layer_queries(shp.seed0, shp.n_cal, Hq, scales, d, shp.rope_base, 0, "cuda", tag=4)
    bits = P.allocate(P.block_energy(qcal, k[:T].contiguous()), shp.b_k * 64, shp.b_min, shp.b_max).cpu().numpy()
    lay = P.Layout(bits[None], Hq, d, shp.b_v, tab128.rot)
    max_tokens = T + 128
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    P.quantize_append(lay, 0, cache, k[None, :T].contiguous(), v[None, :T].contiguous(), seq, max_tokens)
    P.quantize_append(lay, 0, cache, k[None, T:].contiguous(), v[None, T:].contiguous(), seq, max_tokens)   # the decode-step append
    assert int(seq.item()) == T + 1
    q = GS.layer_queries(shp.seed0, 1, Hq, scales, d, shp.rope_base, T, "cuda", tag=3, dtype=torch.bfloat16)
    scale = 1.0 / math.sqrt(d)
    out = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    h = 1
    head = O.quantize_head(k[:, h].double().cpu().numpy(), v[:, h].double().cpu().numpy(), bits[h], shp.b_v, tab128)
    stride = lay.tile_stride(0, h)
    off = lay.region_offset(0, 0, h, 1, max_tokens)
    exp = np.zeros(((max_tokens + 127) // 128) * stride, dtype=np.uint8)
    O.pack_region(head, d, exp)
    assert np.array_equal(cache[off:off + exp.size].cpu().numpy(), exp)
    G = Hq // Hkv
    ref = O.decode_attention_head(q[0, h * G:(h + 1) * G].double().cpu().numpy(), head, tab128, d, scale)
    _, V = O.dequantize_head(head, tab128, d)
    rv = math.sqrt(np.mean(np.sum(V * V, axis=1)))
    err = np.max(np.abs(out[0, h * G:(h + 1) * G].double().cpu().numpy() - ref)) / rv
    assert err <= 2e-3, err


# ----------------------------------------------------------------------------- NEXT #1: prefill attention
@pytest.mark.parametrize("T,n_q,Hq,Hkv,bk,bv", [(40, 40, 8, 1, 3, 3), (300, 77, 16, 2, 3, 3), (333, 333, 8, 2, 2, 2),
                                              (260, 5, 4, 1, 3, 4), (1100, 190, 8, 2, 3, 3), (515, 130, 2, 2, 4, 2),
                                              (200, 9, 8, 1, 6, 6)])
def test_prefill_attention_vs_oracle(P, tab128, T, n_q, Hq, Hkv, bk, bv):
    """bgtq_prefill_attention: causal attention of the last n_q tokens' queries over the packed cache
    against the oracle's plain definition, row by row."""
    p = H.make_problem(70 + T, T, Hq, Hkv, bk, bv, 1, 8, rope_base=1e6)
    lay, cache, seq, heads = _append_and_compare(P, p, tab128, [T], ((T + 127) // 128) * 128, "f32")
    max_tokens = ((T + 127) // 128) * 128
    rng = np.random.default_rng(T)
    scales = W.block_scales(70 + T, Hkv, 64)
    q_pre = W.pre_rope_gaussian(70 + T, 9, n_q, Hq, 128, scales)
    q_post = W.round_to_bf16(O.rope(q_pre, np.arange(T - n_q, T, dtype=np.float64), 1e6)).astype(np.float64)   # [n_q,Hq,d]
    scale = 1.0 / math.sqrt(128)
    out = P.prefill_attention(lay, 0, cache, _cuda(q_post[None], torch.bfloat16), seq, max_tokens, scale)
    torch.cuda.synchronize()
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    for h in range(Hkv):
        ref = O.prefill_attention_head(q_post[:, h * G:(h + 1) * G], heads[h], tab128, 128, scale, T - n_q)
        _, V = O.dequantize_head(heads[h], tab128, 128)
        rv = math.sqrt(np.mean(np.sum(V * V, axis=1)))
        err = np.max(np.abs(got[:, h * G:(h + 1) * G] - ref)) / rv
        assert err <= 2e-3, (h, err)


# ----------------------------------------------------------------------------- randomised allocations
@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_random_allocations_append_and_attention(P, tab128, seed):
    """Arbitrary width patterns (not only greedy outputs): every width 0..8 present, tiny groups of one block,
    a single 8-bit group, many zero-width blocks ... packed bytes bit-exact and attention within tolerance."""
    rng = np.random.default_rng(1000 + seed)
    Hq, Hkv, T = 8, 2, 200 + 37 * seed
    p = H.make_problem(80 + seed, T, Hq, Hkv, 3, 1 + (seed % 8), 1, 8, rope_base=1e4)
    pats = [rng.integers(0, 9, size=64), rng.integers(1, 9, size=64)]
    if seed == 1:
        pats[0] = np.array([0] * 60 + [8, 7, 6, 5])               # almost everything dropped, tiny wide groups
    if seed == 2:
        pats[1] = np.full(64, 8)
    if seed == 3:
        pats[0] = np.array(list(range(1, 9)) * 8)                  # 8 groups of 16 coordinates
    if seed == 4:
        pats[1] = np.array([1] * 63 + [4])                         # a one-block group
    p.bits = np.stack(pats).astype(np.uint8)
    max_tokens = ((T + 127) // 128) * 128
    lay, cache, seq, heads = _append_and_compare(P, p, tab128, [T - 3, 3], max_tokens, "f32")
    scale = 1.0 / math.sqrt(p.d_h)
    out = P.decode_attention(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, max_tokens, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    exp, rv = H.oracle_attention(p, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    err = max(np.max(np.abs(got[a] - exp[a])) / max(rv[a // G], 1e-30) for a in range(Hq))
    assert err <= 2e-3, err


@pytest.mark.parametrize("Hq,Hkv,bk,bv,T", [(4, 2, 1, 1, 260), (6, 2, 4, 4, 200), (5, 1, 2, 8, 130), (2, 2, 6, 5, 140), (16, 2, 3, 2, 515)])
def test_attention_more_shapes_and_budgets(P, tab128, Hq, Hkv, bk, bv, T):
    """GQA groups 1, 2, 3, 5, 8 and budgets K1V1 .. K6V5 / V8 (greedy allocation at that budget)."""
    err = _attention_case(P, tab128, 90 + T, T, Hq, Hkv, bk, bv, 1, 8, base=5e5)
    assert err.max() <= 2e-3, err


def test_paged_cache_append_and_attention(P, tab128):
    """bgtq_quantize_append_paged + bgtq_decode_attention_paged.  A paged cache holds the same
    tiles as the contiguous one at addresses given by a page table, so every page must equal the oracle's packed
    tile byte for byte and attention must match the oracle; pages are scattered, shared across 2 layers, and the
    sequences grow in uneven chunks (a page boundary inside a chunk, an incremental single token)."""
    Lyr, B, Hq, Hkv, d = 2, 3, 8, 2, 128
    lens = [389, 150, 0]
    probs = [[H.make_problem(160 + 10 * l + b, max(lens[b], 1), Hq, Hkv, 3, 3, 1, 8, rope_base=1e6) for b in range(B)]
             for l in range(Lyr)]
    for l in range(Lyr):
        for b in range(B):
            probs[l][b].bits = probs[l][0].bits
    bits = np.stack([probs[l][0].bits for l in range(Lyr)])
    lay = P.Layout(bits, Hq, d, 3, probs[0][0].rot)
    table_stride, n_pages = 5, 23
    rng = np.random.default_rng(7)
    perm = rng.permutation(n_pages)[:B * table_stride].astype(np.int32).reshape(B, table_stride)   # distinct pages
    table = torch.from_numpy(perm).cuda()
    cache = torch.full((lay.paged_cache_bytes(n_pages),), 0xAB, dtype=torch.uint8, device="cuda")   # pages start dirty
    assert lay.paged_cache_bytes(n_pages) == n_pages * sum(lay.tile_stride(l, h) for l in range(Lyr) for h in range(Hkv))
    seq = torch.zeros(B, dtype=torch.int32, device="cuda")
    done = [0] * B
    for chunk in (100, 1, 49, 239):                       # sequence 1 stops at 150, sequence 2 never grows
        n_app = [min(chunk, lens[b] - done[b]) for b in range(B)]
        kk = np.zeros((Lyr, B, chunk, Hkv, d)); vv = np.zeros((Lyr, B, chunk, Hkv, d))
        for l in range(Lyr):
            for b in range(B):
                kk[l, b, :n_app[b]] = probs[l][b].k_post[done[b]:done[b] + n_app[b]]
                vv[l, b, :n_app[b]] = probs[l][b].v[done[b]:done[b] + n_app[b]]
        assert all(n in (0, chunk) for n in n_app)
        # one call for every layer and sequence; a sequence that is done is presented as full, so nothing is appended
        sq = torch.tensor([done[b] if n_app[b] else table_stride * 128 for b in range(B)], dtype=torch.int32, device="cuda")
        P.quantize_append_paged(lay, 0, cache, _cuda(kk, torch.float32), _cuda(vv, torch.float32), sq, table, n_pages,
                                advance_seq_len=(chunk == 100), n_layers=Lyr)
        if chunk == 100:                                  # the library advanced the lengths (and saturated the full one)
            assert sq.tolist() == [100, 100, table_stride * 128]
        seq = torch.tensor([done[b] + n_app[b] for b in range(B)], dtype=torch.int32, device="cuda")
        done = [done[b] + n_app[b] for b in range(B)]
        assert seq.tolist() == done
    assert done == lens
    host = cache.cpu().numpy()
    heads = [[H.oracle_heads(probs[l][b], tab128) if lens[b] else None for b in range(B)] for l in range(Lyr)]
    touched = set()
    for l in range(Lyr):
        for b in range(B):
            if not lens[b]:
                continue
            n_t = (lens[b] + 127) // 128
            for h in range(Hkv):
                stride = lay.tile_stride(l, h)
                pool = lay.paged_pool_offset(l, h, n_pages)
                exp = np.zeros(n_t * stride, dtype=np.uint8)
                O.pack_region(heads[l][b][h], d, exp)
                for j in range(n_t):
                    pg = int(perm[b, j])
                    touched.add((l, h, pg))
                    got = host[pool + pg * stride: pool + (pg + 1) * stride]
                    assert np.array_equal(got, exp[j * stride:(j + 1) * stride]), (l, b, h, j)
    for l in range(Lyr):                                  # pages no live tile maps to were not written
        for h in range(Hkv):
            stride, pool = lay.tile_stride(l, h), lay.paged_pool_offset(l, h, n_pages)
            for pg in range(n_pages):
                if (l, h, pg) not in touched:
                    assert np.all(host[pool + pg * stride: pool + (pg + 1) * stride] == 0xAB)
    scale = 1.0 / math.sqrt(d)
    q = np.stack([np.stack([probs[l][b].q_post for b in range(B)]) for l in range(Lyr)])
    qd = _cuda(q, torch.bfloat16)
    out_b = P.decode_attention_paged(lay, 0, cache, qd, seq, table, n_pages, scale, lay.new_workspace(B, Lyr), n_layers=Lyr)
    ws1 = lay.new_workspace(B, 1)
    out_l = torch.stack([P.decode_attention_paged(lay, l, cache, qd[l].contiguous(), seq, table, n_pages, scale, ws1)
                         for l in range(Lyr)])
    torch.cuda.synchronize()
    for l in range(Lyr):
        for b in range(B):
            for name, out in (("batched", out_b), ("per-layer", out_l)):
                got = out[l, b].double().cpu().numpy()
                if not lens[b]:
                    assert np.all(got == 0.0)
                    continue
                exp, rv = H.oracle_attention(probs[l][b], heads[l][b], tab128, scale)
                err = max(np.max(np.abs(got[a] - exp[a])) / rv[a // (Hq // Hkv)] for a in range(Hq))
                assert err <= 2e-3, (name, l, b, err)
    with pytest.raises(P.BgtqError):
        P.decode_attention_paged(lay, 0, cache, qd[0].contiguous(), seq, table, 0, scale, ws1)


@pytest.mark.parametrize("kv_dtype,pairing", [("f32", 0), ("bf16", 0), ("bf16", 1)])
def test_append_with_fused_rope_bit_exact(P, tab128, kv_dtype, pairing):
    """bgtq_quantize_append_rope on PRE-RoPE keys == oracle rope_table (fp64, no intermediate
    rounding) -> quantise -> pack, byte for byte; two layers in one call, ragged chunks, both pairings."""
    import workloads as W
    Lyr, B, Hq, Hkv, d, T, max_tokens = 2, 1, 8, 2, 128, 300, 384
    L = d // 2
    rng = np.random.default_rng(3)
    base = 1.0e6
    ang = np.arange(max_tokens, dtype=np.float64)[:, None] * base ** (-2.0 * np.arange(L) / d)[None, :]
    cos32, sin32 = np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)
    probs, k_pre = [], []
    for l in range(Lyr):
        p = H.make_problem(300 + l, T, Hq, Hkv, 3, 3, 1, 8, rope_base=base, kv_dtype=kv_dtype)
        scales = W.block_scales(300 + l, Hkv, L)
        kp = W.pre_rope_gaussian(300 + l, 1, T, Hkv, d, scales)
        kp = W.round_to_bf16(kp).astype(np.float64) if kv_dtype == "bf16" else kp.astype(np.float32).astype(np.float64)
        p.k_post = O.rope_table(kp, cos32[:T].astype(np.float64), sin32[:T].astype(np.float64), pairing)
        if pairing == 1:                                   # allocation per interleaved block: any valid bits will do
            p.bits = np.stack([rng.permutation(p.bits[h]) for h in range(Hkv)])
        probs.append(p); k_pre.append(kp)
    bits = np.stack([p.bits for p in probs])
    lay = P.Layout(bits, Hq, d, 3, probs[0].rot, pairing=pairing)
    cache = lay.new_cache(B, max_tokens)
    seq = torch.zeros(B, dtype=torch.int32, device="cuda")
    tdt = torch.float32 if kv_dtype == "f32" else torch.bfloat16
    cs, sn = torch.from_numpy(cos32).cuda(), torch.from_numpy(sin32).cuda()
    t = 0
    for n in (130, 1, 169):
        k = _cuda(np.stack([k_pre[l][None, t:t + n] for l in range(Lyr)]), tdt)
        v = _cuda(np.stack([probs[l].v[None, t:t + n] for l in range(Lyr)]), tdt)
        P.quantize_append_rope(lay, 0, cache, k, v, seq, max_tokens, cs, sn, n_layers=Lyr)
        t += n
    assert int(seq.item()) == T
    host = cache.cpu().numpy()
    n_cap = max_tokens // 128
    for l in range(Lyr):
        heads = [O.quantize_head(probs[l].k_post[:, h], probs[l].v[:, h], probs[l].bits[h], 3, tab128, pairing=pairing)
                 for h in range(Hkv)]
        for h in range(Hkv):
            stride, off = lay.tile_stride(l, h), lay.region_offset(l, 0, h, B, max_tokens)
            exp = np.zeros(n_cap * stride, dtype=np.uint8)
            O.pack_region(heads[h], d, exp)
            assert np.array_equal(host[off:off + n_cap * stride], exp), (l, h)
    with pytest.raises(P.BgtqError):                       # tables shorter than the capacity
        P.quantize_append_rope(lay, 0, cache, k, v, seq, max_tokens, cs[:100].contiguous(), sn[:100].contiguous(), n_layers=Lyr)


# ----------------------------------------------------------------------------- protected regime
def _protected_expected(p, heads, tab, scale, n_sink, n_recent):
    k16 = p.k_post.astype(np.float16).astype(np.float64)
    v16 = p.v.astype(np.float16).astype(np.float64)
    G = p.Hq // p.Hkv
    return np.concatenate([O.decode_attention_protected_head(p.q_post[h * G:(h + 1) * G], heads[h], tab, p.d_h, scale,
                                                             k16[:, h], v16[:, h], n_sink, n_recent) for h in range(p.Hkv)])


def _host_windows(p, n_sink, n_recent):
    """The window buffers as the layout rule defines them (oracle.window_slot), filled on the host."""
    wk = np.zeros((p.Hkv, n_sink + n_recent, p.d_h), dtype=np.float16); wv = np.zeros_like(wk)
    prot, _ = O.protected_sets(p.T, n_sink, n_recent)
    for t in prot:
        s = O.window_slot(int(t), n_sink, n_recent)
        wk[:, s] = p.k_post[t].astype(np.float16); wv[:, s] = p.v[t].astype(np.float16)
    return wk, wv, prot


@pytest.mark.parametrize("T,n_sink,n_recent,chunks", [(300, 4, 128, [300]), (700, 4, 128, [100, 250, 1, 349]), (132, 4, 128, [132]),
                                                      (133, 4, 128, [3, 130]), (100, 4, 128, [100]), (3, 4, 128, [3]),
                                                      (260, 0, 7, [255, 5]), (260, 5, 0, [2, 258]), (1000, 100, 300, [1000])])
def test_protected_windows_attention_and_append(P, tab128, T, n_sink, n_recent, chunks):
    """bgtq_window_append + bgtq_decode_attention_protected == the oracle's one-softmax definition with fp16 rows for
    the first n_sink / last n_recent tokens; the window slots hold exactly the fp16-rounded rows; the packed cache
    is untouched by the regime (still bit-exact, checked by _append_and_compare's path below)."""
    Hq, Hkv = 8, 2
    p = H.make_problem(900 + T + n_recent, T, Hq, Hkv, 3, 2, 1, 8, rope_base=1e6)       # K3V2: the AIME budget
    lay = P.Layout(p.bits[None], Hq, p.d_h, p.b_v, p.rot)
    max_tokens = (T + 127) // 128 * 128 + 128
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    win_k, win_v = P.new_windows(lay, 1, n_sink, n_recent)
    t0 = 0
    for n in chunks:
        kk = _cuda(p.k_post[None, t0:t0 + n], torch.float32); vv = _cuda(p.v[None, t0:t0 + n], torch.float32)
        P.window_append(lay, 0, kk, vv, seq, win_k, win_v, n_sink, n_recent)
        P.quantize_append(lay, 0, cache, kk, vv, seq, max_tokens)
        t0 += n
    assert seq.tolist() == [T]
    wk, wv, prot = _host_windows(p, n_sink, n_recent)
    slots = sorted(O.window_slot(int(t), n_sink, n_recent) for t in prot)
    got_k = win_k[0, 0].cpu().numpy(); got_v = win_v[0, 0].cpu().numpy()
    assert np.array_equal(got_k[:, slots].view(np.uint16), wk[:, slots].view(np.uint16))
    assert np.array_equal(got_v[:, slots].view(np.uint16), wv[:, slots].view(np.uint16))
    heads = H.oracle_heads(p, tab128)
    scale = 1.0 / math.sqrt(p.d_h)
    q = _cuda(p.q_post[None], torch.bfloat16)
    out = P.decode_attention_protected(lay, 0, cache, q, seq, max_tokens, scale, win_k, win_v, n_sink, n_recent,
                                       lay.new_workspace(1))
    torch.cuda.synchronize()
    exp = _protected_expected(p, heads, tab128, scale, n_sink, n_recent)
    _, rv = H.oracle_attention(p, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    err = max(np.max(np.abs(got[a] - exp[a])) / rv[a // G] for a in range(Hq))
    assert err <= 2e-3, err
    # the buffer-free entry point on the same cache still gives the buffer-free answer (nothing leaked into the packed path)
    plain = P.decode_attention(lay, 0, cache, q, seq, max_tokens, scale, lay.new_workspace(1))[0].double().cpu().numpy()
    exp0, _ = H.oracle_attention(p, heads, tab128, scale)
    assert max(np.max(np.abs(plain[a] - exp0[a])) / rv[a // G] for a in range(Hq)) <= 2e-3


def test_protected_windows_layers_and_ragged_batch(P, tab128):
    """3 layers x 3 sequences (one of them empty, one shorter than the windows) in one launch and per layer."""
    Lyr, B, Hq, Hkv, d, ns, nr = 3, 3, 8, 2, 128, 4, 128
    lens = [389, 0, 100]
    probs = [[H.make_problem(1200 + 10 * l + b, max(lens[b], 1), Hq, Hkv, 3, 2, 1, 8, rope_base=1e6) for b in range(B)] for l in range(Lyr)]
    for l in range(Lyr):
        for b in range(B):
            probs[l][b].bits = probs[l][0].bits
    lay = P.Layout(np.stack([probs[l][0].bits for l in range(Lyr)]), Hq, d, 2, probs[0][0].rot)
    max_tokens = 512
    cache = lay.new_cache(B, max_tokens)
    win_k, win_v = P.new_windows(lay, B, ns, nr)
    for l in range(Lyr):
        for b in range(B):
            if lens[b] == 0:
                continue
            pb = probs[l][b]
            kk = np.zeros((B, lens[b], Hkv, d)); vv = np.zeros_like(kk)
            kk[b] = pb.k_post; vv[b] = pb.v
            seq_l = torch.full((B,), max_tokens, dtype=torch.int32, device="cuda"); seq_l[b] = 0     # the others are "full"
            P.quantize_append(lay, l, cache, _cuda(kk, torch.float32), _cuda(vv, torch.float32), seq_l, max_tokens,
                              advance_seq_len=False)
            wk, wv, _ = _host_windows(pb, ns, nr)
            win_k[l, b] = torch.from_numpy(wk).cuda(); win_v[l, b] = torch.from_numpy(wv).cuda()
    seq = torch.tensor(lens, dtype=torch.int32, device="cuda")
    scale = 1.0 / math.sqrt(d)
    qd = _cuda(np.stack([np.stack([probs[l][b].q_post for b in range(B)]) for l in range(Lyr)]), torch.bfloat16)
    out_b = P.decode_attention_protected(lay, 0, cache, qd, seq, max_tokens, scale, win_k, win_v, ns, nr,
                                         lay.new_workspace(B, Lyr), n_layers=Lyr)
    ws1 = lay.new_workspace(B, 1)
    out_l = torch.stack([P.decode_attention_protected(lay, l, cache, qd[l].contiguous(), seq, max_tokens, scale, win_k, win_v,
                                                      ns, nr, ws1) for l in range(Lyr)])
    torch.cuda.synchronize()
    assert torch.all(out_b[:, 1] == 0) and torch.all(out_l[:, 1] == 0)
    for l in range(Lyr):
        for b in (0, 2):
            pb = probs[l][b]
            heads = H.oracle_heads(pb, tab128)
            exp = _protected_expected(pb, heads, tab128, scale, ns, nr)
            _, rv = H.oracle_attention(pb, heads, tab128, scale)
            for name, out in (("batched", out_b), ("per-layer", out_l)):
                got = out[l, b].double().cpu().numpy()
                err = max(np.max(np.abs(got[a] - exp[a])) / rv[a // (Hq // Hkv)] for a in range(Hq))
                assert err <= 2e-3, (name, l, b, err)


def test_protected_argument_errors(P):
    p = H.make_problem(43, 4, 8, 1, 3, 3, 1, 8)
    lay = P.Layout(p.bits[None], 8, 128, 3, p.rot)
    cache = lay.new_cache(1, 128)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    q = _cuda(p.q_post[None], torch.bfloat16)
    wk, wv = P.new_windows(lay, 1, 4, 128)
    for ns, nr in [(128, 4), (0, 0), (-1, 4), (4, 2000)]:
        with pytest.raises(P.BgtqError):
            P.decode_attention_protected(lay, 0, cache, q, seq, 128, 0.1, wk, wv, ns, nr, lay.new_workspace(1))


# ----------------------------------------------------------------------------- capacity that is not a whole number of tiles
@pytest.mark.parametrize("fmt", [1, 2])
def test_append_past_a_capacity_that_is_not_a_tile_multiple(P, tab128, fmt):
    """max_tokens = 1000 (not a multiple of 128): tokens at positions >= 1000 are dropped, seq_len saturates at 1000 and the
    bytes equal the oracle's packing of the first 1000 tokens -- also with the fused-RoPE append, whose cos / sin tables
    have exactly max_tokens rows (nothing beyond them may be read)."""
    T, cap = 1030, 1000
    p = H.make_problem(77, T, 4, 2, 3, 3, 1, 8, rope_base=1e6)
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, p.b_v, p.rot, fmt=fmt)
    cache = lay.new_cache(1, cap)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    for (a, b) in [(0, 990), (990, 1030)]:
        P.quantize_append(lay, 0, cache, _cuda(p.k_post[None, a:b], torch.float32), _cuda(p.v[None, a:b], torch.float32), seq, cap)
    assert seq.tolist() == [cap]
    heads = H.oracle_heads(p, tab128, 0, cap)
    host = cache.cpu().numpy()
    for h in range(p.Hkv):
        stride = lay.tile_stride(0, h)
        off = lay.region_offset(0, 0, h, 1, cap)
        exp = np.zeros(8 * stride, dtype=np.uint8)
        O.pack_region(heads[h], p.d_h, exp, version=fmt)
        assert np.array_equal(host[off:off + 8 * stride], exp), h
    # one more append at capacity: nothing changes
    P.quantize_append(lay, 0, cache, _cuda(p.k_post[None, :5], torch.float32), _cuda(p.v[None, :5], torch.float32), seq, cap)
    assert seq.tolist() == [cap] and np.array_equal(cache.cpu().numpy(), host)
    # attention over the saturated cache
    scale = 1.0 / math.sqrt(p.d_h)
    out = P.decode_attention(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, cap, scale, lay.new_workspace(1))
    pc = H.Problem(p.d_h, p.Hq, p.Hkv, cap, p.b_v, p.bits, p.k_post[:cap], p.v[:cap], p.q_post, p.scores, p.rot)
    exp, rv = H.oracle_attention(pc, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    assert max(np.max(np.abs(got[a] - exp[a])) / rv[a // 2] for a in range(p.Hq)) <= 2e-3


def test_rope_append_with_tables_of_exactly_max_tokens_rows(P, tab128):
    T, cap, d = 1010, 1000, 128
    p = H.make_problem(78, T, 4, 2, 3, 3, 1, 8, rope_base=1e6)
    scales = W.block_scales(78, 2, 64)
    k_pre = W.pre_rope_gaussian(78, 1, T, 2, d, scales).astype(np.float32).astype(np.float64)
    inv = 1e6 ** (-np.arange(64) / 64.0)
    ang = np.arange(cap)[:, None] * inv[None, :]
    cos, sin = np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)      # exactly `cap` rows
    lay = P.Layout(p.bits[None], p.Hq, d, p.b_v, p.rot)
    cache = lay.new_cache(1, cap)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    for (a, b) in [(0, 995), (995, 1010)]:
        P.quantize_append_rope(lay, 0, cache, _cuda(k_pre[None, None, a:b], torch.float32), _cuda(p.v[None, None, a:b], torch.float32),
                               seq, cap, torch.from_numpy(cos).cuda(), torch.from_numpy(sin).cuda(), n_layers=1)
    torch.cuda.synchronize()
    assert seq.tolist() == [cap]
    k_rot = O.rope_table(k_pre[:cap], cos.astype(np.float64), sin.astype(np.float64))
    host = cache.cpu().numpy()
    for h in range(2):
        head = O.quantize_head(k_rot[:, h], p.v[:cap, h], p.bits[h], p.b_v, tab128)
        stride = lay.tile_stride(0, h)
        off = lay.region_offset(0, 0, h, 1, cap)
        exp = np.zeros(8 * stride, dtype=np.uint8)
        O.pack_region(head, d, exp)
        assert np.array_equal(host[off:off + 8 * stride], exp), h


@pytest.mark.parametrize("bits_kind", ["mostly_zero", "all_zero"])
def test_attention_sparse_keys_b_v1_multi_cta(P, tab128, bits_kind):
    """Tile stride below the partial-record size (zero-width K blocks, b_V = 1) at a context long enough for CTAs to merge
    their warps' records in shared memory; and a head without any K group (every logit 0: uniform attention)."""
    T = 128 * 640
    p = H.make_problem(79, T, 8, 1, 3, 1, 0, 8, rope_base=1e6, n_cal=32)
    p.bits[:] = 0
    if bits_kind == "mostly_zero":
        p.bits[0, :6] = [1, 1, 2, 1, 0, 1]
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, 1, p.rot)
    assert lay.tile_stride(0, 0) < 8 * 130 * 4
    cache = lay.new_cache(1, T)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    P.quantize_append(lay, 0, cache, _cuda(p.k_post[None], torch.float32), _cuda(p.v[None], torch.float32), seq, T)
    scale = 1.0 / math.sqrt(p.d_h)
    out = P.decode_attention(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, T, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    heads = H.oracle_heads(p, tab128)
    exp, rv = H.oracle_attention(p, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    err = max(np.max(np.abs(got[a] - exp[a])) / rv[0] for a in range(p.Hq))
    assert err <= 2e-3, err


def test_window_append_respects_capacity(P, tab128):
    """Tokens beyond max_tokens are dropped by bgtq_window_append exactly as by the append: the ring keeps the rows of the
    last n_recent CACHED tokens, and the protected attention over the saturated cache matches the oracle on those tokens."""
    T, cap, ns, nr = 300, 256, 4, 64
    p = H.make_problem(80, T, 8, 2, 3, 2, 1, 8, rope_base=1e6)
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, p.b_v, p.rot)
    cache = lay.new_cache(1, cap)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    win_k, win_v = P.new_windows(lay, 1, ns, nr)
    for (a, b) in [(0, 200), (200, 300)]:
        kk, vv = _cuda(p.k_post[None, a:b], torch.float32), _cuda(p.v[None, a:b], torch.float32)
        P.window_append(lay, 0, kk, vv, seq, win_k, win_v, ns, nr, max_tokens=cap)
        P.quantize_append(lay, 0, cache, kk, vv, seq, cap)
    assert seq.tolist() == [cap]
    pc = H.Problem(p.d_h, p.Hq, p.Hkv, cap, p.b_v, p.bits, p.k_post[:cap], p.v[:cap], p.q_post, p.scores, p.rot)
    wk, wv, prot = _host_windows(pc, ns, nr)
    slots = sorted(O.window_slot(int(t), ns, nr) for t in prot)
    assert np.array_equal(win_k[0, 0].cpu().numpy()[:, slots].view(np.uint16), wk[:, slots].view(np.uint16))
    assert np.array_equal(win_v[0, 0].cpu().numpy()[:, slots].view(np.uint16), wv[:, slots].view(np.uint16))
    heads = H.oracle_heads(pc, tab128)
    scale = 1.0 / math.sqrt(p.d_h)
    out = P.decode_attention_protected(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, cap, scale, win_k, win_v, ns, nr,
                                       lay.new_workspace(1))
    exp = _protected_expected(pc, heads, tab128, scale, ns, nr)
    _, rv = H.oracle_attention(pc, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    assert max(np.max(np.abs(got[a] - exp[a])) / rv[a // 4] for a in range(p.Hq)) <= 2e-3
    with pytest.raises(P.BgtqError):
        P.window_append(lay, 0, _cuda(p.k_post[None, :1], torch.float32), _cuda(p.v[None, :1], torch.float32), seq, win_k, win_v, 128, 64)


# ----------------------------------------------------------------------------- exact-density codebooks
@pytest.mark.parametrize("T,Hq,Hkv,b_k,b_v,bmin,bmax", [(333, 8, 2, 3, 3, 1, 8), (1000, 16, 2, 3, 3, 0, 8), (300, 8, 2, 2, 2, 1, 8),
                                                       (200, 4, 1, 5, 5, 1, 8), (150, 8, 2, 4, 6, 1, 8)])
def test_exact_density_codebooks_append_and_attention(P, rot128, T, Hq, Hkv, b_k, b_v, bmin, bmax):
    """BGTQ_CODEBOOK_EXACT: every group quantises against C_{b, m_g} (V against C_{b_V, 128}); packed bytes bit-exact and
    attention <= 2e-3 against the oracle run with the same per-(b, m) tables (its own solver)."""
    tab = O.Tables(rot128, 128, cb_kind="sphere")
    p = H.make_problem(300 + T, T, Hq, Hkv, b_k, b_v, bmin, bmax, rope_base=1e6)
    lay = P.Layout(p.bits[None], Hq, p.d_h, b_v, p.rot, exact_codebooks=True)
    assert lay.exact_codebooks and lay.fmt == 1
    max_tokens = (T + 127) // 128 * 128
    cache = lay.new_cache(1, max_tokens)
    seq = torch.zeros(1, dtype=torch.int32, device="cuda")
    half = T // 2
    for (a, b) in [(0, half), (half, T)]:
        P.quantize_append(lay, 0, cache, _cuda(p.k_post[None, a:b], torch.float32), _cuda(p.v[None, a:b], torch.float32), seq, max_tokens)
    heads = H.oracle_heads(p, tab)
    host = cache.cpu().numpy()
    differs_from_gaussian = False
    tabg = O.Tables(rot128, 128)
    for h in range(Hkv):
        stride = lay.tile_stride(0, h)
        off = lay.region_offset(0, 0, h, 1, max_tokens)
        exp = np.zeros((max_tokens // 128) * stride, dtype=np.uint8)
        O.pack_region(heads[h], p.d_h, exp)
        assert np.array_equal(host[off:off + exp.size], exp), h
        hg = O.quantize_head(p.k_post[:, h], p.v[:, h], p.bits[h], b_v, tabg)
        differs_from_gaussian |= not np.array_equal(hg.kidx, heads[h].kidx)
    assert differs_from_gaussian                                    # (the tables really are different ones)
    scale = 1.0 / math.sqrt(p.d_h)
    out = P.decode_attention(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, max_tokens, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    exp, rv = H.oracle_attention(p, heads, tab, scale)
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    err = max(H.record_error("exact-density codebooks", got[a], exp[a], rv[a // G], T=T, b_k=b_k, b_v=b_v) for a in range(Hq))
    assert err <= 2e-3, err
    with pytest.raises(P.BgtqError):
        P.prefill_attention(lay, 0, cache, _cuda(p.q_post[None, None], torch.bfloat16), seq, max_tokens, scale)


# ----------------------------------------------------------------------------- a4 fast path (tensor cores + exact recheck)
@pytest.mark.parametrize("kv_dtype,n_new", [("f32", 1000), ("bf16", 16), ("f32", 130)])
def test_append_fast_path_writes_the_exact_kernels_bytes(P, tab128, kv_dtype, n_new):
    """Bulk appends (>= 16 tokens) run the TF32 tensor-core path with an exact fp64 recheck inside the guard band; the
    bytes must equal those of the exact fp64 kernel (forced with the test hook) and of the oracle, for every width 1..8
    on both sides of the cache."""
    p = H.make_problem(77, n_new, 8, 2, 3, 3, 1, 8, kv_dtype=kv_dtype)
    p.bits[0, :] = np.resize(np.arange(1, 9), 64)            # every K width, eight groups of 16 coordinates
    bits_v = np.array([[1, 2, 3, 4, 5, 6, 7, 8], [3] * 8], np.uint8)
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, 0, p.rot, bits_v=bits_v[None])
    tdt = torch.float32 if kv_dtype == "f32" else torch.bfloat16
    k, v = _cuda(p.k_post[None], tdt), _cuda(p.v[None], tdt)
    caches = []
    try:
        for exact_only in (False, True):
            assert P.append_exact_only(exact_only) in (False, True)
            cache = lay.new_cache(1, 1024)
            seq = torch.zeros(1, dtype=torch.int32, device="cuda")
            P.quantize_append(lay, 0, cache, k, v, seq, 1024)
            caches.append(cache.cpu().numpy())
    finally:
        P.append_exact_only(False)
    assert np.array_equal(caches[0], caches[1])
    for h in range(2):
        qh = O.quantize_head(p.k_post[:, h], p.v[:, h], p.bits[h], 0, tab128, bits_v=bits_v[h])
        stride, off = lay.tile_stride(0, h), lay.region_offset(0, 0, h, 1, 1024)
        exp = np.zeros(8 * stride, dtype=np.uint8)
        O.pack_region(qh, p.d_h, exp)
        assert np.array_equal(caches[0][off:off + 8 * stride], exp), h


@pytest.mark.parametrize("kv_dtype,n_old,n_new", [("bf16", 0, 300), ("f32", 50, 700), ("bf16", 128, 256)])
def test_append_whole_tile_path_matches_the_exact_kernel_and_the_oracle(P, tab128, kv_dtype, n_old, n_new):
    """Bulk appends send every tile whose 128 tokens are all new to quantize_tile_kernel (one pass per tile) and leave
    the partly filled first / last tile to the sub-batch kernel: an unaligned start (n_old tokens already cached), a
    ragged end and two sequences of different lengths in one call must give the exact kernel's bytes and the oracle's."""
    T = n_old + n_new
    p = H.make_problem(91, T + 64, 8, 2, 3, 3, 1, 8, kv_dtype=kv_dtype)
    lay = P.Layout(p.bits[None], p.Hq, p.d_h, p.b_v, p.rot)
    tdt = torch.float32 if kv_dtype == "f32" else torch.bfloat16
    cap = 1152
    starts = [n_old, n_old + 64]                                       # the second sequence starts 64 tokens later
    caches = []
    try:
        for exact_only in (False, True):
            P.append_exact_only(exact_only)
            cache = lay.new_cache(2, cap)
            seq = torch.zeros(2, dtype=torch.int32, device="cuda")
            if n_old:                                                  # older tokens of both sequences
                k0, v0 = np.stack([p.k_post[:n_old]] * 2), np.stack([p.v[:n_old]] * 2)
                P.quantize_append(lay, 0, cache, _cuda(k0, tdt), _cuda(v0, tdt), seq, cap)
            # sequence 1 gets 64 more old tokens through a second call that appends nothing to sequence 0: emulate by
            # appending them to both and rewinding sequence 0
            k64 = np.stack([p.k_post[n_old:n_old + 64]] * 2)
            v64 = np.stack([p.v[n_old:n_old + 64]] * 2)
            P.quantize_append(lay, 0, cache, _cuda(k64, tdt), _cuda(v64, tdt), seq, cap)
            seq[0] = n_old
            knew = np.stack([p.k_post[starts[b]:starts[b] + n_new] for b in range(2)])
            vnew = np.stack([p.v[starts[b]:starts[b] + n_new] for b in range(2)])
            P.quantize_append(lay, 0, cache, _cuda(knew, tdt), _cuda(vnew, tdt), seq, cap)
            assert seq.cpu().tolist() == [starts[0] + n_new, starts[1] + n_new]
            caches.append(cache.cpu().numpy())
    finally:
        P.append_exact_only(False)
    assert np.array_equal(caches[0], caches[1])
    n_cap = cap // 128
    for b in range(2):
        Tb = starts[b] + n_new
        for h in range(2):
            qh = O.quantize_head(p.k_post[:Tb, h], p.v[:Tb, h], p.bits[h], p.b_v, tab128)
            stride, off = lay.tile_stride(0, h), lay.region_offset(0, b, h, 2, cap)
            exp = np.zeros(n_cap * stride, dtype=np.uint8)
            O.pack_region(qh, p.d_h, exp)
            assert np.array_equal(caches[0][off:off + n_cap * stride], exp), (b, h)


@pytest.mark.parametrize("counts", [[1, 3, 5, 7, 9, 11, 13, 15], [2, 4, 6, 8, 10, 12, 14, 8], [17, 1, 1, 1, 1, 1, 1, 41]])
def test_attention_every_unit_count_and_partial_lane_pattern(P, tab128, counts):
    """decode_kernel takes a group's 8-coordinate units in pairs (m16n8k16), an odd last unit alone (m16n8k8), and loads a
    trailing partial unit without predicates (its idle lanes decode words they do not own and meet the zero rows of q').
    Group sizes m = 2 * counts[w - 1] for width w cover: a single partial unit, odd and even unit counts, 1, 2 and 3 data
    lanes in the last unit, and a partial unit as the second of a pair -- on tiles that end ragged."""
    assert sum(counts) == 64
    Hq, Hkv, T = 8, 2, 517
    p = H.make_problem(123, T, Hq, Hkv, 3, 3, 1, 8, rope_base=1e4)
    order = np.random.default_rng(7).permutation(64)
    for h in range(Hkv):
        bits = np.concatenate([np.full(c, w + 1) for w, c in enumerate(counts if h == 0 else counts[::-1])])
        p.bits[h] = bits[order]                                       # widths scattered over the RoPE blocks
    max_tokens = 640
    lay, cache, seq, heads = _append_and_compare(P, p, tab128, [T], max_tokens, "f32")
    scale = 1.0 / math.sqrt(p.d_h)
    out = P.decode_attention(lay, 0, cache, _cuda(p.q_post[None], torch.bfloat16), seq, max_tokens, scale, lay.new_workspace(1))
    torch.cuda.synchronize()
    exp, rv = H.oracle_attention(p, heads, tab128, scale)
    got = out[0].double().cpu().numpy()
    G = Hq // Hkv
    err = max(H.record_error("unit-count / partial-lane patterns", got[a], exp[a], rv[a // G], T=T, b_k=3, b_v=3) for a in range(Hq))
    assert err <= 2e-3, err


def test_back_to_back_per_layer_calls_share_a_workspace(P, tab128):
    """A layer-by-layer decode issues its calls back to back on one stream with ONE workspace: every call's q-fold kernel is
    launched programmatically behind the previous call's merge kernel and must not touch the q' workspace before that call
    is done with it.  40 unsynchronised calls alternating layers and queries == the same calls with a device synchronise
    after each (bit for bit: every reduction has a fixed order)."""
    Lyr, Hq, Hkv, d, T = 2, 16, 2, 128, 3000
    probs = [H.make_problem(140 + l, T, Hq, Hkv, 3, 3, 1, 8, rope_base=1e6) for l in range(Lyr)]
    bits = np.stack([p.bits for p in probs])
    lay = P.Layout(bits, Hq, d, 3, probs[0].rot)
    max_tokens = 3072
    cache = lay.new_cache(1, max_tokens)
    for l in range(Lyr):
        seq = torch.zeros(1, dtype=torch.int32, device="cuda")
        P.quantize_append(lay, l, cache, _cuda(probs[l].k_post[None], torch.float32), _cuda(probs[l].v[None], torch.float32), seq, max_tokens)
    rng = np.random.default_rng(5)
    qs = [_cuda(H.W.round_to_bf16(rng.standard_normal((1, Hq, d)) * 3.0), torch.bfloat16) for _ in range(4)]
    ws = lay.new_workspace(1, 1)
    scale = 1.0 / math.sqrt(d)
    calls = [(i % Lyr, qs[(i * 7) % 4]) for i in range(40)]
    ref = []
    for l, q in calls:
        ref.append(P.decode_attention(lay, l, cache, q, seq, max_tokens, scale, ws).clone())
        torch.cuda.synchronize()
    outs = [torch.empty_like(ref[0]) for _ in calls]
    for (l, q), o in zip(calls, outs):
        P.decode_attention(lay, l, cache, q, seq, max_tokens, scale, ws, out=o)
    torch.cuda.synchronize()
    for i, (a, b) in enumerate(zip(ref, outs)):
        assert torch.equal(a, b), i
    exp, rv = H.oracle_attention(probs[0], H.oracle_heads(probs[0], tab128), tab128, scale)    # and the chain still computes the method
    got = P.decode_attention(lay, 0, cache, _cuda(probs[0].q_post[None], torch.bfloat16), seq, max_tokens, scale, ws)[0].double().cpu().numpy()
    err = max(np.max(np.abs(got[a] - exp[a])) / rv[a // (Hq // Hkv)] for a in range(Hq))
    assert err <= 2e-3, err

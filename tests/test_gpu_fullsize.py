"""-m gpu: parity at the sizes north_star names, in the launch configuration bench.py times.

The cache is built by bench.build_workload (energy -> allocate -> layout -> append of every layer), the attention call is
the layers-batched launch of the timed step, and ONE sampled (layer, sequence, KV head) is checked against the oracle run
on the same K, V tensors (regenerated from the seeded generator and copied to the host): packed bytes bit-exact, attention
max-abs / R_V <= 2e-3.  The sampled head is the LAST one, whose region starts beyond byte 2^31 (cfg2 at 524,288 tokens) or
2^32 (cfg4's shape) of the cache, so the 64-bit address paths of the append and decode kernels are checked, not only timed.
"""
import argparse
import math
import os
import sys

import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
import bgtq_helpers as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_24033_b200 import binding
    return binding


def _workload(P, config, layers, ctx, batch, prefill_chunk=0):
    import bench
    args = argparse.Namespace(config=config, layers=layers, ctx=ctx, batch=batch, alloc="greedy", format=1,
                              prefill_chunk=prefill_chunk, compare_fp16=False, paged=False, protected=False)
    return bench.build_workload(args, P, torch, torch.device("cuda", 0)), W.CONFIGS[config]


def _host_kv(shp, l, b, T, h):
    """K, V of (layer l, sequence b, KV head h), regenerated exactly as bench.build_workload generated them."""
    from workloads import gpu_synth as GS
    ks, vs = [], []
    for c0 in range(0, T, 32768):
        n = min(32768, T - c0)
        k, v, _ = GS.layer_kv(shp.seed0 + l + 100000 * b, n, shp.n_kv_heads, shp.d_h, shp.rope_base, "cuda", t0=c0, chunk_tag=c0 // 32768)
        ks.append(k[:, h].double().cpu().numpy()); vs.append(v[:, h].double().cpu().numpy())
    return np.concatenate(ks), np.concatenate(vs)


def _check_sampled_head(P, wl, shp, tab, l, b, h, T, B, name):
    lay, cache, q, ws = wl["lay"], wl["cache"], wl["q"], wl["ws"]
    Lyr, Hq, Hkv, d = q.shape[0], shp.n_q_heads, shp.n_kv_heads, shp.d_h
    G = Hq // Hkv
    assert wl["seq"].tolist() == [T] * B
    out = P.decode_attention(lay, 0, cache, q, wl["seq"], wl["max_tokens"], wl["scale"], ws, n_layers=Lyr)
    torch.cuda.synchronize()
    k_h, v_h = _host_kv(shp, l, b, T, h)
    head = O.quantize_head(k_h, v_h, wl["bits"][l, h], shp.b_v, tab)
    stride = lay.tile_stride(l, h)
    off = lay.region_offset(l, b, h, B, wl["max_tokens"])
    exp = np.zeros((T // 128) * stride, dtype=np.uint8)
    O.pack_region(head, d, exp)
    got = cache[off:off + exp.size].cpu().numpy()
    assert np.array_equal(got, exp), f"{name}: packed region differs"
    q_h = q[l, b, h * G:(h + 1) * G].double().cpu().numpy()
    ref = O.decode_attention_head(q_h, head, tab, d, wl["scale"])
    _, V = O.dequantize_head(head, tab, d)
    rv = math.sqrt(np.mean(np.sum(V * V, axis=1)))
    err = H.record_error(name, out[l, b, h * G:(h + 1) * G].double().cpu().numpy(), ref, rv, tokens=T, layer=l, seq=b,
                         kv_head=h, region_offset=int(off), cache_bytes=int(cache.numel()))
    assert err <= 2e-3, err
    return off


@pytest.mark.timeout(2400)
def test_cfg2_at_524288_tokens_36_layers_last_head(P, tab128):
    """BASELINE.json configs[2] at its longest context: 36 layers x 2 KV heads x 524,288 tokens (4.1 GB of packed cache)."""
    T = 524288
    wl, shp = _workload(P, 2, 36, T, 1)
    off = _check_sampled_head(P, wl, shp, tab128, 35, 0, 1, T, 1, "cfg2@524288x36L")
    assert off > 2 ** 31           # (the whole cache is 4.12e9 bytes: beyond int32, just below 2^32; cfg4 below passes 2^32)


@pytest.mark.timeout(2400)
def test_cfg4_shape_beyond_4gb_last_sequence(P, tab128):
    """BASELINE.json configs[4]'s shape (64q / 8kv, K3V2, batch 8, 131,072 tokens) over enough layers to pass 4 GB."""
    T, Lyr, B = 131072, 6, 8
    wl, shp = _workload(P, 4, Lyr, T, B)
    assert wl["cache"].numel() > 2 ** 32
    off = _check_sampled_head(P, wl, shp, tab128, Lyr - 1, B - 1, shp.n_kv_heads - 1, T, B, "cfg4-shape@131072x6Lxb8")
    assert off > 2 ** 32


@pytest.mark.timeout(2400)
def test_prefill_chunk_8192_at_131072_tokens_sampled_rows(P, tab128):
    """The timed prefill call (last 8,192 queries of a 131,072-token layer of cfg2): 16 sampled query rows, among them the
    first and last rows of a 256-row CTA block, the first and the last query of the chunk."""
    from workloads import gpu_synth as GS
    T, n_q = 131072, 8192
    wl, shp = _workload(P, 2, 1, T, 1, prefill_chunk=n_q)
    lay, cache, d, Hq, Hkv = wl["lay"], wl["cache"], shp.d_h, shp.n_q_heads, shp.n_kv_heads
    G = Hq // Hkv
    scales = W.block_scales(shp.seed0, Hkv, d // 2)
    q = GS.layer_queries(shp.seed0, n_q, Hq, scales, d, shp.rope_base, T - n_q, "cuda", tag=9, dtype=torch.bfloat16)[None].contiguous()
    out = P.prefill_attention(lay, 0, cache, q, wl["seq"], wl["max_tokens"], wl["scale"])
    torch.cuda.synchronize()
    h = 1
    k_h, v_h = _host_kv(shp, 0, 0, T, h)
    head = O.quantize_head(k_h, v_h, wl["bits"][0, h], shp.b_v, tab128)
    K, V = O.dequantize_head(head, tab128, d)
    rv = math.sqrt(np.mean(np.sum(V * V, axis=1)))
    # a CTA owns 256 query rows = 32 tokens x 8 heads: tokens 32j .. 32j+31 of the chunk
    rows = sorted({0, 1, 31, 32, 33, 63, 64, 4095, 4096, 4127, 4128, 8159, 8160, 8190, 8191, 5000})
    worst = 0.0
    for i in rows:
        pos = T - n_q + i
        for a in range(h * G, (h + 1) * G):
            ref = O.attention(q[0, i, a].double().cpu().numpy(), K[:pos + 1], V[:pos + 1], wl["scale"])
            got = out[0, i, a].double().cpu().numpy()
            worst = max(worst, H.record_error("prefill@131072,n_q=8192", got, ref, rv, row=i, q_head=a))
    assert worst <= 2e-3, worst

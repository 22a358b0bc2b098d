#!/usr/bin/env python
"""bench.py -- decode-attention throughput of the Block-GTQ packed-cache path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--ctx T] [--layers L]

Workload (BASELINE.json configs[2] at 131,072 tokens, the configuration the metric is quoted on):
Qwen2.5-3B-shaped attention, 36 independent layers, 16 query / 2 KV heads, d_h = 128, RoPE base 1e6,
K3V3 Block-GTQ (greedy allocation, widths 1..8, from the library's own energy -> allocate path),
batch 1.  One STEP = one decode step of the whole stack: quantize-on-append of one new token to
every layer (bgtq_quantize_append_layers) + split-KV decode attention over the packed cache of
every layer (bgtq_decode_attention_layers: q-fold, decode, combine).  Calibration (block energy,
allocation, layout) and the cache fill run once before the timed region and are reported under
"setup".  Inputs are seeded synthetic draws generated on the GPU; the
per-step cache footprint (~1 GB) is far larger than L2 (126 MB), so every step streams from HBM.

Prints ONE JSON line (see the keys below).  `--impl reference` times the fp64 CPU oracle
(oracle/) on a bounded sample of the same workload instead.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "decode-attention effective HBM GB/s on packed bytes at 128K ctx, K3V3 (us/step in us_per_step)"
ROT_SEED = 20260624
NOMINAL_HBM_GBS = 8000.0


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ctx", type=int, default=None, help="cached tokens per sequence (default: the config's first context)")
    ap.add_argument("--layers", type=int, default=None, help="layers (default: the config's)")
    ap.add_argument("--batch", type=int, default=None, help="sequences (default: the config's)")
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config supplying the head shape")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--microbench", action="store_true",
                    help="print the instruction-rate microbenchmarks (bgtq_debug_microbench) that profiles/ and DESIGN.md quote, then exit")
    ap.add_argument("--format", type=int, default=1, choices=[1, 2],
                    help="physical cache format: 1 = BGTQ-v1 fragment order (mma.sync decode kernel, default), 2 = BGTQ-v2 row order (tcgen05 decode kernel, measured slower: DESIGN.md section 7b)")
    ap.add_argument("--prefill-chunk", type=int, default=None,
                    help="also time bgtq_prefill_attention for the last N cached tokens of layer 0 (default: 8192 in the "
                         "default single-GPU configs[2] run so that the driver's line carries it, else 0)")
    ap.add_argument("--compare-fp16", action="store_true", default=None,
                    help="also time the fp16-cache comparison kernel (bgtq_fp16_decode_attention) on the same K, V "
                         "(default: on in the default single-GPU configs[2] run)")
    ap.add_argument("--lean", action="store_true", help="default run without the prefill and fp16-comparison legs")
    ap.add_argument("--paged", action="store_true",
                    help="also time bgtq_decode_attention_paged on a scattered-page copy of the same cache")
    ap.add_argument("--protected", action="store_true",
                    help="also time bgtq_decode_attention_protected (fp16 sink-4 / recent-128 windows, PAPER.md:813) on the same cache")
    ap.add_argument("--alloc", default="greedy", choices=["greedy", "uniform", "paper_like"],
                    help="K allocation: greedy = Block-GTQ from the library's energy->allocate path (the metric's workload); "
                         "uniform = one group at b_k bits (uniform TQ-MSE, PAPER.md:108); paper_like = greedy on scores whose "
                         "histogram resembles the paper's Qwen2.5-3B row (Table 8, PAPER.md:476)")
    args = ap.parse_args()
    shp = W.CONFIGS[args.config]
    args.ctx = args.ctx or shp.contexts[0]
    args.layers = args.layers or shp.n_layers
    args.batch = args.batch or shp.batch
    # the default run (configs[2] at its first context, BGTQ-v1, one GPU) also reports the prefill and fp16-comparison legs
    default_run = (args.config == 2 and args.ctx == shp.contexts[0] and args.layers == shp.n_layers and args.format == 1 and
                   args.gpus == 1 and args.alloc == "greedy" and not args.lean and int(os.environ.get("WORLD_SIZE", "1")) == 1)
    if args.prefill_chunk is None:
        args.prefill_chunk = 8192 if default_run else 0
    if args.compare_fp16 is None:
        args.compare_fp16 = default_run
    return args


def l2_note(args):
    """How the timed steps stay HBM-cold: the packed bytes one step reads against the 126 MB L2."""
    shp = W.CONFIGS[args.config]
    approx = args.layers * args.batch * shp.n_kv_heads * args.ctx * (16.0 * shp.b_k + 16.0 * shp.b_v + 12.0)
    if approx >= 2 * 126e6:
        return f"inputs larger than L2 (per-step footprint ~{approx / 1e6:.0f} MB >> 126 MB); no flush needed"
    return (f"per-step footprint ~{approx / 1e6:.0f} MB fits the 126 MB L2 and is NOT flushed between steps: this "
            "configuration is L2-warm (a parity / latency case, not a roofline line); the per-layer-launch figure is taken "
            "over all layers of the default configuration, which sweeps ~1 GB per step and is HBM-cold")


def workload_config(args):
    shp = W.CONFIGS[args.config]
    return {
        "workload": f"BASELINE.json configs[{args.config}] ({shp.name}) at ctx {args.ctx}: {args.layers} independent layers, "
                    f"{shp.n_q_heads}q/{shp.n_kv_heads}kv heads, d_h {shp.d_h}, K{shp.b_k}V{shp.b_v}, batch {args.batch}",
        "ctx": args.ctx, "layers": args.layers, "n_q_heads": shp.n_q_heads, "n_kv_heads": shp.n_kv_heads,
        "d_h": shp.d_h, "b_k": shp.b_k, "b_v": shp.b_v, "b_min": shp.b_min, "b_max": shp.b_max,
        "rope_base": shp.rope_base, "batch": args.batch,
        "step": "append 1 token to every layer + decode attention over every layer (one launch each, CUDA graph)",
        "l2": l2_note(args),
        "alloc": args.alloc,
    }


# ----------------------------------------------------------------------------- clocks sampler
class ClockSampler:
    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.002)

    def __enter__(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(args, T_s: int):
    """Oracle-side sample of the workload: one (layer, KV head) with T_s cached tokens, generated on
    the host with the same recipe.  Returns a closure timing one oracle decode-attention pass and
    the packed bytes it covers."""
    from oracle import oracle as O
    shp = W.CONFIGS[args.config]
    d, G, L = shp.d_h, shp.group, shp.d_h // 2
    seed = shp.seed0
    scales = W.block_scales(seed, 1, L)
    pos = np.arange(T_s, dtype=np.float64)
    k_pre = W.pre_rope_gaussian(seed, 1, T_s, 1, d, scales)
    k_post = O.rope(k_pre, pos, shp.rope_base).astype(np.float32).astype(np.float64)
    v = W.values_gaussian(seed, 2, T_s, 1, d).astype(np.float32).astype(np.float64)
    q_post = W.round_to_bf16(O.rope(W.pre_rope_gaussian(seed, 3, 1, G, d, scales), np.array([float(T_s)]),
                                    shp.rope_base)[0]).astype(np.float64)
    q_cal = W.pre_rope_gaussian(seed, 4, shp.n_cal, G, d, scales)
    s, _, _ = O.block_energy(q_cal, k_pre)
    bits = O.allocate(s[0], shp.b_k * L, shp.b_min, shp.b_max)
    tab = O.Tables(W.rotations(ROT_SEED, d), d)
    t0 = time.perf_counter()
    head = O.quantize_head(k_post[:, 0], v[:, 0], bits, shp.b_v, tab)
    t_quant = time.perf_counter() - t0
    nbytes = T_s * O.token_bytes(head.groups, d, shp.b_v)
    scale = 1.0 / math.sqrt(d)

    def one_pass():
        t = time.perf_counter()
        O.decode_attention_head(q_post, head, tab, d, scale)
        return time.perf_counter() - t

    return one_pass, nbytes, t_quant


def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    T_s = min(args.ctx, 32768)
    one_pass, nbytes, t_quant = oracle_sample(args, T_s)
    for _ in range(max(1, min(args.warmup, 2))):
        one_pass()
    times = [one_pass() for _ in range(args.steps)]
    t = float(np.mean(times))
    val = nbytes / t / 1e9
    cores = blas_threads()
    sample = (f"oracle decode attention (dequantise every key, exact softmax, fp64) over 1 layer x 1 KV head x "
              f"{T_s} tokens x {W.CONFIGS[args.config].group} query heads per step")
    cfg = workload_config(args)
    cfg["reference_sample"] = sample
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample,
                         "oracle_quantize_tokens_per_s": T_s / t_quant},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ----------------------------------------------------------------------------- N > 1: replicas only
def max_over_ranks(ms: float, world: int, device) -> float:
    """Device time of the slowest rank (the contract's max-over-ranks); identity for one rank.  Any backend: the GPU arm
    calls it under NCCL, tests/test_bench_cli.py under gloo."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_value(bytes_per_step_per_rank: float, ms_max: float, steps: int, world: int) -> float:
    """Whole-job GB/s of `world` independent replicas (weak scaling, no data-path collective): every rank moves its own
    bytes, the job takes as long as its slowest rank."""
    return world * bytes_per_step_per_rank / (ms_max / steps * 1e-3) / 1e9


def replica_seed_shift(rank: int) -> int:
    """Seed shift of a replica: rank r draws its own workload (bench.build_workload(seed_shift=r))."""
    return rank


# ----------------------------------------------------------------------------- GPU arm
def build_workload(args, P, torch, device, seed_shift: int = 0):
    """Calibrate (energy -> allocate -> layout) and fill the packed cache through the library.
    Two passes over seeded generators (pass 1: block energy per layer; pass 2: regenerate and append), so only one
    layer of fp32 K, V is resident at a time.  Returns everything a step needs plus setup timings."""
    from workloads import gpu_synth as GS
    shp = W.CONFIGS[args.config]
    Lyr, T, d, Hq, Hkv, B = args.layers, args.ctx, shp.d_h, shp.n_q_heads, shp.n_kv_heads, args.batch
    chunk = 32768
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def seed_of(l, b):
        return shp.seed0 + l + 1000 * seed_shift + 100000 * b

    def gen_chunk(l, b, c0, n):
        return GS.layer_kv(seed_of(l, b), n, Hkv, d, shp.rope_base, device, t0=c0, chunk_tag=c0 // chunk)

    # ---- pass 1: block energy from n_cal calibration queries and the T keys of sequence 0 of every layer
    scales_all, scores = [], []
    t_energy, energy_bytes = 0.0, 0
    for l in range(Lyr):
        ks = []
        for c0 in range(0, T, chunk):
            k, _, scales = gen_chunk(l, 0, c0, min(chunk, T - c0))
            ks.append(k)
        k = torch.cat(ks) if len(ks) > 1 else ks[0]
        qcal = GS.layer_queries(seed_of(l, 0), shp.n_cal, Hq, scales, d, shp.rope_base, 0, device, tag=4)
        if l == 0:
            ews = P.block_energy_workspace(Hq, Hkv, d, device)    # caller-owned scratch, reused by every layer
            P.block_energy(qcal, k, workspace=ews)                # warm-up (module load, caches)
        e0, e1 = ev(), ev()
        torch.cuda._sleep(400_000)                            # ~0.2 ms of GPU idling queued first: the host enqueues e0, the
        e0.record()                                           # (cooperative) launch and e1 meanwhile, so the event pair times the
        scores.append(P.block_energy(qcal, k, workspace=ews))  # kernel and not the host's launch latency
        e1.record()
        torch.cuda.synchronize()
        t_energy += e0.elapsed_time(e1)
        energy_bytes += qcal.numel() * qcal.element_size() + k.numel() * k.element_size()
        scales_all.append(scales)
        del k, ks
    s_all = torch.cat(scores)                                   # [Lyr*Hkv, 64]
    e0, e1 = ev(), ev()
    e0.record()
    bits_d = P.allocate(s_all, shp.b_k * (d // 2), shp.b_min, shp.b_max)
    e1.record()
    torch.cuda.synchronize()
    t_alloc = e0.elapsed_time(e1)
    bits = bits_d.cpu().numpy().reshape(Lyr, Hkv, d // 2)
    if args.alloc == "uniform":                                   # comparison path: uniform TQ-MSE (one group)
        bits = np.full_like(bits, shp.b_k)
    elif args.alloc == "paper_like":                              # labelled extra profile, not a BASELINE config
        sc = torch.from_numpy(W.paper_like_scores(shp.seed0, Lyr * Hkv, d // 2).astype(np.float32)).to(device)
        bits = P.allocate(sc, shp.b_k * (d // 2), shp.b_min, shp.b_max).cpu().numpy().reshape(Lyr, Hkv, d // 2)
    t0 = time.perf_counter()
    rot = W.rotations(ROT_SEED, d)
    lay = P.Layout(bits, Hq, d, shp.b_v, rot, fmt=(1 if getattr(args, "prefill_chunk", 0) else args.format))
    t_layout = (time.perf_counter() - t0) * 1e3
    max_tokens = T + 4096
    cache = lay.new_cache(B, max_tokens, device)
    seq = torch.zeros(B, dtype=torch.int32, device=device)
    fp16 = None
    if getattr(args, "compare_fp16", False):                     # comparison path: the same K, V as a plain fp16 cache
        fp16 = (torch.zeros((Lyr, B, Hkv, max_tokens, d), dtype=torch.float16, device=device),
                torch.zeros((Lyr, B, Hkv, max_tokens, d), dtype=torch.float16, device=device))
    # ---- pass 2: regenerate layer by layer and fill the cache through bgtq_quantize_append (timed without the generation)
    # (one untimed 1-token call first: module load and function attributes are not part of the fill rate; the fill
    #  restarts at position 0 and rebuilds that tile from zeros)
    k, v, _ = gen_chunk(0, 0, 0, 1)
    P.quantize_append(lay, 0, cache, k[None].expand(B, -1, -1, -1).contiguous(), v[None].expand(B, -1, -1, -1).contiguous(),
                      seq, max_tokens, advance_seq_len=False)
    torch.cuda.synchronize()
    t_fill = 0.0
    for l in range(Lyr):
        for c0 in range(0, T, chunk):
            n = min(chunk, T - c0)
            kb, vb = [], []
            for b in range(B):
                k, v, _ = gen_chunk(l, b, c0, n)
                kb.append(k)
                vb.append(v)
            k = torch.stack(kb) if B > 1 else kb[0][None]
            v = torch.stack(vb) if B > 1 else vb[0][None]
            seq.fill_(c0)
            e0, e1 = ev(), ev()
            e0.record()
            P.quantize_append(lay, l, cache, k, v, seq, max_tokens, advance_seq_len=True)
            e1.record()
            torch.cuda.synchronize()
            t_fill += e0.elapsed_time(e1)
            if fp16 is not None:
                fp16[0][l, :, :, c0:c0 + n] = k.permute(0, 2, 1, 3).to(torch.float16)
                fp16[1][l, :, :, c0:c0 + n] = v.permute(0, 2, 1, 3).to(torch.float16)
            del k, v, kb, vb
    assert seq.tolist() == [T] * B
    # the decode-step inputs: one query and one new token per (layer, sequence)
    q = torch.stack([torch.cat([GS.layer_queries(seed_of(l, b), 1, Hq, scales_all[l], d, shp.rope_base, T, device, tag=3,
                                                 dtype=torch.bfloat16) for b in range(B)]) for l in range(Lyr)])   # [Lyr,B,Hq,d]
    k_new = torch.stack([torch.stack([gen_chunk(l, b, T, 1)[0] for b in range(B)]) for l in range(Lyr)]).contiguous()  # [Lyr,B,1,Hkv,d]
    v_new = torch.randn_like(k_new)
    # the step's inputs live in ONE device buffer (q | k_new | v_new views), so that the end-to-end leg moves them with a
    # single host-to-device copy
    nq, nk = q.numel() * 2, k_new.numel() * 4
    step_in = torch.empty(nq + 2 * nk, dtype=torch.uint8, device=device)
    qv = step_in[:nq].view(torch.bfloat16).view(q.shape); qv.copy_(q)
    kv_ = step_in[nq:nq + nk].view(torch.float32).view(k_new.shape); kv_.copy_(k_new)
    vv_ = step_in[nq + nk:].view(torch.float32).view(v_new.shape); vv_.copy_(v_new)
    q, k_new, v_new = qv, kv_, vv_
    tok_bytes = B * sum(lay.token_bytes(l, h) for l in range(Lyr) for h in range(Hkv))
    ws = lay.new_workspace(B, Lyr, device)
    torch.cuda.empty_cache()
    n_th = Lyr * B * T * Hkv
    return dict(lay=lay, cache=cache, seq=seq, q=q, k_new=k_new, v_new=v_new, step_in=step_in, ws=ws, max_tokens=max_tokens,
                tok_bytes=tok_bytes, bits=bits, scale=1.0 / math.sqrt(d), fp16=fp16,
                setup={"block_energy_ms": t_energy, "block_energy_GBs": energy_bytes / (t_energy * 1e-3) / 1e9,
                       "allocate_ms": t_alloc, "allocate_heads": Lyr * Hkv, "layout_create_ms": t_layout,
                       "cache_fill_ms": t_fill, "cache_fill_tokens_per_s": Lyr * B * T / (t_fill * 1e-3),
                       "append_codes_per_s": n_th * 2 * d / (t_fill * 1e-3),
                       "cache_bytes": int(cache.numel()),
                       "packed_bytes_per_token_per_kv_head": tok_bytes / (Lyr * Hkv * B)})


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_24033_b200 import binding as P

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    Lyr = args.layers
    wl = build_workload(args, P, torch, device, seed_shift=replica_seed_shift(rank))
    lay, cache, seq, q, k_new, v_new, ws = (wl[k] for k in ("lay", "cache", "seq", "q", "k_new", "v_new", "ws"))
    out = torch.empty_like(q)

    def step():
        P.quantize_append(lay, 0, cache, k_new, v_new, seq, wl["max_tokens"], advance_seq_len=True, n_layers=Lyr)
        P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)

    stream = torch.cuda.Stream(device)
    with torch.cuda.stream(stream):
        step()                                          # one eager step sets function attributes
        stream.synchronize()
        l0 = P.launch_count()
        step()
        launches_per_step = P.launch_count() - l0
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            step()
        for _ in range(args.warmup):
            graph.replay()
        stream.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        seq_start = int(seq[0].item())
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(local) as clk:
            marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
            e0.record(stream)
            for i in range(args.steps):
                graph.replay()
                marks[i].record(stream)
            e1.record(stream)
            stream.synchronize()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ms = e0.elapsed_time(e1)
        per = np.array([(e0 if i == 0 else marks[i - 1]).elapsed_time(marks[i]) * 1e3 for i in range(args.steps)])
        step_stats = {"median": float(np.median(per)), "mean": float(per.mean()), "p5": float(np.percentile(per, 5)),
                      "p95": float(np.percentile(per, 95))}
        ms = max_over_ranks(ms, world, device)
        ms_step = ms / args.steps
        seq_avg = seq_start + (args.steps + 1) / 2.0
        io_bytes = 2 * q.numel() * 2 + 2 * k_new.numel() * 4
        bytes_step = seq_avg * wl["tok_bytes"] + io_bytes
        value = replica_value(bytes_step, ms, args.steps, world)

        # ---- roofline of the dominant kernel (split-KV decode), timed alone with CUDA events on its stream
        P.profile_decode(True)
        for _ in range(3):
            P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)
        P.profile_decode_read()
        n_rf = max(10, min(args.steps, 50))
        for _ in range(n_rf):
            P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)
        k_ms, k_n = P.profile_decode_read()
        P.profile_decode(False)
        k_ms /= max(k_n, 1)
        seq_now = int(seq[0].item())
        alg_bytes = seq_now * wl["tok_bytes"]
        peak, peak_src = 6650.0, "fallback"
        try:
            mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            peak, peak_src = float(mp["hbm_gbs"]), "measured"
        except Exception:
            pass
        traffic, traffic_src = None, None                   # static: an ncu capture of this kernel at this workload, not measured in this run
        try:
            tr = json.load(open(os.path.join(ROOT, "profiles", "decode_traffic.json")))
            if tr.get("ctx") == args.ctx and tr.get("layers") == Lyr and lay.fmt == 1 and args.alloc == "greedy" and args.config == 2:
                traffic = tr.get("dram_bytes_per_launch")
                traffic_src = "static, from profiles/decode_traffic.json (" + tr.get("source", "") + ")"
        except Exception:
            pass
        achieved = alg_bytes / (k_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "bgtq::decode2_kernel" if lay.fmt == 2 else "bgtq::decode_kernel", "achieved": achieved, "peak": peak,
                    "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                    "kernel_us": k_ms * 1e3, "algorithmic_bytes_per_launch": alg_bytes,
                    "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS}

        # ---- comparison: own split-KV kernel over an fp16 cache of the same K, V (PAPER.md:308-310 restated on this box)
        comparison = None
        if wl["fp16"] is not None:
            k16, v16 = wl["fp16"]
            o16 = torch.empty_like(q)
            for _ in range(3):
                P.fp16_decode_attention(k16, v16, q, seq, wl["scale"], out=o16)
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            n16 = 10
            c0.record(stream)
            for _ in range(n16):
                P.fp16_decode_attention(k16, v16, q, seq, wl["scale"], out=o16)
            c1.record(stream)
            stream.synchronize()
            us16 = c0.elapsed_time(c1) / n16 * 1e3
            P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)
            stream.synchronize()
            rel = float((out.float() - o16.float()).abs().max() / o16.float().abs().max())
            bytes16 = int(seq[0].item()) * args.batch * Lyr * W.CONFIGS[args.config].n_kv_heads * 512
            comparison = {"fp16_cache_attention_us": us16, "fp16_cache_GBs": bytes16 / (us16 * 1e-6) / 1e9,
                          "fp16_cache_bytes": bytes16, "packed_attention_us": k_ms * 1e3 + 0.0,
                          "speedup_packed_vs_fp16_attention_call": None, "compression_vs_fp16": 512.0 * args.batch * Lyr * W.CONFIGS[args.config].n_kv_heads / wl["tok_bytes"],
                          "max_rel_diff_packed_vs_fp16_outputs": rel,
                          "note": "fp16 call = fp16_decode_kernel + combine; packed = decode_kernel alone (q-fold + combine add ~25 us)"}
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(stream)
            for _ in range(n16):
                P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)
            p1.record(stream)
            stream.synchronize()
            usp = p0.elapsed_time(p1) / n16 * 1e3
            comparison["packed_attention_call_us"] = usp
            comparison["speedup_packed_vs_fp16_attention_call"] = us16 / usp
            del k16, v16

        # ---- NEXT #4: the same attention over a paged copy of the cache (random page table), device-timed
        paged = None
        if args.paged:
            shp_ = W.CONFIGS[args.config]
            n_cap = (wl["max_tokens"] + 127) // 128
            n_pages = args.batch * n_cap
            gen = torch.Generator(device="cpu")
            gen.manual_seed(1234)
            table = torch.randperm(n_pages, generator=gen).to(torch.int32).reshape(args.batch, n_cap).to(device)
            pc = torch.empty(lay.paged_cache_bytes(n_pages), dtype=torch.uint8, device=device)
            for l in range(Lyr):                          # harness-side scatter of the contiguous tiles into pages
                for h in range(shp_.n_kv_heads):
                    st_, po = lay.tile_stride(l, h), lay.paged_pool_offset(l, h, n_pages)
                    pool = pc[po:po + n_pages * st_].view(n_pages, st_)
                    for b in range(args.batch):
                        ro = lay.region_offset(l, b, h, args.batch, wl["max_tokens"])
                        pool[table[b].long()] = cache[ro:ro + n_cap * st_].view(n_cap, st_)
            outp = torch.empty_like(q)
            tms = {}
            for name in ("contiguous", "paged"):
                def call():
                    if name == "paged":
                        P.decode_attention_paged(lay, 0, pc, q, seq, table, n_pages, wl["scale"], ws, out=outp, n_layers=Lyr)
                    else:
                        P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)
                for _ in range(3):
                    call()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record(stream)
                for _ in range(10):
                    call()
                g1.record(stream)
                stream.synchronize()
                tms[name] = g0.elapsed_time(g1) / 10 * 1e3
            paged = {"attention_call_us": tms["paged"], "contiguous_attention_call_us": tms["contiguous"],
                     "n_pages": n_pages, "outputs_bit_identical": bool(torch.equal(out, outp)),
                     "note": "random page table over batch*ceil(max_tokens/128) pages; same tiles, scattered"}
            del pc

        # ---- NEXT #4: protected regime (fp16 sink-4 / recent-128 windows), device-timed
        protected = None
        if args.protected:
            n_sink, n_recent = 4, 128
            win_k, win_v = P.new_windows(lay, args.batch, n_sink, n_recent)
            win_k.normal_(); win_v.normal_()              # synthetic fp16 rows (timing only; parity is tests/test_gpu_parity.py)
            outw = torch.empty_like(q)
            tms = {}
            for name in ("buffer_free", "protected"):
                def call():
                    if name == "protected":
                        P.decode_attention_protected(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], win_k, win_v,
                                                     n_sink, n_recent, ws, out=outw, n_layers=Lyr)
                    else:
                        P.decode_attention(lay, 0, cache, q, seq, wl["max_tokens"], wl["scale"], ws, out=out, n_layers=Lyr)
                for _ in range(3):
                    call()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record(stream)
                for _ in range(10):
                    call()
                g1.record(stream)
                stream.synchronize()
                tms[name] = g0.elapsed_time(g1) / 10 * 1e3
            protected = {"attention_call_us": tms["protected"], "buffer_free_attention_call_us": tms["buffer_free"],
                         "n_sink": n_sink, "n_recent": n_recent, "window_bytes": int(win_k.numel() * 2 * 2),
                         "note": "q-fold + window_kernel + decode_kernel + combine_kernel over [sink fp16 | packed | recent fp16]"}
            del win_k, win_v

        # ---- NEXT #1: causal prefill attention of the last N cached tokens (layer 0), device-timed
        prefill = None
        if args.prefill_chunk > 0:
            from workloads import gpu_synth as GS
            shp_ = W.CONFIGS[args.config]
            nq = min(args.prefill_chunk, int(seq[0].item()))
            qpf = torch.randn((args.batch, nq, shp_.n_q_heads, shp_.d_h), device=device, dtype=torch.float32).to(torch.bfloat16)
            for _ in range(2):
                opf = P.prefill_attention(lay, 0, cache, qpf, seq, wl["max_tokens"], wl["scale"])
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record(stream)
            for _ in range(3):
                opf = P.prefill_attention(lay, 0, cache, qpf, seq, wl["max_tokens"], wl["scale"])
            f1.record(stream)
            stream.synchronize()
            ms_pf = f0.elapsed_time(f1) / 3
            T_now = int(seq[0].item())
            pairs = args.batch * sum(T_now - nq + i + 1 for i in range(nq))          # causal (query, key) pairs per head
            flops = pairs * shp_.n_q_heads * 4 * shp_.d_h
            prefill = {"n_q": nq, "ms": ms_pf, "tflops": flops / (ms_pf * 1e-3) / 1e12,
                       "note": "layer 0, q-fold + prefill_kernel + derotate; 4*d_h flop per (query, key, head) pair"}

        # ---- per-layer-launch variant (model-faithful dependency order), device-timed, for the record
        per_layer_us = None
        if world == 1:
            g2 = torch.cuda.CUDAGraph()
            wsl = lay.new_workspace(args.batch, 1, device)
            with torch.cuda.graph(g2, stream=stream):
                for l in range(Lyr):
                    P.decode_attention(lay, l, cache, q[l], seq, wl["max_tokens"], wl["scale"], wsl, out=out[l])
            for _ in range(3):
                g2.replay()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record(stream)
            for _ in range(10):
                g2.replay()
            a1.record(stream)
            stream.synchronize()
            per_layer_us = a0.elapsed_time(a1) / 10 * 1e3

        # ---- a4 at prefill shape on a warm GPU: 8192 new tokens per sequence into a scratch cache (layer 0), device-timed
        append_bulk = None
        if rank == 0:
            shp_ = W.CONFIGS[args.config]
            n_app = 8192
            ac = lay.new_cache(args.batch, n_app, device)
            kk = torch.randn((args.batch, n_app, shp_.n_kv_heads, shp_.d_h), device=device, dtype=torch.float32)
            vv = torch.randn_like(kk)
            sq = torch.zeros(args.batch, dtype=torch.int32, device=device)
            def time_append():
                h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                for it in range(2 + 5):
                    if it == 2:
                        h0.record(stream)
                    sq.zero_()
                    P.quantize_append(lay, 0, ac, kk, vv, sq, n_app)
                h1.record(stream)
                stream.synchronize()
                return h0.elapsed_time(h1) / 5
            ms_app = time_append()                       # library default: the tensor-core fast path for a bulk append
            P.append_exact_only(True)
            try:
                ms_exact = time_append()                 # the exact fp64 kernel on the same input (same bytes out)
            finally:
                P.append_exact_only(False)
            vecs = args.batch * n_app * shp_.n_kv_heads
            append_bulk = {"tokens_per_seq": n_app, "ms": ms_app, "codes_per_s": vecs * 2 * shp_.d_h / (ms_app * 1e-3),
                           "input_GBs": vecs * 2 * shp_.d_h * 4 / (ms_app * 1e-3) / 1e9,
                           "exact_kernel_ms": ms_exact, "exact_kernel_codes_per_s": vecs * 2 * shp_.d_h / (ms_exact * 1e-3),
                           "note": "K and V of 8192 tokens per sequence, fp32 in, layer 0; default = whole tiles of new tokens in "
                                   "quantize_tile_kernel (one pass per 128-token tile: TF32 tensor-core rotation, exact fp64 radii, exact "
                                   "fp64 recheck inside the guard band), partly filled tiles in the 16-token sub-batch kernel; bit-identical "
                                   "to the exact fp64 kernel, timed beside it"}
            del ac, kk, vv

        # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
        step_in = wl["step_in"]                       # q | k_new | v_new, one buffer on each side
        hin = step_in.cpu().pin_memory()
        hout = torch.empty_like(out, device="cpu").pin_memory()
        n_e2e = max(5, min(args.steps, 30))
        for it in range(3 + n_e2e):
            if it == 3:
                stream.synchronize()
                b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                b0.record(stream)
            step_in.copy_(hin, non_blocking=True)
            graph.replay()
            hout.copy_(out, non_blocking=True)
            stream.synchronize()
        b1.record(stream)
        stream.synchronize()
        e2e_ms = b0.elapsed_time(b1) / n_e2e
        e2e_ms = max_over_ranks(e2e_ms, world, device)
        seq_e2e = int(seq[0].item()) - n_e2e / 2.0
        e2e_val = world * (seq_e2e * wl["tok_bytes"] + io_bytes) / (e2e_ms * 1e-3) / 1e9
        h2d = hin.numel()
        d2h = hout.numel() * 2

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        T_s = min(args.ctx, 32768)
        one_pass, nbytes, t_quant = oracle_sample(args, T_s)
        one_pass()
        reps, tt = 0, 0.0
        while tt < 12.0 and reps < 400:
            tt += one_pass()
            reps += 1
        cpu_baseline = {"value": nbytes / (tt / reps) / 1e9, "unit": "GB/s", "cores": blas_threads(), "kind": "oracle",
                        "sample": f"oracle decode attention over 1 layer x 1 KV head x {T_s} tokens x "
                                  f"{W.CONFIGS[args.config].group} query heads, {reps} passes ({tt:.1f} s); "
                                  f"oracle quantize of that sample took {t_quant:.1f} s",
                        "ms_per_pass": tt / reps * 1e3}
    if rank == 0:
        cfg = workload_config(args)
        cfg["setup"] = wl["setup"]
        cfg["per_layer_launch_us_per_step"] = per_layer_us
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "us_per_step": ms_step * 1e3, "step_us_stats": step_stats,
            "pct_of_8TBs": 100.0 * value / world / NOMINAL_HBM_GBS, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f16 codes x bf16 query, f32 accumulate (append: f64)", "data": "synthetic",
            "config": cfg, "clocks": clk.summary(), "roofline": roofline, "cpu_baseline": cpu_baseline,
            "e2e": {"value": e2e_val, "unit": "GB/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms},
            "gpu_launches": int(launches_per_step) * args.steps, "gpu_launches_per_step": int(launches_per_step),
            "comparison": comparison, "prefill": prefill, "paged": paged, "protected": protected, "append_bulk": append_bulk,
        }))
    if world > 1:
        dist.destroy_process_group()


def run_microbench():
    """`bench.py --microbench`: one line per microbenchmark (markdown table rows), at 12 warps per SM."""
    from paper_2606_24033_b200 import binding as P
    print("| quantity | value |")
    print("|---|---|")
    for i in range(P.MICROBENCH_COUNT):
        name, v = P.microbench(i, 12)
        print(f"| {name} | {v:.3f} |")


def main():
    args = parse_args()
    if args.microbench:
        run_microbench()
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

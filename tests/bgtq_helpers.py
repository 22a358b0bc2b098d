"""Shared test scaffolding: seeded synthetic problems (workloads/) + oracle-side expected values.

Nothing here comes from the CUDA path: inputs are drawn by workloads.synth, RoPE and every
expected value are computed by oracle/.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List

import numpy as np

import workloads as W
from oracle import oracle as O

ROT_SEED = 20260624


@dataclass
class Problem:
    d_h: int
    Hq: int
    Hkv: int
    T: int
    b_v: int
    bits: np.ndarray          # [Hkv, L] uint8
    k_post: np.ndarray        # [T, Hkv, d_h]  values of the boundary dtype (fp32-exact), post-RoPE
    v: np.ndarray             # [T, Hkv, d_h]
    q_post: np.ndarray        # [Hq, d_h] bf16-exact values, post-RoPE at position T
    scores: np.ndarray        # [Hkv, L] oracle block energies (fp64)
    rot: np.ndarray           # flat fp32 rotation table


def make_problem(seed: int, T: int, Hq: int, Hkv: int, b_k: int, b_v: int, b_min: int, b_max: int,
                 rope_base: float = 1.0e4, n_cal: int = 256, kv_dtype: str = "f32",
                 d_h: int = 128, rot=None) -> Problem:
    L = d_h // 2
    scales = W.block_scales(seed, Hkv, L)
    pos = np.arange(T, dtype=np.float64)
    k_pre = W.pre_rope_gaussian(seed, 1, T, Hkv, d_h, scales)
    k_post = O.rope(k_pre, pos, rope_base)
    v = W.values_gaussian(seed, 2, T, Hkv, d_h)
    q_pre = W.pre_rope_gaussian(seed, 3, 1, Hq, d_h, scales)
    q_post = O.rope(q_pre, np.array([float(T)]), rope_base)[0]
    q_cal = W.pre_rope_gaussian(seed, 4, n_cal, Hq, d_h, scales)
    if kv_dtype == "bf16":
        k_post = W.round_to_bf16(k_post).astype(np.float64)
        v = W.round_to_bf16(v).astype(np.float64)
    else:
        k_post = k_post.astype(np.float32).astype(np.float64)
        v = v.astype(np.float32).astype(np.float64)
    q_post = W.round_to_bf16(q_post).astype(np.float64)
    s, _, _ = O.block_energy(q_cal, k_pre)          # norm-invariant under RoPE
    bits = np.stack([O.allocate(s[h], b_k * L, b_min, b_max) for h in range(Hkv)])
    if rot is None:
        rot = W.rotations(ROT_SEED, d_h)
    return Problem(d_h, Hq, Hkv, T, b_v, bits, k_post, v, q_post, s, rot)


def oracle_heads(p: Problem, tab: O.Tables, t0: int = 0, t1: int | None = None) -> List[O.QuantizedHead]:
    t1 = p.T if t1 is None else t1
    return [O.quantize_head(p.k_post[t0:t1, h], p.v[t0:t1, h], p.bits[h], p.b_v, tab) for h in range(p.Hkv)]


def oracle_attention(p: Problem, heads: List[O.QuantizedHead], tab: O.Tables, scale: float):
    """-> (out [Hq, d_h] fp64, R_V [Hkv]) over the fully dequantised cache."""
    G = p.Hq // p.Hkv
    out = np.zeros((p.Hq, p.d_h))
    rv = np.zeros(p.Hkv)
    for h in range(p.Hkv):
        K, V = O.dequantize_head(heads[h], tab, p.d_h)
        rv[h] = math.sqrt(np.mean(np.sum(V * V, axis=1)))
        for a in range(h * G, (h + 1) * G):
            out[a] = O.attention(p.q_post[a], K, V, scale)
    return out, rv


def record_error(name: str, got: np.ndarray, exp: np.ndarray, rv: float, **extra) -> float:
    """Achieved attention error of a parity case: max-abs / R_V (the bar of north_star) and max-abs / max|o| (how large
    the error is against the output itself).  Appended to gpurun_out/achieved_errors.jsonl when that folder exists, so
    that BASELINE.md can quote measured numbers; returns max-abs / R_V."""
    import json
    import os
    d = float(np.max(np.abs(got - exp)))
    rec = {"case": name, "max_abs_over_R_V": d / rv, "max_abs_over_max_abs_o": d / float(np.max(np.abs(exp))), **extra}
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "achieved_errors.jsonl"), "a") as f:
            f.write(json.dumps(rec) + "\n")
    return d / rv

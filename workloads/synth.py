"""Workload shapes (BASELINE.json configs) and seeded numpy generators.

No method arithmetic lives here (see package docstring).  The recipe is stated in
DESIGN.md section "Input recipe"; the citations for the shapes are the model table
of the paper (Table 7) via BASELINE.json ``configs``.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Tuple

import numpy as np

PAIR_HALF = 0          # block i = coordinates (i, i + d_h/2)   (HF rotate_half)
PAIR_INTERLEAVED = 1   # block i = coordinates (2i, 2i + 1)


@dataclass(frozen=True)
class WorkloadShape:
    """One BASELINE.json config.  ``contexts`` lists the cached lengths T."""
    name: str
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    d_h: int
    rope_base: float
    contexts: Tuple[int, ...]
    batch: int
    b_k: int              # average K bits / dim  (b-bar)
    b_v: int              # uniform V bits / dim
    b_min: int
    b_max: int
    n_cal: int            # calibration queries
    seed0: int            # seed of layer 0 (layer l uses seed0 + l)
    q_dtype: str = "bf16"
    kv_dtype: str = "f32"
    prefill_append: int = 0
    notes: str = ""

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def n_blocks(self) -> int:
        return self.d_h // 2


# BASELINE.json ``configs`` 0..4.  b_min/b_max: DESIGN.md reading Q3 (cfg0 says 0-8
# explicitly; the others follow the paper's 1-8).
CONFIGS: Dict[int, WorkloadShape] = {
    0: WorkloadShape("cfg0-1head-4k", 1, 1, 1, 128, 1.0e4, (4096,), 1, 3, 3, 0, 8, 512, 0,
                     q_dtype="f32", kv_dtype="f32",
                     notes="correctness config; decode query at position 4096"),
    1: WorkloadShape("cfg1-qwen2.5-3b-layer-32k", 1, 16, 2, 128, 1.0e6, (32768,), 1, 3, 3, 1, 8,
                     512, 1, notes="append one token then decode, per step"),
    2: WorkloadShape("cfg2-qwen2.5-3b-36L", 36, 16, 2, 128, 1.0e6, (131072, 262144, 524288), 1,
                     3, 3, 1, 8, 512, 2, notes="36 independent layers, seeds 2..37"),
    3: WorkloadShape("cfg3-llama3.1-8b-layer-128k-b4", 1, 32, 8, 128, 5.0e5, (131072,), 4, 2, 2,
                     1, 8, 1024, 100, prefill_append=8192,
                     notes="K2V2; batch 4 independent seeds; prefill-append 8192 tokens/seq"),
    4: WorkloadShape("cfg4-70b-class-80L-128k-b8", 80, 64, 8, 128, 5.0e5, (131072,), 8, 3, 2, 1,
                     8, 4096, 1000, notes="K3V2; on-device energy + allocator for 640 heads"),
}


def pair_indices(d_h: int, pairing: int) -> Tuple[np.ndarray, np.ndarray]:
    """Coordinate indices (a(i), b(i)) of RoPE block i (index bookkeeping only)."""
    L = d_h // 2
    i = np.arange(L)
    if pairing == PAIR_HALF:
        return i, i + L
    if pairing == PAIR_INTERLEAVED:
        return 2 * i, 2 * i + 1
    raise ValueError("pairing")


def block_scales(seed: int, n_heads: int, n_blocks: int, lo: float = 1e-2,
                 hi: float = 10.0) -> np.ndarray:
    """Per-head, per-block scale s_i drawn log-uniform over [lo, hi] (BASELINE.json cfg0)."""
    rng = np.random.default_rng([seed, 0x5CA1E])
    u = rng.random((n_heads, n_blocks))
    return np.exp(np.log(lo) + u * (np.log(hi) - np.log(lo)))


def pre_rope_gaussian(seed, stream: int, n: int, n_heads: int, d_h: int, scales: np.ndarray,
                      pairing: int = PAIR_HALF, reading: str = "variance") -> np.ndarray:
    """Pre-RoPE Gaussian activations x[n, n_heads, d_h] (fp64).

    ``scales`` is [n_kv_heads or n_heads, L]; if it has fewer heads than ``n_heads`` the
    query heads of a GQA group share their KV head's row (head a -> a // G).
    reading='variance': block i has per-coordinate variance s_i (reading Q16,
    energies span ~3 decades); reading='amplitude': coordinates are multiplied by s_i.
    ``stream`` separates keys / queries / calibration draws of one seed.
    """
    rng = np.random.default_rng([int(seed), int(stream), 0xDA7A])
    x = rng.standard_normal((n, n_heads, d_h))
    hs = scales.shape[0]
    G = n_heads // hs
    a, b = pair_indices(d_h, pairing)
    amp = np.sqrt(scales) if reading == "variance" else scales
    amp_full = np.empty((n_heads, d_h))
    for h in range(n_heads):
        amp_full[h, a] = amp[h // G]
        amp_full[h, b] = amp[h // G]
    return x * amp_full[None, :, :]


def values_gaussian(seed, stream: int, n: int, n_heads: int, d_h: int) -> np.ndarray:
    """V entries N(0, 1), fp64."""
    rng = np.random.default_rng([int(seed), int(stream), 0x7A1E5])
    return rng.standard_normal((n, n_heads, d_h))


def values_block_scaled(seed, stream: int, n: int, n_heads: int, d_h: int, block: int = 16,
                        lo: float = 0.05, hi: float = 5.0) -> np.ndarray:
    """V entries whose 16-coordinate blocks have per-(head, block) variances drawn log-uniform over [lo, hi]:
    an input with something for a V-side allocator to find (reading Q19 / section 5).  fp64."""
    rng = np.random.default_rng([int(seed), int(stream), 0x7B10C])
    var = np.exp(np.log(lo) + rng.random((n_heads, d_h // block)) * (np.log(hi) - np.log(lo)))
    x = rng.standard_normal((n, n_heads, d_h))
    return x * np.repeat(np.sqrt(var), block, axis=1)[None, :, :]


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round-to-nearest-even (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))
    return (r >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round to bf16 and return the values as fp32 (exactly representable)."""
    return bf16_bits_to_f32(f32_to_bf16_bits(np.asarray(x, dtype=np.float32)))


def rotation_offsets(d_h: int) -> Dict[int, int]:
    """Element offset of Pi^(m) inside the flat rotation table, m = 2, 4, ..., d_h."""
    off, o = {}, 0
    for m in range(2, d_h + 1, 2):
        off[m] = o
        o += m * m
    off["total"] = o
    return off


def rotations(seed: int, d_h: int) -> np.ndarray:
    """The random orthogonal matrices TQ-MSE draws ("shared orthogonal
    rotation"), one per group dimension m = 2, 4, ..., d_h, as a flat fp32 table
    (row-major Pi^(m)[j][k] at ``rotation_offsets(d_h)[m] + j*m + k``).

    Drawn as a seeded Gaussian matrix orthonormalised by numpy's QR with the sign
    convention diag(R) > 0 (Haar measure), then rounded to fp32.  The fp32 table is the
    format: both sides receive it as data.
    """
    offs = rotation_offsets(d_h)
    out = np.empty(offs["total"], dtype=np.float32)
    for m in range(2, d_h + 1, 2):
        rng = np.random.default_rng([int(seed), m, 0x207A7E])
        g = rng.standard_normal((m, m))
        q, r = np.linalg.qr(g)
        q = q * np.sign(np.diag(r))[None, :]
        out[offs[m]:offs[m] + m * m] = q.astype(np.float32).ravel()
    return out


def paper_like_scores(seed: int, n_heads: int, n_blocks: int) -> np.ndarray:
    """Scores whose greedy allocation at b-bar=3 resembles the paper's Qwen2.5-3B histogram
    (Table 8: ~0.5/23.5/57.2/14.6/3.1/0.9/0.2 % at 1..7 bits): log-normal
    log4-scores with a heavy upper tail.  A labelled extra profile, not a BASELINE config.
    """
    rng = np.random.default_rng([int(seed), 0xFA9E4])
    z = rng.standard_normal((n_heads, n_blocks)) * 0.62
    tail = rng.random((n_heads, n_blocks)) < 0.05
    z = np.where(tail, z + rng.exponential(1.3, size=z.shape) + 1.0, z)
    return np.power(4.0, z)

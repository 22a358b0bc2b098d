"""Seeded synthetic inputs generated ON THE GPU for the large configs (BASELINE.json cfg2-4).

Same recipe as workloads/synth.py with a torch CUDA generator: per (layer
seed, KV head) block scales from synth.block_scales (host, tiny), pre-RoPE Gaussians with block
variance s_i, RoPE in fp64 angles, rounded to fp32.  The tensors produced here are INPUTS: the
library and the oracle both consume the post-RoPE tensor as given (parity never depends on this
file's rotation being "right"; a GPU test still checks it against the oracle's RoPE).
No quantiser, codebook, packing or attention arithmetic lives here.
"""
from __future__ import annotations

import numpy as np
import torch

from . import synth


def _amp(scales: np.ndarray, n_heads: int, d_h: int, device) -> torch.Tensor:
    """[n_heads, d_h] amplitude sqrt(s_i) on both coordinates of block i (half-split pairing)."""
    hs, L = scales.shape
    G = n_heads // hs
    a = np.sqrt(scales)
    full = np.concatenate([a, a], axis=1)                 # coords i and i + L share block i
    full = np.repeat(full, G, axis=0)
    return torch.from_numpy(full).to(device=device, dtype=torch.float64)


def rope_half(x: torch.Tensor, pos: torch.Tensor, base: float) -> torch.Tensor:
    """x [n, H, d] fp64, pos [n] fp64 -> R_pos x with blocks (i, i+d/2), theta_i = base^(-2i/d)."""
    n, H, d = x.shape
    L = d // 2
    i = torch.arange(L, device=x.device, dtype=torch.float64)
    theta = torch.pow(torch.tensor(base, dtype=torch.float64, device=x.device), -2.0 * i / d)
    ang = pos[:, None] * theta[None, :]
    c, s = torch.cos(ang)[:, None, :], torch.sin(ang)[:, None, :]
    a, b = x[..., :L], x[..., L:]
    return torch.cat([c * a - s * b, s * a + c * b], dim=-1)


def layer_kv(seed: int, T: int, n_kv_heads: int, d_h: int, base: float, device="cuda", t0: int = 0,
             chunk_tag: int = 0):
    """Post-RoPE keys and values of one layer: fp32 [T, n_kv_heads, d_h] each, positions t0..t0+T-1."""
    scales = synth.block_scales(seed, n_kv_heads, d_h // 2)
    g = torch.Generator(device=device)
    g.manual_seed((int(seed) * 1000003 + 17 * chunk_tag + 1) & 0x7FFFFFFFFFFF)
    x = torch.randn((T, n_kv_heads, d_h), generator=g, device=device, dtype=torch.float64)
    x = x * _amp(scales, n_kv_heads, d_h, device)[None]
    pos = torch.arange(t0, t0 + T, device=device, dtype=torch.float64)
    k = rope_half(x, pos, base).to(torch.float32)
    v = torch.randn((T, n_kv_heads, d_h), generator=g, device=device, dtype=torch.float32)
    return k, v, scales


def layer_queries(seed: int, n: int, n_q_heads: int, scales: np.ndarray, d_h: int, base: float, pos0: int,
                  device="cuda", tag: int = 7, dtype=torch.float32):
    """n post-RoPE queries [n, n_q_heads, d_h] at positions pos0..pos0+n-1 (same block profile)."""
    g = torch.Generator(device=device)
    g.manual_seed((int(seed) * 1000003 + 7919 * tag + 3) & 0x7FFFFFFFFFFF)
    x = torch.randn((n, n_q_heads, d_h), generator=g, device=device, dtype=torch.float64)
    x = x * _amp(scales, n_q_heads, d_h, device)[None]
    pos = torch.arange(pos0, pos0 + n, device=device, dtype=torch.float64)
    return rope_half(x, pos, base).to(dtype)

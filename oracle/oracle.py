"""fp64 CPU oracle of the Block-GTQ hot path (TEST INFRASTRUCTURE -- not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It imports nothing from paper_2606_24033_b200/.  Heavy loops live in
bgtq_oracle.c (same directory, same status); this file holds the ctypes glue and the parts
whose plain definition is a numpy one-liner (softmax attention, split merge).

Citations are PAPER.md:<line>; "Qn" are the readings listed in DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import math
from dataclasses import dataclass
from typing import List, Sequence, Tuple

import numpy as np

from . import build as _build
from . import codebook as _cb

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, u8p, u16p, fp, ip = (C.POINTER(C.c_double), C.POINTER(C.c_uint8), C.POINTER(C.c_uint16),
                                 C.POINTER(C.c_float), C.POINTER(C.c_int))
        L.orc_f64_to_f16_bits.restype = C.c_uint16
        L.orc_f64_to_f16_bits.argtypes = [C.c_double]
        L.orc_f16_bits_to_f64.restype = C.c_double
        L.orc_f16_bits_to_f64.argtypes = [C.c_uint16]
        L.orc_rope.restype = None
        L.orc_rope.argtypes = [dp, C.c_long, C.c_int, C.c_int, dp, C.c_double, C.c_int, dp]
        L.orc_block_energy.restype = None
        L.orc_block_energy.argtypes = [dp, C.c_long, C.c_int, dp, C.c_long, C.c_int, C.c_int, C.c_int, dp, dp]
        L.orc_score.restype = C.c_double
        L.orc_score.argtypes = [C.c_double, C.c_double, C.c_int]
        L.orc_allocate_linear.restype = C.c_int
        L.orc_allocate_linear.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_int, u8p, dp]
        L.orc_allocate_heap.restype = C.c_int
        L.orc_allocate_heap.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_int, u8p]
        L.orc_objective.restype = C.c_double
        L.orc_objective.argtypes = [dp, u8p, C.c_int]
        L.orc_quantize_group.restype = None
        L.orc_quantize_group.argtypes = [dp, C.c_int, fp, dp, C.c_int, u8p, u16p, dp]
        L.orc_dequantize_group.restype = None
        L.orc_dequantize_group.argtypes = [u8p, C.c_int, C.c_uint16, fp, dp, dp]
        L.orc_put_field.restype = None
        L.orc_put_field.argtypes = [C.POINTER(C.c_uint32), C.c_int, C.c_int, C.c_uint]
        L.orc_get_field.restype = C.c_uint
        L.orc_get_field.argtypes = [C.POINTER(C.c_uint32), C.c_int, C.c_int]
        L.orc_pack_region.restype = None
        L.orc_pack_region.argtypes = [u8p, C.c_long, C.c_int, ip, ip, C.c_int, C.c_int, C.c_long,
                                      C.c_long, u8p, u16p, u8p, u16p, C.c_int]
        L.orc_pack_region_kv.restype = None
        L.orc_pack_region_kv.argtypes = [u8p, C.c_long, C.c_int, ip, ip, C.c_int, C.c_int, ip, ip, C.c_long,
                                         C.c_long, u8p, u16p, u8p, u16p, C.c_int]
        L.orc_chunk_words_v2.restype = C.c_int
        L.orc_chunk_words_v2.argtypes = [C.c_int, C.c_int]
        L.orc_put_field_v2.restype = None
        L.orc_put_field_v2.argtypes = [C.POINTER(C.c_uint32), C.c_int, C.c_int, C.c_int, C.c_uint]
        L.orc_get_field_v2.restype = C.c_uint
        L.orc_get_field_v2.argtypes = [C.POINTER(C.c_uint32), C.c_int, C.c_int, C.c_int]
        L.orc_kquad_bytes_v2.restype = C.c_long
        L.orc_kquad_bytes_v2.argtypes = [C.c_int, ip, ip]
        L.orc_pack_region_v2.restype = None
        L.orc_pack_region_v2.argtypes = L.orc_pack_region.argtypes
        _lib = L
    return _lib


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def _c64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


PAIR_HALF, PAIR_INTERLEAVED = 0, 1
SCORE_KINDS = {"qk_avg": 0, "qk_max": 1, "qk_product": 2, "k_only": 3, "q_only": 4}


def pair_indices(d_h: int, pairing: int) -> Tuple[np.ndarray, np.ndarray]:
    """(a(i), b(i)) of RoPE block i (Q1)."""
    i = np.arange(d_h // 2)
    return (i, i + d_h // 2) if pairing == PAIR_HALF else (2 * i, 2 * i + 1)


# ----------------------------------------------------------------------------- fp16
def f16_bits(x: float) -> int:
    return int(lib().orc_f64_to_f16_bits(float(x)))


def f16_value(bits: int) -> float:
    return float(lib().orc_f16_bits_to_f64(int(bits)))


# ----------------------------------------------------------------------------- RoPE
def rope(x: np.ndarray, pos: np.ndarray, base: float, pairing: int = PAIR_HALF) -> np.ndarray:
    """x[n, heads, d_h] (pre-RoPE) -> R_pos x (post-RoPE), fp64.  PAPER.md:43, 53; Q1, Q2."""
    x = _c64(x)
    n, H, d = x.shape
    pos = _c64(pos)
    assert pos.shape == (n,)
    out = np.empty_like(x)
    lib().orc_rope(_p(x, C.c_double), n, H, d, _p(pos, C.c_double), float(base), int(pairing),
                   _p(out, C.c_double))
    return out


def rope_table(x: np.ndarray, cos: np.ndarray, sin: np.ndarray, pairing: int = PAIR_HALF) -> np.ndarray:
    """RoPE from caller-supplied tables (the fused-append variant): x[n, heads, d_h], cos/sin
    [n, d_h/2] -> for block i = pair (a(i), b(i)):  a' = x_a cos_i - x_b sin_i,  b' = x_a sin_i + x_b cos_i,
    each evaluated as two fp64 products and one fp64 sum (plain numpy).  With fp32/bf16-valued x and fp32-valued
    tables the products are exact, so every output is the correctly rounded value of its expression."""
    x = _c64(x)
    n, H, d = x.shape
    cos, sin = _c64(cos), _c64(sin)
    assert cos.shape == (n, d // 2) and sin.shape == (n, d // 2)
    a, b = pair_indices(d, pairing)
    out = np.empty_like(x)
    xa, xb = x[:, :, a], x[:, :, b]
    c, s_ = cos[:, None, :], sin[:, None, :]
    out[:, :, a] = xa * c - xb * s_
    out[:, :, b] = xa * s_ + xb * c
    return out


# ----------------------------------------------------------------------------- energy
def block_energy(q: np.ndarray, k: np.ndarray, pairing: int = PAIR_HALF, kind: str = "qk_avg"):
    """Eq. 4.  q[N_q, H_q, d_h], k[N_k, H_kv, d_h] -> (s, Eq, Ek) each [H_kv, L]."""
    q, k = _c64(q), _c64(k)
    nq, Hq, d = q.shape
    nk, Hkv, d2 = k.shape
    assert d == d2 and Hq % Hkv == 0
    L = d // 2
    Eq = np.empty((Hkv, L))
    Ek = np.empty((Hkv, L))
    lib().orc_block_energy(_p(q, C.c_double), nq, Hq, _p(k, C.c_double), nk, Hkv, d, int(pairing),
                           _p(Eq, C.c_double), _p(Ek, C.c_double))
    kd = SCORE_KINDS[kind]
    s = np.array([[lib().orc_score(Eq[h, i], Ek[h, i], kd) for i in range(L)] for h in range(Hkv)])
    return s, Eq, Ek


# ----------------------------------------------------------------------------- Algorithm 1
def allocate(s: Sequence[float], B: int, b_min: int, b_max: int, method: str = "linear",
             return_gains: bool = False):
    """Alg. 1 for one head.  Returns uint8 bits[L] (and the popped gains)."""
    s = _c64(s)
    if not np.all(np.isfinite(s)) or np.any(s < 0):
        raise ValueError("scores must be finite and non-negative (Q5)")
    Lb = len(s)
    bits = np.zeros(Lb, dtype=np.uint8)
    if method == "linear":
        gains = np.zeros(max(B - Lb * b_min, 0))
        rc = lib().orc_allocate_linear(_p(s, C.c_double), Lb, b_min, b_max, B, _p(bits, C.c_uint8),
                                       _p(gains, C.c_double) if len(gains) else None)
    else:
        gains = None
        rc = lib().orc_allocate_heap(_p(s, C.c_double), Lb, b_min, b_max, B, _p(bits, C.c_uint8))
    if rc != 0:
        raise ValueError("infeasible budget B")
    return (bits, gains) if return_gains else bits


def objective(s, bits) -> float:
    """J(b) = sum_i s_i 4^-b_i."""
    s = _c64(s)
    bits = np.ascontiguousarray(bits, dtype=np.uint8)
    return float(lib().orc_objective(_p(s, C.c_double), _p(bits, C.c_uint8), len(s)))


# ----------------------------------------------------------------------------- grouping
@dataclass
class Group:
    width: int                 # bits per coordinate
    blocks: np.ndarray         # member RoPE blocks, ascending
    coords: np.ndarray         # [a(i1), b(i1), a(i2), b(i2), ...]   (Q9)

    @property
    def m(self) -> int:
        return len(self.coords)


def groups_from_bits(bits: Sequence[int], d_h: int, pairing: int = PAIR_HALF) -> List[Group]:
    """G_b = {i : b_i = b} for every non-empty b >= 1, ascending width.  Width-0
    blocks are not stored and decode to zero (Q3)."""
    bits = np.asarray(bits, dtype=np.int64)
    a, b = pair_indices(d_h, pairing)
    out = []
    for w in range(1, 9):
        blk = np.nonzero(bits == w)[0]
        if len(blk) == 0:
            continue
        coords = np.empty(2 * len(blk), dtype=np.int64)
        coords[0::2] = a[blk]
        coords[1::2] = b[blk]
        out.append(Group(w, blk, coords))
    return out


V_BLOCK = 16   # coordinates per V block (reading Q19: the V-side allocator's unit)


def v_groups_from_bits(bits_v: Sequence[int], d_h: int, block: int = V_BLOCK) -> List[Group]:
    """V-side groups ("a V-side allocator", reading Q19): V block j = coordinates
    [block*j, block*j + block); blocks of equal width form one group, ascending width, member blocks and their
    coordinates in ascending order.  Every V block is stored (width >= 1)."""
    bits_v = np.asarray(bits_v, dtype=np.int64)
    assert len(bits_v) * block == d_h and bits_v.min() >= 1 and bits_v.max() <= 8
    out = []
    for w in range(1, 9):
        blk = np.nonzero(bits_v == w)[0]
        if len(blk) == 0:
            continue
        coords = (blk[:, None] * block + np.arange(block)[None, :]).reshape(-1)
        out.append(Group(w, blk, coords))
    return out


def v_block_energy(v: np.ndarray, block: int = V_BLOCK) -> np.ndarray:
    """V-side score (reading Q19): s^V_j = E_t ||v_t^(j)||^2, the mean squared norm of V block j.  With the
    TQ-MSE rate law the expected squared error of the attention output contributed by block j is
    proportional to s^V_j 4^-b_j, the same objective J(b) = sum_j s_j 4^-b_j Alg. 1 minimises for K.
    v[N, H_kv, d_h] -> s[H_kv, d_h / block].  The plain definition."""
    v = _c64(v)
    N, H, d = v.shape
    return np.mean(np.sum(v.reshape(N, H, d // block, block) ** 2, axis=3), axis=0)


class Tables:
    """Codebooks (oracle's own Lloyd-Max, fp16-rounded) + the rotation table passed in as data.
    cb_kind "gaussian": one table per width, the Lloyd-Max quantiser of N(0,1) (reading Q7);
    cb_kind "sphere":   one table per (width, group size m): the Lloyd-Max quantiser of the exact density of a rotated
                        coordinate of a normalised m-vector (oracle/codebook.py sphere_codebook)."""

    def __init__(self, rotations_flat: np.ndarray, d_h: int, cb_table: np.ndarray | None = None,
                 cb_kind: str = "gaussian"):
        assert cb_kind in ("gaussian", "sphere")
        self.d_h = d_h
        self.cb_kind = cb_kind
        self.cb = _cb.codebook_table() if cb_table is None else _c64(cb_table)
        self.rot = np.ascontiguousarray(rotations_flat, dtype=np.float32)
        self.off = {}
        o = 0
        for m in range(2, d_h + 1, 2):
            self.off[m] = o
            o += m * m
        assert o == self.rot.size

    def C(self, b: int, m: int | None = None) -> np.ndarray:
        if self.cb_kind == "sphere":
            assert m is not None
            return np.ascontiguousarray(_cb.sphere_codebook(b, m))
        return np.ascontiguousarray(self.cb[(1 << b) - 1:(1 << (b + 1)) - 1])

    def Pi(self, m: int) -> np.ndarray:
        return np.ascontiguousarray(self.rot[self.off[m]:self.off[m] + m * m]).reshape(m, m)


# ----------------------------------------------------------------------------- TQ-MSE
def quantize_group(x: np.ndarray, b: int, tab: Tables):
    """One TQ-MSE encoder (oracle step 5).  x: m exact fp64 values.
    Returns (idx uint8[m], h_bits, r)."""
    x = _c64(x)
    m = len(x)
    Pi, Cb = tab.Pi(m), tab.C(b, m)
    idx = np.zeros(m, dtype=np.uint8)
    h = C.c_uint16(0)
    r = C.c_double(0.0)
    lib().orc_quantize_group(_p(x, C.c_double), m, _p(Pi, C.c_float), _p(Cb, C.c_double), b,
                             _p(idx, C.c_uint8), C.byref(h), C.byref(r))
    return idx, int(h.value), float(r.value)


def dequantize_group(idx: np.ndarray, h_bits: int, b: int, tab: Tables) -> np.ndarray:
    """Oracle step 6: xhat = (h/sqrt(m)) * Pi^T C[idx]."""
    idx = np.ascontiguousarray(idx, dtype=np.uint8)
    m = len(idx)
    Pi, Cb = tab.Pi(m), tab.C(b, m)
    out = np.empty(m)
    lib().orc_dequantize_group(_p(idx, C.c_uint8), m, int(h_bits), _p(Pi, C.c_float),
                               _p(Cb, C.c_double), _p(out, C.c_double))
    return out


@dataclass
class QuantizedHead:
    """Codes of T tokens of one (layer, KV head): the logical (unpacked) cache content."""
    groups: List[Group]
    b_v: int
    kidx: np.ndarray      # [T, kdim] uint8, grouped coordinate order
    knorm: np.ndarray     # [T, n_groups] uint16 (fp16 bits)
    vidx: np.ndarray      # [T, d_h] uint8 (grouped V order when vgroups is set)
    vnorm: np.ndarray     # [T] uint16, or [T, n_vgroups] when vgroups is set
    vgroups: List[Group] | None = None     # V-side groups (reading Q19); None = one group of all d_h coordinates at b_v

    def v_groups(self, d_h: int) -> List[Group]:
        return self.vgroups if self.vgroups is not None else [Group(self.b_v, np.arange(d_h // V_BLOCK), np.arange(d_h))]


def quantize_head(k_post: np.ndarray, v: np.ndarray, bits: Sequence[int], b_v: int, tab: Tables,
                  pairing: int = PAIR_HALF, bits_v: Sequence[int] | None = None) -> QuantizedHead:
    """Quantise T tokens of one KV head.  k_post[T, d_h] post-RoPE keys, v[T, d_h] (exact values of
    the boundary dtype).  K: one encoder per same-width group; V: one group of all
    d_h coordinates at width b_v, or -- bits_v[d_h/16] given -- one encoder per same-width group of
    16-coordinate V blocks (reading Q19; b_v is then ignored)."""
    k_post, v = _c64(k_post), _c64(v)
    T, d = k_post.shape
    groups = groups_from_bits(bits, d, pairing)
    kdim = sum(g.m for g in groups)
    q = QuantizedHead(groups, b_v, np.zeros((T, kdim), np.uint8), np.zeros((T, len(groups)), np.uint16),
                      np.zeros((T, d), np.uint8), np.zeros(T, np.uint16))
    if bits_v is not None:
        q.vgroups = v_groups_from_bits(bits_v, d)
        q.b_v = q.vgroups[0].width
        q.vnorm = np.zeros((T, len(q.vgroups)), np.uint16)
    for t in range(T):
        o = 0
        for gi, g in enumerate(groups):
            idx, h, _ = quantize_group(k_post[t, g.coords], g.width, tab)
            q.kidx[t, o:o + g.m] = idx
            q.knorm[t, gi] = h
            o += g.m
        if q.vgroups is None:
            idx, h, _ = quantize_group(v[t], b_v, tab)
            q.vidx[t] = idx
            q.vnorm[t] = h
            continue
        o = 0
        for gi, g in enumerate(q.vgroups):
            idx, h, _ = quantize_group(v[t, g.coords], g.width, tab)
            q.vidx[t, o:o + g.m] = idx
            q.vnorm[t, gi] = h
            o += g.m
    return q


def dequantize_head(q: QuantizedHead, tab: Tables, d_h: int) -> Tuple[np.ndarray, np.ndarray]:
    """Fully dequantised (de-rotated) cache: K_hat[T, d_h] in the original coordinate order
    (width-0 blocks are 0), V_hat[T, d_h].  numpy matmul stands in for the sum of step 6."""
    T = q.kidx.shape[0]
    K = np.zeros((T, d_h))
    o = 0
    for gi, g in enumerate(q.groups):
        Cb, Pi = tab.C(g.width, g.m), tab.Pi(g.m).astype(np.float64)
        h = np.array([f16_value(x) for x in q.knorm[:, gi]]) if T < 64 else _f16_array(q.knorm[:, gi])
        K[:, g.coords] = (h / math.sqrt(g.m))[:, None] * (Cb[q.kidx[:, o:o + g.m]] @ Pi)
        o += g.m
    V = np.zeros((T, d_h))
    vnorm = q.vnorm.reshape(T, -1)
    o = 0
    for gi, g in enumerate(q.v_groups(d_h)):
        Cv, Piv = tab.C(g.width, g.m), tab.Pi(g.m).astype(np.float64)
        hv = _f16_array(vnorm[:, gi])
        V[:, g.coords] = (hv / math.sqrt(g.m))[:, None] * (Cv[q.vidx[:, o:o + g.m]] @ Piv)
        o += g.m
    return K, V


def _f16_array(bits: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(bits, dtype=np.uint16).view(np.float16).astype(np.float64)


# ----------------------------------------------------------------------------- physical layout
def tile_geometry(groups: List[Group], d_h: int, b_v: int, version: int = 1, vgroups: List[Group] | None = None):
    """Byte offsets inside one 128-token tile: [K codes | K norms | V norms | V codes].
    version 1 = BGTQ-v1 (fragment order, no padding); 2 = BGTQ-v2 (row order: a K chunk of r <= 32 coordinates of one
    token takes whole 32-bit words)."""
    if version == 2:
        gb = np.array([g.width for g in groups] + [0], dtype=np.int32)
        gm = np.array([g.m for g in groups] + [0], dtype=np.int32)
        kcode = 4 * int(lib().orc_kquad_bytes_v2(len(groups), _p(gb, C.c_int), _p(gm, C.c_int)))
    else:
        kcode = sum(16 * g.m * g.width for g in groups)
    knorm_off = kcode
    vnorm_off = knorm_off + 256 * len(groups)
    if vgroups is not None:           # V-side groups (reading Q19): one norm row and one code section per group
        assert version == 1
        vcode_off = vnorm_off + 256 * len(vgroups)
        stride = vcode_off + sum(16 * g.m * g.width for g in vgroups)
    else:
        vcode_off = vnorm_off + 256
        stride = vcode_off + 16 * d_h * b_v
    return dict(kcode=kcode, knorm_off=knorm_off, vnorm_off=vnorm_off, vcode_off=vcode_off,
                stride=stride)


def token_bytes(groups: List[Group], d_h: int, b_v: int, version: int = 1, vgroups: List[Group] | None = None) -> float:
    """Packed bytes per token of one KV head = tile stride / 128
    (v1: = 16*bbar_K + 16*b_V + 2*(n_g+1) at d_h = 128; PAPER.md:837 for the 96-byte ideal)."""
    return tile_geometry(groups, d_h, b_v, version, vgroups)["stride"] / 128.0


def pack_region(q: QuantizedHead, d_h: int, region: np.ndarray | None = None,
                t_offset: int = 0, version: int = 1) -> np.ndarray:
    """Write the T tokens of q at positions [t_offset, t_offset + T) into the packed region of
    one (sequence, layer, KV head); all other fields of ``region`` are preserved.  ``region``
    (uint8, zero-initialised) is created when None."""
    T = q.kidx.shape[0]
    geo = tile_geometry(q.groups, d_h, q.b_v, version, q.vgroups)
    n_tiles = (t_offset + T + 127) // 128
    if region is None:
        region = np.zeros(n_tiles * geo["stride"], dtype=np.uint8)
    assert region.dtype == np.uint8 and region.flags.c_contiguous
    assert region.size >= n_tiles * geo["stride"]
    ng = len(q.groups)
    gb = np.array([g.width for g in q.groups] + [0], dtype=np.int32)
    gm = np.array([g.m for g in q.groups] + [0], dtype=np.int32)
    kdim = int(gm.sum())
    # the C routine indexes its arrays by absolute token position
    kidx = np.zeros((t_offset + T, kdim), np.uint8); kidx[t_offset:] = q.kidx
    knorm = np.zeros((t_offset + T, ng), np.uint16); knorm[t_offset:] = q.knorm
    vidx = np.zeros((t_offset + T, d_h), np.uint8); vidx[t_offset:] = q.vidx
    if q.vgroups is not None:
        nvg = len(q.vgroups)
        vgb = np.array([g.width for g in q.vgroups], dtype=np.int32)
        vgm = np.array([g.m for g in q.vgroups], dtype=np.int32)
        vnorm = np.zeros((t_offset + T, nvg), np.uint16); vnorm[t_offset:] = q.vnorm
        lib().orc_pack_region_kv(_p(region, C.c_uint8), geo["stride"], ng, _p(gb, C.c_int), _p(gm, C.c_int), d_h,
                                 nvg, _p(vgb, C.c_int), _p(vgm, C.c_int), t_offset, t_offset + T,
                                 _p(kidx, C.c_uint8), _p(knorm, C.c_uint16), _p(vidx, C.c_uint8), _p(vnorm, C.c_uint16), 0)
        return region
    vnorm = np.zeros(t_offset + T, np.uint16); vnorm[t_offset:] = q.vnorm
    fn = lib().orc_pack_region_v2 if version == 2 else lib().orc_pack_region
    fn(_p(region, C.c_uint8), geo["stride"], ng, _p(gb, C.c_int),
       _p(gm, C.c_int), d_h, q.b_v, t_offset, t_offset + T,
       _p(kidx, C.c_uint8), _p(knorm, C.c_uint16),
       _p(vidx, C.c_uint8), _p(vnorm, C.c_uint16), 0)
    return region


def unpack_region(region: np.ndarray, groups: List[Group], d_h: int, b_v: int, T: int,
                  version: int = 1, vgroups: List[Group] | None = None) -> QuantizedHead:
    geo = tile_geometry(groups, d_h, b_v, version, vgroups)
    gb = np.array([g.width for g in groups], dtype=np.int32)
    gm = np.array([g.m for g in groups], dtype=np.int32)
    kdim = int(gm.sum())
    q = QuantizedHead(groups, b_v, np.zeros((T, kdim), np.uint8), np.zeros((T, len(groups)), np.uint16),
                      np.zeros((T, d_h), np.uint8), np.zeros(T, np.uint16))
    region = np.ascontiguousarray(region, dtype=np.uint8)
    if vgroups is not None:
        q.vgroups, q.b_v = vgroups, vgroups[0].width
        q.vnorm = np.zeros((T, len(vgroups)), np.uint16)
        vgb = np.array([g.width for g in vgroups], dtype=np.int32)
        vgm = np.array([g.m for g in vgroups], dtype=np.int32)
        lib().orc_pack_region_kv(_p(region, C.c_uint8), geo["stride"], len(groups), _p(gb, C.c_int), _p(gm, C.c_int), d_h,
                                 len(vgroups), _p(vgb, C.c_int), _p(vgm, C.c_int), 0, T, _p(q.kidx, C.c_uint8),
                                 _p(q.knorm, C.c_uint16), _p(q.vidx, C.c_uint8), _p(q.vnorm, C.c_uint16), 1)
        return q
    fn = lib().orc_pack_region_v2 if version == 2 else lib().orc_pack_region
    fn(_p(region, C.c_uint8), geo["stride"], len(groups), _p(gb, C.c_int),
       _p(gm, C.c_int), d_h, b_v, 0, T, _p(q.kidx, C.c_uint8),
       _p(q.knorm, C.c_uint16), _p(q.vidx, C.c_uint8), _p(q.vnorm, C.c_uint16), 1)
    return q


def put_field(W: np.ndarray, b: int, k: int, idx: int) -> None:
    lib().orc_put_field(_p(W, C.c_uint32), b, k, idx)


def get_field(W: np.ndarray, b: int, k: int) -> int:
    return int(lib().orc_get_field(_p(W, C.c_uint32), b, k))


def chunk_words_v2(b: int, r: int) -> int:
    return int(lib().orc_chunk_words_v2(b, r))


def put_field_v2(W: np.ndarray, b: int, r: int, k: int, idx: int) -> None:
    lib().orc_put_field_v2(_p(W, C.c_uint32), b, r, k, idx)


def get_field_v2(W: np.ndarray, b: int, r: int, k: int) -> int:
    return int(lib().orc_get_field_v2(_p(W, C.c_uint32), b, r, k))


# ----------------------------------------------------------------------------- attention
def attention(q: np.ndarray, K: np.ndarray, V: np.ndarray, scale: float) -> np.ndarray:
    """Exact softmax attention of one query over T cached tokens (oracle step 8):
    l_t = scale * <q, K_t>;  p = softmax(l) with max subtraction;  o = sum_t p_t V_t.  fp64."""
    q, K, V = _c64(q), _c64(K), _c64(V)
    l = scale * (K @ q)
    l = l - np.max(l)
    p = np.exp(l)
    p = p / np.sum(p)
    return p @ V


def attention_partial(q, K, V, scale):
    """(max, sum, acc) of one key-axis split."""
    q, K, V = _c64(q), _c64(K), _c64(V)
    l = scale * (K @ q)
    m = float(np.max(l))
    p = np.exp(l - m)
    return m, float(np.sum(p)), p @ V


def merge_partials(parts):
    """Exact log-sum-exp merge: M = max m_s; l = sum l_s e^(m_s-M);
    o = sum acc_s e^(m_s-M) / l."""
    M = max(p[0] for p in parts)
    l = sum(p[1] * math.exp(p[0] - M) for p in parts)
    acc = sum(p[2] * math.exp(p[0] - M) for p in parts)
    return acc / l


def decode_attention_head(q_post: np.ndarray, qh: QuantizedHead, tab: Tables, d_h: int,
                          scale: float) -> np.ndarray:
    """Attention outputs of the query heads q_post[G, d_h] sharing this KV head, over the fully
    dequantised cache (the slow plain definition: every key is de-rotated)."""
    K, V = dequantize_head(qh, tab, d_h)
    return np.stack([attention(q_post[a], K, V, scale) for a in range(q_post.shape[0])])


def protected_sets(T: int, n_sink: int, n_recent: int) -> Tuple[np.ndarray, np.ndarray]:
    """Token index sets of the *protected-buffer* regime: the cache is
    [sink (fp16) | compressed | recent (fp16)] with the first n_sink tokens and the most recent n_recent
    tokens kept as fp16.  Returns (protected, compressed) index arrays over tokens 0..T-1 (disjoint, covering);
    a token that is both among the first n_sink and the last n_recent is protected once."""
    t = np.arange(T)
    prot = (t < n_sink) | (t >= T - n_recent)
    return t[prot], t[~prot]


def window_slot(t: int, n_sink: int, n_recent: int) -> int:
    """Slot of token t in the fp16 window buffer of n_sink + n_recent rows: the sink tokens keep
    slots 0..n_sink-1, every later token t lives in the ring slot n_sink + (t mod n_recent) while it is recent."""
    return t if t < n_sink else n_sink + (t % n_recent)


def decode_attention_protected_head(q_post: np.ndarray, qh: QuantizedHead, tab: Tables, d_h: int, scale: float,
                                    k16: np.ndarray, v16: np.ndarray, n_sink: int, n_recent: int) -> np.ndarray:
    """Decode attention in the protected regime, the plain definition: one exact softmax
    over ALL T cached tokens, where a protected token contributes its fp16 key / value row (k16, v16 [T, d_h]: the
    exact post-RoPE rows rounded to fp16 by the caller) and every other token its dequantised packed row.
    n_sink = n_recent = 0 is decode_attention_head (the paper's buffer-free packed path)."""
    K, V = dequantize_head(qh, tab, d_h)
    T = K.shape[0]
    prot, _ = protected_sets(T, n_sink, n_recent)
    K = K.copy(); V = V.copy()
    K[prot] = _c64(k16)[prot]
    V[prot] = _c64(v16)[prot]
    return np.stack([attention(q_post[a], K, V, scale) for a in range(q_post.shape[0])])


def prefill_attention_head(q_post: np.ndarray, qh: QuantizedHead, tab: Tables, d_h: int, scale: float,
                           pos0: int) -> np.ndarray:
    """Causal prefill attention over the (fully dequantised) packed cache: query token i of the
    chunk sits at position pos0 + i and attends to cached tokens [0, pos0 + i] (itself included; the chunk's K, V
    are already in the cache).  q_post[n_q, G, d_h] -> out[n_q, G, d_h].  The plain definition: one exact softmax
    per (query token, head), nothing shared between rows."""
    K, V = dequantize_head(qh, tab, d_h)
    n_q, G, _ = q_post.shape
    out = np.zeros((n_q, G, d_h))
    for i in range(n_q):
        T = pos0 + i + 1
        for a in range(G):
            out[i, a] = attention(q_post[i, a], K[:T], V[:T], scale)
    return out


# ----------------------------------------------------------------------------- RoPE-logit MAE (App. B.3)
def rope_logit_mae(q_pre: np.ndarray, k_pre: np.ndarray, bits: np.ndarray, tab: Tables, base: float,
                   offsets: np.ndarray | None = None, pairing: int = PAIR_HALF) -> float:
    """MAE = E_h E_{g in G(h)} E_(q,k) E_{Delta in D} | q^T R_Delta k - q^T R_Delta khat |, K-only: khat is the TQ-MSE /
    Block-GTQ reconstruction of the PRE-RoPE key under the allocation bits[h] (uniform TQ-MSE = all blocks at one width,
    PAPER.md:108), the analytic rotation R_Delta is applied identically to k and khat, D = 50 evenly spaced offsets in
    [-1024, 1024].  q_pre [N, Hq, d], k_pre [N, Hkv, d] are paired sample by sample; bits [Hkv, d/2]."""
    q_pre, k_pre = np.asarray(q_pre, np.float64), np.asarray(k_pre, np.float64)
    N, Hq, d = q_pre.shape
    Hkv = k_pre.shape[1]
    G = Hq // Hkv
    if offsets is None:
        offsets = np.linspace(-1024.0, 1024.0, 50)
    a, b = pair_indices(d, pairing)
    theta = np.array([base ** (-2.0 * i / d) for i in range(d // 2)])
    total, count = 0.0, 0
    for h in range(Hkv):
        groups = groups_from_bits(bits[h], d, pairing)
        khat = np.zeros((N, d))
        for t in range(N):
            for g in groups:
                idx, hb, _ = quantize_group(k_pre[t, h, g.coords], g.width, tab)
                khat[t, g.coords] = dequantize_group(idx, hb, g.width, tab)
        e = k_pre[:, h] - khat                                      # [N, d]
        ea, eb = e[:, a], e[:, b]                                  # block members
        for gq in range(h * G, (h + 1) * G):
            qa, qb = q_pre[:, gq][:, a], q_pre[:, gq][:, b]
            # q^(i)T R(phi) e^(i) = cos(phi) (qa ea + qb eb) + sin(phi) (qb ea - qa eb),  phi = Delta * theta_i
            dot, cross = qa * ea + qb * eb, qb * ea - qa * eb     # [N, L]
            for D in offsets:
                phi = D * theta
                total += float(np.sum(np.abs(dot @ np.cos(phi) + cross @ np.sin(phi))))
                count += N
    return total / count

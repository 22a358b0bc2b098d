"""Thin ctypes binding of libbgtq.so (include/bgtq.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch supplies device memory
and streams.  There is NO CPU fallback: importing this module without a built libbgtq.so raises,
and every device entry point needs a CUDA tensor.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbgtq.so")

F32, BF16 = 0, 1
PAIR_HALF, PAIR_INTERLEAVED = 0, 1
QK_AVG, QK_MAX, QK_PRODUCT, K_ONLY, Q_ONLY = range(5)
TILE_TOKENS = 128

# every symbol include/bgtq.h declares (tests check the library exports each one)
SYMBOLS = [
    "bgtq_last_error", "bgtq_codebook", "bgtq_block_energy_workspace_bytes", "bgtq_block_energy",
    "bgtq_allocate", "bgtq_layout_create", "bgtq_layout_destroy", "bgtq_cache_bytes",
    "bgtq_token_bytes", "bgtq_workspace_bytes", "bgtq_region_offset", "bgtq_tile_stride",
    "bgtq_quantize_append", "bgtq_quantize_append_layers", "bgtq_profile_decode",
    "bgtq_profile_decode_read", "bgtq_decode_attention", "bgtq_decode_attention_layers",
    "bgtq_prefill_workspace_bytes", "bgtq_prefill_attention", "bgtq_fp16_workspace_bytes", "bgtq_fp16_decode_attention", "bgtq_debug_decode_unit", "bgtq_launch_count",
    "bgtq_paged_cache_bytes", "bgtq_paged_pool_offset", "bgtq_quantize_append_paged", "bgtq_decode_attention_paged",
    "bgtq_quantize_append_rope",
    "bgtq_window_bytes", "bgtq_window_append", "bgtq_decode_attention_protected",
    "bgtq_layout_create_format", "bgtq_layout_format", "bgtq_codebook_exact",
    "bgtq_debug_microbench", "bgtq_debug_microbench_name",
    "bgtq_v_block_energy_workspace_bytes", "bgtq_v_block_energy", "bgtq_layout_create_kv",
    "bgtq_block_energy_static", "bgtq_block_energy_static_max_row_elems", "bgtq_debug_append_exact_only",
]
MICROBENCH_COUNT = 22
FORMAT_V1, FORMAT_V2 = 1, 2
CODEBOOK_EXACT = 0x100


class BgtqError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"bgtq error {code}: {msg}")
        self.code = code


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: build it with `python -m paper_2606_24033_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, f32, sz = C.c_void_p, C.c_int, C.c_int64, C.c_float, C.c_size_t
    lib.bgtq_last_error.restype = C.c_char_p
    lib.bgtq_last_error.argtypes = []
    lib.bgtq_launch_count.restype = i64
    lib.bgtq_launch_count.argtypes = []
    lib.bgtq_codebook.restype = i32
    lib.bgtq_codebook.argtypes = [i32, vp]
    lib.bgtq_block_energy_workspace_bytes.restype = sz
    lib.bgtq_block_energy_workspace_bytes.argtypes = [i32, i32, i32]
    lib.bgtq_block_energy.restype = i32
    lib.bgtq_block_energy.argtypes = [vp, i64, vp, i64, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp, sz, vp]
    lib.bgtq_block_energy_static.restype = i32
    lib.bgtq_block_energy_static.argtypes = [vp, i64, vp, i64, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp]
    lib.bgtq_debug_append_exact_only.restype = i32
    lib.bgtq_debug_append_exact_only.argtypes = [i32]
    lib.bgtq_block_energy_static_max_row_elems.restype = i32
    lib.bgtq_block_energy_static_max_row_elems.argtypes = []
    lib.bgtq_v_block_energy_workspace_bytes.restype = sz
    lib.bgtq_v_block_energy_workspace_bytes.argtypes = [i32, i32]
    lib.bgtq_v_block_energy.restype = i32
    lib.bgtq_v_block_energy.argtypes = [vp, i64, i32, i32, i32, vp, vp, sz, vp]
    lib.bgtq_layout_create_kv.restype = i32
    lib.bgtq_layout_create_kv.argtypes = [vp, vp, i32, i32, i32, i32, i32, vp, i32, vp]
    lib.bgtq_allocate.restype = i32
    lib.bgtq_allocate.argtypes = [vp, i32, i32, i32, i32, i32, vp, i32, vp]
    lib.bgtq_layout_create.restype = i32
    lib.bgtq_layout_create.argtypes = [vp, i32, i32, i32, i32, i32, i32, vp, C.POINTER(vp)]
    lib.bgtq_layout_create_format.restype = i32
    lib.bgtq_layout_create_format.argtypes = [vp, i32, i32, i32, i32, i32, i32, vp, i32, C.POINTER(vp)]
    lib.bgtq_debug_microbench.restype = i32
    lib.bgtq_debug_microbench.argtypes = [i32, i32, C.POINTER(C.c_double)]
    lib.bgtq_debug_microbench_name.restype = C.c_char_p
    lib.bgtq_debug_microbench_name.argtypes = [i32]
    lib.bgtq_codebook_exact.restype = i32
    lib.bgtq_codebook_exact.argtypes = [i32, i32, vp]
    lib.bgtq_layout_format.restype = i32
    lib.bgtq_layout_format.argtypes = [vp]
    lib.bgtq_layout_destroy.restype = None
    lib.bgtq_layout_destroy.argtypes = [vp]
    lib.bgtq_cache_bytes.restype = sz
    lib.bgtq_cache_bytes.argtypes = [vp, i32, i64]
    lib.bgtq_token_bytes.restype = C.c_double
    lib.bgtq_token_bytes.argtypes = [vp, i32, i32]
    lib.bgtq_workspace_bytes.restype = sz
    lib.bgtq_workspace_bytes.argtypes = [vp, i32, i32]
    lib.bgtq_region_offset.restype = i64
    lib.bgtq_region_offset.argtypes = [vp, i32, i32, i32, i32, i64]
    lib.bgtq_tile_stride.restype = i64
    lib.bgtq_tile_stride.argtypes = [vp, i32, i32]
    lib.bgtq_quantize_append.restype = i32
    lib.bgtq_quantize_append.argtypes = [vp, i32, vp, vp, vp, i32, i32, i32, vp, i32, i64, vp]
    lib.bgtq_quantize_append_layers.restype = i32
    lib.bgtq_quantize_append_layers.argtypes = [vp, i32, i32, vp, vp, vp, i32, i32, i32, vp, i32, i64, vp]
    lib.bgtq_profile_decode.restype = None
    lib.bgtq_profile_decode.argtypes = [i32]
    lib.bgtq_profile_decode_read.restype = i32
    lib.bgtq_profile_decode_read.argtypes = [vp, vp]
    lib.bgtq_decode_attention.restype = i32
    lib.bgtq_decode_attention.argtypes = [vp, i32, vp, vp, vp, i32, i64, f32, vp, vp, sz, vp]
    lib.bgtq_decode_attention_layers.restype = i32
    lib.bgtq_decode_attention_layers.argtypes = [vp, i32, i32, vp, vp, vp, i32, i64, f32, vp, vp, sz, vp]
    lib.bgtq_prefill_workspace_bytes.restype = sz
    lib.bgtq_prefill_workspace_bytes.argtypes = [vp, i32, i32]
    lib.bgtq_prefill_attention.restype = i32
    lib.bgtq_prefill_attention.argtypes = [vp, i32, vp, vp, vp, i32, i32, i64, f32, vp, vp, sz, vp]
    lib.bgtq_fp16_workspace_bytes.restype = sz
    lib.bgtq_fp16_workspace_bytes.argtypes = [i32, i32, i32]
    lib.bgtq_fp16_decode_attention.restype = i32
    lib.bgtq_fp16_decode_attention.argtypes = [i32, i32, i32, i32, i32, vp, vp, vp, vp, i64, f32, vp, vp, sz, vp]
    lib.bgtq_debug_decode_unit.restype = i32
    lib.bgtq_debug_decode_unit.argtypes = [i32, vp, vp]
    lib.bgtq_paged_cache_bytes.restype = sz
    lib.bgtq_paged_cache_bytes.argtypes = [vp, i64]
    lib.bgtq_paged_pool_offset.restype = i64
    lib.bgtq_paged_pool_offset.argtypes = [vp, i32, i32, i64]
    lib.bgtq_quantize_append_paged.restype = i32
    lib.bgtq_quantize_append_paged.argtypes = [vp, i32, i32, vp, vp, vp, i32, i32, i32, vp, i32, vp, i32, i64, vp]
    lib.bgtq_quantize_append_rope.restype = i32
    lib.bgtq_quantize_append_rope.argtypes = [vp, i32, i32, vp, vp, vp, i32, i32, i32, vp, i32, i64, vp, vp, i64, vp]
    lib.bgtq_window_bytes.restype = sz
    lib.bgtq_window_bytes.argtypes = [vp, i32, i32, i32]
    lib.bgtq_window_append.restype = i32
    lib.bgtq_window_append.argtypes = [vp, i32, i32, vp, vp, i32, i32, i32, vp, i64, vp, vp, i32, i32, vp]
    lib.bgtq_decode_attention_protected.restype = i32
    lib.bgtq_decode_attention_protected.argtypes = [vp, i32, i32, vp, vp, vp, i32, i64, f32, vp, vp, i32, i32, vp, vp, sz, vp]
    lib.bgtq_decode_attention_paged.restype = i32
    lib.bgtq_decode_attention_paged.argtypes = [vp, i32, i32, vp, vp, vp, i32, vp, i32, i64, f32, vp, vp, sz, vp]
    return lib


_lib = _load()


def lib() -> C.CDLL:
    return _lib


def _check(rc: int) -> None:
    if rc != 0:
        raise BgtqError(rc, _lib.bgtq_last_error().decode())


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dev(t: torch.Tensor, dtype=None) -> int:
    if not t.is_cuda:
        raise ValueError("expected a CUDA tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError("expected a contiguous tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return t.data_ptr()


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.bfloat16:
        return BF16
    raise ValueError("activations must be float32 or bfloat16")


def launch_count() -> int:
    return int(_lib.bgtq_launch_count())


def codebook(b: int) -> np.ndarray:
    """bgtq_codebook: the 2^b fp16-representable Lloyd-Max levels (float32)."""
    out = np.zeros(1 << b, dtype=np.float32)
    _check(_lib.bgtq_codebook(b, out.ctypes.data))
    return out


def microbench(which: int, warps: int = 12):
    """bgtq_debug_microbench -> (name, value)."""
    v = C.c_double(0.0)
    _check(_lib.bgtq_debug_microbench(which, warps, C.byref(v)))
    return _lib.bgtq_debug_microbench_name(which).decode(), float(v.value)


def codebook_exact(b: int, m: int) -> np.ndarray:
    """bgtq_codebook_exact: the 2^b fp16-representable levels of C_{b,m} (exact-density codebook, float32)."""
    out = np.zeros(1 << b, dtype=np.float32)
    _check(_lib.bgtq_codebook_exact(b, m, out.ctypes.data))
    return out


def block_energy_workspace(n_q_heads: int, n_kv_heads: int, d_h: int, device="cuda") -> torch.Tensor:
    """Caller-owned scratch for block_energy / v_block_energy (reusable across calls)."""
    return torch.empty(int(_lib.bgtq_block_energy_workspace_bytes(n_q_heads, n_kv_heads, d_h)), dtype=torch.uint8, device=device)


def block_energy(q: torch.Tensor, k: torch.Tensor, pairing: int = PAIR_HALF, kind: int = QK_AVG,
                 return_parts: bool = False, workspace: Optional[torch.Tensor] = None):
    """bgtq_block_energy.  q [N_q, H_q, d_h], k [N_k, H_kv, d_h] (CUDA, same dtype) ->
    scores [H_kv, d_h/2] float32 (and Eq, Ek)."""
    nq, Hq, d = q.shape
    nk, Hkv, d2 = k.shape
    assert d == d2 and _dt(q) == _dt(k)
    L = d // 2
    scores = torch.empty((Hkv, L), dtype=torch.float32, device=k.device)
    eq = torch.empty_like(scores) if return_parts else None
    ek = torch.empty_like(scores) if return_parts else None
    nws = int(_lib.bgtq_block_energy_workspace_bytes(Hq, Hkv, d))
    ws = workspace if workspace is not None else torch.empty(nws, dtype=torch.uint8, device=k.device)
    nws = ws.numel()
    _check(_lib.bgtq_block_energy(_dev(q) if nq else None, nq, _dev(k) if nk else None, nk, _dt(k), Hq, Hkv, d,
                                  pairing, kind, _dev(scores), _dev(eq) if return_parts else None,
                                  _dev(ek) if return_parts else None, _dev(ws), nws, _stream()))
    return (scores, eq, ek) if return_parts else scores


def block_energy_static(q: torch.Tensor, k: torch.Tensor, scores: torch.Tensor, pairing: int = PAIR_HALF,
                        kind: int = QK_AVG, eq: Optional[torch.Tensor] = None, ek: Optional[torch.Tensor] = None) -> torch.Tensor:
    """bgtq_block_energy_static: block_energy without any allocation -- the caller passes the output tensor(s)
    [H_kv, d_h/2] float32, the scratch is the library's static 4 MiB device array (shared by all calls: do not overlap
    calls on the GPU).  Limit (H_q + H_kv) * d_h <= block_energy_static_max_row_elems()."""
    nq, Hq, d = q.shape
    nk, Hkv, d2 = k.shape
    assert d == d2 and _dt(q) == _dt(k) and scores.shape == (Hkv, d // 2)
    _check(_lib.bgtq_block_energy_static(_dev(q) if nq else None, nq, _dev(k) if nk else None, nk, _dt(k), Hq, Hkv, d,
                                         pairing, kind, _dev(scores, torch.float32),
                                         _dev(eq, torch.float32) if eq is not None else None,
                                         _dev(ek, torch.float32) if ek is not None else None, _stream()))
    return scores


def append_exact_only(on: bool) -> bool:
    """bgtq_debug_append_exact_only: force the exact fp64 append kernel for bulk appends (test / bench hook)."""
    return bool(_lib.bgtq_debug_append_exact_only(1 if on else 0))


def block_energy_static_max_row_elems() -> int:
    return int(_lib.bgtq_block_energy_static_max_row_elems())


V_BLOCK = 16


def v_block_energy(v: torch.Tensor, workspace: Optional[torch.Tensor] = None) -> torch.Tensor:
    """bgtq_v_block_energy.  v [N, H_kv, d_h] (CUDA) -> V-side scores [H_kv, d_h/16] float32."""
    n, Hkv, d = v.shape
    scores = torch.empty((Hkv, d // V_BLOCK), dtype=torch.float32, device=v.device)
    nws = int(_lib.bgtq_v_block_energy_workspace_bytes(Hkv, d))
    ws = workspace if workspace is not None else torch.empty(nws, dtype=torch.uint8, device=v.device)
    nws = ws.numel()
    _check(_lib.bgtq_v_block_energy(_dev(v), n, _dt(v), Hkv, d, _dev(scores), _dev(ws), nws, _stream()))
    return scores


def allocate(scores, total_bits: int, b_min: int, b_max: int):
    """bgtq_allocate.  scores [n_heads, L] float32: a CUDA tensor runs the device kernel and returns
    a CUDA uint8 tensor; a numpy array runs the library's host variant."""
    if isinstance(scores, torch.Tensor):
        n_heads, L = scores.shape
        bits = torch.empty((n_heads, L), dtype=torch.uint8, device=scores.device)
        _check(_lib.bgtq_allocate(_dev(scores, torch.float32), n_heads, L, b_min, b_max, total_bits,
                                  _dev(bits), 1, _stream()))
        return bits
    s = np.ascontiguousarray(scores, dtype=np.float32)
    n_heads, L = s.shape
    bits = np.zeros((n_heads, L), dtype=np.uint8)
    _check(_lib.bgtq_allocate(s.ctypes.data, n_heads, L, b_min, b_max, total_bits, bits.ctypes.data, 0, None))
    return bits


class Layout:
    """bgtq_layout: static metadata of the packed cache for an allocation bits[n_layers, H_kv, L]."""

    def __init__(self, bits: np.ndarray, n_q_heads: int, d_h: int, b_v: int, rotations: np.ndarray,
                 pairing: int = PAIR_HALF, fmt: int = FORMAT_V1, exact_codebooks: bool = False,
                 bits_v: np.ndarray | None = None):
        """bits_v [n_layers, H_kv, d_h/16] (V-side allocator, bgtq_layout_create_kv) replaces the uniform width b_v."""
        bits = np.ascontiguousarray(bits, dtype=np.uint8)
        assert bits.ndim == 3
        self.n_layers, self.n_kv_heads, _ = bits.shape
        self.n_q_heads, self.d_h, self.b_v = n_q_heads, d_h, b_v
        rot = np.ascontiguousarray(rotations, dtype=np.float32)
        h = C.c_void_p()
        flags = fmt | (CODEBOOK_EXACT if exact_codebooks else 0)
        if bits_v is not None:
            bits_v = np.ascontiguousarray(bits_v, dtype=np.uint8)
            assert bits_v.shape == (self.n_layers, self.n_kv_heads, d_h // V_BLOCK)
            _check(_lib.bgtq_layout_create_kv(bits.ctypes.data, bits_v.ctypes.data, self.n_layers, self.n_kv_heads,
                                              n_q_heads, d_h, pairing, rot.ctypes.data, flags, C.byref(h)))
        else:
            _check(_lib.bgtq_layout_create_format(bits.ctypes.data, self.n_layers, self.n_kv_heads, n_q_heads, d_h, b_v,
                                                  pairing, rot.ctypes.data, flags, C.byref(h)))
        self._h = h
        self.fmt = int(_lib.bgtq_layout_format(h)) & 0xFF
        self.exact_codebooks = bool(int(_lib.bgtq_layout_format(h)) & CODEBOOK_EXACT)

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:            # (module globals are already gone at interpreter shutdown)
            _lib.bgtq_layout_destroy(h)
            self._h = None

    def cache_bytes(self, batch: int, max_tokens: int) -> int:
        return int(_lib.bgtq_cache_bytes(self._h, batch, max_tokens))

    def token_bytes(self, layer: int, kv_head: int) -> float:
        return float(_lib.bgtq_token_bytes(self._h, layer, kv_head))

    def workspace_bytes(self, batch: int, n_layers: int = 1) -> int:
        return int(_lib.bgtq_workspace_bytes(self._h, batch, n_layers))

    def region_offset(self, layer: int, seq: int, kv_head: int, batch: int, max_tokens: int) -> int:
        return int(_lib.bgtq_region_offset(self._h, layer, seq, kv_head, batch, max_tokens))

    def paged_cache_bytes(self, n_pages: int) -> int:
        return int(_lib.bgtq_paged_cache_bytes(self._h, n_pages))

    def paged_pool_offset(self, layer: int, kv_head: int, n_pages: int) -> int:
        return int(_lib.bgtq_paged_pool_offset(self._h, layer, kv_head, n_pages))

    def tile_stride(self, layer: int, kv_head: int) -> int:
        return int(_lib.bgtq_tile_stride(self._h, layer, kv_head))

    def new_cache(self, batch: int, max_tokens: int, device="cuda") -> torch.Tensor:
        """Zero-initialised cache buffer (torch owns the memory)."""
        return torch.zeros(self.cache_bytes(batch, max_tokens), dtype=torch.uint8, device=device)

    def new_workspace(self, batch: int, n_layers: int = 1, device="cuda") -> torch.Tensor:
        return torch.empty(self.workspace_bytes(batch, n_layers), dtype=torch.uint8, device=device)


def quantize_append(layout: Layout, layer: int, cache: torch.Tensor, k_new: torch.Tensor,
                    v_new: torch.Tensor, seq_len: torch.Tensor, max_tokens: int,
                    advance_seq_len: bool = True, n_layers: int = 1) -> None:
    """bgtq_quantize_append (k_new, v_new [batch, n_new, H_kv, d_h]) or, with n_layers > 1,
    bgtq_quantize_append_layers ([n_layers, batch, n_new, H_kv, d_h]); seq_len int32 [batch] (CUDA)."""
    batch, n_new, Hkv, d = k_new.shape[-4:]
    assert v_new.shape == k_new.shape and Hkv == layout.n_kv_heads and d == layout.d_h
    assert _dt(k_new) == _dt(v_new)
    if k_new.dim() == 5:
        assert k_new.shape[0] == n_layers
        _check(_lib.bgtq_quantize_append_layers(layout._h, layer, n_layers, _dev(cache, torch.uint8), _dev(k_new),
                                                _dev(v_new), _dt(k_new), batch, n_new, _dev(seq_len, torch.int32),
                                                1 if advance_seq_len else 0, max_tokens, _stream()))
        return
    _check(_lib.bgtq_quantize_append(layout._h, layer, _dev(cache, torch.uint8), _dev(k_new), _dev(v_new),
                                     _dt(k_new), batch, n_new, _dev(seq_len, torch.int32),
                                     1 if advance_seq_len else 0, max_tokens, _stream()))


def quantize_append_rope(layout: Layout, layer: int, cache: torch.Tensor, k_pre: torch.Tensor, v_new: torch.Tensor,
                         seq_len: torch.Tensor, max_tokens: int, rope_cos: torch.Tensor, rope_sin: torch.Tensor,
                         advance_seq_len: bool = True, n_layers: int = 1) -> None:
    """bgtq_quantize_append_rope: PRE-RoPE k_pre [batch, n_new, H_kv, d_h] (n_layers = 1) or
    [n_layers, batch, n_new, H_kv, d_h]; rope_cos, rope_sin fp32 [rows >= max_tokens, d_h/2] (CUDA)."""
    batch, n_new, Hkv, d = k_pre.shape[-4:]
    assert v_new.shape == k_pre.shape and Hkv == layout.n_kv_heads and d == layout.d_h
    assert _dt(k_pre) == _dt(v_new)
    assert k_pre.dim() == 4 and n_layers == 1 or k_pre.dim() == 5 and k_pre.shape[0] == n_layers
    assert rope_cos.shape == rope_sin.shape and rope_cos.dim() == 2 and rope_cos.shape[1] == d // 2
    _check(_lib.bgtq_quantize_append_rope(layout._h, layer, n_layers, _dev(cache, torch.uint8), _dev(k_pre), _dev(v_new),
                                          _dt(k_pre), batch, n_new, _dev(seq_len, torch.int32),
                                          1 if advance_seq_len else 0, max_tokens, _dev(rope_cos, torch.float32),
                                          _dev(rope_sin, torch.float32), rope_cos.shape[0], _stream()))


def quantize_append_paged(layout: Layout, layer: int, cache: torch.Tensor, k_new: torch.Tensor,
                          v_new: torch.Tensor, seq_len: torch.Tensor, page_table: torch.Tensor, n_pages: int,
                          advance_seq_len: bool = True, n_layers: int = 1) -> None:
    """bgtq_quantize_append_paged: k_new, v_new [batch, n_new, H_kv, d_h] (n_layers = 1) or
    [n_layers, batch, n_new, H_kv, d_h]; page_table int32 [batch, table_stride] (CUDA)."""
    batch, n_new, Hkv, d = k_new.shape[-4:]
    assert v_new.shape == k_new.shape and Hkv == layout.n_kv_heads and d == layout.d_h
    assert _dt(k_new) == _dt(v_new)
    assert k_new.dim() == 4 and n_layers == 1 or k_new.dim() == 5 and k_new.shape[0] == n_layers
    assert page_table.dim() == 2 and page_table.shape[0] == batch
    _check(_lib.bgtq_quantize_append_paged(layout._h, layer, n_layers, _dev(cache, torch.uint8), _dev(k_new), _dev(v_new),
                                           _dt(k_new), batch, n_new, _dev(seq_len, torch.int32),
                                           1 if advance_seq_len else 0, _dev(page_table, torch.int32),
                                           page_table.shape[1], n_pages, _stream()))


def decode_attention_paged(layout: Layout, layer: int, cache: torch.Tensor, q: torch.Tensor, seq_len: torch.Tensor,
                           page_table: torch.Tensor, n_pages: int, softmax_scale: float, workspace: torch.Tensor,
                           out: Optional[torch.Tensor] = None, n_layers: int = 1) -> torch.Tensor:
    """bgtq_decode_attention_paged: q bf16 [batch, H_q, d_h] (n_layers = 1) or [n_layers, batch, H_q, d_h]."""
    if out is None:
        out = torch.empty_like(q)
    batch = q.shape[-3]
    assert q.shape[-2] == layout.n_q_heads and q.shape[-1] == layout.d_h
    assert q.dim() == 3 and n_layers == 1 or q.dim() == 4 and q.shape[0] == n_layers
    assert page_table.dim() == 2 and page_table.shape[0] == batch
    _check(_lib.bgtq_decode_attention_paged(layout._h, layer, n_layers, _dev(cache, torch.uint8), _dev(q, torch.bfloat16),
                                            _dev(seq_len, torch.int32), batch, _dev(page_table, torch.int32),
                                            page_table.shape[1], n_pages, float(softmax_scale),
                                            _dev(out, torch.bfloat16), _dev(workspace, torch.uint8),
                                            workspace.numel(), _stream()))
    return out


def profile_decode(enable: bool) -> None:
    _lib.bgtq_profile_decode(1 if enable else 0)


def profile_decode_read():
    """-> (summed milliseconds of the decode kernel alone, launches) since the last read."""
    ms, n = C.c_double(0.0), C.c_int(0)
    _check(_lib.bgtq_profile_decode_read(C.byref(ms), C.byref(n)))
    return float(ms.value), int(n.value)


def decode_attention(layout: Layout, layer: int, cache: torch.Tensor, q: torch.Tensor,
                     seq_len: torch.Tensor, max_tokens: int, softmax_scale: float,
                     workspace: torch.Tensor, out: Optional[torch.Tensor] = None,
                     n_layers: int = 1) -> torch.Tensor:
    """bgtq_decode_attention (n_layers = 1: q [batch, H_q, d_h]) or bgtq_decode_attention_layers
    (q [n_layers, batch, H_q, d_h], layers layer..layer+n_layers-1 in one launch).  bf16 in / out."""
    if out is None:
        out = torch.empty_like(q)
    batch = q.shape[-3]
    assert q.shape[-2] == layout.n_q_heads and q.shape[-1] == layout.d_h
    if q.dim() == 3:
        _check(_lib.bgtq_decode_attention(layout._h, layer, _dev(cache, torch.uint8), _dev(q, torch.bfloat16),
                                          _dev(seq_len, torch.int32), batch, max_tokens, float(softmax_scale),
                                          _dev(out, torch.bfloat16), _dev(workspace, torch.uint8),
                                          workspace.numel(), _stream()))
        return out
    assert q.shape[0] == n_layers
    _check(_lib.bgtq_decode_attention_layers(layout._h, layer, n_layers, _dev(cache, torch.uint8),
                                             _dev(q, torch.bfloat16), _dev(seq_len, torch.int32), batch,
                                             max_tokens, float(softmax_scale), _dev(out, torch.bfloat16),
                                             _dev(workspace, torch.uint8), workspace.numel(), _stream()))
    return out


def new_windows(layout: Layout, batch: int, n_sink: int, n_recent: int, device="cuda"):
    """Zeroed fp16 window buffers (win_k, win_v) [n_layers, batch, H_kv, n_sink + n_recent, d_h] (bgtq_window_bytes each)."""
    shape = (layout.n_layers, batch, layout.n_kv_heads, n_sink + n_recent, layout.d_h)
    assert int(_lib.bgtq_window_bytes(layout._h, batch, n_sink, n_recent)) == int(np.prod(shape)) * 2
    return torch.zeros(shape, dtype=torch.float16, device=device), torch.zeros(shape, dtype=torch.float16, device=device)


def window_append(layout: Layout, layer: int, k_new: torch.Tensor, v_new: torch.Tensor, seq_len: torch.Tensor,
                  win_k: torch.Tensor, win_v: torch.Tensor, n_sink: int, n_recent: int, n_layers: int = 1,
                  max_tokens: int = 2**31 - 1) -> None:
    """bgtq_window_append: k_new, v_new [batch, n_new, H_kv, d_h] (n_layers = 1) or [n_layers, batch, n_new, H_kv, d_h];
    call before the quantize_append that advances seq_len."""
    batch, n_new, Hkv, d = k_new.shape[-4:]
    assert v_new.shape == k_new.shape and Hkv == layout.n_kv_heads and d == layout.d_h and _dt(k_new) == _dt(v_new)
    assert k_new.dim() == 4 or k_new.shape[0] == n_layers
    _check(_lib.bgtq_window_append(layout._h, layer, n_layers, _dev(k_new), _dev(v_new), _dt(k_new), batch, n_new,
                                   _dev(seq_len, torch.int32), max_tokens, _dev(win_k, torch.float16),
                                   _dev(win_v, torch.float16), n_sink, n_recent, _stream()))


def decode_attention_protected(layout: Layout, layer: int, cache: torch.Tensor, q: torch.Tensor, seq_len: torch.Tensor,
                               max_tokens: int, softmax_scale: float, win_k: torch.Tensor, win_v: torch.Tensor,
                               n_sink: int, n_recent: int, workspace: torch.Tensor,
                               out: Optional[torch.Tensor] = None, n_layers: int = 1) -> torch.Tensor:
    """bgtq_decode_attention_protected: q bf16 [batch, H_q, d_h] (n_layers = 1) or [n_layers, batch, H_q, d_h]."""
    if out is None:
        out = torch.empty_like(q)
    batch = q.shape[-3]
    assert q.shape[-2] == layout.n_q_heads and q.shape[-1] == layout.d_h
    assert q.dim() == 3 or q.shape[0] == n_layers
    _check(_lib.bgtq_decode_attention_protected(layout._h, layer, n_layers, _dev(cache, torch.uint8), _dev(q, torch.bfloat16),
                                                _dev(seq_len, torch.int32), batch, max_tokens, float(softmax_scale),
                                                _dev(win_k, torch.float16), _dev(win_v, torch.float16), n_sink, n_recent,
                                                _dev(out, torch.bfloat16), _dev(workspace, torch.uint8), workspace.numel(),
                                                _stream()))
    return out


def prefill_attention(layout: Layout, layer: int, cache: torch.Tensor, q: torch.Tensor, seq_len: torch.Tensor,
                      max_tokens: int, softmax_scale: float, workspace: Optional[torch.Tensor] = None,
                      out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """bgtq_prefill_attention: causal attention of the last n_q cached tokens' queries.  q bf16 [batch, n_q, H_q, d_h]."""
    batch, n_q, Hq, d = q.shape
    assert Hq == layout.n_q_heads and d == layout.d_h
    if out is None:
        out = torch.empty_like(q)
    if workspace is None:
        workspace = torch.empty(int(_lib.bgtq_prefill_workspace_bytes(layout._h, batch, n_q)), dtype=torch.uint8, device=q.device)
    _check(_lib.bgtq_prefill_attention(layout._h, layer, _dev(cache, torch.uint8), _dev(q, torch.bfloat16),
                                       _dev(seq_len, torch.int32), batch, n_q, max_tokens, float(softmax_scale),
                                       _dev(out, torch.bfloat16), _dev(workspace, torch.uint8), workspace.numel(), _stream()))
    return out


def fp16_decode_attention(k_cache: torch.Tensor, v_cache: torch.Tensor, q: torch.Tensor, seq_len: torch.Tensor,
                          softmax_scale: float, workspace: Optional[torch.Tensor] = None,
                          out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """bgtq_fp16_decode_attention (comparison path).  k_cache, v_cache fp16 [n_layers, batch, H_kv, max_tokens, 128];
    q bf16 [n_layers, batch, H_q, 128]."""
    n_layers, batch, Hkv, max_tokens, d = k_cache.shape
    Hq = q.shape[-2]
    if out is None:
        out = torch.empty_like(q)
    if workspace is None:
        workspace = torch.empty(int(_lib.bgtq_fp16_workspace_bytes(batch, n_layers, Hkv)), dtype=torch.uint8, device=q.device)
    _check(_lib.bgtq_fp16_decode_attention(n_layers, batch, Hq, Hkv, d, _dev(k_cache, torch.float16), _dev(v_cache, torch.float16),
                                           _dev(q, torch.bfloat16), _dev(seq_len, torch.int32), max_tokens, float(softmax_scale),
                                           _dev(out, torch.bfloat16), _dev(workspace, torch.uint8), workspace.numel(), _stream()))
    return out


def debug_decode_unit(b: int, words: np.ndarray) -> np.ndarray:
    """Test hook: decode one unit (uint32 [b, 32] plane-major) with the kernel's unpack routine ->
    float32 [32 lanes, 32 slots]."""
    w = np.ascontiguousarray(words, dtype=np.uint32).reshape(b * 32)
    out = np.zeros((32, 32), dtype=np.float32)
    _check(_lib.bgtq_debug_decode_unit(b, w.ctypes.data, out.ctypes.data))
    return out

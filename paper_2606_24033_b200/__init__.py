"""B200-native Block-GTQ packed-cache decode path (arxiv/paper_2606_24033).

``paper_2606_24033_b200.binding`` is the thin ctypes layer over ``libbgtq.so`` (C-ABI in
``include/bgtq.h``); ``paper_2606_24033_b200.build`` compiles it in-tree.  The names of the
binding are re-exported lazily so that ``build`` can be imported before the library exists;
touching any of them without a built library raises ImportError (no CPU fallback).
"""
_BINDING_NAMES = (
    "Layout", "BgtqError", "block_energy", "block_energy_workspace", "block_energy_static", "block_energy_static_max_row_elems", "append_exact_only", "v_block_energy", "V_BLOCK", "allocate", "quantize_append", "decode_attention", "quantize_append_paged", "quantize_append_rope", "decode_attention_paged",
    "new_windows", "window_append", "decode_attention_protected",
    "codebook", "fp16_decode_attention", "prefill_attention", "debug_decode_unit", "profile_decode", "profile_decode_read", "launch_count", "lib", "SYMBOLS", "LIB_PATH",
    "F32", "BF16", "PAIR_HALF", "PAIR_INTERLEAVED", "QK_AVG", "QK_MAX", "QK_PRODUCT", "K_ONLY",
    "Q_ONLY", "TILE_TOKENS", "FORMAT_V1", "FORMAT_V2", "CODEBOOK_EXACT", "codebook_exact", "microbench", "MICROBENCH_COUNT",
)


def __getattr__(name):
    if name in _BINDING_NAMES:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)

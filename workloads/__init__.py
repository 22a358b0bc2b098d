"""Seeded synthetic inputs for the Block-GTQ hot path.

This module serves BOTH the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2606_24033_b200/``).  It holds none of the method's arithmetic: no
quantiser, no codebook, no packing, no attention, and no RoPE on the CPU side (the GPU-resident
generator ``gpu_synth`` rotates its own keys -- they are inputs handed to both sides as given).  It only draws random numbers
(numpy ``default_rng``), names the workload shapes of ``BASELINE.json`` and rounds
arrays to the boundary dtypes.  Everything the method itself draws at random (the
TQ-MSE rotation) is produced here as an *input* and handed to both
sides as data.
"""
from .synth import (  # noqa: F401
    CONFIGS,
    WorkloadShape,
    block_scales,
    pre_rope_gaussian,
    values_gaussian,
    values_block_scaled,
    round_to_bf16,
    bf16_bits_to_f32,
    f32_to_bf16_bits,
    rotations,
    rotation_offsets,
    paper_like_scores,
)

"""Seeded synthetic inputs (Wan-2.2-shaped Q/K/V) shared by the oracle tests and the CUDA path.

This package holds input generation only: no attention arithmetic, no thresholds.
Neither `oracle/` nor `paper_2606_16317_b200/` is imported from here.
"""
from .generator import (  # noqa: F401
    CONFIGS,
    WorkloadConfig,
    bf16_bits_to_f64,
    f32_to_bf16_bits,
    make_head,
    make_qkv,
    num_tiles,
)

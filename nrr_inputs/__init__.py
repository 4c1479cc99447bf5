"""Seeded synthetic inputs for the block-matching hot path.

This package is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests/bench.
It holds none of the method's arithmetic (no variance, no NCC, no selection, no search): it only
manufactures volumes, masks and the parameter sets of the five BASELINE.json configs.
The recipe is stated in DESIGN.md ("Input recipe") and follows SURVEY.md section 8(d).
"""
from .configs import CONFIGS, BatchSetting, Config, batch_settings, get_config
from .generate import make_mask, make_pair, make_fixed, spherical_mask

__all__ = [
    "CONFIGS", "Config", "BatchSetting", "batch_settings", "get_config",
    "make_pair", "make_fixed", "make_mask", "spherical_mask",
]

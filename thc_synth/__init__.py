"""Seeded synthetic inputs for the THC-RR-CCSD doubles-residual hot path.

This module holds NO arithmetic of the method itself: it only draws the input
tensors (BASELINE.json `configs`; recipe restated in DESIGN.md section 4).  It is
the one module both the CPU oracle tests and the CUDA path tests may import.
"""
from .generators import (CONFIGS, ThcInputs, make_inputs, make_config, config_dims,
                         normal_block, uniform_block, bvv_block, TENSOR_IDS, LazyCholesky)

__all__ = ["CONFIGS", "ThcInputs", "make_inputs", "make_config", "config_dims",
           "normal_block", "uniform_block", "bvv_block", "TENSOR_IDS", "LazyCholesky"]

"""Seeded synthetic inputs for the grouped-MoE-layer hot path (shared by oracle tests, GPU tests, bench).

This module holds NONE of the method's arithmetic (no router, no top-k, no FFN): it only draws
tensors, group maps and router biases from seeded generators, with the shapes and distributions of
BASELINE.json's configs (recipe: DESIGN.md "Input recipe").  Both the CPU oracle
(`oracle/`) and the CUDA path (`paper_2607_04164_b200/`) are fed from here; neither imports the
other.

The paper's own workloads (Qwen1.5-MoE-A2.7B on ShareGPT / Alpaca) are not in
this container; these synthetic layers stand in for them.
"""
from .configs import LayerConfig, CONFIGS, sweep_points, get_config
from .generate import (
    make_group_map,
    make_router_bias,
    make_cold_mask,
    make_layer,
    identity_variant,
    bf16_bits,
)

__all__ = [
    "LayerConfig",
    "CONFIGS",
    "sweep_points",
    "get_config",
    "make_group_map",
    "make_router_bias",
    "make_cold_mask",
    "make_layer",
    "identity_variant",
    "bf16_bits",
]

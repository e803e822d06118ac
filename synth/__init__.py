"""Seeded synthetic inputs shared by the CUDA path and the CPU oracle.

This module holds NO arithmetic of the method (no norm, attention, routing, cache
logic): only model shapes (BASELINE.json configs 1-5), seeded random weights and
seeded random prompts.  Both `oracle/` and `paper_2410_22134_b200/` are fed from
here; neither imports the other.
"""
from .configs import Shape, RunConfig, CONFIGS, get_config, expert_elems, expert_bytes, moe_layer_ids, mini
from .weights import Weights, make_weights, make_prompt, make_decode_ids

__all__ = [
    "Shape", "RunConfig", "CONFIGS", "get_config", "expert_elems", "expert_bytes", "moe_layer_ids", "mini",
    "Weights", "make_weights", "make_prompt", "make_decode_ids",
]

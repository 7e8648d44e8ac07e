"""Seeded synthetic inputs and weights for the candidate evaluator.

This package is DATA only: configs, random draws, bf16 rounding of the drawn
weights and the weight-file writer.  It holds none of the method's arithmetic
(no embedding, transition, scorer or top-k code) and imports neither `oracle/`
nor the CUDA package, so both sides can consume exactly the same inputs.

Recipe and draw order: SURVEY.md §8(d), restated in DESIGN.md §4.
"""
from .configs import WMConfig, CONFIGS, get_config
from .weights import make_weights, write_weight_file, round_to_bf16, tensor_order
from .inputs import make_inputs, Batch

__all__ = [
    "WMConfig", "CONFIGS", "get_config", "make_weights", "write_weight_file",
    "round_to_bf16", "tensor_order", "make_inputs", "Batch",
]

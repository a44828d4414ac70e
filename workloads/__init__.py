"""Seeded synthetic input generators shared by the tests, bench.py, the oracle
legs and the CUDA path.

This package holds NONE of the method's arithmetic (no scoring, selection,
softmax-attention or quantisation): it only draws seeded random tensors with
the shapes and structure of the paper's decode / prefill workloads
(DESIGN.md section 5 states each recipe) and rounds them once to BF16 bit
patterns, so the oracle and the GPU library read the very same bits.
"""
from .bf16 import f32_to_bf16_bits, bf16_bits_to_f32  # noqa: F401
from .decode import DecodeWorkload, make_decode_workload, CONFIGS, make_config  # noqa: F401
from .prefill import PrefillWorkload, make_prefill_workload  # noqa: F401
from .project import make_project_workload  # noqa: F401

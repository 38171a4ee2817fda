"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the oracle-side tests and the CUDA-side
tests/bench.  It holds none of the method's arithmetic: it draws shapes and
values, and stores them in the storage dtype (fp32, or bf16 as raw uint16
bits).  Recipe and readings: DESIGN.md "Input recipe" (SURVEY.md 8(c) Q7, Q8,
Q15, Q22).
"""
from .gen import (  # noqa: F401
    BF16, F32,
    bf16_bits_from_f32, f32_from_bf16_bits,
    tensor_normal, tensor_uniform,
    config0, config1, config2, config3, config4,
    listing2_example,
)

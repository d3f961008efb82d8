"""Seeded synthetic inputs for the BASE-Q W4A4 linear hot path.

This package is the ONLY code shared by the oracle side (oracle/, tests/) and the CUDA
side (paper_2506_15689_b200, bench.py).  It holds data synthesis only -- random draws,
the outlier / channel-mean structure of the paper's activation model (Eq. 1 P:54-58,
section 3.2), bf16 storage rounding and the int4 RTN draw of the weight operand
(BASELINE.json: "W is int4 per-output-channel symmetric, drawn by quantizing a N(0, 0.02)
fp32 matrix").  None of the hot path's arithmetic (activation quantizer, GEMM, epilogue)
lives here, and it imports neither oracle/ nor the product package.

The recipe for every config is stated in DESIGN.md section "Input recipe".
"""
from .synth import (  # noqa: F401
    CONFIGS,
    LayerSpec,
    bf16_bits_to_f32,
    f32_to_bf16_bits,
    layer_specs,
    make_layer,
    make_weights,
    make_activations,
    unpack_nibbles,
)

"""CPU oracle for the BASE-Q W4A4 linear hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2506_15689_b200 and never
imports it.  The arithmetic lives in baseq_oracle.cpp (plain single-threaded C++17);
this package only builds that file with g++ and marshals numpy arrays through ctypes.
"""
from .binding import (  # noqa: F401
    build,
    bf16_from_double,
    hadamard_blocks,
    quantize_act,
    fused_bias,
    gemm_i32,
    epilogue,
    linear,
    quantize_act_asym,
    gemm_i32_asym,
    epilogue_asym,
    linear_asym,
    quantize_kv,
    dense_hadamard_u64,
    dense_mode_bounds,
    dense_mode_check,
)

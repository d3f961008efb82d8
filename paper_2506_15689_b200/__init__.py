"""paper_2506_15689_b200 -- B200-native W4A4 linear hot path of BASE-Q (arxiv 2506.15689).

Thin Python binding over the C-ABI library libbaseq.so (include/baseq.h).  Argument
marshalling only: every step of the path runs in the CUDA kernels under csrc/.  There is no
CPU fallback -- importing works anywhere (the library is built in-tree by build.py), but
every compute call raises BaseqError unless it runs on an sm_100 device.
"""
from .binding import (  # noqa: F401
    ActParams,
    BaseqError,
    PackedWeight,
    lib,
    lib_path,
    linear,
    linear_fused,
    linear_fused_asym,
    linear_host,
    linear_host_scratch_bytes,
    linear_static,
    linear_static_scratch_bytes,
    pack_weights,
    quantize_act,
    quantize_act_asym,
    quantize_act_tc,
    w4a4_gemm_asym,
    quantize_kv,
    sync_status,
    w4a4_gemm,
    EXPORTED_SYMBOLS,
)

"""CPU-only checks (-m "not gpu"): the C-ABI library loads and exports every symbol
include/baseq.h declares, host-side argument validation returns the documented status codes
before any launch, the bench's multi-rank plumbing works over gloo, and the input recipe has
the statistics DESIGN.md states.  No compute call is made here (there is no CPU fallback)."""
import ctypes
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    import paper_2506_15689_b200 as bq
    return bq, bq.lib()


def test_header_symbols_are_exported():
    bq, L = _lib()
    header = open(os.path.join(ROOT, "include", "baseq.h")).read()
    declared = set(re.findall(r"\b(baseq_[a-z0-9_]+)\s*\(", header))
    declared -= {"baseq_status_t", "baseq_act_params_t"}
    assert declared == set(bq.EXPORTED_SYMBOLS), declared ^ set(bq.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    # nothing but the ABI is visible (internal launchers are hidden)
    out = subprocess.run(["nm", "-D", "--defined-only", bq.lib_path()], capture_output=True,
                         text=True).stdout
    exported = {l.split()[-1] for l in out.splitlines() if " T " in l}
    assert {e for e in exported if e.startswith("baseq_")} == declared
    assert not [e for e in exported if "launch_" in e]


def test_version_and_status_strings():
    _, L = _lib()
    assert L.baseq_version() >= 2
    seen = set()
    for code in range(8):
        s = L.baseq_status_string(code).decode()
        assert s.startswith("BASEQ_") and s not in seen
        seen.add(s)


def test_size_queries_and_blob_layout():
    _, L = _lib()
    assert L.baseq_packed_weight_bytes(7, 256) == 0            # N % 8
    assert L.baseq_packed_weight_bytes(8, 200) == 0            # K % 128
    for N, K in [(8, 128), (256, 256), (4096, 4096), (11008, 4096), (8192, 28672)]:
        nb = L.baseq_packed_weight_bytes(N, K)
        npad = -(-N // 192) * 192                               # tile N extent
        assert nb == 128 + 12 * npad + npad * K // 2
    assert L.baseq_fused_workspace_bytes(0, 8, 128) == 0
    assert L.baseq_fused_workspace_bytes(16, 256, 256) == 512 + 16 * 128     # control + counters + codes [T, K/2]
    assert L.baseq_fused_workspace_bytes(4096, 8192, 28672) == 512 + 4096 * 14336
    assert L.baseq_linear_host_scratch_bytes(16, 256, 256) >= 16 * 256 * 2 + 16 * 128 + 64 + 16 * 256 * 2


def test_validation_happens_before_any_launch():
    """NULL / shape / alignment / parameter errors are reported without touching a device."""
    bq, L = _lib()
    P = bq.binding._ActParamsC
    ok = P(0.9, 1.0, None, None, 0)
    buf = ctypes.create_string_buffer(4096 + 256)
    base = (ctypes.addressof(buf) + 255) // 256 * 256           # 256-byte aligned fake pointer
    q = L.baseq_quantize_act
    assert q(None, 256, 4, 256, ctypes.byref(ok), base, base, None) == 1          # NULL
    assert q(base, 256, 0, 256, ctypes.byref(ok), base, base, None) == 2          # empty T
    assert q(base, 200, 4, 200, ctypes.byref(ok), base, base, None) == 2          # K % 128
    assert q(base, 65536, 4, 65536, ctypes.byref(ok), base, base, None) == 2      # K too long
    assert q(base, 128, 4, 256, ctypes.byref(ok), base, base, None) == 3          # ldx < K
    assert q(base + 2, 256, 4, 256, ctypes.byref(ok), base, base, None) == 3      # misaligned x
    for bad in (P(0.0, 1.0, None, None, 0), P(1.5, 1.0, None, None, 0), P(0.9, -1.0, None, None, 0),
                P(0.9, float("nan"), None, None, 0), P(0.9, 1.0, None, None, 96),
                P(0.9, 1.0, None, None, 512)):
        assert q(base, 256, 4, 256, ctypes.byref(bad), base, base, None) == 4
    g = L.baseq_w4a4_gemm
    assert g(base, base, None, 4, 8, 128, base, 8, None, None) == 1
    assert g(base, base, base, 4, 12, 128, base, 16, None, None) == 2             # N % 8
    assert g(base, base, base, 4, 8, 128, base, 4, None, None) == 3               # ldy < N
    f = L.baseq_linear_fused
    assert f(base, 256, 4, 256, ctypes.byref(ok), base, 8, base, 8, base, 0, None, base, None,
             None) == 5                                                            # workspace
    # the fused and the host-buffer entry points run every check of BOTH stages before the first
    # launch or copy (a failing call enqueues nothing): these all fail before the device is queried
    assert f(base, 256, 4, 256, ctypes.byref(ok), base, 8, base, 8, base, 512, None, base, None,
             None) == 5                                   # workspace = control 256 + counters 256 + codes 512
    bad_alpha = P(0.0, 1.0, None, None, 0)
    assert f(base, 256, 4, 256, ctypes.byref(bad_alpha), base, 8, base, 8, base, 4096, None, base, None,
             None) == 4
    assert f(base, 256, 4, 256, ctypes.byref(ok), base, 12, base, 16, base, 4096, None, base, None,
             None) == 2                                                            # N % 8 (second stage)
    fa = L.baseq_linear_fused_asym
    assert fa(base, 256, 4, 256, ctypes.byref(ok), base, 8, base, 8, base, 4096, None, base, None, None,
              None) == 1                                                           # zeros_out required
    assert fa(base, 256, 4, 256, ctypes.byref(bad_alpha), base, 8, base, 8, base, 4096, None, base, base,
              None, None) == 4
    assert fa(base, 256, 4, 256, ctypes.byref(ok), base, 8, base, 8, base, 512, None, base, base, None,
              None) == 5
    h = L.baseq_linear_host
    assert h(base, 4, 256, ctypes.byref(bad_alpha), base, 8, base, base, 1 << 20, None) == 4
    assert h(base, 4, 65536, ctypes.byref(ok), base, 8, base, base, 1 << 30, None) == 2
    assert h(base, 4, 256, ctypes.byref(ok), base, 8, base, base, 16, None) == 5   # scratch too small
    assert g(base, base, base, 4, 8, 65536, base, 8, None, None) == 2              # K <= 32768 everywhere
    assert L.baseq_packed_weight_bytes(8, 65536) == 0
    assert L.baseq_pack_weights(base, base, None, None, 8, 128, base + 16, None, None) == 3
    kv = L.baseq_quantize_kv
    assert kv(None, 1024, 4, 8, 128, 1.0, base, base, base, None) == 1               # NULL
    assert kv(base, 1024, 0, 8, 128, 1.0, base, base, base, None) == 2               # empty T
    assert kv(base, 768, 4, 8, 96, 1.0, base, base, base, None) == 6                 # head_dim
    assert kv(base, 1024, 4, 8, 128, 0.0, base, base, base, None) == 4               # alpha
    assert kv(base, 512, 4, 8, 128, 1.0, base, base, base, None) == 3                # ldx < H * D
    assert kv(base + 2, 1024, 4, 8, 128, 1.0, base, base, base, None) == 3           # misaligned x


def test_no_cpu_fallback_without_a_device():
    """Without an sm_100 device every compute entry point refuses (UNSUPPORTED or CUDA error)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    bq, L = _lib()
    P = bq.binding._ActParamsC
    ok = P(0.9, 1.0, None, None, 0)
    buf = ctypes.create_string_buffer(8192 + 256)
    base = (ctypes.addressof(buf) + 255) // 256 * 256
    st = L.baseq_quantize_act(base, 256, 4, 256, ctypes.byref(ok), base, base, None)
    assert st in (6, 7)
    assert np.all(np.frombuffer(buf, dtype=np.uint8) == 0)      # nothing was computed on the host


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2506_15689_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src, fn
                assert "_work/" not in src, fn


# ------------------------------------------------------------------------------- input recipe
def _kurtosis(a):
    a = a - a.mean()
    return float((a ** 4).mean() / (a ** 2).mean() ** 2)


def test_input_recipe_statistics():
    """The seeded generators have the value statistics DESIGN.md section 4 states."""
    from baseq_inputs import CONFIGS, make_activations, make_weights
    from baseq_inputs.synth import bf16_bits_to_f32, unpack_nibbles
    # c3 down: SiLU-gated product, heavy-tailed (kurtosis about 10)
    A = make_activations("c3", "x_down", T=64)
    x = bf16_bits_to_f32(A["x"]).astype(np.float64)
    assert 7.0 < _kurtosis(x - x.mean(axis=0, keepdims=True)) < 14.0
    # c5: Laplace(0, 1) around per-channel means (kurtosis 6, variance 2)
    A5 = make_activations("c5", "x_down", T=32)
    x5 = bf16_bits_to_f32(A5["x"]).astype(np.float64)
    c5 = x5 - bf16_bits_to_f32(A5["calib"]).astype(np.float64).mean(axis=0, keepdims=True)
    assert 4.5 < _kurtosis(c5) < 7.5 and 1.7 < c5.var() < 2.4
    assert A5["b"].shape == (28672,) and A5["b"].dtype == np.float32
    # c1: four outlier channels x20 (Eq. 1), b = column mean of gamma * X
    A1 = make_activations("c1", "x")
    x1 = bf16_bits_to_f32(A1["x"]).astype(np.float64)
    std = x1.std(axis=0)
    assert set(np.argsort(std)[-4:]) == {17, 101, 170, 233}
    assert np.allclose(A1["b"], (1.05 * x1).mean(axis=0), rtol=0, atol=1e-5)
    # weights: per-output-channel symmetric RTN int4 of N(0, 0.02^2): codes in [-8, 7], max |q| = 7
    W = make_weights("c1", "linear")
    q = unpack_nibbles(W["w_nibbles"])
    assert q.min() >= -8 and q.max() <= 7 and np.all(np.abs(q).max(axis=1) == 7)
    assert 0.005 < float(W["w_scale"].mean()) < 0.012      # ~ 0.02 * E[max of 256 |N(0,1)|] / 7
    # shapes follow BASELINE.json
    assert [(s.T, s.K, s.N) for s in CONFIGS["c3"]] == [(4096, 4096, 11008)] * 2 + [(4096, 11008, 4096)]
    assert (CONFIGS["c5"][0].T, CONFIGS["c5"][0].K, CONFIGS["c5"][0].N, CONFIGS["c5"][0].had_block) == \
        (4096, 28672, 8192, 128)


def test_generators_are_deterministic():
    from baseq_inputs import make_activations
    a = make_activations("c2", "x", T=8)
    b = make_activations("c2", "x", T=8)
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["b"], b["b"])

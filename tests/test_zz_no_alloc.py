"""baseq_linear_static (-m gpu): the two-kernel linear with its scratch (codes, scales) in the
library's static __device__ array -- the entry point for callers that cannot allocate.

Collected last on purpose (pytest -x: a failure here must not hide the parity tests).  Checks the new
entry point against the existing path (quantize_act + w4a4_gemm with caller buffers) bit for bit --
the tolerance every GPU test here uses -- on two calls in a row that share the array: a prefill
shape (ring quantiser + tcgen05 GEMM) followed by a smaller decode shape (register quantiser +
decode GEMM) whose rows must not see what the first call left behind, then the first again.
"""
import numpy as np
import pytest
import torch

from baseq_inputs import f32_to_bf16_bits

pytestmark = pytest.mark.gpu


def _case(bq, rng, T, K, N, had_block=0):
    x = f32_to_bf16_bits((0.5 * rng.standard_normal(K)[None, :] + rng.standard_normal((T, K)))
                         .astype(np.float32))
    x = torch.from_numpy(x.view(np.int16)).cuda().view(torch.bfloat16)
    wn = torch.from_numpy(rng.integers(0, 256, (N, K // 2), dtype=np.uint8)).cuda()
    ws = torch.from_numpy((0.002 + 0.001 * rng.random(N)).astype(np.float32)).cuda()
    b = torch.from_numpy((0.5 * rng.standard_normal(K)).astype(np.float32)).cuda()
    bias = torch.from_numpy((0.1 * rng.standard_normal(N)).astype(np.float32)).cuda()
    pw = bq.pack_weights(wn, ws, b, bias)
    params = bq.ActParams(0.9, 1.05, None, b, had_block)
    return x, pw, params


def _bits(t):
    return t.contiguous().view(torch.int16).cpu().numpy()


def test_linear_static_matches_the_two_kernel_path_on_consecutive_calls():
    import paper_2506_15689_b200 as bq
    assert torch.cuda.is_available()
    assert bq.linear_static_scratch_bytes() == (4 << 20) + 8192 * 4
    rng = np.random.default_rng(20250615)
    big = _case(bq, rng, 300, 4096, 520)            # 2 M tiles x 3 N tiles, ragged in both
    small = _case(bq, rng, 19, 512, 264, 128)       # decode-size, with the block Hadamard
    expect = {}
    for name, (x, pw, params) in (("big", big), ("small", small)):
        expect[name] = _bits(bq.linear(x, params, pw))
    bq.sync_status()
    for name, (x, pw, params) in (("big", big), ("small", small), ("big", big)):
        T = x.shape[0]
        y = torch.full((T, pw.N), float("nan"), dtype=torch.bfloat16, device="cuda")
        bq.linear_static(x, params, pw, y)          # back to back on one stream, no sync between
        got = _bits(y)
        assert np.array_equal(got, expect[name]), "%s: %d of %d outputs differ" % (
            name, int((got != expect[name]).sum()), got.size)
    bq.sync_status()


def test_linear_static_rejects_sizes_beyond_the_array():
    import paper_2506_15689_b200 as bq
    rng = np.random.default_rng(3)
    x, pw, params = _case(bq, rng, 8, 256, 64)
    L = bq.lib()
    import ctypes
    cs = params.c_struct()
    y = torch.empty((8, 64), dtype=torch.bfloat16, device="cuda")
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)

    def call(T, K, N):
        return L.baseq_linear_static(ctypes.c_void_p(x.data_ptr()), K, T, K, ctypes.byref(cs),
                                     ctypes.c_void_p(pw.blob.data_ptr()), N,
                                     ctypes.c_void_p(y.data_ptr()), N, st)

    # status codes only: these calls must return before anything is enqueued (the buffers are tiny)
    assert call(8193, 128, 64) == 5                  # T beyond the scales area
    assert call(2049, 4096, 64) == 5                 # T * K / 2 beyond 4 MiB
    assert call(4096, 4096, 64) == 5
    assert call(0, 256, 64) == 2                     # shape errors keep their own code
    with pytest.raises(bq.BaseqError):
        bq.linear_static(torch.empty((4100, 4096), dtype=torch.bfloat16, device="cuda"), params,
                         bq.PackedWeight(pw.blob, 64, 4096, None),
                         torch.empty((4100, 64), dtype=torch.bfloat16, device="cuda"))
    torch.cuda.synchronize()

"""ctypes binding of libbaseq.so.  Same names as include/baseq.h minus the `baseq_` prefix.

torch is used for device memory and the current stream only.
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libbaseq.so")
_lib = None

EXPORTED_SYMBOLS = [
    "baseq_status_string", "baseq_version", "baseq_sync_status", "baseq_packed_weight_bytes", "baseq_pack_weights",
    "baseq_set_fused_bias", "baseq_quantize_act", "baseq_quantize_act_tc", "baseq_w4a4_gemm",
    "baseq_fused_workspace_bytes", "baseq_linear_fused", "baseq_linear_host_scratch_bytes",
    "baseq_linear_host", "baseq_quantize_act_asym", "baseq_w4a4_gemm_asym", "baseq_quantize_kv",
    "baseq_linear_static_scratch_bytes", "baseq_linear_static", "baseq_linear_fused_asym",
]


class BaseqError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        msg = lib().baseq_status_string(self.status).decode()
        super().__init__("%s failed: %s" % (where, msg))


class _ActParamsC(ctypes.Structure):
    _fields_ = [("alpha", ctypes.c_float), ("gamma", ctypes.c_float),
                ("sa", ctypes.c_void_p), ("b", ctypes.c_void_p), ("had_block", ctypes.c_int)]


def lib_path():
    return _LIB_PATH


def lib():
    """Loads libbaseq.so (built by paper_2506_15689_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("libbaseq.so is missing: run `python paper_2506_15689_b200/build.py` "
                              "(there is no fallback path)")
        L = ctypes.CDLL(_LIB_PATH)
        c = ctypes
        vp, i32, i64, sz = c.c_void_p, c.c_int, c.c_int64, c.c_size_t
        L.baseq_status_string.restype = c.c_char_p
        L.baseq_status_string.argtypes = [i32]
        L.baseq_version.restype = i32
        L.baseq_version.argtypes = []
        L.baseq_sync_status.restype = i32
        L.baseq_sync_status.argtypes = [vp]
        L.baseq_packed_weight_bytes.restype = sz
        L.baseq_packed_weight_bytes.argtypes = [i32, i32]
        L.baseq_pack_weights.restype = i32
        L.baseq_pack_weights.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, vp]
        L.baseq_set_fused_bias.restype = i32
        L.baseq_set_fused_bias.argtypes = [vp, i32, i32, vp, vp]
        L.baseq_quantize_act.restype = i32
        L.baseq_quantize_act.argtypes = [vp, i64, i32, i32, c.POINTER(_ActParamsC), vp, vp, vp]
        L.baseq_quantize_act_tc.restype = i32
        L.baseq_quantize_act_tc.argtypes = [vp, i64, i32, i32, c.POINTER(_ActParamsC), vp, vp, vp]
        L.baseq_w4a4_gemm.restype = i32
        L.baseq_w4a4_gemm.argtypes = [vp, vp, vp, i32, i32, i32, vp, i64, vp, vp]
        L.baseq_fused_workspace_bytes.restype = sz
        L.baseq_fused_workspace_bytes.argtypes = [i32, i32, i32]
        L.baseq_linear_fused.restype = i32
        L.baseq_linear_fused.argtypes = [vp, i64, i32, i32, c.POINTER(_ActParamsC), vp, i32, vp,
                                         i64, vp, sz, vp, vp, vp, vp]
        L.baseq_linear_fused_asym.restype = i32
        L.baseq_linear_fused_asym.argtypes = [vp, i64, i32, i32, c.POINTER(_ActParamsC), vp, i32, vp,
                                              i64, vp, sz, vp, vp, vp, vp, vp]
        L.baseq_linear_host_scratch_bytes.restype = sz
        L.baseq_linear_host_scratch_bytes.argtypes = [i32, i32, i32]
        L.baseq_linear_host.restype = i32
        L.baseq_linear_host.argtypes = [vp, i32, i32, c.POINTER(_ActParamsC), vp, i32, vp, vp, sz, vp]
        L.baseq_quantize_act_asym.restype = i32
        L.baseq_quantize_act_asym.argtypes = [vp, i64, i32, i32, c.POINTER(_ActParamsC), vp, vp, vp, vp]
        L.baseq_w4a4_gemm_asym.restype = i32
        L.baseq_w4a4_gemm_asym.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, i64, vp, vp]
        L.baseq_quantize_kv.restype = i32
        L.baseq_quantize_kv.argtypes = [vp, i64, i32, i32, i32, c.c_float, vp, vp, vp, vp]
        L.baseq_linear_static_scratch_bytes.restype = sz
        L.baseq_linear_static_scratch_bytes.argtypes = []
        L.baseq_linear_static.restype = i32
        L.baseq_linear_static.argtypes = [vp, i64, i32, i32, c.POINTER(_ActParamsC), vp, i32, vp, i64, vp]
        _lib = L
    return _lib


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _p(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _check(status, where):
    if status != 0:
        raise BaseqError(status, where)


def sync_status():
    """Synchronises the current stream and raises BaseqError(BASEQ_ERR_WORKSPACE) if a GEMM since the
    last call found a packed blob that does not match its (N, K)."""
    _check(lib().baseq_sync_status(_stream()), "baseq_sync_status")


class ActParams:
    """Per-quantizer parameters of Eq. 15: alpha, gamma | sa[K], b[K], had_block."""

    def __init__(self, alpha, gamma=1.0, sa=None, b=None, had_block=0):
        self.alpha, self.gamma, self.sa, self.b, self.had_block = alpha, gamma, sa, b, had_block

    def c_struct(self):
        for t in (self.sa, self.b):
            if t is not None:
                assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        return _ActParamsC(self.alpha, self.gamma,
                           None if self.sa is None else self.sa.data_ptr(),
                           None if self.b is None else self.b.data_ptr(), self.had_block)


class PackedWeight:
    """Opaque packed weight blob (device uint8 tensor) + its logical shape."""

    def __init__(self, blob, N, K, fused_bias):
        self.blob, self.N, self.K, self.fused_bias = blob, N, K, fused_bias

    def set_fused_bias(self, fb):
        assert fb.is_cuda and fb.dtype == torch.float32 and fb.numel() == self.N
        _check(lib().baseq_set_fused_bias(_p(self.blob), self.N, self.K, _p(fb), _stream()),
               "baseq_set_fused_bias")
        self.fused_bias = fb.clone()


def pack_weights(w_nibbles, w_scale, b=None, layer_bias=None):
    """w_nibbles [N,K/2] uint8 cuda, w_scale [N] f32, b [K] f32|None, layer_bias [N] f32|None."""
    N, Kh = w_nibbles.shape
    K = 2 * Kh
    L = lib()
    nbytes = L.baseq_packed_weight_bytes(N, K)
    if nbytes == 0:
        raise BaseqError(2, "baseq_packed_weight_bytes")
    blob = torch.empty(nbytes, dtype=torch.uint8, device=w_nibbles.device)
    fb = torch.empty(N, dtype=torch.float32, device=w_nibbles.device)
    _check(L.baseq_pack_weights(_p(w_nibbles.contiguous()), _p(w_scale), _p(b), _p(layer_bias),
                                N, K, _p(blob), _p(fb), _stream()), "baseq_pack_weights")
    return PackedWeight(blob, N, K, fb)


def quantize_act(x, params, codes=None, scales=None):
    """x [T,K] bf16 cuda (row stride may exceed K).  Returns (codes [T,K/2] u8, scales [T] f32)."""
    T, K = x.shape
    assert x.dtype == torch.bfloat16 and x.stride(1) == 1
    if codes is None:
        codes = torch.empty((T, K // 2), dtype=torch.uint8, device=x.device)
    if scales is None:
        scales = torch.empty((T,), dtype=torch.float32, device=x.device)
    cs = params.c_struct()
    _check(lib().baseq_quantize_act(_p(x), x.stride(0), T, K, ctypes.byref(cs), _p(codes),
                                    _p(scales), _stream()), "baseq_quantize_act")
    return codes, scales


def quantize_act_tc(x, params, codes=None, scales=None):
    """NEXT-2: quantize_act with the block-128 Hadamard on the tensor cores (tolerance parity)."""
    T, K = x.shape
    assert x.dtype == torch.bfloat16 and x.stride(1) == 1
    if codes is None:
        codes = torch.empty((T, K // 2), dtype=torch.uint8, device=x.device)
    if scales is None:
        scales = torch.empty((T,), dtype=torch.float32, device=x.device)
    cs = params.c_struct()
    _check(lib().baseq_quantize_act_tc(_p(x), x.stride(0), T, K, ctypes.byref(cs), _p(codes),
                                       _p(scales), _stream()), "baseq_quantize_act_tc")
    return codes, scales


def w4a4_gemm(codes, scales, pw, y=None, acc_dump=None):
    """codes [T,K/2] u8, scales [T] f32, pw PackedWeight -> y [T,N] bf16."""
    T = codes.shape[0]
    if y is None:
        y = torch.empty((T, pw.N), dtype=torch.bfloat16, device=codes.device)
    _check(lib().baseq_w4a4_gemm(_p(codes), _p(scales), _p(pw.blob), T, pw.N, pw.K, _p(y),
                                 y.stride(0), _p(acc_dump), _stream()), "baseq_w4a4_gemm")
    return y


def quantize_act_asym(x, params):
    """NEXT-1: per-token asymmetric int4.  Returns (codes [T,K/2] u8 unsigned nibbles, scales, zeros)."""
    T, K = x.shape
    assert x.dtype == torch.bfloat16 and x.stride(1) == 1
    codes = torch.empty((T, K // 2), dtype=torch.uint8, device=x.device)
    scales = torch.empty((T,), dtype=torch.float32, device=x.device)
    zeros = torch.empty((T,), dtype=torch.float32, device=x.device)
    cs = params.c_struct()
    _check(lib().baseq_quantize_act_asym(_p(x), x.stride(0), T, K, ctypes.byref(cs), _p(codes),
                                         _p(scales), _p(zeros), _stream()), "baseq_quantize_act_asym")
    return codes, scales, zeros


def w4a4_gemm_asym(codes, scales, zeros, pw, y=None, acc_dump=None):
    T = codes.shape[0]
    if y is None:
        y = torch.empty((T, pw.N), dtype=torch.bfloat16, device=codes.device)
    _check(lib().baseq_w4a4_gemm_asym(_p(codes), _p(scales), _p(zeros), _p(pw.blob), T, pw.N, pw.K,
                                      _p(y), y.stride(0), _p(acc_dump), _stream()),
           "baseq_w4a4_gemm_asym")
    return y


def quantize_kv(x, n_heads, head_dim, alpha=1.0, codes=None, scales=None, zeros=None):
    """NEXT-3: KV-cache per-head asymmetric int4.  x bf16 [T, >= n_heads*head_dim] (row stride free).
    Returns (codes u8 [T, n_heads*head_dim/2], scales f32 [T, n_heads], zeros f32 [T, n_heads])."""
    T = x.shape[0]
    assert x.dtype == torch.bfloat16 and x.stride(1) == 1
    hd = n_heads * head_dim
    if codes is None:
        codes = torch.empty((T, hd // 2), dtype=torch.uint8, device=x.device)
    if scales is None:
        scales = torch.empty((T, n_heads), dtype=torch.float32, device=x.device)
    if zeros is None:
        zeros = torch.empty((T, n_heads), dtype=torch.float32, device=x.device)
    _check(lib().baseq_quantize_kv(_p(x), x.stride(0), T, n_heads, head_dim, alpha, _p(codes),
                                   _p(scales), _p(zeros), _stream()), "baseq_quantize_kv")
    return codes, scales, zeros


def linear(x, params, pw, y=None):
    """quantize_act followed by w4a4_gemm (the two-kernel path)."""
    codes, scales = quantize_act(x, params)
    return w4a4_gemm(codes, scales, pw, y)


def linear_fused(x, params, pw, y=None, codes_dump=None, acc_dump=None, scales=None, workspace=None):
    """Fused variant: one launch, background quantiser warps inside the GEMM kernel.  `workspace`
    (uint8, >= baseq_fused_workspace_bytes) may be reused between calls; allocated here if None."""
    T, K = x.shape
    L = lib()
    if y is None:
        y = torch.empty((T, pw.N), dtype=torch.bfloat16, device=x.device)
    if scales is None:
        scales = torch.empty((T,), dtype=torch.float32, device=x.device)
    ws = workspace
    if ws is None:
        ws = torch.empty(max(L.baseq_fused_workspace_bytes(T, pw.N, K), 256), dtype=torch.uint8,
                         device=x.device)
    cs = params.c_struct()
    _check(L.baseq_linear_fused(_p(x), x.stride(0), T, K, ctypes.byref(cs), _p(pw.blob), pw.N,
                                _p(y), y.stride(0), _p(ws), ws.numel(), _p(codes_dump), _p(scales),
                                _p(acc_dump), _stream()), "baseq_linear_fused")
    return y, scales


def linear_fused_asym(x, params, pw, y=None, codes_dump=None, acc_dump=None, scales=None, zeros=None,
                      workspace=None):
    """Fused single-launch variant with per-token asymmetric activations.  Returns (y, scales, zeros)."""
    T, K = x.shape
    L = lib()
    if y is None:
        y = torch.empty((T, pw.N), dtype=torch.bfloat16, device=x.device)
    if scales is None:
        scales = torch.empty((T,), dtype=torch.float32, device=x.device)
    if zeros is None:
        zeros = torch.empty((T,), dtype=torch.float32, device=x.device)
    ws = workspace
    if ws is None:
        ws = torch.empty(max(L.baseq_fused_workspace_bytes(T, pw.N, K), 256), dtype=torch.uint8,
                         device=x.device)
    cs = params.c_struct()
    _check(L.baseq_linear_fused_asym(_p(x), x.stride(0), T, K, ctypes.byref(cs), _p(pw.blob), pw.N,
                                     _p(y), y.stride(0), _p(ws), ws.numel(), _p(codes_dump), _p(scales),
                                     _p(zeros), _p(acc_dump), _stream()), "baseq_linear_fused_asym")
    return y, scales, zeros


def linear_host(x_host, params, pw, y_host, scratch):
    """x_host [T,K] bf16 pinned CPU tensor, y_host [T,N] bf16 pinned CPU tensor (e2e leg)."""
    T, K = x_host.shape
    cs = params.c_struct()
    _check(lib().baseq_linear_host(_p(x_host), T, K, ctypes.byref(cs), _p(pw.blob), pw.N,
                                   _p(y_host), _p(scratch), scratch.numel(), _stream()),
           "baseq_linear_host")
    return y_host


def linear_host_scratch_bytes(T, N, K):
    return lib().baseq_linear_host_scratch_bytes(T, N, K)


def linear_static_scratch_bytes():
    return lib().baseq_linear_static_scratch_bytes()


def linear_static(x, params, pw, y):
    """quantize_act + w4a4_gemm with the codes / scales in the library's static device array: the
    call allocates nothing (y is the caller's).  T * K / 2 <= 4 MiB, T <= 8192, else BaseqError."""
    T, K = x.shape
    assert x.dtype == torch.bfloat16 and x.stride(1) == 1
    assert y.dtype == torch.bfloat16 and y.stride(1) == 1 and tuple(y.shape) == (T, pw.N)
    cs = params.c_struct()
    _check(lib().baseq_linear_static(_p(x), x.stride(0), T, K, ctypes.byref(cs), _p(pw.blob), pw.N,
                                     _p(y), y.stride(0), _stream()), "baseq_linear_static")
    return y

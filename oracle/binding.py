"""ctypes marshalling for oracle/baseq_oracle.cpp.  TEST INFRASTRUCTURE, NOT PRODUCT.

No arithmetic of the method lives here: every function checks dtypes/shapes, allocates
numpy outputs and calls the C++ routine of the same name.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "baseq_oracle.cpp")
_LIB = os.path.join(_HERE, "libbaseq_oracle.so")
_lib = None

# -ffp-contract=off: the compiler must not fuse a*b+c; no -march/-ffast-math: every fp32
# line of the oracle is one correctly rounded IEEE operation (oracle contract).
_CXXFLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


def build(force=False):
    """Compile the oracle with g++ (no CUDA).  Returns the path of the shared object."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", *_CXXFLAGS, _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c = ctypes
        lib.oracle_bf16_from_double.restype = c.c_uint16
        lib.oracle_bf16_from_double.argtypes = [c.c_double]
        lib.oracle_hadamard_blocks.restype = None
        lib.oracle_hadamard_blocks.argtypes = [c.c_void_p, c.c_int, c.c_int]
        lib.oracle_quantize_act.restype = c.c_int
        lib.oracle_quantize_act.argtypes = [c.c_void_p, c.c_int64, c.c_int, c.c_int, c.c_float,
                                            c.c_float, c.c_void_p, c.c_void_p, c.c_int,
                                            c.c_void_p, c.c_void_p, c.c_void_p]
        lib.oracle_fused_bias.restype = c.c_int
        lib.oracle_fused_bias.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                                          c.c_int, c.c_int, c.c_void_p]
        lib.oracle_gemm_i32.restype = c.c_int
        lib.oracle_gemm_i32.argtypes = [c.c_void_p, c.c_void_p, c.c_int, c.c_int, c.c_int,
                                        c.c_void_p]
        lib.oracle_epilogue.restype = c.c_int
        lib.oracle_epilogue.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                                        c.c_int, c.c_int, c.c_void_p, c.c_void_p]
        lib.oracle_quantize_act_asym.restype = c.c_int
        lib.oracle_quantize_act_asym.argtypes = [c.c_void_p, c.c_int64, c.c_int, c.c_int, c.c_float,
                                                 c.c_float, c.c_void_p, c.c_void_p, c.c_int,
                                                 c.c_void_p, c.c_void_p, c.c_void_p]
        lib.oracle_gemm_i32_asym.restype = c.c_int
        lib.oracle_gemm_i32_asym.argtypes = [c.c_void_p, c.c_void_p, c.c_int, c.c_int, c.c_int,
                                             c.c_void_p, c.c_void_p]
        lib.oracle_epilogue_asym.restype = c.c_int
        lib.oracle_epilogue_asym.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                                             c.c_void_p, c.c_void_p, c.c_int, c.c_int, c.c_void_p,
                                             c.c_void_p]
        lib.oracle_dense_hadamard_u64.restype = c.c_int
        lib.oracle_dense_hadamard_u64.argtypes = [c.c_void_p, c.c_int64, c.c_int, c.c_int, c.c_float,
                                                  c.c_void_p, c.c_void_p, c.c_int, c.c_void_p, c.c_void_p]
        _lib = lib
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _chk(a, dtype, name):
    if a is None:
        return None
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous:
        raise TypeError("%s must be a C-contiguous numpy array of %s" % (name, np.dtype(dtype)))
    return a


def bf16_from_double(y):
    """bf16 bit pattern (int) of a Python float, one RNE rounding."""
    return int(_load().oracle_bf16_from_double(float(y)))


def hadamard_blocks(x, block):
    """In-place fp32 block Hadamard of a 1-D float32 array (Q1)."""
    _chk(x, np.float32, "x")
    if x.ndim != 1 or x.size % block:
        raise ValueError("x must be 1-D with length a multiple of block")
    _load().oracle_hadamard_blocks(_ptr(x), x.size, block)
    return x


def quantize_act(x_bf16, alpha, gamma=1.0, sa=None, b=None, had_block=0, return_u=False):
    """x_bf16: [T,K] uint16 bf16 bit patterns.  Returns (codes [T,K/2] u8, scales [T] f32[, u])."""
    _chk(x_bf16, np.uint16, "x_bf16")
    if x_bf16.ndim != 2:
        raise ValueError("x_bf16 must be [T,K]")
    T, K = x_bf16.shape
    _chk(sa, np.float32, "sa")
    _chk(b, np.float32, "b")
    for v, n in ((sa, "sa"), (b, "b")):
        if v is not None and v.shape != (K,):
            raise ValueError("%s must have shape [K]" % n)
    codes = np.empty((T, max(K // 2, 0)), dtype=np.uint8)
    scales = np.empty((T,), dtype=np.float32)
    u = np.empty((T, K), dtype=np.float32) if return_u else None
    rc = _load().oracle_quantize_act(_ptr(x_bf16), K, T, K, alpha, gamma, _ptr(sa), _ptr(b),
                                     had_block, _ptr(codes), _ptr(scales), _ptr(u))
    if rc:
        raise ValueError("oracle_quantize_act: invalid arguments (status %d)" % rc)
    return (codes, scales, u) if return_u else (codes, scales)


def fused_bias(w_nibbles, w_scale, b=None, layer_bias=None):
    """fb[n] = s_w[n] * sum_k qw[n,k] b[k] + bias[n]  (fp64 accumulate, fp32 result)."""
    _chk(w_nibbles, np.uint8, "w_nibbles")
    _chk(w_scale, np.float32, "w_scale")
    _chk(b, np.float32, "b")
    _chk(layer_bias, np.float32, "layer_bias")
    N, Kh = w_nibbles.shape
    fb = np.empty((N,), dtype=np.float32)
    rc = _load().oracle_fused_bias(_ptr(w_nibbles), _ptr(w_scale), _ptr(b), _ptr(layer_bias),
                                   N, 2 * Kh, _ptr(fb))
    if rc:
        raise ValueError("oracle_fused_bias: invalid arguments (status %d)" % rc)
    return fb


def gemm_i32(codes, w_nibbles):
    """acc[t,n] = sum_k qa[t,k] qw[n,k], int32, triple loop."""
    _chk(codes, np.uint8, "codes")
    _chk(w_nibbles, np.uint8, "w_nibbles")
    T, Kh = codes.shape
    N, Kh2 = w_nibbles.shape
    if Kh != Kh2:
        raise ValueError("K mismatch")
    acc = np.empty((T, N), dtype=np.int32)
    rc = _load().oracle_gemm_i32(_ptr(codes), _ptr(w_nibbles), T, N, 2 * Kh, _ptr(acc))
    if rc:
        raise ValueError("oracle_gemm_i32: invalid arguments (status %d)" % rc)
    return acc


def epilogue(acc, scales, w_scale, fb=None, return_y64=False):
    """Y = bf16_rne(fma(s_t*s_w[n], acc, fb[n])) in fp64.  Returns uint16 [T,N] (and y64)."""
    _chk(acc, np.int32, "acc")
    _chk(scales, np.float32, "scales")
    _chk(w_scale, np.float32, "w_scale")
    _chk(fb, np.float32, "fb")
    T, N = acc.shape
    y = np.empty((T, N), dtype=np.uint16)
    y64 = np.empty((T, N), dtype=np.float64) if return_y64 else None
    rc = _load().oracle_epilogue(_ptr(acc), _ptr(scales), _ptr(w_scale), _ptr(fb), T, N,
                                 _ptr(y), _ptr(y64))
    if rc:
        raise ValueError("oracle_epilogue: invalid arguments (status %d)" % rc)
    return (y, y64) if return_y64 else y


def linear(x_bf16, w_nibbles, w_scale, fb, alpha, gamma=1.0, sa=None, b=None, had_block=0):
    """quantize_act -> gemm_i32 -> epilogue.  Returns dict(codes, scales, acc, y, y64)."""
    codes, scales = quantize_act(x_bf16, alpha, gamma, sa, b, had_block)
    acc = gemm_i32(codes, w_nibbles)
    y, y64 = epilogue(acc, scales, w_scale, fb, return_y64=True)
    return {"codes": codes, "scales": scales, "acc": acc, "y": y, "y64": y64}


# ------------------------------------------------------------------ NEXT-1: asymmetric activations
def quantize_act_asym(x_bf16, alpha, gamma=1.0, sa=None, b=None, had_block=0):
    """Per-token asymmetric int4 (Eq. 4).  Returns (codes u8 [T,K/2] with UNSIGNED
    nibbles, scales [T] f32, zeros [T] f32 = the lattice lower bounds z_t)."""
    _chk(x_bf16, np.uint16, "x_bf16")
    T, K = x_bf16.shape
    _chk(sa, np.float32, "sa")
    _chk(b, np.float32, "b")
    codes = np.empty((T, K // 2), dtype=np.uint8)
    scales = np.empty((T,), dtype=np.float32)
    zeros = np.empty((T,), dtype=np.float32)
    rc = _load().oracle_quantize_act_asym(_ptr(x_bf16), K, T, K, alpha, gamma, _ptr(sa), _ptr(b),
                                          had_block, _ptr(codes), _ptr(scales), _ptr(zeros))
    if rc:
        raise ValueError("oracle_quantize_act_asym: invalid arguments (status %d)" % rc)
    return codes, scales, zeros


def quantize_kv(x_bf16, n_heads, head_dim, alpha=1.0):
    """NEXT-3: KV-cache "per-head asymmetric dynamic quantization", heads =
    contiguous column blocks of head_dim that never straddle groups.  Each (token, head)
    group is quantised by the asymmetric rule of Eq. 4 on its own min / max -- i.e.
    oracle_quantize_act_asym applied to the [T * n_heads, head_dim] view with gamma = 1, no bias.
    Returns (codes u8 [T, n_heads*head_dim/2], scales f32 [T, n_heads], zeros f32 [T, n_heads])."""
    _chk(x_bf16, np.uint16, "x_bf16")
    T, HD = x_bf16.shape
    if HD != n_heads * head_dim or head_dim % 2:
        raise ValueError("quantize_kv: x must be [T, n_heads * head_dim]")
    groups = np.ascontiguousarray(x_bf16).reshape(T * n_heads, head_dim)
    codes = np.empty((T * n_heads, head_dim // 2), dtype=np.uint8)
    scales = np.empty((T * n_heads,), dtype=np.float32)
    zeros = np.empty((T * n_heads,), dtype=np.float32)
    rc = _load().oracle_quantize_act_asym(_ptr(groups), head_dim, T * n_heads, head_dim, alpha, 1.0,
                                          None, None, 0, _ptr(codes), _ptr(scales), _ptr(zeros))
    if rc:
        raise ValueError("oracle_quantize_act_asym (kv view): invalid arguments (status %d)" % rc)
    return (codes.reshape(T, HD // 2), scales.reshape(T, n_heads), zeros.reshape(T, n_heads))


def gemm_i32_asym(codes, w_nibbles):
    """Unsigned activation codes x signed weights.  Returns (acc [T,N] i32, wsum [N] i32)."""
    _chk(codes, np.uint8, "codes")
    _chk(w_nibbles, np.uint8, "w_nibbles")
    T, Kh = codes.shape
    N = w_nibbles.shape[0]
    acc = np.empty((T, N), dtype=np.int32)
    wsum = np.empty((N,), dtype=np.int32)
    rc = _load().oracle_gemm_i32_asym(_ptr(codes), _ptr(w_nibbles), T, N, 2 * Kh, _ptr(acc), _ptr(wsum))
    if rc:
        raise ValueError("oracle_gemm_i32_asym: invalid arguments (status %d)" % rc)
    return acc, wsum


def epilogue_asym(acc, wsum, scales, zeros, w_scale, fb=None, return_y64=False):
    T, N = acc.shape
    y = np.empty((T, N), dtype=np.uint16)
    y64 = np.empty((T, N), dtype=np.float64) if return_y64 else None
    rc = _load().oracle_epilogue_asym(_ptr(acc), _ptr(wsum), _ptr(scales), _ptr(zeros), _ptr(w_scale),
                                      _ptr(fb), T, N, _ptr(y), _ptr(y64))
    if rc:
        raise ValueError("oracle_epilogue_asym: invalid arguments (status %d)" % rc)
    return (y, y64) if return_y64 else y


def linear_asym(x_bf16, w_nibbles, w_scale, fb, alpha, gamma=1.0, sa=None, b=None, had_block=0):
    codes, scales, zeros = quantize_act_asym(x_bf16, alpha, gamma, sa, b, had_block)
    acc, wsum = gemm_i32_asym(codes, w_nibbles)
    y, y64 = epilogue_asym(acc, wsum, scales, zeros, w_scale, fb, return_y64=True)
    return {"codes": codes, "scales": scales, "zeros": zeros, "acc": acc, "wsum": wsum, "y": y,
            "y64": y64}


# ------------------------------------------------------------------ NEXT-2: dense (tensor-core) Hadamard
def dense_hadamard_u64(x_bf16, had_block, gamma=1.0, sa=None, b=None):
    """Exact (fp64) u = g * (H_B x) / sqrt(B) - b per block of had_block channels, and the L1 norm of
    every block of x (the scale of a tensor core's accumulation error).  Returns (u64 [T,K], l1 [T,K/B])."""
    _chk(x_bf16, np.uint16, "x_bf16")
    T, K = x_bf16.shape
    _chk(sa, np.float32, "sa")
    _chk(b, np.float32, "b")
    u = np.empty((T, K), dtype=np.float64)
    l1 = np.empty((T, K // had_block), dtype=np.float64)
    rc = _load().oracle_dense_hadamard_u64(_ptr(x_bf16), K, T, K, gamma, _ptr(sa), _ptr(b), had_block,
                                           _ptr(u), _ptr(l1))
    if rc:
        raise ValueError("oracle_dense_hadamard_u64: invalid arguments (status %d)" % rc)
    return u, l1


def dense_mode_bounds(u64, l1, alpha, had_block, sa=None, gamma=1.0, eps=2.0 ** -16):
    """The acceptance band of the dense (tensor-core) Hadamard mode: a result u' is
    admissible iff |u' - u64| <= tol with tol[t,c] = eps * |g_c| * l1[t, block(c)] / sqrt(B) +
    2^-21 |u64| (accumulation error of block(c)'s 128-term sum, then two fp32 roundings).  Returns
    (tol [T,K], m_lo [T], m_hi [T]): the band of the row absmax."""
    T, K = u64.shape
    g = np.abs(sa.astype(np.float64)) if sa is not None else np.full(K, abs(float(gamma)))
    tol = eps * g[None, :] * np.repeat(l1, had_block, axis=1) / np.sqrt(float(had_block)) + 2.0 ** -21 * np.abs(u64)
    a = np.abs(u64)
    return tol, (a - tol).max(axis=1).clip(min=0.0), (a + tol).max(axis=1)


def dense_mode_check(codes, scales, u64, tol, m_lo, m_hi, alpha):
    """True iff (codes, scales) is an admissible output of the dense Hadamard mode: every scale is
    max((alpha m) / 7, 1e-12) for some absmax m inside [m_lo, m_hi] (up to the two fp32 roundings of
    Q4), and every code q satisfies clamp(rne(lo)) <= q <= clamp(rne(hi)) where [lo, hi] is the image
    of [u64 - tol, u64 + tol] under multiplication by the RECIPROCAL OF THE RETURNED SCALE, rounded
    as in Q5 (rounding is monotonic, so this says: some admissible u rounds to q).  Returns
    (ok, n_bad_scales, n_bad_codes)."""
    s = scales.astype(np.float64)
    a = np.float64(np.float32(alpha))
    floor = np.float64(np.float32(1e-12))
    s_lo = np.maximum(a * m_lo / 7.0, floor) * (1 - 2.0 ** -22)
    s_hi = np.maximum(a * m_hi / 7.0, floor) * (1 + 2.0 ** -22)
    bad_s = (s < s_lo) | (s > s_hi)
    inv = (np.float32(1.0) / scales.astype(np.float32)).astype(np.float64)[:, None]
    lo = (u64 - tol) * inv
    hi = (u64 + tol) * inv
    lo -= np.abs(lo) * 2.0 ** -22
    hi += np.abs(hi) * 2.0 ** -22
    q_lo = np.clip(np.rint(lo), -8, 7)
    q_hi = np.clip(np.rint(hi), -8, 7)
    lo_n = (codes & 0xF).astype(np.int16)
    hi_n = (codes >> 4).astype(np.int16)
    q = np.empty(u64.shape, dtype=np.int16)
    q[:, 0::2] = np.where(lo_n >= 8, lo_n - 16, lo_n)
    q[:, 1::2] = np.where(hi_n >= 8, hi_n - 16, hi_n)
    bad_q = (q < q_lo) | (q > q_hi)
    return (not bad_s.any()) and (not bad_q.any()), int(bad_s.sum()), int(bad_q.sum())

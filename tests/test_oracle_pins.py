"""Pins for the CPU oracle (-m "not gpu").

Each test checks oracle/ against something OTHER than itself: values the paper or SPEC.md
print, closed forms, exact rational arithmetic (Python fractions), brute force on tiny
inputs, library routines on special cases.  P:n / S:n = PAPER.md / SPEC.md line n.
"""
from fractions import Fraction
import json
import math
import os
import struct

import numpy as np
import pytest

import oracle
from baseq_inputs import bf16_bits_to_f32, f32_to_bf16_bits, unpack_nibbles

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def bf16(a):
    return f32_to_bf16_bits(np.asarray(a, dtype=np.float32))


def codes_to_int(codes):
    return unpack_nibbles(codes).astype(np.int32)


def pad_row(vals, K):
    row = np.zeros((1, K), dtype=np.float32)
    row[0, :len(vals)] = vals
    return row



def _round_f32(exact):
    """Round an exact Fraction to the nearest fp32 (ties to even) without double rounding."""
    approx = np.float32(float(exact))
    cands = [approx, np.nextafter(approx, np.float32(np.inf)),
             np.nextafter(approx, np.float32(-np.inf))]
    return min(cands, key=lambda c: (abs(Fraction(float(c)) - exact),
                                     int(np.float32(c).view(np.uint32)) & 1))


# --------------------------------------------------------------------------- bf16 rounding
def _bf16_exact(y):
    """bf16 RNE of a double via exact rational arithmetic (independent of the oracle)."""
    if y == 0:
        return 0x8000 if math.copysign(1.0, y) < 0 else 0
    sign = 0x8000 if y < 0 else 0
    a = Fraction(abs(y))
    e = math.floor(math.log2(abs(y)))
    while Fraction(2) ** e > a:
        e -= 1
    while Fraction(2) ** (e + 1) <= a:
        e += 1
    ulp_e = max(e - 7, -133)
    q = a / Fraction(2) ** ulp_e
    fl = q.numerator // q.denominator
    rem = q - fl
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl % 2 == 1):
        fl += 1
    val = Fraction(fl) * Fraction(2) ** ulp_e
    if val >= Fraction(2) ** 128:
        return sign | 0x7F80
    f = float(val)
    bits = struct.unpack("<I", struct.pack("<f", f))[0]
    assert float(struct.unpack("<f", struct.pack("<I", bits & 0xFFFF0000))[0]) == f
    return sign | (bits >> 16)


def test_bf16_from_double_against_exact_rational():
    rng = np.random.default_rng(0)
    vals = list(rng.standard_normal(2000) * 3.0)
    vals += list(rng.standard_normal(200) * 1e-3) + list(rng.standard_normal(200) * 1e4)
    # exact ties and their neighbours
    for base in (1.0, 2.0, 0.75, 100.0, -3.0):
        ulp = 2.0 ** (math.floor(math.log2(abs(base))) - 7)
        for k in range(0, 6):
            mid = base + (k + 0.5) * ulp
            vals += [mid, np.nextafter(mid, 1e9), np.nextafter(mid, -1e9)]
    vals += [2.0 ** -133, 1.5 * 2.0 ** -133, 0.5 * 2.0 ** -133, 2.0 ** -126, 2.0 ** -127 * 1.01,
             3.3895313892515355e38, 3.4e38, 0.0, -0.0]
    for v in vals:
        assert oracle.bf16_from_double(float(v)) == _bf16_exact(float(v)), v


def test_bf16_known_patterns():
    assert oracle.bf16_from_double(1.0) == 0x3F80
    assert oracle.bf16_from_double(-2.5) == 0xC020
    assert oracle.bf16_from_double(1.0 + 2.0 ** -8) == 0x3F80       # tie -> even (down)
    assert oracle.bf16_from_double(1.0 + 3 * 2.0 ** -8) == 0x3F82   # tie -> even (up)
    assert oracle.bf16_from_double(float("inf")) == 0x7F80


# --------------------------------------------------------------------------- Hadamard (Q1)
def _dense_hadamard(B):
    H = np.array([[1.0]])
    while H.shape[0] < B:
        H = np.block([[H, H], [H, -H]])
    return H


@pytest.mark.parametrize("B", [2, 8, 128])
def test_hadamard_small_integers_equal_dense_matrix_product(B):
    # small-integer inputs: every butterfly sum is exact in fp32, so the result must equal
    # the dense +-1 Sylvester matrix product times (float)(1/sqrt(B)) (Eq. 2).
    rng = np.random.default_rng(B)
    x = rng.integers(-8, 9, size=3 * B).astype(np.float32)
    want = np.concatenate([_dense_hadamard(B) @ x[i * B:(i + 1) * B].astype(np.float64)
                           for i in range(3)])
    c = np.float32(1.0 / math.sqrt(B))
    want = (want.astype(np.float32) * c).astype(np.float32)
    got = oracle.hadamard_blocks(x.copy(), B)
    assert np.array_equal(got, want)


def test_hadamard_one_hot_spreads_a_over_sqrt_n():
    # Eq. 2: a one-hot outlier a*e_i becomes a dense vector of magnitude a/sqrt(n).
    B = 128
    for i in (0, 5, 127):
        x = np.zeros(B, dtype=np.float32)
        x[i] = 64.0
        y = oracle.hadamard_blocks(x, B)
        assert np.array_equal(np.abs(y), np.full(B, np.float32(64.0) * np.float32(1 / math.sqrt(128)),
                                                 dtype=np.float32))
        assert np.array_equal(np.sign(y), _dense_hadamard(B)[:, i])


def test_hadamard_is_involution():
    # H H = I within 1e-6.
    rng = np.random.default_rng(3)
    x = rng.standard_normal(1024).astype(np.float32)
    y = oracle.hadamard_blocks(oracle.hadamard_blocks(x.copy(), 128), 128)
    assert np.max(np.abs(y - x)) < 1e-5


# --------------------------------------------------------------------------- quantizer
def _rtn_independent(xf, alpha):
    """Independent 6-line per-token symmetric RTN using numpy fp32 ops (QuaRot-style)."""
    m = np.max(np.abs(xf), axis=1).astype(np.float32)
    s = np.maximum((np.float32(alpha) * m) / np.float32(7.0), np.float32(1e-12)).astype(np.float32)
    inv = (np.float32(1.0) / s).astype(np.float32)
    r = xf.astype(np.float64) * inv[:, None].astype(np.float64)      # exact product, one rounding (C-17)
    q = np.clip(np.rint(r), -8, 7).astype(np.int32)
    return q, s


def test_quantizer_reduces_to_plain_rtn():
    # north_star: "with b=0 and gamma=1 it must reduce to plain RTN per-token quantization".
    rng = np.random.default_rng(1)
    x = bf16(rng.standard_normal((37, 384)) * 2.0)
    for alpha in (1.0, 0.9, 0.5):
        codes, scales = oracle.quantize_act(x, alpha)
        q, s = _rtn_independent(bf16_bits_to_f32(x), alpha)
        assert np.array_equal(codes_to_int(codes), q)
        assert np.array_equal(scales, s)


def test_quantizer_lattice_rows_exact():
    # integers -7..7, symmetric, alpha=1 -> s=1, all values exact.
    vals = np.arange(-7, 8, dtype=np.float32)
    x = bf16(pad_row(vals, 128))
    codes, scales = oracle.quantize_act(x, 1.0)
    assert scales[0] == np.float32(1.0)
    assert np.array_equal(codes_to_int(codes)[0, :15], np.arange(-7, 8))
    assert np.all(codes_to_int(codes)[0, 15:] == 0)
    # constant group -> codes +-7, dequantised value = c within 1 fp32 ulp.
    x = bf16(np.full((1, 128), 5.0, dtype=np.float32))
    codes, scales = oracle.quantize_act(x, 1.0)
    assert np.all(codes_to_int(codes) == 7)
    assert abs(float(scales[0]) * 7 - 5.0) <= np.spacing(np.float32(5.0))


def test_quantizer_tie_rule_is_half_to_even():
    # Reading C-6 (north_star) vs SPEC's half-away: 0.5->0, 1.5->2, 2.5->2, ...
    vals = [0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 7.0, 3.5, -3.5]
    x = bf16(pad_row(vals, 128))
    codes, scales = oracle.quantize_act(x, 1.0)
    assert scales[0] == np.float32(1.0)
    assert list(codes_to_int(codes)[0, :9]) == [0, 2, 2, 0, -2, -2, 7, 4, -4]


def test_quantizer_clip_and_range():
    # Eq. 4 P:74 clip; reading C-7: scale uses 7, clamp uses [-8, 7].
    vals = [14.0, 9.0, -9.0, -14.0, 7.4, -7.6, -8.4]
    x = bf16(pad_row(vals, 128))
    codes, scales = oracle.quantize_act(x, 0.5)
    assert scales[0] == np.float32(1.0)                       # 0.5 * 14 / 7
    assert list(codes_to_int(codes)[0, :7]) == [7, 7, -8, -8, 7, -8, -8]


def test_quantizer_nibble_packing_order():
    # D2: byte j = (q[2j] & 15) | ((q[2j+1] & 15) << 4).
    vals = [1.0, -1.0, 7.0, -7.0]
    x = bf16(pad_row(vals, 128))
    codes, _ = oracle.quantize_act(x, 1.0)
    assert codes[0, 0] == (1 | (0xF << 4))
    assert codes[0, 1] == (7 | (0x9 << 4))


def test_quantizer_zero_row_uses_floor():
    # Reading C-10 / S:224: all-equal (zero) row -> s = 1e-12, codes 0.
    x = bf16(np.zeros((2, 128), dtype=np.float32))
    codes, scales = oracle.quantize_act(x, 0.9)
    assert np.all(codes == 0)
    assert np.all(scales == np.float32(1e-12))


def test_quantizer_scale_then_bias_order():
    # Reading C-1: u = g*x - b (Eq. 15), NOT g*(x - b).
    x = bf16(pad_row([2.0, 4.0, -6.0], 128))
    b = np.zeros(128, dtype=np.float32)
    b[:3] = [1.0, 1.0, 1.0]
    _, _, u = oracle.quantize_act(x, 1.0, gamma=1.5, b=b, return_u=True)
    assert list(u[0, :3]) == [2.0, 5.0, -10.0]
    # per-channel vector s^a wins over gamma (reading C-2)
    sa = np.full(128, 2.0, dtype=np.float32)
    _, _, u = oracle.quantize_act(x, 1.0, gamma=1.5, sa=sa, b=b, return_u=True)
    assert list(u[0, :3]) == [3.0, 7.0, -13.0]


def test_quantizer_u_is_single_rounded_fma():
    # Q2 is ONE rounding: compare with exact rational g*x - b rounded once to fp32.
    rng = np.random.default_rng(5)
    K = 128
    x = bf16(rng.standard_normal((4, K)))
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    b = (0.3 * rng.standard_normal(K)).astype(np.float32)
    _, _, u = oracle.quantize_act(x, 0.9, sa=sa, b=b, return_u=True)
    xf = bf16_bits_to_f32(x)
    for t in range(4):
        for k in range(K):
            exact = Fraction(float(sa[k])) * Fraction(float(xf[t, k])) - Fraction(float(b[k]))
            assert u[t, k] == _round_f32(exact)


def test_reconstruction_within_half_step():
    # north_star: "the dequantised x-b plus b must reconstruct x within one quantization
    # step per element"; tighter here: |s_t q + b - g x| <= s_t/2 (1 + 2^-20) for in-range u.
    rng = np.random.default_rng(7)
    T, K = 32, 512
    mu = rng.standard_normal(K).astype(np.float32)
    x = bf16(mu[None, :] + rng.standard_normal((T, K)))
    b = mu.copy()
    for alpha in (1.0, 0.8):
        codes, scales, u = oracle.quantize_act(x, alpha, gamma=1.05, b=b, return_u=True)
        q = codes_to_int(codes).astype(np.float64)
        gx = 1.05 * bf16_bits_to_f32(x).astype(np.float64)
        rec = scales[:, None].astype(np.float64) * q + b[None, :].astype(np.float64)
        inrange = np.abs(u).astype(np.float64) <= 7.0 * scales[:, None].astype(np.float64) * (1 + 1e-6)
        err = np.abs(rec - gx)
        bound = scales[:, None].astype(np.float64) / 2 * (1 + 2.0 ** -20) + 1e-6 * np.abs(gx)
        assert np.all(err[inrange] <= bound[inrange])
        if alpha == 1.0:
            assert inrange.all()
        else:
            assert (~inrange).any()
            assert np.all(np.abs(q[~inrange]) >= 7)


def test_rounding_energy_is_s2_over_12():
    # P:79 "E||eps_round||^2 = s^2/12"; S:238 / acceptance S:583: within 5% at 1e6 samples.
    rng = np.random.default_rng(11)
    T, K = 512, 2048
    xf = rng.uniform(-7.0, 7.0, size=(T, K)).astype(np.float32)
    xf[:, 0] = 7.0          # pins absmax = 7 -> s_t = 1 with alpha = 1
    x = bf16(xf)
    codes, scales = oracle.quantize_act(x, 1.0)
    assert np.all(scales == np.float32(1.0))
    err = codes_to_int(codes).astype(np.float64) - bf16_bits_to_f32(x).astype(np.float64)
    mse = np.mean(err[:, 1:] ** 2)
    assert abs(mse - 1.0 / 12.0) < 0.05 / 12.0


def test_bias_correction_removes_variance_of_means():
    # Eq. 6: sigma^2 = mean_j sigma_j^2 + Var(mu_j).  With b = channel means the
    # quantizer input u has var-of-means fraction < 0.01, and the mean squared
    # step shrinks accordingly (Eq. 5 P:118-122 "s^2 prop. to sigma^2").
    rng = np.random.default_rng(13)
    T, K = 256, 1024
    mu = (2.0 * rng.standard_normal(K)).astype(np.float32)
    x = bf16(mu[None, :] + rng.standard_normal((T, K)))
    xf = bf16_bits_to_f32(x).astype(np.float64)
    total = xf.var()
    mean_ch_var = xf.var(axis=0).mean()
    var_of_means = xf.mean(axis=0).var()
    assert abs(total - (mean_ch_var + var_of_means)) < 1e-10 * total        # the identity itself
    b = xf.mean(axis=0).astype(np.float32)
    _, s_raw, u_raw = oracle.quantize_act(x, 1.0, return_u=True)
    _, s_cor, u_cor = oracle.quantize_act(x, 1.0, b=b, return_u=True)
    frac_raw = u_raw.astype(np.float64).mean(axis=0).var() / u_raw.astype(np.float64).var()
    frac_cor = u_cor.astype(np.float64).mean(axis=0).var() / u_cor.astype(np.float64).var()
    assert frac_raw > 0.7 and frac_cor < 0.01
    ratio = np.mean(s_raw.astype(np.float64) ** 2) / np.mean(s_cor.astype(np.float64) ** 2)
    assert 0.6 * (1 + 4.0) < ratio < 1.4 * (1 + 4.0)        # sigma^2 drops from 1+4 to 1


def test_clipped_energy_fraction_18_4_percent():
    # Eq. 8: clipping N(0,1) at +-2.2 sigma loses ~18.4% of the energy of the
    # clipped values' region; closed form 2(t phi(t) + 1 - Phi(t)).  Pins the
    # generator's Gaussian draw + the paper constant used in DESIGN.md's alpha discussion.
    t = 2.2
    phi = math.exp(-t * t / 2) / math.sqrt(2 * math.pi)
    tail = 0.5 * math.erfc(t / math.sqrt(2))
    closed = 2 * (t * phi + tail)
    assert abs(closed - 0.184) < 0.0005 + 0.0005
    rng = np.random.default_rng(17)
    z = rng.standard_normal(1_000_000)
    emp = np.sum(z[np.abs(z) > t] ** 2) / np.sum(z ** 2)
    assert abs(emp - 0.184) < 0.005


def test_quantizer_argument_errors():
    x = bf16(np.ones((1, 128), dtype=np.float32))
    with pytest.raises(ValueError):
        oracle.quantize_act(x, 0.0)                  # alpha in (0,1]
    with pytest.raises(ValueError):
        oracle.quantize_act(x, 1.5)
    with pytest.raises(ValueError):
        oracle.quantize_act(x, 1.0, had_block=96)    # non power of two
    with pytest.raises(ValueError):
        oracle.quantize_act(np.zeros((0, 128), dtype=np.uint16), 1.0)   # empty


def test_quantizer_with_hadamard_matches_composition():
    # had_block: the quantizer must see exactly hadamard_blocks(x) (R^-1 before s^a, Eq. 15).
    rng = np.random.default_rng(19)
    T, K = 8, 512
    x = bf16(rng.standard_normal((T, K)))
    b = (0.1 * rng.standard_normal(K)).astype(np.float32)
    codes, scales, u = oracle.quantize_act(x, 0.9, gamma=1.1, b=b, had_block=128, return_u=True)
    xf = bf16_bits_to_f32(x)
    for t in range(T):
        h = oracle.hadamard_blocks(xf[t].copy(), 128)
        g = np.float32(1.1)
        for k in range(0, K, 7):
            exact = Fraction(float(g)) * Fraction(float(h[k])) - Fraction(float(b[k]))
            assert u[t, k] == _round_f32(exact)
    # one-hot in a block -> all |h| equal -> all |codes| equal when b = 0
    one = np.zeros((1, K), dtype=np.float32)
    one[0, 130] = 128.0
    c2, s2 = oracle.quantize_act(bf16(one), 1.0, had_block=128)
    q = codes_to_int(c2)[0]
    assert np.all(np.abs(q[128:256]) == 7) and np.all(q[:128] == 0) and np.all(q[256:] == 0)


# --------------------------------------------------------------------------- GEMM
def _pack(q):
    u = (np.ascontiguousarray(q).astype(np.int8).astype(np.uint8) & 0xF)
    return np.ascontiguousarray((u[:, 0::2] | (u[:, 1::2] << 4)).astype(np.uint8))


def test_gemm_closed_forms():
    K = 256
    ones = _pack(np.ones((3, K), dtype=np.int8))
    assert np.all(oracle.gemm_i32(ones, ones) == K)
    a = _pack(np.full((2, K), 7, dtype=np.int8))
    w = _pack(np.full((5, K), -8, dtype=np.int8))
    assert np.all(oracle.gemm_i32(a, w) == -56 * K)


def test_gemm_one_hot_rows_pick_weights():
    rng = np.random.default_rng(23)
    K, N = 128, 16
    wq = rng.integers(-8, 8, size=(N, K)).astype(np.int8)
    for k in (0, 1, 77, 127):
        a = np.zeros((1, K), dtype=np.int8)
        a[0, k] = 3
        acc = oracle.gemm_i32(_pack(a), _pack(wq))
        assert np.array_equal(acc[0], 3 * wq[:, k].astype(np.int32))


def test_gemm_matches_brute_force_and_numpy():
    # north_star: "the INT32 GEMM must agree with brute-force triple loops on tiny shapes".
    rng = np.random.default_rng(29)
    T, N, K = 16, 16, 256
    aq = rng.integers(-8, 8, size=(T, K)).astype(np.int8)
    wq = rng.integers(-8, 8, size=(N, K)).astype(np.int8)
    acc = oracle.gemm_i32(_pack(aq), _pack(wq))
    brute = [[sum(int(aq[t, k]) * int(wq[n, k]) for k in range(K)) for n in range(N)]
             for t in range(T)]
    assert acc.tolist() == brute
    assert np.array_equal(acc, aq.astype(np.int64) @ wq.astype(np.int64).T)
    # permuting K on both operands leaves the contraction unchanged
    perm = rng.permutation(K)
    assert np.array_equal(acc, oracle.gemm_i32(_pack(aq[:, perm]), _pack(wq[:, perm])))


# --------------------------------------------------------------------------- epilogue / fb
def test_epilogue_hand_case():
    acc = np.array([[8]], dtype=np.int32)
    y = oracle.epilogue(acc, np.array([0.5], np.float32), np.array([0.25], np.float32),
                        np.array([1.0], np.float32))
    assert y[0, 0] == 0x4000          # 0.5*0.25*8 + 1 = 2.0


def test_epilogue_against_exact_rational():
    rng = np.random.default_rng(31)
    T, N = 24, 40
    acc = rng.integers(-200000, 200000, size=(T, N)).astype(np.int32)
    st = (np.abs(rng.standard_normal(T)) * 0.3 + 0.01).astype(np.float32)
    sw = (np.abs(rng.standard_normal(N)) * 0.004 + 0.001).astype(np.float32)
    fb = rng.standard_normal(N).astype(np.float32)
    y, y64 = oracle.epilogue(acc, st, sw, fb, return_y64=True)
    for t in range(T):
        for n in range(N):
            exact = Fraction(float(st[t])) * Fraction(float(sw[n])) * int(acc[t, n]) + Fraction(float(fb[n]))
            assert abs(Fraction(float(y64[t, n])) - exact) <= abs(exact) * Fraction(1, 2 ** 52)
            assert y64[t, n] == float(exact)        # s_t s_w is exact in double: the fma is ONE rounding
            assert y[t, n] == _bf16_exact(float(y64[t, n]))


def test_fused_bias_against_exact_rational():
    rng = np.random.default_rng(37)
    N, K = 12, 256
    wq = rng.integers(-8, 8, size=(N, K)).astype(np.int8)
    sw = (np.abs(rng.standard_normal(N)) * 0.004 + 0.001).astype(np.float32)
    b = rng.standard_normal(K).astype(np.float32)
    bias = rng.standard_normal(N).astype(np.float32)
    fb = oracle.fused_bias(_pack(wq), sw, b, bias)
    for n in range(N):
        exact = Fraction(float(sw[n])) * sum(int(wq[n, k]) * Fraction(float(b[k])) for k in range(K)) \
            + Fraction(float(bias[n]))
        assert abs(Fraction(float(fb[n])) - exact) <= Fraction(float(np.spacing(np.abs(fb[n]))))
    assert np.array_equal(oracle.fused_bias(_pack(wq), sw, None, bias), bias)
    assert np.all(oracle.fused_bias(_pack(wq), sw, None, None) == 0)


def test_eq14_cancellation_on_lattice_rows():
    # Eq. 14: W(x - b) + W b = W x.  Integer-lattice rows make the quantizer exact, so
    # Y must equal bf16(W_deq (g x)) exactly ("quantizers disabled => equals FP forward").
    rng = np.random.default_rng(41)
    T, K, N = 8, 128, 32
    u_int = rng.integers(-7, 8, size=(T, K)).astype(np.float32)
    u_int[:, 0] = 7.0                                   # s_t = 1 with alpha = 1
    b = rng.integers(-3, 4, size=K).astype(np.float32)
    x = bf16(u_int + b[None, :])                        # small integers: exact in bf16
    wq = rng.integers(-8, 8, size=(N, K)).astype(np.int8)
    sw = np.full(N, 0.125, dtype=np.float32)
    fb = oracle.fused_bias(_pack(wq), sw, b, None)
    out = oracle.linear(x, _pack(wq), sw, fb, alpha=1.0, gamma=1.0, b=b)
    assert np.all(out["scales"] == 1.0)
    want = 0.125 * (wq.astype(np.float64) @ bf16_bits_to_f32(x).astype(np.float64).T).T
    assert np.array_equal(out["y64"], want)
    assert np.array_equal(out["y"], f32_to_bf16_bits(want.astype(np.float32)))


def test_output_noise_variance_follows_eq_9_11():
    # Eq. 9-11: rounding noise ~ U(-s/2, s/2) propagates as
    # Var(y_Q - y_ref) ~= sum_k W_deq[n,k]^2 s_t^2 / 12 on unclipped rows, within ~10%.
    rng = np.random.default_rng(43)
    T, K, N = 256, 1024, 64
    x = bf16(rng.standard_normal((T, K)))
    wq = rng.integers(-8, 8, size=(N, K)).astype(np.int8)
    sw = np.full(N, 0.01, dtype=np.float32)
    out = oracle.linear(x, _pack(wq), sw, None, alpha=1.0)
    wd = 0.01 * wq.astype(np.float64)
    ref = bf16_bits_to_f32(x).astype(np.float64) @ wd.T
    err = out["y64"] - ref
    pred = (out["scales"].astype(np.float64) ** 2 / 12.0)[:, None] * (wd ** 2).sum(axis=1)[None, :]
    ratio = (err ** 2).mean() / pred.mean()
    assert 0.9 < ratio < 1.1


def test_golden_fixture_matches_oracle():
    # Stored expected values written by tests/golden/make_golden.py (calls only oracle/).
    path = os.path.join(GOLDEN, "c1_digest.json")
    if not os.path.exists(path):
        pytest.skip("golden digest not generated")
    from baseq_inputs import make_layer
    import hashlib
    g = json.load(open(path))
    L = make_layer("c1", "linear")
    sp = L["spec"]
    fb = oracle.fused_bias(L["w_nibbles"], L["w_scale"], L["b"], L["layer_bias"])
    out = oracle.linear(L["x"], L["w_nibbles"], L["w_scale"], fb, sp.alpha, sp.gamma, None, L["b"])
    for key in ("codes", "scales", "acc", "y"):
        assert hashlib.sha256(out[key].tobytes()).hexdigest() == g[key], key


# =========================================================================== NEXT-1: asymmetric
def ucodes(codes):
    lo = (codes & 0xF).astype(np.int64)
    hi = (codes >> 4).astype(np.int64)
    out = np.empty((codes.shape[0], codes.shape[1] * 2), dtype=np.int64)
    out[:, 0::2], out[:, 1::2] = lo, hi
    return out


def test_asym_lattice_rows_exact():
    # group [0..15], b = 4, asymmetric, alpha = 1 -> z = 0, s = 1, codes = the integers
    row = np.tile(np.arange(16, dtype=np.float32), (3, 8))
    c, s, z = oracle.quantize_act_asym(bf16(row), 1.0)
    assert np.all(s == 1.0) and np.all(z == 0.0)
    assert np.array_equal(ucodes(c), row.astype(np.int64))
    # shifted lattice: values -5 .. 10 -> z = -5, s = 1, codes = value + 5
    c, s, z = oracle.quantize_act_asym(bf16(row - 5.0), 1.0)
    assert np.all(s == 1.0) and np.all(z == -5.0)
    assert np.array_equal(ucodes(c), row.astype(np.int64))


def test_asym_constant_row_and_floor():
    # degenerate all-equal group -> floor scale, value reproduced exactly by z
    row = np.full((2, 128), 5.0, dtype=np.float32)
    c, s, z = oracle.quantize_act_asym(bf16(row), 1.0)
    assert np.all(s == np.float32(1e-12)) and np.all(z == 5.0) and np.all(ucodes(c) == 0)


def test_asym_matches_independent_restatement_and_reconstructs():
    rng = np.random.default_rng(5)
    x = (rng.standard_normal((7, 256)) * 2.0 + 1.5).astype(np.float32)
    xb = bf16(x)
    xf = (xb.astype(np.uint32) << 16).view(np.float32)
    b = (0.3 * rng.standard_normal(256)).astype(np.float32)
    for alpha in (1.0, 0.9):
        c, s, z = oracle.quantize_act_asym(xb, alpha, 1.05, None, b)
        # independent numpy restatement, every op in float32 (Eq. 4)
        u = (np.float64(np.float32(1.05)) * xf.astype(np.float64) - b.astype(np.float64)).astype(np.float32)
        mn, mx = u.min(axis=1), u.max(axis=1)
        st = np.maximum((np.float32(alpha) * (mx - mn)) / np.float32(15.0), np.float32(1e-12)).astype(np.float32)
        zz = (np.float32(alpha) * mn).astype(np.float32)
        inv = (np.float32(1.0) / st).astype(np.float32)
        q = np.clip(np.rint((u - zz[:, None]).astype(np.float32).astype(np.float64) * inv[:, None].astype(np.float64)), 0, 15)
        assert np.array_equal(s.view(np.uint32), st.view(np.uint32))
        assert np.array_equal(z.view(np.uint32), zz.view(np.uint32))
        assert np.array_equal(ucodes(c), q.astype(np.int64))
        if alpha == 1.0:
            # reconstruction: |s q + z - u| <= s / 2 for every element (nothing is clipped)
            rec = s[:, None].astype(np.float64) * ucodes(c) + z[:, None].astype(np.float64)
            assert np.all(np.abs(rec - u.astype(np.float64)) <= 0.5 * s[:, None] * (1 + 2.0 ** -18))


def test_asym_gemm_and_epilogue_identity():
    # sum_k Wdeq[n,k] (s q_k + z) == s s_w acc + z s_w wsum  (the algebra the epilogue relies on),
    # brute force on a tiny shape with exact rational arithmetic
    rng = np.random.default_rng(9)
    T, K, N = 3, 64, 5
    qa = rng.integers(0, 16, size=(T, K))
    qw = rng.integers(-8, 8, size=(N, K))
    codes = (qa[:, 0::2] | (qa[:, 1::2] << 4)).astype(np.uint8)
    wn = ((qw[:, 0::2] & 0xF) | ((qw[:, 1::2] & 0xF) << 4)).astype(np.uint8)
    acc, wsum = oracle.gemm_i32_asym(codes, wn)
    assert np.array_equal(acc, qa @ qw.T) and np.array_equal(wsum, qw.sum(axis=1))
    s = np.array([0.5, 0.25, 0.125], dtype=np.float32)
    z = np.array([-1.0, 0.5, 2.0], dtype=np.float32)
    sw = np.array([0.5, 1.0, 2.0, 0.25, 4.0], dtype=np.float32)
    fb = np.array([1.0, -2.0, 0.0, 0.5, 3.0], dtype=np.float32)
    y, y64 = oracle.epilogue_asym(acc, wsum, s, z, sw, fb, return_y64=True)
    for t in range(T):
        for n in range(N):
            exact = sum(Fraction(float(sw[n])) * int(qw[n, k]) * (Fraction(float(s[t])) * int(qa[t, k])
                        + Fraction(float(z[t]))) for k in range(K)) + Fraction(float(fb[n]))
            assert Fraction(float(y64[t, n])) == exact          # powers of two: no rounding at all
            assert y[t, n] == oracle.bf16_from_double(float(exact))


def test_asym_epilogue_against_exact_rational_on_general_scales():
    # oracle_epilogue_asym on scales that are NOT powers of two (every fma really rounds):
    #   c = fma(z s_w, wsum, fb);  y64 = fma(s s_w, acc, c)
    # s s_w and z s_w are exact in double (24 x 24 bits), so each fma is ONE rounding of an exact
    # rational; int / int true division in Python is correctly rounded, so float(Fraction) is that
    # rounding.  Equality is required bit for bit, and the pin must tell the stated nesting from the
    # other one (lower-bound term added last), which differs on some elements.
    rng = np.random.default_rng(131)
    T, N = 20, 36
    acc = rng.integers(0, 900000, size=(T, N)).astype(np.int32)          # unsigned codes: acc >= 0 mostly
    wsum = rng.integers(-30000, 30000, size=N).astype(np.int32)
    st = (np.abs(rng.standard_normal(T)) * 0.3 + 0.013).astype(np.float32)
    zt = (-8.3 * st * (1.0 + 0.2 * rng.standard_normal(T))).astype(np.float32)
    sw = (np.abs(rng.standard_normal(N)) * 0.004 + 0.0011).astype(np.float32)
    fb = rng.standard_normal(N).astype(np.float32)
    y, y64 = oracle.epilogue_asym(acc, wsum, st, zt, sw, fb, return_y64=True)
    other_nesting_differs = 0
    for t in range(T):
        for n in range(N):
            S, Z, W, F = (Fraction(float(v)) for v in (st[t], zt[t], sw[n], fb[n]))
            c = float(Z * W * int(wsum[n]) + F)                         # one rounding
            want = float(S * W * int(acc[t, n]) + Fraction(c))          # one rounding
            assert y64[t, n] == want, (t, n)
            assert y[t, n] == _bf16_exact(want)
            exact = S * W * int(acc[t, n]) + Z * W * int(wsum[n]) + F
            assert abs(Fraction(want) - exact) <= (abs(Fraction(c)) + abs(exact)) * Fraction(1, 2 ** 52)
            c2 = float(S * W * int(acc[t, n]) + F)
            other_nesting_differs += float(Z * W * int(wsum[n]) + Fraction(c2)) != want
    assert other_nesting_differs > 0


# =========================================================================== NEXT-3: KV cache
def test_kv_groups_are_heads_and_do_not_straddle():
    # contiguous blocks of head_dim; a head's codes / scale / zero depend on that head only
    rng = np.random.default_rng(9)
    T, H, D = 5, 4, 64
    x = rng.standard_normal((T, H * D)).astype(np.float32)
    c0, s0, z0 = oracle.quantize_kv(bf16(x), H, D, 1.0)
    x2 = x.copy()
    x2[:, 2 * D:3 * D] = 37.0 * rng.standard_normal((T, D)).astype(np.float32)   # disturb head 2 only
    c1, s1, z1 = oracle.quantize_kv(bf16(x2), H, D, 1.0)
    for h in (0, 1, 3):
        assert np.array_equal(c0[:, h * D // 2:(h + 1) * D // 2], c1[:, h * D // 2:(h + 1) * D // 2])
        assert np.array_equal(s0[:, h], s1[:, h]) and np.array_equal(z0[:, h], z1[:, h])
    assert not np.array_equal(s0[:, 2], s1[:, 2])


def test_kv_lattice_heads_exact_and_reconstruct():
    # each head a shifted integer lattice (S:227 per group): head h holds h*3 - 4 + (0..15)
    T, H, D = 3, 4, 64
    base = np.tile(np.arange(16, dtype=np.float32), D // 16)
    x = np.concatenate([base + (3.0 * h - 4.0) for h in range(H)])[None, :].repeat(T, axis=0)
    c, s, z = oracle.quantize_kv(bf16(x), H, D, 1.0)
    assert np.all(s == 1.0)
    assert np.array_equal(z, np.tile(3.0 * np.arange(H, dtype=np.float32) - 4.0, (T, 1)))
    assert np.array_equal(ucodes(c), np.tile(np.tile(base, H), (T, 1)).astype(np.int64))
    # random data: per-head reconstruction error <= half a step of THAT head (alpha = 1)
    rng = np.random.default_rng(10)
    xr = (rng.standard_normal((6, H * D)) * np.repeat([0.1, 1.0, 10.0, 100.0], D)).astype(np.float32)
    xb = bf16(xr)
    xf = (xb.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    c, s, z = oracle.quantize_kv(xb, H, D, 1.0)
    rec = np.repeat(s, D, axis=1).astype(np.float64) * ucodes(c) + np.repeat(z, D, axis=1)
    assert np.all(np.abs(rec - xf) <= 0.5 * np.repeat(s, D, axis=1) * (1 + 2.0 ** -18))
    # and the steps really are per head: they follow the heads' spreads
    assert np.all(s[:, 0] < s[:, 1]) and np.all(s[:, 1] < s[:, 2]) and np.all(s[:, 2] < s[:, 3])


def test_rounding_is_of_the_exact_product():
    # C-17: q = rne(u * inv) rounds the EXACT product once.  Steer inv with alpha until the exact
    # u * inv lies strictly on one side of k + 1/2 while its fp32-rounded value is the tie itself
    # (a separately rounded product would then go to the even neighbour): the code must follow the
    # exact product.
    f32 = np.float32
    m = f32(8.0)
    found = {"below": 0, "above": 0}
    separating = 0        # cases where rounding the fp32 product (ties to even) gives another code
    # bf16-representable u with full 8-bit significands, |u| < m; odd and even k
    for u, k in ((f32(191 / 128), 1), (f32(147 / 128), 2), (f32(221 / 128), 3), (f32(1.5), 4),
                 (f32(253 / 128), 5), (f32(163 / 128), 6)):
        a0 = f32(7.0 * (float(u) / (k + 0.5)) / float(m))
        alpha = a0
        for _ in range(64):
            alpha = np.nextafter(alpha, f32(0.0))
        for _ in range(129):
            st = f32(f32(alpha * m) / f32(7.0))
            inv = f32(f32(1.0) / st)
            exact = float(u) * float(inv)           # exact in double: 8 x 24 significant bits
            if f32(exact) == f32(k + 0.5) and exact != k + 0.5 and 2.0 ** -16 <= alpha <= 1.0:
                row = np.zeros((1, 128), dtype=f32)
                row[0, 0], row[0, 1] = m, u
                c, s = oracle.quantize_act(bf16(row), float(alpha))
                assert s[0] == st
                side = "above" if exact > k + 0.5 else "below"
                assert codes_to_int(c)[0, 1] == (k + 1 if side == "above" else k)
                found[side] += 1
                separating += (side == "above") == (k % 2 == 0)
            alpha = np.nextafter(alpha, f32(2.0))
    assert found["below"] > 0 and found["above"] > 0     # the search exercised both sides
    assert separating > 0


# =========================================================================== NEXT-2: dense Hadamard mode
def test_dense_hadamard_equals_library_matrix_product():
    # oracle_dense_hadamard_u64 against scipy.linalg.hadamard (Sylvester construction, the library
    # routine) applied in fp64: u = g * (H x) / sqrt(B) - b, per block
    from scipy.linalg import hadamard
    rng = np.random.default_rng(61)
    for B, K in ((128, 384), (16, 64), (2, 8)):
        x = bf16(rng.standard_normal((5, K)) * 3.0)
        xf = bf16_bits_to_f32(x).astype(np.float64)
        sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
        b = rng.standard_normal(K).astype(np.float32)
        u, l1 = oracle.dense_hadamard_u64(x, B, 1.0, sa, b)
        H = hadamard(B).astype(np.float64)
        want = (xf.reshape(5, K // B, B) @ H.T).reshape(5, K) / np.sqrt(B) * sa.astype(np.float64) - b
        assert np.allclose(u, want, rtol=0, atol=1e-12 * np.abs(want).max())
        assert np.allclose(l1, np.abs(xf).reshape(5, K // B, B).sum(axis=2), rtol=1e-15)


def test_dense_hadamard_equals_butterflies_where_both_are_exact():
    # small-integer inputs: every butterfly of Q1 is exact in fp32 and the dense sum is exact in
    # fp64, so the two oracle modes must agree (before the 1/sqrt(B) rounding: use B = 4, 16, 64,
    # whose 1/sqrt(B) is a power of two)
    rng = np.random.default_rng(62)
    for B in (4, 16, 64):
        K = 4 * B
        xi = rng.integers(-60, 61, size=(3, K)).astype(np.float32)
        x = bf16(xi)
        u, _ = oracle.dense_hadamard_u64(x, B)
        for t in range(3):
            h = bf16_bits_to_f32(x[t]).copy()
            oracle.hadamard_blocks(h, B)
            assert np.array_equal(h.astype(np.float64), u[t])
    # and H H = B I: applying the dense transform twice returns the input (g = 1, b = 0, exact here)
    x = bf16(rng.integers(-7, 8, size=(2, 64)).astype(np.float32))
    u, _ = oracle.dense_hadamard_u64(x, 16)
    u2, _ = oracle.dense_hadamard_u64(bf16(u.astype(np.float32)), 16)
    assert np.array_equal(u2, bf16_bits_to_f32(x).astype(np.float64))


def test_dense_mode_band_accepts_the_contract_and_rejects_mistakes():
    # The acceptance band of the tensor-core mode (oracle.dense_mode_check): the bit-exact
    # butterfly quantiser is itself an admissible dense-mode result (its fp32 error is far inside the
    # band); a result with a wrong sign convention, a dropped bias, or codes off by one level on
    # elements that are not near a rounding boundary is rejected.
    rng = np.random.default_rng(63)
    T, K, B = 6, 1024, 128
    x = bf16(rng.standard_normal((T, K)) + 0.3)
    b = (0.3 * rng.standard_normal(K)).astype(np.float32)
    u, l1 = oracle.dense_hadamard_u64(x, B, 1.0, None, b)
    tol, m_lo, m_hi = oracle.dense_mode_bounds(u, l1, 0.9, B)
    codes, scales = oracle.quantize_act(x, 0.9, 1.0, None, b, B)
    ok, bs, bq_ = oracle.dense_mode_check(codes, scales, u, tol, m_lo, m_hi, 0.9)
    assert ok, (bs, bq_)
    # no bias
    c2, s2 = oracle.quantize_act(x, 0.9, 1.0, None, None, B)
    assert not oracle.dense_mode_check(c2, s2, u, tol, m_lo, m_hi, 0.9)[0]
    # scale off by 2^-12
    assert not oracle.dense_mode_check(codes, (scales * np.float32(1 + 2.0 ** -12)).astype(np.float32),
                                       u, tol, m_lo, m_hi, 0.9)[0]
    # one code moved by one level (an element in the middle of its rounding interval)
    q = codes_to_int(codes)
    r = u / scales[:, None].astype(np.float64)
    t, k = np.unravel_index(np.argmin(np.abs(r - np.rint(r)) + 10.0 * (np.abs(q) >= 7)), r.shape)
    q2 = q.copy()
    q2[t, k] += 1
    u8 = (q2.astype(np.int16) & 0xF).astype(np.uint8)
    c3 = (u8[:, 0::2] | (u8[:, 1::2] << 4)).astype(np.uint8)
    ok3, _, nb = oracle.dense_mode_check(c3, scales, u, tol, m_lo, m_hi, 0.9)
    assert not ok3 and nb == 1
    # the band is narrow: at most a small fraction of the elements may take two values
    lo = np.rint((u - tol) / scales[:, None]); hi = np.rint((u + tol) / scales[:, None])
    assert (lo != hi).mean() < 2e-3

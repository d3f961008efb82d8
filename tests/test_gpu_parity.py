"""GPU-vs-oracle parity (-m gpu): bit-exact codes, scales, int32 accumulators and bf16 output.

Every call goes through the C-ABI library (paper_2506_15689_b200.binding -> libbaseq.so).
Expected values come from oracle/ only, on the same seeded inputs (baseq_inputs).
"""
import numpy as np
import pytest
import torch

import oracle
from baseq_inputs import f32_to_bf16_bits, make_activations, make_layer, make_weights

pytestmark = pytest.mark.gpu

bq = None


def setup_module(module):
    global bq
    import paper_2506_15689_b200 as _bq
    bq = _bq
    assert torch.cuda.is_available()


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.view(dtype)


def bf16_dev(bits):
    return torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)


def bits_host(t):
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def run_quant(x_bits, alpha, gamma=1.0, sa=None, b=None, had_block=0):
    params = bq.ActParams(alpha, gamma, None if sa is None else dev(sa),
                          None if b is None else dev(b), had_block)
    codes, scales = bq.quantize_act(bf16_dev(x_bits), params)
    torch.cuda.synchronize()
    return codes.cpu().numpy(), scales.cpu().numpy()


def check_quant(x_bits, alpha, gamma=1.0, sa=None, b=None, had_block=0):
    codes, scales = run_quant(x_bits, alpha, gamma, sa, b, had_block)
    ocodes, oscales = oracle.quantize_act(x_bits, alpha, gamma, sa, b, had_block)
    assert np.array_equal(scales.view(np.uint32), oscales.view(np.uint32)), "scales differ"
    assert np.array_equal(codes, ocodes), "codes differ: %d bytes" % int((codes != ocodes).sum())


def rand_x(rng, T, K, spread=0.5):
    mu = spread * rng.standard_normal(K)
    return f32_to_bf16_bits((mu[None, :] + rng.standard_normal((T, K))).astype(np.float32))


# ------------------------------------------------------------------------------- quantizer
@pytest.mark.parametrize("T,K", [(1, 128), (16, 256), (37, 384), (130, 4096), (33, 11008),
                                 (9, 14336), (5, 28672), (257, 1024), (3, 32768)])
def test_quantizer_bit_exact_shapes(T, K):
    rng = np.random.default_rng(T * 100003 + K)
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    check_quant(x, 0.9, 1.05, None, b)


def test_quantizer_variants():
    rng = np.random.default_rng(7)
    T, K = 67, 2048
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    check_quant(x, 1.0)                          # plain RTN
    check_quant(x, 0.5, 1.2)                     # heavy clipping: saturates at -8 / 7
    check_quant(x, 0.9, 1.0, sa, b)              # per-channel s^a
    check_quant(x, 0.9, 1.0, sa, None)
    zero = np.zeros((4, 256), dtype=np.uint16)   # degenerate rows: floor scale, codes 0
    check_quant(zero, 0.9)
    ties = f32_to_bf16_bits(np.tile(np.array([0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 7.0, 3.5],
                                             dtype=np.float32), (3, 32)))
    check_quant(ties, 1.0)


@pytest.mark.parametrize("K,B", [(256, 128), (4096, 128), (28672, 128), (1024, 16), (512, 256),
                                 (384, 2)])
def test_quantizer_hadamard_bit_exact(K, B):
    rng = np.random.default_rng(K + B)
    x = rand_x(rng, 19, K, 0.3)
    b = (0.2 * rng.standard_normal(K)).astype(np.float32)
    check_quant(x, 0.9, 1.0, None, b, B)


def test_quantizer_per_channel_sa_long_rows():
    # a per-channel s^a vector: the ring's split kernel at K = 4096 without Hadamard, the
    # register-resident kernel otherwise
    rng = np.random.default_rng(17)
    for K in (4096, 8192, 11008, 14336, 28672):
        x = rand_x(rng, 9, K)
        b = (0.5 * rng.standard_normal(K)).astype(np.float32)
        sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
        check_quant(x, 0.9, 1.0, sa, b)
        check_quant(x, 0.9, 1.0, sa, None)
        check_quant(x, 0.9, 1.0, sa, b, 128)
    x = rand_x(rng, 1030, 4096)                  # many stages per CTA, ragged last stage
    sa = (1.0 + 0.1 * rng.standard_normal(4096)).astype(np.float32)
    check_quant(x, 0.9, 1.0, sa, (0.5 * rng.standard_normal(4096)).astype(np.float32))


def test_quantizer_strided_input():
    rng = np.random.default_rng(11)
    T, K, ld = 21, 512, 640
    full = rand_x(rng, T, ld)
    xt = bf16_dev(full)[:, :K]
    params = bq.ActParams(0.9)
    codes, scales = bq.quantize_act(xt, params)
    oc, os_ = oracle.quantize_act(np.ascontiguousarray(full[:, :K]), 0.9)
    assert np.array_equal(codes.cpu().numpy(), oc)
    assert np.array_equal(scales.cpu().numpy(), os_)


# ------------------------------------------------------------------------------- NEXT-2: tensor-core Hadamard
def check_quant_tc(x_bits, alpha, gamma=1.0, sa=None, b=None, rows=None):
    """baseq_quantize_act_tc against the dense-Hadamard oracle mode: every scale and every code
    must be admissible (oracle.dense_mode_check); beside it, the fraction of codes
    that differ from the bit-exact butterfly contract (must be tiny: only elements whose u / s_t sits
    within the band of a rounding boundary may move, and then by one level)."""
    params = bq.ActParams(alpha, gamma, None if sa is None else dev(sa), None if b is None else dev(b), 128)
    codes, scales = bq.quantize_act_tc(bf16_dev(x_bits), params)
    torch.cuda.synchronize()
    codes, scales = codes.cpu().numpy(), scales.cpu().numpy()
    sel = np.arange(x_bits.shape[0]) if rows is None else rows
    xs = np.ascontiguousarray(x_bits[sel])
    u64, l1 = oracle.dense_hadamard_u64(xs, 128, gamma, sa, b)
    tol, m_lo, m_hi = oracle.dense_mode_bounds(u64, l1, alpha, 128, sa, gamma)
    ok, bad_s, bad_q = oracle.dense_mode_check(codes[sel], scales[sel], u64, tol, m_lo, m_hi, alpha)
    assert ok, "tensor-core Hadamard: %d inadmissible scales, %d inadmissible codes" % (bad_s, bad_q)
    ocodes, oscales = oracle.quantize_act(xs, alpha, gamma, sa, b, 128)
    frac = float((codes[sel] != ocodes).mean())
    assert frac < 2e-3, "too many codes differ from the butterfly contract: %.2e of the bytes" % frac
    assert np.allclose(scales[sel], oscales, rtol=2.0 ** -18, atol=0)
    return frac


@pytest.mark.parametrize("T,K", [(16, 128), (1, 256), (37, 384), (100, 4096), (33, 11008), (21, 14336),
                                 (50, 28672), (130, 3584), (17, 7168)])
def test_quantizer_tc_shapes(T, K):
    # one CTA (K <= 3584), clusters of 2 / 4 / 8 (uneven block split at K = 11008), ragged token groups
    rng = np.random.default_rng(T * 7 + K)
    x = rand_x(rng, T, K, 0.3)
    b = (0.2 * rng.standard_normal(K)).astype(np.float32)
    check_quant_tc(x, 0.9, 1.0, None, b)


def test_quantizer_tc_variants():
    rng = np.random.default_rng(909)
    T, K = 45, 4096
    x = rand_x(rng, T, K, 0.5)
    b = (0.3 * rng.standard_normal(K)).astype(np.float32)
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    check_quant_tc(x, 1.0)                                # no bias, no clipping
    check_quant_tc(x, 0.5, 1.2, None, b)                  # heavy clipping
    check_quant_tc(x, 0.9, 1.0, sa, b)                    # per-channel s^a
    zero = np.zeros((20, 256), dtype=np.uint16)           # floor scale, codes 0
    params = bq.ActParams(0.9, 1.0, None, None, 128)
    codes, scales = bq.quantize_act_tc(bf16_dev(zero), params)
    torch.cuda.synchronize()
    assert torch.all(codes == 0) and torch.all(scales == float(np.float32(1e-12)))
    # small integers: the 128-term sums are exact in any order -- the transform itself must then be
    # exact (one-hot rows spread a / sqrt(128) with the signs of H's columns, Eq. 2)
    onehot = np.zeros((128, 128), dtype=np.float32)
    onehot[np.arange(128), np.arange(128)] = 16.0
    codes, scales = bq.quantize_act_tc(bf16_dev(f32_to_bf16_bits(onehot)), bq.ActParams(1.0, 1.0, None, None, 128))
    torch.cuda.synchronize()
    oc, os_ = oracle.quantize_act(f32_to_bf16_bits(onehot), 1.0, 1.0, None, None, 128)
    assert np.array_equal(codes.cpu().numpy(), oc) and np.array_equal(scales.cpu().numpy(), os_)


def test_quantizer_tc_config5_full_size_sampled_rows():
    # config 5's activation at full size (T = 4096, K = 28672: clusters of 8, 16 groups per cluster)
    L = cached_layer("c5", "down")
    rows = half_rows(L["spec"].T)
    frac = check_quant_tc(L["x"], L["spec"].alpha, L["spec"].gamma, None, L["b"], rows=rows)
    assert frac < 1e-3


def test_quantizer_tc_feeds_the_gemm():
    # the codes of the tensor-core mode through the unchanged GEMM: the accumulators equal the
    # oracle's integer GEMM of THOSE codes, the output its epilogue with THOSE scales
    rng = np.random.default_rng(4711)
    T, K, N = 130, 1024, 264
    x = rand_x(rng, T, K, 0.3)
    b = (0.2 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
    codes, scales = bq.quantize_act_tc(bf16_dev(x), bq.ActParams(0.9, 1.0, None, dev(b), 128))
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    y = bq.w4a4_gemm(codes, scales, pw, acc_dump=acc)
    bq.sync_status()
    oacc = oracle.gemm_i32(codes.cpu().numpy(), W["w_nibbles"])
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    assert np.array_equal(acc.cpu().numpy(), oacc)
    assert np.array_equal(bits_host(y), oracle.epilogue(oacc, scales.cpu().numpy(), W["w_scale"], fb))


def test_quantizer_tc_rejects_other_blocks():
    x = torch.zeros((4, 256), dtype=torch.bfloat16, device="cuda")
    for B in (0, 64, 256):
        with pytest.raises(bq.BaseqError) as e:
            bq.quantize_act_tc(x, bq.ActParams(0.9, had_block=B))
        assert e.value.status == 6
    with pytest.raises(bq.BaseqError) as e:
        bq.quantize_act_tc(torch.zeros((4, 32768), dtype=torch.bfloat16, device="cuda"), bq.ActParams(0.9, had_block=128))
    assert e.value.status == 6


# ------------------------------------------------------------------------------- packer
def test_pack_weights_fused_bias_matches_oracle():
    W = make_weights("c1", "linear")
    rng = np.random.default_rng(3)
    b = rng.standard_normal(W["K"]).astype(np.float32)
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
    torch.cuda.synchronize()
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    assert np.array_equal(pw.fused_bias.cpu().numpy().view(np.uint32), fb.view(np.uint32))


# ------------------------------------------------------------------------------- GEMM + epilogue
def run_linear(x_bits, W, alpha, gamma, b, had_block=0, rows=None, with_bias=True):
    """Runs quantize + GEMM on the GPU and the oracle; compares everything bit for bit."""
    N, K = W["N"], W["K"]
    lb = W["layer_bias"] if with_bias else None
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, lb)
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), None if b is None else dev(b),
                         None if lb is None else dev(lb))
    torch.cuda.synchronize()
    assert np.array_equal(pw.fused_bias.cpu().numpy().view(np.uint32), fb.view(np.uint32))
    params = bq.ActParams(alpha, gamma, None, None if b is None else dev(b), had_block)
    xd = bf16_dev(x_bits)
    T = x_bits.shape[0]
    codes, scales = bq.quantize_act(xd, params)
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    y = bq.w4a4_gemm(codes, scales, pw, acc_dump=acc)
    y2 = bq.w4a4_gemm(codes, scales, pw)            # timed configuration: no dump
    torch.cuda.synchronize()
    assert torch.equal(y.view(torch.int16), y2.view(torch.int16))
    sel = np.arange(T) if rows is None else rows
    ref = oracle.linear(np.ascontiguousarray(x_bits[sel]), W["w_nibbles"], W["w_scale"], fb,
                        alpha, gamma, None, b, had_block)
    assert np.array_equal(codes.cpu().numpy()[sel], ref["codes"])
    assert np.array_equal(scales.cpu().numpy()[sel], ref["scales"])
    gacc = acc.cpu().numpy()[sel]
    assert np.array_equal(gacc, ref["acc"]), "int32 accumulators differ at %d places" % int(
        (gacc != ref["acc"]).sum())
    gy = bits_host(y)[sel]
    nbad = int((gy != ref["y"]).sum())
    assert nbad == 0, "bf16 output differs at %d of %d places" % (nbad, gy.size)
    return ref, gy


def test_config1_full():
    L = make_layer("c1", "linear")
    sp = L["spec"]
    run_linear(L["x"], L, sp.alpha, sp.gamma, L["b"])


@pytest.mark.parametrize("T,K,N", [(16, 256, 256), (1, 128, 8), (130, 384, 264), (257, 1024, 520),
                                   (128, 128, 256), (300, 2048, 1024)])
def test_linear_ragged_shapes(T, K, N):
    rng = np.random.default_rng(T + 7 * K + 13 * N)
    x = rand_x(rng, T, K)
    q = rng.integers(-8, 8, size=(N, K)).astype(np.int8).astype(np.uint8) & 0xF
    W = {"N": N, "K": K, "w_nibbles": np.ascontiguousarray(q[:, 0::2] | (q[:, 1::2] << 4)),
         "w_scale": (0.002 + 0.004 * rng.random(N)).astype(np.float32),
         "layer_bias": rng.standard_normal(N).astype(np.float32)}
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    run_linear(x, W, 0.9, 1.05, b)


def test_gemm_extreme_codes():
    # qa = 7, qw = -8 everywhere: acc = -56 K (closed form), largest |raw| accumulator
    T, K, N = 130, 4096, 256
    codes = torch.full((T, K // 2), 0x77, dtype=torch.uint8, device="cuda")
    scales = torch.full((T,), 0.25, dtype=torch.float32, device="cuda")
    wn = np.full((N, K // 2), 0x88, dtype=np.uint8)
    sw = np.full((N,), 0.5, dtype=np.float32)
    pw = bq.pack_weights(dev(wn), dev(sw))
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    y = bq.w4a4_gemm(codes, scales, pw, acc_dump=acc)
    torch.cuda.synchronize()
    assert torch.all(acc == -56 * K)
    assert torch.all(y.float() == -56.0 * K * 0.125)


def test_config2_sampled_rows():
    L = make_layer("c2", "qkvo")
    sp = L["spec"]
    rows = np.r_[0:8, 1020:1030, 2040:2048]
    run_linear(L["x"], L, sp.alpha, sp.gamma, L["b"], rows=rows)


def test_config5_hadamard_small_T():
    # config 5's K = 28672 + Hadamard-128 with a small token count (full N would take the
    # oracle minutes: use the first 512 output channels of the seeded weight).
    A = make_activations("c5", "x_down", T=40)
    rng = np.random.default_rng(5)
    K, N = 28672, 512
    q = rng.integers(-8, 8, size=(N, K)).astype(np.int8).astype(np.uint8) & 0xF
    W = {"N": N, "K": K, "w_nibbles": np.ascontiguousarray(q[:, 0::2] | (q[:, 1::2] << 4)),
         "w_scale": (0.002 + 0.004 * rng.random(N)).astype(np.float32), "layer_bias": None}
    run_linear(A["x"], W, 0.9, 1.0, A["b"], had_block=128)


# ------------------------------------------------------------------------------- ABI errors
def test_abi_error_codes():
    x = torch.zeros((4, 256), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(bq.BaseqError) as e:
        bq.quantize_act(x, bq.ActParams(0.0))
    assert e.value.status == 4
    with pytest.raises(bq.BaseqError) as e:
        bq.quantize_act(x, bq.ActParams(0.9, had_block=96))
    assert e.value.status == 4
    with pytest.raises(bq.BaseqError) as e:
        bq.quantize_act(torch.zeros((4, 192), dtype=torch.bfloat16, device="cuda"), bq.ActParams(0.9))
    assert e.value.status == 2
    with pytest.raises(bq.BaseqError) as e:
        bq.quantize_act(torch.zeros((0, 256), dtype=torch.bfloat16, device="cuda"), bq.ActParams(0.9))
    assert e.value.status == 2


# ------------------------------------------------------------------------------- fused variant (a10)
def run_fused(x_bits, W, alpha, gamma, b, had_block=0, sa=None):
    """baseq_linear_fused vs the oracle: scales, producer codes, int32 accumulators, bf16 Y."""
    N, K = W["N"], W["K"]
    T = x_bits.shape[0]
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), None if b is None else dev(b),
                         None if W["layer_bias"] is None else dev(W["layer_bias"]))
    params = bq.ActParams(alpha, gamma, None if sa is None else dev(sa),
                          None if b is None else dev(b), had_block)
    codes = torch.zeros((T, K // 2), dtype=torch.uint8, device="cuda")
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    y, scales = bq.linear_fused(bf16_dev(x_bits), params, pw, codes_dump=codes, acc_dump=acc)
    y2, _ = bq.linear_fused(bf16_dev(x_bits), params, pw)          # timed configuration: no dumps
    torch.cuda.synchronize()
    assert torch.equal(y.view(torch.int16), y2.view(torch.int16))
    ref = oracle.linear(x_bits, W["w_nibbles"], W["w_scale"], fb, alpha, gamma, sa, b, had_block)
    assert np.array_equal(scales.cpu().numpy().view(np.uint32), ref["scales"].view(np.uint32))
    assert np.array_equal(codes.cpu().numpy(), ref["codes"])
    assert np.array_equal(acc.cpu().numpy(), ref["acc"])
    assert np.array_equal(bits_host(y), ref["y"])


def _rand_w(rng, N, K, bias=True):
    q = rng.integers(-8, 8, size=(N, K)).astype(np.int8).astype(np.uint8) & 0xF
    return {"N": N, "K": K, "w_nibbles": np.ascontiguousarray(q[:, 0::2] | (q[:, 1::2] << 4)),
            "w_scale": (0.002 + 0.004 * rng.random(N)).astype(np.float32),
            "layer_bias": rng.standard_normal(N).astype(np.float32) if bias else None}


def test_fused_config1():
    L = make_layer("c1", "linear")
    sp = L["spec"]
    run_fused(L["x"], L, sp.alpha, sp.gamma, L["b"])


@pytest.mark.parametrize("T,K,N,B", [(1, 128, 8, 0), (130, 384, 264, 0), (257, 1024, 520, 128),
                                     (300, 2048, 200, 16), (40, 4096, 192, 128)])
def test_fused_ragged_and_hadamard(T, K, N, B):
    rng = np.random.default_rng(T + 3 * K + 5 * N + B)
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    run_fused(x, _rand_w(rng, N, K), 0.9, 1.05, b, had_block=B)


def test_fused_per_channel_sa_and_no_bias():
    rng = np.random.default_rng(99)
    T, K, N = 70, 512, 136
    x = rand_x(rng, T, K)
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    run_fused(x, _rand_w(rng, N, K, bias=False), 1.0, 1.0, None, sa=sa)


def test_fused_hadamard_256_and_many_rows_per_quantiser_warp():
    # a 256-channel block spans the whole quantiser warp; few tiles = few CTAs = many rows per warp
    rng = np.random.default_rng(256)
    T, K, N = 700, 1024, 136
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    run_fused(x, _rand_w(rng, N, K), 0.9, 1.05, b, had_block=256)
    T, K, N = 1500, 640, 72                     # K / 8 = 80 vectors: a ragged last step per lane
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    run_fused(x, _rand_w(rng, N, K), 1.0, 1.0, b, had_block=128)


def test_fused_workspace_is_reused_without_clearing():
    # the ready counters are reset by the call itself: same workspace, garbage in it, three calls
    rng = np.random.default_rng(77)
    T, K, N = 300, 512, 200
    x_bits = rand_x(rng, T, K)
    W = _rand_w(rng, N, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
    params = bq.ActParams(0.9, 1.05, None, dev(b), 0)
    ref = oracle.linear(x_bits, W["w_nibbles"], W["w_scale"], fb, 0.9, 1.05, None, b, 0)
    ws = torch.full((bq.lib().baseq_fused_workspace_bytes(T, N, K),), 0xFF, dtype=torch.uint8, device="cuda")
    x = bf16_dev(x_bits)
    for _ in range(3):
        y, scales = bq.linear_fused(x, params, pw, workspace=ws)
        assert np.array_equal(bits_host(y), ref["y"])
        assert np.array_equal(scales.cpu().numpy().view(np.uint32), ref["scales"].view(np.uint32))
    off = ws.numel() - T * K // 2                                     # [ counters | codes ]
    assert np.array_equal(ws[off:].cpu().numpy().reshape(T, K // 2), ref["codes"])


def test_fused_and_static_calls_replay_in_a_cuda_graph():
    # neither call enqueues anything but kernels (the fused workspace is cleared by the kernel itself,
    # the static entry point owns its scratch): capture once, replay with new inputs in place
    rng = np.random.default_rng(909)
    T, K, N = 520, 1024, 392
    W = _rand_w(rng, N, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
    params = bq.ActParams(0.9, 1.0, None, dev(b), 0)
    x = torch.empty((T, K), dtype=torch.bfloat16, device="cuda")
    yf = torch.empty((T, N), dtype=torch.bfloat16, device="cuda")
    ys = torch.empty_like(yf)
    scales = torch.empty((T,), dtype=torch.float32, device="cuda")
    ws = torch.full((bq.lib().baseq_fused_workspace_bytes(T, N, K),), 0xAB, dtype=torch.uint8, device="cuda")
    xs = [rand_x(rng, T, K) for _ in range(3)]
    stream = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(stream):
        x.copy_(bf16_dev(xs[0]))
        bq.linear_fused(x, params, pw, yf, scales=scales, workspace=ws)        # warm-up outside capture
        bq.linear_static(x, params, pw, ys)
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=stream):
            bq.linear_fused(x, params, pw, yf, scales=scales, workspace=ws)
            bq.linear_static(x, params, pw, ys)
    for xb in xs:
        x.copy_(bf16_dev(xb))
        graph.replay()
        torch.cuda.synchronize()
        ref = oracle.linear(xb, W["w_nibbles"], W["w_scale"], fb, 0.9, 1.0, None, b, 0)
        assert np.array_equal(bits_host(yf), ref["y"])
        assert np.array_equal(bits_host(ys), ref["y"])
        assert np.array_equal(scales.cpu().numpy().view(np.uint32), ref["scales"].view(np.uint32))


def test_fused_launches_overlapping_on_two_streams():
    # two fused launches in flight at once, each with its own workspace: neither fits the GPU next
    # to the other, so CTAs of both wait for SMs while resident ones wait for quantised rows --
    # rows are claimed, so nobody waits for a CTA that is not running (w4a4_gemm.cu)
    rng = np.random.default_rng(2024)
    cases = []
    for T, K, N in ((1536, 1024, 4096), (1100, 2048, 4800)):
        x_bits = rand_x(rng, T, K)
        W = _rand_w(rng, N, K)
        b = (0.5 * rng.standard_normal(K)).astype(np.float32)
        fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
        pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
        ref = oracle.linear(x_bits, W["w_nibbles"], W["w_scale"], fb, 0.9, 1.0, None, b, 0)
        ws = torch.empty(bq.lib().baseq_fused_workspace_bytes(T, N, K), dtype=torch.uint8, device="cuda")
        cases.append((bf16_dev(x_bits), bq.ActParams(0.9, 1.0, None, dev(b), 0), pw, ws, ref,
                      torch.empty((T, N), dtype=torch.bfloat16, device="cuda"), torch.cuda.Stream()))
    torch.cuda.synchronize()
    for _ in range(10):
        for x, params, pw, ws, ref, y, stream in cases:
            with torch.cuda.stream(stream):
                bq.linear_fused(x, params, pw, y, workspace=ws)
    torch.cuda.synchronize()
    for x, params, pw, ws, ref, y, stream in cases:
        assert np.array_equal(bits_host(y), ref["y"])


# ------------------------------------------------------------------------------- full BASELINE sizes
# Launch configuration = the one bench.py times (full T, N, K; the timed output comes from a call
# without dumps).  Three layers of comparison, so that every tile, both CTAs of every pair and every
# TMEM lane quarter of the persistent GEMM are covered:
#   1. the ORACLE quantises every row: codes and scales of all T rows, bit for bit;
#   2. every int32 accumulator (acc_dump, all T x N) against an integer matmul of the unpacked
#      codes and weights that shares nothing with the product kernels (torch._int_mm / fp64 matmul:
#      both exact here), and every bf16 output against the fp64 expression of the contract evaluated
#      in torch from those accumulators;
#   3. the ORACLE's GEMM and epilogue on sampled rows: at least one row in every 128-row CTA half,
#      rotating through the four 32-lane TMEM quarters, plus the first and last rows.
_ACT_CACHE = {}


def cached_layer(config, name):
    from baseq_inputs import CONFIGS
    sp = [s_ for s_ in CONFIGS[config] if s_.name == name][0]
    key = (config, sp.act)
    if key not in _ACT_CACHE:
        if len(_ACT_CACHE) >= 2:
            _ACT_CACHE.pop(next(iter(_ACT_CACHE)))
        _ACT_CACHE[key] = make_activations(config, sp.act)
    L = {"spec": sp}
    L.update(_ACT_CACHE[key])
    L.update(make_weights(config, name))
    return L


def half_rows(T):
    """One row per 128-row CTA half h, in lane quarter h mod 4, plus the first and last rows."""
    rows = [128 * h + 32 * (h % 4) + (7 * h) % 32 for h in range((T + 127) // 128)]
    rows = [r if r < T else T - 1 for r in rows]
    return np.unique(np.r_[0:2, rows, 255:258, T - 2:T].clip(0, T - 1))


def gpu_unpack(nib, signed=True):
    """[R, K/2] packed nibbles (device uint8) -> [R, K] int8 on the device."""
    lo = (nib & 0xF).to(torch.int16)
    hi = (nib >> 4).to(torch.int16)
    if signed:
        lo = torch.where(lo >= 8, lo - 16, lo)
        hi = torch.where(hi >= 8, hi - 16, hi)
    return torch.stack([lo, hi], dim=2).reshape(nib.shape[0], -1).to(torch.int8)


def int_matmul(qa, qw):
    """acc[t, n] = sum_k qa[t, k] qw[n, k], exact, independent of the product kernels."""
    try:
        if qa.shape[0] > 16:
            return torch._int_mm(qa, qw.t())
    except RuntimeError:
        pass
    out = torch.empty((qa.shape[0], qw.shape[0]), dtype=torch.int32, device=qa.device)
    wd = qw.to(torch.float64).t().contiguous()
    for r0 in range(0, qa.shape[0], 512):          # fp64: every partial sum is an integer < 2^53
        out[r0:r0 + 512] = (qa[r0:r0 + 512].to(torch.float64) @ wd).to(torch.int32)
    return out


def bf16_bits_from_f64(y):
    """One round-half-to-even from double to bf16 (round-to-odd to fp32 first), as int32 bit patterns."""
    f = y.to(torch.float32)
    fd = f.to(torch.float64)
    bits = f.view(torch.int32).to(torch.int64) & 0xFFFFFFFF
    over = fd.abs() > y.abs()                       # RN went away from zero: step back (truncate)
    bits = torch.where(over, bits - 1, bits)
    bits = bits | (fd != y).to(torch.int64)         # sticky bit
    return ((bits + 0x7FFF + ((bits >> 16) & 1)) >> 16).to(torch.int32)


def check_all_rows_on_device(codes, w_nibbles_dev, acc, y, scales, w_scale, fb, zeros=None, wsum=None):
    """Layer 2 of the full-size comparison (see above).  Unsettled outputs of the torch evaluation
    (it multiplies and adds in two roundings where the contract has one fma) go to the oracle."""
    qa = gpu_unpack(codes, signed=zeros is None)
    qw = gpu_unpack(w_nibbles_dev)
    if zeros is not None:
        # _int_mm takes signed bytes: recentre the unsigned codes and add 8 wsum back (exact)
        ref = int_matmul((qa.to(torch.int16) - 8).to(torch.int8), qw) + 8 * wsum.to(torch.int32)[None, :]
    else:
        ref = int_matmul(qa, qw)
    nbad = int((ref != acc).sum())
    assert nbad == 0, "%d of %d int32 accumulators differ from the integer matmul" % (nbad, acc.numel())
    sw64, fb64 = w_scale.to(torch.float64), fb.to(torch.float64)
    bad_idx = []
    for r0 in range(0, acc.shape[0], 1024):
        a = acc[r0:r0 + 1024].to(torch.float64)
        p = scales[r0:r0 + 1024].to(torch.float64)[:, None] * sw64[None, :]            # exact
        c = fb64[None, :]
        if zeros is not None:
            c = (zeros[r0:r0 + 1024].to(torch.float64)[:, None] * sw64[None, :]) * wsum.to(torch.float64)[None, :] + c
        want = bf16_bits_from_f64(p * a + c)
        got = y[r0:r0 + 1024].view(torch.int16).to(torch.int32) & 0xFFFF
        d = (want != got).nonzero()
        if d.numel():
            d[:, 0] += r0
            bad_idx.append(d)
    if bad_idx:
        bad = torch.cat(bad_idx).cpu().numpy()
        assert len(bad) <= 64, "%d bf16 outputs differ from the fp64 expression" % len(bad)
        yh = bits_host(y)
        acch, sch, swh, fbh = acc.cpu().numpy(), scales.cpu().numpy(), w_scale.cpu().numpy(), fb.cpu().numpy()
        for t, n in bad:                                   # settle each one with the oracle's epilogue
            if zeros is None:
                o = oracle.epilogue(acch[t:t + 1, n:n + 1].copy(), sch[t:t + 1].copy(), swh[n:n + 1].copy(),
                                    fbh[n:n + 1].copy())
            else:
                o = oracle.epilogue_asym(acch[t:t + 1, n:n + 1].copy(), wsum.cpu().numpy()[n:n + 1].astype(np.int32),
                                         sch[t:t + 1].copy(), zeros.cpu().numpy()[t:t + 1].copy(),
                                         swh[n:n + 1].copy(), fbh[n:n + 1].copy())
            assert o[0, 0] == yh[t, n], (t, n)


def check_full(config, name, fused=False, gamma=None, sa_seed=None, asym=False):
    L = cached_layer(config, name)
    sp = L["spec"]
    T, N, K = sp.T, sp.N, sp.K
    gamma = sp.gamma if gamma is None else gamma
    sa = None
    if sa_seed is not None:
        sa = (1.0 + 0.1 * np.random.default_rng(sa_seed).standard_normal(K)).astype(np.float32)
    rows = half_rows(T)
    fb = oracle.fused_bias(L["w_nibbles"], L["w_scale"], L["b"], L["layer_bias"])
    wn_dev = dev(L["w_nibbles"])
    pw = bq.pack_weights(wn_dev, dev(L["w_scale"]), dev(L["b"]),
                         None if L["layer_bias"] is None else dev(L["layer_bias"]))
    params = bq.ActParams(sp.alpha, gamma, None if sa is None else dev(sa), dev(L["b"]), sp.had_block)
    xd = bf16_dev(L["x"])
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    zeros = None
    if fused:
        y, scales = bq.linear_fused(xd, params, pw)                       # timed configuration
        codes = torch.zeros((T, K // 2), dtype=torch.uint8, device="cuda")
        y2, scales2 = bq.linear_fused(xd, params, pw, codes_dump=codes, acc_dump=acc)
        assert torch.equal(scales, scales2)
    elif asym:
        codes, scales, zeros = bq.quantize_act_asym(xd, params)
        y = bq.w4a4_gemm_asym(codes, scales, zeros, pw)
        y2 = bq.w4a4_gemm_asym(codes, scales, zeros, pw, acc_dump=acc)
    else:
        codes, scales = bq.quantize_act(xd, params)
        y = bq.w4a4_gemm(codes, scales, pw)                               # timed configuration
        y2 = bq.w4a4_gemm(codes, scales, pw, acc_dump=acc)
    bq.sync_status()
    assert torch.equal(y.view(torch.int16), y2.view(torch.int16))
    assert np.array_equal(pw.fused_bias.cpu().numpy().view(np.uint32), fb.view(np.uint32))
    # 1. the oracle's quantiser on every row
    if asym:
        ocodes, oscales, ozeros = oracle.quantize_act_asym(L["x"], sp.alpha, gamma, sa, L["b"], sp.had_block)
        assert np.array_equal(zeros.cpu().numpy().view(np.uint32), ozeros.view(np.uint32))
    else:
        ocodes, oscales = oracle.quantize_act(L["x"], sp.alpha, gamma, sa, L["b"], sp.had_block)
    assert np.array_equal(scales.cpu().numpy().view(np.uint32), oscales.view(np.uint32)), "scales differ"
    cbad = int((codes.cpu().numpy() != ocodes).sum())
    assert cbad == 0, "%s/%s: %d code bytes differ from the oracle" % (config, name, cbad)
    # 2. every accumulator and every output, on the device
    wsum = None
    if asym:
        wsum = gpu_unpack(wn_dev).to(torch.int32).sum(dim=1)
    check_all_rows_on_device(codes, wn_dev, acc, y, scales, dev(L["w_scale"]), dev(fb), zeros, wsum)
    # 3. the oracle's GEMM and epilogue on the sampled rows
    rsel = torch.from_numpy(rows).cuda()
    if asym:
        oacc, owsum = oracle.gemm_i32_asym(np.ascontiguousarray(ocodes[rows]), L["w_nibbles"])
        oy = oracle.epilogue_asym(oacc, owsum, np.ascontiguousarray(oscales[rows]),
                                  np.ascontiguousarray(ozeros[rows]), L["w_scale"], fb)
    else:
        oacc = oracle.gemm_i32(np.ascontiguousarray(ocodes[rows]), L["w_nibbles"])
        oy = oracle.epilogue(oacc, np.ascontiguousarray(oscales[rows]), L["w_scale"], fb)
    assert np.array_equal(acc[rsel].cpu().numpy(), oacc), "%s/%s: sampled accumulators differ" % (config, name)
    gy = bits_host(y[rsel])
    nbad = int((gy != oy).sum())
    assert nbad == 0, "%s/%s: %d of %d sampled bf16 outputs differ" % (config, name, nbad, gy.size)


ALL_LAYERS = [("c2", "qkvo"), ("c3", "up"), ("c3", "gate"), ("c3", "down"), ("c4", "q"), ("c4", "k"),
              ("c4", "v"), ("c4", "o"), ("c4", "up"), ("c4", "gate"), ("c4", "down"), ("c5", "down")]


@pytest.mark.parametrize("config,name", ALL_LAYERS)
def test_full_size_all_layers(config, name):
    check_full(config, name)


@pytest.mark.parametrize("config,name", [("c3", "down"), ("c4", "k"), ("c5", "down")])
def test_full_size_fused(config, name):
    # north_star config 5 "exercises the fused quantize-in-producer GEMM path at a large K"
    check_full(config, name, fused=True)


def test_full_size_gamma_and_per_channel_sa():
    # the C-12 grid picks gamma = 1.00 for c3; a scalar s^a != 1 and a per-channel s^a vector
    # (Eq. 15) at full size: K = 4096 (split ring kernel) and K = 11008
    check_full("c3", "down", gamma=1.1)
    check_full("c2", "qkvo", sa_seed=71)
    check_full("c3", "down", sa_seed=72)
    check_full("c3", "down", fused=True, sa_seed=73)


@pytest.mark.parametrize("config,name", [("c3", "up"), ("c4", "down"), ("c5", "down")])
def test_full_size_asym(config, name):
    check_full(config, name, asym=True)


@pytest.mark.parametrize("mode", ["sym", "asym", "fused"])
def test_multi_tile_persistent_loop_full_compare(mode):
    # 10 x 22 = 220 tiles of 256 x 192 on 74 CTA pairs: three tiles per pair, so the accumulator
    # ping-pong wraps, the column-operand buffers and the Y staging tiles are reused and the flat
    # k-block phases run across tile boundaries -- every element compared with the ORACLE.
    # Ragged in T (2500 = 9 x 256 + 196) and in N (4040 = 21 x 192 + 8).
    T, K, N = 2500, 384, 4040
    rng = np.random.default_rng(2500 + len(mode))
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    if mode == "sym":
        run_linear(x, W, 0.9, 1.05, b)
    elif mode == "asym":
        run_asym(x, W, 0.9, 1.05, b)
    else:
        run_fused(x, W, 0.9, 1.05, b)


def test_back_to_back_set_fused_bias_quantise_decode_no_sync():
    # set_fused_bias -> ring quantiser (K = 4096, triggers its dependents early) ->
    # decode GEMM with no synchronisation in between; the decode kernel must not read fb before its
    # griddepcontrol.wait.  fb alternates between two vectors, every output is checked.
    rng = np.random.default_rng(4242)
    T, K, N = 16, 4096, 1024
    x = bf16_dev(rand_x(rng, T, K))
    W = _rand_w(rng, N, K, bias=False)
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]))
    params = bq.ActParams(0.9)
    fbs = [dev(rng.standard_normal(N).astype(np.float32)) for _ in range(2)]
    want = []
    for fbv in fbs:
        pw.set_fused_bias(fbv)
        torch.cuda.synchronize()
        codes, scales = bq.quantize_act(x, params)
        want.append(bq.w4a4_gemm(codes, scales, pw).clone())
        torch.cuda.synchronize()
    assert not torch.equal(want[0], want[1])
    codes = torch.empty((T, K // 2), dtype=torch.uint8, device="cuda")
    scales = torch.empty((T,), dtype=torch.float32, device="cuda")
    ys = [torch.empty((T, N), dtype=torch.bfloat16, device="cuda") for _ in range(40)]
    for i, y in enumerate(ys):
        bq.lib().baseq_set_fused_bias(pw.blob.data_ptr(), N, K, fbs[i % 2].data_ptr(),
                                      torch.cuda.current_stream().cuda_stream)
        bq.quantize_act(x, params, codes, scales)
        bq.w4a4_gemm(codes, scales, pw, y)
    torch.cuda.synchronize()
    for i, y in enumerate(ys):
        assert torch.equal(y.view(torch.int16), want[i % 2].view(torch.int16)), i


def test_mismatched_blob_is_refused_on_the_device():
    # a blob packed for another (N, K): the GEMM kernels compare the header, do no work, leave Y
    # untouched and raise the status word (baseq_sync_status -> BASEQ_ERR_WORKSPACE)
    rng = np.random.default_rng(5150)
    K, N = 384, 264
    W = _rand_w(rng, N, K)
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]))
    bq.sync_status()
    for T in (8, 130):                                   # decode kernel, tcgen05 kernel
        codes, scales = bq.quantize_act(bf16_dev(rand_x(rng, T, K)), bq.ActParams(0.9))
        y = torch.full((T, 200), 3.0, dtype=torch.bfloat16, device="cuda")
        wrong = bq.PackedWeight(pw.blob, 200, K, None)    # same K, smaller N: reads stay in bounds
        bq.w4a4_gemm(codes, scales, wrong, y)
        with pytest.raises(bq.BaseqError) as e:
            bq.sync_status()
        assert e.value.status == 5
        assert torch.all(y == 3.0)
        bq.sync_status()                                 # the word was cleared
        y_ok = bq.w4a4_gemm(codes, scales, pw)
        bq.sync_status()
        ref = oracle.gemm_i32(codes.cpu().numpy(), W["w_nibbles"])
        oy = oracle.epilogue(ref, scales.cpu().numpy(), W["w_scale"],
                             oracle.fused_bias(W["w_nibbles"], W["w_scale"], None, None))
        assert np.array_equal(bits_host(y_ok), oy)


def test_config5_fused_hadamard_small_T():
    A = make_activations("c5", "x_down", T=70)
    rng = np.random.default_rng(55)
    W = _rand_w(rng, 200, 28672, bias=False)
    run_fused(A["x"], W, 0.9, 1.0, A["b"], had_block=128)


# ------------------------------------------------------------------------------- randomised sweep
def test_random_shapes_and_parameters():
    """Seeded random (T, K, N, alpha, gamma, Hadamard block, bias on/off) cases, both paths."""
    rng = np.random.default_rng(20260604)
    for case in range(14):
        T = int(rng.integers(1, 400))
        K = 128 * int(rng.integers(1, 24))
        N = 8 * int(rng.integers(1, 80))
        alpha = float(rng.choice([1.0, 0.9, 0.75, 0.5]))
        gamma = float(rng.choice([1.0, 1.05, 1.2]))
        pow2 = [b for b in (2, 8, 32, 128) if K % b == 0]
        B = int(rng.choice([0, 0] + pow2))
        x = rand_x(rng, T, K, spread=float(rng.choice([0.0, 0.5, 2.0])))
        b = (0.5 * rng.standard_normal(K)).astype(np.float32) if rng.random() < 0.8 else None
        W = _rand_w(rng, N, K, bias=bool(rng.random() < 0.5))
        run_linear(x, W, alpha, gamma, b, had_block=B, with_bias=W["layer_bias"] is not None)
        run_fused(x, W, alpha, gamma, b, had_block=B)


# ------------------------------------------------------------------------------- NEXT-1: asymmetric
def run_asym(x_bits, W, alpha, gamma, b, had_block=0, rows=None, sa=None):
    """baseq_quantize_act_asym + baseq_w4a4_gemm_asym vs the oracle, everything bit for bit."""
    N, K = W["N"], W["K"]
    T = x_bits.shape[0]
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), None if b is None else dev(b),
                         None if W["layer_bias"] is None else dev(W["layer_bias"]))
    params = bq.ActParams(alpha, gamma, None if sa is None else dev(sa), None if b is None else dev(b),
                          had_block)
    codes, scales, zeros = bq.quantize_act_asym(bf16_dev(x_bits), params)
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    y = bq.w4a4_gemm_asym(codes, scales, zeros, pw, acc_dump=acc)
    y2 = bq.w4a4_gemm_asym(codes, scales, zeros, pw)
    torch.cuda.synchronize()
    assert torch.equal(y.view(torch.int16), y2.view(torch.int16))
    sel = np.arange(T) if rows is None else rows
    ref = oracle.linear_asym(np.ascontiguousarray(x_bits[sel]), W["w_nibbles"], W["w_scale"], fb,
                             alpha, gamma, sa, b, had_block)
    assert np.array_equal(scales.cpu().numpy()[sel].view(np.uint32), ref["scales"].view(np.uint32))
    assert np.array_equal(zeros.cpu().numpy()[sel].view(np.uint32), ref["zeros"].view(np.uint32))
    assert np.array_equal(codes.cpu().numpy()[sel], ref["codes"])
    assert np.array_equal(acc.cpu().numpy()[sel], ref["acc"])
    gy = bits_host(y)[sel]
    nbad = int((gy != ref["y"]).sum())
    assert nbad == 0, "asym bf16 output differs at %d of %d places" % (nbad, gy.size)


def run_fused_asym(x_bits, W, alpha, gamma, b, had_block=0, sa=None):
    """baseq_linear_fused_asym vs the oracle AND vs the two asymmetric calls, everything bit for bit."""
    N, K = W["N"], W["K"]
    T = x_bits.shape[0]
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), None if b is None else dev(b),
                         None if W["layer_bias"] is None else dev(W["layer_bias"]))
    params = bq.ActParams(alpha, gamma, None if sa is None else dev(sa), None if b is None else dev(b),
                          had_block)
    x = bf16_dev(x_bits)
    codes = torch.zeros((T, K // 2), dtype=torch.uint8, device="cuda")
    acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
    y, scales, zeros = bq.linear_fused_asym(x, params, pw, codes_dump=codes, acc_dump=acc)
    y2, _, _ = bq.linear_fused_asym(x, params, pw)                    # timed configuration: no dumps
    c3, s3, z3 = bq.quantize_act_asym(x, params)
    y3 = bq.w4a4_gemm_asym(c3, s3, z3, pw)
    torch.cuda.synchronize()
    assert torch.equal(y.view(torch.int16), y2.view(torch.int16))
    assert torch.equal(y.view(torch.int16), y3.view(torch.int16))
    assert torch.equal(codes, c3) and torch.equal(scales, s3) and torch.equal(zeros, z3)
    ref = oracle.linear_asym(x_bits, W["w_nibbles"], W["w_scale"], fb, alpha, gamma, sa, b, had_block)
    assert np.array_equal(scales.cpu().numpy().view(np.uint32), ref["scales"].view(np.uint32))
    assert np.array_equal(zeros.cpu().numpy().view(np.uint32), ref["zeros"].view(np.uint32))
    assert np.array_equal(codes.cpu().numpy(), ref["codes"])
    assert np.array_equal(acc.cpu().numpy(), ref["acc"])
    assert np.array_equal(bits_host(y), ref["y"])


@pytest.mark.parametrize("T,K,N,B", [(1, 128, 8, 0), (130, 384, 264, 0), (257, 1024, 520, 128),
                                     (300, 2048, 200, 16), (700, 4096, 392, 0), (520, 1280, 136, 256)])
def test_fused_asym_shapes(T, K, N, B):
    # the single-launch variant with asymmetric activations: pipelined chunks with and without the
    # Hadamard-128, generic steps (other block sizes), gamma a bf16 value and not
    rng = np.random.default_rng(31 * T + 3 * K + 5 * N + B)
    x = rand_x(rng, T, K, spread=1.0)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    run_fused_asym(x, _rand_w(rng, N, K), 0.9, 1.0 if T % 2 else 1.05, b, had_block=B)


def test_fused_asym_per_channel_sa_and_offsets():
    rng = np.random.default_rng(41)
    T, K, N = 70, 512, 136
    x = f32_to_bf16_bits((5.0 + rng.standard_normal((T, K))).astype(np.float32))     # far from zero
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    run_fused_asym(x, _rand_w(rng, N, K, bias=False), 1.0, 1.0, None, sa=sa)


def test_fused_asym_full_size_c3_up():
    L = cached_layer("c3", "up")
    sp = L["spec"]
    pw = bq.pack_weights(dev(L["w_nibbles"]), dev(L["w_scale"]), dev(L["b"]),
                         None if L["layer_bias"] is None else dev(L["layer_bias"]))
    params = bq.ActParams(sp.alpha, sp.gamma, None, dev(L["b"]), sp.had_block)
    x = bf16_dev(L["x"])
    y, scales, zeros = bq.linear_fused_asym(x, params, pw)
    c3, s3, z3 = bq.quantize_act_asym(x, params)
    y3 = bq.w4a4_gemm_asym(c3, s3, z3, pw)
    torch.cuda.synchronize()
    # the two-call path is checked against the oracle at full size by test_full_size_asym
    assert torch.equal(scales, s3) and torch.equal(zeros, z3)
    assert torch.equal(y.view(torch.int16), y3.view(torch.int16))


def test_asym_config1():
    L = make_layer("c1", "linear")
    sp = L["spec"]
    run_asym(L["x"], L, sp.alpha, sp.gamma, L["b"])


@pytest.mark.parametrize("T,K,N,B", [(1, 128, 8, 0), (130, 384, 264, 0), (257, 1024, 520, 128),
                                     (70, 4096, 200, 0), (33, 11008, 136, 0), (9, 28672, 64, 128)])
def test_asym_shapes(T, K, N, B):
    rng = np.random.default_rng(3 * T + 5 * K + 7 * N + B)
    x = rand_x(rng, T, K, spread=1.0)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    run_asym(x, _rand_w(rng, N, K), 0.9, 1.05, b, had_block=B)


def test_asym_degenerate_rows_and_offsets():
    # constant rows (floor scale), all-positive rows far from zero, and alpha = 1 (no clipping)
    rng = np.random.default_rng(41)
    K, N = 512, 72
    x = np.zeros((6, K), dtype=np.float32)
    x[0] = 5.0
    x[1] = rng.random(K) + 100.0
    x[2] = -rng.random(K) - 50.0
    x[3] = rng.standard_normal(K)
    x[4] = 0.0
    x[5] = np.arange(K) % 16
    W = _rand_w(rng, N, K, bias=False)
    run_asym(f32_to_bf16_bits(x), W, 1.0, 1.0, None)
    run_asym(f32_to_bf16_bits(x), W, 0.5, 1.0, None)


@pytest.mark.parametrize("T,K,N,B", [(9, 256, 72, 0), (70, 4096, 136, 0), (33, 11008, 72, 0),
                                     (12, 14336, 64, 128), (5, 28672, 64, 128)])
def test_asym_per_channel_sa(T, K, N, B):
    # NEXT-4 second half: the per-channel s^a vector (Eq. 15) through the asymmetric
    # quantiser (the paper's deployed setting), every ring-kernel instantiation family
    rng = np.random.default_rng(17 * T + K + N + B)
    x = rand_x(rng, T, K, spread=1.0)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    run_asym(x, _rand_w(rng, N, K), 0.9, 1.0, b, had_block=B, sa=sa)


# =========================================================================== NEXT-3: KV cache
def run_kv(x_bits, H, D, alpha, ldx=None, rows=None):
    """baseq_quantize_kv vs oracle.quantize_kv: codes, scales, zeros bit for bit."""
    T = x_bits.shape[0]
    if ldx is None:
        xd = bf16_dev(x_bits)
    else:                                    # row stride larger than H * D: the extra columns are junk
        pad = np.full((T, ldx), 0x7FC0, dtype=np.uint16)          # NaNs that must never be read
        pad[:, :H * D] = x_bits
        xd = bf16_dev(pad)[:, :H * D]
    codes, scales, zeros = bq.quantize_kv(xd, H, D, alpha)
    torch.cuda.synchronize()
    sel = np.arange(T) if rows is None else rows
    rc, rs, rz = oracle.quantize_kv(np.ascontiguousarray(x_bits[sel]), H, D, alpha)
    assert np.array_equal(scales.cpu().numpy()[sel].view(np.uint32), rs.view(np.uint32))
    assert np.array_equal(zeros.cpu().numpy()[sel].view(np.uint32), rz.view(np.uint32))
    assert np.array_equal(codes.cpu().numpy()[sel], rc)


@pytest.mark.parametrize("T,H,D", [(1, 1, 64), (1, 1, 128), (7, 3, 128), (33, 8, 128), (130, 32, 64),
                                   (5, 5, 64), (257, 9, 128)])
def test_kv_shapes(T, H, D):
    rng = np.random.default_rng(11 * T + 13 * H + D)
    x = rand_x(rng, T, H * D, spread=1.0)
    for alpha in (1.0, 0.9):
        run_kv(x, H, D, alpha)


def test_kv_strided_rows_and_degenerate_groups():
    rng = np.random.default_rng(77)
    T, H, D = 19, 4, 128
    x = rand_x(rng, T, H * D, spread=1.0)
    xf = (x.astype(np.uint32) << 16).view(np.float32).copy()
    xf[0, :D] = 3.5                      # constant head: floor scale, z = the value, codes 0
    xf[1, D:2 * D] = 0.0                 # all-zero head
    xf[2, 2 * D:3 * D] = np.abs(xf[2, 2 * D:3 * D]) + 100.0     # all positive, far from zero
    xf[3, 3 * D:] *= 1e-30               # tiny magnitudes
    xb = (xf.view(np.uint32) >> 16).astype(np.uint16)           # truncation: still bf16 patterns
    run_kv(xb, H, D, 1.0)
    run_kv(xb, H, D, 0.9, ldx=H * D + 64)


def test_kv_full_size_sampled_rows():
    # Llama-3-8B K or V of an 8192-token prefill (8 KV heads x 128) and Llama-2-7B (32 x 128, T = 4096)
    for T, H, D, seed in ((8192, 8, 128, 5), (4096, 32, 128, 6)):
        rng = np.random.default_rng(seed)
        x = rand_x(rng, T, H * D, spread=1.0)
        rows = np.unique(np.concatenate([np.arange(4), rng.integers(0, T, 24), np.arange(T - 4, T)]))
        run_kv(x, H, D, 0.9, rows=rows)


def test_kv_rejects_other_head_dims():
    x = torch.zeros((4, 96 * 2), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(bq.BaseqError):
        bq.quantize_kv(x, 2, 96)


# ------------------------------------------------------------------------------- clip ratios below 2^-16
def _tiny_alpha_x(rng, T, K):
    # N(0.3, 1) rows with a fifth of the entries scaled down to the size of the step alpha * max / 7,
    # so that codes other than the saturated ones occur
    x = 0.3 + rng.standard_normal((T, K))
    small = rng.random((T, K)) < 0.2
    x[small] *= 1e-6
    return f32_to_bf16_bits(x.astype(np.float32))


@pytest.mark.parametrize("alpha", [2.0 ** -17, 2.0 ** -20, 1e-9])
def test_small_alpha_every_entry_point(alpha):
    # include/baseq.h allows 0 < alpha <= 1; below 2^-16 the clamping kernel (quantize_small_alpha.cu)
    # takes over behind every entry point: same contract, same bits as the oracle
    rng = np.random.default_rng(int(-np.log2(alpha)))
    T, K, N = 75, 1024, 200
    x = _tiny_alpha_x(rng, T, K)
    b = (1e-7 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    for B in (0, 128, 256):
        check_quant(x, alpha, 1.05, None, b, B)
        run_linear(x, W, alpha, 1.0, b, had_block=B)
        run_asym(x, W, alpha, 1.0, b, had_block=B)
        run_fused(x, W, alpha, 1.0, b, had_block=B)
        run_fused_asym(x, W, alpha, 1.05, b, had_block=B)
    sa = (1.0 + 0.1 * rng.standard_normal(K)).astype(np.float32)
    check_quant(x, alpha, 1.0, sa, None)
    # the ring kernels' shapes route there too
    x2 = _tiny_alpha_x(rng, 9, 11008)
    check_quant(x2, alpha, 1.0, None, (1e-7 * rng.standard_normal(11008)).astype(np.float32))
    # KV cache: (token, head) groups, strided rows
    xk = _tiny_alpha_x(rng, 33, 5 * 128)
    run_kv(xk, 5, 128, alpha)
    run_kv(_tiny_alpha_x(rng, 17, 3 * 64), 3, 64, alpha, ldx=3 * 64 + 24)
    # the tensor-core Hadamard variant keeps the limit
    with pytest.raises(bq.BaseqError) as e:
        bq.quantize_act_tc(bf16_dev(x), bq.ActParams(alpha, 1.0, None, dev(b), 128))
    assert e.value.status == 6


def test_small_alpha_static_entry_point():
    rng = np.random.default_rng(5)
    T, K, N = 40, 512, 72
    x_bits = _tiny_alpha_x(rng, T, K)
    W = _rand_w(rng, N, K)
    b = (1e-7 * rng.standard_normal(K)).astype(np.float32)
    alpha = 2.0 ** -18
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
    y = torch.empty((T, N), dtype=torch.bfloat16, device="cuda")
    bq.linear_static(bf16_dev(x_bits), bq.ActParams(alpha, 1.0, None, dev(b), 0), pw, y)
    torch.cuda.synchronize()
    ref = oracle.linear(x_bits, W["w_nibbles"], W["w_scale"], fb, alpha, 1.0, None, b, 0)
    assert np.array_equal(bits_host(y), ref["y"])


# ------------------------------------------------------------------------------- NEXT-4: decode shapes
# T <= 64 takes the W-streaming decode kernel (w4a4_decode.cu) behind the same baseq_w4a4_gemm /
# baseq_w4a4_gemm_asym calls; same contract, same bits.
@pytest.mark.parametrize("T", [1, 7, 8, 9, 16, 17, 32, 33, 63, 64])
def test_decode_token_counts(T):
    # every token-tile instantiation (8 / 16 / 32 / 64), ragged token tails, N % 16 == 8,
    # K = 11 k-blocks (8 warps: three take two k-blocks, five take one)
    rng = np.random.default_rng(100 + T)
    K, N = 1408, 200
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    run_linear(x, W, 0.9, 1.05, b)
    run_asym(x, W, 0.9, 1.05, b)


@pytest.mark.parametrize("T,K,N", [(1, 128, 8), (5, 256, 96), (64, 4096, 112), (16, 11008, 208),
                                   (24, 28672, 64), (40, 4224, 1000)])
def test_decode_k_and_n_edges(T, K, N):
    # one k-block (seven idle warps), several rounds of the in-flight window (K = 28672: 224
    # k-blocks), row groups at the end of / across 96-row weight boxes, N below one group
    rng = np.random.default_rng(T + 3 * K + 11 * N)
    x = rand_x(rng, T, K, spread=1.0)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    run_linear(x, W, 0.9, 1.0, b)
    run_asym(x, W, 1.0, 1.0, b)


@pytest.mark.parametrize("T,K,N", [(8, 28672, 64), (3, 6144, 72), (16, 6144, 40), (8, 8192, 7112),
                                   (5, 512, 7120), (2, 1280, 7104), (6, 3072, 7104), (1, 11008, 7104)])
def test_decode_straight_line_pieces(T, K, N):
    # T <= 16 walks a warp's k-blocks in branch-free pieces (w4a4_decode.cu): every piece kind --
    # several full pieces + an exact short one (K = 28672: 28 k-blocks per warp), a masked full piece
    # (K = 6144: 6), a masked short one, warps without any k-block (K = 512) -- and, for T <= 8 and
    # N >= 48 x 148, the two-groups-per-CTA instantiation (window of 2: full + full, exact short,
    # masked full at K = 3072, full + masked at K = 11008), N % 32 != 0 included
    rng = np.random.default_rng(7 * T + 3 * K + 11 * N)
    x = rand_x(rng, T, K, spread=1.0)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    run_linear(x, W, 0.9, 1.0, b)
    run_asym(x, W, 1.0, 1.0, b)


def test_decode_extreme_codes():
    # largest raw accumulators: qa = -8, qw = -8 -> acc = 64 K; qa = 7, qw = -8 -> -56 K (closed forms)
    T, K, N = 48, 28672, 64
    scales = torch.full((T,), 0.25, dtype=torch.float32, device="cuda")
    wn = np.full((N, K // 2), 0x88, dtype=np.uint8)
    pw = bq.pack_weights(dev(wn), dev(np.full((N,), 0.5, dtype=np.float32)))
    for byte, per_k in ((0x88, 64), (0x77, -56)):
        codes = torch.full((T, K // 2), byte, dtype=torch.uint8, device="cuda")
        acc = torch.empty((T, N), dtype=torch.int32, device="cuda")
        y = bq.w4a4_gemm(codes, scales, pw, acc_dump=acc)
        torch.cuda.synchronize()
        assert torch.all(acc == per_k * K)
        assert torch.all(y.float() == float(torch.tensor(per_k * K * 0.125).bfloat16()))


def test_decode_matches_prefill_kernel_on_shared_rows():
    # the same codes through both kernels: rows 0..T-1 of a 130-token call (tcgen05 GEMM) and a
    # T-token call (decode kernel) must agree bit for bit, Llama-2-7B q/k/v/o shape, full N
    L = make_layer("c2", "qkvo", T=130)
    sp = L["spec"]
    pw = bq.pack_weights(dev(L["w_nibbles"]), dev(L["w_scale"]), dev(L["b"]),
                         None if L["layer_bias"] is None else dev(L["layer_bias"]))
    params = bq.ActParams(sp.alpha, sp.gamma, None, dev(L["b"]), sp.had_block)
    codes, scales = bq.quantize_act(bf16_dev(L["x"]), params)
    y_big = bq.w4a4_gemm(codes, scales, pw)
    for T in (1, 8, 20, 64):
        acc = torch.empty((T, sp.N), dtype=torch.int32, device="cuda")
        y = bq.w4a4_gemm(codes[:T].contiguous(), scales[:T].contiguous(), pw, acc_dump=acc)
        torch.cuda.synchronize()
        assert torch.equal(y.view(torch.int16), y_big[:T].view(torch.int16)), T
    # and against the oracle on the first two tokens
    fb = oracle.fused_bias(L["w_nibbles"], L["w_scale"], L["b"], L["layer_bias"])
    ref = oracle.linear(np.ascontiguousarray(L["x"][:2]), L["w_nibbles"], L["w_scale"], fb,
                        sp.alpha, sp.gamma, None, L["b"], sp.had_block)
    assert np.array_equal(bits_host(y_big[:2]), ref["y"])


def test_decode_strided_output():
    # ldy > N and guard rows around Y / acc_dump: the decode kernel writes only the T x N outputs
    rng = np.random.default_rng(77)
    K, N = 512, 136
    for T in (3, 12, 30, 57):
        x = rand_x(rng, T, K)
        W = _rand_w(rng, N, K)
        pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), None, dev(W["layer_bias"]))
        codes, scales = bq.quantize_act(bf16_dev(x), bq.ActParams(0.9))
        acc_ref = torch.empty((T, N), dtype=torch.int32, device="cuda")
        y_ref = bq.w4a4_gemm(codes, scales, pw, acc_dump=acc_ref)
        buf = torch.full((T + 2, 160), -1.0, dtype=torch.bfloat16, device="cuda")
        accbuf = torch.full((T + 2, N), -7, dtype=torch.int32, device="cuda")
        bq.w4a4_gemm(codes, scales, pw, y=buf[1:T + 1, :N], acc_dump=accbuf[1:T + 1])
        torch.cuda.synchronize()
        assert torch.equal(buf[1:T + 1, :N].contiguous().view(torch.int16), y_ref.view(torch.int16))
        assert torch.all(buf[1:T + 1, N:] == -1.0) and torch.all(buf[0] == -1.0) and torch.all(buf[T + 1] == -1.0)
        assert torch.equal(accbuf[1:T + 1], acc_ref)
        assert torch.all(accbuf[0] == -7) and torch.all(accbuf[T + 1] == -7)


# ------------------------------------------------------------------------------- host-buffer entry
@pytest.mark.parametrize("T", [16, 130])
def test_linear_host_matches_oracle(T):
    # baseq_linear_host (bench.py's e2e leg): pinned host X in, pinned host Y out, H2D / quantise /
    # GEMM / D2H enqueued by the library; T = 16 takes the decode GEMM, T = 130 the tcgen05 one
    rng = np.random.default_rng(900 + T)
    K, N = 512, 264
    x = rand_x(rng, T, K)
    b = (0.5 * rng.standard_normal(K)).astype(np.float32)
    W = _rand_w(rng, N, K)
    fb = oracle.fused_bias(W["w_nibbles"], W["w_scale"], b, W["layer_bias"])
    pw = bq.pack_weights(dev(W["w_nibbles"]), dev(W["w_scale"]), dev(b), dev(W["layer_bias"]))
    params = bq.ActParams(0.9, 1.05, None, dev(b), 0)
    x_host = torch.from_numpy(x.view(np.int16)).view(torch.bfloat16).pin_memory()
    y_host = torch.zeros((T, N), dtype=torch.bfloat16).pin_memory()
    scratch = torch.empty(bq.linear_host_scratch_bytes(T, N, K), dtype=torch.uint8, device="cuda")
    bq.linear_host(x_host, params, pw, y_host, scratch)
    torch.cuda.synchronize()
    ref = oracle.linear(x, W["w_nibbles"], W["w_scale"], fb, 0.9, 1.05, None, b, 0)
    assert np.array_equal(pw.fused_bias.cpu().numpy().view(np.uint32), fb.view(np.uint32))
    assert np.array_equal(y_host.view(torch.int16).numpy().view(np.uint16), ref["y"])

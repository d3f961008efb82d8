// Decode-shaped W4A4 GEMM: the same contract as w4a4_gemm.cu (steps a7-a9 of
// DESIGN.md; int32-exact accumulation, fp64 epilogue, bf16 out) for T <= 64 tokens, where the
// work is streaming the packed weights once (N K / 2 bytes) and the 128 x 192 tcgen05 tile would
// be 1-50 % full.  HBM-bound: algorithmic bytes = N K / 2 (W) + T K / 2 (codes) + 2 T N (Y).
//
//   CTA            MT groups of 16 output channels (MT = 2 for T > 16 and N >= 64 SMs, for T <= 8 and
//                  N >= 48 SMs, else 1; a group is 16 rows x
//                  64 bytes = 1 KB contiguous per k-block of the weight blob), all of K, all T
//                  tokens; grid = ceil(N / (16 MT))
//   8 warps        k-blocks w, w + 8, ... each, through a window of kDepth register slots (T <= 16:
//                  branch-free straight-line pieces, see the main loop; T > 16: a rolling window)
//                  (2 MT x LDG.128 per lane and k-block, streaming; the first window is issued
//                  BEFORE griddepcontrol.wait: the weights do not depend on the preceding
//                  quantiser, and griddepcontrol.launch_dependents right after it lets a following
//                  decode GEMM stream its weights while this one drains)
//   MMA            mma.sync.m16n8k32 s8 x s8 -> s32 with M = output channels, N = 8 tokens: at
//                  T <= 64 the contraction is 0.4-3 % of the tensor peak, the legacy warp-level MMA
//                  is ample and needs no shared-memory operand staging
//   expansion      a 32-bit word holds 8 nibbles; (w << 4) & 0xF0F0F0F0 and w & 0xF0F0F0F0 are the
//                  bytes 16 q of the even and odd nibbles (a signed nibble in the top half of a
//                  byte IS 16 q as int8).  Both operands are split the same way, so every k meets
//                  its partner (a permutation of k inside the dot product); raw = 256 acc exactly.
//                  Asymmetric codes (NEXT-1, unsigned) are re-centred to q - 8 by flipping the top
//                  bit, as in the tcgen05 kernel.
//   epilogue       the 8 partial sums meet in shared memory (integer atomics: order-free); every
//                  output is evaluated with the fp64 expression of the contract itself
//                  (<= 2048 outputs per CTA), 32-64 contiguous bytes of a Y row per half-warp / warp.
#include <type_traits>

#include "epilogue_math.cuh"
#include "kernels.cuh"
#include "ptx.cuh"

namespace baseq {
namespace {

constexpr int kRows = 16;          // output channels per CTA (MMA M)

struct DecodeParams {
  const uint32_t* header;   // blob header: magic, N, K, ... (checked against N, K)
  unsigned int* status;     // device status word
  const uint8_t* tiles;
  const float* sw;
  const float* fb;
  const float* wsum;
  const uint8_t* codes;     // [T, K/2]
  const float* scales;      // [T]
  const float* zeros;       // [T] (asymmetric) or nullptr
  uint16_t* y;
  int64_t ldy;
  int32_t* acc_dump;
  int T, N, K, num_kb;
};

__device__ __forceinline__ void mma_s8(int32_t (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                       uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, "
      "{%8, %9}, {%0, %1, %2, %3};"
      : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint32_t word(const uint4& v, int i) {
  return i == 0 ? v.x : i == 1 ? v.y : i == 2 ? v.z : v.w;
}

// NT = token tiles of 8 (T <= 8 NT); MT = groups of 16 output channels per CTA (a warp multiplies
// all of them with the same activation fragments); kWarps warps split K; kDepth k-blocks of W in
// flight per warp.
template <int NT, int MT, bool ASYM, int kWarps, int kDepth>
__global__ void __launch_bounds__(kWarps * 32, NT == 1 ? 3 : (NT * MT <= 8 ? 2 : 1)) w4a4_decode_kernel(const DecodeParams p) {
  constexpr int kThreads = kWarps * 32;
  constexpr int kCh = kRows * MT;                       // output channels per CTA
  constexpr int kOut = (NT * 8 * kCh + kThreads - 1) / kThreads;   // outputs per thread
  static_assert(kThreads % kCh == 0, "epilogue mapping");
  __shared__ int32_t red[MT * NT * 4 * 32];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t4 = lane & 3;
  const int n0 = blockIdx.x * kCh;
  // weight rows g and g + 8 of the first group, k-block 0 (boxes of kTileRows rows x 64 bytes);
  // group m is 16 rows = 1 KB further on in the same box
  const uint8_t* wrow = p.tiles +
      (static_cast<size_t>(n0 / kTileRows) * p.num_kb * kTileRows + (n0 % kTileRows) + g) * 64 + t4 * 16;

  // epilogue: this thread's outputs are one channel (ch) x tokens tok0 + i * (kThreads / kCh)
  const int ch = threadIdx.x % kCh, tok0 = threadIdx.x / kCh;
  const int n = n0 + ch;
  // requested with the first weight window, compared after the wait: a blob packed for another
  // (N, K) makes the whole grid write nothing and raises the status word (as in w4a4_gemm.cu)
  const uint4 hdr = ptx::ldg_nc(reinterpret_cast<const uint4*>(p.header));
  for (int i = threadIdx.x; i < MT * NT * 4 * 32; i += kThreads) red[i] = 0;

  int32_t acc[MT][NT][4];
#pragma unroll
  for (int m = 0; m < MT; ++m)
#pragma unroll
    for (int j = 0; j < NT; ++j)
#pragma unroll
      for (int c = 0; c < 4; ++c) acc[m][j][c] = 0;

  // this warp's k-blocks: warp, warp + kWarps, ... (`count` of them), consumed through a rolling
  // window of kDepth register slots: slot d is refilled with k-block it + kDepth as soon as
  // k-block it has been multiplied, so kDepth loads stay in flight until the row group ends
  const int count = (p.num_kb - warp + kWarps - 1) / kWarps;
  uint4 wa[kDepth][MT], wb[kDepth][MT];
  auto load_w = [&](int d, int it) {
    const uint8_t* src = wrow + static_cast<size_t>(warp + it * kWarps) * (kTileRows * 64);
#pragma unroll
    for (int m = 0; m < MT; ++m) {
      wa[d][m] = ptx::ldg_nc_stream(reinterpret_cast<const uint4*>(src + m * (kRows * 64)));
      wb[d][m] = ptx::ldg_nc_stream(reinterpret_cast<const uint4*>(src + m * (kRows * 64) + 8 * 64));
    }
  };
#pragma unroll
  for (int d = 0; d < kDepth; ++d) {
#pragma unroll
    for (int m = 0; m < MT; ++m) {
      wa[d][m] = make_uint4(0, 0, 0, 0);
      wb[d][m] = make_uint4(0, 0, 0, 0);
    }
    if (d < count) load_w(d, d);
  }
  // The first window of W is in flight.  Only the weight BOXES may be read up here: they are written
  // by the packer's retile kernel, which is followed by a fully serialised kernel boundary inside
  // baseq_pack_weights (its scales / fused-bias kernel is a plain launch), so they are complete and
  // visible before any programmatically launched kernel can start.  s_w, fb and wsum are written by
  // the LAST packer kernel and by baseq_set_fused_bias, possibly the direct predecessor of a
  // quantiser that triggers its dependents early: they are read after griddepcontrol.wait.
  // Let the next kernel of the stream start on the SMs this grid leaves free (a following decode
  // GEMM streams ITS weights meanwhile; every kernel of this library writes only after its own
  // griddepcontrol.wait), then wait for the preceding kernel: codes and scales are its output.
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  const bool blob_ok = hdr.x == kBlobMagic && hdr.y == static_cast<uint32_t>(p.N) &&
                       hdr.z == static_cast<uint32_t>(p.K);
  if (!blob_ok) {
    if (threadIdx.x == 0 && blockIdx.x == 0) atomicOr(p.status, kStatusBadBlob);
    return;
  }
  const bool n_ok = n < p.N;
  // per-channel epilogue operands from the blob header area
  const float sw = n_ok ? p.sw[n] : 0.0f, fb = n_ok ? p.fb[n] : 0.0f;
  const float ws = (ASYM && n_ok) ? p.wsum[n] : 0.0f;

  // per-token epilogue operands, requested with the first activation fragments: their L2 round
  // trip is over long before the partial sums meet
  float st[kOut], zt[kOut];
#pragma unroll
  for (int i = 0; i < kOut; ++i) {
    const int tok = tok0 + i * (kThreads / kCh);
    st[i] = tok < p.T ? p.scales[tok] : 0.0f;
    zt[i] = (ASYM && tok < p.T) ? p.zeros[tok] : 0.0f;
  }

  // T <= 16: the activation fragments travel with the window (one or two vectors per k-block), so
  // a k-block's MMAs never wait for an L2 round trip of their own; larger T loads them per k-block
  // (8 NT registers each)
  constexpr bool kXPre = NT <= 2;
  uint4 xs[kXPre ? kDepth : 1][NT];
  // kXPre: unconditional loads -- a token row beyond T is clamped to the last row (its accumulators
  // are never written out) -- so that the load sits in the same basic block as the MMAs that use it
  auto load_x = [&](uint4 (&dst)[NT], int it) {
#pragma unroll
    for (int j = 0; j < NT; ++j) {
      const uint8_t* src = p.codes + t4 * 16 + static_cast<size_t>(warp + it * kWarps) * 64;
      if (kXPre) {
        const int tok = j * 8 + g < p.T ? j * 8 + g : p.T - 1;
        dst[j] = ptx::ldg_nc(reinterpret_cast<const uint4*>(src + static_cast<size_t>(tok) * (p.K / 2)));
      } else {
        dst[j] = make_uint4(0, 0, 0, 0);
        if (j * 8 + g < p.T)
          dst[j] = ptx::ldg_nc(reinterpret_cast<const uint4*>(src + static_cast<size_t>(j * 8 + g) * (p.K / 2)));
      }
    }
  };
  if (kXPre) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d)
      if (d < count) load_x(xs[kXPre ? d : 0], d);
  }

  // The k-blocks of this warp in straight-line pieces without a single branch.  ptxas puts every
  // load whose value is consumed across a branch or a loop back-edge on ONE scoreboard, and the wait
  // for window slot d then also waits for the refill issued one k-block earlier: the rolling window
  // of round 1 (refills under `if (it + kDepth < count)`, consumed in the next loop iteration) ran
  // at one memory round trip per k-block for K > 4096 (decoded from the SASS control words; the
  // same effect as in the fused GEMM's background quantiser, w4a4_gemm.cu).  A full piece is
  // 2 kDepth k-blocks: the window it starts with, refilled once while it is consumed.  The window of
  // the NEXT piece is loaded at its start (the ring drains at piece boundaries).  The last, partial
  // piece is kDepth steps with the k-blocks beyond `count` clamped (loads) and zeroed (weights).
  auto step = [&](int d, int it, bool valid) {
    uint4 xa[NT];
    if (kXPre) {
#pragma unroll
      for (int j = 0; j < NT; ++j) xa[j] = xs[kXPre ? d : 0][j];
    } else {
      load_x(xa, it);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      uint32_t a0[MT], a1[MT], a2[MT], a3[MT];
#pragma unroll
      for (int m = 0; m < MT; ++m) {
        const uint32_t a = valid ? word(wa[d][m], i) : 0u, b = valid ? word(wb[d][m], i) : 0u;
        a0[m] = (a << 4) & 0xF0F0F0F0u, a2[m] = a & 0xF0F0F0F0u;
        a1[m] = (b << 4) & 0xF0F0F0F0u, a3[m] = b & 0xF0F0F0F0u;
      }
#pragma unroll
      for (int j = 0; j < NT; ++j) {
        const uint32_t x = word(xa[j], i);
        uint32_t b0 = (x << 4) & 0xF0F0F0F0u, b1 = x & 0xF0F0F0F0u;
        if (ASYM) {
          b0 ^= 0x80808080u;        // 16 q -> 16 (q - 8) as int8
          b1 ^= 0x80808080u;
        }
#pragma unroll
        for (int m = 0; m < MT; ++m) mma_s8(acc[m][j], a0[m], a1[m], a2[m], a3[m], b0, b1);
      }
    }
  };
  constexpr int kPiece = 2 * kDepth;
  const int last = count - 1;
  // kSteps k-blocks from `base`; the first kDepth are in the window (loaded by the prologue for
  // base = 0, here otherwise), the others are refilled while the piece runs.  kMasked: k-blocks
  // beyond `count` exist in the piece (clamped loads, zeroed weights).
  auto piece = [&](int base, auto steps_tag, auto masked_tag) {
    constexpr int kSteps = decltype(steps_tag)::value;
    constexpr bool kMasked = decltype(masked_tag)::value;
    auto clamp = [&](int it) { return (kMasked && it > last) ? last : it; };
    if (base > 0) {
#pragma unroll
      for (int d = 0; d < kDepth; ++d) {
        load_w(d, clamp(base + d));
        if (kXPre) load_x(xs[kXPre ? d : 0], clamp(base + d));
      }
    }
#pragma unroll
    for (int t = 0; t < kSteps; ++t) {
      const int d = t % kDepth;
      step(d, clamp(base + t), !kMasked || base + t < count);
      if (t + kDepth < kSteps) {
        load_w(d, clamp(base + t + kDepth));
        if (kXPre) load_x(xs[kXPre ? d : 0], clamp(base + t + kDepth));
      }
    }
  };
  using Full = std::integral_constant<int, kPiece>;
  using Short = std::integral_constant<int, kDepth>;
  if (kXPre) {
    int base = 0;
#pragma unroll 1
    for (; base + kPiece <= count; base += kPiece) piece(base, Full{}, std::false_type{});
    if (count - base > kDepth) {
      piece(base, Full{}, std::true_type{});
    } else if (count - base == kDepth) {
      piece(base, Short{}, std::false_type{});
    } else if (count - base > 0) {
      piece(base, Short{}, std::true_type{});
    }
  } else {
    // T > 16: the activation fragments are loaded per k-block and the MMAs dominate; the rolling
    // window in a loop measured 3-8 % faster here than the pieces (smaller code, no masked steps)
    for (int base = 0; base < count; base += kDepth) {
#pragma unroll
      for (int d = 0; d < kDepth; ++d) {
        const int it = base + d;
        if (it < count) {
          step(d, it, true);
          if (it + kDepth < count) load_w(d, it + kDepth);
        }
      }
    }
  }

  // the kWarps partial sums meet in shared memory (integer adds: any order, same result)
  __syncthreads();                                        // red is zero
#pragma unroll
  for (int m = 0; m < MT; ++m)
#pragma unroll
    for (int j = 0; j < NT; ++j)
#pragma unroll
      for (int c = 0; c < 4; ++c) atomicAdd(&red[((m * NT + j) * 4 + c) * 32 + lane], acc[m][j][c]);
  __syncthreads();

  // thread -> (token, channel): kCh consecutive threads write 2 kCh contiguous bytes of one Y row
#pragma unroll
  for (int i = 0; i < kOut; ++i) {
    const int tok = tok0 + i * (kThreads / kCh);
    if (tok >= NT * 8 || tok >= p.T || !n_ok) continue;
    // accumulator fragment: c0, c1 = row g, tokens 2 t4 + {0, 1}; c2, c3 = row g + 8
    const int j = tok >> 3, col = tok & 7, m = ch >> 4, r = ch & 15;
    const int idx = ((m * NT + j) * 4 + (r >> 3) * 2 + (col & 1)) * 32 + (r & 7) * 4 + (col >> 1);
    int32_t a = red[idx] >> 8;                             // raw = 256 acc exactly
    uint32_t out;
    if (ASYM) {
      out = epi::dequant_f64_asym(a, st[i], zt[i], sw, fb, ws);
      a += 8 * static_cast<int32_t>(ws);                   // the accumulator over the unsigned codes
    } else {
      out = epi::dequant_f64(a, st[i], sw, fb);
    }
    p.y[static_cast<size_t>(tok) * p.ldy + n] = static_cast<uint16_t>(out);
    if (p.acc_dump != nullptr) p.acc_dump[static_cast<size_t>(tok) * p.N + n] = a;
  }
}

// kDepth x MT = 4: the same bytes of W in flight per warp either way.
template <int NT, int MT, bool ASYM>
cudaError_t launch_nt(const DecodeParams& p, cudaStream_t stream) {
  constexpr int kWarps = 8, kThreads = kWarps * 32, kDepth = 4 / MT;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>((p.N + kRows * MT - 1) / (kRows * MT)), 1, 1);
  cfg.blockDim = dim3(kThreads, 1, 1);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, w4a4_decode_kernel<NT, MT, ASYM, kWarps, kDepth>, p);
}

// T <= 16: one 16-channel group per CTA.  T > 16: two groups per CTA share the activation
// fragments (half the L2 -> SM activation traffic and half the B-operand expansion); at T <= 32
// only where that still leaves two CTAs per SM (measured: at N = 4096 the halved grid of 128 CTAs
// costs more than the sharing saves there, and less at T = 64).
template <bool ASYM>
cudaError_t launch_asym(const DecodeParams& p, int num_sms, cudaStream_t stream) {
  const bool wide = p.N >= 2 * kRows * 2 * num_sms;
  // T <= 8: two groups per CTA (64 KB per CTA and k-sweep, half as many CTAs) where that still
  // leaves 1.5 CTAs per SM (measured with the straight-line pieces: c3 17.9 -> 15.7 us, c5 24.4 ->
  // 21.3 us at T = 1; at N = 4096 the 128-CTA grid loses, and T = 16 does not gain)
  if (p.T <= 8 && p.N >= 48 * num_sms) return launch_nt<1, 2, ASYM>(p, stream);
  if (p.T <= 8) return launch_nt<1, 1, ASYM>(p, stream);
  if (p.T <= 16) return launch_nt<2, 1, ASYM>(p, stream);
  if (p.T <= 32) return wide ? launch_nt<4, 2, ASYM>(p, stream) : launch_nt<4, 1, ASYM>(p, stream);
  return launch_nt<8, 2, ASYM>(p, stream);
}

}  // namespace

cudaError_t launch_w4a4_decode(const GemmLaunch& g) {
  if (g.x != nullptr || g.T > kDecodeMaxT) return cudaErrorNotSupported;
  const BlobHeader h = blob_header(g.N, g.K);
  const uint8_t* base = static_cast<const uint8_t*>(g.blob);
  static_assert(kTileRows % (2 * kRows) == 0, "a CTA's row groups must not straddle two weight boxes");
  DecodeParams p{};
  p.header = reinterpret_cast<const uint32_t*>(base);
  p.status = g.status_word;
  p.tiles = base + h.off_tiles;
  p.sw = reinterpret_cast<const float*>(base + h.off_sw);
  p.fb = reinterpret_cast<const float*>(base + h.off_fb);
  p.wsum = reinterpret_cast<const float*>(base + h.off_wsum);
  p.codes = g.codes;
  p.scales = g.scales;
  p.zeros = g.zeros;
  p.y = static_cast<uint16_t*>(g.y);
  p.ldy = g.ldy;
  p.acc_dump = g.acc_dump;
  p.T = g.T;
  p.N = g.N;
  p.K = g.K;
  p.num_kb = g.K / kTileK;
  const int sms = g.num_sms > 0 ? g.num_sms : 148;
  return g.zeros != nullptr ? launch_asym<true>(p, sms, g.stream) : launch_asym<false>(p, sms, g.stream);
}

}  // namespace baseq

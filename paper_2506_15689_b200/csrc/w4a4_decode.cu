// Decode-shaped W4A4 GEMM: the same contract as w4a4_gemm.cu (steps a7-a9 of
// DESIGN.md; int32-exact accumulation, fp64 epilogue, bf16 out) for T <= 64 tokens, where the
// work is streaming the packed weights once (N K / 2 bytes) and the 128 x 192 tcgen05 tile would
// be 1-50 % full.  HBM-bound: algorithmic bytes = N K / 2 (W) + T K / 2 (codes) + 2 T N (Y).
//
//   CTA            one group of 16 output channels (16 rows x 64 bytes = 1 KB contiguous per k-block
//                  of the weight blob), all of K, all T tokens; grid = ceil(N / 16)
//   8 warps        k-blocks w, w + 8, ... each; kDepth k-blocks of W (2 x LDG.128 per lane and
//                  k-block, streaming, issued BEFORE griddepcontrol.wait: the weights do not depend
//                  on the preceding quantiser) are in flight per warp
//   MMA            mma.sync.m16n8k32 s8 x s8 -> s32 with M = output channels, N = 8 tokens: at
//                  T <= 64 the contraction is 0.4-3 % of the tensor peak, the legacy warp-level MMA
//                  is ample and needs no shared-memory operand staging
//   expansion      a 32-bit word holds 8 nibbles; (w << 4) & 0xF0F0F0F0 and w & 0xF0F0F0F0 are the
//                  bytes 16 q of the even and odd nibbles (a signed nibble in the top half of a
//                  byte IS 16 q as int8).  Both operands are split the same way, so every k meets
//                  its partner (a permutation of k inside the dot product); raw = 256 acc exactly.
//                  Asymmetric codes (NEXT-1, unsigned) are re-centred to q - 8 by flipping the top
//                  bit, as in the tcgen05 kernel.
//   epilogue       partial sums of the 8 warps meet in shared memory; every output is evaluated
//                  with the fp64 expression of the contract itself (<= 1024 outputs per CTA).
#include "epilogue_math.cuh"
#include "kernels.cuh"
#include "ptx.cuh"

namespace baseq {
namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;
constexpr int kRows = 16;          // output channels per CTA (MMA M)
constexpr int kDepth = 4;          // k-blocks of W in flight per warp

struct DecodeParams {
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

// NT = token tiles of 8 (T <= 8 NT)
template <int NT, bool ASYM>
__global__ void __launch_bounds__(kThreads) w4a4_decode_kernel(const DecodeParams p) {
  __shared__ int32_t red[kWarps][NT * 4 * 32];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t4 = lane & 3;
  const int n0 = blockIdx.x * kRows;
  // weight rows g and g + 8 of this group, k-block 0 (boxes of kTileRows rows x 64 bytes)
  const uint8_t* wrow = p.tiles +
      (static_cast<size_t>(n0 / kTileRows) * p.num_kb * kTileRows + (n0 % kTileRows) + g) * 64 + t4 * 16;
  const uint8_t* xrow = p.codes + static_cast<size_t>(g) * (p.K / 2) + t4 * 16;

  int32_t acc[NT][4];
#pragma unroll
  for (int j = 0; j < NT; ++j)
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[j][c] = 0;

  bool waited = false;
  for (int kb0 = warp; kb0 < p.num_kb; kb0 += kWarps * kDepth) {
    uint4 wa[kDepth], wb[kDepth];
#pragma unroll
    for (int d = 0; d < kDepth; ++d) {
      const int kb = kb0 + d * kWarps;
      wa[d] = make_uint4(0, 0, 0, 0);
      wb[d] = make_uint4(0, 0, 0, 0);
      if (kb < p.num_kb) {
        const uint8_t* src = wrow + static_cast<size_t>(kb) * (kTileRows * 64);
        wa[d] = ptx::ldg_nc_stream(reinterpret_cast<const uint4*>(src));
        wb[d] = ptx::ldg_nc_stream(reinterpret_cast<const uint4*>(src + 8 * 64));
      }
    }
    if (!waited) {
      ptx::griddep_wait();      // codes and scales are the preceding kernel's output
      waited = true;
    }
#pragma unroll
    for (int d = 0; d < kDepth; ++d) {
      const int kb = kb0 + d * kWarps;
      if (kb < p.num_kb) {
        uint4 xa[NT];
#pragma unroll
        for (int j = 0; j < NT; ++j) {
          xa[j] = make_uint4(0, 0, 0, 0);
          if (j * 8 + g < p.T)
            xa[j] = ptx::ldg_nc(reinterpret_cast<const uint4*>(
                xrow + static_cast<size_t>(j) * 8 * (p.K / 2) + kb * 64));
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const uint32_t a = word(wa[d], i), b = word(wb[d], i);
          const uint32_t a0 = (a << 4) & 0xF0F0F0F0u, a2 = a & 0xF0F0F0F0u;
          const uint32_t a1 = (b << 4) & 0xF0F0F0F0u, a3 = b & 0xF0F0F0F0u;
#pragma unroll
          for (int j = 0; j < NT; ++j) {
            const uint32_t x = word(xa[j], i);
            uint32_t b0 = (x << 4) & 0xF0F0F0F0u, b1 = x & 0xF0F0F0F0u;
            if (ASYM) {
              b0 ^= 0x80808080u;        // 16 q -> 16 (q - 8) as int8
              b1 ^= 0x80808080u;
            }
            mma_s8(acc[j], a0, a1, a2, a3, b0, b1);
          }
        }
      }
    }
  }
  if (!waited) ptx::griddep_wait();

#pragma unroll
  for (int j = 0; j < NT; ++j)
#pragma unroll
    for (int c = 0; c < 4; ++c) red[warp][(j * 4 + c) * 32 + lane] = acc[j][c];
  __syncthreads();

  // thread o -> (token, channel): 16 consecutive lanes write 32 contiguous bytes of one Y row
  for (int o = threadIdx.x; o < NT * 8 * kRows; o += kThreads) {
    const int tok = o >> 4, ch = o & 15;
    const int n = n0 + ch;
    if (tok >= p.T || n >= p.N) continue;
    // accumulator fragment: c0, c1 = row g, tokens 2 t4 + {0, 1}; c2, c3 = row g + 8
    const int j = tok >> 3, col = tok & 7;
    const int idx = (j * 4 + (ch >> 3) * 2 + (col & 1)) * 32 + (ch & 7) * 4 + (col >> 1);
    int32_t raw = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) raw += red[w][idx];
    int32_t a = raw >> 8;                                  // raw = 256 acc exactly
    const float st = p.scales[tok], sw = p.sw[n], fb = p.fb[n];
    uint32_t out;
    if (ASYM) {
      const float ws = p.wsum[n];
      out = epi::dequant_f64_asym(a, st, p.zeros[tok], sw, fb, ws);
      a += 8 * static_cast<int32_t>(ws);                   // the accumulator over the unsigned codes
    } else {
      out = epi::dequant_f64(a, st, sw, fb);
    }
    p.y[static_cast<size_t>(tok) * p.ldy + n] = static_cast<uint16_t>(out);
    if (p.acc_dump != nullptr) p.acc_dump[static_cast<size_t>(tok) * p.N + n] = a;
  }
}

template <int NT, bool ASYM>
cudaError_t launch_nt(const DecodeParams& p, cudaStream_t stream) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>((p.N + kRows - 1) / kRows), 1, 1);
  cfg.blockDim = dim3(kThreads, 1, 1);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, w4a4_decode_kernel<NT, ASYM>, p);
}

template <bool ASYM>
cudaError_t launch_asym(const DecodeParams& p, cudaStream_t stream) {
  if (p.T <= 8) return launch_nt<1, ASYM>(p, stream);
  if (p.T <= 16) return launch_nt<2, ASYM>(p, stream);
  if (p.T <= 32) return launch_nt<4, ASYM>(p, stream);
  return launch_nt<8, ASYM>(p, stream);
}

}  // namespace

cudaError_t launch_w4a4_decode(const GemmLaunch& g) {
  if (g.x != nullptr || g.T > kDecodeMaxT) return cudaErrorNotSupported;
  const BlobHeader h = blob_header(g.N, g.K);
  const uint8_t* base = static_cast<const uint8_t*>(g.blob);
  static_assert(kTileRows % kRows == 0, "a 16-row group must not straddle two weight boxes");
  DecodeParams p{};
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
  return g.zeros != nullptr ? launch_asym<true>(p, g.stream) : launch_asym<false>(p, g.stream);
}

}  // namespace baseq

// W4A4 GEMM + fused de-quantisation epilogue (steps a7-a10 of DESIGN.md; K1 + K3 of SURVEY;
// PAPER.md:307).  sm_100a has no int4 MMA kind, so int4 nibbles are expanded on-chip to int8
// and multiplied with tcgen05.mma kind::i8 (exact int32 accumulation in TMEM).
//
// Persistent, warp-specialised, one CTA per SM, 128x256 output tile, K-block = 128:
//   warp 0      producer  : TMA (2-D tensor map for A codes, 1-D bulk copies for the packed
//                           weight boxes) into a ring of PACKED stages
//   warps 8-15  unpackers : packed int4 -> int8 (x16 trick, below) into a ring of UNPACKED
//                           stages in the SWIZZLE_128B K-major layout the MMA reads
//   warp 1      MMA       : one elected thread issues 4 x tcgen05.mma (K = 32 each) per K-block
//                           into one of two 256-column TMEM accumulators
//   warps 4-7   epilogue  : tcgen05.ld -> dequant (+ fused bias) -> bf16 -> global; overlaps the
//                           next tile's main loop through the second TMEM accumulator
//
// x16 unpack: for a 32-bit word w holding 8 two's-complement nibbles,
//   lo = (w << 4) & 0xF0F0F0F0   -> 4 signed bytes = 16 * (even-k codes)
//   hi =  w       & 0xF0F0F0F0   -> 4 signed bytes = 16 * (odd-k codes)
// Both operands use the same even/odd permutation of K inside each 32-element group, so the
// dot products are unchanged and the raw accumulator is exactly 256 * acc
// (|256 * acc| <= 256 * 64 * K < 2^31 for K <= 131072); acc = raw >> 8 is exact.
#include <cuda.h>

#include "kernels.cuh"
#include "ptx.cuh"

namespace baseq {
namespace {

constexpr int BM = 128;                 // tokens per tile (UMMA M)
constexpr int BN = 256;                 // output channels per tile (UMMA N)
constexpr int BK = 128;                 // int4 elements along K per stage
constexpr int kPackedA = BM * BK / 2;   // 8 KB
constexpr int kPackedB = BN * BK / 2;   // 16 KB
constexpr int kPackedStage = kPackedA + kPackedB;
constexpr int kUnpackedA = BM * BK;     // 16 KB (int8)
constexpr int kUnpackedB = BN * BK;     // 32 KB
constexpr int kUnpackedStage = kUnpackedA + kUnpackedB;
constexpr int kPStages = 3;
constexpr int kUStages = 3;
constexpr int kAccStages = 2;
constexpr int kTmemCols = 512;

constexpr int kNumThreads = 512;
constexpr int kProducerWarp = 0;
constexpr int kMmaWarp = 1;
constexpr int kEpiWarp0 = 4;            // warps 4..7  (warp % 4 = TMEM lane quarter)
constexpr int kUnpackWarp0 = 8;         // warps 8..15
constexpr int kNumUnpackWarps = 8;

struct __align__(8) Barriers {
  uint64_t pfull[kPStages], pempty[kPStages];
  uint64_t ufull[kUStages], uempty[kUStages];
  uint64_t tfull[kAccStages], tempty[kAccStages];
  uint32_t tmem_base;
};

constexpr int kSmemBytes = 1024 /*align slack*/ + kUStages * kUnpackedStage +
                           kPStages * kPackedStage + 256 /*barriers*/;
static_assert(sizeof(Barriers) <= 256, "barrier block too large");
static_assert(kSmemBytes <= 232448, "exceeds 227 KB of dynamic shared memory");

struct GemmParams {
  const uint8_t* tiles;     // blob tiles
  const float* sw;          // [Npad]
  const float* fb;          // [Npad]
  const float* scales;      // [T]
  uint16_t* y;              // bf16 [T, ldy]
  int64_t ldy;
  int32_t* acc_dump;        // optional [T, N]
  int T, N, K;
  int num_m, num_n, num_kb;
};

__device__ __forceinline__ void advance(int& stage, uint32_t& phase, int n) {
  if (++stage == n) {
    stage = 0;
    phase ^= 1u;
  }
}

// ------------------------------------------------------------------------------ epilogue math
// Contract (C-9): Y = bf16_rne( fma((double)s_t * (double)s_w, (double)acc, (double)fb) ).
// Fast path in fp32 with a proven error bracket; any element whose bracket straddles a bf16
// rounding boundary (about 1e-4 of them) is recomputed with the fp64 expression itself, so the
// result is bit-identical to the fp64 definition for every element.
//
//   t   = RN(s_t * acc)            rel. error <= 2^-24
//   y   = RN(t * s_w + fb)         one more rounding
//   |y - y*| <= 2^-24 (|t s_w| + |y|) (1 + eps)  <  E := 2^-23 (|RN(t s_w)| + |y|)
// If bf16(y - E) == bf16(y + E) every real number in the bracket -- including the fp64 value --
// rounds to that bf16.
__device__ __forceinline__ uint32_t bf16_from_double_rne(double v) {
  // round-to-odd to fp32 (keeps a sticky bit), then RNE to bf16: a single rounding overall
  float f = __double2float_rz(v);
  uint32_t u = __float_as_uint(f);
  if (static_cast<double>(f) != v) u |= 1u;
  const uint32_t r = u + 0x7FFFu + ((u >> 16) & 1u);
  return r >> 16;
}

__device__ __forceinline__ uint32_t dequant_bf16(int32_t acc, float st, float sw, float fb) {
  const float accf = __int2float_rn(acc);                 // exact: |acc| < 2^24
  const float t = __fmul_rn(st, accf);
  const float p = __fmul_rn(t, sw);
  const float y = __fmaf_rn(t, sw, fb);
  const float e = __fmul_rn(__fadd_rn(fabsf(p), fabsf(y)), 1.1920928955078125e-07f);   // 2^-23
  const float lo = __fsub_rn(y, e);
  const float hi = __fadd_rn(y, e);
  uint32_t pk;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pk) : "f"(hi), "f"(lo));   // hi -> upper half
  const uint32_t a = pk & 0xFFFFu, b = pk >> 16;
  if (a == b && fabsf(y) > 1e-30f) return a;
  const double pd = __dmul_rn(static_cast<double>(st), static_cast<double>(sw));
  const double yd = __fma_rn(pd, static_cast<double>(acc), static_cast<double>(fb));
  return bf16_from_double_rne(yd);
}

// ------------------------------------------------------------------------------ the kernel
__global__ void __launch_bounds__(kNumThreads, 1)
w4a4_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const GemmParams p) {
  extern __shared__ uint8_t smem_raw[];
  // SWIZZLE_128B operands need 1024-byte alignment
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
  const uint32_t unpacked0 = smem_base;                                   // kUStages x 48 KB
  const uint32_t packed0 = smem_base + kUStages * kUnpackedStage;         // kPStages x 24 KB
  uint8_t* packed_ptr = smem + kUStages * kUnpackedStage;
  uint8_t* unpacked_ptr = smem;
  Barriers* bars = reinterpret_cast<Barriers*>(smem + kUStages * kUnpackedStage +
                                               kPStages * kPackedStage);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (warp == kProducerWarp && lane == 0) {
    ptx::prefetch_tensormap(&tmap_a);
    for (int i = 0; i < kPStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->pfull[i]), 1);
      ptx::mbar_init(ptx::smem_u32(&bars->pempty[i]), kNumUnpackWarps);
    }
    for (int i = 0; i < kUStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->ufull[i]), kNumUnpackWarps);
      ptx::mbar_init(ptx::smem_u32(&bars->uempty[i]), 1);
    }
    for (int i = 0; i < kAccStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->tfull[i]), 1);
      ptx::mbar_init(ptx::smem_u32(&bars->tempty[i]), 4);
    }
    ptx::fence_barrier_init();
  }
  if (warp == kMmaWarp) {
    ptx::tmem_alloc<kTmemCols>(ptx::smem_u32(&bars->tmem_base));
  }
  ptx::tcgen05_fence_before();
  __syncthreads();
  ptx::tcgen05_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&bars->tmem_base);

  const int num_tiles = p.num_m * p.num_n;

  if (warp == kProducerWarp) {
    // ===================================================================== TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        const int m_blk = tile % p.num_m, n_blk = tile / p.num_m;
        const uint8_t* b0 = p.tiles + static_cast<size_t>(2 * n_blk) * p.num_kb * kTileBytes;
        const uint8_t* b1 = b0 + static_cast<size_t>(p.num_kb) * kTileBytes;
        for (int kb = 0; kb < p.num_kb; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&bars->pempty[stage]), phase ^ 1u);
          const uint32_t full = ptx::smem_u32(&bars->pfull[stage]);
          const uint32_t dst = packed0 + stage * kPackedStage;
          ptx::mbar_arrive_expect_tx(full, kPackedStage);
          ptx::tma_load_2d(dst, &tmap_a, kb * (BK / 2), m_blk * BM, full);
          ptx::bulk_load_1d(dst + kPackedA, b0 + static_cast<size_t>(kb) * kTileBytes,
                            kTileBytes, full);
          ptx::bulk_load_1d(dst + kPackedA + kTileBytes, b1 + static_cast<size_t>(kb) * kTileBytes,
                            kTileBytes, full);
          advance(stage, phase, kPStages);
        }
      }
    }
  } else if (warp == kMmaWarp) {
    // ===================================================================== MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_i8(BM, BN);
      int stage = 0, as = 0;
      uint32_t phase = 0, aphase = 0;
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        ptx::mbar_wait(ptx::smem_u32(&bars->tempty[as]), aphase ^ 1u);
        ptx::tcgen05_fence_after();
        const uint32_t tmem_d = tmem_base + as * BN;
        for (int kb = 0; kb < p.num_kb; ++kb) {
          ptx::mbar_wait(ptx::smem_u32(&bars->ufull[stage]), phase);
          ptx::tcgen05_fence_after();
          const uint32_t a_addr = unpacked0 + stage * kUnpackedStage;
          const uint32_t b_addr = a_addr + kUnpackedA;
#pragma unroll
          for (int k = 0; k < BK / 32; ++k) {
            const uint64_t da = ptx::make_smem_desc_sw128(a_addr + k * 32);
            const uint64_t db = ptx::make_smem_desc_sw128(b_addr + k * 32);
            ptx::mma_i8_ss(tmem_d, da, db, idesc, (kb | k) != 0 ? 1u : 0u);
          }
          ptx::tcgen05_commit(ptx::smem_u32(&bars->uempty[stage]));    // frees the smem stage
          advance(stage, phase, kUStages);
        }
        ptx::tcgen05_commit(ptx::smem_u32(&bars->tfull[as]));          // accumulator ready
        advance(as, aphase, kAccStages);
      }
    }
  } else if (warp >= kUnpackWarp0) {
    // ===================================================================== int4 -> int8 unpack
    const int uw = warp - kUnpackWarp0;                 // 0..7
    int ps = 0, us = 0;
    uint32_t pphase = 0, uphase = 0;
    const int rsub = lane >> 2, c = lane & 3;           // row in 8-row group, 16-byte chunk
    for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
      for (int kb = 0; kb < p.num_kb; ++kb) {
        ptx::mbar_wait(ptx::smem_u32(&bars->pfull[ps]), pphase);
        ptx::mbar_wait(ptx::smem_u32(&bars->uempty[us]), uphase ^ 1u);
        const uint8_t* src = packed_ptr + ps * kPackedStage;
        uint8_t* dst = unpacked_ptr + us * kUnpackedStage;
        // 384 rows (A 128 + B 256) = 48 groups of 8 rows; warp uw takes groups uw, uw+8, ...
        uint4 v[6];
#pragma unroll
        for (int i = 0; i < 6; ++i) {
          const int rg = uw + i * kNumUnpackWarps;
          v[i] = *reinterpret_cast<const uint4*>(src + rg * 512 + lane * 16);
        }
#pragma unroll
        for (int i = 0; i < 6; ++i) {
          const int rg = uw + i * kNumUnpackWarps;
          uint4 lo, hi;
          lo.x = (v[i].x << 4) & 0xF0F0F0F0u; hi.x = v[i].x & 0xF0F0F0F0u;
          lo.y = (v[i].y << 4) & 0xF0F0F0F0u; hi.y = v[i].y & 0xF0F0F0F0u;
          lo.z = (v[i].z << 4) & 0xF0F0F0F0u; hi.z = v[i].z & 0xF0F0F0F0u;
          lo.w = (v[i].w << 4) & 0xF0F0F0F0u; hi.w = v[i].w & 0xF0F0F0F0u;
          uint8_t* row = dst + rg * 1024 + rsub * 128;
          *reinterpret_cast<uint4*>(row + (((2 * c) ^ rsub) << 4)) = lo;
          *reinterpret_cast<uint4*>(row + (((2 * c + 1) ^ rsub) << 4)) = hi;
        }
        ptx::fence_proxy_async_smem();      // generic-proxy writes -> visible to tcgen05.mma
        __syncwarp();
        if (lane == 0) {
          ptx::mbar_arrive(ptx::smem_u32(&bars->ufull[us]));
          ptx::mbar_arrive(ptx::smem_u32(&bars->pempty[ps]));
        }
        advance(ps, pphase, kPStages);
        advance(us, uphase, kUStages);
      }
    }
  } else if (warp >= kEpiWarp0 && warp < kEpiWarp0 + 4) {
    // ===================================================================== epilogue
    const int q = warp & 3;                             // TMEM lane quarter
    int as = 0;
    uint32_t aphase = 0;
    for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
      const int m_blk = tile % p.num_m, n_blk = tile / p.num_m;
      const int row = m_blk * BM + q * 32 + lane;
      const bool row_ok = row < p.T;
      const float st = row_ok ? p.scales[row] : 0.0f;
      ptx::mbar_wait(ptx::smem_u32(&bars->tfull[as]), aphase);
      ptx::tcgen05_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + as * BN;
      const int n0 = n_blk * BN;
#pragma unroll 1
      for (int c0 = 0; c0 < BN; c0 += 32) {
        if (n0 + c0 >= p.N) break;                      // warp-uniform
        uint32_t r[32];
        ptx::tmem_ld_32x32b_x32(taddr + c0, r);
        ptx::tmem_ld_wait();
        uint32_t out[16];
#pragma unroll
        for (int j = 0; j < 32; j += 2) {
          const int n = n0 + c0 + j;
          const int32_t a0 = static_cast<int32_t>(r[j]) >> 8;       // raw = 256 * acc
          const int32_t a1 = static_cast<int32_t>(r[j + 1]) >> 8;
          r[j] = static_cast<uint32_t>(a0);
          r[j + 1] = static_cast<uint32_t>(a1);
          const float2 sw = __ldg(reinterpret_cast<const float2*>(p.sw + n));
          const float2 fb = __ldg(reinterpret_cast<const float2*>(p.fb + n));
          const uint32_t y0 = dequant_bf16(a0, st, sw.x, fb.x);
          const uint32_t y1 = dequant_bf16(a1, st, sw.y, fb.y);
          out[j >> 1] = y0 | (y1 << 16);
        }
        if (row_ok) {
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            const int n = n0 + c0 + g * 8;
            if (n < p.N) {
              *reinterpret_cast<uint4*>(p.y + static_cast<int64_t>(row) * p.ldy + n) =
                  make_uint4(out[4 * g], out[4 * g + 1], out[4 * g + 2], out[4 * g + 3]);
              if (p.acc_dump != nullptr) {
                int32_t* d = p.acc_dump + static_cast<int64_t>(row) * p.N + n;
                *reinterpret_cast<uint4*>(d) = make_uint4(r[8 * g], r[8 * g + 1], r[8 * g + 2], r[8 * g + 3]);
                *reinterpret_cast<uint4*>(d + 4) =
                    make_uint4(r[8 * g + 4], r[8 * g + 5], r[8 * g + 6], r[8 * g + 7]);
              }
            }
          }
        }
      }
      // all TMEM reads of this warp are complete (wait::ld above): release the accumulator
      ptx::tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&bars->tempty[as]));
      advance(as, aphase, kAccStages);
    }
  }

  // ---- teardown
  ptx::tcgen05_fence_before();
  __syncthreads();
  if (warp == kMmaWarp) {
    ptx::tcgen05_fence_after();
    ptx::tmem_dealloc<kTmemCols>(tmem_base);
  }
}

// ------------------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  // resolved through the runtime so that libbaseq.so has no link-time dependency on libcuda
  static EncodeTiledFn fn = nullptr;
  if (fn == nullptr) {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) ==
            cudaSuccess && qres == cudaDriverEntryPointSuccess) {
      fn = reinterpret_cast<EncodeTiledFn>(sym);
    }
  }
  return fn;
}

}  // namespace

cudaError_t launch_w4a4_gemm(const GemmLaunch& g) {
  if (g.x != nullptr) return cudaErrorNotSupported;     // fused producer: separate kernel (TODO)
  EncodeTiledFn encode = get_encode_fn();
  if (encode == nullptr) return cudaErrorNotSupported;

  const BlobHeader h = blob_header(g.N, g.K);
  const uint8_t* base = static_cast<const uint8_t*>(g.blob);

  // A operand: codes [T, K/2] bytes; box = 64 bytes (128 int4) x 128 rows; rows beyond T are
  // zero-filled by TMA, so a ragged last M tile needs no special case in the main loop.
  CUtensorMap tmap;
  const cuuint64_t dims[2] = {static_cast<cuuint64_t>(g.K / 2), static_cast<cuuint64_t>(g.T)};
  const cuuint64_t strides[1] = {static_cast<cuuint64_t>(g.K / 2)};
  const cuuint32_t box[2] = {static_cast<cuuint32_t>(BK / 2), static_cast<cuuint32_t>(BM)};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = encode(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2,
                            const_cast<uint8_t*>(g.codes), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;

  GemmParams p;
  p.tiles = base + h.off_tiles;
  p.sw = reinterpret_cast<const float*>(base + h.off_sw);
  p.fb = reinterpret_cast<const float*>(base + h.off_fb);
  p.scales = g.scales;
  p.y = static_cast<uint16_t*>(g.y);
  p.ldy = g.ldy;
  p.acc_dump = g.acc_dump;
  p.T = g.T;
  p.N = g.N;
  p.K = g.K;
  p.num_m = (g.T + BM - 1) / BM;
  p.num_n = h.Npad / BN;
  p.num_kb = g.K / BK;

  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(w4a4_gemm_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int tiles = p.num_m * p.num_n;
  const int grid = tiles < g.num_sms ? tiles : g.num_sms;
  w4a4_gemm_kernel<<<grid, kNumThreads, kSmemBytes, g.stream>>>(tmap, p);
  return cudaGetLastError();
}

}  // namespace baseq

// W4A4 GEMM + fused de-quantisation epilogue (steps a7-a10 of DESIGN.md; K1 + K3 of SURVEY;
// PAPER.md:307).  sm_100a has no int4 MMA kind, so int4 nibbles are expanded on-chip to int8
// and multiplied with tcgen05.mma kind::i8 (exact int32 accumulation in TMEM).
//
// The r1a kernel staged both operands packed -> smem -> unpack -> smem -> MMA and ran exactly at
// the shared-memory bandwidth limit (144 KB of smem traffic per 128x256x128 k-block against a
// 64 KB budget at the int8 MMA rate; profiles/r1a.md).  This version removes most of it:
//   * the expanded activation operand A never touches shared memory: the packed codes arrive by
//     TMA (SWIZZLE_64B), A warps (thread = token row) read them with conflict-free 16-byte LDS,
//     expand them and write int8 to TENSOR MEMORY with tcgen05.st; the MMA takes A from TMEM
//     (.ts form);
//   * a CTA PAIR (cta_group::2, M = 256) shares the weight operand: each CTA stages and
//     expands only half of the tile's N rows.
// Per CTA and k-block the shared-memory traffic is  BN/2 x (64 B TMA write + 64 B unpack read +
// 128 B unpack write + 128 B MMA read) = 36 KB at BN = 192, plus 16 KB for A's packed codes,
// against 48 KB of budget.
//
// Persistent, warp-specialised, one CTA per SM, 896 threads; the single-lane roles
// sit at the highest warp ids (the scheduler of a sub-partition favours the higher id):
//   warps 0-7     epilogue: tcgen05.ld -> dequant (+ fused bias) -> bf16 -> staging tile -> TMA
//                 store; overlaps the next tile's main loop through the second accumulator
//   warps 8-15    A: LDS -> x16 expand -> tcgen05.st (two sets alternate k-blocks)
//   warps 16-23   B: packed int4 -> int8 into SWIZZLE_128B K-major stages (two sets)
//   warps 24, 25  TMA producers: A codes (2-D tensor map) / this CTA's weight box (bulk copy),
//                 8-deep packed ring
//   warp 27       MMA issuer (leader CTA of the pair only): 4 x tcgen05.mma.kind::i8 (K = 32) per
//                 k-block into one of two BN-column TMEM accumulators; commits multicast to both CTAs
// Fused variant (a10, 1024 threads): warps 0-3 are the background quantiser -- one token row per
// warp (quant_math.cuh), codes into an L2-resident workspace, per-128-row ready counters -- and
// every role above moves up by four.
//
// x16 unpack: for a 32-bit word w holding 8 two's-complement nibbles,
//   lo = (w << 4) & 0xF0F0F0F0   -> 4 signed bytes = 16 * (even-k codes)
//   hi =  w       & 0xF0F0F0F0   -> 4 signed bytes = 16 * (odd-k codes)
// Both operands use the same even/odd permutation of K inside each 32-element group, so the
// dot products are unchanged and the raw accumulator is exactly 256 * acc
// (|256 * acc| <= 256 * 64 * K < 2^31 for K <= 131072); acc = raw >> 8 is exact.
#include <cuda.h>

#include <mutex>

#include "epilogue_math.cuh"
#include "kernels.cuh"
#include "ptx.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr int BM = 128;                 // token rows per CTA (TMEM lanes)
constexpr int BN = kGemmBN;             // output channels per tile (UMMA N)
constexpr int BK = 128;                 // int4 elements along K per stage
constexpr int kStages = 4;              // operand stages: A in TMEM (32 columns), B unpacked in smem
constexpr int kPStagesMax = 8;          // packed ring depth (TMA latency from L2 is ~1.5k clk)
constexpr int kAccStages = 2;
constexpr int kACol0 = kAccStages * BN; // first TMEM column of the A stages
constexpr int kTmemCols = 512;
constexpr int kPackedA = BM * BK / 2;    // 8 KB of packed codes per CTA and k-block
static_assert(kACol0 + kStages * (BK / 4) <= kTmemCols, "TMEM budget");
static_assert(BN % 32 == 0 && BN <= 256, "UMMA N");

constexpr int kSets = 2;                // A and B warp sets alternate k-blocks: one warp's serial
                                        // chain per k-block (two try_waits, LDS, expand, store,
                                        // fence, arrive: 400-700 clk) exceeds the 384 clk MMA time
constexpr int kNumUnpackWarps = 4;      // per set

// A tile belongs to a CTA pair (cta_group::2, M = 256).  FUSED = the single-launch variant (a10):
// four more warps quantise bf16 X in the background -- one token row per warp, the same
// quant_math.cuh contract as the stand-alone quantiser -- into a workspace the size of the codes
// that lives in L2, raise a counter per 128-row group, and the A producer of a tile waits for its
// group's counter before it issues the tile's first TMA load.  Tiles are walked M-major there, so
// that the first wave needs the first one or two 256-row strips only.
constexpr int CG = 2;                   // CTAs per tile
constexpr int kQuantWarps = 4;          // fused variant: background quantiser warps per CTA
template <bool FUSED>
struct Cfg {
  // per-tile column operands of the epilogue (s_w, fb, wsum), one copy per accumulator stage
  static constexpr int kColParamBytes = kAccStages * 3 * BN * 4;
  // [barriers 256 | column operands | pad] then the Y staging tiles of the TMA-store epilogue: per
  // epilogue warp 32 rows x BN/2 columns of bf16 as 3 boxes of 32 rows x 64 bytes
  static constexpr int kTailBytes = (256 + kColParamBytes + 1023) / 1024 * 1024;
  static constexpr int kStoreWarpBytes = 32 * (BN / 2) * 2;
  static constexpr int kEpiWarps = 8;                       // x 32 rows; 2 column halves
  static constexpr int kStoreBytes = kEpiWarps * kStoreWarpBytes;
  // fused: the quantiser warps take the LOWEST warp ids (the scheduler of a sub-partition favours
  // the higher id among eligible warps: background work must never beat a GEMM role to an issue slot)
  static constexpr int kQuantWarp0 = 0;
  static constexpr int kEpiWarp0 = FUSED ? kQuantWarps : 0;   // epilogue: warp % 4 = TMEM lane quarter
  static constexpr int kAWarp0 = kEpiWarp0 + kEpiWarps;     // 8 A warps
  static constexpr int kUnpackWarp0 = kAWarp0 + 8;
  // the single-lane roles sit ABOVE the data warps: the warp scheduler of a sub-partition favours the
  // higher warp id among eligible warps, and a late TMA issue or MMA issue stalls everybody else
  static constexpr int kRoleWarp0 = kUnpackWarp0 + kNumUnpackWarps * kSets;
  static constexpr int kProducerWarp = kRoleWarp0;        // A operand (tensor-map TMA)
  static constexpr int kProducerWarpB = kRoleWarp0 + 1;   // B operand (bulk TMA)
  static constexpr int kMmaWarp = kRoleWarp0 + 3;
  static constexpr int kThreads = 32 * (kRoleWarp0 + 4);      // 896, fused 1024
  static constexpr int kBRows = BN / CG;                   // weight rows staged per CTA
  static constexpr int kPackedB = kBRows * BK / 2;
  static constexpr int kPackedStage = kPackedA + kPackedB;   // multiple of 1024
  static constexpr int kUnpackedStage = kBRows * BK;
  static constexpr int kPFullCount = 2;
  static constexpr int kPEmptyCount = kNumUnpackWarps + 4;
  static constexpr int kFullCount = CG * (4 + kNumUnpackWarps);
  static constexpr int kTemptyCount = CG * kEpiWarps;
  static constexpr int kPStages = kPStagesMax;
  static constexpr int kSmemBytes =
      1024 + kStages * kUnpackedStage + kPStages * kPackedStage + kTailBytes + kStoreBytes;
  static_assert(kSmemBytes <= 232448, "exceeds 227 KB of dynamic shared memory");
};

struct __align__(8) Barriers {
  uint64_t pfull[kPStagesMax], pempty[kPStagesMax];   // packed-B ring, CTA-local
  uint64_t full[kStages];                       // operand stage ready   (waited on in the leader CTA)
  uint64_t empty[kStages];                      // operand stage free    (every CTA; MMA commit)
  uint64_t tfull[kAccStages];                   // accumulator ready     (every CTA; MMA commit)
  uint64_t tempty[kAccStages];                  // accumulator drained   (waited on in the leader CTA)
  uint32_t tmem_base;
};
static_assert(sizeof(Barriers) <= 256, "barrier block too large");

struct GemmParams {
  const uint32_t* header;   // blob header: magic, N, K, Npad, ... (checked against N, K below)
  unsigned int* status;     // device status word: kStatusBadBlob is raised on a mismatch
  const uint8_t* tiles;     // blob boxes
  const float* sw;          // [Npad]
  const float* fb;          // [Npad]
  const float* scales;      // [T]
  const float* zeros;       // [T] lattice lower bounds z_t (asymmetric variant)
  const float* wsum;        // [Npad] sum_k qw[n,k] as fp32 (asymmetric variant)
  uint16_t* y;              // bf16 [T, ldy]
  int64_t ldy;
  int32_t* acc_dump;        // optional [T, N]
  int T, N, K;
  int num_m, num_n, num_kb;
  // fused variant only
  const uint4* x;           // bf16 [T, ldx] viewed as 16-byte vectors
  int64_t ldxv;             // ldx / 8
  float alpha, gamma;
  const float* sa;
  const float* bvec;
  int had_block;
  float had_scale;
  uint32_t* codes_out;      // [T, K/8] words of 8 nibbles: the workspace (or the caller's codes_dump)
  float* scales_out;        // [T] (= scales)
  float* zeros_out;         // [T] (= zeros; asymmetric fused variant)
  unsigned int* ready;      // [ceil(T / 128)] rows quantised per 128-row group
  unsigned long long* ctrl; // workspace control block: [0] = kFusedReady once the counters are zero,
                            // [1] (low word) = CTAs that have finished, [2] = next row to quantise
  int ngroups;
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
// If bf16(y - E) == bf16(y + E) for a proven bound E >= |y - y*| every real number in the bracket
// -- including the fp64 value -- rounds to that bf16 (all but ~2.4e-4 of the elements); otherwise
// the fp64 expression itself is evaluated.  The bound is derived at dequant_bracket below.
__device__ __noinline__ uint32_t dequant_f64(int32_t acc, float st, float sw, float fb) {
  return epi::dequant_f64(acc, st, sw, fb);
}
// `raw` is the TMEM accumulator 256 * acc (|acc| < 2^22, so raw has at most 22 significant bits
// and converts to fp32 exactly) and st256 = s_t * 2^-8 (exact): st256 * float(raw) is the same
// real number as s_t * acc and rounds to the same t.
// Branch-free fast path: returns the bracket ends  hi, lo = y +- 2^-23 (2 |y| + |fb| + 2^-100)
// (the 2^-100 keeps the bracket wider than the absolute rounding errors when y is denormal; the
// caller passes fbt = |fb| + 2^-100, formed once per column when the tile's operands are staged).
// With P = s_t s_w acc:  y = (P (1 + d1) + fb)(1 + d2), |d| <= 2^-24, so
//   |y - y*| <= 2^-24 (|P| + |y|)(1 + 2^-23)  and  |P| = |y* - fb| <= |y| + |y - y*| + |fb|,
// i.e. |y - y*| < 2^-24 (2 |y| + |fb|)(1 + 2^-22): E is twice that, which also covers the rounding of
// hi / lo themselves (half an ulp of y).  Five fma-pipe instructions per output (t, y, s, hi, lo)
// instead of seven: the epilogue's FMUL / FFMA / FADD are what a tile costs the main loop
// (r1i capture: ~2400 clk per tile, the fma pipe issues one warp instruction per two clocks).
// The element is settled iff both ends round to the same bf16.
__device__ __forceinline__ void dequant_bracket(int32_t raw, float st256, float sw, float fb, float fbt,
                                                float& lo, float& hi) {
  const float t = __fmul_rn(st256, __int2float_rn(raw));
  const float y = __fmaf_rn(t, sw, fb);
  const float s = __fmaf_rn(2.0f, fabsf(y), fbt);
  hi = __fmaf_rn(s, 1.1920928955078125e-07f, y);
  lo = __fmaf_rn(s, -1.1920928955078125e-07f, y);
}
// bf16(a1) << 16 | bf16(a0), both RNE: two bracket ends of neighbouring columns -> one output word
__device__ __forceinline__ uint32_t pack_bf16x2(float a1, float a0) {
  uint32_t pk;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pk) : "f"(a1), "f"(a0));
  return pk;
}
// Asymmetric variant (NEXT-1): the oracle's value is yd = fma(s_t s_w, acc, fma(z_t s_w, wsum, fb))
// in fp64 with acc = sum_k q w over the UNSIGNED codes.  Evaluated like that in fp32 the two
// products are ~80x larger than y and nearly cancel (q = q' + 8 puts 8 s_t wsum into the first and
// z_t ~ -8 s_t into the second), so the bracket almost never settled (measured).  The MMA therefore
// accumulates acc' = sum_k (q - 8) w = acc - 8 wsum, and the fast path evaluates the algebraically
// identical  y* = (s_t s_w) acc' + (mid_t s_w) wsum + fb,  mid_t = z_t + 8 s_t  (the centre of the
// row's range; no structural cancellation):
//   t = RN(s_t acc'), p = RN(t s_w), midf = RN(8 s_t + z_t), mw = RN(midf wsum), m = RN(mw s_w),
//   c = RN(mw s_w + fb), y = RN(t s_w + c)
//   |y - y*| <= 2^-24 (|p| + |y| + |c| + 2 |m|) (1 + 2^-22)      [one term per rounding above]
// and |yd - y*| is ~2^-52 of the same magnitudes, so E = 2^-23 (|p| + |y| + |c| + 2 |m| + 2^-100)
// is a bracket for yd; unsettled elements take the fp64 expression itself, with acc rebuilt
// exactly as acc' + 8 wsum.
__device__ __noinline__ uint32_t dequant_f64_asym(int32_t acc_c, float st, float zt, float sw,
                                                  float fb, float ws) {
  return epi::dequant_f64_asym(acc_c, st, zt, sw, fb, ws);
}
__device__ __forceinline__ void dequant_bracket_asym(int32_t raw, float st256, float midf, float sw,
                                                     float fb, float ws, float& lo, float& hi) {
  const float t = __fmul_rn(st256, __int2float_rn(raw));
  const float p = __fmul_rn(t, sw);
  const float mw = __fmul_rn(midf, ws);
  const float m = __fmul_rn(mw, sw);
  const float c = __fmaf_rn(mw, sw, fb);
  const float y = __fmaf_rn(t, sw, c);
  float s = __fadd_rn(__fadd_rn(fabsf(p), 7.888609052210118e-31f), fabsf(y));
  s = __fmaf_rn(fabsf(m), 2.0f, __fadd_rn(s, fabsf(c)));
  hi = __fmaf_rn(s, 1.1920928955078125e-07f, y);
  lo = __fmaf_rn(s, -1.1920928955078125e-07f, y);
}

// ------------------------------------------------------------------------------ background quantiser
// One pass (PASS 0: absmax; PASS 1: round, clamp, pack, store) of a quantiser warp over kQC vector
// steps of its row, lane l owning vectors l, l + 32, ....  ONE BASIC BLOCK by construction -- no
// branch, idle lanes and steps beyond the row are clamped to the row's last vector and masked where
// the values are used -- because ptxas tracks loads that cross a branch with a single scoreboard, and
// then the wait for ring slot d also waits for the refill issued one step earlier (measured: one
// memory round trip per step).  In straight-line code the kQD-deep register ring {x vector, its 8 b
// values} is a true software pipeline.  HAD: 0 = no rotation, 128 = block-128 Hadamard (compile
// time: qm::hadamard8 unrolls to 32 shuffles); everything else takes the generic step below.
constexpr int kQD = 4;     // ring slots = loads in flight per lane: x + 2 x b per slot
constexpr int kQC = 8;     // vector steps per chunk (16 without the Hadamard measured 4 % slower for
                           // the whole launch on K = 4096: twice the code in the instruction cache)
// GBF16 (HAD == 0 only): the scalar s^a is a bf16 value, so Q0 + Q2 are ONE mixed-precision fma per
// element (as in the stand-alone quantiser, quant_math.cuh) -- computed as -u = fma(x, -gamma, b),
// which needs no negated copy of b; |-u| = |u| for the absmax, and pass 1 rounds (-u) * (-inv), the
// same exact product as u * inv.
// AQ (NEXT-1): per-token asymmetric codes -- pass 0 tracks max u (m) and max -u (m2), pass 1 rounds
// (u - z) * inv to 0 .. 15 (quant_math.cuh A1-A3).  With GBF16 the chunk holds -u: the two maxima
// swap roles, and (-u) - (-z) = -(u - z) times -inv is the same exact product.
template <int PASS, int HAD, bool GBF16, int QC, bool AQ>
__device__ __forceinline__ void quant_chunk(const uint4* __restrict__ xr, const float* __restrict__ bvec,
                                            float gamma, float had_scale, int lane, int nv, int nvl,
                                            int c0, float inv, float z, float& m, float& m2,
                                            uint32_t* __restrict__ cr) {
  static_assert(!(GBF16 && HAD != 0), "the bf16 fma consumes the packed activations as they are");
  uint4 sx[kQD];
  float4 sb0[kQD], sb1[kQD];
  auto issue = [&](int d, int j) {
    int i = lane + 32 * j;
    i = i < nv ? i : nv - 1;
    sx[d] = __ldg(xr + i);
    sb0[d] = __ldg(reinterpret_cast<const float4*>(bvec) + 2 * i);
    sb1[d] = __ldg(reinterpret_cast<const float4*>(bvec) + 2 * i + 1);
  };
#pragma unroll
  for (int d = 0; d < kQD; ++d) issue(d, c0 + d);
  if (PASS == 0) {
    // the chunk after the next one, towards L2: the ring's own depth covers an L2 hit, not an HBM miss
    // (measured: asking for the next row's head during pass 1 as well cost 4 % of the fused launch)
    const int jp = c0 + 2 * QC + (lane >> 2);             // 8 steps x 4 lines of 128 bytes
    const int vp = 32 * jp + 8 * (lane & 3);              // first vector of this lane's line
    if (vp < nv) ptx::prefetch_l2(xr + vp);               // never past the end of the row
  }
#pragma unroll
  for (int t = 0; t < QC; ++t) {
    const int d = t % kQD;
    const int j = c0 + t;
    const int i = lane + 32 * j;
    const bool valid = j < nvl && i < nv;
    float u[8];
    const float bb[8] = {sb0[d].x, sb0[d].y, sb0[d].z, sb0[d].w, sb1[d].x, sb1[d].y, sb1[d].z, sb1[d].w};
    if (GBF16) {
      const uint32_t ng = (__float_as_uint(gamma) >> 16) ^ 0x8000u;       // -gamma as bf16 bits
      qm::affine8_bf16(sx[d], ng, bb, u);                                 // u := -(gamma x - b)
    } else {
      float f[8];
      qm::unpack8(sx[d], f);
      if (HAD != 0) qm::hadamard8(f, HAD, had_scale, lane);
#pragma unroll
      for (int e = 0; e < 8; ++e) u[e] = qm::affine(gamma, f[e], bb[e]);
    }
    if (PASS == 0) {
      if (AQ) {
        float mx = m, mn = m2;
        if (GBF16) qm::maxmin8(mn, mx, u);
        else qm::maxmin8(mx, mn, u);
        m = valid ? mx : m;
        m2 = valid ? mn : m2;
      } else {
        const float mm = qm::absmax8(m, u);
        m = valid ? mm : m;
      }
    } else {
      const uint32_t w = AQ ? qm::quantize_pack8_asym(u, GBF16 ? -z : z, GBF16 ? -inv : inv)
                            : qm::quantize_pack8(u, GBF16 ? -inv : inv);
      if (valid) cr[i] = w;
    }
    if (t + kQD < QC) issue(d, j + kQD);
  }
}
// Any parameter combination, one vector step at a time (loads not pipelined).
template <int PASS, bool AQ>
__device__ __forceinline__ void quant_step_generic(const uint4* __restrict__ xr, const float* __restrict__ bvec,
                                                   const float* __restrict__ sa, float gamma, int had_block,
                                                   float had_scale, int lane, int nv, int j, float inv,
                                                   float z, float& m, float& m2, uint32_t* __restrict__ cr) {
  const int i = lane + 32 * j;
  const bool ok = i < nv;
  const uint4 v = ok ? __ldg(xr + i) : make_uint4(0u, 0u, 0u, 0u);
  float f[8], g[8], bb[8], u[8];
  qm::unpack8(v, f);
  if (had_block) qm::hadamard8(f, had_block, had_scale, lane);
  qm::load_gb(sa, bvec, gamma, i, ok, g, bb);
#pragma unroll
  for (int e = 0; e < 8; ++e) u[e] = qm::affine(g[e], f[e], bb[e]);
  if (ok) {
    if (PASS == 0) {
      if (AQ) qm::maxmin8(m, m2, u);
      else m = qm::absmax8(m, u);
    } else {
      cr[i] = AQ ? qm::quantize_pack8_asym(u, z, inv) : qm::quantize_pack8(u, inv);
    }
  }
}

// Fused variant: the workspace's counters start from whatever the last user of the memory left.
// CTA 0 clears them (and the CTA-exit count) and then publishes kFusedReady in the control block;
// every reader or incrementer of a counter first waits for that word; the last CTA to finish puts
// the word back to 0, so the next call on this workspace -- or the next replay of a captured graph
// -- finds it unset again.  (A memset node in front of the kernel would do, but it serialises the
// launch against its predecessor: ~6 us per call.)  Memory that has never been a workspace holds
// the 64-bit word by chance with probability 2^-64.
constexpr unsigned long long kFusedReady = 0x51534142465553EDull;
__device__ __forceinline__ void fused_wait_ready(const unsigned long long* ctrl) {
  while (ptx::ld_acquire_gpu_u64(ctrl) != kFusedReady) ptx::nanosleep(64);
}

// ------------------------------------------------------------------------------ the kernel
// ASYM (NEXT-1): unsigned activation codes, re-centred to q - 8 while they are expanded, and the
// epilogue term (z_t + 8 s_t) s_w wsum[n].
template <bool FUSED, bool ASYM>
__global__ void __launch_bounds__((Cfg<FUSED>::kThreads), 1)
w4a4_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_y,
                 const GemmParams p) {
  using C = Cfg<FUSED>;
  constexpr int kEpiWarps = C::kEpiWarps;
  constexpr int kEpiWarp0 = C::kEpiWarp0;
  constexpr int kAWarp0 = C::kAWarp0;
  constexpr int kUnpackWarp0 = C::kUnpackWarp0;
  constexpr int kProducerWarp = C::kProducerWarp, kProducerWarpB = C::kProducerWarpB, kMmaWarp = C::kMmaWarp;
  extern __shared__ uint8_t smem_raw[];
  // SWIZZLE_128B operands need 1024-byte alignment
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
  // [ int8 B stages | packed ring | barriers | column operands | Y staging ]
  const uint32_t unpacked0 = smem_base;
  const uint32_t packed0 = unpacked0 + kStages * C::kUnpackedStage;
  uint8_t* unpacked_ptr = smem;
  uint8_t* packed_ptr = unpacked_ptr + kStages * C::kUnpackedStage;
  Barriers* bars = reinterpret_cast<Barriers*>(packed_ptr + C::kPStages * C::kPackedStage);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();
  const bool leader = rank == 0;
  // The blob's header (written by the packer's first kernel, complete long before any dependent
  // launch can start: see w4a4_decode.cu) is requested now and compared with the call's (N, K) after
  // the prologue: a blob packed for another shape would be read out of bounds, so such a call does
  // no work at all and raises the status word (baseq_sync_status -> BASEQ_ERR_WORKSPACE).
  const uint4 hdr = ptx::ldg_nc(reinterpret_cast<const uint4*>(p.header));

  if (warp == kProducerWarp && lane == 0) {
    ptx::prefetch_tensormap(&tmap_a);
    ptx::prefetch_tensormap(&tmap_y);
    for (int i = 0; i < C::kPStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->pfull[i]), C::kPFullCount);
      ptx::mbar_init(ptx::smem_u32(&bars->pempty[i]), C::kPEmptyCount);
    }
    for (int i = 0; i < kStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->full[i]), C::kFullCount);
      ptx::mbar_init(ptx::smem_u32(&bars->empty[i]), 1);
    }
    for (int i = 0; i < kAccStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->tfull[i]), 1);
      ptx::mbar_init(ptx::smem_u32(&bars->tempty[i]), C::kTemptyCount);
    }
    ptx::fence_barrier_init();
  }
  if (warp == kMmaWarp) {
    ptx::tmem_alloc_2cta<kTmemCols>(ptx::smem_u32(&bars->tmem_base));
  }
  ptx::tcgen05_fence_before();
  __syncthreads();
  ptx::cluster_sync_all();                    // peer barriers initialised before any remote arrive
  ptx::tcgen05_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&bars->tmem_base);
  // prologue done (barriers, TMEM, tensor maps): from here on the predecessor's outputs are read
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  const bool blob_ok = hdr.x == kBlobMagic && hdr.y == static_cast<uint32_t>(p.N) &&
                       hdr.z == static_cast<uint32_t>(p.K);
  if (!blob_ok && threadIdx.x == 0 && blockIdx.x == 0) atomicOr(p.status, kStatusBadBlob);
  const int num_tiles = blob_ok ? p.num_m * p.num_n : 0;
  const int first_tile = static_cast<int>(blockIdx.x) / CG;
  const int tile_step = static_cast<int>(gridDim.x) / CG;
  const int n_it = first_tile < num_tiles
                       ? ((num_tiles - first_tile + tile_step - 1) / tile_step) * p.num_kb : 0;
  // tile -> (m_blk, n_blk).  Unfused: N-major walk (consecutive tiles share a weight strip).  Fused:
  // M-major, so that a wave of tiles needs one or two 256-row strips of codes, in increasing order.
  auto tile_m = [&](int tile) { return FUSED ? tile / p.num_n : tile % p.num_m; };
  auto tile_n = [&](int tile) { return FUSED ? tile % p.num_n : tile / p.num_m; };
  // fused: rows of this CTA's 128-row group of strip m that the quantiser warps will deliver
  auto group_rows = [&](int m_blk) {
    const int r0 = m_blk * (BM * CG) + static_cast<int>(rank) * BM;
    return r0 >= p.T ? 0 : (p.T - r0 < BM ? p.T - r0 : BM);
  };

  // Fused variant: 1024 threads start with 64 registers each; the warpgroups trade them so that
  // the epilogue warps get 80 and the quantiser group can hold a token row (up to kQV vectors per
  // thread) in registers:
  //   2 x 4 x 32 x 80 (epilogue) + 2 x 4 x 32 x 48 (A) + 2 x 4 x 32 x 40 (B) + 4 x 32 x 48 (roles)
  //   + 4 x 32 x 128 (quantiser) = 65536.
  if (warp >= C::kRoleWarp0 && warp < C::kRoleWarp0 + 4) {
    if (FUSED) ptx::setmaxnreg_dec<48>();
  }
  if (warp == kProducerWarp || warp == kProducerWarpB) {
    // ===================================================================== producers (TMA)
    // Two warps, one per operand: a single warp's wait + expect_tx + two copy issues per k-block
    // is a ~350 clk serial chain (measured with everything else stubbed out).
    const bool is_a = warp == kProducerWarp;
    int stage = 0;
    uint32_t phase = 0;
    for (int tile = first_tile; tile < num_tiles; tile += tile_step) {
      const int m_blk = tile_m(tile), n_blk = tile_n(tile);
      const int row0 = m_blk * (BM * CG) + static_cast<int>(rank) * BM;
      // row groups of kTileRows rows: this CTA streams its half of the tile's N rows
      const uint8_t* g0 = p.tiles + static_cast<size_t>(2 * n_blk + rank) * p.num_kb * kTileBytes;
      if (FUSED && is_a) {
        // the codes of this CTA's 128 rows come from the quantiser warps of the whole grid
        const unsigned int need = static_cast<unsigned int>(group_rows(m_blk));
        const unsigned int* flag = p.ready + (2 * m_blk + static_cast<int>(rank));
        if (tile == first_tile) fused_wait_ready(p.ctrl);
        while (ptx::ld_acquire_gpu(flag) < need) ptx::nanosleep(64);
        ptx::fence_proxy_async_global();          // their generic-proxy stores -> this warp's TMA reads
      }
      for (int kb = 0; kb < p.num_kb; ++kb) {
        ptx::mbar_wait(ptx::smem_u32(&bars->pempty[stage]), phase ^ 1u);
        const uint32_t full = ptx::smem_u32(&bars->pfull[stage]);
        const uint32_t dst = packed0 + stage * C::kPackedStage;
        if (ptx::elect_one()) {
          if (is_a) {
            // A: 128 rows x 64 B of codes, SWIZZLE_64B; rows beyond T are zero-filled by TMA
            ptx::mbar_arrive_expect_tx(full, kPackedA);
            ptx::tma_load_2d(dst, &tmap_a, kb * (BK / 2), row0, full);
          } else {
            ptx::mbar_arrive_expect_tx(full, C::kPackedB);
            ptx::bulk_load_1d(dst + kPackedA, g0 + static_cast<size_t>(kb) * kTileBytes,
                              kTileBytes, full);
          }
        }
        __syncwarp();
        advance(stage, phase, C::kPStages);
      }
    }
  } else if (warp == kMmaWarp) {
    // ===================================================================== MMA issuer
    // The whole warp runs the loop in uniform control flow and one elected lane issues: with a
    // divergent `lane == 0` region ptxas wraps every tcgen05 instruction in a vote/elect/R2UR
    // waterfall (~95 SASS instructions and ~670 clk per k-block, measured -- slower than the
    // 384 clk the four MMAs take).
    if (leader) {
      constexpr uint32_t idesc = ptx::make_idesc_i8(BM * CG, BN);
      int as = 0;
      uint32_t phase = 0, aphase = 0;
      const uint64_t desc0 = ptx::make_smem_desc_sw128(unpacked0);
      // Flat k-block index over all of this CTA pair's tiles, unrolled over the kStages operand
      // stages: the stage index is a compile-time constant, so the barrier addresses, the TMEM
      // column of A and the descriptor of B are constants off loop-invariant bases (r1i capture:
      // the issuing warp spent ~60 % of a k-block period executing a 52-instruction loop body,
      // eight of them R2UR moves of per-stage values -- close to the 384 clk the MMAs take).
      int kb = 0;
      uint32_t tmem_d = tmem_base;
      if (n_it > 0) {
        ptx::mbar_wait(ptx::smem_u32(&bars->tempty[0]), 1u);
        ptx::tcgen05_fence_after();
      }
      for (int base = 0; base < n_it; base += kStages) {
#pragma unroll
        for (int stage = 0; stage < kStages; ++stage) {
          if (base + stage < n_it) {
            ptx::mbar_wait(ptx::smem_u32(&bars->full[stage]), phase);
            ptx::tcgen05_fence_after();
            if (ptx::elect_one()) {
              const uint32_t a_col = tmem_base + kACol0 + stage * (BK / 4);
              // descriptor start-address field is in 16-byte units: + stage bytes/16, + 2 per K chunk
              const uint64_t db = desc0 + static_cast<uint64_t>(stage * (C::kUnpackedStage >> 4));
#pragma unroll
              for (int k = 0; k < BK / 32; ++k) {
                const uint32_t accum = (k != 0 || kb != 0) ? 1u : 0u;
                ptx::mma_i8_ts_2cta(tmem_d, a_col + k * 8, db + 2 * k, idesc, accum);
              }
              // frees the operand stage (A columns + B smem) in every CTA of the pair
              ptx::tcgen05_commit_2cta(ptx::smem_u32(&bars->empty[stage]), 3);
            }
            __syncwarp();
            if (++kb == p.num_kb) {
              // tile complete: publish the accumulator, move to the other accumulator stage
              kb = 0;
              if (ptx::elect_one()) {
                ptx::tcgen05_commit_2cta(ptx::smem_u32(&bars->tfull[as]), 3);
              }
              __syncwarp();
              advance(as, aphase, kAccStages);
              tmem_d = tmem_base + as * BN;
              if (base + stage + 1 < n_it) {
                ptx::mbar_wait(ptx::smem_u32(&bars->tempty[as]), aphase ^ 1u);
                ptx::tcgen05_fence_after();
              }
            }
          }
        }
        phase ^= 1u;
      }
    }
  } else if (warp >= kUnpackWarp0 && warp < kUnpackWarp0 + kNumUnpackWarps * kSets) {
    // ===================================================================== B: int4 -> int8
    if (FUSED) ptx::setmaxnreg_dec<40>();
    const int ut = (threadIdx.x - kUnpackWarp0 * 32) & 127;   // 0..127 inside the set
    const int set = (warp - kUnpackWarp0) >> 2;
    constexpr int kTasks = C::kBRows * 4 / (kNumUnpackWarps * 32);   // 16-byte chunks per thread
    static_assert(C::kBRows * 4 % (kNumUnpackWarps * 32) == 0, "unpack tasks");
    const uint32_t full_remote = ptx::mapa_cluster(ptx::smem_u32(&bars->full[0]), 0);
    // flat k-block index over all of this CTA's tiles; this set takes every kSets-th one (the
    // operand warps never need the tile coordinates)
    {
      for (uint32_t it = set; it < static_cast<uint32_t>(n_it); it += kSets) {
        const uint32_t ps = it % C::kPStages, us = it % kStages;      // unsigned: plain masks
        const uint32_t pphase = (it / C::kPStages) & 1u, uphase = (it / kStages) & 1u;
        ptx::mbar_wait(ptx::smem_u32(&bars->pfull[ps]), pphase);
        const uint8_t* src = packed_ptr + ps * C::kPackedStage + kPackedA;
        uint4 v[kTasks];
#pragma unroll
        for (int i = 0; i < kTasks; ++i)
          v[i] = *reinterpret_cast<const uint4*>(src + (ut + i * 128) * 16);
        ptx::mbar_wait(ptx::smem_u32(&bars->empty[us]), uphase ^ 1u);
        uint8_t* dst = unpacked_ptr + us * C::kUnpackedStage;
#pragma unroll
        for (int i = 0; i < kTasks; ++i) {
          const int task = ut + i * 128;
          const int row = task >> 2, c = task & 3, rsub = row & 7;
          uint4 lo, hi;
          lo.x = (v[i].x << 4) & 0xF0F0F0F0u; hi.x = v[i].x & 0xF0F0F0F0u;
          lo.y = (v[i].y << 4) & 0xF0F0F0F0u; hi.y = v[i].y & 0xF0F0F0F0u;
          lo.z = (v[i].z << 4) & 0xF0F0F0F0u; hi.z = v[i].z & 0xF0F0F0F0u;
          lo.w = (v[i].w << 4) & 0xF0F0F0F0u; hi.w = v[i].w & 0xF0F0F0F0u;
          uint8_t* rp = dst + row * 128;                  // 8-row swizzle atoms of 1024 bytes
          *reinterpret_cast<uint4*>(rp + (((2 * c) ^ rsub) << 4)) = lo;
          *reinterpret_cast<uint4*>(rp + (((2 * c + 1) ^ rsub) << 4)) = hi;
        }
        ptx::fence_proxy_async_smem();      // generic-proxy writes -> visible to tcgen05.mma
        __syncwarp();
        if (lane == 0) {
          ptx::mbar_arrive(ptx::smem_u32(&bars->pempty[ps]));
          ptx::mbar_arrive_cluster(full_remote + us * 8);
        }
      }
    }
  } else if (FUSED && warp < C::kQuantWarp0 + kQuantWarps) {
    // ===================================================================== background quantiser
    // One token row per warp, claimed from a counter (see below).  Lane l owns the 16-byte vectors
    // l, l + 32, ... of the row, so an aligned half-warp holds 128 consecutive channels (what qm::hadamard8's shuffle
    // stages expect; a 256-channel block spans the warp).  Same arithmetic (quant_math.cuh) and
    // therefore the same codes as the stand-alone quantiser.  Two passes over the row -- absmax,
    // then round and pack; the second one re-reads the row from L2 and recomputes u.  No
    // shared-memory staging: the GEMM around these warps runs at the shared-memory bandwidth
    // limit, and it leaves 40 % of the issue slots and most of HBM idle.
    ptx::setmaxnreg_inc<128>();
    const int gw = static_cast<int>(blockIdx.x) * kQuantWarps + (warp - C::kQuantWarp0);
    const int nv = p.K >> 3;
    const int nvl = (nv + 31) >> 5;                   // vectors per lane (the last one may be idle)
    // 0 / 1: pipelined chunks without / with the block-128 Hadamard; 3: as 0 with the bf16 fma
    // (scalar s^a that is a bf16 value: 1.0 in four of the five configs); 2: generic steps
    const int mode = (p.bvec == nullptr || p.sa != nullptr) ? 2
                     : p.had_block == 0 ? (qm::is_bf16_value(p.gamma) ? 3 : 0)
                     : p.had_block == 128 ? 1 : 2;
    if (gw == 0 && num_tiles > 0) {
      // clear the counters and the exit count, then publish: see kFusedReady
      for (int i = lane; i < p.ngroups; i += 32) p.ready[i] = 0u;
      if (lane == 0) {
        p.ctrl[1] = 0ull;          // CTAs that have finished
        p.ctrl[2] = 0ull;          // next token row to quantise
      }
      __syncwarp();
      if (lane == 0) {
        __threadfence();
        ptx::st_release_gpu_u64(p.ctrl, kFusedReady);
      }
    }
    // Rows are CLAIMED, not assigned: a warp takes the next row from a counter in the control block
    // (in increasing order, so 256-row strips complete in the order the tile walk needs them).  With
    // a static assignment the GEMM warps of a resident CTA would wait for rows owned by a CTA that
    // is not resident yet -- a second spin-waiting kernel on another stream holding the remaining SMs
    // would then deadlock both.  Claimed rows need nothing from a CTA that is not running (CTA 0,
    // which clears the control block, is the first to be placed).  The claim for the next row is
    // issued before the current one is processed, so its L2 round trip is hidden; the first one costs
    // the launch about 2 us (measured against the static assignment: c3 up 135.7 -> 138.7 us; long
    // rows gain from the balancing: c3 down 162.6 -> 158.3 us).
    unsigned int* next_row = reinterpret_cast<unsigned int*>(p.ctrl + 2);
    int row = p.T;
    if (num_tiles > 0) {
      if (lane == 0) {
        fused_wait_ready(p.ctrl);
        row = static_cast<int>(atomicAdd(next_row, 1u));
      }
      row = __shfl_sync(0xffffffffu, row, 0);
    }
    while (row < p.T) {
      int claimed = 0;
      if (lane == 0) claimed = static_cast<int>(atomicAdd(next_row, 1u));
      const uint4* xr = p.x + static_cast<int64_t>(row) * p.ldxv;
      uint32_t* cr = p.codes_out + static_cast<int64_t>(row) * nv;
      // symmetric: m = max |u|; asymmetric: m = max u, m2 = max -u
      float m = ASYM ? -3.402823466e38f : 0.0f, m2 = -3.402823466e38f;
      if (mode == 0) {
#pragma unroll 1
        for (int c0 = 0; c0 < nvl; c0 += kQC)
          quant_chunk<0, 0, false, kQC, ASYM>(xr, p.bvec, p.gamma, p.had_scale, lane, nv, nvl, c0, 0.0f, 0.0f, m, m2, cr);
      } else if (mode == 3) {
#pragma unroll 1
        for (int c0 = 0; c0 < nvl; c0 += kQC)
          quant_chunk<0, 0, true, kQC, ASYM>(xr, p.bvec, p.gamma, p.had_scale, lane, nv, nvl, c0, 0.0f, 0.0f, m, m2, cr);
      } else if (mode == 1) {
#pragma unroll 1
        for (int c0 = 0; c0 < nvl; c0 += kQC)
          quant_chunk<0, 128, false, kQC, ASYM>(xr, p.bvec, p.gamma, p.had_scale, lane, nv, nvl, c0, 0.0f, 0.0f, m, m2, cr);
      } else {
#pragma unroll 1
        for (int j = 0; j < nvl; ++j)
          quant_step_generic<0, ASYM>(xr, p.bvec, p.sa, p.gamma, p.had_block, p.had_scale, lane, nv, j, 0.0f, 0.0f, m, m2, cr);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (ASYM) m2 = fmaxf(m2, __shfl_xor_sync(0xffffffffu, m2, o));
      }
      const float st = ASYM ? qm::step_size_asym(p.alpha, -m2, m) : qm::step_size(p.alpha, m);
      const float zt = ASYM ? qm::lower_bound_asym(p.alpha, -m2) : 0.0f;
      const float inv = qm::reciprocal(st);
      if (mode == 0) {
#pragma unroll 1
        for (int c0 = 0; c0 < nvl; c0 += kQC)
          quant_chunk<1, 0, false, kQC, ASYM>(xr, p.bvec, p.gamma, p.had_scale, lane, nv, nvl, c0, inv, zt, m, m2, cr);
      } else if (mode == 3) {
#pragma unroll 1
        for (int c0 = 0; c0 < nvl; c0 += kQC)
          quant_chunk<1, 0, true, kQC, ASYM>(xr, p.bvec, p.gamma, p.had_scale, lane, nv, nvl, c0, inv, zt, m, m2, cr);
      } else if (mode == 1) {
#pragma unroll 1
        for (int c0 = 0; c0 < nvl; c0 += kQC)
          quant_chunk<1, 128, false, kQC, ASYM>(xr, p.bvec, p.gamma, p.had_scale, lane, nv, nvl, c0, inv, zt, m, m2, cr);
      } else {
#pragma unroll 1
        for (int j = 0; j < nvl; ++j)
          quant_step_generic<1, ASYM>(xr, p.bvec, p.sa, p.gamma, p.had_block, p.had_scale, lane, nv, j, inv, zt, m, m2, cr);
      }
      if (ASYM && lane == 0) p.zeros_out[row] = zt;
      if (lane == 0) p.scales_out[row] = st;
      __syncwarp();
      if (lane == 0) ptx::red_release_gpu_add(p.ready + (row >> 7), 1u);
      row = __shfl_sync(0xffffffffu, claimed, 0);
    }
  } else if (warp >= kAWarp0 && warp < kAWarp0 + 8) {
    // ===================================================================== A: smem -> TMEM
    if (FUSED) ptx::setmaxnreg_dec<48>();
    // thread = token row = TMEM lane.  The packed tile is [128 rows][64 B] with TMA's SWIZZLE_64B
    // (16-byte chunk index ^= (row >> 1) & 3), so the 32 lanes' 16-byte reads of one chunk column
    // spread over all banks (4 wavefronts per 512 B: the minimum).
    const int q = warp & 3;                               // TMEM lane quarter
    const int arow = q * 32 + lane;
    const uint32_t full_remote = ptx::mapa_cluster(ptx::smem_u32(&bars->full[0]), 0);
    const uint32_t a_taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + kACol0;
    const int sw = (arow >> 1) & 3;
    const int set = (warp - kAWarp0) >> 2;
    {
      for (uint32_t it = set; it < static_cast<uint32_t>(n_it); it += kSets) {
        const uint32_t ps = it % C::kPStages, us = it % kStages;      // unsigned: plain masks
        const uint32_t pphase = (it / C::kPStages) & 1u, uphase = (it / kStages) & 1u;
        ptx::mbar_wait(ptx::smem_u32(&bars->pfull[ps]), pphase);
        const uint8_t* src = packed_ptr + ps * C::kPackedStage + arow * 64;
        uint4 w4[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) w4[c] = *reinterpret_cast<const uint4*>(src + ((c ^ sw) << 4));
        uint32_t r[32];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const uint4 w = w4[c];
          // ASYM: the unsigned code q becomes the signed byte 16 (q - 8) (flip the byte's top bit;
          // the xor folds into the same LOP3), so the MMA accumulates acc' = acc - 8 wsum
          constexpr uint32_t kFlip = ASYM ? 0x80808080u : 0u;
          r[8 * c + 0] = ((w.x << 4) & 0xF0F0F0F0u) ^ kFlip; r[8 * c + 4] = (w.x & 0xF0F0F0F0u) ^ kFlip;
          r[8 * c + 1] = ((w.y << 4) & 0xF0F0F0F0u) ^ kFlip; r[8 * c + 5] = (w.y & 0xF0F0F0F0u) ^ kFlip;
          r[8 * c + 2] = ((w.z << 4) & 0xF0F0F0F0u) ^ kFlip; r[8 * c + 6] = (w.z & 0xF0F0F0F0u) ^ kFlip;
          r[8 * c + 3] = ((w.w << 4) & 0xF0F0F0F0u) ^ kFlip; r[8 * c + 7] = (w.w & 0xF0F0F0F0u) ^ kFlip;
        }
        ptx::mbar_wait(ptx::smem_u32(&bars->empty[us]), uphase ^ 1u);
        ptx::tcgen05_fence_after();
        ptx::tmem_st_32x32b_x32(a_taddr + us * (BK / 4), r);
        ptx::tmem_st_wait();
        ptx::tcgen05_fence_before();
        __syncwarp();
        if (lane == 0) {
          ptx::mbar_arrive_cluster(full_remote + us * 8);
          // the store consumed every lane's smem reads: the packed stage may be refilled
          ptx::mbar_arrive(ptx::smem_u32(&bars->pempty[ps]));
        }
      }
    }
  } else if (warp >= kEpiWarp0 && warp < kEpiWarp0 + kEpiWarps) {
    // ===================================================================== epilogue
    if (FUSED) ptx::setmaxnreg_inc<80>();
    // 8 warps: warp % 4 = TMEM lane quarter (32 token rows), (warp - kEpiWarp0) / 4 = which half
    // of the tile's BN columns.  16 columns per tcgen05.ld keep the register footprint small.
    const int q = warp & 3;
    const int half = (warp - kEpiWarp0) >> 2;
    // The tile's column operands are staged in shared memory by the epilogue threads themselves:
    // fetched one tile ahead into registers (latency hidden behind the previous tile), published
    // before the accumulator wait, read back with broadcast LDS.128 -- no global-load latency
    // inside the chunk loop (r1h capture: 44 % of the epilogue warps' time).  Reuse of a stage's
    // copy is ordered by the per-tile named barrier (a warp arrives at tile i's barrier only after
    // it finished tile i-1, so nobody still reads the copy of tile i-2).
    constexpr int kEpiThreads = kEpiWarps * 32;
    constexpr int kPer = (BN + kEpiThreads - 1) / kEpiThreads;
    float* colp = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(bars) + 256);
    const int et = static_cast<int>(threadIdx.x) - kEpiWarp0 * 32;
    float pre[kPer][3];
    auto fetch = [&](int tile) {
      const int nb = tile_n(tile) * BN;
#pragma unroll
      for (int i = 0; i < kPer; ++i) {
        const int c = et + i * kEpiThreads;
        if (c < BN) {
          pre[i][0] = __ldg(p.sw + nb + c);
          pre[i][1] = __ldg(p.fb + nb + c);
          pre[i][2] = ASYM ? __ldg(p.wsum + nb + c) : 0.0f;
        }
      }
    };
    if (first_tile < num_tiles) fetch(first_tile);
    // TMA-store epilogue: this warp's 32 x 96 bf16 block is staged in shared memory in the
    // SWIZZLE_64B layout of three 32-row x 64-byte boxes (lane = row, conflict-free STS.128) and
    // written by three bulk tensor stores -- a per-lane STG.128 touches 32 different 128-byte lines
    // (32 L1 tag cycles per instruction: 20 % of the LSU pipe's load in the r1h capture); TMA also
    // clips rows >= T and columns >= N.
    const uint32_t stage_y = ptx::smem_u32(bars) + C::kTailBytes + (warp - kEpiWarp0) * C::kStoreWarpBytes;
    const uint32_t stage_lane = stage_y + lane * 64;
    const uint32_t stage_sw = (lane >> 1) & 3;
    constexpr int kColsPerWarp = BN / (kEpiWarps / 4);
    const uint32_t tempty_remote = ptx::mapa_cluster(ptx::smem_u32(&bars->tempty[0]), 0);
    int as = 0;
    uint32_t aphase = 0;
    for (int tile = first_tile; tile < num_tiles; tile += tile_step) {
      const int m_blk = tile_m(tile), n_blk = tile_n(tile);
      const int row = m_blk * (BM * CG) + static_cast<int>(rank) * BM + q * 32 + lane;
      const bool row_ok = row < p.T;
      float st = 0.0f;
      if (FUSED) {
        // the scale was written by a quantiser warp of some CTA during this launch: observe the
        // group's counter (long complete: the A producer waited for it before this tile's first
        // load) and read the scale past L1
        const unsigned int need = static_cast<unsigned int>(group_rows(m_blk));
        const unsigned int* flag = p.ready + (2 * m_blk + static_cast<int>(rank));
        if (tile == first_tile) fused_wait_ready(p.ctrl);
        while (ptx::ld_acquire_gpu(flag) < need) ptx::nanosleep(64);
        if (row_ok) st = ptx::ld_relaxed_gpu_f32(p.scales + row);
      } else if (row_ok) {
        st = p.scales[row];
      }
      const float st256 = __fmul_rn(st, 0.00390625f);
      const float zt = (ASYM && row_ok) ? (FUSED ? ptx::ld_relaxed_gpu_f32(p.zeros + row) : p.zeros[row]) : 0.0f;
      const float midf = __fmaf_rn(8.0f, st, zt);
      float* cs = colp + as * 3 * BN;
#pragma unroll
      for (int i = 0; i < kPer; ++i) {
        const int c = et + i * kEpiThreads;
        if (c < BN) {
          cs[c] = pre[i][0];
          cs[BN + c] = pre[i][1];
          // third column operand: wsum (asymmetric) or |fb| + 2^-100 for the bracket
          cs[2 * BN + c] = ASYM ? pre[i][2] : __fadd_rn(fabsf(pre[i][1]), 7.888609052210118e-31f);
        }
      }
      ptx::bar_sync(1, kEpiThreads);
      if (tile + tile_step < num_tiles) fetch(tile + tile_step);
      cs += half * kColsPerWarp;
      if (lane == 0) ptx::bulk_wait_group_read<0>();   // the previous tile's stores have read the staging tile
      __syncwarp();
      ptx::mbar_wait(ptx::smem_u32(&bars->tfull[as]), aphase);
      ptx::tcgen05_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + as * BN +
                             half * kColsPerWarp;
      const int n0 = n_blk * BN + half * kColsPerWarp;
      // 8 columns: two groups of 4 -> one 16-byte store per row
      auto process8 = [&](const uint32_t (&r)[8], int c0) {
        uint32_t out[4];
#pragma unroll
        for (int j = 0; j < 8; j += 4) {
          const float4 sw = *reinterpret_cast<const float4*>(cs + c0 + j);
          const float4 fb = *reinterpret_cast<const float4*>(cs + BN + c0 + j);
          const float4 ws = *reinterpret_cast<const float4*>(cs + 2 * BN + c0 + j);
          const float swv[4] = {sw.x, sw.y, sw.z, sw.w}, fbv[4] = {fb.x, fb.y, fb.z, fb.w};
          const float wsv[4] = {ws.x, ws.y, ws.z, ws.w};
          float lo[4], hi[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            if (ASYM) dequant_bracket_asym(static_cast<int32_t>(r[j + e]), st256, midf, swv[e], fbv[e], wsv[e], lo[e], hi[e]);
            else dequant_bracket(static_cast<int32_t>(r[j + e]), st256, swv[e], fbv[e], wsv[e], lo[e], hi[e]);
          }
          // output words of the low ends and of the high ends of the four brackets
          uint32_t lo01 = pack_bf16x2(lo[1], lo[0]), lo23 = pack_bf16x2(lo[3], lo[2]);
          const uint32_t d01 = lo01 ^ pack_bf16x2(hi[1], hi[0]), d23 = lo23 ^ pack_bf16x2(hi[3], hi[2]);
          if ((d01 | d23) != 0) {
            // rare (2.4e-4 of the elements, symmetric; ~1e-3 asymmetric): some bracket of this
            // group straddles a bf16 rounding boundary -- evaluate the fp64 expression itself for
            // those elements (operands are still in registers)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const uint32_t d = (e < 2) ? d01 : d23;
              if (((e & 1) ? (d >> 16) : (d & 0xFFFFu)) != 0) {
                const int32_t a = static_cast<int32_t>(r[j + e]) >> 8;
                const uint32_t v = ASYM ? dequant_f64_asym(a, st, zt, swv[e], fbv[e], wsv[e])
                                        : dequant_f64(a, st, swv[e], fbv[e]);
                uint32_t& w = (e < 2) ? lo01 : lo23;
                w = (e & 1) ? ((w & 0x0000FFFFu) | (v << 16)) : ((w & 0xFFFF0000u) | v);
              }
            }
          }
          out[j >> 1] = lo01;
          out[(j >> 1) + 1] = lo23;
        }
        const int n = n0 + c0;
        const uint32_t dst = stage_lane + ((c0 >> 5) << 11) + ((((c0 >> 3) & 3) ^ stage_sw) << 4);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "r"(out[0]), "r"(out[1]),
                     "r"(out[2]), "r"(out[3]) : "memory");
        if (row_ok && n < p.N) {
          if (p.acc_dump != nullptr) {
            int32_t* d = p.acc_dump + static_cast<int64_t>(row) * p.N + n;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
              int32_t a = static_cast<int32_t>(r[e]) >> 8;                      // raw = 256 * acc
              if (ASYM) a += 8 * static_cast<int32_t>(__ldg(p.wsum + n + e));   // acc' -> acc
              d[e] = a;
            }
          }
        }
      };
      // double-buffered TMEM reads: the load of the next 8 columns is in flight while these 8 are
      // converted
      static_assert(kColsPerWarp % 16 == 0, "chunk pairs");
      uint32_t ra[8], rb[8];
      ptx::tmem_ld_32x32b_x8(taddr, ra);
#pragma unroll 1
      for (int c0 = 0; c0 < kColsPerWarp; c0 += 16) {
        if (n0 + c0 >= p.N) break;                      // warp-uniform
        ptx::tmem_ld_wait_for(ra);
        ptx::tmem_ld_32x32b_x8(taddr + c0 + 8, rb);
        process8(ra, c0);
        ptx::tmem_ld_wait_for(rb);
        if (c0 + 16 < kColsPerWarp) ptx::tmem_ld_32x32b_x8(taddr + c0 + 16, ra);
        process8(rb, c0 + 8);
      }
      ptx::tmem_ld_wait();
      ptx::fence_proxy_async_smem();                  // this lane's STS -> visible to the TMA engine
      __syncwarp();
      const int row0 = m_blk * (BM * CG) + static_cast<int>(rank) * BM + q * 32;
      if (lane == 0 && row0 < p.T) {
#pragma unroll
        for (int bx = 0; bx < kColsPerWarp / 32; ++bx)
          if (n0 + bx * 32 < p.N) ptx::tma_store_2d(&tmap_y, stage_y + bx * 2048, n0 + bx * 32, row0);
        ptx::bulk_commit_group();
      }
      // all TMEM reads of this warp are complete (wait::ld above): release the accumulator
      ptx::tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster(tempty_remote + as * 8);
      advance(as, aphase, kAccStages);
    }
  }

  // ---- teardown: nobody leaves while the peer may still touch this CTA's barriers / smem
  if (warp >= kEpiWarp0 && warp < kEpiWarp0 + kEpiWarps && lane == 0)
    ptx::bulk_wait_group<0>();                          // Y stores complete before the CTA exits
  ptx::tcgen05_fence_before();
  __syncthreads();
  if (FUSED && num_tiles > 0 && threadIdx.x == 0) {
    // every role of this CTA is past its last look at the control word: count the exit
    const unsigned int done = atomicAdd(reinterpret_cast<unsigned int*>(p.ctrl + 1), 1u);
    if (done == gridDim.x - 1) ptx::st_release_gpu_u64(p.ctrl, 0ull);
  }
  ptx::cluster_sync_all();
  if (warp == kMmaWarp) {
    ptx::tcgen05_fence_after();
    ptx::tmem_dealloc_2cta<kTmemCols>(tmem_base);
  }
}

}  // namespace


// ------------------------------------------------------------------------------ host side
namespace {

// fused variant: [ control block 256 B | ready counters, one per 128-row group, padded to 256 B |
// codes [T, K/2] ]
struct FusedWorkspace {
  size_t off_ready, off_codes, bytes;
  int ngroups;
};
FusedWorkspace fused_workspace_layout(int T, int K) {
  FusedWorkspace w{};
  w.ngroups = (T + BM - 1) / BM;
  w.off_ready = 256;
  w.off_codes = w.off_ready + (static_cast<size_t>(w.ngroups) * 4 + 255) / 256 * 256;
  w.bytes = w.off_codes + (static_cast<size_t>(T) * (K / 2) + 255) / 256 * 256;
  return w;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  // resolved through the runtime so that libbaseq.so has no link-time dependency on libcuda
  static std::once_flag once;
  static EncodeTiledFn fn = nullptr;
  std::call_once(once, []() {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) ==
            cudaSuccess && qres == cudaDriverEntryPointSuccess) {
      fn = reinterpret_cast<EncodeTiledFn>(sym);
    }
  });
  return fn;
}

// 2-D row-major tensor map (SWIZZLE_64B boxes), memoised: a tensor map is a pure function of
// (address, extents, row pitch, box, element type), and a serving loop calls the GEMM with the same
// handful of buffers over and over -- the driver's encode call costs about as much as the rest of
// the launch path.  Small direct-mapped table under a mutex (any host thread, any device: device
// pointers of different GPUs are distinct in the unified address space).
struct TmapKey {
  const void* ptr;
  uint64_t d0, d1, pitch;
  uint32_t b0, b1, type, l2;
  bool operator==(const TmapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && pitch == o.pitch && b0 == o.b0 && b1 == o.b1 &&
           type == o.type && l2 == o.l2;
  }
};
struct TmapSlot {
  bool valid = false;
  TmapKey key{};
  CUtensorMap map{};
};
constexpr int kTmapSlots = 256;

cudaError_t tensor_map_2d(const void* ptr, uint64_t d0, uint64_t d1, uint64_t pitch_bytes, uint32_t b0,
                          uint32_t b1, CUtensorMapDataType type, CUtensorMapL2promotion l2,
                          CUtensorMap* out) {
  static std::mutex mu;
  static TmapSlot table[kTmapSlots];
  const TmapKey key{ptr, d0, d1, pitch_bytes, b0, b1, static_cast<uint32_t>(type), static_cast<uint32_t>(l2)};
  uint64_t h = reinterpret_cast<uintptr_t>(ptr) * 0x9E3779B97F4A7C15ull;
  h ^= (d0 * 0xC2B2AE3D27D4EB4Full) ^ (d1 * 0x165667B19E3779F9ull) ^ (pitch_bytes << 7) ^ (b1 << 3) ^ type;
  TmapSlot& slot = table[(h >> 40) % kTmapSlots];
  {
    std::lock_guard<std::mutex> lock(mu);
    if (slot.valid && slot.key == key) {
      *out = slot.map;
      return cudaSuccess;
    }
  }
  EncodeTiledFn encode = get_encode_fn();
  if (encode == nullptr) return cudaErrorNotSupported;
  const cuuint64_t dims[2] = {d0, d1};
  const cuuint64_t strides[1] = {pitch_bytes};
  const cuuint32_t box[2] = {b0, b1};
  const cuuint32_t estr[2] = {1, 1};
  CUtensorMap m{};
  const CUresult r = encode(&m, type, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, l2,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  {
    std::lock_guard<std::mutex> lock(mu);
    slot.valid = true;
    slot.key = key;
    slot.map = m;
  }
  *out = m;
  return cudaSuccess;
}

template <bool FUSED, bool ASYM>
cudaError_t launch_pair(const CUtensorMap& tmap_a, const CUtensorMap& tmap_y, const GemmParams& p,
                        int num_sms, int device, cudaStream_t stream) {
  using C = Cfg<FUSED>;
  static std::atomic<int> attr_smem[kMaxDevices];
  const cudaError_t ea = ensure_dynamic_smem(w4a4_gemm_kernel<FUSED, ASYM>, C::kSmemBytes, device, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int tiles = p.num_m * p.num_n;
  const int slots = num_sms / CG;                        // CTA pairs
  const int groups = tiles < slots ? tiles : slots;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(groups * CG), 1, 1);
  cfg.blockDim = dim3(C::kThreads, 1, 1);
  cfg.dynamicSmemBytes = C::kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CG;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, w4a4_gemm_kernel<FUSED, ASYM>, tmap_a, tmap_y, p);
}

}  // namespace

cudaError_t launch_w4a4_gemm(const GemmLaunch& g) {
  const bool fused = g.x != nullptr;
  if (!fused && g.T <= kDecodeMaxT) return launch_w4a4_decode(g);   // decode shapes: W-streaming kernel
  if (fused && !fused_supported(g.had_block)) return cudaErrorNotSupported;
  const BlobHeader h = blob_header(g.N, g.K);
  const uint8_t* base = static_cast<const uint8_t*>(g.blob);

  // Fused variant: the workspace is [ control block | ready counters | codes ]; the codes go to the
  // caller's codes_dump instead when there is one (same layout, [T, K/2]).
  const FusedWorkspace ws = fused_workspace_layout(g.T, g.K);
  uint8_t* wsb = static_cast<uint8_t*>(g.workspace);
  const uint8_t* codes = fused ? (g.codes_dump != nullptr ? g.codes_dump : wsb + ws.off_codes) : g.codes;

  // A operand: codes [T, K/2] bytes; box = 64 bytes (128 int4) x 128 rows, SWIZZLE_64B;
  // rows beyond T are zero-filled by TMA, so a ragged last M tile needs no special case.
  // Y: bf16 [T, ldy]; box = 32 columns (64 bytes) x 32 rows, SWIZZLE_64B; the store clips
  // rows >= T and columns >= N.
  CUtensorMap tmap_a{}, tmap_y{};
  cudaError_t e = tensor_map_2d(codes, static_cast<uint64_t>(g.K / 2), static_cast<uint64_t>(g.T),
                                static_cast<uint64_t>(g.K / 2), BK / 2, BM, CU_TENSOR_MAP_DATA_TYPE_UINT8,
                                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, &tmap_a);
  if (e != cudaSuccess) return e;
  e = tensor_map_2d(g.y, static_cast<uint64_t>(g.N), static_cast<uint64_t>(g.T),
                    static_cast<uint64_t>(g.ldy) * 2, 32, 32, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, &tmap_y);
  if (e != cudaSuccess) return e;

  GemmParams p{};
  p.header = reinterpret_cast<const uint32_t*>(base);
  p.status = g.status_word;
  p.tiles = base + h.off_tiles;
  p.sw = reinterpret_cast<const float*>(base + h.off_sw);
  p.fb = reinterpret_cast<const float*>(base + h.off_fb);
  p.scales = g.scales;
  p.zeros = g.zeros;
  p.wsum = reinterpret_cast<const float*>(base + h.off_wsum);
  p.y = static_cast<uint16_t*>(g.y);
  p.ldy = g.ldy;
  p.acc_dump = g.acc_dump;
  p.T = g.T;
  p.N = g.N;
  p.K = g.K;
  p.num_m = (g.T + BM * CG - 1) / (BM * CG);
  p.num_n = h.Npad / BN;
  p.num_kb = g.K / BK;
  if (fused) {
    p.x = static_cast<const uint4*>(g.x);
    p.ldxv = g.ldx / 8;
    p.alpha = g.alpha;
    p.gamma = g.gamma;
    p.sa = g.sa;
    p.bvec = g.b;
    p.had_block = g.had_block;
    p.had_scale = g.had_scale;
    p.codes_out = reinterpret_cast<uint32_t*>(const_cast<uint8_t*>(codes));
    p.scales_out = const_cast<float*>(g.scales);
    p.zeros_out = const_cast<float*>(g.zeros);
    p.ctrl = reinterpret_cast<unsigned long long*>(wsb);
    p.ready = reinterpret_cast<unsigned int*>(wsb + ws.off_ready);
    p.ngroups = ws.ngroups;
    if (g.zeros != nullptr) return launch_pair<true, true>(tmap_a, tmap_y, p, g.num_sms, g.device, g.stream);
    return launch_pair<true, false>(tmap_a, tmap_y, p, g.num_sms, g.device, g.stream);
  }
  if (g.zeros != nullptr) return launch_pair<false, true>(tmap_a, tmap_y, p, g.num_sms, g.device, g.stream);
  return launch_pair<false, false>(tmap_a, tmap_y, p, g.num_sms, g.device, g.stream);
}

// ------------------------------------------------------------------------------ fused variant (a10)
size_t fused_workspace_bytes(int T, int N, int K) {
  (void)N;
  return fused_workspace_layout(T, K).bytes;
}

bool fused_supported(int had_block) { return had_block <= 256; }   // a block spans at most one warp

cudaError_t launch_linear_fused(const GemmLaunch& g) {
  if (g.alpha >= kMinFastAlpha) return launch_w4a4_gemm(g);
  // clip ratios below 2^-16: the background quantiser rounds like the fast kernels do; quantise with
  // the clamping kernel into the codes buffer of the call, then run the plain GEMM on it
  const FusedWorkspace ws = fused_workspace_layout(g.T, g.K);
  uint8_t* codes = g.codes_dump != nullptr ? g.codes_dump : static_cast<uint8_t*>(g.workspace) + ws.off_codes;
  QuantLaunch q{};
  q.x = g.x;
  q.ldx = g.ldx;
  q.T = g.T;
  q.K = g.K;
  q.alpha = g.alpha;
  q.gamma = g.gamma;
  q.sa = g.sa;
  q.b = g.b;
  q.had_block = g.had_block;
  q.had_scale = g.had_scale;
  q.codes = codes;
  q.scales = const_cast<float*>(g.scales);
  q.zeros = const_cast<float*>(g.zeros);
  q.asym = g.zeros != nullptr;
  q.stream = g.stream;
  q.num_sms = g.num_sms;
  q.device = g.device;
  const cudaError_t e = launch_quantize_small_alpha(q, true);
  if (e != cudaSuccess) return e;
  GemmLaunch u = g;
  u.x = nullptr;
  u.codes = codes;
  return launch_w4a4_gemm(u);
}

}  // namespace baseq

// NEXT-2: activation quantiser with the online block-128 Hadamard on the tensor cores.
//
// The paper runs its online rotations as matrix products because a butterfly FWHT "does not fully
// leverage tensor core parallelism" (R_qk "128 x 128" as a direct matmul).  The
// bit-exact contract of this library (quant_math.cuh: fp32 butterflies in a fixed order) costs
// seven adds and four shuffles per element and runs at 28 % of the HBM rate on config 5.  This kernel
// computes the same transform as  D = H_128 X^T  with tcgen05.mma kind::f16 (bf16 x bf16 -> fp32):
// +-1 and the bf16 activations are exact operands, only the order of the 128-term fp32 sum is the
// tensor core's own, so the result is NOT bit-reproducible against the butterfly contract -- it is
// accepted iff it lies inside the band DESIGN.md 6.9 states around the exact (fp64) values
// (oracle/: dense_hadamard_u64, dense_mode_check).  Everything after the transform is the contract
// unchanged: u = g h - b, s_t = max((alpha max|u|) / 7, 1e-12), q = clamp(rne(u / s_t), -8, 7).
//
// Shape of the computation (one CTA, inside a cluster of C CTAs that split K):
//   A = H_128 (M = 128 output channels x K = 128 input channels, +-1 as bf16) lives in TENSOR MEMORY
//       for the whole kernel (64 columns) -- no shared-memory traffic for it at all;
//   B = tiles of X: 8 tokens x 128 channels per block, K-major, SWIZZLE_128B, streamed by TMA (one
//       4-D tensor copy brings up to 14 blocks x 8 tokens = 28 KB laid out [half][block][token][64 ch]).
//       H is the same matrix for every block, so the (block, token) rows of a stage are the rows of
//       ONE operand: one N = 112 instruction per K = 16 step serves fourteen blocks.  Measured
//       (a probe of back-to-back instructions): an M = 128 kind::f16 MMA with A in tensor memory
//       takes 130 clk whatever N is (16 ... 224) -- the 4 KB of A are re-read by every instruction
//       at 32 B/clk -- so N must be as large as the data in flight allows (N = 16: 224 instructions
//       and 29 k clk per 8 token rows; N = 112: 16 and 2.1 k).  Every element of X is read ONCE;
//   D = 128 lanes (channels) x 8 columns (tokens) per block.  The CTA's share of a group of 8 token
//       rows (<= 28 blocks = 3584 channels = 224 columns) stays RESIDENT in tensor memory while
//       the epilogue warps read it twice -- pass 1 (u = g h - b written back over h, absmax), pass 2
//       (round, pack) -- and tensor memory holds TWO such groups (64 + 2 x 224 = 512 columns): the
//       MMAs of group g + 1 run under the epilogue of group g.
//   The per-token absmax needs the whole row: the C CTAs of a cluster exchange 8 floats each through
//   distributed shared memory (st.async + a transaction mbarrier).  A dedicated warp does the
//   exchange and the two divisions while the epilogue warps are already in pass 1 of the NEXT group:
//   no epilogue warp ever waits for another one (all hand-overs are mbarriers).
//   The 16 epilogue warps form two teams of 8; a team owns one of the group's two slots (half of the
//   CTA's blocks), so its waits concern that slot's MMAs only.
//   Epilogue thread <-> data: tcgen05.ld.16x256b hands a thread two TMEM lanes (r, r + 8) and four
//   columns; H's rows are permuted so that these two lanes are the channels 2j and 2j + 1 -- the two
//   nibbles of one output byte -- so the saturating pack (cvt.pack.sat.s4.s32) builds whole bytes
//   with no shuffle.  Per-channel operands (g / sqrt(128), b) sit in shared memory (the CTA's slice:
//   <= 28 KB).  Codes leave through a shared-memory tile and row-contiguous bulk stores issued by
//   another otherwise idle warp.
#include <cuda.h>

#include <cstring>
#include <mutex>

#include "kernels.cuh"
#include "ptx.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr int kTok = 8;                  // tokens per group
constexpr int kBlk = 128;                // Hadamard block = MMA M = MMA K extent
constexpr int kSBMax = 14;               // blocks per TMA stage / per D slot (MMA N <= 112); a group = 2 slots
constexpr int kUPSMax = kSBMax / 2;      // epilogue units (two blocks each) of a warp: it owns ONE slot
constexpr int kMaxBlocks = 28;           // per CTA: 28 x 8 = 224 D columns per group
constexpr int kHCols = 64;               // A operand: 128 bf16 per lane
constexpr int kDCols = kMaxBlocks * kTok;               // 224 columns per resident group
constexpr int kXStages = 5;              // smem ring: 2.5 groups in flight
constexpr int kStageBytes = kSBMax * 2 * kTok * 128;    // [2 halves][<= 14 blocks][8 tokens][128 B] = 28 KB
constexpr int kCodePitch = kMaxBlocks * 64 + 16;        // bytes per token row of the codes tile (+16: banks)
constexpr int kCodeTile = kTok * kCodePitch;
constexpr int kMaxCluster = 8;
// Warp roles.  The warp scheduler of a sub-partition favours high warp ids; the single-thread,
// latency-critical roles sit at the top.
constexpr int kEpiWarps = 16;            // warps 0-15 (warp & 3 = TMEM lane quarter)
constexpr int kTmaWarp = 16, kScaleWarp = 17, kStoreWarp = 18, kMmaWarp = 19;
constexpr int kTcThreads = 640;

struct TcBarriers {
  uint64_t xfull[kXStages], xempty[kXStages];
  uint64_t dfull[2][2], dempty[2][2];    // [D buffer][slot]: MMAs done / pass 2 has the slot in registers (8 warps)
  uint64_t pmfull[2];                    // the 16 warps' partial maxima of a group are in wmax
  uint64_t xchg[4];                      // the cluster's partial maxima have arrived (transaction count)
  uint64_t invfull[2];                   // 1 / s_t of a group is in inv
  uint64_t tfull[2], tempty[2];          // codes tile written (16 warps) / read by the bulk stores
  uint32_t tmem_base;
};

struct TcSmem {                          // after the 1024-aligned X ring and the codes tiles
  float4 gb[kMaxBlocks * kBlk / 2];      // per channel pair (2j, 2j + 1): g / sqrt(128) of both, then b of both
  float xmax[4][kMaxCluster][kTok];      // partial row maxima of every CTA of the cluster (see the scale warp)
  float wmax[2][kEpiWarps][kTok];
  float inv[2][kTok];
  TcBarriers bars;
};

constexpr int kTcSmemBytes = 1024 + kXStages * kStageBytes + 2 * kCodeTile + static_cast<int>(sizeof(TcSmem));
static_assert(kTcSmemBytes <= 232448, "shared memory budget");
static_assert(kHCols + 2 * kDCols <= 512, "tensor memory budget");

struct TcParams {
  const float* sa;
  const float* bvec;
  float gamma, alpha, had_scale;
  uint8_t* codes;
  float* scales;
  int T, K, nblk_total;
};

__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
// 4-D tiled tensor copy global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_4d(uint32_t dst_smem, const void* tmap, int32_t c0, int32_t c1,
                                            int32_t c2, int32_t c3, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst_smem), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]; bf16 x bf16 -> fp32
__device__ __forceinline__ void mma_f16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b,
                                           uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
      "}\n"
      ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
// kind::f16 instruction descriptor: D = F32 (1), A = B = BF16 (1), both K-major
__host__ __device__ constexpr uint32_t make_idesc_bf16(uint32_t M, uint32_t N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((N >> 3) << 17) | ((M >> 4) << 24);
}
// this warp's TMEM lanes (r, r + 8) of a 16-lane group x columns (2c, 2c+1, 8+2c, 9+2c):
// registers 0, 1 = lane r, columns 2c, 2c+1; 2, 3 = lane r + 8, same columns; 4..7 = columns 8 + ...
__device__ __forceinline__ void tmem_ld_16x256b_x2(uint32_t taddr, uint32_t (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_st_16x256b_x2(uint32_t taddr, const float (&r)[8]) {
  asm volatile("tcgen05.st.sync.aligned.16x256b.x2.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
               ::"r"(taddr), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7])
               : "memory");
}
__device__ __forceinline__ void tmem_st_32x32b_x16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]),
        "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]),
        "r"(r[15])
      : "memory");
}
// remote (or local) 4-byte store into a cluster CTA's shared memory that completes 4 bytes of a
// transaction on an mbarrier of the SAME CTA: the data is visible to whoever observes the phase flip
__device__ __forceinline__ void st_async_f32(uint32_t cluster_addr, float v, uint32_t cluster_bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];"
               ::"r"(cluster_addr), "r"(__float_as_uint(v)), "r"(cluster_bar)
               : "memory");
}
__device__ __forceinline__ void bulk_store_1d(void* gdst, uint32_t src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               ::"l"(reinterpret_cast<uint64_t>(gdst)), "r"(src_smem), "r"(bytes)
               : "memory");
}

// UPS = sb / 2: units (two blocks each) of an epilogue warp, a compile-time constant so that its
// loops over tensor-memory loads unroll (a run-time trip count cost 2x on config 5)
template <int UPS>
__global__ void __launch_bounds__(kTcThreads, 1)
quantize_had_tc_kernel(const __grid_constant__ CUtensorMap tmap_x, const TcParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t ring0 = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;     // SWIZZLE_128B: 1024-aligned
  uint8_t* ring = smem_raw + (ring0 - ptx::smem_u32(smem_raw));
  uint8_t* code_tile = ring + kXStages * kStageBytes;
  TcSmem* sm = reinterpret_cast<TcSmem*>(code_tile + 2 * kCodeTile);
  TcBarriers* bars = &sm->bars;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank(), csize = cluster_nctarank();
  const int cluster_id = static_cast<int>(blockIdx.x / csize), n_clusters = static_cast<int>(gridDim.x / csize);
  // this CTA's blocks of every row: [blk0, blk0 + nb)
  const int per = (p.nblk_total + static_cast<int>(csize) - 1) / static_cast<int>(csize);
  const int blk0 = static_cast<int>(rank) * per;
  const int nb = max(0, min(per, p.nblk_total - blk0));
  constexpr int sb = 2 * UPS;
  const int nslots = (nb + sb - 1) / sb;                 // 0, 1 or 2
  const uint32_t stage_bytes = static_cast<uint32_t>(sb) * 2u * kTok * 128u;
  const int num_groups = (p.T + kTok - 1) / kTok;
  // this cluster's groups: cluster_id, cluster_id + n_clusters, ...
  const int my_groups = cluster_id < num_groups ? (num_groups - cluster_id + n_clusters - 1) / n_clusters : 0;

  if (warp == kTmaWarp && lane == 0) {
    ptx::prefetch_tensormap(&tmap_x);
    for (int i = 0; i < kXStages; ++i) {
      ptx::mbar_init(ptx::smem_u32(&bars->xfull[i]), 1);
      ptx::mbar_init(ptx::smem_u32(&bars->xempty[i]), 1);
    }
    for (int i = 0; i < 2; ++i) {
      for (int j = 0; j < 2; ++j) {
        ptx::mbar_init(ptx::smem_u32(&bars->dfull[i][j]), 1);
        ptx::mbar_init(ptx::smem_u32(&bars->dempty[i][j]), kEpiWarps / 2);
      }
      ptx::mbar_init(ptx::smem_u32(&bars->pmfull[i]), kEpiWarps);
      ptx::mbar_init(ptx::smem_u32(&bars->invfull[i]), 1);
      ptx::mbar_init(ptx::smem_u32(&bars->tfull[i]), kEpiWarps);
      ptx::mbar_init(ptx::smem_u32(&bars->tempty[i]), 1);
    }
    for (int i = 0; i < 4; ++i) ptx::mbar_init(ptx::smem_u32(&bars->xchg[i]), 1);
    ptx::fence_barrier_init();
  }
  if (warp == kMmaWarp) ptx::tmem_alloc<512>(ptx::smem_u32(&bars->tmem_base));
  ptx::tcgen05_fence_before();
  __syncthreads();
  ptx::tcgen05_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&bars->tmem_base);

  // H_128 into tensor memory: TMEM lane L holds row ch(L) of H, ch(L) = 16 (L / 16) + (rr < 8 ? 2 rr :
  // 2 (rr - 8) + 1) with rr = L % 16, so that the lanes (r, r + 8) a 16x256b load gives one thread
  // are the channels 2j and 2j + 1.  Column j of the operand = the bf16 pair H[ch][2j], H[ch][2j + 1];
  // H[c][k] = (-1)^popcount(c & k) (Sylvester), +1 = 0x3F80, -1 = 0xBF80.
  if (warp < 4) {
    const int L = warp * 32 + lane;
    const int rr = L & 15;
    const uint32_t ch = static_cast<uint32_t>((L & ~15) + (rr < 8 ? 2 * rr : 2 * (rr - 8) + 1));
#pragma unroll
    for (int j0 = 0; j0 < kHCols; j0 += 16) {
      uint32_t w[16];
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const uint32_t k0 = 2u * static_cast<uint32_t>(j0 + j);
        const uint32_t lo = (__popc(ch & k0) & 1) ? 0xBF80u : 0x3F80u;
        const uint32_t hi = (__popc(ch & (k0 + 1u)) & 1) ? 0xBF80u : 0x3F80u;
        w[j] = lo | (hi << 16);
      }
      tmem_st_32x32b_x16(tmem_base + (static_cast<uint32_t>(warp * 32) << 16) + j0, w);
    }
    ptx::tmem_st_wait();
  }
  // per-channel operands of the CTA's slice (parameters of the call, not a predecessor's output)
  for (int i = threadIdx.x; i < nb * kBlk / 2; i += kTcThreads) {
    const int col = blk0 * kBlk + 2 * i;
    const float g0 = p.sa != nullptr ? __ldg(p.sa + col) : p.gamma, g1 = p.sa != nullptr ? __ldg(p.sa + col + 1) : p.gamma;
    sm->gb[i] = make_float4(__fmul_rn(g0, p.had_scale), __fmul_rn(g1, p.had_scale),
                            p.bvec != nullptr ? __ldg(p.bvec + col) : 0.0f, p.bvec != nullptr ? __ldg(p.bvec + col + 1) : 0.0f);
  }
  ptx::tcgen05_fence_before();
  __syncthreads();
  ptx::cluster_sync_all();                   // every CTA's barriers exist before any remote store
  ptx::tcgen05_fence_after();
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  if (warp == kTmaWarp) {
    // ===================================================================== TMA producer
    if (lane == 0 && nb > 0) {
      int xs = 0;
      uint32_t ph = 0;
      for (int gi = 0; gi < my_groups; ++gi) {
        const int g = cluster_id + gi * n_clusters;
        for (int j = 0; j < nslots; ++j) {
          ptx::mbar_wait(ptx::smem_u32(&bars->xempty[xs]), ph ^ 1u);
          const uint32_t bar = ptx::smem_u32(&bars->xfull[xs]);
          ptx::mbar_arrive_expect_tx(bar, stage_bytes);
          // box (64 channels, 8 tokens, sb blocks, 2 halves of a block): rows >= T and blocks >= K / 128
          // are zero-filled; blocks of a neighbouring CTA (last, partial slot) are read and ignored
          tma_load_4d(ring0 + xs * kStageBytes, &tmap_x, 0, g * kTok, blk0 + j * sb, 0, bar);
          if (++xs == kXStages) { xs = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == kMmaWarp) {
    // ===================================================================== MMA issuer
    if (nb > 0) {
      int xs = 0;
      uint32_t ph = 0;
      for (int gi = 0; gi < my_groups; ++gi) {
        const uint32_t buf = static_cast<uint32_t>(gi) & 1u;
        for (int j = 0; j < nslots; ++j) {
          // pass 2 of group gi - 2 has this slot of the D buffer in registers
          if (gi >= 2) ptx::mbar_wait(ptx::smem_u32(&bars->dempty[buf][j]), ((static_cast<uint32_t>(gi) >> 1) - 1u) & 1u);
          ptx::mbar_wait(ptx::smem_u32(&bars->xfull[xs]), ph);
          ptx::tcgen05_fence_after();
          if (ptx::elect_one()) {
            // MMA N: the slot's blocks x 8 tokens, rounded up to the multiple of 16 that M = 128 needs
            // (an odd last block computes 8 spare columns that stay inside this group's D buffer)
            const int blocks = min(sb, nb - j * sb);
            const uint32_t idesc = make_idesc_bf16(kBlk, static_cast<uint32_t>(((blocks * kTok + 15) / 16) * 16));
            const uint64_t desc0 = ptx::make_smem_desc_sw128(ring0 + xs * kStageBytes);
            const uint32_t d = tmem_base + kHCols + buf * kDCols + static_cast<uint32_t>(j * sb * kTok);
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              // half k / 4 of the blocks (sb KB further on), 32 bytes per K = 16 step inside the 128-byte row
              const uint64_t db = desc0 + static_cast<uint64_t>(((k >> 2) * (sb * kTok * 128) + (k & 3) * 32) >> 4);
              mma_f16_ts(d, tmem_base + 8 * k, db, idesc, k != 0 ? 1u : 0u);
            }
            ptx::tcgen05_commit(ptx::smem_u32(&bars->xempty[xs]));
            ptx::tcgen05_commit(ptx::smem_u32(&bars->dfull[buf][j]));
          }
          __syncwarp();
          if (++xs == kXStages) { xs = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == kScaleWarp) {
    // ===================================================================== row maxima -> 1 / s_t
    // lane t < 8: token t of the group.  CTA maximum -> every CTA of the cluster (st.async) -> cluster
    // maximum -> s_t, 1 / s_t (Q4, Q5).  Runs beside pass 1 of the next group.
    // The exchange slots rotate over FOUR groups: a CTA reaches the send of group g + 3 only after
    // its pass 2 of group g + 1, i.e. after every peer's scale warp has sent group g + 1 -- which it
    // does after having read group g.  (With two slots a fast CTA could overwrite a value a slow
    // peer has not read yet.)
    for (int gi = 0; gi < my_groups; ++gi) {
      const uint32_t par = static_cast<uint32_t>(gi) & 1u, phase = (static_cast<uint32_t>(gi) >> 1) & 1u;
      const uint32_t x4 = static_cast<uint32_t>(gi) & 3u, xphase = (static_cast<uint32_t>(gi) >> 2) & 1u;
      const int g = cluster_id + gi * n_clusters;
      ptx::mbar_wait(ptx::smem_u32(&bars->pmfull[par]), phase);
      if (lane == 0) ptx::mbar_arrive_expect_tx(ptx::smem_u32(&bars->xchg[x4]), csize * kTok * 4u);
      if (lane < kTok) {
        float mm = sm->wmax[par][0][lane];
#pragma unroll
        for (int w = 1; w < kEpiWarps; ++w) mm = fmaxf(mm, sm->wmax[par][w][lane]);
        const uint32_t slot = ptx::smem_u32(&sm->xmax[x4][rank][lane]);
        const uint32_t bar = ptx::smem_u32(&bars->xchg[x4]);
        for (uint32_t rk = 0; rk < csize; ++rk)
          st_async_f32(ptx::mapa_cluster(slot, rk), mm, ptx::mapa_cluster(bar, rk));
      }
      ptx::mbar_wait(ptx::smem_u32(&bars->xchg[x4]), xphase);
      if (lane < kTok) {
        float mm = sm->xmax[x4][0][lane];
        for (uint32_t rk = 1; rk < csize; ++rk) mm = fmaxf(mm, sm->xmax[x4][rk][lane]);
        const float st = qm::step_size(p.alpha, mm);
        sm->inv[par][lane] = qm::reciprocal(st);
        const int row = g * kTok + lane;
        if (rank == 0 && row < p.T) p.scales[row] = st;
      }
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&bars->invfull[par]));
    }
  } else if (warp == kStoreWarp) {
    // ===================================================================== codes tile -> global
    if (lane == 0) {
      for (int gi = 0; gi < my_groups; ++gi) {
        const uint32_t par = static_cast<uint32_t>(gi) & 1u, phase = (static_cast<uint32_t>(gi) >> 1) & 1u;
        const int g = cluster_id + gi * n_clusters;
        ptx::mbar_wait(ptx::smem_u32(&bars->tfull[par]), phase);
        if (nb > 0) {
          const uint8_t* tile = code_tile + par * kCodeTile;
          const int rows = min(kTok, p.T - g * kTok);
          for (int t = 0; t < rows; ++t) {
            bulk_store_1d(p.codes + static_cast<size_t>(g * kTok + t) * (p.K / 2) + static_cast<size_t>(blk0) * 64,
                          ptx::smem_u32(tile + t * kCodePitch), static_cast<uint32_t>(nb) * 64u);
          }
        }
        ptx::bulk_commit_group();
        // at most this group's stores may still be reading: the OTHER tile is free again
        ptx::bulk_wait_group_read<1>();
        if (gi >= 1) ptx::mbar_arrive(ptx::smem_u32(&bars->tempty[par ^ 1u]));
      }
      ptx::bulk_wait_group<0>();
    }
  } else if (warp < kEpiWarps) {
    // ===================================================================== epilogue (16 warps)
    // warp e: TMEM lane quarter e & 3 (fixed by the hardware), 16-lane half (e >> 2) & 1, team e >> 3:
    // the team owns slot `team` of every group (blocks team * sb ...), two blocks per load
    const int e = warp;
    const int q = e & 3, hh = (e >> 2) & 1, team = e >> 3;
    const int lane_base = 32 * q + 16 * hh;              // this warp's 16 TMEM lanes
    const int r = lane >> 2, c = lane & 3;
    const int pair = lane_base / 2 + r;                  // channel pair (2 pair, 2 pair + 1) of the block =
                                                         // TMEM lanes lane_base + r, + 8 = byte column
    const uint32_t taddr0 = tmem_base + (static_cast<uint32_t>(lane_base) << 16) + kHCols;
    // A load covers two blocks (lb, lb + 1) x this thread's tokens 2c, 2c + 1 x its two channels:
    // registers 0, 1 = (even channel, token 2c / 2c+1, block lb), 2, 3 = odd channel, 4..7 = block lb + 1.
    const int bl0 = team * sb;
    const int my_blocks = max(0, min(sb, nb - bl0));     // blocks of this team's slot
    const int nunits = (my_blocks + 1) / 2;              // <= UPS

    // ---- pass 1 of group gi: u = g h - b written back over h, partial absmax of tokens 2c, 2c + 1
    auto pass1 = [&](int gi) {
      const uint32_t buf = static_cast<uint32_t>(gi) & 1u, phase = (static_cast<uint32_t>(gi) >> 1) & 1u;
      const uint32_t tbuf = taddr0 + buf * kDCols + static_cast<uint32_t>(bl0 * kTok);
      float m0 = 0.0f, m1 = 0.0f;
      if (nunits > 0) {
        ptx::mbar_wait(ptx::smem_u32(&bars->dfull[buf][team]), phase);       // this slot's MMAs are complete
        ptx::tcgen05_fence_after();
        uint32_t va[8], vb[8];
        float4 ga[2], gb[2];
        auto load = [&](int u, uint32_t (&v)[8], float4 (&gg)[2]) {
          tmem_ld_16x256b_x2(tbuf + static_cast<uint32_t>(2 * u * kTok), v);
#pragma unroll
          for (int i = 0; i < 2; ++i) gg[i] = sm->gb[min(bl0 + 2 * u + i, kMaxBlocks - 1) * (kBlk / 2) + pair];
        };
        auto math = [&](int u, const uint32_t (&v)[8], const float4 (&gg)[2]) {
          float uu[8];
          uu[0] = qm::affine(gg[0].x, __uint_as_float(v[0]), gg[0].z);
          uu[1] = qm::affine(gg[0].x, __uint_as_float(v[1]), gg[0].z);
          uu[2] = qm::affine(gg[0].y, __uint_as_float(v[2]), gg[0].w);
          uu[3] = qm::affine(gg[0].y, __uint_as_float(v[3]), gg[0].w);
          uu[4] = qm::affine(gg[1].x, __uint_as_float(v[4]), gg[1].z);
          uu[5] = qm::affine(gg[1].x, __uint_as_float(v[5]), gg[1].z);
          uu[6] = qm::affine(gg[1].y, __uint_as_float(v[6]), gg[1].w);
          uu[7] = qm::affine(gg[1].y, __uint_as_float(v[7]), gg[1].w);
          m0 = qm::max3_abs(m0, uu[0], uu[2]);
          m1 = qm::max3_abs(m1, uu[1], uu[3]);
          if (2 * u + 1 < my_blocks) {                   // an odd last block: the spare columns hold no data
            m0 = qm::max3_abs(m0, uu[4], uu[6]);
            m1 = qm::max3_abs(m1, uu[5], uu[7]);
          }
          tmem_st_16x256b_x2(tbuf + static_cast<uint32_t>(2 * u * kTok), uu);
        };
        load(0, va, ga);
#pragma unroll
        for (int u = 0; u < UPS; u += 2) {
          ptx::tmem_ld_wait();
          if (u + 1 < UPS) load(u + 1, vb, gb);
          if (u < nunits) math(u, va, ga);
          if (u + 1 < UPS) {
            ptx::tmem_ld_wait();
            if (u + 2 < UPS) load(u + 2, va, ga);
            if (u + 1 < nunits) math(u + 1, vb, gb);
          }
        }
        ptx::tmem_st_wait();
      }
      // over r (lane bits 2..4) inside the warp; the 16 warps meet in shared memory
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) {
        m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, o));
        m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, o));
      }
      if (r == 0) {
        sm->wmax[buf][e][2 * c] = m0;
        sm->wmax[buf][e][2 * c + 1] = m1;
      }
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&bars->pmfull[buf]));
    };

    // ---- pass 2 of group gi: u back from tensor memory, round, pack whole bytes, stage
    auto pass2 = [&](int gi) {
      const uint32_t buf = static_cast<uint32_t>(gi) & 1u, phase = (static_cast<uint32_t>(gi) >> 1) & 1u;
      const uint32_t tbuf = taddr0 + buf * kDCols + static_cast<uint32_t>(bl0 * kTok);
      uint8_t* tile = code_tile + buf * kCodeTile + bl0 * 64 + pair;
      ptx::mbar_wait(ptx::smem_u32(&bars->invfull[buf]), phase);
      const float inv0 = sm->inv[buf][2 * c], inv1 = sm->inv[buf][2 * c + 1];
      // the bulk stores of group gi - 2 have read this tile
      if (gi >= 2) ptx::mbar_wait(ptx::smem_u32(&bars->tempty[buf]), ((static_cast<uint32_t>(gi) >> 1) - 1u) & 1u);
      auto math = [&](int u, const uint32_t (&vv)[8]) {
        // byte = (q[2j + 1] & 15) << 4 | (q[2j] & 15), both clamped to [-8, 7] by the pack
        const uint32_t b0 = qm::pack2_sat(qm::code_int(__uint_as_float(vv[2]), inv0), qm::code_int(__uint_as_float(vv[0]), inv0), 0u);
        const uint32_t b1 = qm::pack2_sat(qm::code_int(__uint_as_float(vv[3]), inv1), qm::code_int(__uint_as_float(vv[1]), inv1), 0u);
        uint8_t* dst = tile + 2 * u * 64;
        dst[(2 * c) * kCodePitch] = static_cast<uint8_t>(b0);
        dst[(2 * c + 1) * kCodePitch] = static_cast<uint8_t>(b1);
        if (2 * u + 1 < my_blocks) {
          const uint32_t b2 = qm::pack2_sat(qm::code_int(__uint_as_float(vv[6]), inv0), qm::code_int(__uint_as_float(vv[4]), inv0), 0u);
          const uint32_t b3 = qm::pack2_sat(qm::code_int(__uint_as_float(vv[7]), inv1), qm::code_int(__uint_as_float(vv[5]), inv1), 0u);
          dst[64 + (2 * c) * kCodePitch] = static_cast<uint8_t>(b2);
          dst[64 + (2 * c + 1) * kCodePitch] = static_cast<uint8_t>(b3);
        }
      };
      // the warp's units in two chunks of registers; once the last loads have completed the slot is
      // released to the MMAs of group gi + 2 (they run under the rest of the rounding work)
      constexpr int kHalf = (UPS + 1) / 2;
      uint32_t va[kHalf][8], vb[UPS - kHalf + 1][8];
      if (nunits > 0) {
#pragma unroll
        for (int i = 0; i < kHalf; ++i) tmem_ld_16x256b_x2(tbuf + static_cast<uint32_t>(2 * i * kTok), va[i]);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int i = kHalf; i < UPS; ++i) tmem_ld_16x256b_x2(tbuf + static_cast<uint32_t>(2 * i * kTok), vb[i - kHalf]);
#pragma unroll
        for (int i = 0; i < kHalf; ++i)
          if (i < nunits) math(i, va[i]);
        ptx::tmem_ld_wait();
      }
      ptx::tcgen05_fence_before();
      __syncwarp();
      if (lane == 0 && team < nslots) ptx::mbar_arrive(ptx::smem_u32(&bars->dempty[buf][team]));
#pragma unroll
      for (int i = kHalf; i < UPS; ++i)
        if (i < nunits) math(i, vb[i - kHalf]);
      ptx::fence_proxy_async_smem();                    // this lane's tile bytes -> the bulk-copy engine
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&bars->tfull[buf]));
    };

    // software pipeline over the groups: pass 1 of group gi + 1 runs while the scale warp exchanges
    // the maxima of group gi
    if (my_groups > 0) pass1(0);
    for (int gi = 0; gi < my_groups; ++gi) {
      if (gi + 1 < my_groups) pass1(gi + 1);
      pass2(gi);
    }
  }

  // ---- teardown: no CTA leaves while a peer may still store into its shared memory
  ptx::tcgen05_fence_before();
  __syncthreads();
  ptx::cluster_sync_all();
  if (warp == kMmaWarp) {
    ptx::tcgen05_fence_after();
    ptx::tmem_dealloc<512>(tmem_base);
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn tc_encode_fn() {
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

template <int UPS>
cudaError_t launch_ups(const QuantLaunch& q, const CUtensorMap& tmap, int nblk, int C) {
  static std::atomic<int> attr_smem[kMaxDevices];
  const cudaError_t ea = ensure_dynamic_smem(quantize_had_tc_kernel<UPS>, kTcSmemBytes, q.device, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int groups = (q.T + kTok - 1) / kTok;

  TcParams p{};
  p.sa = q.sa;
  p.bvec = q.b;
  p.gamma = q.gamma;
  p.alpha = q.alpha;
  p.had_scale = q.had_scale;
  p.codes = q.codes;
  p.scales = q.scales;
  p.T = q.T;
  p.K = q.K;
  p.nblk_total = nblk;

  cudaLaunchConfig_t cfg{};
  cfg.blockDim = dim3(kTcThreads, 1, 1);
  cfg.dynamicSmemBytes = kTcSmemBytes;
  cfg.stream = q.stream;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = static_cast<unsigned>(C);
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  // Persistent clusters, every one of them resident at once: the groups are dealt round-robin, so a
  // cluster that had to wait for a free GPC slot would start a whole wave late.  How many clusters
  // of C CTAs with this much shared memory fit depends on the GPC layout of the part (15 of 8 on a
  // B200, not 148 / 8 = 18): ask once per device and cluster size.
  static std::atomic<int> max_clusters[kMaxDevices][4];   // per UPS instantiation
  const int ci = C == 1 ? 0 : C == 2 ? 1 : C == 4 ? 2 : 3;
  int fit = max_clusters[q.device][ci].load(std::memory_order_acquire);
  if (fit == 0) {
    cfg.gridDim = dim3(static_cast<unsigned>(q.num_sms / C * C), 1, 1);
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, quantize_had_tc_kernel<UPS>, &cfg) != cudaSuccess || n < 1) {
      (void)cudaGetLastError();
      n = q.num_sms / C > 2 ? q.num_sms / C - 2 : 1;
    }
    fit = n;
    max_clusters[q.device][ci].store(fit, std::memory_order_release);
  }
  const int clusters = fit < groups ? fit : groups;
  cfg.gridDim = dim3(static_cast<unsigned>(clusters * C), 1, 1);
  return cudaLaunchKernelEx(&cfg, quantize_had_tc_kernel<UPS>, tmap, p);
}

}  // namespace

bool quantize_tc_supported(int K, int had_block) {
  return had_block == kBlk && K % kBlk == 0 && K / kBlk <= kMaxBlocks * kMaxCluster;
}

cudaError_t launch_quantize_tc(const QuantLaunch& q) {
  if (!quantize_tc_supported(q.K, q.had_block) || q.asym) return cudaErrorNotSupported;
  EncodeTiledFn encode = tc_encode_fn();
  if (encode == nullptr) return cudaErrorNotSupported;
  const int nblk = q.K / kBlk;
  int C = 1;
  while ((nblk + C - 1) / C > kMaxBlocks) C *= 2;
  // a CTA's blocks (at most ceil(nblk / C)) in two slots of sb blocks, sb even: both epilogue teams
  // get the same amount of work
  const int per = (nblk + C - 1) / C;
  const int sb = (((per + 1) / 2) + 1) / 2 * 2;
  // X as a 4-D tensor [2 halves of a block][K / 128 blocks][T tokens][64 channels]: a box lands in
  // shared memory as [half][block][8 tokens x 128 bytes] -- for each half the 64 (block, token) rows
  // of one K-major SWIZZLE_128B operand of tcgen05.mma
  CUtensorMap tmap{};
  const cuuint64_t dims[4] = {64, static_cast<cuuint64_t>(q.T), static_cast<cuuint64_t>(q.K / kBlk), 2};
  const cuuint64_t strides[3] = {static_cast<cuuint64_t>(q.ldx) * 2, 256, 128};
  const cuuint32_t box[4] = {64, kTok, static_cast<cuuint32_t>(sb), 2};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUresult r = encode(&tmap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(q.x), dims, strides,
                            box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;

  switch (sb / 2) {
    case 1: return launch_ups<1>(q, tmap, nblk, C);
    case 2: return launch_ups<2>(q, tmap, nblk, C);
    case 3: return launch_ups<3>(q, tmap, nblk, C);
    case 4: return launch_ups<4>(q, tmap, nblk, C);
    case 5: return launch_ups<5>(q, tmap, nblk, C);
    case 6: return launch_ups<6>(q, tmap, nblk, C);
    case 7: return launch_ups<7>(q, tmap, nblk, C);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace baseq

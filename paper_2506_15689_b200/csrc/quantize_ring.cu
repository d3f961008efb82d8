// Activation quantiser for long rows (K >= 4096, and every K of the asymmetric variant): the
// arithmetic contract of quant_math.cuh (Q0-Q7), fed by a bulk-TMA ring.
//
// One producer lane streams whole token rows (row-contiguous cp.async.bulk copies, completion on an
// mbarrier) into a ring of shared-memory stages that fills whatever the 227 KB allow -- 150-200 KB
// of loads in flight per SM, no registers involved -- and 16 consumer warps read each stage once
// from shared memory, conflict-free.
//
// Per stage: pass 1 (u = g h - b, absmax) -> the stage is released to the producer -> reduction
// (partials in smem, one designated thread per row finishes the max and computes s_t and 1 / s_t
// once) -> pass 2 from registers (round, clamp, pack, store).
//
// Instruction budget (r2): with the mixed-precision fma (FHFMA.BF16 consumes the bf16 activations in
// place), three-input max (FMNMX3), fma-with-magic rounding and the saturating nibble pack the two
// passes cost 4 issue slots per element (FHFMA, 1/2 FMNMX3, FFMA, IADD, 1/2 I2IP) instead of the ~9
// of r1 (unpack, FFMA, FMNMX, FFMA, IADD, I2IP plus address arithmetic).
#include <cstring>

#include "kernels.cuh"
#include "ptx.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr int kConsumers = 512;                 // threads per row (row-wide kernel)
constexpr int kConsumerWarps = kConsumers / 32;
constexpr int kRingThreads = kConsumers + 32;   // + the producer warp
constexpr int kMaxStages = 8;
constexpr int kRingSmemBudget = 220 * 1024;
constexpr float kNegHuge = -3.402823466e38f;

// How the scale factor g of u = g h - b reaches the kernel:
//   kGBf16  scalar s^a that is itself a bf16 value (1.0 in four of the five BASELINE configs): the
//           mixed-precision fma consumes the bf16 activations in place (quant_math.cuh), no unpack
//   kGF32   any other scalar s^a: unpack + FFMA
//   kGVec   per-channel s^a vector (Eq. 15; NEXT-4): the thread's values live in private
//           slots of shared memory behind the ring (V <= 4) or come through L1 for every row
enum : int { kGBf16 = 0, kGF32 = 1, kGVec = 2 };

struct RingParams {
  const uint8_t* x;        // bf16 rows
  int64_t row_bytes_stride;
  int T, K, nvec;
  float alpha, gamma;
  uint32_t gamma_bf16;     // the scalar s^a as a bf16 bit pattern (kGBf16 only)
  const float* bvec;
  const float* sa;         // per-channel s^a (kGVec), else NULL
  int had_block;
  float had_scale;
  uint32_t* codes;         // NULL: scales only
  float* scales;
  float* zeros;            // asymmetric variant only
  int stages;
  int stage_bytes;
};

__device__ __forceinline__ void named_barrier_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

// launch with programmatic stream serialisation allowed (see ptx::griddep_wait)
template <typename Kern>
cudaError_t launch_pdl(Kern kern, int blocks, int threads, int smem, cudaStream_t stream, const RingParams& p) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(blocks), 1, 1);
  cfg.blockDim = dim3(static_cast<unsigned>(threads), 1, 1);
  cfg.dynamicSmemBytes = static_cast<size_t>(smem);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, p);
}

// ------------------------------------------------------------------ shared pieces
// The producer: one lane streams the RL rows of every stage this CTA owns.
template <int RL>
__device__ __forceinline__ void produce_rows(const RingParams& p, uint8_t* ring, uint64_t* full,
                                             uint64_t* empty, int num_groups) {
  int s = 0;
  uint32_t ph = 0;
  const uint32_t row_bytes = static_cast<uint32_t>(p.K) * 2u;
  for (int g = blockIdx.x; g < num_groups; g += gridDim.x) {
    ptx::mbar_wait(ptx::smem_u32(&empty[s]), ph ^ 1u);
    const int row0 = g * RL;
    const int rows = (p.T - row0) < RL ? (p.T - row0) : RL;
    const uint32_t bar = ptx::smem_u32(&full[s]);
    ptx::mbar_arrive_expect_tx(bar, row_bytes * rows);
    const uint32_t dst = ptx::smem_u32(ring) + s * p.stage_bytes;
    for (int j = 0; j < rows; ++j) {
      ptx::bulk_load_1d(dst + j * row_bytes, p.x + static_cast<int64_t>(row0 + j) * p.row_bytes_stride,
                        row_bytes, bar);
    }
    if (++s == p.stages) { s = 0; ph ^= 1u; }
  }
}

// Q0-Q2 for one 16-byte vector: u = g h - b.  `g8` is read for kGVec only.
template <bool HAD, int GMODE>
__device__ __forceinline__ void vector_u(const RingParams& p, const uint4& xv, const float (&b8)[8],
                                         const float (&g8)[8], int lane, float (&u)[8]) {
  if (!HAD && GMODE == kGBf16) {
    float nb[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) nb[e] = -b8[e];          // folds into the fma's operand modifier
    qm::affine8_bf16(xv, p.gamma_bf16, nb, u);
  } else {
    float f[8];
    qm::unpack8(xv, f);
    if (HAD) qm::hadamard8(f, p.had_block, p.had_scale, lane);
#pragma unroll
    for (int e = 0; e < 8; ++e) u[e] = qm::affine(GMODE == kGVec ? g8[e] : p.gamma, f[e], b8[e]);
  }
}

__device__ __forceinline__ void load8_shared(const float4* s, float (&v)[8]) {
  const float4 a = s[0], b = s[1];
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
  v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}

// ------------------------------------------------------------------ row-wide kernel
// 512 threads = one row wide, thread r owns the 16-byte vectors r, r + 512, ... of all RL rows of a
// stage, so its slice of b stays in registers for every row (V <= 4).
template <int V, int RL, bool HAD, bool RAGGED, bool ASYM, int GMODE>
__global__ void __launch_bounds__(kRingThreads, 1) quantize_ring_kernel(const RingParams p) {
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ uint64_t full[kMaxStages], empty[kMaxStages];
  __shared__ float s_part[2][RL][kConsumerWarps];
  __shared__ float s_part2[ASYM ? 2 : 1][RL][kConsumerWarps];   // asymmetric: max(-u) = -min(u)
  __shared__ float2 s_scale[2][RL];
  __shared__ float s_zero[2][RL];

  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int num_groups = (p.T + RL - 1) / RL;     // one group = RL rows = one stage

  if (tid == 0) {
    for (int s = 0; s < p.stages; ++s) {
      ptx::mbar_init(ptx::smem_u32(&full[s]), 1);
      ptx::mbar_init(ptx::smem_u32(&empty[s]), kConsumerWarps);
    }
    ptx::fence_barrier_init();
  }
  __syncthreads();
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  if (warp == kConsumerWarps) {
    if (lane == 0) produce_rows<RL>(p, ring, full, empty, num_groups);
    return;
  }

  // ======================================================================= consumers
  const int r = tid;                               // vector r + i * 512 of every row
  constexpr bool kInRegs = V <= 4;                 // b in registers, s^a in private smem slots
  float bb[kInRegs ? V : 1][8];
  float4* sa_s = reinterpret_cast<float4*>(ring + static_cast<size_t>(p.stages) * p.stage_bytes);
  if (kInRegs) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const int idx = r + i * kConsumers;
      const bool ok = !RAGGED || idx < p.nvec;
      if (p.bvec != nullptr && ok) {
        qm::load8_pinned(p.bvec + 8 * idx, bb[kInRegs ? i : 0]);
      } else {
#pragma unroll
        for (int e = 0; e < 8; ++e) bb[kInRegs ? i : 0][e] = 0.0f;
      }
      if (GMODE == kGVec) {
        const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
        sa_s[2 * idx] = ok ? __ldg(reinterpret_cast<const float4*>(p.sa) + 2 * idx) : z4;
        sa_s[2 * idx + 1] = ok ? __ldg(reinterpret_cast<const float4*>(p.sa) + 2 * idx + 1) : z4;
      }
    }
  }

  int s = 0, parity = 0;
  uint32_t ph = 0;
  for (int g = blockIdx.x; g < num_groups; g += gridDim.x, parity ^= 1) {
    const int row0 = g * RL;
    ptx::mbar_wait(ptx::smem_u32(&full[s]), ph);
    const uint8_t* stage = ring + s * p.stage_bytes;

    // ---- pass 1: smem -> registers, Hadamard, u = g*h - b, absmax
    float u[RL][V][8];
    float m[RL];
    float m2[RL];                                      // asymmetric only: running max of -u
#pragma unroll
    for (int j = 0; j < RL; ++j) {
      m[j] = ASYM ? kNegHuge : 0.0f;
      m2[j] = kNegHuge;
    }
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const int idx = r + i * kConsumers;
      const bool ok = !RAGGED || idx < p.nvec;
      float b8[8], g8[8];
      if (kInRegs) {
#pragma unroll
        for (int e = 0; e < 8; ++e) b8[e] = bb[kInRegs ? i : 0][e];
        if (GMODE == kGVec) load8_shared(sa_s + 2 * idx, g8);
      } else {
        qm::load_gb(GMODE == kGVec ? p.sa : nullptr, p.bvec, p.gamma, idx, ok, g8, b8);
      }
#pragma unroll
      for (int j = 0; j < RL; ++j) {
        uint4 xv = make_uint4(0, 0, 0, 0);
        if (ok) xv = *reinterpret_cast<const uint4*>(stage + static_cast<size_t>(j) * p.K * 2 + idx * 16);
        vector_u<HAD, GMODE>(p, xv, b8, g8, lane, u[j][i]);
        if (ASYM) {
          if (ok) qm::maxmin8(m[j], m2[j], u[j][i]);
        } else {
          m[j] = qm::absmax8(m[j], u[j][i]);
        }
      }
    }
    // every lane's shared-memory reads have returned (their values fed the max): release the stage
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&empty[s]));
    if (++s == p.stages) { s = 0; ph ^= 1u; }

    // ---- block reduction: warp shuffle -> partials -> one warp per row finishes.
    // RL row maxima are reduced together: each xor step that halves the live values costs one
    // shuffle per surviving value (6 shuffles for 4 rows instead of 20).
    if (ASYM) {
#pragma unroll
      for (int j = 0; j < RL; ++j) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          m[j] = fmaxf(m[j], __shfl_xor_sync(0xffffffffu, m[j], o));
          m2[j] = fmaxf(m2[j], __shfl_xor_sync(0xffffffffu, m2[j], o));
        }
        if (lane == 0) {
          s_part[parity][j][warp] = m[j];
          s_part2[ASYM ? parity : 0][j][warp] = m2[j];
        }
      }
    } else if (RL == 4) {
      const bool up16 = (lane & 16) != 0, up8 = (lane & 8) != 0;
      float s0 = up16 ? m[0] : m[2], s1 = up16 ? m[1] : m[3];      // what the partner keeps
      float k0 = up16 ? m[2] : m[0], k1 = up16 ? m[3] : m[1];
      k0 = fmaxf(k0, __shfl_xor_sync(0xffffffffu, s0, 16));
      k1 = fmaxf(k1, __shfl_xor_sync(0xffffffffu, s1, 16));
      const float snd = up8 ? k0 : k1;
      float c = up8 ? k1 : k0;
      c = fmaxf(c, __shfl_xor_sync(0xffffffffu, snd, 8));
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) c = fmaxf(c, __shfl_xor_sync(0xffffffffu, c, o));
      // lane 0, 8, 16, 24 hold rows 0, 1, 2, 3
      if ((lane & 7) == 0) s_part[parity][lane >> 3][warp] = c;
    } else if (RL == 2) {
      const bool up16 = (lane & 16) != 0;
      const float snd = up16 ? m[0] : m[1 % RL];
      float c = up16 ? m[1 % RL] : m[0];
      c = fmaxf(c, __shfl_xor_sync(0xffffffffu, snd, 16));
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) c = fmaxf(c, __shfl_xor_sync(0xffffffffu, c, o));
      if ((lane & 15) == 0) s_part[parity][(lane >> 4) % RL][warp] = c;
    } else {
#pragma unroll
      for (int j = 0; j < RL; ++j) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m[j] = fmaxf(m[j], __shfl_xor_sync(0xffffffffu, m[j], o));
        if (lane == 0) s_part[parity][j][warp] = m[j];
      }
    }
    named_barrier_sync(1, kConsumers);
    if (warp < RL) {
      float mm = lane < kConsumerWarps ? s_part[parity][warp][lane] : (ASYM ? kNegHuge : 0.0f);
      float mm2 = (ASYM && lane < kConsumerWarps) ? s_part2[ASYM ? parity : 0][warp][lane] : kNegHuge;
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) {
        mm = fmaxf(mm, __shfl_xor_sync(0xffffffffu, mm, o));
        if (ASYM) mm2 = fmaxf(mm2, __shfl_xor_sync(0xffffffffu, mm2, o));
      }
      if (lane == 0) {
        const float st = ASYM ? qm::step_size_asym(p.alpha, -mm2, mm) : qm::step_size(p.alpha, mm);
        s_scale[parity][warp] = make_float2(st, qm::reciprocal(st));
        if (ASYM) s_zero[parity][warp] = qm::lower_bound_asym(p.alpha, -mm2);
        if (row0 + warp < p.T) {
          p.scales[row0 + warp] = st;
          if (ASYM) p.zeros[row0 + warp] = qm::lower_bound_asym(p.alpha, -mm2);
        }
      }
    }
    named_barrier_sync(2, kConsumers);

    // ---- pass 2: round, clamp, pack, store
    if (p.codes != nullptr) {
#pragma unroll
      for (int j = 0; j < RL; ++j) {
        const float inv = s_scale[parity][j].y;
        if (row0 + j < p.T) {
          uint32_t* crow = p.codes + static_cast<int64_t>(row0 + j) * p.nvec;
#pragma unroll
          for (int i = 0; i < V; ++i) {
            const int idx = r + i * kConsumers;
            const uint32_t w = ASYM ? qm::quantize_pack8_asym(u[j][i], s_zero[parity][j], inv)
                                    : qm::quantize_pack8(u[j][i], inv);
            if (!RAGGED || idx < p.nvec) crow[idx] = w;
          }
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Split variant for short rows (K = 1024 * V, V <= 4; every K = 4096 shape of the benchmark): the
// 16 consumer warps form four independent groups of 128 threads, and row j of a 4-row stage
// belongs to group j (thread r' of the group owns vectors r', r' + 128, ...).  Same work per
// thread and stage as the row-wide layout (32 elements, one reduction, two barriers), but the
// barriers are group-local, so while one group waits for its row's s_t (shuffles, barrier, two IEEE
// divisions, barrier) the other three keep the issue slots busy.
constexpr int kGroupThreads = 128;
constexpr int kGroupWarps = kGroupThreads / 32;

// G groups of 128 threads (+ the producer warp).  G = 4: one CTA per SM with the whole shared memory
// as its ring.  G = 2: a CTA of 288 threads and half the shared memory, so that the NEXT kernel's CTA
// is already resident (prologue done, parked in griddepcontrol.wait) while this one streams -- the
// hand-over between two launches then costs one DRAM round trip instead of a CTA launch on top.
template <int V, int G, bool ASYM, int GMODE>
__global__ void __launch_bounds__(G * kGroupThreads + 32, G == 4 ? 1 : 2) quantize_ring_split_kernel(const RingParams p) {
  constexpr int RL = G;
  constexpr int kWarps = G * kGroupWarps;          // consumer warps
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ uint64_t full[kMaxStages], empty[kMaxStages];
  __shared__ float s_part[2][RL][kGroupWarps];
  __shared__ float s_part2[ASYM ? 2 : 1][RL][kGroupWarps];   // asymmetric: max(-u) = -min(u)
  __shared__ float2 s_scale[2][RL];
  __shared__ float s_zero[2][RL];

  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int num_groups = (p.T + RL - 1) / RL;     // one stage = RL rows

  if (tid == 0) {
    for (int s = 0; s < p.stages; ++s) {
      ptx::mbar_init(ptx::smem_u32(&full[s]), 1);
      ptx::mbar_init(ptx::smem_u32(&empty[s]), kWarps);
    }
    ptx::fence_barrier_init();
  }
  __syncthreads();
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  if (warp == kWarps) {
    if (lane == 0) produce_rows<RL>(p, ring, full, empty, num_groups);
    return;
  }

  const int grp = warp / kGroupWarps;              // this thread's row inside every stage
  const int gw = warp % kGroupWarps;
  const int r = tid & (kGroupThreads - 1);         // vectors r, r + 128, ... of that row
  float bb[V][8];
#pragma unroll
  for (int i = 0; i < V; ++i) {
    if (p.bvec != nullptr) {
      qm::load8_pinned(p.bvec + 8 * (r + i * kGroupThreads), bb[i]);
    } else {
#pragma unroll
      for (int e = 0; e < 8; ++e) bb[i][e] = 0.0f;
    }
  }

  // per-channel s^a (NEXT-4): u, the bias and s^a together do not fit the register file (ptxas
  // spilled), so this thread's V x 8 values of s^a live in shared memory behind the ring, written
  // and read by this thread only (every group writes the same values: a benign duplicate)
  float4* sa_s = reinterpret_cast<float4*>(ring + static_cast<size_t>(p.stages) * p.stage_bytes);
  if (GMODE == kGVec) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const int idx = r + i * kGroupThreads;
      sa_s[2 * idx] = __ldg(reinterpret_cast<const float4*>(p.sa) + 2 * idx);
      sa_s[2 * idx + 1] = __ldg(reinterpret_cast<const float4*>(p.sa) + 2 * idx + 1);
    }
  }

  int s = 0, parity = 0;
  uint32_t ph = 0;
  for (int g = blockIdx.x; g < num_groups; g += gridDim.x, parity ^= 1) {
    const int row = g * RL + grp;
    const bool row_ok = row < p.T;
    ptx::mbar_wait(ptx::smem_u32(&full[s]), ph);
    const uint8_t* srow = ring + s * p.stage_bytes + static_cast<size_t>(grp) * p.K * 2;

    float u[V][8];
    float m = ASYM ? kNegHuge : 0.0f;
    float m2 = kNegHuge;                            // asymmetric only: running max of -u
    if (row_ok) {                                   // rows past T were not loaded
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const int idx = r + i * kGroupThreads;
        const uint4 xv = *reinterpret_cast<const uint4*>(srow + idx * 16);
        float g8[8];
        if (GMODE == kGVec) load8_shared(sa_s + 2 * idx, g8);
        vector_u<false, GMODE>(p, xv, bb[i], g8, lane, u[i]);
        if (ASYM) qm::maxmin8(m, m2, u[i]);
        else m = qm::absmax8(m, u[i]);
      }
    }
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&empty[s]));
    if (++s == p.stages) { s = 0; ph ^= 1u; }
    if (!row_ok) continue;                          // group-uniform: the whole group skips

#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
      if (ASYM) m2 = fmaxf(m2, __shfl_xor_sync(0xffffffffu, m2, o));
    }
    if (lane == 0) {
      s_part[parity][grp][gw] = m;
      if (ASYM) s_part2[ASYM ? parity : 0][grp][gw] = m2;
    }
    named_barrier_sync(1 + grp, kGroupThreads);
    if (gw == 0 && lane == 0) {
      float mm = s_part[parity][grp][0];
#pragma unroll
      for (int w = 1; w < kGroupWarps; ++w) mm = fmaxf(mm, s_part[parity][grp][w]);
      float mm2 = kNegHuge;
      if (ASYM) {
#pragma unroll
        for (int w = 0; w < kGroupWarps; ++w) mm2 = fmaxf(mm2, s_part2[ASYM ? parity : 0][grp][w]);
      }
      const float st = ASYM ? qm::step_size_asym(p.alpha, -mm2, mm) : qm::step_size(p.alpha, mm);
      s_scale[parity][grp] = make_float2(st, qm::reciprocal(st));
      p.scales[row] = st;
      if (ASYM) {
        const float zt = qm::lower_bound_asym(p.alpha, -mm2);
        s_zero[parity][grp] = zt;
        p.zeros[row] = zt;
      }
    }
    named_barrier_sync(5 + grp, kGroupThreads);

    if (p.codes != nullptr) {
      const float inv = s_scale[parity][grp].y;
      uint32_t* crow = p.codes + static_cast<int64_t>(row) * p.nvec;
#pragma unroll
      for (int i = 0; i < V; ++i) {
        crow[r + i * kGroupThreads] = ASYM ? qm::quantize_pack8_asym(u[i], s_zero[parity][grp], inv)
                                           : qm::quantize_pack8(u[i], inv);
      }
    }
  }
}

// ------------------------------------------------------------------ host side
RingParams make_params(const QuantLaunch& q, bool write_codes) {
  RingParams p{};
  p.x = static_cast<const uint8_t*>(q.x);
  p.row_bytes_stride = q.ldx * 2;
  p.T = q.T;
  p.K = q.K;
  p.nvec = q.K / 8;
  p.alpha = q.alpha;
  p.gamma = q.gamma;
  uint32_t gbits;
  static_assert(sizeof(gbits) == sizeof(q.gamma), "float bits");
  std::memcpy(&gbits, &q.gamma, sizeof gbits);
  p.gamma_bf16 = gbits >> 16;
  p.bvec = q.b;
  p.sa = q.sa;
  p.had_block = q.had_block;
  p.had_scale = q.had_scale;
  p.codes = write_codes ? reinterpret_cast<uint32_t*>(q.codes) : nullptr;
  p.scales = q.scales;
  p.zeros = q.zeros;
  return p;
}

int gmode_of(const QuantLaunch& q) {
  if (q.sa != nullptr) return kGVec;
  uint32_t gbits;
  std::memcpy(&gbits, &q.gamma, sizeof gbits);
  return ((gbits & 0xFFFFu) == 0u && q.had_block == 0) ? kGBf16 : kGF32;
}

template <int V, int G, bool ASYM, int GMODE>
cudaError_t launch_ring_split_g(const QuantLaunch& q, bool write_codes) {
  RingParams p = make_params(q, write_codes);
  p.stage_bytes = G * q.K * 2;
  const int sa_bytes = GMODE == kGVec ? q.K * 4 : 0;
  int stages = (kRingSmemBudget - sa_bytes) / p.stage_bytes;
  p.stages = stages > kMaxStages ? kMaxStages : stages;
  if (p.stages < 2) return cudaErrorInvalidValue;
  const int smem = p.stages * p.stage_bytes + sa_bytes;
  static std::atomic<int> attr_smem[kMaxDevices];
  const cudaError_t ea = ensure_dynamic_smem(quantize_ring_split_kernel<V, G, ASYM, GMODE>, smem, q.device, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int groups = (q.T + G - 1) / G;
  const int blocks = groups < q.num_sms ? groups : q.num_sms;
  return launch_pdl(quantize_ring_split_kernel<V, G, ASYM, GMODE>, blocks, G * kGroupThreads + 32, smem, q.stream, p);
}

template <int V, bool ASYM, int GMODE>
cudaError_t launch_ring_split(const QuantLaunch& q, bool write_codes) {
  return launch_ring_split_g<V, 4, ASYM, GMODE>(q, write_codes);
}

template <int V, int RL, bool HAD, bool RAGGED, bool ASYM, int GMODE>
cudaError_t launch_ring_g(const QuantLaunch& q, bool write_codes) {
  RingParams p = make_params(q, write_codes);
  p.stage_bytes = RL * q.K * 2;
  const int slots = (q.K / 8 + kConsumers - 1) / kConsumers * kConsumers;     // padded to whole threads
  const int sa_bytes = (GMODE == kGVec && V <= 4) ? slots * 32 : 0;
  int stages = (kRingSmemBudget - sa_bytes) / p.stage_bytes;
  p.stages = stages > kMaxStages ? kMaxStages : stages;
  if (p.stages < 2) return cudaErrorInvalidValue;
  const int smem = p.stages * p.stage_bytes + sa_bytes;
  static std::atomic<int> attr_smem[kMaxDevices];
  const cudaError_t ea =
      ensure_dynamic_smem(quantize_ring_kernel<V, RL, HAD, RAGGED, ASYM, GMODE>, smem, q.device, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int groups = (q.T + RL - 1) / RL;
  const int blocks = groups < q.num_sms ? groups : q.num_sms;
  return launch_pdl(quantize_ring_kernel<V, RL, HAD, RAGGED, ASYM, GMODE>, blocks, kRingThreads, smem, q.stream, p);
}

template <int V, int RL, bool HAD, bool RAGGED, bool ASYM>
cudaError_t launch_ring_a(const QuantLaunch& q, bool wc, int gmode) {
  if (gmode == kGVec) return launch_ring_g<V, RL, HAD, RAGGED, ASYM, kGVec>(q, wc);
  if (gmode == kGBf16 && !HAD) return launch_ring_g<V, RL, HAD, RAGGED, ASYM, HAD ? kGF32 : kGBf16>(q, wc);
  return launch_ring_g<V, RL, HAD, RAGGED, ASYM, kGF32>(q, wc);
}

template <int V, int RL, bool HAD>
cudaError_t launch_ring_t(const QuantLaunch& q, bool wc, int gmode) {
  const bool ragged = (q.K / 8) % kConsumers != 0;
  if (q.asym) {
    return ragged ? launch_ring_a<V, RL, HAD, true, true>(q, wc, gmode)
                  : launch_ring_a<V, RL, HAD, false, true>(q, wc, gmode);
  }
  return ragged ? launch_ring_a<V, RL, HAD, true, false>(q, wc, gmode)
                : launch_ring_a<V, RL, HAD, false, false>(q, wc, gmode);
}

template <bool HAD>
cudaError_t launch_ring_hw(const QuantLaunch& q, bool wc, int gmode, int V, int RL) {
  // reachable (V, RL): RL = 4 for K <= 5120 (V <= 2), RL = 2 for K <= 10240 (V = 2, 3), else RL = 1
  if (RL == 4) {
    if (V == 1) return launch_ring_t<1, 4, HAD>(q, wc, gmode);
    if (V == 2) return launch_ring_t<2, 4, HAD>(q, wc, gmode);
  } else if (RL == 2) {
    if (V == 2) return launch_ring_t<2, 2, HAD>(q, wc, gmode);
    if (V == 3) return launch_ring_t<3, 2, HAD>(q, wc, gmode);
  } else {
    switch (V) {
      case 3: return launch_ring_t<3, 1, HAD>(q, wc, gmode);
      case 4: return launch_ring_t<4, 1, HAD>(q, wc, gmode);
      case 5: return launch_ring_t<5, 1, HAD>(q, wc, gmode);
      case 6: return launch_ring_t<6, 1, HAD>(q, wc, gmode);
      case 7: return launch_ring_t<7, 1, HAD>(q, wc, gmode);
      case 8: return launch_ring_t<8, 1, HAD>(q, wc, gmode);
      default: break;
    }
  }
  return cudaErrorInvalidValue;
}

}  // namespace

bool quantize_ring_supported(int K) { return K >= 4096 && K <= kMaxK; }

cudaError_t launch_quantize_ring(const QuantLaunch& q, bool write_codes) {
  if (q.asym && !write_codes) return cudaErrorInvalidValue;
  const int nvec = q.K / 8;
  const int V = (nvec + kConsumers - 1) / kConsumers;
  const int RL = q.K <= 5120 ? 4 : (q.K <= 10240 ? 2 : 1);
  const int gmode = gmode_of(q);
  if (q.had_block == 0 && q.K == 4096) {
    if (q.asym) {
      if (gmode == kGVec) return launch_ring_split<4, true, kGVec>(q, write_codes);
      return gmode == kGBf16 ? launch_ring_split<4, true, kGBf16>(q, write_codes)
                             : launch_ring_split<4, true, kGF32>(q, write_codes);
    }
    if (gmode == kGVec) return launch_ring_split<4, false, kGVec>(q, write_codes);
    return gmode == kGBf16 ? launch_ring_split<4, false, kGBf16>(q, write_codes)
                           : launch_ring_split<4, false, kGF32>(q, write_codes);
  }
  return q.had_block ? launch_ring_hw<true>(q, write_codes, gmode, V, RL)
                     : launch_ring_hw<false>(q, write_codes, gmode, V, RL);
}

}  // namespace baseq

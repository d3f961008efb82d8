// Activation quantiser for long rows (K >= 4096): the same arithmetic contract as
// quantize_act.cu (quant_math.cuh), fed by a bulk-TMA ring.
//
// Why: the register-resident row kernel keeps only its own loads in flight (32-64 KB per SM) and
// measured 2.5-3.0 TB/s (profiles/).  Here one producer lane streams whole token rows
// (row-contiguous cp.async.bulk copies, completion on an mbarrier) into a ring of shared-memory
// stages that fills whatever the 227 KB allow -- 150-200 KB of loads in flight per SM, no
// registers involved -- and 16 consumer warps (512 threads = one row wide, thread r owns the
// 16-byte vectors r, r + 512, ...) read each stage once from shared memory, conflict-free.
//
// Per stage of RL rows: pass 1 (u = g h - b, absmax) -> the stage is released to the producer ->
// block reduction (partials in smem, one designated warp per row finishes the max and computes
// s_t and 1 / s_t once) -> pass 2 from registers (round, clamp, pack, store).
#include "kernels.cuh"
#include "ptx.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr int kConsumers = 512;                 // threads per row
constexpr int kConsumerWarps = kConsumers / 32;
constexpr int kRingThreads = kConsumers + 32;   // + the producer warp
constexpr int kMaxStages = 8;
constexpr int kRingSmemBudget = 220 * 1024;

struct RingParams {
  const uint8_t* x;        // bf16 rows
  int64_t row_bytes_stride;
  int T, K, nvec;
  float alpha, gamma;
  const float* bvec;
  const float* sa;         // per-channel s^a (split kernel only), or NULL for the scalar gamma
  int had_block;
  float had_scale;
  uint32_t* codes;
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

template <int V, int RL, bool HAD, bool WRITE_CODES, bool RAGGED, bool ASYM>
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
    // ===================================================================== producer
    if (lane == 0) {
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
    return;
  }

  // ======================================================================= consumers
  const int r = tid;                               // vector r + i * 512 of every row
  constexpr bool kBiasInRegs = V <= 4;
  float bb[kBiasInRegs ? V : 1][8];
  if (kBiasInRegs) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const int idx = r + i * kConsumers;
      if (p.bvec != nullptr && (!RAGGED || idx < p.nvec)) {
        qm::load8_pinned(p.bvec + 8 * idx, bb[kBiasInRegs ? i : 0]);
      } else {
#pragma unroll
        for (int e = 0; e < 8; ++e) bb[kBiasInRegs ? i : 0][e] = 0.0f;
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
      m[j] = ASYM ? -3.402823466e38f : 0.0f;
      m2[j] = -3.402823466e38f;
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const int idx = r + i * kConsumers;
        const bool ok = !RAGGED || idx < p.nvec;
        uint4 xv = make_uint4(0, 0, 0, 0);
        if (ok) xv = *reinterpret_cast<const uint4*>(stage + static_cast<size_t>(j) * p.K * 2 + idx * 16);
        float f[8];
        qm::unpack8(xv, f);
        if (HAD) qm::hadamard8(f, p.had_block, p.had_scale, lane);
        float bl[8];
        if (!kBiasInRegs) {
          float g_unused[8];
          qm::load_gb(nullptr, p.bvec, p.gamma, idx, ok, g_unused, bl);
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          const float bv = kBiasInRegs ? bb[kBiasInRegs ? i : 0][e] : bl[e];
          u[j][i][e] = qm::affine(p.gamma, f[e], bv);          // scalar s^a only (see the launcher)
          if (ASYM) {
            if (ok) {
              m[j] = fmaxf(m[j], u[j][i][e]);
              m2[j] = fmaxf(m2[j], -u[j][i][e]);
            }
          } else {
            m[j] = fmaxf(m[j], fabsf(u[j][i][e]));
          }
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
      float mm = lane < kConsumerWarps ? s_part[parity][warp][lane] : (ASYM ? -3.402823466e38f : 0.0f);
      float mm2 = (ASYM && lane < kConsumerWarps) ? s_part2[ASYM ? parity : 0][warp][lane]
                                                  : -3.402823466e38f;
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
    if (WRITE_CODES) {
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
// divisions, barrier: ~1 us of latency in the row-wide kernel, where all 16 warps waited together)
// the other three keep the issue slots busy.
constexpr int kSplitGroups = 4;
constexpr int kGroupThreads = kConsumers / kSplitGroups;   // 128
constexpr int kGroupWarps = kGroupThreads / 32;

template <int V, bool WRITE_CODES, bool ASYM, bool SA>
__global__ void __launch_bounds__(kRingThreads, 1) quantize_ring_split_kernel(const RingParams p) {
  constexpr int RL = kSplitGroups;
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
      ptx::mbar_init(ptx::smem_u32(&empty[s]), kConsumerWarps);
    }
    ptx::fence_barrier_init();
  }
  __syncthreads();
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  if (warp == kConsumerWarps) {
    if (lane == 0) {
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
  if (SA) {
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
    float m = ASYM ? -3.402823466e38f : 0.0f;
    float m2 = -3.402823466e38f;                    // asymmetric only: running max of -u
    if (row_ok) {                                   // rows past T were not loaded
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const uint4 xv = *reinterpret_cast<const uint4*>(srow + (r + i * kGroupThreads) * 16);
        float f[8];
        qm::unpack8(xv, f);
        float gv[8];
        if (SA) {
          const float4 g0 = sa_s[2 * (r + i * kGroupThreads)], g1 = sa_s[2 * (r + i * kGroupThreads) + 1];
          gv[0] = g0.x; gv[1] = g0.y; gv[2] = g0.z; gv[3] = g0.w;
          gv[4] = g1.x; gv[5] = g1.y; gv[6] = g1.z; gv[7] = g1.w;
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          u[i][e] = qm::affine(SA ? gv[e] : p.gamma, f[e], bb[i][e]);
          if (ASYM) {
            m = fmaxf(m, u[i][e]);
            m2 = fmaxf(m2, -u[i][e]);
          } else {
            m = fmaxf(m, fabsf(u[i][e]));
          }
        }
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
      float mm2 = -3.402823466e38f;
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

    if (WRITE_CODES) {
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

template <int V, bool WC, bool ASYM, bool SA>
cudaError_t launch_ring_split(const QuantLaunch& q) {
  RingParams p{};
  p.x = static_cast<const uint8_t*>(q.x);
  p.row_bytes_stride = q.ldx * 2;
  p.T = q.T;
  p.K = q.K;
  p.nvec = q.K / 8;
  p.alpha = q.alpha;
  p.gamma = q.gamma;
  p.bvec = q.b;
  p.sa = q.sa;
  p.codes = reinterpret_cast<uint32_t*>(q.codes);
  p.scales = q.scales;
  p.zeros = q.zeros;
  p.stage_bytes = kSplitGroups * q.K * 2;
  const int sa_bytes = SA ? q.K * 4 : 0;
  int stages = (kRingSmemBudget - sa_bytes) / p.stage_bytes;
  p.stages = stages > kMaxStages ? kMaxStages : stages;
  if (p.stages < 2) return cudaErrorInvalidValue;
  const int smem = p.stages * p.stage_bytes + sa_bytes;
  static std::atomic<int> attr_smem[kMaxDevices];
  const cudaError_t ea = ensure_dynamic_smem(quantize_ring_split_kernel<V, WC, ASYM, SA>, smem, q.device, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int groups = (q.T + kSplitGroups - 1) / kSplitGroups;
  const int blocks = groups < q.num_sms ? groups : q.num_sms;
  return launch_pdl(quantize_ring_split_kernel<V, WC, ASYM, SA>, blocks, kRingThreads, smem, q.stream, p);
}

template <int V, int RL, bool HAD, bool WC, bool RAGGED, bool ASYM>
cudaError_t launch_ring_a(const QuantLaunch& q) {
  RingParams p{};
  p.x = static_cast<const uint8_t*>(q.x);
  p.row_bytes_stride = q.ldx * 2;
  p.T = q.T;
  p.K = q.K;
  p.nvec = q.K / 8;
  p.alpha = q.alpha;
  p.gamma = q.gamma;
  p.bvec = q.b;
  p.had_block = q.had_block;
  p.had_scale = q.had_scale;
  p.codes = reinterpret_cast<uint32_t*>(q.codes);
  p.scales = q.scales;
  p.zeros = q.zeros;
  p.stage_bytes = RL * q.K * 2;
  int stages = kRingSmemBudget / p.stage_bytes;
  p.stages = stages > kMaxStages ? kMaxStages : stages;
  if (p.stages < 2) return cudaErrorInvalidValue;
  const int smem = p.stages * p.stage_bytes;
  static std::atomic<int> attr_smem[kMaxDevices];
  const cudaError_t ea = ensure_dynamic_smem(quantize_ring_kernel<V, RL, HAD, WC, RAGGED, ASYM>, smem, q.device, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int groups = (q.T + RL - 1) / RL;
  const int blocks = groups < q.num_sms ? groups : q.num_sms;
  return launch_pdl(quantize_ring_kernel<V, RL, HAD, WC, RAGGED, ASYM>, blocks, kRingThreads, smem, q.stream, p);
}

template <int V, int RL, bool HAD, bool WC, bool RAGGED>
cudaError_t launch_ring_r(const QuantLaunch& q) {
  // the asymmetric variant (NEXT-1) always writes codes
  if (q.asym) return WC ? launch_ring_a<V, RL, HAD, true, RAGGED, true>(q) : cudaErrorInvalidValue;
  return launch_ring_a<V, RL, HAD, WC, RAGGED, false>(q);
}

template <int V, int RL, bool HAD, bool WC>
cudaError_t launch_ring_t(const QuantLaunch& q) {
  return (q.K / 8) % kConsumers != 0 ? launch_ring_r<V, RL, HAD, WC, true>(q)
                                     : launch_ring_r<V, RL, HAD, WC, false>(q);
}

template <bool HAD, bool WC>
cudaError_t launch_ring_hw(const QuantLaunch& q, int V, int RL) {
  // reachable (V, RL): RL = 4 for K <= 5120 (V <= 2), RL = 2 for K <= 10240 (V = 2, 3), else RL = 1
  if (RL == 4) {
    if (V == 1) return launch_ring_t<1, 4, HAD, WC>(q);
    if (V == 2) return launch_ring_t<2, 4, HAD, WC>(q);
  } else if (RL == 2) {
    if (V == 2) return launch_ring_t<2, 2, HAD, WC>(q);
    if (V == 3) return launch_ring_t<3, 2, HAD, WC>(q);
  } else {
    switch (V) {
      case 3: return launch_ring_t<3, 1, HAD, WC>(q);
      case 4: return launch_ring_t<4, 1, HAD, WC>(q);
      case 5: return launch_ring_t<5, 1, HAD, WC>(q);
      case 6: return launch_ring_t<6, 1, HAD, WC>(q);
      case 7: return launch_ring_t<7, 1, HAD, WC>(q);
      case 8: return launch_ring_t<8, 1, HAD, WC>(q);
      default: break;
    }
  }
  return cudaErrorInvalidValue;
}

}  // namespace

bool quantize_ring_supported(int K) { return K >= 4096 && K <= 32768; }
// a per-channel s^a vector is handled by the split kernel only
bool quantize_ring_supports_sa(int K, int had_block) { return K == 4096 && had_block == 0; }

cudaError_t launch_quantize_ring(const QuantLaunch& q, bool write_codes) {
  const int nvec = q.K / 8;
  const int V = (nvec + kConsumers - 1) / kConsumers;
  const int RL = q.K <= 5120 ? 4 : (q.K <= 10240 ? 2 : 1);
  if (q.had_block == 0 && q.K == 4096) {
    if (q.asym) {
      if (q.sa != nullptr || !write_codes) return cudaErrorInvalidValue;
      return launch_ring_split<4, true, true, false>(q);
    }
    if (q.sa != nullptr) {
      return write_codes ? launch_ring_split<4, true, false, true>(q) : launch_ring_split<4, false, false, true>(q);
    }
    return write_codes ? launch_ring_split<4, true, false, false>(q) : launch_ring_split<4, false, false, false>(q);
  }
  if (q.had_block) {
    return write_codes ? launch_ring_hw<true, true>(q, V, RL) : launch_ring_hw<true, false>(q, V, RL);
  }
  return write_codes ? launch_ring_hw<false, true>(q, V, RL) : launch_ring_hw<false, false>(q, V, RL);
}

}  // namespace baseq

// NEXT-3: KV-cache "per-head asymmetric dynamic quantization".  A group is one
// (token, head) block of head_dim contiguous channels (heads never straddle groups); each
// group gets its own step and lower bound by the asymmetric rule of Eq. 4, in the
// arithmetic of NEXT-1 (quant_math.cuh A1-A3) with u = x (no gamma, bias or Hadamard).
//
// HBM-bound: 2 B read + 0.5 B written per element, 8 / head_dim B of (scale, zero).
// r2: the same skeleton as the activation quantiser (quantize_ring.cu) instead of register-resident
// loads -- one producer lane streams 32 KB runs of groups with cp.async.bulk into a shared-memory
// ring (~190 KB of loads in flight per SM, whatever the consumers do), 16 consumer warps read each
// stage once.  LPG = head_dim / 8 lanes hold one group (one 16-byte vector each): the group's
// min / max need log2(LPG) shuffle steps inside the sub-warp and no barrier at all; lane 0 of the
// sub-warp does the two IEEE divisions and writes (scale, zero); the bf16 -> fp32 conversion is
// one mixed-precision FMA per element (x * 1 + 0, exact) on the FMA pipe.
#include "kernels.cuh"
#include "ptx.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr int kKvConsumers = 512;
constexpr int kKvThreads = kKvConsumers + 32;     // + the producer warp
constexpr int kKvStageBytes = 32 * 1024;
constexpr int kKvStages = 6;
constexpr int kKvSmem = kKvStages * kKvStageBytes;
constexpr float kNegHuge = -3.402823466e38f;

struct KvParams {
  const uint8_t* x;          // bf16
  int64_t row_stride_bytes;  // ldx * 2
  int64_t n_groups;          // T * heads
  int heads;
  int contiguous;            // ldx == heads * head_dim: X is one flat array of groups
  int stages_per_row;        // strided input: a stage never crosses a row
  float alpha;
  uint32_t* codes;
  float* scales;
  float* zeros;
};

// groups [g0, g0 + n) of stage `st`: a run of consecutive groups (contiguous input), or a run inside
// one token row (strided input)
template <int LPG>
__device__ __forceinline__ void kv_stage(const KvParams& p, int64_t st, int64_t& g0, int& n) {
  constexpr int kGS = kKvStageBytes / (LPG * 16);          // groups per full stage
  if (p.contiguous) {
    g0 = st * kGS;
    const int64_t left = p.n_groups - g0;
    n = left < kGS ? static_cast<int>(left) : kGS;
  } else {
    const int64_t row = st / p.stages_per_row;
    const int h0 = static_cast<int>(st % p.stages_per_row) * kGS;
    g0 = row * p.heads + h0;
    n = p.heads - h0 < kGS ? p.heads - h0 : kGS;
  }
}

template <int LPG>
__global__ void __launch_bounds__(kKvThreads, 1) quantize_kv_kernel(const KvParams p, int64_t n_stages) {
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ uint64_t full[kKvStages], empty[kKvStages];
  constexpr int kGroupBytes = LPG * 16;
  constexpr int kSub = kKvConsumers / LPG;                 // sub-warps (one group at a time each)
  constexpr int kGS = kKvStageBytes / kGroupBytes;
  constexpr int kPer = kGS / kSub;                         // groups per sub-warp and stage: 4
  static_assert(kGS % kSub == 0, "stage layout");

  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int s = 0; s < kKvStages; ++s) {
      ptx::mbar_init(ptx::smem_u32(&full[s]), 1);
      ptx::mbar_init(ptx::smem_u32(&empty[s]), kKvConsumers / 32);
    }
    ptx::fence_barrier_init();
  }
  __syncthreads();
  ptx::griddep_launch_dependents();
  ptx::griddep_wait();

  if (warp == kKvConsumers / 32) {
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      for (int64_t st = blockIdx.x; st < n_stages; st += gridDim.x) {
        ptx::mbar_wait(ptx::smem_u32(&empty[s]), ph ^ 1u);
        int64_t g0;
        int n;
        kv_stage<LPG>(p, st, g0, n);
        const uint32_t bytes = static_cast<uint32_t>(n) * kGroupBytes;
        const uint8_t* src = p.contiguous
                                 ? p.x + g0 * kGroupBytes
                                 : p.x + (g0 / p.heads) * p.row_stride_bytes + (g0 % p.heads) * kGroupBytes;
        const uint32_t bar = ptx::smem_u32(&full[s]);
        ptx::mbar_arrive_expect_tx(bar, bytes);
        ptx::bulk_load_1d(ptx::smem_u32(ring) + s * kKvStageBytes, src, bytes, bar);
        if (++s == kKvStages) { s = 0; ph ^= 1u; }
      }
    }
    return;
  }

  const int sub = tid / LPG;                               // this sub-warp's groups: sub, sub + kSub, ...
  const int l = tid & (LPG - 1);
  const int leader = lane & ~(LPG - 1);
  // the contract's u = fma(1, x, -0): the addend is MINUS zero, so that x = -0 stays -0 (as in the oracle)
  const float zero8[8] = {-0.f, -0.f, -0.f, -0.f, -0.f, -0.f, -0.f, -0.f};
  int s = 0;
  uint32_t ph = 0;
  for (int64_t st = blockIdx.x; st < n_stages; st += gridDim.x) {
    int64_t g0;
    int n;
    kv_stage<LPG>(p, st, g0, n);
    ptx::mbar_wait(ptx::smem_u32(&full[s]), ph);
    const uint8_t* stage = ring + s * kKvStageBytes;

    float u[kPer][8];
    float mx[kPer], mneg[kPer];
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
      const int gi = sub + j * kSub;
      uint4 xv = make_uint4(0u, 0u, 0u, 0u);
      if (gi < n) xv = *reinterpret_cast<const uint4*>(stage + (gi * LPG + l) * 16);
      qm::affine8_bf16(xv, 0x3F80u, zero8, u[j]);          // Q0: x * 1 + 0, exact
      mx[j] = kNegHuge;
      mneg[j] = kNegHuge;
      qm::maxmin8(mx[j], mneg[j], u[j]);                   // A1
    }
    // the stage's data is in registers: release it
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(ptx::smem_u32(&empty[s]));
    if (++s == kKvStages) { s = 0; ph ^= 1u; }

    // Reduction over the LPG lanes of a sub-warp, the four groups together: a TRANSPOSING butterfly
    // (a lane keeps half of the values and sends the other half at each of the first two steps)
    // needs 2 + 1 exchanges and leaves lane l with the partial of group (l / (LPG / 4)) & 3; the
    // remaining log2(LPG) - 2 steps reduce that single value.  5 shuffles per quantity instead of
    // 16 (a shuffle costs four issue slots).
    constexpr int kQ = LPG / 4;                            // lanes that end up owning the same group
    {
      const bool hi2 = (l & (LPG / 2)) != 0, hi1 = (l & (LPG / 4)) != 0;
      // step 1 (partner l ^ LPG/2): upper lanes keep groups 2, 3, lower lanes keep groups 0, 1
      float kx0 = hi2 ? mx[2] : mx[0], kx1 = hi2 ? mx[3] : mx[1];
      float sx0 = hi2 ? mx[0] : mx[2], sx1 = hi2 ? mx[1] : mx[3];
      float kn0 = hi2 ? mneg[2] : mneg[0], kn1 = hi2 ? mneg[3] : mneg[1];
      float sn0 = hi2 ? mneg[0] : mneg[2], sn1 = hi2 ? mneg[1] : mneg[3];
      kx0 = fmaxf(kx0, __shfl_xor_sync(0xffffffffu, sx0, LPG / 2));
      kx1 = fmaxf(kx1, __shfl_xor_sync(0xffffffffu, sx1, LPG / 2));
      kn0 = fmaxf(kn0, __shfl_xor_sync(0xffffffffu, sn0, LPG / 2));
      kn1 = fmaxf(kn1, __shfl_xor_sync(0xffffffffu, sn1, LPG / 2));
      // step 2 (partner l ^ LPG/4): upper lanes keep the odd group of their pair
      float vx = hi1 ? kx1 : kx0, tx = hi1 ? kx0 : kx1;
      float vn = hi1 ? kn1 : kn0, tn = hi1 ? kn0 : kn1;
      vx = fmaxf(vx, __shfl_xor_sync(0xffffffffu, tx, LPG / 4));
      vn = fmaxf(vn, __shfl_xor_sync(0xffffffffu, tn, LPG / 4));
#pragma unroll
      for (int o = kQ / 2; o > 0; o >>= 1) {
        vx = fmaxf(vx, __shfl_xor_sync(0xffffffffu, vx, o));
        vn = fmaxf(vn, __shfl_xor_sync(0xffffffffu, vn, o));
      }
      // lane l now holds the max / -min of group jown = 2 * hi2 + hi1; A2 by the first lane of each
      // quarter (the two IEEE divisions: ~30 instructions, once per group)
      const int jown = (hi2 ? 2 : 0) + (hi1 ? 1 : 0);
      const int gown = sub + jown * kSub;
      float zt_own = 0.0f, inv_own = 0.0f;
      if ((l & (kQ - 1)) == 0) {
        const float st_ = qm::step_size_asym(p.alpha, -vn, vx);
        zt_own = qm::lower_bound_asym(p.alpha, -vn);
        inv_own = qm::reciprocal(st_);
        if (gown < n) {
          p.scales[g0 + gown] = st_;
          p.zeros[g0 + gown] = zt_own;
        }
      }
      // hand (z, 1 / s) of group j back to all lanes of the sub-warp: its owner is lane j * kQ
#pragma unroll
      for (int j = 0; j < kPer; ++j) {
        const int gi = sub + j * kSub;
        const float zt = __shfl_sync(0xffffffffu, zt_own, leader + j * kQ);
        const float inv = __shfl_sync(0xffffffffu, inv_own, leader + j * kQ);
        const uint32_t w = qm::quantize_pack8_asym(u[j], zt, inv);   // A3
        if (gi < n) p.codes[(g0 + gi) * LPG + l] = w;
      }
    }
  }
}

template <int LPG>
cudaError_t launch_lpg(const KvLaunch& q) {
  KvParams p{};
  p.x = static_cast<const uint8_t*>(q.x);
  p.row_stride_bytes = q.ldx * 2;
  p.n_groups = static_cast<int64_t>(q.T) * q.heads;
  p.heads = q.heads;
  p.contiguous = q.ldx == static_cast<int64_t>(q.heads) * q.head_dim ? 1 : 0;
  constexpr int kGS = kKvStageBytes / (LPG * 16);
  p.stages_per_row = (q.heads + kGS - 1) / kGS;
  p.alpha = q.alpha;
  p.codes = reinterpret_cast<uint32_t*>(q.codes);
  p.scales = q.scales;
  p.zeros = q.zeros;
  const int64_t n_stages = p.contiguous ? (p.n_groups + kGS - 1) / kGS
                                        : static_cast<int64_t>(q.T) * p.stages_per_row;
  static std::atomic<int> attr_smem[kMaxDevices];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return cudaErrorInvalidDevice;
  const cudaError_t ea = ensure_dynamic_smem(quantize_kv_kernel<LPG>, kKvSmem, dev, attr_smem);
  if (ea != cudaSuccess) return ea;
  const int64_t blocks = n_stages < q.num_sms ? n_stages : q.num_sms;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(blocks), 1, 1);
  cfg.blockDim = dim3(kKvThreads, 1, 1);
  cfg.dynamicSmemBytes = kKvSmem;
  cfg.stream = q.stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, quantize_kv_kernel<LPG>, p, n_stages);
}

}  // namespace

cudaError_t launch_quantize_kv(const KvLaunch& q) {
  if (q.head_dim != 64 && q.head_dim != 128) return cudaErrorNotSupported;
  if (q.alpha < kMinFastAlpha) return launch_quantize_kv_small_alpha(q);
  switch (q.head_dim) {
    case 64: return launch_lpg<8>(q);
    case 128: return launch_lpg<16>(q);
    default: return cudaErrorNotSupported;
  }
}

}  // namespace baseq

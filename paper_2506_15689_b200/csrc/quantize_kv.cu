// NEXT-3: KV-cache "per-head asymmetric dynamic quantization".  A group is one
// (token, head) block of head_dim contiguous channels (heads never straddle groups); each
// group gets its own step and lower bound by the asymmetric rule of Eq. 4, in the
// arithmetic of NEXT-1 (quant_math.cuh A1-A3) with u = x (no gamma, bias or Hadamard).
//
// HBM-bound: 2 B read + 0.5 B written per element, 8 / head_dim B of (scale, zero).  Layout of the
// work: LPG = head_dim / 8 lanes hold one group (one 16-byte vector each), and every such sub-warp
// handles LPG groups per pass, so a lane has LPG independent 16-byte loads in flight.  The LPG
// (min, max) pairs are reduced with a transposing butterfly (LPG - 1 exchanges instead of
// LPG * log2 LPG): afterwards lane l of the sub-warp owns group l, computes its step, reciprocal
// and lower bound once (the two IEEE divisions are ~25 instructions), writes scale and zero
// coalesced, and the values are handed back by shuffle for the rounding pass.
#include "kernels.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr int kKvThreads = 256;

template <int LPG, bool CONTIG>
// (197 registers at LPG = 16: one 256-thread block per SM with 64 KB of loads in flight; forcing two
// blocks per SM spills 230 bytes per thread)
__global__ void __launch_bounds__(kKvThreads)
quantize_kv_kernel(const uint4* __restrict__ x, int64_t ldxv, int64_t n_groups, int heads, float alpha,
                   uint32_t* __restrict__ codes, float* __restrict__ scales, float* __restrict__ zeros) {
  constexpr int G = LPG;                      // groups per sub-warp and pass
  constexpr int kSub = 32 / LPG;              // sub-warps per warp
  const int lane = threadIdx.x & 31;
  const int l = lane & (LPG - 1);             // vector index inside the group
  const int sub = lane / LPG;
  const int64_t warp_id = (static_cast<int64_t>(blockIdx.x) * kKvThreads + threadIdx.x) >> 5;
  const int64_t n_warps = (static_cast<int64_t>(gridDim.x) * kKvThreads) >> 5;
  const int64_t per_pass = static_cast<int64_t>(kSub) * G;
  const int64_t n_pass = (n_groups + per_pass - 1) / per_pass;

  for (int64_t pass = warp_id; pass < n_pass; pass += n_warps) {
    const int64_t g0 = pass * per_pass + static_cast<int64_t>(sub) * G;
    uint4 v[G];
#pragma unroll
    for (int j = 0; j < G; ++j) {
      const int64_t g = g0 + j;
      v[j] = make_uint4(0u, 0u, 0u, 0u);
      if (g < n_groups) {
        // vector index of (group g, lane l): contiguous rows, or token * ldx + head * head_dim
        const int64_t idx = CONTIG ? g * LPG + l : (g / heads) * ldxv + (g % heads) * LPG + l;
        v[j] = __ldg(x + idx);
      }
    }
    // A1: this lane's 8 channels of each group
    float mx[G], mn[G];
#pragma unroll
    for (int j = 0; j < G; ++j) {
      float f[8];
      qm::unpack8(v[j], f);
      mx[j] = fmaxf(fmaxf(fmaxf(f[0], f[1]), fmaxf(f[2], f[3])), fmaxf(fmaxf(f[4], f[5]), fmaxf(f[6], f[7])));
      mn[j] = fminf(fminf(fminf(f[0], f[1]), fminf(f[2], f[3])), fminf(fminf(f[4], f[5]), fminf(f[6], f[7])));
    }
    // transposing butterfly: after the step with stride s a lane keeps the half of the group
    // indices whose bit s equals its own lane bit; at the end lane l holds group l's totals in [0]
#pragma unroll
    for (int s = LPG / 2; s >= 1; s >>= 1) {
      const bool up = (l & s) != 0;
#pragma unroll
      for (int i = 0; i < s; ++i) {
        const float send_x = up ? mx[i] : mx[i + s], keep_x = up ? mx[i + s] : mx[i];
        const float send_n = up ? mn[i] : mn[i + s], keep_n = up ? mn[i + s] : mn[i];
        mx[i] = fmaxf(keep_x, __shfl_xor_sync(0xffffffffu, send_x, s));
        mn[i] = fminf(keep_n, __shfl_xor_sync(0xffffffffu, send_n, s));
      }
    }
    // A2 for group g0 + l
    const float st = qm::step_size_asym(alpha, mn[0], mx[0]);
    const float zt = qm::lower_bound_asym(alpha, mn[0]);
    const float inv = qm::reciprocal(st);
    if (g0 + l < n_groups) {
      scales[g0 + l] = st;
      zeros[g0 + l] = zt;
    }
    // A3: hand (z, 1/s) of group j back to its lanes, round, clamp, pack
#pragma unroll
    for (int j = 0; j < G; ++j) {
      const int src = (lane & ~(LPG - 1)) + j;
      const float zj = __shfl_sync(0xffffffffu, zt, src);
      const float ij = __shfl_sync(0xffffffffu, inv, src);
      float f[8];
      qm::unpack8(v[j], f);
      const uint32_t w = qm::quantize_pack8_asym(f, zj, ij);
      const int64_t g = g0 + j;
      if (g < n_groups) codes[g * LPG + l] = w;
    }
  }
}

template <int LPG>
cudaError_t launch_lpg(const KvLaunch& q) {
  const int64_t n_groups = static_cast<int64_t>(q.T) * q.heads;
  const int64_t per_pass = 32;                                   // kSub * G = 32 groups per warp pass
  const int64_t n_pass = (n_groups + per_pass - 1) / per_pass;
  const int64_t warps_per_block = kKvThreads / 32;
  int64_t blocks = (n_pass + warps_per_block - 1) / warps_per_block;
  const int64_t cap = static_cast<int64_t>(q.num_sms) * 8;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  const bool contig = q.ldx == static_cast<int64_t>(q.heads) * q.head_dim;
  const uint4* x = static_cast<const uint4*>(q.x);
  uint32_t* codes = reinterpret_cast<uint32_t*>(q.codes);
  if (contig) {
    quantize_kv_kernel<LPG, true><<<static_cast<unsigned>(blocks), kKvThreads, 0, q.stream>>>(
        x, q.ldx / 8, n_groups, q.heads, q.alpha, codes, q.scales, q.zeros);
  } else {
    quantize_kv_kernel<LPG, false><<<static_cast<unsigned>(blocks), kKvThreads, 0, q.stream>>>(
        x, q.ldx / 8, n_groups, q.heads, q.alpha, codes, q.scales, q.zeros);
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_quantize_kv(const KvLaunch& q) {
  switch (q.head_dim) {
    case 64: return launch_lpg<8>(q);
    case 128: return launch_lpg<16>(q);
    default: return cudaErrorNotSupported;
  }
}

}  // namespace baseq

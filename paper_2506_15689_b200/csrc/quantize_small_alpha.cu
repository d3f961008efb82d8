// Clip ratios below 2^-16 (include/baseq.h allows 0 < alpha <= 1).
//
// Every other quantiser kernel rounds with  fma(u, 1 / s_t, 1.5 * 2^23): exact as long as
// |u / s_t| < 2^22, which |u| <= max|u| = 7 s_t / alpha guarantees for alpha >= 2^-16.  Below that
// the quotient can be arbitrarily large -- but every |u / s_t| >= 8.5 saturates anyway, so clamping
// u to +-16 s_t first (asymmetric: u - z_t to [-16 s_t, 32 s_t]) changes no code and keeps the
// quotient inside the exact range.  No calibrated alpha is anywhere near, so this path is a plain,
// slow kernel of its own instead of two more instructions per element in the fast ones: one warp
// per group (token row, or (token, head) for the KV cache), lane l owning the 16-byte vectors
// l, l + 32, ... (an aligned half-warp = 128 channels, what qm::hadamard8 expects), two passes with
// the arithmetic of quant_math.cuh.  launch_quantize_act / launch_quantize_kv route here, and the
// fused entry points quantise through it and then run the plain GEMM.
#include "kernels.cuh"
#include "quant_math.cuh"

namespace baseq {
namespace {

constexpr float kNegHuge = -3.402823466e38f;

struct SmallAlphaParams {
  const uint4* x;          // bf16 as 16-byte vectors
  int64_t ldxv;            // vectors between the starts of two token rows
  int64_t n_groups;        // T (activations) or T * heads (KV cache)
  int groups_per_row;      // 1, or heads
  int nv;                  // vectors per group
  float alpha, gamma;
  const float* sa;
  const float* b;
  int had_block;
  float had_scale;
  uint32_t* codes;         // [n_groups, nv] words of 8 nibbles, or nullptr (scales only)
  float* scales;
  float* zeros;
};

template <bool ASYM>
__global__ void __launch_bounds__(256) quantize_small_alpha_kernel(const SmallAlphaParams p) {
  const int lane = threadIdx.x & 31;
  const int64_t warps = static_cast<int64_t>(gridDim.x) * (blockDim.x >> 5);
  const int nvl = (p.nv + 31) >> 5;
  for (int64_t grp = static_cast<int64_t>(blockIdx.x) * (blockDim.x >> 5) + (threadIdx.x >> 5);
       grp < p.n_groups; grp += warps) {
    const int64_t row = grp / p.groups_per_row;
    const int sub = static_cast<int>(grp % p.groups_per_row);
    const uint4* xr = p.x + row * p.ldxv + static_cast<int64_t>(sub) * p.nv;
    uint32_t* cr = p.codes ? p.codes + grp * p.nv : nullptr;
    auto vector_u = [&](int j, float (&u)[8]) {
      const int i = lane + 32 * j;
      const bool ok = i < p.nv;
      const uint4 v = ok ? __ldg(xr + i) : make_uint4(0u, 0u, 0u, 0u);
      float f[8], g[8], bb[8];
      qm::unpack8(v, f);
      if (p.had_block) qm::hadamard8(f, p.had_block, p.had_scale, lane);
      // per-channel operands are indexed inside the group's row (one group per row whenever they exist)
      qm::load_gb(p.sa, p.b, p.gamma, i, ok, g, bb);
#pragma unroll
      for (int e = 0; e < 8; ++e) u[e] = qm::affine(g[e], f[e], bb[e]);
      return ok;
    };
    float m = ASYM ? kNegHuge : 0.0f, m2 = kNegHuge;
    for (int j = 0; j < nvl; ++j) {
      float u[8];
      if (vector_u(j, u)) {
        if (ASYM) qm::maxmin8(m, m2, u);
        else m = qm::absmax8(m, u);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
      if (ASYM) m2 = fmaxf(m2, __shfl_xor_sync(0xffffffffu, m2, o));
    }
    const float st = ASYM ? qm::step_size_asym(p.alpha, -m2, m) : qm::step_size(p.alpha, m);
    const float zt = ASYM ? qm::lower_bound_asym(p.alpha, -m2) : 0.0f;
    const float inv = qm::reciprocal(st);
    if (lane == 0) {
      p.scales[grp] = st;
      if (ASYM) p.zeros[grp] = zt;
    }
    if (cr == nullptr) continue;
    const float lo = __fmul_rn(-16.0f, st), hi = __fmul_rn(ASYM ? 32.0f : 16.0f, st);
    for (int j = 0; j < nvl; ++j) {
      float u[8];
      const bool ok = vector_u(j, u);
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const float d = ASYM ? __fsub_rn(u[e], zt) : u[e];       // A3 subtracts first
        u[e] = fminf(fmaxf(d, lo), hi);
      }
      if (ok) cr[lane + 32 * j] = ASYM ? qm::quantize_pack8_asym(u, 0.0f, inv) : qm::quantize_pack8(u, inv);
    }
  }
}

template <bool ASYM>
cudaError_t launch(const SmallAlphaParams& p, int num_sms, cudaStream_t stream) {
  const int64_t want = (p.n_groups + 7) / 8;
  const int64_t cap = static_cast<int64_t>(num_sms > 0 ? num_sms : 148) * 8;
  const int blocks = static_cast<int>(want < cap ? want : cap);
  quantize_small_alpha_kernel<ASYM><<<blocks, 256, 0, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_quantize_small_alpha(const QuantLaunch& q, bool write_codes) {
  SmallAlphaParams p{};
  p.x = static_cast<const uint4*>(q.x);
  p.ldxv = q.ldx / 8;
  p.n_groups = q.T;
  p.groups_per_row = 1;
  p.nv = q.K / 8;
  p.alpha = q.alpha;
  p.gamma = q.gamma;
  p.sa = q.sa;
  p.b = q.b;
  p.had_block = q.had_block;
  p.had_scale = q.had_scale;
  p.codes = write_codes ? reinterpret_cast<uint32_t*>(q.codes) : nullptr;
  p.scales = q.scales;
  p.zeros = q.zeros;
  return q.asym ? launch<true>(p, q.num_sms, q.stream) : launch<false>(p, q.num_sms, q.stream);
}

cudaError_t launch_quantize_kv_small_alpha(const KvLaunch& q) {
  SmallAlphaParams p{};
  p.x = static_cast<const uint4*>(q.x);
  p.ldxv = q.ldx / 8;
  p.n_groups = static_cast<int64_t>(q.T) * q.heads;
  p.groups_per_row = q.heads;
  p.nv = q.head_dim / 8;
  p.alpha = q.alpha;
  p.gamma = 1.0f;
  p.sa = nullptr;
  p.b = nullptr;
  p.had_block = 0;
  p.had_scale = 1.0f;
  p.codes = reinterpret_cast<uint32_t*>(q.codes);
  p.scales = q.scales;
  p.zeros = q.zeros;
  return launch<true>(p, q.num_sms, q.stream);
}

}  // namespace baseq

// Fused activation quantiser (steps a0-a5 of DESIGN.md; K2 of SURVEY; "fuse the
// online bias and scaling ... within quantization", Eq. 15).
//
// HBM-bound row kernel: each token row is read from HBM exactly once (128-bit coalesced
// streaming loads), stays in registers as fp32 u between the absmax pass and the rounding
// pass, and leaves as packed int4 nibbles (0.5 B/element) plus one fp32 scale.  Algorithmic
// traffic: 2.5 B/element.
//
// Arithmetic contract (Q0-Q7), every line one correctly rounded fp32 operation --
// explicit __f*_rn intrinsics are never contracted or re-associated by nvcc:
//   Q1  h   = block Hadamard of x: butterflies (a,b) <- (a+b, a-b) for stride 1,2,..,B/2,
//             then h *= (float)(1/sqrt(B))
//   Q2  u   = fma(g, h, -b)                     g = sa ? sa[k] : gamma
//   Q3  m   = max |u|
//   Q4  s_t = max((alpha * m) / 7, 1e-12)
//   Q5  inv = 1 / s_t
//   Q6  q   = clamp(rne(u * inv), -8, 7)
//   Q7  byte j = (q[2j] & 15) | ((q[2j+1] & 15) << 4)
#include "kernels.cuh"
#include "ptx.cuh"
#include "quant_math.cuh"

namespace baseq {

namespace {

constexpr int kMaxV = 8;          // 16-byte vectors (8 bf16) a thread keeps in registers

// One row = TPR threads; thread r holds vectors r, r + TPR, ..., r + (V-1) TPR of the row.
// A block holds THREADS = max(256, TPR) threads = RPB rows at a time (TPR <= 512 so that 8 vectors
// of fp32 u fit the register file) and walks over row groups blockIdx.x, + gridDim.x, ...; the
// next group's loads are issued before the current group is processed, so every thread keeps V
// 16-byte loads in flight all the time (the r1a kernel only had loads in flight during its load
// phase: 2.0-2.5 TB/s, profiles/r1a.md).
template <int V, bool HAD, bool WRITE_CODES, int THREADS>
__global__ void __launch_bounds__(THREADS, 512 / THREADS) quantize_act_kernel(
    const uint4* __restrict__ x, int64_t ldx_vec, int T, int nvec, int tpr_log2,
    float alpha, float gamma, const float* __restrict__ sa, const float* __restrict__ bvec,
    int had_block, float had_scale, uint32_t* __restrict__ codes, float* __restrict__ scales) {
  __shared__ float s_red[2][THREADS / 32];

  const int tpr = 1 << tpr_log2;
  const int tid = threadIdx.x;
  const int r = tid & (tpr - 1);
  const int row_in_block = tid >> tpr_log2;
  const int rows_per_block = blockDim.x >> tpr_log2;
  const int lane = tid & 31;
  const int num_groups = (T + rows_per_block - 1) / rows_per_block;

  auto load_group = [&](int group, uint4 (&xv)[V]) {
    const int row = group * rows_per_block + row_in_block;
    const bool row_ok = group < num_groups && row < T;
    const uint4* xrow = x + static_cast<int64_t>(row_ok ? row : 0) * ldx_vec;
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const int idx = r + i * tpr;
      xv[i] = (row_ok && idx < nvec) ? ptx::ldg_nc_stream(xrow + idx) : make_uint4(0, 0, 0, 0);
    }
  };

  // per-channel bias of this thread's columns: the same for every row, kept in registers
  // (channels beyond K get g = gamma, b = 0, x = 0, hence u = 0: no per-element select)
  // -- for up to 4 vectors per thread; longer rows re-read it from L1 for every row
  constexpr bool kBiasInRegs = V <= 4;
  float bb[kBiasInRegs ? V : 1][8];
  if (kBiasInRegs) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const int idx = r + i * tpr;
      float g_unused[8];
      qm::load_gb(nullptr, bvec, gamma, idx, idx < nvec, g_unused, bb[kBiasInRegs ? i : 0]);
    }
  }

  auto process = [&](int group, const uint4 (&xv)[V], int parity) {
    const int row = group * rows_per_block + row_in_block;
    const bool row_ok = row < T;
    // ---- pass 1: Hadamard, u = g*h - b, absmax
    float u[V][8];
    float m = 0.0f;
#pragma unroll
    for (int i = 0; i < V; ++i) {
      float f[8];
      qm::unpack8(xv[i], f);
      if (HAD) qm::hadamard8(f, had_block, had_scale, lane);
      const int idx = r + i * tpr;
      float g[8], bl[8];
      if (sa != nullptr || !kBiasInRegs) {
        qm::load_gb(sa, kBiasInRegs ? nullptr : bvec, gamma, idx, idx < nvec, g, bl);
      }
      if (sa != nullptr) {
#pragma unroll
        for (int j = 0; j < 8; ++j)
          u[i][j] = qm::affine(g[j], f[j], kBiasInRegs ? bb[kBiasInRegs ? i : 0][j] : bl[j]);
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j)
          u[i][j] = qm::affine(gamma, f[j], kBiasInRegs ? bb[kBiasInRegs ? i : 0][j] : bl[j]);
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) m = fmaxf(m, fabsf(u[i][j]));
    }

    // ---- row absmax: warp shuffle, then (TPR > 32) across the row's warps through smem
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (tpr > 32) {
      const int warp = tid >> 5;
      if (lane == 0) s_red[parity][warp] = m;
      __syncthreads();                 // s_red is double-buffered: one barrier per group
      const int wpr = tpr >> 5;        // warps per row
      const int w0 = row_in_block * wpr;
      float mm = s_red[parity][w0];
      for (int w = 1; w < wpr; ++w) mm = fmaxf(mm, s_red[parity][w0 + w]);
      m = mm;
    }

    // ---- Q4, Q5
    const float st = qm::step_size(alpha, m);
    const float inv = qm::reciprocal(st);
    if (row_ok && r == 0) scales[row] = st;

    // ---- pass 2: round, clamp, pack, store (one 32-bit word = 8 codes per vector)
    if (WRITE_CODES && row_ok) {
      uint32_t* crow = codes + static_cast<int64_t>(row) * nvec;
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const int idx = r + i * tpr;
        uint32_t t[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) t[j] = qm::code_bits(u[i][j], inv);
        const uint32_t w = qm::pack_nibbles(t);
        if (idx < nvec) crow[idx] = w;
      }
    }
  };

  // two groups per trip with ping-pong buffers: the next group's loads are in flight while the
  // current one is processed, and no register copies are needed
  uint4 xa[V], xb[V];
  load_group(blockIdx.x, xa);
  for (int group = blockIdx.x; group < num_groups; group += 2 * gridDim.x) {
    load_group(group + gridDim.x, xb);
    process(group, xa, 0);
    load_group(group + 2 * gridDim.x, xa);
    if (group + gridDim.x < num_groups || tpr > 32) process(group + gridDim.x, xb, 1);
  }
}

template <int V, bool HAD, bool WC, int THREADS>
cudaError_t launch_t(const QuantLaunch& q) {
  const int tpr = 1 << q.tpr_log2;
  const int rpb = THREADS / tpr;
  const int groups = (q.T + rpb - 1) / rpb;
  const int max_blocks = q.num_sms * q.blocks_per_sm;
  const int blocks = groups < max_blocks ? groups : max_blocks;
  quantize_act_kernel<V, HAD, WC, THREADS><<<blocks, THREADS, 0, q.stream>>>(
      reinterpret_cast<const uint4*>(q.x), q.ldx / 8, q.T, q.K / 8, q.tpr_log2, q.alpha, q.gamma,
      q.sa, q.b, q.had_block, q.had_scale, reinterpret_cast<uint32_t*>(q.codes), q.scales);
  return cudaGetLastError();
}

template <int V, bool HAD, bool WC>
cudaError_t launch_v(const QuantLaunch& q) {
  return q.tpr_log2 > 8 ? launch_t<V, HAD, WC, 512>(q) : launch_t<V, HAD, WC, 256>(q);
}

template <bool HAD, bool WC>
cudaError_t launch_hw(const QuantLaunch& q, int V) {
  switch (V) {
    case 1: return launch_v<1, HAD, WC>(q);
    case 2: return launch_v<2, HAD, WC>(q);
    case 3: return launch_v<3, HAD, WC>(q);
    case 4: return launch_v<4, HAD, WC>(q);
    case 5: return launch_v<5, HAD, WC>(q);
    case 6: return launch_v<6, HAD, WC>(q);
    case 7: return launch_v<7, HAD, WC>(q);
    case 8: return launch_v<8, HAD, WC>(q);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

static_assert(512 * kMaxV * 8 >= kMaxK, "a row of kMaxK channels fits 512 threads x kMaxV vectors");

cudaError_t launch_quantize_act(QuantLaunch q, bool write_codes) {
  if (q.alpha < kMinFastAlpha) return launch_quantize_small_alpha(q, write_codes);
  // the asymmetric variant (NEXT-1) lives in the ring kernels only (any K)
  if (q.asym) return launch_quantize_ring(q, write_codes);
  // long rows (every benchmark shape): bulk-TMA ring kernels; short rows: the register-resident
  // kernel below
  if (quantize_ring_supported(q.K)) return launch_quantize_ring(q, write_codes);
  const int nvec = q.K / 8;
  // smallest power-of-two threads-per-row (>= 32) with at most 4 vectors per thread (the fp32 row
  // segment plus the prefetched next segment must leave room for two 256-thread blocks per SM);
  // rows longer than 512 threads x 4 vectors take up to kMaxV vectors per thread
  int tl = 5;
  while (tl < 9 && ((nvec + (1 << tl) - 1) >> tl) > 4) ++tl;
  if (((nvec + (1 << tl) - 1) >> tl) > kMaxV) return cudaErrorInvalidValue;
  q.tpr_log2 = tl;
  const int V = (nvec + (1 << tl) - 1) >> tl;
  if (q.had_block) {
    return write_codes ? launch_hw<true, true>(q, V) : launch_hw<true, false>(q, V);
  }
  return write_codes ? launch_hw<false, true>(q, V) : launch_hw<false, false>(q, V);
}

}  // namespace baseq

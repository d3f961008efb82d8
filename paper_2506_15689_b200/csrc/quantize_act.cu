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

namespace baseq {

namespace {

constexpr int kMaxV = 8;          // 16-byte vectors (8 bf16) a thread keeps in registers

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

// One row = TPR threads; thread r holds vectors r, r + TPR, ..., r + (V-1) TPR of the row.
// A block holds THREADS = max(256, TPR) threads = RPB rows (TPR <= 512 so that 8 vectors of
// fp32 u fit the register file: 512 threads x 128 registers).
template <int V, bool HAD, bool WRITE_CODES, int THREADS>
__global__ void __launch_bounds__(THREADS) quantize_act_kernel(
    const uint4* __restrict__ x, int64_t ldx_vec, int T, int nvec, int tpr_log2,
    float alpha, float gamma, const float* __restrict__ sa, const float* __restrict__ bvec,
    int had_block, float had_scale, uint32_t* __restrict__ codes, float* __restrict__ scales) {
  __shared__ float s_red[THREADS / 32];

  const int tpr = 1 << tpr_log2;
  const int tid = threadIdx.x;
  const int r = tid & (tpr - 1);
  const int row_in_block = tid >> tpr_log2;
  const int rows_per_block = blockDim.x >> tpr_log2;
  const int row = blockIdx.x * rows_per_block + row_in_block;
  const bool row_ok = row < T;
  const int lane = tid & 31;

  float u[V][8];
  float m = 0.0f;

  // ---- pass 1: load (all V loads issued back to back), Hadamard, u = g*h - b, absmax
  uint4 xv[V];
  const uint4* xrow = x + static_cast<int64_t>(row_ok ? row : 0) * ldx_vec;
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int idx = r + i * tpr;
    xv[i] = (row_ok && idx < nvec) ? ptx::ldg_nc_stream(xrow + idx) : make_uint4(0, 0, 0, 0);
  }

#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int idx = r + i * tpr;
    const bool ok = idx < nvec;
    float f[8];
    f[0] = bf16_lo(xv[i].x); f[1] = bf16_hi(xv[i].x);
    f[2] = bf16_lo(xv[i].y); f[3] = bf16_hi(xv[i].y);
    f[4] = bf16_lo(xv[i].z); f[5] = bf16_hi(xv[i].z);
    f[6] = bf16_lo(xv[i].w); f[7] = bf16_hi(xv[i].w);

    if (HAD) {
      // strides 1, 2, 4 inside the thread's 8 contiguous channels
#pragma unroll
      for (int h = 1; h < 8; h <<= 1) {
        if (h < had_block) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            if ((j & h) == 0) {
              const float a = f[j], b2 = f[j + h];
              f[j] = __fadd_rn(a, b2);
              f[j + h] = __fsub_rn(a, b2);
            }
          }
        }
      }
      // strides 8 .. B/2 across lanes: lane l holds vector idx, partner holds idx ^ (h/8).
      // lower lane: a + b = own + other; upper lane: a - b = other - own = fma(own, -1, other).
      for (int h = 8; h < had_block; h <<= 1) {
        const int lm = h >> 3;
        const float sgn = (lane & lm) ? -1.0f : 1.0f;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float other = __shfl_xor_sync(0xffffffffu, f[j], lm);
          f[j] = __fmaf_rn(f[j], sgn, other);
        }
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) f[j] = __fmul_rn(f[j], had_scale);
    }

    float g[8], bb[8];
    if (sa != nullptr && ok) {
      const float4 g0 = __ldg(reinterpret_cast<const float4*>(sa) + 2 * idx);
      const float4 g1 = __ldg(reinterpret_cast<const float4*>(sa) + 2 * idx + 1);
      g[0] = g0.x; g[1] = g0.y; g[2] = g0.z; g[3] = g0.w;
      g[4] = g1.x; g[5] = g1.y; g[6] = g1.z; g[7] = g1.w;
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j) g[j] = gamma;
    }
    if (bvec != nullptr && ok) {
      const float4 b0 = __ldg(reinterpret_cast<const float4*>(bvec) + 2 * idx);
      const float4 b1 = __ldg(reinterpret_cast<const float4*>(bvec) + 2 * idx + 1);
      bb[0] = b0.x; bb[1] = b0.y; bb[2] = b0.z; bb[3] = b0.w;
      bb[4] = b1.x; bb[5] = b1.y; bb[6] = b1.z; bb[7] = b1.w;
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j) bb[j] = 0.0f;
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float uu = ok ? __fmaf_rn(g[j], f[j], -bb[j]) : 0.0f;
      u[i][j] = uu;
      m = fmaxf(m, fabsf(uu));
    }
  }

  // ---- row absmax: warp shuffle, then (TPR > 32) across the row's warps through smem
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (tpr > 32) {
    const int warp = tid >> 5;
    if (lane == 0) s_red[warp] = m;
    __syncthreads();
    const int wpr = tpr >> 5;                      // warps per row
    const int w0 = row_in_block * wpr;
    float mm = s_red[w0];
    for (int w = 1; w < wpr; ++w) mm = fmaxf(mm, s_red[w0 + w]);
    m = mm;
  }

  // ---- Q4, Q5
  const float st = fmaxf(__fdiv_rn(__fmul_rn(alpha, m), 7.0f), 1e-12f);
  const float inv = __fdiv_rn(1.0f, st);
  if (row_ok && r == 0) scales[row] = st;
  if (!WRITE_CODES || !row_ok) return;

  // ---- pass 2: round, clamp, pack, store (one 32-bit word = 8 codes per vector)
  uint32_t* crow = codes + static_cast<int64_t>(row) * nvec;
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int idx = r + i * tpr;
    if (idx < nvec) {
      uint32_t t[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float rr = __fmul_rn(u[i][j], inv);
        rr = fminf(fmaxf(rr, -8.0f), 7.0f);
        // magic add: bits = 0x4B400000 + rne(rr); low nibble = two's-complement code
        t[j] = __float_as_uint(__fadd_rn(rr, 12582912.0f));
      }
      uint32_t p0 = (t[0] & 0xFu) | (t[1] << 4);
      uint32_t p1 = (t[2] & 0xFu) | (t[3] << 4);
      uint32_t p2 = (t[4] & 0xFu) | (t[5] << 4);
      uint32_t p3 = (t[6] & 0xFu) | (t[7] << 4);
      const uint32_t lo = __byte_perm(p0, p1, 0x0040);   // bytes: p0.b0, p1.b0, -, -
      const uint32_t hi = __byte_perm(p2, p3, 0x0040);
      crow[idx] = __byte_perm(lo, hi, 0x5410);           // lo.b0 lo.b1 hi.b0 hi.b1
    }
  }
}

template <int V, bool HAD, bool WC, int THREADS>
cudaError_t launch_t(const QuantLaunch& q) {
  const int tpr = 1 << q.tpr_log2;
  const int rpb = THREADS / tpr;
  const int blocks = (q.T + rpb - 1) / rpb;
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

int quant_max_k() { return 512 * kMaxV * 8; }

cudaError_t launch_quantize_act(QuantLaunch q, bool write_codes) {
  const int nvec = q.K / 8;
  // smallest power-of-two threads-per-row (>= 32) with at most kMaxV vectors per thread
  int tl = 5;
  while (((nvec + (1 << tl) - 1) >> tl) > kMaxV) ++tl;
  if (tl > 9) return cudaErrorInvalidValue;
  if (q.tpr_log2_override >= 5 && q.tpr_log2_override <= 9 &&
      ((nvec + (1 << q.tpr_log2_override) - 1) >> q.tpr_log2_override) <= kMaxV)
    tl = q.tpr_log2_override;
  q.tpr_log2 = tl;
  const int V = (nvec + (1 << tl) - 1) >> tl;
  if (q.had_block) {
    return write_codes ? launch_hw<true, true>(q, V) : launch_hw<true, false>(q, V);
  }
  return write_codes ? launch_hw<false, true>(q, V) : launch_hw<false, false>(q, V);
}

}  // namespace baseq

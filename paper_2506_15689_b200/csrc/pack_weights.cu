// Offline weight packer (step a6 of DESIGN.md).  Untimed: runs once per layer.
//  - re-tiles [N, K/2] int4 nibbles into 128-row x 64-byte boxes so that one (n-tile, k-block)
//    operand of the GEMM is a single contiguous 8 KB bulk-TMA copy;
//  - copies the per-output-channel scales s_w ("per-channel symmetric");
//  - computes the fused bias fb[n] = s_w[n] * sum_k qw[n,k] b[k] + bias[n]  ("fused bias"
//    W R b^c + b of Eq. 14; reading C-3), fp64, k ascending, one thread per
//    output channel so that the summation order is the sequential one.
#include "kernels.cuh"

namespace baseq {
namespace {

__global__ void retile_kernel(const uint8_t* __restrict__ w, int N, int K, int Npad,
                              uint8_t* __restrict__ tiles) {
  // one thread per 16-byte chunk of the destination
  const int kb_count = K / kTileK;
  const int64_t chunks = static_cast<int64_t>(Npad) * (K / 2) / 16;
  const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
  for (int64_t c = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; c < chunks;
       c += stride) {
    // destination chunk c -> (tile, row in tile, 16-byte chunk in the 64-byte row)
    const int64_t tile = c / (kTileBytes / 16);
    const int in_tile = static_cast<int>(c % (kTileBytes / 16));
    const int r = in_tile >> 2, ch = in_tile & 3;
    const int nt = static_cast<int>(tile / kb_count), kb = static_cast<int>(tile % kb_count);
    const int n = nt * kTileRows + r;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (n < N) {
      v = *reinterpret_cast<const uint4*>(w + static_cast<int64_t>(n) * (K / 2) + kb * 64 + ch * 16);
    }
    *reinterpret_cast<uint4*>(tiles + c * 16) = v;
  }
}

__global__ void scales_bias_kernel(const uint8_t* __restrict__ w, const float* __restrict__ w_scale,
                                   const float* __restrict__ b, const float* __restrict__ bias,
                                   int N, int K, int Npad, float* __restrict__ sw_out,
                                   float* __restrict__ fb_out, float* __restrict__ wsum_out,
                                   float* __restrict__ fb_copy) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= Npad) return;
  if (n >= N) {
    sw_out[n] = 0.0f;
    fb_out[n] = 0.0f;
    wsum_out[n] = 0.0f;
    return;
  }
  double s = 0.0;
  int wsum = 0;
  const uint8_t* row = w + static_cast<int64_t>(n) * (K / 2);
  for (int j = 0; j < K / 2; ++j) {
    const uint32_t byte = row[j];
    const int q0 = static_cast<int>(byte << 28) >> 28;        // sign-extend low nibble
    const int q1 = static_cast<int>(byte << 24) >> 28;        // sign-extend high nibble
    wsum += q0 + q1;
    if (b != nullptr) {
      // q * b is exact in fp64, so fma(q, b, s) == s + q*b rounded once (same as the oracle)
      s = __fma_rn(static_cast<double>(q0), static_cast<double>(b[2 * j]), s);
      s = __fma_rn(static_cast<double>(q1), static_cast<double>(b[2 * j + 1]), s);
    }
  }
  wsum_out[n] = static_cast<float>(wsum);                      // exact: |wsum| <= 8 K < 2^24
  double v = __dmul_rn(static_cast<double>(w_scale[n]), s);
  if (bias != nullptr) v = __dadd_rn(v, static_cast<double>(bias[n]));
  const float f = __double2float_rn(v);
  sw_out[n] = w_scale[n];
  fb_out[n] = f;
  if (fb_copy != nullptr) fb_copy[n] = f;
}

__global__ void header_kernel(BlobHeader h, uint32_t* __restrict__ out) {
  // header by value through the kernel parameters: no host staging, no synchronisation
  const uint32_t* src = reinterpret_cast<const uint32_t*>(&h);
  for (int i = threadIdx.x; i < kBlobHeaderBytes / 4; i += 32)
    out[i] = i < static_cast<int>(sizeof(BlobHeader) / 4) ? src[i] : 0u;
}

__global__ void set_fb_kernel(float* __restrict__ fb_out, const float* __restrict__ fb, int N) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < N) fb_out[n] = fb[n];
}

}  // namespace

cudaError_t launch_pack_weights(const uint8_t* w_nibbles, const float* w_scale, const float* b,
                                const float* layer_bias, int N, int K, void* blob,
                                float* fused_bias_out, cudaStream_t stream) {
  const BlobHeader h = blob_header(N, K);
  uint8_t* base = static_cast<uint8_t*>(blob);
  static_assert(sizeof(BlobHeader) <= kBlobHeaderBytes, "header too large");
  header_kernel<<<1, 32, 0, stream>>>(h, reinterpret_cast<uint32_t*>(base));
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const int64_t chunks = static_cast<int64_t>(h.Npad) * (K / 2) / 16;
  const int blocks = static_cast<int>(chunks / 256 < 148 * 16 ? (chunks + 255) / 256 : 148 * 16);
  retile_kernel<<<blocks, 256, 0, stream>>>(w_nibbles, N, K, h.Npad, base + h.off_tiles);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  scales_bias_kernel<<<(h.Npad + 63) / 64, 64, 0, stream>>>(
      w_nibbles, w_scale, b, layer_bias, N, K, h.Npad, reinterpret_cast<float*>(base + h.off_sw),
      reinterpret_cast<float*>(base + h.off_fb), reinterpret_cast<float*>(base + h.off_wsum),
      fused_bias_out);
  return cudaGetLastError();
}

cudaError_t launch_set_fused_bias(void* blob, int N, int K, const float* fb, cudaStream_t stream) {
  const BlobHeader h = blob_header(N, K);
  uint8_t* base = static_cast<uint8_t*>(blob);
  set_fb_kernel<<<(N + 255) / 256, 256, 0, stream>>>(reinterpret_cast<float*>(base + h.off_fb), fb, N);
  return cudaGetLastError();
}

}  // namespace baseq

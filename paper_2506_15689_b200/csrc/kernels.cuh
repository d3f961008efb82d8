// Internal launch interfaces between baseq_api.cu and the kernel translation units.
#pragma once
#include <atomic>
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

namespace baseq {

constexpr int kMaxDevices = 64;        // per-device host state (attributes set, status word) is indexed by device
constexpr int kMaxK = 32768;           // library-wide bound on K (include/baseq.h, shape rules)
constexpr unsigned int kStatusBadBlob = 1u;   // status-word bit: a GEMM found a blob header != its (N, K)

// Raises a kernel's dynamic shared-memory limit once per device (thread-safe; setting the attribute
// twice from two racing threads is harmless).  `slots` is one zero-initialised array per kernel.
template <typename Kern>
inline cudaError_t ensure_dynamic_smem(Kern kern, int bytes, int device, std::atomic<int>* slots) {
  if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
  if (slots[device].load(std::memory_order_acquire) >= bytes) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  int cur = slots[device].load(std::memory_order_relaxed);
  while (cur < bytes && !slots[device].compare_exchange_weak(cur, bytes, std::memory_order_release)) {
  }
  return cudaSuccess;
}

// ------------------------------------------------------------------ packed weight blob
// [ header 128 B | s_w[Npad] f32 | fb[Npad] f32 | wsum[Npad] f32 | boxes ]
// wsum[n] = sum_k qw[n,k] (an exact integer, |wsum| <= 8 K < 2^24, stored as fp32): the term the
// lattice lower bound z_t of the asymmetric activation quantiser multiplies (NEXT-1).
// boxes: [Npad/kTileRows][K/128] boxes of kTileRows rows x 64 bytes (= 128 int4 along K),
// row-major inside the box, so one (row group, k-block) box is contiguous and consecutive
// k-blocks of one row group are adjacent -- each is fetched with a single bulk-TMA copy.
// kTileRows = half a GEMM tile's N extent: each CTA of a CTA pair streams one row group.
// Npad = N rounded up to the tile's N extent (zero rows), so no partial B load exists.
constexpr uint32_t kBlobMagic = 0x51534142u;   // "BASQ"
constexpr int kBlobHeaderBytes = 128;
constexpr int kGemmBN = 192;                   // output channels per GEMM tile (UMMA N)
constexpr int kTileRows = kGemmBN / 2;         // rows per weight box
constexpr int kTileK = 128;                    // int4 elements along K per box
constexpr int kTileBytes = kTileRows * kTileK / 2;

struct BlobHeader {
  uint32_t magic;
  int32_t N, K, Npad;
  uint64_t off_sw, off_fb, off_wsum, off_tiles, total_bytes;
};

inline int blob_npad(int N) { return (N + kGemmBN - 1) / kGemmBN * kGemmBN; }
inline size_t blob_bytes(int N, int K) {
  const size_t npad = static_cast<size_t>(blob_npad(N));
  return kBlobHeaderBytes + npad * 4 * 3 + npad * static_cast<size_t>(K) / 2;
}
inline BlobHeader blob_header(int N, int K) {
  BlobHeader h{};
  h.magic = kBlobMagic;
  h.N = N;
  h.K = K;
  h.Npad = blob_npad(N);
  h.off_sw = kBlobHeaderBytes;
  h.off_fb = h.off_sw + static_cast<uint64_t>(h.Npad) * 4;
  h.off_wsum = h.off_fb + static_cast<uint64_t>(h.Npad) * 4;
  h.off_tiles = h.off_wsum + static_cast<uint64_t>(h.Npad) * 4;
  h.total_bytes = blob_bytes(N, K);
  return h;
}

// ------------------------------------------------------------------ activation quantiser
struct QuantLaunch {
  const void* x;       // bf16 [T, ldx]
  int64_t ldx;
  int T, K;
  float alpha, gamma;
  const float* sa;
  const float* b;
  int had_block;
  float had_scale;     // (float)(1 / sqrt((double)had_block)), computed on the host
  uint8_t* codes;      // [T, K/2]
  float* scales;       // [T]
  float* zeros;        // [T] lattice lower bounds z_t (asymmetric variant), else nullptr
  bool asym;           // NEXT-1: per-token asymmetric int4 (unsigned codes)
  cudaStream_t stream;
  int tpr_log2;            // filled by the launcher
  int num_sms;             // persistent grid = num_sms * blocks_per_sm
  int device;              // current device ordinal (per-device attribute cache)
  int blocks_per_sm;
};
cudaError_t launch_quantize_act(QuantLaunch q, bool write_codes);
// alpha < kMinFastAlpha: the fast kernels' single-fma rounding needs |u / s_t| < 2^22; a plain kernel
// that clamps first takes over (quantize_small_alpha.cu)
constexpr float kMinFastAlpha = 1.0f / 65536.0f;
cudaError_t launch_quantize_small_alpha(const QuantLaunch& q, bool write_codes);
// long rows (K >= 4096): bulk-TMA ring variant of the same contract (quantize_ring.cu)
bool quantize_ring_supported(int K);
cudaError_t launch_quantize_ring(const QuantLaunch& q, bool write_codes);

// NEXT-2: the block-128 Hadamard on the tensor cores (quantize_had_tc.cu); tolerance parity
bool quantize_tc_supported(int K, int had_block);
cudaError_t launch_quantize_tc(const QuantLaunch& q);

// ------------------------------------------------------------------ KV-cache quantiser (NEXT-3)
struct KvLaunch {
  const void* x;        // bf16 [T, ldx], row t = heads blocks of head_dim channels
  int64_t ldx;
  int T, heads, head_dim;
  float alpha;
  uint8_t* codes;       // [T, heads * head_dim / 2] unsigned nibbles
  float* scales;        // [T, heads]
  float* zeros;         // [T, heads]
  int num_sms;
  cudaStream_t stream;
};
cudaError_t launch_quantize_kv(const KvLaunch& q);   // cudaErrorNotSupported: head_dim not 64 / 128
cudaError_t launch_quantize_kv_small_alpha(const KvLaunch& q);

cudaError_t launch_pack_weights(const uint8_t* w_nibbles, const float* w_scale, const float* b,
                                const float* layer_bias, int N, int K, void* blob,
                                float* fused_bias_out, cudaStream_t stream);
cudaError_t launch_set_fused_bias(void* blob, int N, int K, const float* fb, cudaStream_t stream);

// ------------------------------------------------------------------ GEMM
struct GemmLaunch {
  const uint8_t* codes;    // [T, K/2]   (unfused) or nullptr (fused)
  const float* scales;     // [T]
  const float* zeros;      // [T] asymmetric variant (unsigned codes), else nullptr
  const void* blob;
  int T, N, K;
  void* y;                 // bf16 [T, ldy]
  int64_t ldy;
  int32_t* acc_dump;       // optional [T, N]
  // fused single-launch variant (x != nullptr selects it): the background quantiser's inputs
  const void* x;
  int64_t ldx;
  float alpha, gamma;
  const float* sa;
  const float* b;
  int had_block;
  float had_scale;
  uint8_t* codes_dump;     // optional [T, K/2]
  void* workspace;         // fused variant: baseq_fused_workspace_bytes(T, N, K) bytes
  cudaStream_t stream;
  int num_sms;
  int device;              // current device ordinal
  unsigned int* status_word;   // this device's status word (kStatusBadBlob)
};
// Returns cudaSuccess, or an error (cudaErrorNotSupported when the tensor map cannot be built).
cudaError_t launch_w4a4_gemm(const GemmLaunch& g);
// Fused variant (a10): GEMM with background quantiser warps, one launch; g.x != nullptr,
// g.scales = scales_out (g.zeros = zeros_out selects asymmetric codes).
size_t fused_workspace_bytes(int T, int N, int K);
bool fused_supported(int had_block);
cudaError_t launch_linear_fused(const GemmLaunch& g);
// Decode shapes (NEXT-4, w4a4_decode.cu): the same contract and the same bits for T <= kDecodeMaxT,
// bound by streaming the packed weights once; launch_w4a4_gemm routes the unfused calls there.
constexpr int kDecodeMaxT = 64;
cudaError_t launch_w4a4_decode(const GemmLaunch& g);

}  // namespace baseq

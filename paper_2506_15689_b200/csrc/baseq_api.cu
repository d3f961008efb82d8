// extern "C" entry points of libbaseq (include/baseq.h): host-side validation + dispatch.
// No compute happens here and nothing falls back to the CPU.
#include <cmath>
#include <cstring>
#include <mutex>

#include "../../include/baseq.h"
#include "kernels.cuh"

namespace {

using namespace baseq;

// One word per device (a __device__ variable exists once per context): bit 0 is raised by a GEMM
// kernel that finds a packed-weight header not matching its (N, K) arguments.
__device__ unsigned int g_status_word;

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// Per-device state, filled once per device under std::call_once (any number of host threads, any
// number of GPUs in one process): compute capability, SM count, and the address of this device's
// copy of the library's status word (see baseq_sync_status).
struct DeviceState {
  std::once_flag once;
  baseq_status_t st = BASEQ_ERR_CUDA;
  int num_sms = 0;
  unsigned int* status_word = nullptr;
};
DeviceState g_dev[kMaxDevices];

struct DeviceRef {
  int device = 0;
  int num_sms = 0;
  unsigned int* status_word = nullptr;
};

baseq_status_t device_check(DeviceRef* out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return BASEQ_ERR_CUDA;
  if (dev < 0 || dev >= kMaxDevices) return BASEQ_ERR_UNSUPPORTED;
  DeviceState& d = g_dev[dev];
  std::call_once(d.once, [&d, dev]() {
    int major = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return;
    if (major != 10) {
      d.st = BASEQ_ERR_UNSUPPORTED;
      return;
    }
    void* sym = nullptr;
    if (cudaGetSymbolAddress(&sym, g_status_word) != cudaSuccess) return;
    d.status_word = static_cast<unsigned int*>(sym);
    d.num_sms = sms;
    d.st = BASEQ_OK;
  });
  if (d.st != BASEQ_OK) return d.st;
  if (out) {
    out->device = dev;
    out->num_sms = d.num_sms;
    out->status_word = d.status_word;
  }
  return BASEQ_OK;
}

// K <= 32768 everywhere: a whole row stays in one CTA (quantiser), and the GEMM's raw accumulator
// 256 * acc stays inside int32 (|256 * 64 * K| = 2^29 symmetric, |256 * 120 * K| < 2^30 asymmetric).
baseq_status_t check_shape(int T, int N, int K) {
  if (T < 1) return BASEQ_ERR_SHAPE;
  if (K < 128 || (K % 128) != 0 || K > kMaxK) return BASEQ_ERR_SHAPE;
  if (N < 8 || (N % 8) != 0) return BASEQ_ERR_SHAPE;
  return BASEQ_OK;
}

baseq_status_t check_act_params(const baseq_act_params_t* p, int K) {
  if (p == nullptr) return BASEQ_ERR_NULL;
  if (!(p->alpha > 0.0f) || !(p->alpha <= 1.0f)) return BASEQ_ERR_PARAM;
  if (p->sa == nullptr && (!(p->gamma > 0.0f) || !std::isfinite(p->gamma))) return BASEQ_ERR_PARAM;
  if (p->had_block != 0) {
    const int B = p->had_block;
    if (B < 2 || B > 256 || (B & (B - 1)) != 0 || (K % B) != 0) return BASEQ_ERR_PARAM;
  }
  if (p->sa != nullptr && !aligned(p->sa, 16)) return BASEQ_ERR_ALIGN;
  if (p->b != nullptr && !aligned(p->b, 16)) return BASEQ_ERR_ALIGN;
  return BASEQ_OK;
}

QuantLaunch make_quant(const void* x, int64_t ldx, int T, int K, const baseq_act_params_t* p,
                       uint8_t* codes, float* scales, void* stream) {
  QuantLaunch q{};
  q.x = x;
  q.ldx = ldx;
  q.T = T;
  q.K = K;
  q.alpha = p->alpha;
  q.gamma = p->gamma;
  q.sa = p->sa;
  q.b = p->b;
  q.had_block = p->had_block;
  q.had_scale = p->had_block
                    ? static_cast<float>(1.0 / std::sqrt(static_cast<double>(p->had_block)))
                    : 1.0f;
  q.codes = codes;
  q.scales = scales;
  q.stream = static_cast<cudaStream_t>(stream);
  q.tpr_log2 = 0;
  q.zeros = nullptr;
  q.asym = false;
  q.num_sms = 148;          // overwritten by the callers from the device query
  q.device = 0;
  q.blocks_per_sm = 2;
  return q;
}

}  // namespace

extern "C" {

const char* baseq_status_string(baseq_status_t s) {
  switch (s) {
    case BASEQ_OK: return "BASEQ_OK";
    case BASEQ_ERR_NULL: return "BASEQ_ERR_NULL: a required pointer is NULL";
    case BASEQ_ERR_SHAPE: return "BASEQ_ERR_SHAPE: need T >= 1, K % 128 == 0, 128 <= K <= 32768, N % 8 == 0";
    case BASEQ_ERR_ALIGN: return "BASEQ_ERR_ALIGN: pointer or leading dimension misaligned";
    case BASEQ_ERR_PARAM: return "BASEQ_ERR_PARAM: alpha / gamma / had_block out of range";
    case BASEQ_ERR_WORKSPACE: return "BASEQ_ERR_WORKSPACE: workspace too small, or a packed blob did not match (N, K)";
    case BASEQ_ERR_UNSUPPORTED: return "BASEQ_ERR_UNSUPPORTED: requires an sm_100 (B200) device, or the combination is not built";
    case BASEQ_ERR_CUDA: return "BASEQ_ERR_CUDA: a CUDA call failed";
  }
  return "BASEQ: unknown status";
}

int baseq_version(void) { return 2; }

baseq_status_t baseq_sync_status(void* stream) {
  DeviceRef d;
  const baseq_status_t st = device_check(&d);
  if (st != BASEQ_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  unsigned int word = 0;
  if (cudaMemcpyAsync(&word, d.status_word, sizeof word, cudaMemcpyDeviceToHost, s) != cudaSuccess)
    return BASEQ_ERR_CUDA;
  if (cudaMemsetAsync(d.status_word, 0, sizeof word, s) != cudaSuccess) return BASEQ_ERR_CUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return BASEQ_ERR_CUDA;
  return (word & kStatusBadBlob) ? BASEQ_ERR_WORKSPACE : BASEQ_OK;
}

size_t baseq_packed_weight_bytes(int N, int K) {
  if (check_shape(1, N, K) != BASEQ_OK) return 0;
  return blob_bytes(N, K);
}

baseq_status_t baseq_pack_weights(const uint8_t* w_nibbles, const float* w_scale, const float* b,
                                  const float* layer_bias, int N, int K, void* packed_out,
                                  float* fused_bias_out, void* stream) {
  if (w_nibbles == nullptr || w_scale == nullptr || packed_out == nullptr) return BASEQ_ERR_NULL;
  baseq_status_t st = check_shape(1, N, K);
  if (st != BASEQ_OK) return st;
  if (!aligned(w_nibbles, 16) || !aligned(packed_out, 128)) return BASEQ_ERR_ALIGN;
  st = device_check(nullptr);
  if (st != BASEQ_OK) return st;
  const cudaError_t e = launch_pack_weights(w_nibbles, w_scale, b, layer_bias, N, K, packed_out,
                                            fused_bias_out, static_cast<cudaStream_t>(stream));
  return e == cudaSuccess ? BASEQ_OK : BASEQ_ERR_CUDA;
}

baseq_status_t baseq_set_fused_bias(void* packed, int N, int K, const float* fb, void* stream) {
  if (packed == nullptr || fb == nullptr) return BASEQ_ERR_NULL;
  baseq_status_t st = check_shape(1, N, K);
  if (st != BASEQ_OK) return st;
  if (!aligned(packed, 128)) return BASEQ_ERR_ALIGN;
  st = device_check(nullptr);
  if (st != BASEQ_OK) return st;
  const cudaError_t e = launch_set_fused_bias(packed, N, K, fb, static_cast<cudaStream_t>(stream));
  return e == cudaSuccess ? BASEQ_OK : BASEQ_ERR_CUDA;
}

namespace {

// Everything baseq_quantize_act / _asym check, without launching: shared with the entry points that
// call them after having enqueued other work (fused, host), so that a failing call enqueues nothing.
baseq_status_t validate_quant(const void* x, int64_t ldx, int T, int K, const baseq_act_params_t* p,
                              const void* codes, const void* scales, bool need_codes) {
  baseq_status_t st = check_shape(T, 8, K);     // empty input is a shape error
  if (st != BASEQ_OK) return st;
  if (x == nullptr || scales == nullptr || p == nullptr || (need_codes && codes == nullptr))
    return BASEQ_ERR_NULL;
  st = check_act_params(p, K);
  if (st != BASEQ_OK) return st;
  if (!aligned(x, 16) || !aligned(codes, 16) || !aligned(scales, 4)) return BASEQ_ERR_ALIGN;
  if (ldx < K || (ldx % 8) != 0) return BASEQ_ERR_ALIGN;
  return BASEQ_OK;
}

baseq_status_t validate_gemm(const void* codes, const void* scales, const void* packed_w, int T, int N,
                             int K, const void* y, int64_t ldy, const void* acc_dump, bool need_codes) {
  if ((need_codes && codes == nullptr) || scales == nullptr || packed_w == nullptr || y == nullptr)
    return BASEQ_ERR_NULL;
  const baseq_status_t st = check_shape(T, N, K);
  if (st != BASEQ_OK) return st;
  if (!aligned(codes, 16) || !aligned(y, 16) || !aligned(packed_w, 128)) return BASEQ_ERR_ALIGN;
  if (acc_dump != nullptr && !aligned(acc_dump, 16)) return BASEQ_ERR_ALIGN;
  if (ldy < N || (ldy % 8) != 0) return BASEQ_ERR_ALIGN;
  return BASEQ_OK;
}

baseq_status_t from_cuda(cudaError_t e) {
  if (e == cudaErrorNotSupported) return BASEQ_ERR_UNSUPPORTED;
  return e == cudaSuccess ? BASEQ_OK : BASEQ_ERR_CUDA;
}

GemmLaunch make_gemm(const uint8_t* codes, const float* scales, const float* zeros, const void* packed_w,
                     int T, int N, int K, void* y, int64_t ldy, int32_t* acc_dump, void* stream,
                     const DeviceRef& d) {
  GemmLaunch g{};
  g.codes = codes;
  g.scales = scales;
  g.zeros = zeros;
  g.blob = packed_w;
  g.T = T;
  g.N = N;
  g.K = K;
  g.y = y;
  g.ldy = ldy;
  g.acc_dump = acc_dump;
  g.stream = static_cast<cudaStream_t>(stream);
  g.num_sms = d.num_sms;
  g.device = d.device;
  g.status_word = d.status_word;
  return g;
}

}  // namespace

baseq_status_t baseq_quantize_act(const void* x_bf16, int64_t ldx, int T, int K,
                                  const baseq_act_params_t* p, uint8_t* codes, float* scales,
                                  void* stream) {
  baseq_status_t st = validate_quant(x_bf16, ldx, T, K, p, codes, scales, true);
  if (st != BASEQ_OK) return st;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  QuantLaunch q = make_quant(x_bf16, ldx, T, K, p, codes, scales, stream);
  q.num_sms = d.num_sms;
  q.device = d.device;
  return from_cuda(launch_quantize_act(q, true));
}

baseq_status_t baseq_quantize_act_tc(const void* x_bf16, int64_t ldx, int T, int K,
                                     const baseq_act_params_t* p, uint8_t* codes, float* scales,
                                     void* stream) {
  baseq_status_t st = validate_quant(x_bf16, ldx, T, K, p, codes, scales, true);
  if (st != BASEQ_OK) return st;
  if (!quantize_tc_supported(K, p->had_block) || p->alpha < kMinFastAlpha) return BASEQ_ERR_UNSUPPORTED;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  QuantLaunch q = make_quant(x_bf16, ldx, T, K, p, codes, scales, stream);
  q.num_sms = d.num_sms;
  q.device = d.device;
  return from_cuda(launch_quantize_tc(q));
}

baseq_status_t baseq_w4a4_gemm(const uint8_t* codes, const float* scales, const void* packed_w,
                               int T, int N, int K, void* y_bf16, int64_t ldy, int32_t* acc_dump,
                               void* stream) {
  baseq_status_t st = validate_gemm(codes, scales, packed_w, T, N, K, y_bf16, ldy, acc_dump, true);
  if (st != BASEQ_OK) return st;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  return from_cuda(launch_w4a4_gemm(
      make_gemm(codes, scales, nullptr, packed_w, T, N, K, y_bf16, ldy, acc_dump, stream, d)));
}

baseq_status_t baseq_quantize_act_asym(const void* x_bf16, int64_t ldx, int T, int K,
                                       const baseq_act_params_t* p, uint8_t* codes, float* scales,
                                       float* zeros, void* stream) {
  baseq_status_t st = validate_quant(x_bf16, ldx, T, K, p, codes, scales, true);
  if (st != BASEQ_OK) return st;
  if (zeros == nullptr) return BASEQ_ERR_NULL;
  if (!aligned(zeros, 4)) return BASEQ_ERR_ALIGN;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  QuantLaunch q = make_quant(x_bf16, ldx, T, K, p, codes, scales, stream);
  q.num_sms = d.num_sms;
  q.device = d.device;
  q.zeros = zeros;
  q.asym = true;
  return from_cuda(launch_quantize_act(q, true));
}

baseq_status_t baseq_w4a4_gemm_asym(const uint8_t* codes, const float* scales, const float* zeros,
                                    const void* packed_w, int T, int N, int K, void* y_bf16,
                                    int64_t ldy, int32_t* acc_dump, void* stream) {
  if (zeros == nullptr) return BASEQ_ERR_NULL;
  baseq_status_t st = validate_gemm(codes, scales, packed_w, T, N, K, y_bf16, ldy, acc_dump, true);
  if (st != BASEQ_OK) return st;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  return from_cuda(launch_w4a4_gemm(
      make_gemm(codes, scales, zeros, packed_w, T, N, K, y_bf16, ldy, acc_dump, stream, d)));
}

baseq_status_t baseq_quantize_kv(const void* x_bf16, int64_t ldx, int T, int n_heads, int head_dim,
                                 float alpha, uint8_t* codes, float* scales, float* zeros,
                                 void* stream) {
  if (x_bf16 == nullptr || codes == nullptr || scales == nullptr || zeros == nullptr)
    return BASEQ_ERR_NULL;
  if (T < 1 || n_heads < 1 || n_heads > 65536 || T > (1 << 24)) return BASEQ_ERR_SHAPE;
  if (head_dim != 64 && head_dim != 128) return BASEQ_ERR_UNSUPPORTED;
  if (!(alpha > 0.0f && alpha <= 1.0f)) return BASEQ_ERR_PARAM;
  if (!aligned(x_bf16, 16) || !aligned(codes, 16) || !aligned(scales, 4) || !aligned(zeros, 4))
    return BASEQ_ERR_ALIGN;
  if (ldx < static_cast<int64_t>(n_heads) * head_dim || (ldx % 8) != 0) return BASEQ_ERR_ALIGN;
  DeviceRef d;
  const baseq_status_t st = device_check(&d);
  if (st != BASEQ_OK) return st;
  KvLaunch q{};
  q.x = x_bf16;
  q.ldx = ldx;
  q.T = T;
  q.heads = n_heads;
  q.head_dim = head_dim;
  q.alpha = alpha;
  q.codes = codes;
  q.scales = scales;
  q.zeros = zeros;
  q.num_sms = d.num_sms;
  q.stream = static_cast<cudaStream_t>(stream);
  return from_cuda(launch_quantize_kv(q));
}

size_t baseq_fused_workspace_bytes(int T, int N, int K) {
  if (check_shape(T, N, K) != BASEQ_OK) return 0;
  return fused_workspace_bytes(T, N, K);
}

baseq_status_t baseq_linear_fused(const void* x_bf16, int64_t ldx, int T, int K,
                                  const baseq_act_params_t* p, const void* packed_w, int N,
                                  void* y_bf16, int64_t ldy, void* workspace, size_t workspace_bytes,
                                  uint8_t* codes_dump, float* scales_out, int32_t* acc_dump,
                                  void* stream) {
  // every check of both stages first: a failing call enqueues nothing
  if (workspace == nullptr) return BASEQ_ERR_NULL;
  baseq_status_t st = validate_quant(x_bf16, ldx, T, K, p, codes_dump, scales_out, false);
  if (st != BASEQ_OK) return st;
  st = validate_gemm(nullptr, scales_out, packed_w, T, N, K, y_bf16, ldy, acc_dump, false);
  if (st != BASEQ_OK) return st;
  if (!aligned(workspace, 256)) return BASEQ_ERR_ALIGN;
  if (workspace_bytes < baseq_fused_workspace_bytes(T, N, K)) return BASEQ_ERR_WORKSPACE;
  if (!fused_supported(p->had_block)) return BASEQ_ERR_UNSUPPORTED;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  GemmLaunch g = make_gemm(nullptr, scales_out, nullptr, packed_w, T, N, K, y_bf16, ldy, acc_dump, stream, d);
  g.x = x_bf16;
  g.ldx = ldx;
  g.alpha = p->alpha;
  g.gamma = p->gamma;
  g.sa = p->sa;
  g.b = p->b;
  g.had_block = p->had_block;
  g.had_scale = p->had_block
                    ? static_cast<float>(1.0 / std::sqrt(static_cast<double>(p->had_block)))
                    : 1.0f;
  g.codes_dump = codes_dump;
  g.workspace = workspace;
  return from_cuda(launch_linear_fused(g));
}

baseq_status_t baseq_linear_fused_asym(const void* x_bf16, int64_t ldx, int T, int K,
                                       const baseq_act_params_t* p, const void* packed_w, int N,
                                       void* y_bf16, int64_t ldy, void* workspace, size_t workspace_bytes,
                                       uint8_t* codes_dump, float* scales_out, float* zeros_out,
                                       int32_t* acc_dump, void* stream) {
  if (workspace == nullptr || zeros_out == nullptr) return BASEQ_ERR_NULL;
  baseq_status_t st = validate_quant(x_bf16, ldx, T, K, p, codes_dump, scales_out, false);
  if (st != BASEQ_OK) return st;
  st = validate_gemm(nullptr, scales_out, packed_w, T, N, K, y_bf16, ldy, acc_dump, false);
  if (st != BASEQ_OK) return st;
  if (!aligned(workspace, 256) || !aligned(zeros_out, 4)) return BASEQ_ERR_ALIGN;
  if (workspace_bytes < baseq_fused_workspace_bytes(T, N, K)) return BASEQ_ERR_WORKSPACE;
  if (!fused_supported(p->had_block)) return BASEQ_ERR_UNSUPPORTED;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  GemmLaunch g = make_gemm(nullptr, scales_out, zeros_out, packed_w, T, N, K, y_bf16, ldy, acc_dump, stream, d);
  g.x = x_bf16;
  g.ldx = ldx;
  g.alpha = p->alpha;
  g.gamma = p->gamma;
  g.sa = p->sa;
  g.b = p->b;
  g.had_block = p->had_block;
  g.had_scale = p->had_block
                    ? static_cast<float>(1.0 / std::sqrt(static_cast<double>(p->had_block)))
                    : 1.0f;
  g.codes_dump = codes_dump;
  g.workspace = workspace;
  return from_cuda(launch_linear_fused(g));
}

size_t baseq_linear_host_scratch_bytes(int T, int N, int K) {
  if (check_shape(T, N, K) != BASEQ_OK) return 0;
  auto up = [](size_t v) { return (v + 255) / 256 * 256; };
  return up(static_cast<size_t>(T) * K * 2) + up(static_cast<size_t>(T) * K / 2) +
         up(static_cast<size_t>(T) * 4) + up(static_cast<size_t>(T) * N * 2);
}

baseq_status_t baseq_linear_host(const void* x_bf16_host, int T, int K, const baseq_act_params_t* p,
                                 const void* packed_w, int N, void* y_bf16_host, void* dev_scratch,
                                 size_t dev_scratch_bytes, void* stream) {
  if (x_bf16_host == nullptr || y_bf16_host == nullptr || dev_scratch == nullptr ||
      packed_w == nullptr || p == nullptr)
    return BASEQ_ERR_NULL;
  baseq_status_t st = check_shape(T, N, K);
  if (st != BASEQ_OK) return st;
  if (dev_scratch_bytes < baseq_linear_host_scratch_bytes(T, N, K)) return BASEQ_ERR_WORKSPACE;
  if (!aligned(dev_scratch, 256) || !aligned(packed_w, 128)) return BASEQ_ERR_ALIGN;
  auto up = [](size_t v) { return (v + 255) / 256 * 256; };
  uint8_t* base = static_cast<uint8_t*>(dev_scratch);
  void* dx = base;
  uint8_t* dcodes = base + up(static_cast<size_t>(T) * K * 2);
  float* dscales = reinterpret_cast<float*>(dcodes + up(static_cast<size_t>(T) * K / 2));
  void* dy = reinterpret_cast<uint8_t*>(dscales) + up(static_cast<size_t>(T) * 4);
  // every check of the two nested calls before the first copy is enqueued
  st = validate_quant(dx, K, T, K, p, dcodes, dscales, true);
  if (st != BASEQ_OK) return st;
  st = validate_gemm(dcodes, dscales, packed_w, T, N, K, dy, N, nullptr, true);
  if (st != BASEQ_OK) return st;
  st = device_check(nullptr);
  if (st != BASEQ_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (cudaMemcpyAsync(dx, x_bf16_host, static_cast<size_t>(T) * K * 2, cudaMemcpyHostToDevice, s) !=
      cudaSuccess)
    return BASEQ_ERR_CUDA;
  st = baseq_quantize_act(dx, K, T, K, p, dcodes, dscales, stream);
  if (st != BASEQ_OK) return st;
  st = baseq_w4a4_gemm(dcodes, dscales, packed_w, T, N, K, dy, N, nullptr, stream);
  if (st != BASEQ_OK) return st;
  if (cudaMemcpyAsync(y_bf16_host, dy, static_cast<size_t>(T) * N * 2, cudaMemcpyDeviceToHost, s) !=
      cudaSuccess)
    return BASEQ_ERR_CUDA;
  return BASEQ_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ baseq_linear_static (no allocation)
// The two-kernel linear needs scratch between its kernels: the int4 codes [T, K/2] and the
// per-token scales [T].  Callers that cannot allocate (CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc) get that scratch from this file-scope array: kStaticCodesBytes of codes
// followed by kStaticMaxT scales.  Every GPU that loads the library holds it until the process
// exits.  In host code `g_static_scratch` is only a host-side stand-in for the symbol, never a
// device address: the address comes from cudaGetSymbolAddress, once per device with that device
// current, and is what the kernels receive.
constexpr size_t kStaticCodesBytes = size_t(4) << 20;   // T * K / 2 <= 4 MiB (c2: 2048 x 4096)
constexpr int kStaticMaxT = 8192;                        // scales: 32 KiB
constexpr size_t kStaticScratchBytes = kStaticCodesBytes + size_t(kStaticMaxT) * sizeof(float);
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {

struct StaticScratchState {
  std::once_flag once;
  cudaError_t err = cudaErrorUnknown;
  unsigned char* ptr = nullptr;
};
StaticScratchState g_static_state[kMaxDevices];

// device_check() has run: `dev` is the current device and inside [0, kMaxDevices)
baseq_status_t static_scratch(int dev, unsigned char** out) {
  StaticScratchState& s = g_static_state[dev];
  std::call_once(s.once, [&s]() {
    void* sym = nullptr;
    s.err = cudaGetSymbolAddress(&sym, g_static_scratch);
    if (s.err == cudaSuccess) s.ptr = static_cast<unsigned char*>(sym);
  });
  if (s.err != cudaSuccess || s.ptr == nullptr) return BASEQ_ERR_CUDA;
  *out = s.ptr;
  return BASEQ_OK;
}

}  // namespace

extern "C" {

size_t baseq_linear_static_scratch_bytes(void) { return kStaticScratchBytes; }

baseq_status_t baseq_linear_static(const void* x_bf16, int64_t ldx, int T, int K,
                                   const baseq_act_params_t* p, const void* packed_w, int N,
                                   void* y_bf16, int64_t ldy, void* stream) {
  if (x_bf16 == nullptr || y_bf16 == nullptr || packed_w == nullptr || p == nullptr)
    return BASEQ_ERR_NULL;
  baseq_status_t st = check_shape(T, N, K);
  if (st != BASEQ_OK) return st;
  // beyond the static array: a clear error, nothing enqueued
  if (T > kStaticMaxT || static_cast<size_t>(T) * K / 2 > kStaticCodesBytes) return BASEQ_ERR_WORKSPACE;
  DeviceRef d;
  st = device_check(&d);
  if (st != BASEQ_OK) return st;
  unsigned char* base = nullptr;
  st = static_scratch(d.device, &base);
  if (st != BASEQ_OK) return st;
  uint8_t* codes = base;
  float* scales = reinterpret_cast<float*>(base + kStaticCodesBytes);
  // every check of both stages before the first launch
  st = validate_quant(x_bf16, ldx, T, K, p, codes, scales, true);
  if (st != BASEQ_OK) return st;
  st = validate_gemm(codes, scales, packed_w, T, N, K, y_bf16, ldy, nullptr, true);
  if (st != BASEQ_OK) return st;
  // Nothing in the scratch has to start at zero: the quantiser writes all T rows of codes and
  // scales before the GEMM reads them, and the GEMM reads no row >= T (its tensor map ends at T).
  QuantLaunch q = make_quant(x_bf16, ldx, T, K, p, codes, scales, stream);
  q.num_sms = d.num_sms;
  q.device = d.device;
  st = from_cuda(launch_quantize_act(q, true));
  if (st != BASEQ_OK) return st;
  return from_cuda(launch_w4a4_gemm(
      make_gemm(codes, scales, nullptr, packed_w, T, N, K, y_bf16, ldy, nullptr, stream, d)));
}

}  // extern "C"

// The epilogue's arithmetic contract (DESIGN.md section 2 / C-9, section 6.6 A4) as the fp64
// expressions themselves, written once and used by the tcgen05 GEMM (w4a4_gemm.cu: the fix-up of
// elements its fp32 bracket does not settle) and by the decode GEMM (w4a4_decode.cu: every output).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace baseq {
namespace epi {

__device__ __forceinline__ uint32_t bf16_from_double_rne(double v) {
  // round-to-odd to fp32 (keeps a sticky bit), then RNE to bf16: a single rounding overall
  float f = __double2float_rz(v);
  uint32_t u = __float_as_uint(f);
  if (static_cast<double>(f) != v) u |= 1u;
  const uint32_t r = u + 0x7FFFu + ((u >> 16) & 1u);
  return r >> 16;
}

// Y = bf16_rne( fma((double)s_t * (double)s_w, (double)acc, (double)fb) )
__device__ __forceinline__ uint32_t dequant_f64(int32_t acc, float st, float sw, float fb) {
  const double pd = __dmul_rn(static_cast<double>(st), static_cast<double>(sw));
  const double yd = __fma_rn(pd, static_cast<double>(acc), static_cast<double>(fb));
  return bf16_from_double_rne(yd);
}

// Asymmetric variant (NEXT-1): yd = fma(s_t s_w, acc, fma(z_t s_w, wsum, fb)) with acc = sum_k q w
// over the UNSIGNED codes; `acc_c` is the accumulator over the re-centred codes q - 8 (what the
// MMA produces), acc = acc_c + 8 wsum exactly.
__device__ __forceinline__ uint32_t dequant_f64_asym(int32_t acc_c, float st, float zt, float sw,
                                                     float fb, float ws) {
  const int32_t acc = acc_c + 8 * static_cast<int32_t>(ws);
  const double swd = static_cast<double>(sw);
  const double c = __fma_rn(__dmul_rn(static_cast<double>(zt), swd), static_cast<double>(ws),
                            static_cast<double>(fb));
  const double yd = __fma_rn(__dmul_rn(static_cast<double>(st), swd), static_cast<double>(acc), c);
  return bf16_from_double_rne(yd);
}

}  // namespace epi
}  // namespace baseq

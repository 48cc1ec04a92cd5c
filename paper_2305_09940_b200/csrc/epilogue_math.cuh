// epilogue_math.cuh — elementwise math of the fused epilogues (device only).
// gelu / gelu' in the tanh form (reading S2):
//   gelu(z)  = 1/2 z (1 + tanh u),  u = c (z + a z^3)
//   gelu'(z) = 1/2 (1 + tanh u) + 1/2 z (1 - tanh^2 u) c (1 + 3 a z^2)
#pragma once
#include "common.cuh"

namespace osdp {

// Precise = tanhf (fp32 config, 1e-4 budget); otherwise the MUFU tanh.approx.f32 (bf16 configs: its
// ~2^-11 relative error is below bf16's own 2^-9 rounding step).
template <bool kPrecise>
__device__ __forceinline__ float tanh_fn(float u) {
  if constexpr (kPrecise) {
    return tanhf(u);
  } else {
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(u));
    return t;
  }
}

template <bool kPrecise>
__device__ __forceinline__ float gelu_fwd(float z) {
  const float z2 = z * z;
  const float u = kGeluC() * z * fmaf(kGeluA(), z2, 1.0f);
  const float t = tanh_fn<kPrecise>(u);
  const float hz = 0.5f * z;
  return fmaf(hz, t, hz);
}

template <bool kPrecise>
__device__ __forceinline__ float gelu_bwd(float z) {
  const float z2 = z * z;
  const float u = kGeluC() * z * fmaf(kGeluA(), z2, 1.0f);
  const float t = tanh_fn<kPrecise>(u);
  const float du = kGeluC() * fmaf(3.0f * kGeluA(), z2, 1.0f);
  const float sech2 = fmaf(-t, t, 1.0f);
  return fmaf(0.5f * z * sech2, du, fmaf(0.5f, t, 0.5f));
}

}  // namespace osdp

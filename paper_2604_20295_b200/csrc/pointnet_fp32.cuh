// fp32 SIMT pieces of the PointNet form of Phi (widths = DESIGN.md R10) shared by the fp32 forward
// (k_pointnet_fp32.cu) and the backward (k_backward_pointnet.cu).
#pragma once
#include "etac_internal.h"

namespace etac {

constexpr int kPnW32Floats = 64 * 9 + 64 + 64 * 64 + 64 + 64 * 64 + 3 * 64 + 3;  // E1 e1 E2 e2 D1[:, :64] D2 d2

__device__ __forceinline__ float silu_exact(float x) { return x / (1.0f + expf(-x)); }
// monotone map float -> uint32 (max of keys = key of the max); 0 is below every float's key
__device__ __forceinline__ uint32_t float_key(float f) {
  const uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key_float(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// point-wise features of one node: x9 = [p(3), n(3), u^(3)], weights in shared memory
__device__ __forceinline__ void pn_features(const float* __restrict__ sw, const float (&x9)[9], float (&f)[64]) {
  const float *E1 = sw, *e1 = E1 + 576, *E2 = e1 + 64, *e2 = E2 + 4096;
  float h1[64];
#pragma unroll
  for (int k = 0; k < 64; ++k) {
    float s = e1[k];
#pragma unroll
    for (int c = 0; c < 9; ++c) s = fmaf(E1[k * 9 + c], x9[c], s);
    h1[k] = silu_exact(s);
  }
  for (int k2 = 0; k2 < 64; ++k2) {
    float s = e2[k2];
    const float4* w = reinterpret_cast<const float4*>(E2 + k2 * 64);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const float4 wv = w[k];
      s = fmaf(wv.x, h1[4 * k], s), s = fmaf(wv.y, h1[4 * k + 1], s), s = fmaf(wv.z, h1[4 * k + 2], s), s = fmaf(wv.w, h1[4 * k + 3], s);
    }
    f[k2] = silu_exact(s);
  }
}

}  // namespace etac

// Measurement helper, not on the hot path: the issue rate of the special-function (MUFU) pipe.
//
// The fused S2-S4 kernel evaluates 128 SiLUs per node-environment (two hidden layers of 64,
// BASELINE.json configs[0]); each is one MUFU.TANH, and that pipe, not the tensor core, is the
// unit the kernel saturates first.  The guides give no unit count for it, so the
// roofline denominator is measured: every thread runs kChains independent dependent chains of
// tanh.approx.f32, 32 warps per SM, a multiple of the SM count of CTAs.
#include "etac_internal.h"

namespace etac {

constexpr int kChains = 8;

__global__ void __launch_bounds__(1024) mufu_rate_kernel(float* __restrict__ out, int iters) {
  float x[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) x[c] = 0.001f * (float)(threadIdx.x + 1) + (float)c;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int c = 0; c < kChains; ++c) asm volatile("tanh.approx.f32 %0, %0;" : "+f"(x[c]));
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < kChains; ++c) s += x[c];
  if (s == 123.456f) out[0] = s;  // never true: keeps the chains alive
}

}  // namespace etac

extern "C" etac_status etac_measure_sfu_rate(void* cuda_stream, double* ops_per_s, double* ops_per_clk_per_sm) {
  using namespace etac;
  if (!ops_per_s) return ETAC_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, n_sm = 0, khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev) != cudaSuccess)
    return ETAC_ERR_CUDA;
  float* d = nullptr;
  cudaEvent_t e0, e1;
  if (cudaMalloc(&d, 4) != cudaSuccess) return ETAC_ERR_CUDA;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return ETAC_ERR_CUDA;
  const int iters = 4096, grid = n_sm * 2, threads = 1024;
  float best = 0.f;
  cudaError_t e = cudaSuccess;
  for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {  // first repetition warms up
    cudaEventRecord(e0, s);
    mufu_rate_kernel<<<grid, threads, 0, s>>>(d, iters);
    cudaEventRecord(e1, s);
    e = cudaStreamSynchronize(s);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && (best == 0.f || ms < best)) best = ms;
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaEventDestroy(e0), cudaEventDestroy(e1), cudaFree(d);
  if (e != cudaSuccess || best <= 0.f) return ETAC_ERR_CUDA;
  const double ops = (double)grid * threads * kChains * iters;
  *ops_per_s = ops / (best * 1e-3);
  if (ops_per_clk_per_sm) *ops_per_clk_per_sm = *ops_per_s / ((double)khz * 1e3) / n_sm;  // at the nominal maximum clock
  return ETAC_OK;
}

// Create-time kernels: the propagation matrix of Eq. (1) per patch, in fp32
// (gather path) and bf16 (tensor-core path), and the environment-independent part of MLP layer 1.
#include "etac_internal.h"

namespace etac {

// K_p[i,j] = exp(-alpha_p * ||p_j - p_i||_2); one thread per (i,j), j fastest (coalesced stores).
__global__ void build_k_kernel(DevModel m, float* __restrict__ k32, __nv_bfloat16* __restrict__ k16, int p) {
  const PatchInfo pi = m.patch[p];
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = blockIdx.y;
  if (j >= pi.n) return;
  const float4 a = m.pos4[pi.off + i];
  const float4 b = m.pos4[pi.off + j];
  const float dx = b.x - a.x, dy = b.y - a.y, dz = b.z - a.z;
  const float dist = sqrtf((dx * dx + dy * dy) + dz * dz);
  const float k = expf(-pi.alpha * dist);
  k32[pi.k32_off + (int64_t)i * pi.n + j] = k;
  k16[(int64_t)(pi.off + i) * m.kw + j] = __float2bfloat16_rn(k);
}

cudaError_t launch_build_k(const DevModel& m, float* k32, __nv_bfloat16* k16, cudaStream_t s) {
  std::vector<PatchInfo> hp(m.n_patches);
  cudaError_t e = cudaMemcpy(hp.data(), m.patch, sizeof(PatchInfo) * m.n_patches, cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return e;
  for (int p = 0; p < m.n_patches; ++p) {
    dim3 grid((hp[p].n + 255) / 256, hp[p].n);
    build_k_kernel<<<grid, 256, 0, s>>>(m, k32, k16, p);
  }
  return cudaGetLastError();
}

// c1t[k][i] = b1[k] + sum_{c<3} W1[k][3+c] p_i[c] + W1[k][6+c] n_i[c]   (fp32 gather path)
__global__ void build_c1_kernel(DevModel m, const float* __restrict__ W1, const float* __restrict__ b1,
                                float* __restrict__ c1t) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int k = blockIdx.y;
  if (i >= m.n_nodes) return;
  const float4 p = m.pos4[i], n = m.nrm4[i];
  const float* w = W1 + k * 9;
  float acc = b1[k];
  acc = fmaf(w[3], p.x, acc);
  acc = fmaf(w[4], p.y, acc);
  acc = fmaf(w[5], p.z, acc);
  acc = fmaf(w[6], n.x, acc);
  acc = fmaf(w[7], n.y, acc);
  acc = fmaf(w[8], n.z, acc);
  c1t[(int64_t)k * m.n_nodes + i] = acc;
}

cudaError_t launch_build_c1(const DevModel& m, const float* W1, const float* b1, float* c1t, cudaStream_t s) {
  dim3 grid((m.n_nodes + 255) / 256, kHidden);
  build_c1_kernel<<<grid, 256, 0, s>>>(m, W1, b1, c1t);
  return cudaGetLastError();
}

}  // namespace etac

// The paper's form of Phi (PointNet encoder, max-pool, global MLP, decoder, widths = DESIGN.md
// R10) on ETAC_PREC_FP32 contexts: plain fp32 SIMT with exact expf, at the fp32 tolerance of the per-node form.
// Three kernels behind S1 (the max-pool over all nodes of a patch separates encoder and decoder):
//   pn_encode_fp32_kernel  f_i = silu(E2 silu(E1 [p, n, u^] + e1) + e2) per node of a contacting (env, patch),
//                          column max over the nodes -> gmax (order-preserving integer keys, atomicMax)
//   pn_global_env_kernel   g' = silu(G1 g + g1),  c = D1[:, 64:] g' + d1   per contacting (env, patch)
//   pn_decode_fp32_kernel  Omega U_a as in gather_fp32_kernel, f_i again, r = D2 silu(D1[:, :64] f_i + c) + d2,
//                          mask + combine (Eq. 2)
// gmax / cvec are the arrays of the bf16 path, indexed by the environment instead of the contact-list slot.
#include "etac_internal.h"
#include "pointnet_fp32.cuh"

namespace etac {

__global__ void __launch_bounds__(kGatherChunk) pn_encode_fp32_kernel(DevModel m, StepIO io) {
  extern __shared__ float s_w[];
  const int e = blockIdx.x / m.n_chunks;
  const ChunkInfo ch = m.chunk[blockIdx.x - e * m.n_chunks];
  if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) return;
  const int t = threadIdx.x, lane = t & 31;
  for (int k = t; k < 576 + 64 + 4096 + 64; k += kGatherChunk) s_w[k] = m.pn_w32[k];
  __syncthreads();
  const bool valid = t < ch.count;
  const int g = ch.node0 + (valid ? t : 0);
  const float4 pos = m.pos4[g], nn = m.nrm4[g];
  const float d = m.delta[(int64_t)e * m.n_nodes + g];
  const float x9[9] = {pos.x, pos.y, pos.z, nn.x, nn.y, nn.z, -d * nn.x, -d * nn.y, -d * nn.z};
  float f[64];
  pn_features(s_w, x9, f);
  uint32_t* gm = m.gmax + ((int64_t)ch.patch * m.max_envs + e) * 64;
  uint32_t mine = 0;  // lane l ends up with the warp's max key of column l (and 32 + l in the second round)
#pragma unroll
  for (int half = 0; half < 2; ++half) {
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const uint32_t key = __reduce_max_sync(0xffffffffu, valid ? float_key(f[32 * half + k]) : 0u);
      if (lane == k) mine = key;
    }
    atomicMax(gm + 32 * half + lane, mine);
  }
}

__global__ void __launch_bounds__(64) pn_global_env_kernel(DevModel m, int n_envs) {
  const int p = blockIdx.y, k = threadIdx.x;
  __shared__ float sG1[64 * 64], sD1[64 * 64], g[64], g2[64];
  const float* G1t = m.pn_f32, *g1 = G1t + 4096, *D1gt = g1 + 64, *d1 = D1gt + 4096;  // both matrices [in][out]
  bool staged = false;
  for (int e = blockIdx.x * 16; e < min(n_envs, blockIdx.x * 16 + 16); ++e) {
    if (!m.flags[(int64_t)e * m.n_patches + p]) continue;  // (uniform over the CTA)
    if (!staged) {
      for (int i = k; i < 4096; i += 64) sG1[i] = G1t[i], sD1[i] = D1gt[i];
      staged = true;
    }
    const int64_t base = ((int64_t)p * m.max_envs + e) * 64;
    __syncthreads();
    g[k] = key_float(m.gmax[base + k]);
    __syncthreads();
    float a = g1[k];
#pragma unroll 8
    for (int j = 0; j < 64; ++j) a = fmaf(sG1[j * 64 + k], g[j], a);
    g2[k] = silu_exact(a);
    __syncthreads();
    float c = d1[k];
#pragma unroll 8
    for (int j = 0; j < 64; ++j) c = fmaf(sD1[j * 64 + k], g2[j], c);
    m.cvec[base + k] = c;
  }
}

__global__ void __launch_bounds__(kGatherChunk) pn_decode_fp32_kernel(DevModel m, StepIO io) {
  extern __shared__ float s_w[];
  __shared__ int s_j[kGatherChunk];
  __shared__ float s_u[kGatherChunk][3];
  __shared__ int s_wcnt[kGatherChunk / 32];
  const int e = blockIdx.x / m.n_chunks;
  const ChunkInfo ch = m.chunk[blockIdx.x - e * m.n_chunks];
  if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) return;  // S1 zero-filled this patch
  const PatchInfo pi = m.patch[ch.patch];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const bool valid = t < ch.count;
  const int g = ch.node0 + (valid ? t : 0);
  const int li = g - pi.off;
  const float* __restrict__ delta = m.delta + (int64_t)e * m.n_nodes + pi.off;
  const float* __restrict__ K = m.k32 + pi.k32_off;
  for (int k = t; k < kPnW32Floats; k += kGatherChunk) s_w[k] = m.pn_w32[k];

  // Omega U_a over the active nodes of the patch, compacted in node order (as gather_fp32_kernel)
  float ax = 0.f, ay = 0.f, az = 0.f;
  for (int base = 0; base < pi.n; base += kGatherChunk) {
    const int j = base + t;
    const float dj = j < pi.n ? delta[j] : 0.0f;
    const bool act = dj > 0.0f;
    const unsigned bal = __ballot_sync(0xffffffffu, act);
    if (lane == 0) s_wcnt[warp] = __popc(bal);
    __syncthreads();
    int pre = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kGatherChunk / 32; ++w) {
      const int c = s_wcnt[w];
      pre += w < warp ? c : 0;
      total += c;
    }
    if (act) {
      const int slot = pre + __popc(bal & ((1u << lane) - 1u));
      const float4 n = m.nrm4[pi.off + j];
      s_j[slot] = j;
      s_u[slot][0] = -dj * n.x, s_u[slot][1] = -dj * n.y, s_u[slot][2] = -dj * n.z;
    }
    __syncthreads();
    for (int a = 0; a < total; ++a) {
      const float k = K[(int64_t)s_j[a] * pi.n + li];
      ax = fmaf(k, s_u[a][0], ax);
      ay = fmaf(k, s_u[a][1], ay);
      az = fmaf(k, s_u[a][2], az);
    }
    __syncthreads();
  }
  if (!valid) return;

  const float4 pos = m.pos4[g], nn = m.nrm4[g];
  const float d = delta[li];
  const float x9[9] = {pos.x, pos.y, pos.z, nn.x, nn.y, nn.z, -d * nn.x, -d * nn.y, -d * nn.z};
  float f[64];
  pn_features(s_w, x9, f);
  const float *D1a = s_w + 576 + 64 + 4096 + 64, *D2 = D1a + 4096, *d2 = D2 + 192;
  const float* __restrict__ cv = m.cvec + ((int64_t)ch.patch * m.max_envs + e) * 64;
  float r0 = d2[0], r1 = d2[1], r2 = d2[2];
  for (int k2 = 0; k2 < 64; ++k2) {
    float s = cv[k2];
    const float4* w = reinterpret_cast<const float4*>(D1a + k2 * 64);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const float4 wv = w[k];
      s = fmaf(wv.x, f[4 * k], s), s = fmaf(wv.y, f[4 * k + 1], s), s = fmaf(wv.z, f[4 * k + 2], s), s = fmaf(wv.w, f[4 * k + 3], s);
    }
    const float h = silu_exact(s);
    r0 = fmaf(D2[k2], h, r0), r1 = fmaf(D2[64 + k2], h, r1), r2 = fmaf(D2[128 + k2], h, r2);
  }
  float ox, oy, oz;
  if (m.residual_only) ox = r0, oy = r1, oz = r2;  // Table II ablation "Residual Network Only"
  else ox = ax + r0, oy = ay + r1, oz = az + r2;
  if (d > 0.0f && m.active_mode == ETAC_ACTIVE_PASSTHROUGH) ox = -d * nn.x, oy = -d * nn.y, oz = -d * nn.z;
  store_out3(io, e, g, ox, oy, oz);
  if (io.analytic_out) {
    float* a = io.analytic_out + ((int64_t)e * m.n_nodes + g) * 3;
    a[0] = ax, a[1] = ay, a[2] = az;
  }
}

// c_(e,p) for every contacting (env, patch) from gmax (also the first half of the backward's global pass)
void launch_pointnet_global_env(const DevModel& m, int n_envs, cudaStream_t s) {
  pn_global_env_kernel<<<dim3((unsigned)((n_envs + 15) / 16), (unsigned)m.n_patches), 64, 0, s>>>(m, n_envs);
}

cudaError_t pointnet_fp32_configure() {
  return cudaFuncSetAttribute(pn_decode_fp32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPnW32Floats * 4);
}

// S2-S4 of an fp32 context with the PointNet form of Phi; *launches receives the number of kernels
cudaError_t launch_pointnet_fp32(const DevModel& m, const StepIO& io, int* launches, cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(m.gmax, 0, sizeof(uint32_t) * 64 * (size_t)m.n_patches * m.max_envs, s);
  if (e != cudaSuccess) return e;
  const unsigned grid = (unsigned)((int64_t)m.n_chunks * io.n_envs);
  pn_encode_fp32_kernel<<<grid, kGatherChunk, (576 + 64 + 4096 + 64) * 4, s>>>(m, io);
  launch_pointnet_global_env(m, io.n_envs, s);
  pn_decode_fp32_kernel<<<grid, kGatherChunk, kPnW32Floats * 4, s>>>(m, io);
  *launches = 3;
  return cudaGetLastError();
}

}  // namespace etac

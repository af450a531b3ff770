// S2+S3+S4, fp32 SIMT "sparse gather" path: Omega U_a literally -- every node of
// a contacting (env, patch) sums exp-decay contributions of the ACTIVE nodes only -- followed by
// the per-node residual MLP (fp32, exact expf) and the mask/combine of Eq. (2).
// Used for ETAC_PREC_FP32 contexts and for ETAC_PATH_SPARSE.
//
// One CTA = kGatherChunk (128) consecutive nodes of one patch in one environment; thread = node.
// K is symmetric, so K[i][j] is read as K[j][i]: for a fixed active j the 128 threads read 128
// consecutive floats of row j (coalesced).  Active nodes are compacted in node order with
// ballots (deterministic summation order).
#include "etac_internal.h"

namespace etac {

constexpr int kWf32Floats = 64 * 3 + 64 * 64 + 64 + 3 * 64 + 3;  // W1u | W2 | b2 | W3 | b3

__device__ __forceinline__ float silu_f32(float x) { return x / (1.0f + expf(-x)); }

__global__ void __launch_bounds__(kGatherChunk) gather_fp32_kernel(DevModel m, StepIO io) {
  __shared__ float s_w[kWf32Floats];
  __shared__ int s_j[kGatherChunk];
  __shared__ float s_u[kGatherChunk][3];
  __shared__ int s_wcnt[kGatherChunk / 32];

  const int e = blockIdx.x / m.n_chunks;  // 1-D grid: n_envs is not bounded by gridDim.y's 65535
  const ChunkInfo ch = m.chunk[blockIdx.x - e * m.n_chunks];
  if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) return;  // S1 zero-filled this patch
  const PatchInfo pi = m.patch[ch.patch];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const bool valid = t < ch.count;
  const int g = ch.node0 + (valid ? t : 0);
  const int li = g - pi.off;
  const float* __restrict__ delta = m.delta + (int64_t)e * m.n_nodes + pi.off;
  const float* __restrict__ K = m.k32 + pi.k32_off;

  if (m.resid != ETAC_RESID_NONE)
    for (int k = t; k < kWf32Floats; k += kGatherChunk) s_w[k] = m.wf32[k];

  float ax = 0.f, ay = 0.f, az = 0.f;
  for (int base = 0; base < pi.n; base += kGatherChunk) {
    const int j = base + t;
    const float d = j < pi.n ? delta[j] : 0.0f;
    const bool act = d > 0.0f;
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
      s_u[slot][0] = -d * n.x, s_u[slot][1] = -d * n.y, s_u[slot][2] = -d * n.z;
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

  float ox = ax, oy = ay, oz = az;
  if (m.resid == ETAC_RESID_NONE && m.residual_only) ox = oy = oz = 0.0f;  // Phi_p of a context without Phi
  if (m.resid != ETAC_RESID_NONE) {
    const float* W1u = s_w;
    const float* W2 = s_w + 192;
    const float* b2 = W2 + 4096;
    const float* W3 = b2 + 64;
    const float* b3 = W3 + 192;
    float h1[kHidden];
#pragma unroll
    for (int k = 0; k < kHidden; ++k) {
      float s = m.c1t[(int64_t)k * m.n_nodes + g];
      s = fmaf(W1u[k * 3 + 0], ax, s);
      s = fmaf(W1u[k * 3 + 1], ay, s);
      s = fmaf(W1u[k * 3 + 2], az, s);
      h1[k] = silu_f32(s);
    }
    float r0 = b3[0], r1 = b3[1], r2 = b3[2];
    for (int k2 = 0; k2 < kHidden; ++k2) {
      float s = b2[k2];
      const float4* w = reinterpret_cast<const float4*>(W2 + k2 * kHidden);
#pragma unroll
      for (int k = 0; k < kHidden / 4; ++k) {
        const float4 wv = w[k];
        s = fmaf(wv.x, h1[4 * k + 0], s);
        s = fmaf(wv.y, h1[4 * k + 1], s);
        s = fmaf(wv.z, h1[4 * k + 2], s);
        s = fmaf(wv.w, h1[4 * k + 3], s);
      }
      const float h2 = silu_f32(s);
      r0 = fmaf(W3[k2], h2, r0);
      r1 = fmaf(W3[kHidden + k2], h2, r1);
      r2 = fmaf(W3[2 * kHidden + k2], h2, r2);
    }
    if (m.residual_only) ox = r0, oy = r1, oz = r2;  // Table II ablation "Residual Network Only"
    else ox += r0, oy += r1, oz += r2;
  }
  const float d = delta[li];
  if (d > 0.0f && m.active_mode == ETAC_ACTIVE_PASSTHROUGH) {
    const float4 n = m.nrm4[g];
    ox = -d * n.x, oy = -d * n.y, oz = -d * n.z;
  }
  const int64_t o = ((int64_t)e * m.n_nodes + g) * 3;
  store_out3(io, e, g, ox, oy, oz);
  if (io.analytic_out) io.analytic_out[o] = ax, io.analytic_out[o + 1] = ay, io.analytic_out[o + 2] = az;
}

cudaError_t launch_gather_fp32(const DevModel& m, const StepIO& io, cudaStream_t s) {
  const unsigned grid = (unsigned)((int64_t)m.n_chunks * io.n_envs);
  gather_fp32_kernel<<<grid, kGatherChunk, 0, s>>>(m, io);
  return cudaGetLastError();
}

}  // namespace etac

// Backward pass of S2-S4 for the calibration of Eq. (3) (alpha and Phi are fitted
// by gradient descent on ||U_p - U_p*||): given G = dL/dU it returns dL/dalpha and dL/d(weights of
// the per-node residual MLP).  fp32 SIMT, same decomposition as the fp32 forward kernel
// (k_gather_fp32.cu): thread = node, work item = 128 consecutive nodes of one patch in one
// environment whose patch is in contact.
//
// For a row i that Eq. (2) does not overwrite (passive rows; all rows in ETAC_ACTIVE_PROPAGATE):
//   u_i = sum_{j active} K_ij u^_j,   U_i = u_i + Phi(u_i, p_i, n_i),   K_ij = exp(-alpha d_ij)
//   dK_ij/dalpha = -d_ij K_ij = K_ij ln(K_ij) / alpha          (no positions needed)
//   dL/dalpha   += (G_i + J_Phi,u^T G_i) . sum_j dK_ij/dalpha u^_j
//   dL/dW       += the usual MLP backward of G_i
// Active rows of Eq. (2) are u^ itself and carry no gradient to alpha or Phi.
//
// The grid is persistent (one CTA per SM, 128 threads).  Per item every thread runs forward and
// backward of its node with its activations in registers and leaves h1, dz1, dz2, h2 as columns of
// four [64 x 128] shared-memory arrays; the weight gradients are then CTA-level products of those
// arrays (dW2 = dZ2^T H1 as a 4 x 8 register tile per thread), accumulated in registers over all
// items of the CTA and added to the global result once at the end (fp32 atomics: the sum order
// across CTAs is not fixed, results agree to fp32 rounding).
#include "etac_internal.h"

namespace etac {

namespace {
constexpr int kT = kGatherChunk;        // threads per CTA = nodes per item
constexpr int kLd = kT + 1;             // row pitch of the [64][128] arrays (conflict-free column and row access)
constexpr int kWf32 = 64 * 3 + 64 * 64 + 64 + 3 * 64 + 3;  // W1u | W2 | b2 | W3 | b3 (DevModel::wf32)

struct BwdSmem {
  float w[kWf32];
  float A[kHidden * kLd];  // silu'(z1) -> dz1
  float B[kHidden * kLd];  // h1
  float C[kHidden * kLd];  // dz2
  float D[kHidden * kLd];  // h2
  float X[9 * kLd];        // layer-1 input [u(3), p(3), n(3)] per node
  float G[3 * kLd];        // upstream gradient of the rows that carry one (0 elsewhere)
  float u[kT][3];
  int j[kT];
  int wcnt[kT / 32];
  float red[kT / 32];
};

__device__ __forceinline__ void silu_and_grad(float z, float& y, float& dy) {
  const float s = 1.0f / (1.0f + expf(-z));
  y = z * s;
  dy = s * (1.0f + z * (1.0f - s));
}
}  // namespace

__global__ void __launch_bounds__(kT, 1) backward_kernel(DevModel m, StepIO io, const float* __restrict__ grad_out,
                                                         float* __restrict__ grad_alpha, int n_alpha,
                                                         float* __restrict__ grad_w) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  BwdSmem& S = *reinterpret_cast<BwdSmem*>(smem_raw);
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const bool mlp = m.resid == ETAC_RESID_PERNODE_MLP;
  if (mlp)
    for (int k = t; k < kWf32; k += kT) S.w[k] = m.wf32[k];
  const float* W1u = S.w;
  const float* W2 = S.w + 192;
  const float* b2 = W2 + 4096;
  const float* W3 = b2 + 64;

  // per-thread shares of the weight gradients, accumulated over all items of this CTA
  const int kt = 4 * (t & 15), jt = 8 * (t >> 4);  // dW2 tile: rows kt..kt+3 (layer-2 output), columns jt..jt+7
  float gw2[4][8];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 8; ++b) gw2[a][b] = 0.f;
  float gw1[5] = {0.f, 0.f, 0.f, 0.f, 0.f};  // dW1 entries t, t+128, ... (< 576) in [64 x 9] order
  float gw3[2] = {0.f, 0.f};                 // dW3 entries t, t+128 (< 192) in [3 x 64] order
  float gb = 0.f;                            // t < 64: db1[t]; else db2[t - 64]
  float gb3 = 0.f;                           // t < 3: db3[t]
  __syncthreads();

  const int64_t n_items = (int64_t)m.n_chunks * io.n_envs;
  for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int e = (int)(item / m.n_chunks);
    const ChunkInfo ch = m.chunk[item - (int64_t)e * m.n_chunks];
    if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) continue;  // contact-free pair: U = 0, no gradient
    const PatchInfo pi = m.patch[ch.patch];
    const bool valid = t < ch.count;
    const int g = ch.node0 + (valid ? t : 0);
    const int li = g - pi.off;
    const float* __restrict__ delta = m.delta + (int64_t)e * m.n_nodes + pi.off;
    const float* __restrict__ K = m.k32 + pi.k32_off;

    // ---- u_i = sum_j K_ij u^_j and v_i = sum_j K_ij ln K_ij u^_j over the active nodes j (node order)
    float ax = 0.f, ay = 0.f, az = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    for (int base = 0; base < pi.n; base += kT) {
      const int j = base + t;
      const float d = j < pi.n ? delta[j] : 0.0f;
      const bool act = d > 0.0f;
      const unsigned bal = __ballot_sync(0xffffffffu, act);
      if (lane == 0) S.wcnt[warp] = __popc(bal);
      __syncthreads();
      int pre = 0, total = 0;
#pragma unroll
      for (int w = 0; w < kT / 32; ++w) {
        const int c = S.wcnt[w];
        pre += w < warp ? c : 0;
        total += c;
      }
      if (act) {
        const int slot = pre + __popc(bal & ((1u << lane) - 1u));
        const float4 n = m.nrm4[pi.off + j];
        S.j[slot] = j;
        S.u[slot][0] = -d * n.x, S.u[slot][1] = -d * n.y, S.u[slot][2] = -d * n.z;
      }
      __syncthreads();
      for (int a = 0; a < total; ++a) {
        const float k = K[(int64_t)S.j[a] * pi.n + li];
        const float kl = k > 0.0f ? k * logf(k) : 0.0f;
        ax = fmaf(k, S.u[a][0], ax), ay = fmaf(k, S.u[a][1], ay), az = fmaf(k, S.u[a][2], az);
        vx = fmaf(kl, S.u[a][0], vx), vy = fmaf(kl, S.u[a][1], vy), vz = fmaf(kl, S.u[a][2], vz);
      }
      __syncthreads();
    }
    // rows that carry a gradient: Eq. (2) overwrites the active rows with u^ (ETAC_ACTIVE_PASSTHROUGH)
    const bool carries = valid && !(m.active_mode == ETAC_ACTIVE_PASSTHROUGH && delta[li] > 0.0f);
    float g0 = 0.f, g1 = 0.f, g2 = 0.f;
    if (carries) {
      const float* go = grad_out + ((int64_t)e * m.n_nodes + g) * 3;
      g0 = go[0], g1 = go[1], g2 = go[2];
    }
    float l0 = g0, l1 = g1, l2 = g2;  // dL/du_i = G_i + J_Phi,u^T G_i
    if (mlp) {
      const float4 pos = m.pos4[g], nrm = m.nrm4[g];
      S.X[0 * kLd + t] = ax, S.X[1 * kLd + t] = ay, S.X[2 * kLd + t] = az;
      S.X[3 * kLd + t] = pos.x, S.X[4 * kLd + t] = pos.y, S.X[5 * kLd + t] = pos.z;
      S.X[6 * kLd + t] = nrm.x, S.X[7 * kLd + t] = nrm.y, S.X[8 * kLd + t] = nrm.z;
      S.G[0 * kLd + t] = g0, S.G[1 * kLd + t] = g1, S.G[2 * kLd + t] = g2;
      // forward layer 1 (position / normal part precomputed at create: c1t), activations in registers
      float h[kHidden];
#pragma unroll
      for (int k = 0; k < kHidden; ++k) h[k] = m.c1t[(int64_t)k * m.n_nodes + g];  // 64 independent loads in flight
#pragma unroll
      for (int k = 0; k < kHidden; ++k) {
        float z = h[k];
        z = fmaf(W1u[k * 3 + 0], ax, z), z = fmaf(W1u[k * 3 + 1], ay, z), z = fmaf(W1u[k * 3 + 2], az, z);
        float dy;
        silu_and_grad(z, h[k], dy);
        S.A[k * kLd + t] = dy;
        S.B[k * kLd + t] = h[k];
      }
      // forward layer 2 and, in the same sweep, dz2 = (W3^T G) * silu'(z2); two rows and two partial sums
      // per row at a time: with one warp per SM sub-partition the FMA latency is not hidden otherwise
      for (int k2 = 0; k2 < kHidden; k2 += 2) {
        float za = b2[k2], zb = b2[k2 + 1], zc = 0.f, zd = 0.f;
        const float4* wa = reinterpret_cast<const float4*>(W2 + k2 * kHidden);
        const float4* wb = reinterpret_cast<const float4*>(W2 + (k2 + 1) * kHidden);
#pragma unroll
        for (int k = 0; k < kHidden / 4; ++k) {
          const float4 u = wa[k], v = wb[k];
          za = fmaf(u.x, h[4 * k + 0], za), zc = fmaf(u.y, h[4 * k + 1], zc);
          zb = fmaf(v.x, h[4 * k + 0], zb), zd = fmaf(v.y, h[4 * k + 1], zd);
          za = fmaf(u.z, h[4 * k + 2], za), zc = fmaf(u.w, h[4 * k + 3], zc);
          zb = fmaf(v.z, h[4 * k + 2], zb), zd = fmaf(v.w, h[4 * k + 3], zd);
        }
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          const int kk = k2 + q;
          float y, dy;
          silu_and_grad(q ? zb + zd : za + zc, y, dy);
          const float gh2 = fmaf(W3[kk], g0, fmaf(W3[kHidden + kk], g1, W3[2 * kHidden + kk] * g2));
          S.C[kk * kLd + t] = gh2 * dy;
          S.D[kk * kLd + t] = y;
        }
      }
      // dh1 = W2^T dz2 (h[] is reused), dz1 = dh1 * silu'(z1), dL/du += W1u^T dz1
#pragma unroll
      for (int k = 0; k < kHidden; ++k) h[k] = 0.f;
      for (int k2 = 0; k2 < kHidden; ++k2) {
        const float gz = S.C[k2 * kLd + t];
        const float4* w = reinterpret_cast<const float4*>(W2 + k2 * kHidden);
#pragma unroll
        for (int k = 0; k < kHidden / 4; ++k) {
          const float4 wv = w[k];
          h[4 * k + 0] = fmaf(wv.x, gz, h[4 * k + 0]), h[4 * k + 1] = fmaf(wv.y, gz, h[4 * k + 1]);
          h[4 * k + 2] = fmaf(wv.z, gz, h[4 * k + 2]), h[4 * k + 3] = fmaf(wv.w, gz, h[4 * k + 3]);
        }
      }
#pragma unroll
      for (int k = 0; k < kHidden; ++k) {
        const float gz1 = h[k] * S.A[k * kLd + t];
        S.A[k * kLd + t] = gz1;
        l0 = fmaf(W1u[k * 3 + 0], gz1, l0), l1 = fmaf(W1u[k * 3 + 1], gz1, l1), l2 = fmaf(W1u[k * 3 + 2], gz1, l2);
      }
    }
    // ---- dL/dalpha of this item: sum_i dL/du_i . v_i / alpha
    {
      float ga = carries ? (l0 * vx + l1 * vy + l2 * vz) / pi.alpha : 0.0f;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) ga += __shfl_xor_sync(0xffffffffu, ga, o);
      if (lane == 0) S.red[warp] = ga;
    }
    __syncthreads();  // columns of A, B, C, D, X, G and red[] complete
    if (t == 0) {
      float ga = 0.f;
#pragma unroll
      for (int w = 0; w < kT / 32; ++w) ga += S.red[w];
      atomicAdd(&grad_alpha[n_alpha == 1 ? 0 : ch.patch], ga);
    }
    if (mlp) {
      // ---- weight gradients as CTA-level products over the item's 128 nodes
      for (int i = 0; i < kT; ++i) {
        float a[4], b[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) a[q] = S.C[(kt + q) * kLd + i];
#pragma unroll
        for (int q = 0; q < 8; ++q) b[q] = S.B[(jt + q) * kLd + i];
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int r = 0; r < 8; ++r) gw2[q][r] = fmaf(a[q], b[r], gw2[q][r]);
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const int idx = t + q * kT;  // (k, c) = (idx / 9, idx % 9)
        if (idx < kHidden * 9) {
          const float* zr = S.A + (idx / 9) * kLd;
          const float* xr = S.X + (idx % 9) * kLd;
          float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
          for (int i = 0; i < kT; i += 4)
            s0 = fmaf(zr[i], xr[i], s0), s1 = fmaf(zr[i + 1], xr[i + 1], s1), s2 = fmaf(zr[i + 2], xr[i + 2], s2),
            s3 = fmaf(zr[i + 3], xr[i + 3], s3);
          gw1[q] += (s0 + s1) + (s2 + s3);
        }
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int idx = t + q * kT;  // (c, k) = (idx / 64, idx % 64)
        if (idx < 3 * kHidden) {
          const float* gr = S.G + (idx / kHidden) * kLd;
          const float* hr = S.D + (idx % kHidden) * kLd;
          float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
          for (int i = 0; i < kT; i += 4)
            s0 = fmaf(gr[i], hr[i], s0), s1 = fmaf(gr[i + 1], hr[i + 1], s1), s2 = fmaf(gr[i + 2], hr[i + 2], s2),
            s3 = fmaf(gr[i + 3], hr[i + 3], s3);
          gw3[q] += (s0 + s1) + (s2 + s3);
        }
      }
      {
        const float* zr = (t < kHidden ? S.A : S.C) + (t & (kHidden - 1)) * kLd;
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
        for (int i = 0; i < kT; i += 4) s0 += zr[i], s1 += zr[i + 1], s2 += zr[i + 2], s3 += zr[i + 3];
        gb += (s0 + s1) + (s2 + s3);
      }
      if (t < 3) {
        float s = 0.f;
        for (int i = 0; i < kT; ++i) s += S.G[t * kLd + i];
        gb3 += s;
      }
    }
    __syncthreads();  // the arrays are rewritten by the next item
  }

  if (mlp && grad_w) {  // layout of d_grad_weights: W1[64x9] b1[64] W2[64x64] b2[64] W3[3x64] b3[3]
    float* gW1 = grad_w;
    float* gb1 = gW1 + 576;
    float* gW2 = gb1 + 64;
    float* gb2 = gW2 + 4096;
    float* gW3 = gb2 + 64;
    float* gB3 = gW3 + 192;
#pragma unroll
    for (int q = 0; q < 5; ++q)
      if (t + q * kT < 576) atomicAdd(&gW1[t + q * kT], gw1[q]);
    atomicAdd(t < kHidden ? &gb1[t] : &gb2[t - kHidden], gb);
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
      for (int r = 0; r < 8; ++r) atomicAdd(&gW2[(kt + q) * kHidden + jt + r], gw2[q][r]);
#pragma unroll
    for (int q = 0; q < 2; ++q)
      if (t + q * kT < 192) atomicAdd(&gW3[t + q * kT], gw3[q]);
    if (t < 3) atomicAdd(&gB3[t], gb3);
  }
}

cudaError_t backward_configure() {
  return cudaFuncSetAttribute(backward_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BwdSmem));
}

cudaError_t launch_backward(const DevModel& m, const StepIO& io, const float* grad_out, float* grad_alpha, int n_alpha,
                            float* grad_w, int n_sm, cudaStream_t s) {
  backward_kernel<<<n_sm, kT, sizeof(BwdSmem), s>>>(m, io, grad_out, grad_alpha, n_alpha, grad_w);
  return cudaGetLastError();
}

}  // namespace etac

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
// Optionally also dL/ddelta (the penetrations of the nodes in contact; the contact set is held fixed),
// from which a caller chains to object / link poses through its SDF gradients.
//
// The grid is persistent (one CTA per SM, 512 threads: four threads per node, each owning 16 of the
// 64 hidden units, so that 16 warps hide each other's FMA and shared-memory latencies; the
// activations take 1 KB of shared memory per node, which limits an SM to 128 nodes in flight).
// Per item the threads run forward and backward of their node's MLP and leave h1, dz1, dz2, h2 as
// columns of four [64 x 128] shared-memory arrays; the weight gradients are then CTA-level products
// of those arrays (dW2 = dZ2^T H1 as 4 x 4 register tiles over half the nodes each), accumulated
// in registers over all items of the CTA and added to the global result once at the end (fp32
// atomics: the sum order across CTAs is not fixed, results agree to fp32 rounding).
#include "etac_internal.h"

namespace etac {

namespace {
constexpr int kT = kGatherChunk;        // nodes per item
constexpr int kParts = 4;               // threads per node: part s owns the hidden units 16 s .. 16 s + 15
constexpr int kThreads = kT * kParts;   // 512: thread t = s * 128 + i (s is warp-uniform)
constexpr int kHp = kHidden / kParts;   // 16
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
  float L[kParts][3][kT];  // per-part shares of W1u^T dz1
  float u[kT][3];
  int j[kT];
  int wcnt[kT / 32];
};

__device__ __forceinline__ void silu_and_grad(float z, float& y, float& dy) {
  const float s = 1.0f / (1.0f + expf(-z));
  y = z * s;
  dy = s * (1.0f + z * (1.0f - s));
}
}  // namespace

__global__ void __launch_bounds__(kThreads, 1) backward_kernel(DevModel m, StepIO io, const float* __restrict__ grad_out,
                                                               float* __restrict__ grad_alpha, int n_alpha,
                                                               float* __restrict__ grad_w,
                                                               float* __restrict__ grad_delta) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  BwdSmem& S = *reinterpret_cast<BwdSmem*>(smem_raw);
  const int t = threadIdx.x, lane = t & 31;
  const int part = t / kT, i = t - part * kT, warp_i = i >> 5;  // node slot i, its warp within the part
  const int k0 = part * kHp;
  const bool mlp = m.resid == ETAC_RESID_PERNODE_MLP;
  if (mlp)
    for (int k = t; k < kWf32; k += kThreads) S.w[k] = m.wf32[k];
  const float* W1u = S.w;
  const float* W2 = S.w + 192;
  const float* b2 = W2 + 4096;
  const float* W3 = b2 + 64;

  // per-thread shares of the weight gradients, accumulated over all items of this CTA.
  // dW2 = dZ2^T H1: 4 x 4 tile (rows kt.., columns jt..) over the nodes [ih, ih + 64) of the item
  const int tile = t & 255, ih = (t >> 8) * (kT / 2);
  const int kt = 4 * (tile & 15), jt = 4 * (tile >> 4);
  float gw2[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) gw2[a][b] = 0.f;
  float gw1[2] = {0.f, 0.f};  // dW1 entries t, t + 512 (< 576) in [64 x 9] order
  float gw3 = 0.f;            // t < 192: dW3 entry t in [3 x 64] order
  float gb = 0.f;             // t < 64: db1[t]; t < 128: db2[t - 64]
  float gb3 = 0.f;            // t < 3: db3[t]
  __syncthreads();

  const int64_t n_items = (int64_t)m.n_chunks * io.n_envs;
  for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int e = (int)(item / m.n_chunks);
    const ChunkInfo ch = m.chunk[item - (int64_t)e * m.n_chunks];
    if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) continue;  // contact-free pair: U = 0, no gradient
    const PatchInfo pi = m.patch[ch.patch];
    const bool valid = i < ch.count;
    const int g = ch.node0 + (valid ? i : 0);
    const int li = g - pi.off;
    const float* __restrict__ delta = m.delta + (int64_t)e * m.n_nodes + pi.off;
    const float* __restrict__ K = m.k32 + pi.k32_off;

    // ---- u_i = sum_j K_ij u^_j and v_i = sum_j K_ij ln K_ij u^_j over the active nodes j (node order);
    // part 0 compacts the active nodes, every part runs the (short) sum for its copy of node i
    float ax = 0.f, ay = 0.f, az = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    for (int base = 0; base < pi.n; base += kT) {
      const int j = base + i;
      const float d = (part == 0 && j < pi.n) ? delta[j] : 0.0f;
      const bool act = d > 0.0f;
      const unsigned bal = __ballot_sync(0xffffffffu, act);
      if (part == 0 && lane == 0) S.wcnt[warp_i] = __popc(bal);
      __syncthreads();
      int pre = 0, total = 0;
#pragma unroll
      for (int w = 0; w < kT / 32; ++w) {
        const int c = S.wcnt[w];
        pre += w < warp_i ? c : 0;
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
    float l0 = g0, l1 = g1, l2 = g2;  // dL/du_i = G_i + J_Phi,u^T G_i (completed by part 0 below)
    if (mlp) {
      if (part == 0) {
        const float4 pos = m.pos4[g], nrm = m.nrm4[g];
        S.X[0 * kLd + i] = ax, S.X[1 * kLd + i] = ay, S.X[2 * kLd + i] = az;
        S.X[3 * kLd + i] = pos.x, S.X[4 * kLd + i] = pos.y, S.X[5 * kLd + i] = pos.z;
        S.X[6 * kLd + i] = nrm.x, S.X[7 * kLd + i] = nrm.y, S.X[8 * kLd + i] = nrm.z;
        S.G[0 * kLd + i] = g0, S.G[1 * kLd + i] = g1, S.G[2 * kLd + i] = g2;
      }
      // forward layer 1 for this part's hidden units (position / normal part precomputed at create: c1t)
      {
        float z[kHp];
#pragma unroll
        for (int q = 0; q < kHp; ++q) z[q] = m.c1t[(int64_t)(k0 + q) * m.n_nodes + g];
#pragma unroll
        for (int q = 0; q < kHp; ++q) {
          const int k = k0 + q;
          float zz = z[q], y, dy;
          zz = fmaf(W1u[k * 3 + 0], ax, zz), zz = fmaf(W1u[k * 3 + 1], ay, zz), zz = fmaf(W1u[k * 3 + 2], az, zz);
          silu_and_grad(zz, y, dy);
          S.A[k * kLd + i] = dy;
          S.B[k * kLd + i] = y;
        }
      }
      __syncthreads();  // h1 of every node complete
      float h[kHidden];
#pragma unroll
      for (int k = 0; k < kHidden; ++k) h[k] = S.B[k * kLd + i];
      // forward layer 2 for this part's rows and, in the same sweep, dz2 = (W3^T G) * silu'(z2);
      // two rows and two partial sums per row at a time (FMA latency)
#pragma unroll 1
      for (int q = 0; q < kHp; q += 2) {
        const int k2 = k0 + q;
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
        for (int r = 0; r < 2; ++r) {
          const int kk = k2 + r;
          float y, dy;
          silu_and_grad(r ? zb + zd : za + zc, y, dy);
          const float gh2 = fmaf(W3[kk], g0, fmaf(W3[kHidden + kk], g1, W3[2 * kHidden + kk] * g2));
          S.C[kk * kLd + i] = gh2 * dy;
          S.D[kk * kLd + i] = y;
        }
      }
      __syncthreads();  // dz2 of every node complete
      // dh1 = W2^T dz2 for this part's 16 hidden units, dz1 = dh1 * silu'(z1), share of W1u^T dz1
#pragma unroll
      for (int k = 0; k < kHidden; ++k) h[k] = S.C[k * kLd + i];  // dz2 of node i
      float gh[kHp];
#pragma unroll
      for (int q = 0; q < kHp; ++q) gh[q] = 0.f;
#pragma unroll
      for (int k2 = 0; k2 < kHidden; ++k2) {
        const float4* w = reinterpret_cast<const float4*>(W2 + k2 * kHidden + k0);
#pragma unroll
        for (int q = 0; q < kHp / 4; ++q) {
          const float4 wv = w[q];
          gh[4 * q + 0] = fmaf(wv.x, h[k2], gh[4 * q + 0]), gh[4 * q + 1] = fmaf(wv.y, h[k2], gh[4 * q + 1]);
          gh[4 * q + 2] = fmaf(wv.z, h[k2], gh[4 * q + 2]), gh[4 * q + 3] = fmaf(wv.w, h[k2], gh[4 * q + 3]);
        }
      }
      float p0 = 0.f, p1 = 0.f, p2 = 0.f;
#pragma unroll
      for (int q = 0; q < kHp; ++q) {
        const int k = k0 + q;
        const float gz1 = gh[q] * S.A[k * kLd + i];
        S.A[k * kLd + i] = gz1;
        p0 = fmaf(W1u[k * 3 + 0], gz1, p0), p1 = fmaf(W1u[k * 3 + 1], gz1, p1), p2 = fmaf(W1u[k * 3 + 2], gz1, p2);
      }
      S.L[part][0][i] = p0, S.L[part][1][i] = p1, S.L[part][2][i] = p2;
      __syncthreads();  // dz1 and the shares of W1u^T dz1 complete
#pragma unroll
      for (int s = 0; s < kParts; ++s) l0 += S.L[s][0][i], l1 += S.L[s][1][i], l2 += S.L[s][2][i];
    }
    // ---- dL/ddelta_j of the patch's active nodes j (optional): u^_j = -delta_j n_j, so
    //   dL/ddelta_j = -n_j . ( sum_{i carrying a gradient} K_ij dL/du_i  +  G_j if row j is u^_j itself )
    // The active nodes are compacted again (their normals this time); part s takes every fourth of them,
    // reduces K_ij (dL/du_i . n_j) over its copy of the item's nodes and adds it with one atomic per warp.
    if (grad_delta) {
      float* gd = grad_delta + (int64_t)e * m.n_nodes + pi.off;
      if (part == 0 && valid && !carries) {  // active row of Eq. (2): U_j = u^_j
        const float* go = grad_out + ((int64_t)e * m.n_nodes + g) * 3;
        const float4 nn = m.nrm4[g];
        atomicAdd(&gd[li], -(nn.x * go[0] + nn.y * go[1] + nn.z * go[2]));
      }
      for (int base = 0; base < pi.n; base += kT) {
        const int j = base + i;
        const bool act = part == 0 && j < pi.n && delta[j] > 0.0f;
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (part == 0 && lane == 0) S.wcnt[warp_i] = __popc(bal);
        __syncthreads();
        int pre = 0, total = 0;
#pragma unroll
        for (int w = 0; w < kT / 32; ++w) {
          const int c = S.wcnt[w];
          pre += w < warp_i ? c : 0;
          total += c;
        }
        if (act) {
          const int slot = pre + __popc(bal & ((1u << lane) - 1u));
          const float4 n = m.nrm4[pi.off + j];
          S.j[slot] = j;
          S.u[slot][0] = n.x, S.u[slot][1] = n.y, S.u[slot][2] = n.z;
        }
        __syncthreads();
        for (int a = part; a < total; a += kParts) {
          float c = 0.0f;
          if (carries) c = K[(int64_t)S.j[a] * pi.n + li] * (l0 * S.u[a][0] + l1 * S.u[a][1] + l2 * S.u[a][2]);
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
          if (lane == 0 && c != 0.0f) atomicAdd(&gd[S.j[a]], -c);
        }
        __syncthreads();
      }
    }
    // ---- dL/dalpha of this item: sum_i dL/du_i . v_i / alpha (part 0's warps, one atomic each)
    if (part == 0) {
      float ga = carries ? (l0 * vx + l1 * vy + l2 * vz) / pi.alpha : 0.0f;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) ga += __shfl_xor_sync(0xffffffffu, ga, o);
      if (lane == 0) atomicAdd(&grad_alpha[n_alpha == 1 ? 0 : ch.patch], ga);
    }
    if (mlp) {
      // ---- weight gradients as CTA-level products over the item's 128 nodes
#pragma unroll 4
      for (int n = ih; n < ih + kT / 2; ++n) {
        float a[4], b[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) a[q] = S.C[(kt + q) * kLd + n], b[q] = S.B[(jt + q) * kLd + n];
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int r = 0; r < 4; ++r) gw2[q][r] = fmaf(a[q], b[r], gw2[q][r]);
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int idx = t + q * kThreads;  // (k, c) = (idx / 9, idx % 9)
        if (idx < kHidden * 9) {
          const float* zr = S.A + (idx / 9) * kLd;
          const float* xr = S.X + (idx % 9) * kLd;
          float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
          for (int n = 0; n < kT; n += 4)
            s0 = fmaf(zr[n], xr[n], s0), s1 = fmaf(zr[n + 1], xr[n + 1], s1), s2 = fmaf(zr[n + 2], xr[n + 2], s2),
            s3 = fmaf(zr[n + 3], xr[n + 3], s3);
          gw1[q] += (s0 + s1) + (s2 + s3);
        }
      }
      if (t < 3 * kHidden) {  // (c, k) = (t / 64, t % 64)
        const float* gr = S.G + (t / kHidden) * kLd;
        const float* hr = S.D + (t % kHidden) * kLd;
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
        for (int n = 0; n < kT; n += 4)
          s0 = fmaf(gr[n], hr[n], s0), s1 = fmaf(gr[n + 1], hr[n + 1], s1), s2 = fmaf(gr[n + 2], hr[n + 2], s2),
          s3 = fmaf(gr[n + 3], hr[n + 3], s3);
        gw3 += (s0 + s1) + (s2 + s3);
      } else if (t >= 256 && t < 256 + 2 * kHidden) {  // (other warps than the dW3 ones)
        const int k = t - 256;
        const float* zr = (k < kHidden ? S.A : S.C) + (k & (kHidden - 1)) * kLd;
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
        for (int n = 0; n < kT; n += 4) s0 += zr[n], s1 += zr[n + 1], s2 += zr[n + 2], s3 += zr[n + 3];
        gb += (s0 + s1) + (s2 + s3);
      } else if (t >= 384 && t < 387) {
        float s = 0.f;
        for (int n = 0; n < kT; ++n) s += S.G[(t - 384) * kLd + n];
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
    for (int q = 0; q < 2; ++q)
      if (t + q * kThreads < 576) atomicAdd(&gW1[t + q * kThreads], gw1[q]);
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
      for (int r = 0; r < 4; ++r) atomicAdd(&gW2[(kt + q) * kHidden + jt + r], gw2[q][r]);
    if (t < 3 * kHidden) atomicAdd(&gW3[t], gw3);
    if (t >= 256 && t < 256 + 2 * kHidden) atomicAdd(t - 256 < kHidden ? &gb1[t - 256] : &gb2[t - 256 - kHidden], gb);
    if (t >= 384 && t < 387) atomicAdd(&gB3[t - 384], gb3);
  }
}

cudaError_t backward_configure() {
  return cudaFuncSetAttribute(backward_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BwdSmem));
}

cudaError_t launch_backward(const DevModel& m, const StepIO& io, const float* grad_out, float* grad_alpha, int n_alpha,
                            float* grad_w, float* grad_delta, int n_sm, cudaStream_t s) {
  backward_kernel<<<n_sm, kThreads, sizeof(BwdSmem), s>>>(m, io, grad_out, grad_alpha, n_alpha, grad_w, grad_delta);
  return cudaGetLastError();
}

}  // namespace etac

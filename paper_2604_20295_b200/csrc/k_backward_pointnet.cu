// Backward pass of the PointNet form of Phi (Eq. (3), calibrates this network
// by gradient descent).  fp32 SIMT on the fp32 copies of the weights, whatever the context's precision.
//
//   forward, per contacting (env, patch):  x_i = [p_i, n_i, u^_i]           u^_i = -delta_i n_i
//       f1 = silu(E1 x + e1), f = silu(E2 f1 + e2), gmax = max_i f_i, g' = silu(G1 gmax + g1),
//       h = silu(D1[:, :64] f_i + D1[:, 64:] g' + d1), r_i = D2 h + d2,  U_i = u_i + r_i on the rows Eq. (2) keeps
//   Phi does not see u_i: dL/dalpha and the K part of dL/ddelta come from backward_kernel (k_backward.cu) run
//   without a residual; this file adds dL/dPhi-weights and the part of dL/ddelta that enters through x_i.
//
// The sum over the rows of the broadcast global feature and the max-pool separate the passes:
//   pn_bwd_encode_kernel   f_i; column max with its arg-max node (64-bit keys: value | ~node) -> gkey, gmax
//   pn_global_env_kernel   (k_pointnet_fp32.cu) c = D1[:, 64:] g' + d1 -> cvec
//   pn_bwd_sum_kernel      S = sum_i dL/dzc_i  (zc = the decoder's hidden pre-activation)           -> ssum
//   pn_bwd_global_kernel   dL/dg' = D1[:, 64:]^T S, through the global MLP -> dL/dgmax (ggmax); dG1, dg1, dD1[:, 64:], dd1
//   pn_bwd_node_kernel     everything per node: decoder, arg-max routing of ggmax, encoder; dD2, dd2, dD1[:, :64], dE2,
//                          de2, dE1, de1 as CTA-level products accumulated in registers over the CTA's items; dL/ddelta
// d_grad_weights layout: E1[64x9] e1[64] E2[64x64] e2[64] G1[64x64] g1[64] D1[64x128] d1[64] D2[3x64] d2[3].
#include "etac_internal.h"
#include "pointnet_fp32.cuh"

namespace etac {

namespace {
constexpr int kOffE1 = 0, kOffe1 = 576, kOffE2 = 640, kOffe2 = 4736, kOffG1 = 4800, kOffg1 = 8896, kOffD1 = 8960,
              kOffd1 = 17152, kOffD2 = 17216, kOffd2 = 17408;
static_assert(kOffd2 + 3 == ETAC_GRAD_WEIGHTS_POINTNET_LEN, "d_grad_weights layout");

__device__ __forceinline__ void silu_val_grad(float z, float& y, float& dy) {
  const float s = 1.0f / (1.0f + expf(-z));
  y = z * s;
  dy = s * (1.0f + z * (1.0f - s));
}
__device__ __forceinline__ float silu_grad(float z) {
  const float s = 1.0f / (1.0f + expf(-z));
  return s * (1.0f + z * (1.0f - s));
}
// rows of a contacting (env, patch) that carry an upstream gradient: Eq. (2) overwrites the active rows with u^
__device__ __forceinline__ bool row_carries(const DevModel& m, float delta_i) {
  return !(m.active_mode == ETAC_ACTIVE_PASSTHROUGH && delta_i > 0.0f);
}
}  // namespace

// ------------------------------------------------------------------------------------------------ encode + arg-max
__global__ void __launch_bounds__(kGatherChunk) pn_bwd_encode_kernel(DevModel m, StepIO io) {
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
  const int64_t base = ((int64_t)ch.patch * m.max_envs + e) * 64;
  // key = order-preserving bits of f in the high word, ~node in the low word: the max picks the largest value and,
  // among equal values, the smallest node index (the first occurrence, as an arg-max over the rows does)
  unsigned long long mine = 0ull;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      unsigned long long key = valid ? (((unsigned long long)float_key(f[32 * half + k]) << 32) | (uint32_t)(~(uint32_t)g)) : 0ull;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
      }
      if (lane == k) mine = key;
    }
    atomicMax(m.pn_gkey + base + 32 * half + lane, mine);
    atomicMax(m.gmax + base + 32 * half + lane, (uint32_t)(mine >> 32));
  }
}

// ------------------------------------------------------------------------------------------------ S = sum_i dL/dzc_i
__global__ void __launch_bounds__(kGatherChunk) pn_bwd_sum_kernel(DevModel m, StepIO io, const float* __restrict__ grad_out) {
  extern __shared__ float s_w[];
  const int e = blockIdx.x / m.n_chunks;
  const ChunkInfo ch = m.chunk[blockIdx.x - e * m.n_chunks];
  if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) return;
  const int t = threadIdx.x, lane = t & 31;
  for (int k = t; k < kPnW32Floats; k += kGatherChunk) s_w[k] = m.pn_w32[k];
  __syncthreads();
  const bool valid = t < ch.count;
  const int g = ch.node0 + (valid ? t : 0);
  const float4 pos = m.pos4[g], nn = m.nrm4[g];
  const float d = m.delta[(int64_t)e * m.n_nodes + g];
  float g0 = 0.f, g1 = 0.f, g2 = 0.f;
  if (valid && row_carries(m, d)) {
    const float* go = grad_out + ((int64_t)e * m.n_nodes + g) * 3;
    g0 = go[0], g1 = go[1], g2 = go[2];
  }
  // (a warp none of whose rows carries a gradient adds nothing)
  if (!__any_sync(0xffffffffu, g0 != 0.0f || g1 != 0.0f || g2 != 0.0f)) return;
  const float x9[9] = {pos.x, pos.y, pos.z, nn.x, nn.y, nn.z, -d * nn.x, -d * nn.y, -d * nn.z};
  float f[64];
  pn_features(s_w, x9, f);
  const float *D1a = s_w + 576 + 64 + 4096 + 64, *D2 = D1a + 4096;
  const int64_t base = ((int64_t)ch.patch * m.max_envs + e) * 64;
  const float* __restrict__ cv = m.cvec + base;
  float mine = 0.f;  // lane l keeps the warp's sums of columns l and 32 + l
  for (int k2 = 0; k2 < 64; ++k2) {
    float s = cv[k2];
    const float4* w = reinterpret_cast<const float4*>(D1a + k2 * 64);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const float4 wv = w[k];
      s = fmaf(wv.x, f[4 * k], s), s = fmaf(wv.y, f[4 * k + 1], s), s = fmaf(wv.z, f[4 * k + 2], s), s = fmaf(wv.w, f[4 * k + 3], s);
    }
    float gz = fmaf(D2[k2], g0, fmaf(D2[64 + k2], g1, D2[128 + k2] * g2)) * silu_grad(s);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) gz += __shfl_xor_sync(0xffffffffu, gz, o);
    if (lane == (k2 & 31)) mine = gz;
    if ((k2 & 31) == 31) atomicAdd(m.pn_ssum + base + (k2 - 31) + lane, mine);
  }
}

// ------------------------------------------------------------------------------------------------ global MLP backward
// One CTA of 64 threads walks kBwdEnvs environments of one patch; thread k owns hidden unit k.  The two 64 x 64
// matrices sit in shared memory with a pitch of 65 floats, so that both M v (thread = output, stride 1 over the
// threads) and M^T v (thread = row) are conflict-free.
constexpr int kBwdEnvs = 64;
__global__ void __launch_bounds__(64) pn_bwd_global_kernel(DevModel m, int n_envs, float* __restrict__ grad_w) {
  const int p = blockIdx.y, k = threadIdx.x;
  __shared__ float sG1[64 * 65], sD1[64 * 65];  // [in j][out n] (DevModel::pn_f32)
  __shared__ float g[64], gp[64], ss[64], gzg[64];
  const float* G1t = m.pn_f32, *g1 = G1t + 4096, *D1gt = g1 + 64;
  float accG1[64], accD1[64];  // rows k of dG1 ([out k][in j]) and of dD1[:, 64:]
  float accg1 = 0.f, accd1 = 0.f;
#pragma unroll
  for (int j = 0; j < 64; ++j) accG1[j] = 0.f, accD1[j] = 0.f;
  bool staged = false;
  for (int e = blockIdx.x * kBwdEnvs; e < min(n_envs, (blockIdx.x + 1) * kBwdEnvs); ++e) {
    if (!m.flags[(int64_t)e * m.n_patches + p]) continue;  // (uniform over the CTA)
    if (!staged) {
      for (int i = k; i < 4096; i += 64) sG1[(i >> 6) * 65 + (i & 63)] = G1t[i], sD1[(i >> 6) * 65 + (i & 63)] = D1gt[i];
      staged = true;
    }
    const int64_t base = ((int64_t)p * m.max_envs + e) * 64;
    __syncthreads();  // previous environment done with the vectors; first pass: matrices staged
    g[k] = key_float(m.gmax[base + k]);
    ss[k] = m.pn_ssum[base + k];
    __syncthreads();
    float zg = g1[k];
#pragma unroll 8
    for (int j = 0; j < 64; ++j) zg = fmaf(sG1[j * 65 + k], g[j], zg);
    float y, dy;
    silu_val_grad(zg, y, dy);
    gp[k] = y;
    // dL/dg'_k = sum_n D1[n][64 + k] S_n = sum_n D1gt[k][n] S_n
    float gg = 0.f;
#pragma unroll 8
    for (int n = 0; n < 64; ++n) gg = fmaf(sD1[k * 65 + n], ss[n], gg);
    const float gz = gg * dy;
    gzg[k] = gz;
    __syncthreads();
    // dL/dgmax_k = sum_n G1[n][k] gzg_n = sum_n G1t[k][n] gzg_n
    float gm = 0.f;
#pragma unroll 8
    for (int n = 0; n < 64; ++n) gm = fmaf(sG1[k * 65 + n], gzg[n], gm);
    m.pn_ggmax[base + k] = gm;
    accg1 += gz, accd1 += ss[k];
#pragma unroll
    for (int j = 0; j < 64; ++j) accG1[j] = fmaf(gz, g[j], accG1[j]), accD1[j] = fmaf(ss[k], gp[j], accD1[j]);
  }
  if (!staged || !grad_w) return;
#pragma unroll
  for (int j = 0; j < 64; ++j) {
    atomicAdd(grad_w + kOffG1 + k * 64 + j, accG1[j]);
    atomicAdd(grad_w + kOffD1 + k * 128 + 64 + j, accD1[j]);
  }
  atomicAdd(grad_w + kOffg1 + k, accg1);
  atomicAdd(grad_w + kOffd1 + k, accd1);
}

// ------------------------------------------------------------------------------------------------ per-node backward
// Persistent grid, one CTA of 256 threads per SM.  A work item is one node chunk (<= 128 nodes of one patch in one
// environment) handled as two halves of kT = 64 nodes; four threads per node, part s owning the hidden units
// 16 s .. 16 s + 15 of every layer.  Every matrix-vector product reads its 64 inputs as a column of a [64][kLd]
// shared-memory array that the previous phase wrote and writes its 16 outputs into another one; the weight
// gradients are products of those arrays over the 64 nodes, accumulated in registers over all items of the CTA.
namespace {
constexpr int kT = 64, kParts = 4, kNodeThreads = kT * kParts, kHp = 64 / kParts, kLd = kT + 1;
struct PnBwdSmem {
  float w[kPnW32Floats + 1];  // E1 e1 E2 e2 D1[:, :64] D2 d2
  float A[64 * kLd];          // silu'(z1) -> dz1
  float B[64 * kLd];          // f1
  float C[64 * kLd];          // silu'(z2) -> dz2
  float D[64 * kLd];          // f
  float H[64 * kLd];          // h (decoder hidden)
  float Z[64 * kLd];          // dzc
  float X[9 * kLd];           // [p, n, u^] per node
  float G[3 * kLd];           // upstream gradient of the rows that carry one
  float L[kParts][3][kT];     // per-part shares of E1[:, 6:9]^T dz1
  float cv[64], gm[64];       // c_(e,p) and dL/dgmax of the item's (env, patch)
  int arg[64];                // arg-max node of every feature column
};
}  // namespace

__global__ void __launch_bounds__(kNodeThreads, 1) pn_bwd_node_kernel(DevModel m, StepIO io, const float* __restrict__ grad_out,
                                                                      float* __restrict__ grad_w, float* __restrict__ grad_delta) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  PnBwdSmem& S = *reinterpret_cast<PnBwdSmem*>(smem_raw);
  const int t = threadIdx.x;
  const int part = t / kT, i = t - part * kT, k0 = part * kHp;
  for (int k = t; k < kPnW32Floats; k += kNodeThreads) S.w[k] = m.pn_w32[k];
  const float *E1 = S.w, *e1 = E1 + 576, *E2 = e1 + 64, *e2 = E2 + 4096, *D1a = e2 + 64, *D2 = D1a + 4096;

  // per-thread shares of the weight gradients: 4 x 4 tiles (rows kt.., columns jt..) of dD1[:, :64] and dE2
  const int kt = 4 * (t & 15), jt = 4 * (t >> 4);
  float gD1[4][4], gE2[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) gD1[a][b] = 0.f, gE2[a][b] = 0.f;
  float gE1[3] = {0.f, 0.f, 0.f};  // dE1 entries t, t + 256, t + 512 (< 576) in [64 x 9] order
  float gD2 = 0.f;                 // t < 192: dD2 entry t in [3 x 64] order
  float gb = 0.f;                  // t < 64: de1[t]; t < 128: de2[t - 64]; 192 <= t < 195: dd2[t - 192]
  __syncthreads();

  const int64_t n_items = (int64_t)m.n_chunks * io.n_envs;
  for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int e = (int)(item / m.n_chunks);
    const ChunkInfo ch = m.chunk[item - (int64_t)e * m.n_chunks];
    if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) continue;
    const int64_t base = ((int64_t)ch.patch * m.max_envs + e) * 64;
    if (t < 64) {
      S.cv[t] = m.cvec[base + t], S.gm[t] = m.pn_ggmax[base + t];
      S.arg[t] = (int)~(uint32_t)(m.pn_gkey[base + t] & 0xffffffffull);
    }
    for (int sub = 0; sub * kT < ch.count; ++sub) {
      const bool valid = sub * kT + i < ch.count;
      const int g = ch.node0 + (valid ? sub * kT + i : 0);
      const float4 pos = m.pos4[g], nn = m.nrm4[g];
      const float d = m.delta[(int64_t)e * m.n_nodes + g];
      const float x9[9] = {pos.x, pos.y, pos.z, nn.x, nn.y, nn.z, -d * nn.x, -d * nn.y, -d * nn.z};
      float g0 = 0.f, g1 = 0.f, g2 = 0.f;
      if (valid && row_carries(m, d)) {
        const float* go = grad_out + ((int64_t)e * m.n_nodes + g) * 3;
        g0 = go[0], g1 = go[1], g2 = go[2];
      }
      if (part == 0) {
#pragma unroll
        for (int c = 0; c < 9; ++c) S.X[c * kLd + i] = valid ? x9[c] : 0.0f;
        S.G[0 * kLd + i] = g0, S.G[1 * kLd + i] = g1, S.G[2 * kLd + i] = g2;
      }
      // ---- encoder layer 1 (this part's 16 units): f1 -> B, silu'(z1) -> A
#pragma unroll
      for (int q = 0; q < kHp; ++q) {
        const int k = k0 + q;
        float z = e1[k], y, dy;
#pragma unroll
        for (int c = 0; c < 9; ++c) z = fmaf(E1[k * 9 + c], x9[c], z);
        silu_val_grad(z, y, dy);
        S.B[k * kLd + i] = y, S.A[k * kLd + i] = dy;
      }
      __syncthreads();  // f1 of every node complete (and cv / gm / arg of the item)
      float v[64];
      // ---- encoder layer 2: f -> D, silu'(z2) -> C
#pragma unroll
      for (int k = 0; k < 64; ++k) v[k] = S.B[k * kLd + i];
#pragma unroll 2
      for (int q = 0; q < kHp; ++q) {
        const int k = k0 + q;
        float za = e2[k], zb = 0.f, y, dy;
        const float4* w = reinterpret_cast<const float4*>(E2 + k * 64);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const float4 wv = w[j];
          za = fmaf(wv.x, v[4 * j], za), zb = fmaf(wv.y, v[4 * j + 1], zb), za = fmaf(wv.z, v[4 * j + 2], za), zb = fmaf(wv.w, v[4 * j + 3], zb);
        }
        silu_val_grad(za + zb, y, dy);
        S.D[k * kLd + i] = y, S.C[k * kLd + i] = dy;
      }
      __syncthreads();  // f complete
      // ---- decoder hidden layer: h -> H, dzc = (D2^T G) silu'(zc) -> Z
#pragma unroll
      for (int k = 0; k < 64; ++k) v[k] = S.D[k * kLd + i];
#pragma unroll 2
      for (int q = 0; q < kHp; ++q) {
        const int k = k0 + q;
        float za = S.cv[k], zb = 0.f, y, dy;
        const float4* w = reinterpret_cast<const float4*>(D1a + k * 64);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const float4 wv = w[j];
          za = fmaf(wv.x, v[4 * j], za), zb = fmaf(wv.y, v[4 * j + 1], zb), za = fmaf(wv.z, v[4 * j + 2], za), zb = fmaf(wv.w, v[4 * j + 3], zb);
        }
        silu_val_grad(za + zb, y, dy);
        S.H[k * kLd + i] = y;
        S.Z[k * kLd + i] = fmaf(D2[k], g0, fmaf(D2[64 + k], g1, D2[128 + k] * g2)) * dy;
      }
      __syncthreads();  // h, dzc complete
      // ---- dL/df = D1[:, :64]^T dzc + the max-pool's share (the arg-max row of column j gets dL/dgmax_j);
      //      dz2 = dL/df silu'(z2) -> C (this part's 16 columns)
#pragma unroll
      for (int k = 0; k < 64; ++k) v[k] = S.Z[k * kLd + i];
      float gh[kHp];
#pragma unroll
      for (int q = 0; q < kHp; ++q) gh[q] = (valid && S.arg[k0 + q] == g) ? S.gm[k0 + q] : 0.0f;
#pragma unroll
      for (int k = 0; k < 64; ++k) {
        const float4* w = reinterpret_cast<const float4*>(D1a + k * 64 + k0);
#pragma unroll
        for (int q = 0; q < kHp / 4; ++q) {
          const float4 wv = w[q];
          gh[4 * q + 0] = fmaf(wv.x, v[k], gh[4 * q + 0]), gh[4 * q + 1] = fmaf(wv.y, v[k], gh[4 * q + 1]);
          gh[4 * q + 2] = fmaf(wv.z, v[k], gh[4 * q + 2]), gh[4 * q + 3] = fmaf(wv.w, v[k], gh[4 * q + 3]);
        }
      }
#pragma unroll
      for (int q = 0; q < kHp; ++q) S.C[(k0 + q) * kLd + i] *= gh[q];
      // weight gradients of the decoder over the 64 nodes (H, Z, D, G are complete and not rewritten below)
#pragma unroll 4
      for (int n = 0; n < kT; ++n) {
        float a[4], b[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) a[q] = S.Z[(kt + q) * kLd + n], b[q] = S.D[(jt + q) * kLd + n];
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int r = 0; r < 4; ++r) gD1[q][r] = fmaf(a[q], b[r], gD1[q][r]);
      }
      if (t < 192) {  // dD2[c][k] = sum_n G_c[n] h_k[n], (c, k) = (t / 64, t % 64)
        const float *gr = S.G + (t >> 6) * kLd, *hr = S.H + (t & 63) * kLd;
        float s0 = 0.f, s1 = 0.f;
        for (int n = 0; n < kT; n += 2) s0 = fmaf(gr[n], hr[n], s0), s1 = fmaf(gr[n + 1], hr[n + 1], s1);
        gD2 += s0 + s1;
      } else if (t >= 192 && t < 195) {  // dd2
        float s = 0.f;
        for (int n = 0; n < kT; ++n) s += S.G[(t - 192) * kLd + n];
        gb += s;
      }
      __syncthreads();  // dz2 complete
      // ---- dL/df1 = E2^T dz2, dz1 = dL/df1 silu'(z1) -> A, share of E1[:, 6:9]^T dz1
#pragma unroll
      for (int k = 0; k < 64; ++k) v[k] = S.C[k * kLd + i];
#pragma unroll
      for (int q = 0; q < kHp; ++q) gh[q] = 0.f;
#pragma unroll
      for (int k = 0; k < 64; ++k) {
        const float4* w = reinterpret_cast<const float4*>(E2 + k * 64 + k0);
#pragma unroll
        for (int q = 0; q < kHp / 4; ++q) {
          const float4 wv = w[q];
          gh[4 * q + 0] = fmaf(wv.x, v[k], gh[4 * q + 0]), gh[4 * q + 1] = fmaf(wv.y, v[k], gh[4 * q + 1]);
          gh[4 * q + 2] = fmaf(wv.z, v[k], gh[4 * q + 2]), gh[4 * q + 3] = fmaf(wv.w, v[k], gh[4 * q + 3]);
        }
      }
      float p0 = 0.f, p1 = 0.f, p2 = 0.f;
#pragma unroll
      for (int q = 0; q < kHp; ++q) {
        const int k = k0 + q;
        const float gz1 = gh[q] * S.A[k * kLd + i];
        S.A[k * kLd + i] = gz1;
        p0 = fmaf(E1[k * 9 + 6], gz1, p0), p1 = fmaf(E1[k * 9 + 7], gz1, p1), p2 = fmaf(E1[k * 9 + 8], gz1, p2);
      }
      S.L[part][0][i] = p0, S.L[part][1][i] = p1, S.L[part][2][i] = p2;
      // dE2 = dz2^T f1 (C and B are complete)
#pragma unroll 4
      for (int n = 0; n < kT; ++n) {
        float a[4], b[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) a[q] = S.C[(kt + q) * kLd + n], b[q] = S.B[(jt + q) * kLd + n];
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int r = 0; r < 4; ++r) gE2[q][r] = fmaf(a[q], b[r], gE2[q][r]);
      }
      __syncthreads();  // dz1 and the shares of E1[:, 6:9]^T dz1 complete
      // ---- dE1 = dz1^T X, de1, de2; dL/ddelta_i = -n_i . dL/du^_i for the nodes in contact
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        const int idx = t + q * kNodeThreads;  // (k, c) = (idx / 9, idx % 9)
        if (idx < 576) {
          const float *zr = S.A + (idx / 9) * kLd, *xr = S.X + (idx % 9) * kLd;
          float s0 = 0.f, s1 = 0.f;
          for (int n = 0; n < kT; n += 2) s0 = fmaf(zr[n], xr[n], s0), s1 = fmaf(zr[n + 1], xr[n + 1], s1);
          gE1[q] += s0 + s1;
        }
      }
      if (t < 128) {
        const float* zr = (t < 64 ? S.A : S.C) + (t & 63) * kLd;
        float s0 = 0.f, s1 = 0.f;
        for (int n = 0; n < kT; n += 2) s0 += zr[n], s1 += zr[n + 1];
        gb += s0 + s1;
      }
      if (grad_delta && part == 0 && valid && d > 0.0f) {
        float u0 = 0.f, u1 = 0.f, u2 = 0.f;
#pragma unroll
        for (int s = 0; s < kParts; ++s) u0 += S.L[s][0][i], u1 += S.L[s][1][i], u2 += S.L[s][2][i];
        atomicAdd(grad_delta + (int64_t)e * m.n_nodes + g, -(nn.x * u0 + nn.y * u1 + nn.z * u2));
      }
      __syncthreads();  // the arrays are rewritten by the next half / item
    }
  }

  if (!grad_w) return;
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      atomicAdd(grad_w + kOffD1 + (kt + q) * 128 + jt + r, gD1[q][r]);
      atomicAdd(grad_w + kOffE2 + (kt + q) * 64 + jt + r, gE2[q][r]);
    }
#pragma unroll
  for (int q = 0; q < 3; ++q)
    if (t + q * kNodeThreads < 576) atomicAdd(grad_w + kOffE1 + t + q * kNodeThreads, gE1[q]);
  if (t < 192) atomicAdd(grad_w + kOffD2 + t, gD2);
  if (t < 64) atomicAdd(grad_w + kOffe1 + t, gb);
  else if (t < 128) atomicAdd(grad_w + kOffe2 + t - 64, gb);
  else if (t >= 192 && t < 195) atomicAdd(grad_w + kOffd2 + t - 192, gb);
}

cudaError_t backward_pointnet_configure() {
  cudaError_t e = cudaFuncSetAttribute(pn_bwd_node_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PnBwdSmem));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(pn_bwd_sum_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPnW32Floats * 4);
  return e;
}

// dL/d(PointNet weights) and the share of dL/ddelta that enters through the encoder input; S1 has run (delta, flags).
// *launches receives the number of kernels.  grad_w / grad_delta may be NULL.
cudaError_t launch_backward_pointnet(const DevModel& m, const StepIO& io, const float* grad_out, float* grad_w, float* grad_delta,
                                     int n_sm, int* launches, cudaStream_t s) {
  const size_t cells = (size_t)64 * m.n_patches * m.max_envs;
  cudaError_t e;
  if ((e = cudaMemsetAsync(m.gmax, 0, sizeof(uint32_t) * cells, s)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(m.pn_gkey, 0, sizeof(unsigned long long) * cells, s)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(m.pn_ssum, 0, sizeof(float) * cells, s)) != cudaSuccess) return e;
  const unsigned grid = (unsigned)((int64_t)m.n_chunks * io.n_envs);
  pn_bwd_encode_kernel<<<grid, kGatherChunk, (576 + 64 + 4096 + 64) * 4, s>>>(m, io);
  launch_pointnet_global_env(m, io.n_envs, s);
  pn_bwd_sum_kernel<<<grid, kGatherChunk, kPnW32Floats * 4, s>>>(m, io, grad_out);
  pn_bwd_global_kernel<<<dim3((unsigned)((io.n_envs + kBwdEnvs - 1) / kBwdEnvs), (unsigned)m.n_patches), 64, 0, s>>>(m, io.n_envs, grad_w);
  pn_bwd_node_kernel<<<n_sm, kNodeThreads, sizeof(PnBwdSmem), s>>>(m, io, grad_out, grad_w, grad_delta);
  *launches = 5;
  return cudaGetLastError();
}

}  // namespace etac

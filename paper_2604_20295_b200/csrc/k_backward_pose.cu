// etac_backward, pose part: chains dL/ddelta (k_backward.cu / k_backward_pointnet.cu) to the poses the penetration came
// from (delta from SDFs between nodes and objects; Table I: differentiability).
//
// For a node in contact  delta_i = -phi_k*(y),  y = R_k^T (x_i - t_k),  x_i = R_p p_i + t_p,  k* = the indenter that
// attains the min of the union (contact set and k* held fixed).  With n_w = R_k grad phi_k*(y), d = x_i - t_k,
// r = x_i - t_p and rotations perturbed on the left in the world frame (R <- exp([theta]x) R):
//     d delta/d t_k = +n_w      d delta/d theta_k = -(n_w x d)
//     d delta/d t_p = -n_w      d delta/d theta_p = -(r x n_w)
// One CTA per (environment, patch): a calibration / trajectory-optimisation step, not on the RL path; fp32 SIMT.
// phi_k is re-evaluated with S1's arithmetic (sdf_device.cuh), so k* is the indenter S1's min picked.
#include "etac_internal.h"
#include "sdf_device.cuh"

namespace etac {

namespace {
constexpr int kPoseThreads = 128;

__device__ __forceinline__ float safe_rcp_len(float a, float b, float c) {
  const float l = sqrtf(fmaf(a, a, fmaf(b, b, c * c)));
  return l > 0.0f ? 1.0f / l : 0.0f;
}

// gradient of the sampled SDF (sdf_grid) in the grid's frame: along an axis on which y is inside the box the
// derivative of the trilinear interpolant, along a clamped axis the distance term's (y - clamp(y)) / |y - clamp(y)|
__device__ __forceinline__ void sdf_grid_grad(const GridDesc& g, const float* y, float* gl) {
  const int n[3] = {g.nx, g.ny, g.nz};
  float yc[3], f[3];
  int i[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float lo = g.o[a], hi = __fadd_rn(lo, __fmul_rn(g.h, (float)(n[a] - 1)));
    yc[a] = fminf(fmaxf(y[a], lo), hi);
    const float t = __fmul_rn(__fsub_rn(yc[a], lo), g.inv_h);
    const float fl = fminf(floorf(t), (float)(n[a] - 2));
    i[a] = (int)fl;
    f[a] = t - fl;
  }
  const float* v = g.v + ((int64_t)i[2] * g.ny + i[1]) * g.nx + i[0];
  const int64_t sy = g.nx, sz = (int64_t)g.nx * g.ny;
  const float c000 = v[0], c001 = v[1], c010 = v[sy], c011 = v[sy + 1];  // c[z][y][x]
  const float c100 = v[sz], c101 = v[sz + 1], c110 = v[sz + sy], c111 = v[sz + sy + 1];
  auto lerp = [](float a, float b, float t) { return fmaf(t, b - a, a); };
  const float dx = lerp(lerp(c001 - c000, c011 - c010, f[1]), lerp(c101 - c100, c111 - c110, f[1]), f[2]);
  const float dy = lerp(lerp(c010 - c000, c011 - c001, f[0]), lerp(c110 - c100, c111 - c101, f[0]), f[2]);
  const float dz = lerp(lerp(c100 - c000, c101 - c001, f[0]), lerp(c110 - c010, c111 - c011, f[0]), f[1]);
  const float off[3] = {y[0] - yc[0], y[1] - yc[1], y[2] - yc[2]};
  const float rl = safe_rcp_len(off[0], off[1], off[2]);
  const float d[3] = {dx, dy, dz};
#pragma unroll
  for (int a = 0; a < 3; ++a) gl[a] = (off[a] == 0.0f ? d[a] * g.inv_h : 0.0f) + off[a] * rl;
}

// n_w = R_k grad phi_k(R_k^T (X - t_k)): the SDF's gradient at world point X, in the world frame
__device__ __forceinline__ void sdf_grad_world(const SInd& s, const float* X, const GridDesc* grids, float* nw) {
  const float d0 = X[0] - s.t[0], d1 = X[1] - s.t[1], d2 = X[2] - s.t[2];
  const float y[3] = {fmaf(s.R[0], d0, fmaf(s.R[3], d1, s.R[6] * d2)), fmaf(s.R[1], d0, fmaf(s.R[4], d1, s.R[7] * d2)),
                      fmaf(s.R[2], d0, fmaf(s.R[5], d1, s.R[8] * d2))};
  float gl[3] = {0.f, 0.f, 0.f};
  if (s.type == ETAC_IND_SPHERE) {
    const float rl = safe_rcp_len(y[0], y[1], y[2]);
    gl[0] = y[0] * rl, gl[1] = y[1] * rl, gl[2] = y[2] * rl;
  } else if (s.type == ETAC_IND_BOX) {
    const float q[3] = {fabsf(y[0]) - s.prm[0], fabsf(y[1]) - s.prm[1], fabsf(y[2]) - s.prm[2]};
    const float o[3] = {fmaxf(q[0], 0.f), fmaxf(q[1], 0.f), fmaxf(q[2], 0.f)};
    const float rl = safe_rcp_len(o[0], o[1], o[2]);
    if (rl > 0.0f) {  // outside: towards the closest point of the box
#pragma unroll
      for (int a = 0; a < 3; ++a) gl[a] = copysignf(o[a] * rl, y[a]);
    } else {          // inside: the face that is closest
      const int a = (q[0] >= q[1] && q[0] >= q[2]) ? 0 : (q[1] >= q[2] ? 1 : 2);
      gl[a] = copysignf(1.0f, y[a]);
    }
  } else if (s.type == ETAC_IND_CAPSULE) {
    const float L = s.prm[1];
    const float dz = y[2] - fminf(fmaxf(y[2], -L), L);
    const float rl = safe_rcp_len(y[0], y[1], dz);
    gl[0] = y[0] * rl, gl[1] = y[1] * rl, gl[2] = dz * rl;
  } else if (s.type == ETAC_IND_GRID) {
    const GridDesc& g = grids[min(max((int)s.prm[0], 0), kMaxGrids - 1)];
    if (g.v) sdf_grid_grad(g, y, gl);
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) nw[a] = fmaf(s.R[3 * a], gl[0], fmaf(s.R[3 * a + 1], gl[1], s.R[3 * a + 2] * gl[2]));
}

struct PoseSmem {
  float R[9], t[3];
  float acc_patch[6];
};
}  // namespace

// grid = n_envs * n_patches; grad_ind (may be NULL) must be zero on entry, grad_patch (may be NULL) is overwritten
__global__ void __launch_bounds__(kPoseThreads) pose_grad_kernel(DevModel m, StepIO io, const float* __restrict__ g_delta,
                                                                 float* __restrict__ grad_ind, float* __restrict__ grad_patch) {
  __shared__ PoseSmem sm;
  extern __shared__ __align__(16) uint8_t pose_dyn[];  // SInd[max_ind] | float acc_ind[max_ind][6]
  SInd* s_ind = reinterpret_cast<SInd*>(pose_dyn);
  float* acc_ind = reinterpret_cast<float*>(s_ind + m.max_ind);
  const int e = blockIdx.x / m.n_patches, p = blockIdx.x - e * m.n_patches;
  const PatchInfo pi = m.patch[p];
  const int tid = threadIdx.x;
  for (int k = tid; k < m.max_ind; k += kPoseThreads) s_ind[k] = load_indenter(io.ind + (int64_t)e * m.max_ind + k);
  for (int a = tid; a < m.max_ind * 6; a += kPoseThreads) acc_ind[a] = 0.0f;
  if (tid < 6) sm.acc_patch[tid] = 0.0f;
  if (tid == 32) {
    if (io.patch_pose) {
      const float* q = io.patch_pose + ((int64_t)e * m.n_patches + p) * 7;
      quat_to_rot(q + 3, sm.R);
      sm.t[0] = q[0], sm.t[1] = q[1], sm.t[2] = q[2];
    } else {
#pragma unroll
      for (int a = 0; a < 9; ++a) sm.R[a] = (a % 4 == 0) ? 1.0f : 0.0f;
      sm.t[0] = sm.t[1] = sm.t[2] = 0.0f;
    }
  }
  __syncthreads();
  float ap[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  const float* gd = g_delta + (int64_t)e * m.n_nodes + pi.off;
  for (int i = tid; i < pi.n; i += kPoseThreads) {
    const float g = gd[i];
    if (g == 0.0f) continue;  // not in contact (or no gradient)
    const float4 x = m.pos4[pi.off + i];
    float X[3];
    to_world(sm.R, sm.t, x.x, x.y, x.z, X[0], X[1], X[2]);
    float best = __int_as_float(0x7f800000);
    int ks = -1;
    for (int k = 0; k < m.max_ind; ++k) {
      if (s_ind[k].skip1 == p + 1) continue;
      const float phi = sdf_one<true>(s_ind[k], X[0], X[1], X[2], m.grid);
      if (phi < best) best = phi, ks = k;  // first minimum in slot order, as S1's running fminf
    }
    if (ks < 0) continue;
    const SInd& s = s_ind[ks];
    float nw[3];
    sdf_grad_world(s, X, m.grid, nw);
    const float d[3] = {X[0] - s.t[0], X[1] - s.t[1], X[2] - s.t[2]};
    const float r[3] = {X[0] - sm.t[0], X[1] - sm.t[1], X[2] - sm.t[2]};
    // indenter: dL/dt_k += g n_w ; dL/dtheta_k += -g (n_w x d)
    float* ai = acc_ind + ks * 6;
    atomicAdd(ai + 0, g * nw[0]), atomicAdd(ai + 1, g * nw[1]), atomicAdd(ai + 2, g * nw[2]);
    atomicAdd(ai + 3, -g * (nw[1] * d[2] - nw[2] * d[1]));
    atomicAdd(ai + 4, -g * (nw[2] * d[0] - nw[0] * d[2]));
    atomicAdd(ai + 5, -g * (nw[0] * d[1] - nw[1] * d[0]));
    // patch: dL/dt_p += -g n_w ; dL/dtheta_p += -g (r x n_w)
    ap[0] -= g * nw[0], ap[1] -= g * nw[1], ap[2] -= g * nw[2];
    ap[3] -= g * (r[1] * nw[2] - r[2] * nw[1]);
    ap[4] -= g * (r[2] * nw[0] - r[0] * nw[2]);
    ap[5] -= g * (r[0] * nw[1] - r[1] * nw[0]);
  }
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    float v = ap[c];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((tid & 31) == 0 && v != 0.0f) atomicAdd(&sm.acc_patch[c], v);
  }
  __syncthreads();
  if (grad_patch && tid < 6) grad_patch[((int64_t)e * m.n_patches + p) * 6 + tid] = io.patch_pose ? sm.acc_patch[tid] : 0.0f;
  if (grad_ind)
    for (int a = tid; a < m.max_ind * 6; a += kPoseThreads)
      if (acc_ind[a] != 0.0f) atomicAdd(grad_ind + (int64_t)e * m.max_ind * 6 + a, acc_ind[a]);
}

cudaError_t launch_backward_pose(const DevModel& m, const StepIO& io, const float* g_delta, float* grad_ind, float* grad_patch,
                                 cudaStream_t s) {
  if (io.n_envs == 0 || m.n_patches == 0) return cudaSuccess;
  const size_t smem = (sizeof(SInd) + 6 * sizeof(float)) * (size_t)m.max_ind;  // <= 48 KB: etac_backward checks kMaxPoseGradIndenters
  pose_grad_kernel<<<(unsigned)((int64_t)io.n_envs * m.n_patches), kPoseThreads, smem, s>>>(m, io, g_delta, grad_ind, grad_patch);
  return cudaGetLastError();
}

}  // namespace etac

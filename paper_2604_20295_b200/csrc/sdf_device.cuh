// Device helpers of S1 shared by k_sdf.cu and k_backward_pose.cu: the indenter as the kernels hold it,
// quaternion -> rotation, the signed distance of every indenter type and the transform of a mesh point into the world
// frame.  The arithmetic of phi is single-rounded fp32 in a fixed order (no FMA contraction ->
// __fmul_rn / __fadd_rn / __fsub_rn / __fsqrt_rn) so that an independent fp32 implementation reproduces the contact
// decision.
#pragma once
#include "etac_internal.h"

namespace etac {

struct SInd {
  int type;
  int skip1;  // etac_indenter::skip_patch1 (self-contact: patch skip1 - 1 ignores this indenter)
  float prm[3];
  float t[3];
  float R[9];
  float rb2;  // square of a radius around t beyond which the shape's SDF is > 0.05 (conservative; +inf: unknown, -1: no shape)
};

__device__ __forceinline__ void quat_to_rot(const float* q, float* R) {
  const float x = q[0], y = q[1], z = q[2], w = q[3];
  const float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z);
  const float xy = __fmul_rn(x, y), xz = __fmul_rn(x, z), yz = __fmul_rn(y, z);
  const float wx = __fmul_rn(w, x), wy = __fmul_rn(w, y), wz = __fmul_rn(w, z);
  R[0] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(yy, zz)));
  R[1] = __fmul_rn(2.0f, __fsub_rn(xy, wz));
  R[2] = __fmul_rn(2.0f, __fadd_rn(xz, wy));
  R[3] = __fmul_rn(2.0f, __fadd_rn(xy, wz));
  R[4] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, zz)));
  R[5] = __fmul_rn(2.0f, __fsub_rn(yz, wx));
  R[6] = __fmul_rn(2.0f, __fsub_rn(xz, wy));
  R[7] = __fmul_rn(2.0f, __fadd_rn(yz, wx));
  R[8] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, yy)));
}

__device__ __forceinline__ float len3(float a, float b, float c) {
  return __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(a, a), __fmul_rn(b, b)), __fmul_rn(c, c)));
}

// Sampled SDF (R21): clamp to the grid's box, trilinear interpolation of the samples
// (x, then y, then z; lerp = a + f*(b - a)), plus the distance from the point to the box.  Same
// single-rounded operations in the same order as the oracle's fp32 twin.
__device__ __forceinline__ float sdf_grid(const GridDesc& g, float y0, float y1, float y2) {
  const float y[3] = {y0, y1, y2};
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
    f[a] = __fsub_rn(t, fl);
  }
  const float* v = g.v + ((int64_t)i[2] * g.ny + i[1]) * g.nx + i[0];
  const int64_t sy = g.nx, sz = (int64_t)g.nx * g.ny;
  auto lerp = [](float a, float b, float t) { return __fadd_rn(a, __fmul_rn(t, __fsub_rn(b, a))); };
  const float c00 = lerp(v[0], v[1], f[0]), c10 = lerp(v[sy], v[sy + 1], f[0]);
  const float c01 = lerp(v[sz], v[sz + 1], f[0]), c11 = lerp(v[sz + sy], v[sz + sy + 1], f[0]);
  const float c = lerp(lerp(c00, c10, f[1]), lerp(c01, c11, f[1]), f[2]);
  return __fadd_rn(c, len3(__fsub_rn(y0, yc[0]), __fsub_rn(y1, yc[1]), __fsub_rn(y2, yc[2])));
}

// Signed distance of world point X to one indenter (+inf for an empty slot).
template <bool kGrid>
__device__ __forceinline__ float sdf_one(const SInd& s, float X0, float X1, float X2, const GridDesc* grids) {
  if (s.type == ETAC_IND_NONE) return __int_as_float(0x7f800000);
  const float d0 = __fsub_rn(X0, s.t[0]), d1 = __fsub_rn(X1, s.t[1]), d2 = __fsub_rn(X2, s.t[2]);
  // y = R^T d
  const float y0 = __fadd_rn(__fadd_rn(__fmul_rn(s.R[0], d0), __fmul_rn(s.R[3], d1)), __fmul_rn(s.R[6], d2));
  const float y1 = __fadd_rn(__fadd_rn(__fmul_rn(s.R[1], d0), __fmul_rn(s.R[4], d1)), __fmul_rn(s.R[7], d2));
  const float y2 = __fadd_rn(__fadd_rn(__fmul_rn(s.R[2], d0), __fmul_rn(s.R[5], d1)), __fmul_rn(s.R[8], d2));
  if (s.type == ETAC_IND_SPHERE) return __fsub_rn(len3(y0, y1, y2), s.prm[0]);
  if constexpr (kGrid) {  // compiled only into the variants launched once a grid is registered
    if (s.type == ETAC_IND_GRID) {
      const GridDesc& g = grids[min(max((int)s.prm[0], 0), kMaxGrids - 1)];
      return g.v ? sdf_grid(g, y0, y1, y2) : __int_as_float(0x7f800000);
    }
  } else {
    if (s.type == ETAC_IND_GRID) return __int_as_float(0x7f800000);  // no grid registered: empty slot
  }
  if (s.type == ETAC_IND_BOX) {
    const float q0 = __fsub_rn(fabsf(y0), s.prm[0]);
    const float q1 = __fsub_rn(fabsf(y1), s.prm[1]);
    const float q2 = __fsub_rn(fabsf(y2), s.prm[2]);
    const float outside = len3(fmaxf(q0, 0.0f), fmaxf(q1, 0.0f), fmaxf(q2, 0.0f));
    const float inside = fminf(fmaxf(fmaxf(q0, q1), q2), 0.0f);
    return __fadd_rn(outside, inside);
  }
  // capsule along local z
  const float L = s.prm[1];
  const float cz = fminf(fmaxf(y2, -L), L);
  return __fsub_rn(len3(y0, y1, __fsub_rn(y2, cz)), s.prm[0]);
}

// Union signed distance at world point X: min over the slots in slot order.
template <bool kGrid>
__device__ __forceinline__ float union_sdf(const SInd* __restrict__ ind, int n_ind, float X0, float X1, float X2,
                                           const GridDesc* grids, int p1) {  // p1 = patch + 1 (self-contact skip)
  float phi = __int_as_float(0x7f800000);
  for (int k = 0; k < n_ind; ++k)
    if (ind[k].skip1 != p1) phi = fminf(phi, sdf_one<kGrid>(ind[k], X0, X1, X2, grids));
  return phi;
}

// Lower bound of the union SDF over a ball of radius rad around X, for the conservative culls:
// the analytic SDFs are 1-Lipschitz; a sampled one is bounded by sqrt(3) inside its box (each
// partial derivative of the trilinear interpolant <= the samples' Lipschitz constant) plus 1
// for the distance term outside.
template <bool kGrid>
__device__ __forceinline__ float union_sdf_lower(const SInd* __restrict__ ind, int n_ind, float X0, float X1, float X2,
                                                 float rad, const GridDesc* grids, int p1) {
  float lo = __int_as_float(0x7f800000);
  for (int k = 0; k < n_ind; ++k) {
    if (ind[k].skip1 == p1) continue;
    const float L = (kGrid && ind[k].type == ETAC_IND_GRID) ? 2.7320508f : 1.0f;
    lo = fminf(lo, sdf_one<kGrid>(ind[k], X0, X1, X2, grids) - L * rad);
  }
  return lo;
}

__device__ __forceinline__ SInd load_indenter(const etac_indenter* __restrict__ p) {
  SInd s;
  s.type = p->type;
  s.skip1 = p->skip_patch1;
  s.prm[0] = p->param[0], s.prm[1] = p->param[1], s.prm[2] = p->param[2];
  s.t[0] = p->pose[0], s.t[1] = p->pose[1], s.t[2] = p->pose[2];
  quat_to_rot(p->pose + 3, s.R);
  // bounding radius of the shape around its origin: sphere r, box |half extents|, capsule r + L; sampled grids: unknown
  const float b = s.type == ETAC_IND_SPHERE  ? s.prm[0]
                  : s.type == ETAC_IND_BOX   ? sqrtf(s.prm[0] * s.prm[0] + s.prm[1] * s.prm[1] + s.prm[2] * s.prm[2])
                  : s.type == ETAC_IND_CAPSULE ? s.prm[0] + s.prm[1]
                                               : __int_as_float(0x7f800000);
  const float rb = fmaf(fabsf(b), 1.001f, 0.05f);
  s.rb2 = s.type == ETAC_IND_NONE ? -1.0f : rb * rb;
  return s;
}

// world position of mesh point x under patch pose (R, t): one fixed order of single-rounded operations
__device__ __forceinline__ void to_world(const float* R, const float* t, float x, float y, float z, float& X0, float& X1,
                                         float& X2) {
  X0 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(R[0], x), __fmul_rn(R[1], y)), __fmul_rn(R[2], z)), t[0]);
  X1 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(R[3], x), __fmul_rn(R[4], y)), __fmul_rn(R[5], z)), t[1]);
  X2 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(R[6], x), __fmul_rn(R[7], y)), __fmul_rn(R[8], z)), t[2]);
}

}  // namespace etac

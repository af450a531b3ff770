// etac_mesh_to_sdf_grid: samples the signed distance field of a closed triangle mesh ("SDFs between
// nodes and object meshes") on a regular grid, in the layout etac_set_sdf_grid takes.  A set-up utility, not on the
// step's path: brute force, one thread per grid point over all triangles (staged through shared memory),
//   distance = min over the triangles of the distance to the closest point of the triangle (vertex / edge / face
//              regions of the point's projection),
//   inside   = |winding number| >= 1/2, the winding number being the sum of the triangles' signed solid angles
//              (2 atan2(a.(b x c), |a||b||c| + (a.b)|c| + (b.c)|a| + (c.a)|b|)) over 4 pi,
// fp32 with the triangle translated to the query point first (the cancellations of the region tests then scale with
// the distance to the triangle, not with the coordinates).
#include "etac_internal.h"

namespace etac {

namespace {
constexpr int kTriChunk = 256, kMeshThreads = 128;

struct V3 {
  float x, y, z;
};
__device__ __forceinline__ V3 sub(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ float dot(V3 a, V3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ V3 axpy(V3 a, float s, V3 d) { return {fmaf(s, d.x, a.x), fmaf(s, d.y, a.y), fmaf(s, d.z, a.z)}; }
__device__ __forceinline__ V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }

// squared distance from the origin to the triangle (a, b, c)
__device__ __forceinline__ float tri_dist2(V3 a, V3 b, V3 c) {
  const V3 ab = sub(b, a), ac = sub(c, a);
  const float d1 = -dot(ab, a), d2 = -dot(ac, a);  // ap = -a
  if (d1 <= 0.f && d2 <= 0.f) return dot(a, a);
  const float d3 = -dot(ab, b), d4 = -dot(ac, b);
  if (d3 >= 0.f && d4 <= d3) return dot(b, b);
  const float vc = d1 * d4 - d3 * d2;
  if (vc <= 0.f && d1 >= 0.f && d3 <= 0.f) {
    const V3 q = axpy(a, d1 / (d1 - d3), ab);
    return dot(q, q);
  }
  const float d5 = -dot(ab, c), d6 = -dot(ac, c);
  if (d6 >= 0.f && d5 <= d6) return dot(c, c);
  const float vb = d5 * d2 - d1 * d6;
  if (vb <= 0.f && d2 >= 0.f && d6 <= 0.f) {
    const V3 q = axpy(a, d2 / (d2 - d6), ac);
    return dot(q, q);
  }
  const float va = d3 * d6 - d5 * d4;
  if (va <= 0.f && (d4 - d3) >= 0.f && (d5 - d6) >= 0.f) {
    const V3 q = axpy(b, (d4 - d3) / ((d4 - d3) + (d5 - d6)), sub(c, b));
    return dot(q, q);
  }
  const float den = 1.0f / (va + vb + vc);
  const V3 q = axpy(axpy(a, vb * den, ab), vc * den, ac);
  return dot(q, q);
}
__device__ __forceinline__ float tri_solid_angle(V3 a, V3 b, V3 c) {
  const float la = sqrtf(dot(a, a)), lb = sqrtf(dot(b, b)), lc = sqrtf(dot(c, c));
  const float det = dot(a, cross(b, c));
  const float den = la * lb * lc + dot(a, b) * lc + dot(b, c) * la + dot(c, a) * lb;
  return 2.0f * atan2f(det, den);
}
}  // namespace

// tri: [n_tri x 9] fp32 (three vertices per triangle); values[(iz*ny + iy)*nx + ix]
__global__ void __launch_bounds__(kMeshThreads) mesh_sdf_grid_kernel(const float* __restrict__ tri, int n_tri, int nx, int ny, int nz,
                                                                     float ox, float oy, float oz, float h, float* __restrict__ values) {
  __shared__ float s_tri[kTriChunk * 9];
  const int64_t idx = (int64_t)blockIdx.x * kMeshThreads + threadIdx.x, total = (int64_t)nx * ny * nz;
  const int ix = (int)(idx % nx), iy = (int)((idx / nx) % ny), iz = (int)(idx / ((int64_t)nx * ny));
  const V3 p = {fmaf(h, (float)ix, ox), fmaf(h, (float)iy, oy), fmaf(h, (float)iz, oz)};
  float best = __int_as_float(0x7f800000), omega = 0.f;
  for (int t0 = 0; t0 < n_tri; t0 += kTriChunk) {
    const int nb = min(kTriChunk, n_tri - t0);
    __syncthreads();
    for (int k = threadIdx.x; k < nb * 9; k += kMeshThreads) s_tri[k] = tri[(int64_t)t0 * 9 + k];
    __syncthreads();
    if (idx < total)
      for (int t = 0; t < nb; ++t) {
        const float* q = s_tri + t * 9;
        const V3 a = sub({q[0], q[1], q[2]}, p), b = sub({q[3], q[4], q[5]}, p), c = sub({q[6], q[7], q[8]}, p);
        best = fminf(best, tri_dist2(a, b, c));
        omega += tri_solid_angle(a, b, c);
      }
  }
  if (idx < total) {
    const float d = sqrtf(best);
    values[idx] = fabsf(omega) >= 6.2831853f ? -d : d;
  }
}

cudaError_t launch_mesh_sdf_grid(const float* tri, int n_tri, int nx, int ny, int nz, const float* origin, float h, float* values,
                                 cudaStream_t s) {
  const int64_t total = (int64_t)nx * ny * nz;
  mesh_sdf_grid_kernel<<<(unsigned)((total + kMeshThreads - 1) / kMeshThreads), kMeshThreads, 0, s>>>(tri, n_tri, nx, ny, nz, origin[0],
                                                                                                      origin[1], origin[2], h, values);
  return cudaGetLastError();
}

}  // namespace etac

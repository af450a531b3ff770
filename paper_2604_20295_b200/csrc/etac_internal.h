// Internal declarations shared by the host API (etac_api.cu) and the kernels.  Not installed.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/etac.h"
#include "../../include/etac_bench.h"

namespace etac {

constexpr int kHidden = 64;
constexpr int kMaxPatches = 1024;

// One sensor patch (contiguous node range; K is zero across patches, R9).
constexpr int kWf32W2t = 4548;  // offset of W2^T in DevModel::wf32 (16-byte aligned, behind the 4547 floats of the blob)

struct PatchInfo {
  int32_t off;        // first node
  int32_t n;          // nodes in the patch
  int32_t uoff;       // first column of the patch in the U^ operand rows (a multiple of 8: TMA wants 16-byte aligned boxes)
  int64_t k32_off;    // element offset of K_p (fp32, [n x n] row-major) in k32
  float alpha;
  float bc[3];        // bounding-sphere centre (patch-local frame)
  float brad;         // bounding-sphere radius
};

// Node chunk of <= kGatherChunk nodes of one patch, for the fp32 gather kernel's grid.
struct ChunkInfo {
  int32_t patch;
  int32_t node0;  // first node (global index)
  int32_t count;
};
constexpr int kGatherChunk = 128;

// tensor-core path tiling: environments per work item (16, or 32 for large patches); the U^ operand and the
// active lists are sized for whole tiles of the larger one
constexpr int kMaxTE = 32;
// Block-sparse contraction: S1 records, per contacting (patch, slot), which 64-node k-blocks of the patch hold an
// active node (kKbWords x 32 bits; k-blocks beyond that are always contracted)
constexpr int kKbWords = 8;

// Shared-memory image of the MLP weights for the tensor-core path (bf16, UMMA K-major
// SWIZZLE_NONE core-matrix layout; see k_fused.cu).
constexpr int kW1ImgBytes = 64 * 16 * 2;   // N=64,  K=16   (9 inputs + bias column)
constexpr int kW2ImgBytes = 64 * 80 * 2;   // N=64,  K=80   (64 + bias column, padded to 5 k-steps)
// The output layer (3 x 64) is not an MMA: the epilogue applies it with FFMAs to the fp32 SiLU
// outputs it holds in registers (DevModel::wout), which saves one tensor-core round trip per unit.
constexpr int kWImgBytes = kW1ImgBytes + kW2ImgBytes;
// PointNet form: E1 [64 x 16] | E2 [64 x 80] | D1[:, 0:64] [64 x 80, zero bias column] | D2 [16 x 80]
constexpr int kPnImgBytes = kW1ImgBytes + 2 * kW2ImgBytes;

// Active node of a contacting (env, patch) pair, for the gather form of the propagation:
// u^ of the node (fp32) and its index within the patch.
struct __align__(16) ActiveEntry {
  float ux, uy, uz;
  int32_t j;
};

// what S1 writes besides delta / flags / env lists
enum : int { kS1WriteUhat = 1, kS1WriteAlist = 2, kS1FillOut = 4, kS1Bucket = 8 };

// Sampled SDF of an object (ETAC_IND_GRID): values[(iz*ny + iy)*nx + ix] at origin + h*(ix, iy, iz).
constexpr int kMaxGrids = 8;
struct GridDesc {
  const float* v;  // device, NULL = slot unused
  int32_t nx, ny, nz;
  float o[3];
  float h, inv_h;  // inv_h = 1.0f / h (IEEE fp32 division)
};

struct PairTask;
struct DevModel {
  int32_t n_nodes, n_patches, n_chunks;
  int32_t max_patch_nodes;    // largest patch
  int32_t kw;                 // padded column count of k16 (multiple of 64)
  int32_t ldu;                // row pitch (elements) of uhat_t
  int32_t max_envs, max_ind;
  int32_t resid, active_mode;
  int32_t residual_only;      // ETAC_OPT_ABLATION: passive rows get Phi_p without the linear term
  int32_t group_bytes;        // ETAC_OPT_L2_GROUP_BYTES: U^ operand bytes of one group of env tiles (fused kernel)
  int32_t ablation;           // ETAC_ABLATE_* (LINEAR_ONLY / NO_PROPAGATION select other kernels on the host)
  const float4* pos4;         // [N] (x,y,z,0)
  const float4* nrm4;         // [N]
  const uint4* a1c;           // [N] constant part of the layer-1 operand of the tensor-core MLP, bf16:
                              //     .x = px (low half), .y = (py, pz), .z = (nx, ny), .w = (nz, 1.0)
  const PatchInfo* patch;     // [P]
  const ChunkInfo* chunk;     // [n_chunks]
  const float* k32;           // per patch [n x n]
  const __nv_bfloat16* k16;   // [N x kw], row i holds K_p[i - off_p][0..n_p) then zeros
  const float* wf32;          // fp32 weights blob: W1u[64x3] | c1t[64 x N] is separate | W2[64x64] b2[64] W3[3x64] b3[3]
                              // | pad | W2^T[64x64] at kWf32W2t
  const float* c1t;           // [64 x N]: W1[:,3:9].[p;n] + b1, transposed for coalescing
  const uint8_t* wimg;        // kWImgBytes
  const uint8_t* wimg_pn;     // kPnImgBytes (ETAC_RESID_POINTNET)
  const float* pn_f32;        // G1^T [in][out] g1[64] D1[:,64:128]^T [in][out] d1[64] (fp32, pn_global_kernel)
  const float* pn_w32;        // E1[64x9] e1 E2[64x64] e2 D1[:, :64] D2[3x64] d2 (fp32: k_pointnet_fp32.cu, k_backward_pointnet.cu)
  uint32_t* gmax;             // [P x max_envs x 64] max-pooled encoder features as order-preserving keys
  float* cvec;                // [P x max_envs x 64] c_(e,p) / 2
  // workspaces of the PointNet backward, [P x max_envs x 64] each (indexed by the environment)
  unsigned long long* pn_gkey;  // column max with its arg-max node: key of the value << 32 | ~node
  float* pn_ssum;               // sum over the rows of dL/d(decoder hidden pre-activation)
  float* pn_ggmax;              // dL/d(max-pooled feature)
  float wout[196];            // output layer of Phi in fp32: W3 (or D2) [3 x 64] row-major, then b3 (d2) at 192..194
  // per-step workspace
  float* delta;               // [max_envs x N]
  __nv_bfloat16* uhat_t;      // [3*max_envs (+pad) x ldu]: row slot*3+c, column = node j
  int32_t* count;             // [P] contacting envs per patch (this step)
  int32_t* envlist;           // [P x max_envs]
  uint8_t* flags;             // [max_envs x P]
  uint32_t* kbmap;            // [P x max_envs x kKbWords] active k-block bitmaps of the contacting pairs (bf16 contexts)
  uint32_t* kbtile;           // [P x kbtile_stride x kKbWords] union of the bitmaps per tile of 32 slots (kbtile_kernel)
  int32_t kbtile_stride;      // tiles per patch in kbtile
  // S1 bucketing of the contacting environments of a large patch by the position of their contact (first active
  // k-block), so that the environments of a tile share their active k-blocks: counting sort
  int32_t* khist;             // [P x 256] environments per key (zeroed per step), NULL = no bucketing on this context
  int32_t* kcursor;           // [P x 256] running rank inside a key (zeroed per step)
  uint8_t* keybuf;            // [max_envs x P] key of every contacting pair
  struct PairTask* tasks;     // [max_envs x P] S1 task list of the cull / evaluate kernel pair (many patches, one indenter)
  int32_t* ntask;             // [1], behind count[P] (zeroed with it)
  int32_t* wq;                // [2], behind ntask: item counter of the fused kernel's dynamic item order and the
                              // number of CTAs that are done with it (zeroed with count; the kernel leaves them at zero)
  GridDesc grid[kMaxGrids];   // sampled-SDF objects (etac_set_sdf_grid)
  ActiveEntry* alist;         // [max_envs (slots) x ldu]: the active nodes of (slot, patch p) start at
                              // slot * ldu + off_p, in node order (allocated when the bf16 gather path is first selected)
  int32_t* acount;            // [P x max_envs]: number of active nodes of (patch, slot)
};

struct StepIO {
  int32_t n_envs, input_mode;
  const etac_indenter* ind;
  const float* patch_pose;
  const float* pen_in;
  void* out;                  // fp32 or bf16 elements (out_bf16), environment e at element e * out_stride
  int64_t out_stride;
  int32_t out_bf16;
  float* pen_out;
  uint32_t* mask_out;
  float* analytic_out;
  uint8_t* contact_out;
  int32_t* nact_out;
};

#ifdef __CUDACC__
// ---- output element access (etac_step_args: d_out, out_env_stride, out_dtype)
// Streaming zero fill of nbytes (even, < 2^31) at a 2-byte aligned address by nthreads (>= 8) cooperating threads.
__device__ __forceinline__ void zero_fill_bytes(void* ptr, int nbytes, int tid, int nthreads) {
  char* p = static_cast<char*>(ptr);
  const int head = min((int)((16u - (uint32_t)((uintptr_t)p & 15u)) & 15u), nbytes);
  if (2 * tid < head) __stcs(reinterpret_cast<unsigned short*>(p + 2 * tid), (unsigned short)0);
  uint4* body = reinterpret_cast<uint4*>(p + head);
  const int nvec = (nbytes - head) >> 4;
  for (int v = tid; v < nvec; v += nthreads) __stcs(body + v, make_uint4(0u, 0u, 0u, 0u));
  const int tail0 = head + (nvec << 4);
  if (tail0 + 2 * tid < nbytes) __stcs(reinterpret_cast<unsigned short*>(p + tail0 + 2 * tid), (unsigned short)0);
}
// rows [g0, g0 + n_rows) of environment env of the displacement output := 0
__device__ __forceinline__ void zero_out_rows(const StepIO& io, int env, int g0, int n_rows, int tid, int nthreads) {
  const int sh = io.out_bf16 ? 1 : 2;
  char* p = static_cast<char*>(io.out) + (((int64_t)env * io.out_stride + 3 * g0) << sh);
  zero_fill_bytes(p, (n_rows * 3) << sh, tid, nthreads);
}
// U[env][g][0..2] := (x, y, z), streaming; kDtype: ETAC_OUT_F32 / ETAC_OUT_BF16, or -1 = io.out_bf16 decides
template <int kDtype = -1>
__device__ __forceinline__ void store_out3_at(const StepIO& io, int64_t o, float x, float y, float z) {
  if (kDtype == ETAC_OUT_BF16 || (kDtype < 0 && io.out_bf16)) {
    unsigned short* q = static_cast<unsigned short*>(io.out) + o;
    __stcs(q, __bfloat16_as_ushort(__float2bfloat16_rn(x)));
    __stcs(q + 1, __bfloat16_as_ushort(__float2bfloat16_rn(y)));
    __stcs(q + 2, __bfloat16_as_ushort(__float2bfloat16_rn(z)));
  } else {
    float* q = static_cast<float*>(io.out) + o;
    __stcs(q, x), __stcs(q + 1, y), __stcs(q + 2, z);
  }
}
template <int kDtype = -1>
__device__ __forceinline__ void store_out3(const StepIO& io, int env, int g, float x, float y, float z) {
  store_out3_at<kDtype>(io, (int64_t)env * io.out_stride + 3 * (int64_t)g, x, y, z);
}
#endif

// kernel launchers (each returns cudaGetLastError())
cudaError_t launch_build_k(const DevModel& m, float* k32, __nv_bfloat16* k16, cudaStream_t s);
cudaError_t launch_build_c1(const DevModel& m, const float* W1, const float* b1, float* c1t, cudaStream_t s);
cudaError_t launch_sdf(const DevModel& m, const StepIO& io, int s1_flags, int* launches, cudaStream_t s);
cudaError_t launch_gather_fp32(const DevModel& m, const StepIO& io, int n_sm, cudaStream_t s);
cudaError_t gather_fp32_configure();
cudaError_t launch_pointnet_fp32(const DevModel& m, const StepIO& io, int* launches, cudaStream_t s);
cudaError_t pointnet_fp32_configure();
void launch_pointnet_global_env(const DevModel& m, int n_envs, cudaStream_t s);
cudaError_t backward_pointnet_configure();
cudaError_t launch_backward_pointnet(const DevModel& m, const StepIO& io, const float* grad_out, float* grad_w, float* grad_delta,
                                     int n_sm, int* launches, cudaStream_t s);
// etac_backward, pose part (k_backward_pose.cu): dL/ddelta chained to the indenter poses ([E x max_ind x 6], zero on
// entry, may be NULL) and the patch poses ([E x P x 6], overwritten, may be NULL); rows are (dL/dt, dL/dtheta)
constexpr int kMaxPoseGradIndenters = 256;
cudaError_t launch_backward_pose(const DevModel& m, const StepIO& io, const float* g_delta, float* grad_ind, float* grad_patch,
                                 cudaStream_t s);
cudaError_t launch_mesh_sdf_grid(const float* tri, int n_tri, int nx, int ny, int nz, const float* origin, float h, float* values,
                                 cudaStream_t s);
cudaError_t launch_penalty_only(const DevModel& m, const StepIO& io, cudaStream_t s);
cudaError_t backward_configure();
cudaError_t launch_backward(const DevModel& m, const StepIO& io, const float* grad_out, float* grad_alpha, int n_alpha,
                            float* grad_w, float* grad_delta, int n_sm, cudaStream_t s);
cudaError_t launch_fused_bf16(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB, int n_sm, bool gather,
                              int* launches, cudaStream_t s);
cudaError_t fused_configure();
bool fused_uses_big_tile(const DevModel& m, int n_envs);
bool fused_fits(int n_patches);

}  // namespace etac

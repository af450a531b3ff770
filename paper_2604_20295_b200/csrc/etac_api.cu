// Host side of the C ABI declared in include/etac.h: validation, patch derivation, device
// staging, workspace, tensor maps, and the per-step launch sequence  S1 -> (S2+S3+S4).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <numeric>

#include "etac_internal.h"

using namespace etac;

struct etac_ctx {
  DevModel m{};
  std::vector<void*> allocs;
  size_t bytes = 0;
  int device = 0, n_sm = 0, precision = 0, path_opt = ETAC_PATH_AUTO, n_alpha = 1;
  int last_path = ETAC_PATH_AUTO, last_launches = 0;
  CUtensorMap tmA{}, tmB{};  // K rows [128 x 64]; U^ rows [48 x 64]: the 16-env tile, half of the 32-env tile
  bool have_tm = false;
  cudaStream_t last_stream = nullptr;
  std::string err;
  // writable aliases of the parameter-dependent device buffers (etac_update_params)
  std::vector<PatchInfo> hp;
  float* k32_w = nullptr;
  __nv_bfloat16* k16_w = nullptr;
  float *dW1_w = nullptr, *db1_w = nullptr;
};

static thread_local std::string g_create_err;

namespace {

struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    ok = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

etac_status fail(etac_ctx* c, etac_status st, const std::string& msg) {
  if (c) c->err = msg; else g_create_err = msg;
  return st;
}
std::string cuda_msg(const char* what, cudaError_t e) {
  return std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
}

uint16_t f2bf(float f) {  // round-to-nearest-even
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

template <class T>
cudaError_t dev_alloc(etac_ctx* c, T** p, size_t count, bool zero) {
  void* q = nullptr;
  const size_t bytes = std::max<size_t>(count * sizeof(T), 16);
  cudaError_t e = cudaMalloc(&q, bytes);
  if (e != cudaSuccess) return e;
  c->allocs.push_back(q);
  c->bytes += bytes;
  if (zero) e = cudaMemset(q, 0, bytes);
  *p = static_cast<T*>(q);
  return e;
}
template <class T>
cudaError_t dev_upload(etac_ctx* c, const T** p, const T* host, size_t count) {
  T* q = nullptr;
  cudaError_t e = dev_alloc(c, &q, count, false);
  if (e != cudaSuccess) return e;
  *p = q;
  return cudaMemcpy(q, host, count * sizeof(T), cudaMemcpyHostToDevice);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 2-D bf16 tensor [rows x cols], row pitch ld elements; box [box_rows x 64 cols], 128-byte swizzle.
bool make_tmap(CUtensorMap* tm, const void* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows,
               std::string* why) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || fn == nullptr || qres != cudaDriverEntryPointSuccess) {
    *why = "cuTensorMapEncodeTiled entry point not available";
    return false;
  }
  const cuuint64_t gdim[2] = {cols, rows};
  const cuuint64_t gstride[1] = {ld * 2};
  const cuuint32_t box[2] = {64, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base),
                                                   gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                   CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    *why = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return false;
  }
  return true;
}

int resolve_path(const etac_ctx* c) {
  if (c->path_opt == ETAC_PATH_AUTO) return c->precision == ETAC_PREC_BF16 ? ETAC_PATH_DENSE : ETAC_PATH_SPARSE;
  return c->path_opt;
}

// byte offset of element (n, k) in a K-major SWIZZLE_NONE UMMA operand with n_rows rows:
// 8x8 core matrices (128 B), core matrices of one k-octet contiguous over the row groups.
size_t wimg_off(int n, int k, int n_rows) {
  return (size_t)(k / 8) * (n_rows / 8) * 128 + (size_t)(n / 8) * 128 + (size_t)(n % 8) * 16 + (size_t)(k % 8) * 2;
}

etac_status step_impl(etac_ctx* ctx, cudaStream_t s, const etac_step_args* a, cudaEvent_t* ev) {
  if (!ctx) return ETAC_ERR_INVALID_ARG;
  if (!a || a->struct_size != sizeof(etac_step_args)) return fail(ctx, ETAC_ERR_INVALID_ARG, "bad etac_step_args");
  if (a->n_envs < 0) return fail(ctx, ETAC_ERR_INVALID_ARG, "n_envs < 0");
  if (a->n_envs > ctx->m.max_envs) return fail(ctx, ETAC_ERR_CAPACITY, "n_envs > max_envs");
  if (a->input_mode != ETAC_IN_INDENTERS && a->input_mode != ETAC_IN_PENETRATION)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "bad input_mode");
  if (!a->d_out) return fail(ctx, ETAC_ERR_INVALID_ARG, "d_out is required");
  if (a->out_dtype != ETAC_OUT_F32 && a->out_dtype != ETAC_OUT_BF16) return fail(ctx, ETAC_ERR_INVALID_ARG, "bad out_dtype");
  if (a->out_env_stride != 0 && a->out_env_stride < 3 * (int64_t)ctx->m.n_nodes)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "out_env_stride < 3 * n_nodes");
  if (a->reserved != 0) return fail(ctx, ETAC_ERR_INVALID_ARG, "reserved must be 0");
  if (reinterpret_cast<uintptr_t>(a->d_out) % (a->out_dtype == ETAC_OUT_BF16 ? 2 : 4))
    return fail(ctx, ETAC_ERR_INVALID_ARG, "d_out is not aligned to its element type");
  if (a->input_mode == ETAC_IN_INDENTERS && ctx->m.max_ind > 0 && !a->d_indenters)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "d_indenters is NULL");
  if (a->input_mode == ETAC_IN_PENETRATION && !a->d_penetration)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "d_penetration is NULL");
  const int path = resolve_path(ctx);
  if (path == ETAC_PATH_DENSE && ctx->precision != ETAC_PREC_BF16)
    return fail(ctx, ETAC_ERR_UNSUPPORTED, "ETAC_PATH_DENSE needs an ETAC_PREC_BF16 context");
  ctx->last_path = path;
  ctx->last_launches = 0;
  ctx->last_stream = s;
  if (a->n_envs == 0) return ETAC_OK;
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, ETAC_ERR_CUDA, "cudaSetDevice failed");

  StepIO io{};
  io.n_envs = a->n_envs, io.input_mode = a->input_mode;
  io.ind = a->d_indenters, io.patch_pose = a->d_patch_pose, io.pen_in = a->d_penetration;
  io.out = a->d_out, io.pen_out = a->d_penetration_out, io.mask_out = a->d_mask_out;
  io.out_stride = a->out_env_stride ? a->out_env_stride : 3 * (int64_t)ctx->m.n_nodes;
  io.out_bf16 = a->out_dtype == ETAC_OUT_BF16;
  io.analytic_out = a->d_analytic_out;
  io.contact_out = a->d_contact_out, io.nact_out = a->d_active_count_out;

  cudaError_t e;
  if (ev) cudaEventRecord(ev[0], s);
  if (io.mask_out) {
    const size_t words = (size_t)((ctx->m.n_nodes + 31) / 32) * a->n_envs;
    if ((e = cudaMemsetAsync(io.mask_out, 0, words * 4, s)) != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("memset mask", e));
  }
  if (io.nact_out && (e = cudaMemsetAsync(io.nact_out, 0, sizeof(int32_t) * a->n_envs, s)) != cudaSuccess)
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("memset active count", e));
  if ((e = cudaMemsetAsync(ctx->m.count, 0, sizeof(int32_t) * (ctx->m.n_patches + 3), s)) != cudaSuccess)
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("memset count", e));
  // bf16 context: tensor-core MLP either way; DENSE = tcgen05 contraction K.U^, SPARSE = gather over the
  // active-node lists.  fp32 context: fp32 SIMT gather kernel (which needs S1 to zero-fill).
  const bool bf16 = ctx->precision == ETAC_PREC_BF16;
  const bool gather16 = bf16 && path == ETAC_PATH_SPARSE;
  const int abl = ctx->m.ablation;
  int s1_flags = abl == ETAC_ABLATE_NO_PROPAGATION ? 0 : !bf16 ? kS1FillOut : (gather16 ? kS1WriteAlist : kS1WriteUhat);
  if ((s1_flags & kS1WriteUhat) && ctx->m.khist && fused_uses_big_tile(ctx->m, a->n_envs)) s1_flags |= kS1Bucket;
  if (gather16 && !ctx->m.alist) return fail(ctx, ETAC_ERR_INVALID_ARG, "select ETAC_PATH_SPARSE with etac_set_option first");
  int n_s1 = 1;
  if ((e = launch_sdf(ctx->m, io, s1_flags, &n_s1, s)) != cudaSuccess)
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("sdf_penetration_kernel", e));
  ctx->last_launches += n_s1;
  if (ev) cudaEventRecord(ev[1], s);
  if (abl == ETAC_ABLATE_NO_PROPAGATION) {
    if ((e = launch_penalty_only(ctx->m, io, s)) != cudaSuccess)
      return fail(ctx, ETAC_ERR_CUDA, cuda_msg("penalty_only_kernel", e));
  } else if (bf16) {
    int n_launch = 1;
    if (abl == ETAC_ABLATE_LINEAR_ONLY) {  // "Linear Decay Only": the kernels compiled without Phi
      DevModel lin = ctx->m;
      lin.resid = ETAC_RESID_NONE;
      e = launch_fused_bf16(lin, io, ctx->tmA, ctx->tmB, ctx->n_sm, gather16, &n_launch, s);
    } else {
      e = launch_fused_bf16(ctx->m, io, ctx->tmA, ctx->tmB, ctx->n_sm, gather16, &n_launch, s);
    }
    if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("fused_mlp_kernel", e));
    ctx->last_launches += n_launch - 1;
  } else {
    if (abl == ETAC_ABLATE_LINEAR_ONLY) {
      DevModel lin = ctx->m;
      lin.resid = ETAC_RESID_NONE;
      e = launch_gather_fp32(lin, io, ctx->n_sm, s);
    } else if (ctx->m.resid == ETAC_RESID_POINTNET) {
      int n_launch = 1;
      e = launch_pointnet_fp32(ctx->m, io, &n_launch, s);
      ctx->last_launches += n_launch - 1;
    } else {
      e = launch_gather_fp32(ctx->m, io, ctx->n_sm, s);
    }
    if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("gather_fp32_kernel", e));
  }
  ++ctx->last_launches;
  if (ev) cudaEventRecord(ev[2], s);
  return ETAC_OK;
}

// Host staging of the per-node MLP: the fp32 blob of the SIMT kernels (W1u | W2 | b2 | W3 | b3) and the
// bf16 shared-memory image of the tensor-core path.  The epilogue evaluates silu(x) = h + h*tanh(h) with
// h = x/2, so the 0.5 is folded into layers 1 and 2 (exact); the output layer runs on the FMA pipe in
// fp32 (DevModel::wout).
struct PerNodeStage {
  std::vector<float> wf;
  std::vector<uint8_t> img;
  float wout[196];
};
void stage_pernode(const float* W1, const float* b1, const float* W2, const float* b2, const float* W3, const float* b3,
                   PerNodeStage* st) {
  st->wf.assign(kWf32W2t + 64 * 64, 0.f);  // W1u | W2 | b2 | W3 | b3 | pad | W2^T (for gather_fp32_kernel)
  for (int k2 = 0; k2 < 64; ++k2)
    for (int k = 0; k < 64; ++k) st->wf[kWf32W2t + k * 64 + k2] = W2[k2 * 64 + k];
  float* q = st->wf.data();
  for (int k = 0; k < 64; ++k)
    for (int cc = 0; cc < 3; ++cc) *q++ = W1[k * 9 + cc];
  memcpy(q, W2, 4096 * 4), q += 4096;
  memcpy(q, b2, 64 * 4), q += 64;
  memcpy(q, W3, 192 * 4), q += 192;
  memcpy(q, b3, 3 * 4);
  st->img.assign(kWImgBytes, 0);
  auto put = [&](size_t base, int n, int k, int rows, float v) {
    const uint16_t b = f2bf(v);
    memcpy(&st->img[base + wimg_off(n, k, rows)], &b, 2);
  };
  for (int n = 0; n < 64; ++n) {
    for (int k = 0; k < 9; ++k) put(0, n, k, 64, 0.5f * W1[n * 9 + k]);
    put(0, n, 9, 64, 0.5f * b1[n]);
    for (int k = 0; k < 64; ++k) put(kW1ImgBytes, n, k, 64, 0.5f * W2[n * 64 + k]);
    put(kW1ImgBytes, n, 64, 64, 0.5f * b2[n]);
  }
  memcpy(st->wout, W3, 192 * 4);
  memcpy(st->wout + 192, b3, 3 * 4);
  st->wout[195] = 0.0f;
}

// The PointNet form of Phi staged for the device: the bf16 shared-memory image of the tensor-core
// passes, the global MLP (fp32, both matrices transposed), the fp32 copies of the node layers, the output layer.
struct PointNetStage {
  std::vector<uint8_t> img;
  std::vector<float> pf, w32;
  float wout[196];
};
void stage_pointnet(const float* E1, const float* e1, const float* E2, const float* e2, const float* G1, const float* g1,
                    const float* D1, const float* d1, const float* D2, const float* d2, PointNetStage* st) {
  // bf16 image; the 0.5 of silu(x) = h + h*tanh(h), h = x/2, is folded into every layer that feeds a SiLU.
  // Layer-1 operand columns are [u^(3), p(3), n(3), 1]; E1's inputs are [p, n, u^].
  st->img.assign(kPnImgBytes, 0);
  auto put = [&](size_t base, int n, int k, int rows, float v) {
    const uint16_t b = f2bf(v);
    memcpy(&st->img[base + wimg_off(n, k, rows)], &b, 2);
  };
  const size_t o1 = kW1ImgBytes, o2 = o1 + kW2ImgBytes;
  for (int n = 0; n < 64; ++n) {
    for (int k = 0; k < 3; ++k) {
      put(0, n, k, 64, 0.5f * E1[n * 9 + 6 + k]);      // u^
      put(0, n, 3 + k, 64, 0.5f * E1[n * 9 + k]);      // p
      put(0, n, 6 + k, 64, 0.5f * E1[n * 9 + 3 + k]);  // n
    }
    put(0, n, 9, 64, 0.5f * e1[n]);
    for (int k = 0; k < 64; ++k) put(o1, n, k, 64, 0.5f * E2[n * 64 + k]);
    put(o1, n, 64, 64, 0.5f * e2[n]);
    for (int k = 0; k < 64; ++k) put(o2, n, k, 64, 0.5f * D1[n * 128 + k]);  // bias column stays 0: c_(e,p) is added in the epilogue
  }
  memcpy(st->wout, D2, 192 * 4);
  memcpy(st->wout + 192, d2, 3 * 4);
  st->wout[195] = 0.0f;
  st->pf.assign(4096 + 64 + 4096 + 64, 0.f);
  for (int n = 0; n < 64; ++n)  // both 64 x 64 matrices transposed to [in][out] (coalesced over the outputs)
    for (int j = 0; j < 64; ++j) st->pf[j * 64 + n] = G1[n * 64 + j], st->pf[4160 + j * 64 + n] = D1[n * 128 + 64 + j];
  memcpy(st->pf.data() + 4096, g1, 64 * 4);
  memcpy(st->pf.data() + 4160 + 4096, d1, 64 * 4);
  st->w32.clear();  // fp32 SIMT forward (k_pointnet_fp32.cu) and backward (k_backward_pointnet.cu)
  st->w32.insert(st->w32.end(), E1, E1 + 576), st->w32.insert(st->w32.end(), e1, e1 + 64);
  st->w32.insert(st->w32.end(), E2, E2 + 4096), st->w32.insert(st->w32.end(), e2, e2 + 64);
  for (int n = 0; n < 64; ++n) st->w32.insert(st->w32.end(), D1 + n * 128, D1 + n * 128 + 64);
  st->w32.insert(st->w32.end(), D2, D2 + 192), st->w32.insert(st->w32.end(), d2, d2 + 3);
}

}  // namespace

extern "C" {

int32_t etac_abi_version(void) { return ETAC_ABI_VERSION; }

const char* etac_last_error(const etac_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

etac_status etac_patches_from_adjacency(int32_t n, const int32_t* rowptr, const int32_t* col, int32_t* off,
                                        int32_t cap, int32_t* n_patches) {
  if (n < 1 || !rowptr || !off || !n_patches || cap < 2) return ETAC_ERR_INVALID_ARG;
  if (rowptr[0] != 0) return ETAC_ERR_INVALID_ARG;
  for (int i = 0; i < n; ++i)
    if (rowptr[i + 1] < rowptr[i]) return ETAC_ERR_INVALID_ARG;
  if (rowptr[n] > 0 && !col) return ETAC_ERR_INVALID_ARG;
  std::vector<int32_t> parent(n);
  std::iota(parent.begin(), parent.end(), 0);
  auto find = [&](int x) {
    while (parent[x] != x) x = parent[x] = parent[parent[x]];
    return x;
  };
  for (int i = 0; i < n; ++i)
    for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
      const int j = col[k];
      if (j < 0 || j >= n) return ETAC_ERR_INVALID_ARG;
      int a = find(i), b = find(j);
      if (a != b) parent[std::max(a, b)] = std::min(a, b);  // representative = smallest index
    }
  int np = 0;
  int cur = -1;
  for (int i = 0; i < n; ++i) {
    const int r = find(i);
    if (r != cur) {
      if (r != i) return ETAC_ERR_UNSUPPORTED;  // component re-entered: not a contiguous range
      if (np + 1 >= cap) return ETAC_ERR_CAPACITY;
      off[np++] = i;
      cur = r;
    }
  }
  off[np] = n;
  *n_patches = np;
  return ETAC_OK;
}

etac_status etac_create(const etac_model_desc* d, etac_ctx** out) {
  if (!out) return fail(nullptr, ETAC_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!d) return fail(nullptr, ETAC_ERR_INVALID_ARG, "desc is NULL");
  if (d->struct_size != sizeof(etac_model_desc)) return fail(nullptr, ETAC_ERR_INVALID_ARG, "struct_size mismatch (ABI)");
  if (d->n_nodes < 1 || !d->node_pos || !d->node_normal) return fail(nullptr, ETAC_ERR_INVALID_ARG, "mesh missing");
  if (d->kernel_type != ETAC_KERNEL_EXP_L2) return fail(nullptr, ETAC_ERR_INVALID_ARG, "unknown kernel_type");
  if (d->max_envs < 1 || d->max_indenters < 0) return fail(nullptr, ETAC_ERR_INVALID_ARG, "bad max_envs / max_indenters");
  if (d->precision != ETAC_PREC_FP32 && d->precision != ETAC_PREC_BF16) return fail(nullptr, ETAC_ERR_INVALID_ARG, "bad precision");
  if (d->active_mode != ETAC_ACTIVE_PASSTHROUGH && d->active_mode != ETAC_ACTIVE_PROPAGATE)
    return fail(nullptr, ETAC_ERR_INVALID_ARG, "bad active_mode");
  if (d->resid_arch != ETAC_RESID_NONE && d->resid_arch != ETAC_RESID_PERNODE_MLP && d->resid_arch != ETAC_RESID_POINTNET)
    return fail(nullptr, ETAC_ERR_INVALID_ARG, "bad resid_arch");
  if (d->resid_arch == ETAC_RESID_POINTNET) {
    if (d->resid_hidden != kHidden) return fail(nullptr, ETAC_ERR_UNSUPPORTED, "only resid_hidden == 64 is built");
    if (!d->E1 || !d->e1 || !d->E2 || !d->e2 || !d->G1 || !d->g1 || !d->D1 || !d->d1 || !d->D2 || !d->d2)
      return fail(nullptr, ETAC_ERR_INVALID_ARG, "PointNet weights missing");
  }
  if (d->resid_arch == ETAC_RESID_PERNODE_MLP) {
    if (d->resid_hidden != kHidden) return fail(nullptr, ETAC_ERR_UNSUPPORTED, "only resid_hidden == 64 is built");
    if (!d->W1 || !d->b1 || !d->W2 || !d->b2 || !d->W3 || !d->b3) return fail(nullptr, ETAC_ERR_INVALID_ARG, "MLP weights missing");
  }
  const int N = d->n_nodes;
  // ---- patches
  std::vector<int32_t> off;
  if (d->patch_offset) {
    if (d->n_patches < 1) return fail(nullptr, ETAC_ERR_INVALID_ARG, "n_patches < 1");
    off.assign(d->patch_offset, d->patch_offset + d->n_patches + 1);
    if (off.front() != 0 || off.back() != N) return fail(nullptr, ETAC_ERR_INVALID_ARG, "patch_offset must span [0, N]");
    for (size_t p = 0; p + 1 < off.size(); ++p)
      if (off[p + 1] <= off[p]) return fail(nullptr, ETAC_ERR_INVALID_ARG, "patch_offset must be strictly increasing");
    if (d->adj_rowptr) {  // validate: no edge may cross a patch boundary
      std::vector<int32_t> pid(N);
      for (size_t p = 0; p + 1 < off.size(); ++p) std::fill(pid.begin() + off[p], pid.begin() + off[p + 1], (int32_t)p);
      for (int i = 0; i < N; ++i)
        for (int k = d->adj_rowptr[i]; k < d->adj_rowptr[i + 1]; ++k) {
          const int j = d->adj_col ? d->adj_col[k] : -1;
          if (j < 0 || j >= N) return fail(nullptr, ETAC_ERR_INVALID_ARG, "adjacency index out of range");
          if (pid[j] != pid[i]) return fail(nullptr, ETAC_ERR_INVALID_ARG, "adjacency edge crosses a patch boundary");
        }
    }
  } else if (d->adj_rowptr) {
    off.resize((size_t)N + 1);
    int32_t np = 0;
    etac_status st = etac_patches_from_adjacency(N, d->adj_rowptr, d->adj_col, off.data(), N + 1, &np);
    if (st != ETAC_OK) return fail(nullptr, st, "patches could not be derived from the adjacency");
    off.resize((size_t)np + 1);
  } else {
    off = {0, N};
  }
  const int P = (int)off.size() - 1;
  if (P > kMaxPatches) return fail(nullptr, ETAC_ERR_UNSUPPORTED, "more than 1024 patches");
  if (d->n_alpha != 1 && d->n_alpha != P) return fail(nullptr, ETAC_ERR_INVALID_ARG, "n_alpha must be 1 or P");
  if (!d->alpha) return fail(nullptr, ETAC_ERR_INVALID_ARG, "alpha is NULL");
  for (int k = 0; k < d->n_alpha; ++k)
    if (!(d->alpha[k] > 0.0f) || !isfinite(d->alpha[k])) return fail(nullptr, ETAC_ERR_INVALID_ARG, "alpha must be > 0");

  // ---- device
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(nullptr, ETAC_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
  }
  if (d->device < 0 || d->device >= ndev) return fail(nullptr, ETAC_ERR_INVALID_ARG, "bad device ordinal");
  cudaDeviceProp prop;
  if ((e = cudaGetDeviceProperties(&prop, d->device)) != cudaSuccess) return fail(nullptr, ETAC_ERR_CUDA, cuda_msg("cudaGetDeviceProperties", e));
  if (prop.major != 10) return fail(nullptr, ETAC_ERR_UNSUPPORTED, "needs a compute-capability 10.x (Blackwell, sm_100a) device");
  DeviceGuard guard(d->device);
  if (!guard.ok) return fail(nullptr, ETAC_ERR_CUDA, "cudaSetDevice failed");

  etac_ctx* c = new (std::nothrow) etac_ctx();
  if (!c) return fail(nullptr, ETAC_ERR_ALLOC, "host allocation failed");
  c->device = d->device, c->n_sm = prop.multiProcessorCount, c->precision = d->precision;
  DevModel& m = c->m;
  m.n_nodes = N, m.n_patches = P, m.max_envs = d->max_envs, m.max_ind = d->max_indenters;
  m.resid = d->resid_arch, m.active_mode = d->active_mode;
  m.group_bytes = 40 << 20;

  auto bail = [&](etac_status st, const std::string& msg) {
    g_create_err = msg;
    for (void* p : c->allocs) cudaFree(p);
    delete c;
    return st;
  };
#define CK(call, what)                                                                              \
  do {                                                                                              \
    cudaError_t e_ = (call);                                                                        \
    if (e_ != cudaSuccess)                                                                          \
      return bail(e_ == cudaErrorMemoryAllocation ? ETAC_ERR_ALLOC : ETAC_ERR_CUDA, cuda_msg(what, e_)); \
  } while (0)

  // mesh as float4 (coalesced 16-byte node loads)
  std::vector<float4> pos4(N), nrm4(N);
  for (int i = 0; i < N; ++i) {
    pos4[i] = make_float4(d->node_pos[3 * i], d->node_pos[3 * i + 1], d->node_pos[3 * i + 2], 0.f);
    nrm4[i] = make_float4(d->node_normal[3 * i], d->node_normal[3 * i + 1], d->node_normal[3 * i + 2], 0.f);
  }
  CK(dev_upload(c, &m.pos4, pos4.data(), N), "upload pos");
  CK(dev_upload(c, &m.nrm4, nrm4.data(), N), "upload normal");
  {
    std::vector<uint4> a1c(N);
    for (int i = 0; i < N; ++i) {
      auto pk = [](float lo, float hi) { return (uint32_t)f2bf(lo) | ((uint32_t)f2bf(hi) << 16); };
      a1c[i] = make_uint4(pk(pos4[i].x, 0.f), pk(pos4[i].y, pos4[i].z), pk(nrm4[i].x, nrm4[i].y), pk(nrm4[i].z, 1.0f));
    }
    CK(dev_upload(c, &m.a1c, a1c.data(), N), "upload layer-1 constants");
  }

  std::vector<PatchInfo> hp(P);
  std::vector<ChunkInfo> chunks;
  int64_t k32_total = 0;
  int max_np = 0, ucols = 0;
  for (int p = 0; p < P; ++p) {
    PatchInfo& pi = hp[p];
    pi.off = off[p], pi.n = off[p + 1] - off[p];
    pi.uoff = ucols;
    ucols += (pi.n + 7) / 8 * 8;
    pi.k32_off = k32_total;
    k32_total += (int64_t)pi.n * pi.n;
    pi.alpha = d->alpha[d->n_alpha == 1 ? 0 : p];
    double c0 = 0, c1 = 0, c2 = 0;
    for (int i = pi.off; i < pi.off + pi.n; ++i) c0 += pos4[i].x, c1 += pos4[i].y, c2 += pos4[i].z;
    c0 /= pi.n, c1 /= pi.n, c2 /= pi.n;
    pi.bc[0] = (float)c0, pi.bc[1] = (float)c1, pi.bc[2] = (float)c2;
    double r2 = 0;
    for (int i = pi.off; i < pi.off + pi.n; ++i) {
      const double dx = pos4[i].x - pi.bc[0], dy = pos4[i].y - pi.bc[1], dz = pos4[i].z - pi.bc[2];
      r2 = std::max(r2, dx * dx + dy * dy + dz * dz);
    }
    pi.brad = (float)(sqrt(r2) * (1.0 + 1e-5) + 1e-6);
    max_np = std::max(max_np, pi.n);
    for (int n0 = 0; n0 < pi.n; n0 += kGatherChunk)
      chunks.push_back(ChunkInfo{p, pi.off + n0, std::min(kGatherChunk, pi.n - n0)});
  }
  m.n_chunks = (int)chunks.size();
  m.max_patch_nodes = max_np;
  m.kw = (max_np + 63) / 64 * 64;
  m.ldu = (ucols + 63) / 64 * 64;
  CK(dev_upload(c, &m.patch, hp.data(), P), "upload patches");
  CK(dev_upload(c, &m.chunk, chunks.data(), chunks.size()), "upload chunks");

  float* k32 = nullptr;
  __nv_bfloat16* k16 = nullptr;
  CK(dev_alloc(c, &k32, (size_t)k32_total, false), "alloc K fp32");
  CK(dev_alloc(c, &k16, (size_t)N * m.kw, true), "alloc K bf16");
  m.k32 = k32, m.k16 = k16;
  c->k32_w = k32, c->k16_w = k16, c->hp = hp;
  CK(launch_build_k(m, k32, k16, 0), "build_k_kernel");

  if (d->resid_arch == ETAC_RESID_PERNODE_MLP) {
    PerNodeStage st;
    stage_pernode(d->W1, d->b1, d->W2, d->b2, d->W3, d->b3, &st);
    CK(dev_upload(c, &m.wf32, st.wf.data(), st.wf.size()), "upload weights");
    const float *dW1 = nullptr, *db1 = nullptr;
    CK(dev_upload(c, &dW1, d->W1, 64 * 9), "upload W1");
    CK(dev_upload(c, &db1, d->b1, 64), "upload b1");
    c->dW1_w = const_cast<float*>(dW1), c->db1_w = const_cast<float*>(db1);
    float* c1t = nullptr;
    CK(dev_alloc(c, &c1t, (size_t)64 * N, false), "alloc c1");
    m.c1t = c1t;
    CK(launch_build_c1(m, dW1, db1, c1t, 0), "build_c1_kernel");
    memcpy(m.wout, st.wout, sizeof(m.wout));
    CK(dev_upload(c, &m.wimg, st.img.data(), st.img.size()), "upload weight image");
  }

  if (d->resid_arch == ETAC_RESID_POINTNET) {
    PointNetStage st;
    stage_pointnet(d->E1, d->e1, d->E2, d->e2, d->G1, d->g1, d->D1, d->d1, d->D2, d->d2, &st);
    memcpy(m.wout, st.wout, sizeof(m.wout));
    CK(dev_upload(c, &m.wimg_pn, st.img.data(), st.img.size()), "upload PointNet weight image");
    CK(dev_upload(c, &m.pn_f32, st.pf.data(), st.pf.size()), "upload PointNet global MLP");
    CK(dev_upload(c, &m.pn_w32, st.w32.data(), st.w32.size()), "upload PointNet fp32 weights");
    CK(pointnet_fp32_configure(), "cudaFuncSetAttribute(pn_decode_fp32_kernel)");
    CK(backward_pointnet_configure(), "cudaFuncSetAttribute(pn_bwd_node_kernel)");
    CK(dev_alloc(c, &m.pn_gkey, (size_t)64 * P * d->max_envs, true), "alloc PointNet arg-max keys");
    CK(dev_alloc(c, &m.pn_ssum, (size_t)64 * P * d->max_envs, true), "alloc PointNet backward sums");
    CK(dev_alloc(c, &m.pn_ggmax, (size_t)64 * P * d->max_envs, true), "alloc PointNet backward dL/dgmax");
    CK(dev_alloc(c, &m.gmax, (size_t)64 * P * d->max_envs, true), "alloc gmax");
    CK(dev_alloc(c, &m.cvec, (size_t)64 * P * d->max_envs, true), "alloc cvec");
  }

  // ---- per-step workspace
  const size_t urows = (size_t)((d->max_envs + kMaxTE - 1) / kMaxTE) * kMaxTE * 3;
  CK(dev_alloc(c, &m.delta, (size_t)d->max_envs * N, true), "alloc delta");
  CK(dev_alloc(c, &m.count, (size_t)P + 3, true), "alloc count");
  m.ntask = m.count + P;
  m.wq = m.count + P + 1;
  if (d->max_indenters == 1 && P >= 4) {  // S1 as cull + evaluate kernels: 128-byte task records
    void* tasks = nullptr;
    CK(dev_alloc(c, reinterpret_cast<uint8_t**>(&tasks), (size_t)128 * P * d->max_envs, false), "alloc S1 tasks");
    m.tasks = static_cast<PairTask*>(tasks);
  }
  CK(dev_alloc(c, &m.envlist, (size_t)P * d->max_envs, true), "alloc envlist");
  CK(dev_alloc(c, &m.flags, (size_t)P * d->max_envs, true), "alloc flags");
  if (d->precision == ETAC_PREC_BF16) {
    if (!fused_fits(P)) return bail(ETAC_ERR_UNSUPPORTED, "too many patches for the shared-memory tables of the tensor-core path");
    CK(dev_alloc(c, &m.uhat_t, urows * m.ldu, true), "alloc uhat");
    CK(dev_alloc(c, &m.kbmap, (size_t)P * ((size_t)(d->max_envs + kMaxTE - 1) / kMaxTE * kMaxTE) * kKbWords, true), "alloc k-block bitmaps");
    m.kbtile_stride = (d->max_envs + kMaxTE - 1) / kMaxTE;
    CK(dev_alloc(c, &m.kbtile, (size_t)P * m.kbtile_stride * kKbWords, true), "alloc tile k-block masks");
    if (P <= 64 && max_np >= 1024) {  // bucketing of the environments by contact position (large patches)
      CK(dev_alloc(c, &m.khist, (size_t)P * 512, true), "alloc bucket histogram");
      m.kcursor = m.khist + (size_t)P * 256;
      CK(dev_alloc(c, &m.keybuf, (size_t)P * d->max_envs, true), "alloc bucket keys");
    }
    std::string why;
    if (!make_tmap(&c->tmA, m.k16, (uint64_t)N, (uint64_t)m.kw, (uint64_t)m.kw, 128, &why) ||
        !make_tmap(&c->tmB, m.uhat_t, (uint64_t)urows, (uint64_t)m.ldu, (uint64_t)m.ldu, 48, &why))
      return bail(ETAC_ERR_CUDA, why);
    c->have_tm = true;
    CK(fused_configure(), "cudaFuncSetAttribute(fused_mlp_kernel)");
  }
  c->n_alpha = d->n_alpha;
  CK(backward_configure(), "cudaFuncSetAttribute(backward_kernel)");
  CK(gather_fp32_configure(), "cudaFuncSetAttribute(gather_fp32_kernel)");
  CK(cudaDeviceSynchronize(), "create-time kernels");
#undef CK
  *out = c;
  return ETAC_OK;
}

etac_status etac_destroy(etac_ctx* ctx) {
  if (!ctx) return ETAC_OK;
  etac_status st = ETAC_OK;
  {
    DeviceGuard guard(ctx->device);
    if (cudaDeviceSynchronize() != cudaSuccess) st = ETAC_ERR_CUDA;
    for (void* p : ctx->allocs) cudaFree(p);
  }
  delete ctx;
  return st;
}

etac_status etac_step(etac_ctx* ctx, void* cuda_stream, const etac_step_args* args) {
  return step_impl(ctx, static_cast<cudaStream_t>(cuda_stream), args, nullptr);
}

etac_status etac_set_option(etac_ctx* ctx, int32_t key, int64_t value) {
  if (!ctx) return ETAC_ERR_INVALID_ARG;
  if (key == ETAC_OPT_ABLATION) {
    if (value < ETAC_ABLATE_FULL || value > ETAC_ABLATE_NO_PROPAGATION) return fail(ctx, ETAC_ERR_INVALID_ARG, "bad ETAC_OPT_ABLATION value");
    ctx->m.residual_only = value == ETAC_ABLATE_RESIDUAL_ONLY;
    ctx->m.ablation = (int32_t)value;
    return ETAC_OK;
  }
  if (key == ETAC_OPT_L2_GROUP_BYTES) {
    if (value < 1 || value > (int64_t)1 << 30) return fail(ctx, ETAC_ERR_INVALID_ARG, "bad ETAC_OPT_L2_GROUP_BYTES value");
    ctx->m.group_bytes = (int32_t)value;
    return ETAC_OK;
  }
  if (key != ETAC_OPT_PATH) return fail(ctx, ETAC_ERR_INVALID_ARG, "unknown option");
  if (value != ETAC_PATH_AUTO && value != ETAC_PATH_DENSE && value != ETAC_PATH_SPARSE)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "bad ETAC_OPT_PATH value");
  if (value == ETAC_PATH_DENSE && ctx->precision != ETAC_PREC_BF16)
    return fail(ctx, ETAC_ERR_UNSUPPORTED, "ETAC_PATH_DENSE needs an ETAC_PREC_BF16 context");
  if (value == ETAC_PATH_SPARSE && ctx->precision == ETAC_PREC_BF16 && !ctx->m.alist) {
    // workspace of the bf16 gather path: active-node lists (allocated here, never inside etac_step)
    DeviceGuard guard(ctx->device);
    ActiveEntry* al = nullptr;
    int32_t* ac = nullptr;
    const size_t rows = (size_t)((ctx->m.max_envs + kMaxTE - 1) / kMaxTE) * kMaxTE;
    cudaError_t e = dev_alloc(ctx, &al, rows * ctx->m.ldu, false);
    if (e == cudaSuccess) e = dev_alloc(ctx, &ac, (size_t)ctx->m.n_patches * ctx->m.max_envs, true);
    if (e != cudaSuccess) return fail(ctx, e == cudaErrorMemoryAllocation ? ETAC_ERR_ALLOC : ETAC_ERR_CUDA, cuda_msg("alloc active lists", e));
    ctx->m.alist = al, ctx->m.acount = ac;
  }
  ctx->path_opt = (int)value;
  return ETAC_OK;
}

etac_status etac_set_sdf_grid(etac_ctx* ctx, int32_t grid_id, int32_t nx, int32_t ny, int32_t nz, const float* origin,
                              float spacing, const float* values) {
  if (!ctx) return ETAC_ERR_INVALID_ARG;
  if (grid_id < 0 || grid_id >= kMaxGrids) return fail(ctx, ETAC_ERR_INVALID_ARG, "grid_id out of range");
  if (nx < 2 || ny < 2 || nz < 2 || !origin || !values || !(spacing > 0.0f) || !isfinite(spacing))
    return fail(ctx, ETAC_ERR_INVALID_ARG, "bad SDF grid");
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, ETAC_ERR_CUDA, "cudaSetDevice failed");
  GridDesc& g = ctx->m.grid[grid_id];
  cudaError_t e = cudaSuccess;
  if (g.v) {  // replacing: nothing in flight may still read the old samples
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("synchronize", e));
    cudaFree(const_cast<float*>(g.v));
    ctx->allocs.erase(std::remove(ctx->allocs.begin(), ctx->allocs.end(), (void*)g.v), ctx->allocs.end());
    g.v = nullptr;
  }
  float* dv = nullptr;
  const size_t count = (size_t)nx * ny * nz;
  if ((e = dev_alloc(ctx, &dv, count, false)) != cudaSuccess)
    return fail(ctx, e == cudaErrorMemoryAllocation ? ETAC_ERR_ALLOC : ETAC_ERR_CUDA, cuda_msg("alloc SDF grid", e));
  if ((e = cudaMemcpy(dv, values, count * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("upload SDF grid", e));
  g.v = dv, g.nx = nx, g.ny = ny, g.nz = nz;
  g.o[0] = origin[0], g.o[1] = origin[1], g.o[2] = origin[2];
  g.h = spacing, g.inv_h = 1.0f / spacing;
  return ETAC_OK;
}

etac_status etac_mesh_to_sdf_grid(int32_t device, int32_t n_vertices, const float* vertices, int32_t n_triangles,
                                  const int32_t* triangles, int32_t nx, int32_t ny, int32_t nz, const float* origin, float spacing,
                                  float* values_out) {
  if (n_vertices < 4 || n_triangles < 4 || !vertices || !triangles || !origin || !values_out)
    return fail(nullptr, ETAC_ERR_INVALID_ARG, "etac_mesh_to_sdf_grid: NULL pointer or fewer than 4 vertices / triangles");
  if (nx < 2 || ny < 2 || nz < 2 || !(spacing > 0.0f) || !isfinite(spacing))
    return fail(nullptr, ETAC_ERR_INVALID_ARG, "etac_mesh_to_sdf_grid: bad grid");
  std::vector<float> tri((size_t)n_triangles * 9);
  for (int t = 0; t < n_triangles; ++t)
    for (int k = 0; k < 3; ++k) {
      const int v = triangles[3 * t + k];
      if (v < 0 || v >= n_vertices) return fail(nullptr, ETAC_ERR_INVALID_ARG, "etac_mesh_to_sdf_grid: vertex index out of range");
      for (int a = 0; a < 3; ++a) {
        if (!isfinite(vertices[3 * v + a])) return fail(nullptr, ETAC_ERR_INVALID_ARG, "etac_mesh_to_sdf_grid: vertex is not finite");
        tri[(size_t)t * 9 + 3 * k + a] = vertices[3 * v + a];
      }
    }
  DeviceGuard guard(device);
  if (!guard.ok) return fail(nullptr, ETAC_ERR_CUDA, "cudaSetDevice failed");
  const size_t count = (size_t)nx * ny * nz;
  float *d_tri = nullptr, *d_val = nullptr;
  cudaError_t e = cudaMalloc(&d_tri, tri.size() * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&d_val, count * sizeof(float));
  if (e == cudaSuccess) e = cudaMemcpy(d_tri, tri.data(), tri.size() * sizeof(float), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = launch_mesh_sdf_grid(d_tri, n_triangles, nx, ny, nz, origin, spacing, d_val, 0);
  if (e == cudaSuccess) e = cudaMemcpy(values_out, d_val, count * sizeof(float), cudaMemcpyDeviceToHost);
  cudaFree(d_tri), cudaFree(d_val);
  if (e != cudaSuccess)
    return fail(nullptr, e == cudaErrorMemoryAllocation ? ETAC_ERR_ALLOC : ETAC_ERR_CUDA, cuda_msg("etac_mesh_to_sdf_grid", e));
  return ETAC_OK;
}

etac_status etac_get_info(const etac_ctx* ctx, int32_t key, int64_t* value) {
  if (!ctx || !value) return ETAC_ERR_INVALID_ARG;
  switch (key) {
    case ETAC_INFO_N_NODES: *value = ctx->m.n_nodes; return ETAC_OK;
    case ETAC_INFO_N_PATCHES: *value = ctx->m.n_patches; return ETAC_OK;
    case ETAC_INFO_MAX_ENVS: *value = ctx->m.max_envs; return ETAC_OK;
    case ETAC_INFO_DEVICE_BYTES: *value = (int64_t)ctx->bytes; return ETAC_OK;
    case ETAC_INFO_LAST_PATH: *value = ctx->last_path; return ETAC_OK;
    case ETAC_INFO_LAST_LAUNCHES: *value = ctx->last_launches; return ETAC_OK;
    case ETAC_INFO_SM_COUNT: *value = ctx->n_sm; return ETAC_OK;
    case ETAC_INFO_LAST_CONTACT_PAIRS: {
      DeviceGuard guard(ctx->device);
      std::vector<int32_t> cnt(ctx->m.n_patches);
      if (cudaStreamSynchronize(ctx->last_stream) != cudaSuccess) return ETAC_ERR_CUDA;
      if (cudaMemcpy(cnt.data(), ctx->m.count, cnt.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return ETAC_ERR_CUDA;
      *value = std::accumulate(cnt.begin(), cnt.end(), (int64_t)0);
      return ETAC_OK;
    }
    default: return ETAC_ERR_INVALID_ARG;
  }
}

etac_status etac_update_params(etac_ctx* ctx, const etac_params* p) {
  if (!ctx) return ETAC_ERR_INVALID_ARG;
  // (a caller built against the header before the PointNet arrays were added passes the shorter struct)
  if (!p || (p->struct_size != sizeof(etac_params) && p->struct_size != offsetof(etac_params, E1)))
    return fail(ctx, ETAC_ERR_INVALID_ARG, "bad etac_params");
  const float* w[6] = {p->W1, p->b1, p->W2, p->b2, p->W3, p->b3};
  int n_w = 0, n_pn = 0;
  for (const float* q : w) n_w += q != nullptr;
  if (n_w != 0 && n_w != 6) return fail(ctx, ETAC_ERR_INVALID_ARG, "give all six weight arrays or none");
  if (n_w && ctx->m.resid != ETAC_RESID_PERNODE_MLP)
    return fail(ctx, ETAC_ERR_UNSUPPORTED, "W1 .. b3 can be replaced on ETAC_RESID_PERNODE_MLP contexts only");
  const float* pn[10] = {};
  if (p->struct_size == sizeof(etac_params)) {
    const float* q[10] = {p->E1, p->e1, p->E2, p->e2, p->G1, p->g1, p->D1, p->d1, p->D2, p->d2};
    for (int k = 0; k < 10; ++k) pn[k] = q[k], n_pn += q[k] != nullptr;
  }
  if (n_pn != 0 && n_pn != 10) return fail(ctx, ETAC_ERR_INVALID_ARG, "give all ten PointNet arrays or none");
  if (n_pn && ctx->m.resid != ETAC_RESID_POINTNET)
    return fail(ctx, ETAC_ERR_UNSUPPORTED, "E1 .. d2 can be replaced on ETAC_RESID_POINTNET contexts only");
  if (p->alpha) {
    if (p->n_alpha != ctx->n_alpha) return fail(ctx, ETAC_ERR_INVALID_ARG, "n_alpha differs from the context's");
    for (int k = 0; k < p->n_alpha; ++k)
      if (!(p->alpha[k] > 0.0f) || !isfinite(p->alpha[k])) return fail(ctx, ETAC_ERR_INVALID_ARG, "alpha must be > 0");
  }
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, ETAC_ERR_CUDA, "cudaSetDevice failed");
  cudaError_t e = cudaDeviceSynchronize();  // steps in flight read the old parameters
  if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("cudaDeviceSynchronize", e));
  DevModel& m = ctx->m;
  if (p->alpha) {  // Eq. (1): K_p is rebuilt on the device
    for (int q = 0; q < m.n_patches; ++q) ctx->hp[q].alpha = p->alpha[ctx->n_alpha == 1 ? 0 : q];
    e = cudaMemcpy(const_cast<PatchInfo*>(m.patch), ctx->hp.data(), sizeof(PatchInfo) * m.n_patches, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_build_k(m, ctx->k32_w, ctx->k16_w, 0);
    if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("rebuild K", e));
  }
  if (n_w) {
    PerNodeStage st;
    stage_pernode(p->W1, p->b1, p->W2, p->b2, p->W3, p->b3, &st);
    e = cudaMemcpy(const_cast<float*>(m.wf32), st.wf.data(), st.wf.size() * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(ctx->dW1_w, p->W1, 64 * 9 * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(ctx->db1_w, p->b1, 64 * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_build_c1(m, ctx->dW1_w, ctx->db1_w, const_cast<float*>(m.c1t), 0);
    if (e == cudaSuccess) e = cudaMemcpy(const_cast<uint8_t*>(m.wimg), st.img.data(), st.img.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("restage weights", e));
    memcpy(m.wout, st.wout, sizeof(m.wout));
  }
  if (n_pn) {
    PointNetStage st;
    stage_pointnet(pn[0], pn[1], pn[2], pn[3], pn[4], pn[5], pn[6], pn[7], pn[8], pn[9], &st);
    e = cudaMemcpy(const_cast<uint8_t*>(m.wimg_pn), st.img.data(), st.img.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(const_cast<float*>(m.pn_f32), st.pf.data(), st.pf.size() * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(const_cast<float*>(m.pn_w32), st.w32.data(), st.w32.size() * 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("restage PointNet weights", e));
    memcpy(m.wout, st.wout, sizeof(m.wout));
  }
  if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("update kernels", e));
  return ETAC_OK;
}

etac_status etac_backward(etac_ctx* ctx, void* cuda_stream, const etac_backward_args* a) {
  if (!ctx) return ETAC_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  // (a caller built against the header before the pose gradients were added passes the shorter struct)
  if (!a || (a->struct_size != sizeof(etac_backward_args) && a->struct_size != offsetof(etac_backward_args, d_grad_indenter_pose)))
    return fail(ctx, ETAC_ERR_INVALID_ARG, "bad etac_backward_args");
  const bool has_pose_fields = a->struct_size == sizeof(etac_backward_args);
  float* const g_ind_pose = has_pose_fields ? a->d_grad_indenter_pose : nullptr;
  float* const g_patch_pose = has_pose_fields ? a->d_grad_patch_pose : nullptr;
  if (a->n_envs < 0) return fail(ctx, ETAC_ERR_INVALID_ARG, "n_envs < 0");
  if (a->n_envs > ctx->m.max_envs) return fail(ctx, ETAC_ERR_CAPACITY, "n_envs > max_envs");
  if (a->input_mode != ETAC_IN_INDENTERS && a->input_mode != ETAC_IN_PENETRATION)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "bad input_mode");
  if (!a->d_grad_out || !a->d_grad_alpha) return fail(ctx, ETAC_ERR_INVALID_ARG, "d_grad_out and d_grad_alpha are required");
  if (a->input_mode == ETAC_IN_INDENTERS && ctx->m.max_ind > 0 && !a->d_indenters)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "d_indenters is NULL");
  if (a->input_mode == ETAC_IN_PENETRATION && !a->d_penetration)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "d_penetration is NULL");
  if (ctx->m.ablation != ETAC_ABLATE_FULL) return fail(ctx, ETAC_ERR_UNSUPPORTED, "etac_backward: ETAC_ABLATE_FULL only");
  if (ctx->m.resid == ETAC_RESID_NONE && a->d_grad_weights)
    return fail(ctx, ETAC_ERR_INVALID_ARG, "d_grad_weights given for a context without a residual network");
  if (g_ind_pose || g_patch_pose) {
    if (a->input_mode != ETAC_IN_INDENTERS)
      return fail(ctx, ETAC_ERR_INVALID_ARG, "pose gradients exist in ETAC_IN_INDENTERS mode only");
    if (!a->d_grad_penetration) return fail(ctx, ETAC_ERR_INVALID_ARG, "pose gradients need d_grad_penetration");
    if (ctx->m.max_ind > kMaxPoseGradIndenters) return fail(ctx, ETAC_ERR_UNSUPPORTED, "pose gradients: max_indenters > 256");
  }
  ctx->last_stream = s;
  if (a->n_envs == 0) return ETAC_OK;
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, ETAC_ERR_CUDA, "cudaSetDevice failed");
  StepIO io{};
  io.n_envs = a->n_envs, io.input_mode = a->input_mode;
  io.ind = a->d_indenters, io.patch_pose = a->d_patch_pose, io.pen_in = a->d_penetration;
  cudaError_t e;
  const bool pointnet = ctx->m.resid == ETAC_RESID_POINTNET;
  if ((e = cudaMemsetAsync(ctx->m.count, 0, sizeof(int32_t) * (ctx->m.n_patches + 3), s)) != cudaSuccess ||
      (e = cudaMemsetAsync(a->d_grad_alpha, 0, sizeof(float) * ctx->n_alpha, s)) != cudaSuccess ||
      (a->d_grad_weights && (e = cudaMemsetAsync(a->d_grad_weights, 0, sizeof(float) * (pointnet ? ETAC_GRAD_WEIGHTS_POINTNET_LEN : ETAC_GRAD_WEIGHTS_LEN), s)) != cudaSuccess) ||
      (a->d_grad_penetration &&
       (e = cudaMemsetAsync(a->d_grad_penetration, 0, sizeof(float) * (size_t)a->n_envs * ctx->m.n_nodes, s)) != cudaSuccess))
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("memset", e));
  int n_s1 = 1;
  if ((e = launch_sdf(ctx->m, io, 0, &n_s1, s)) != cudaSuccess)  // S1: delta and the pair flags only
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("sdf_penetration_kernel", e));
  // (PointNet: Phi does not see u_i, so backward_kernel runs without a residual -- dL/dalpha and the K part of
  //  dL/ddelta -- and k_backward_pointnet.cu adds the weight gradients and the encoder-input part of dL/ddelta)
  if ((e = launch_backward(ctx->m, io, a->d_grad_out, a->d_grad_alpha, ctx->n_alpha, pointnet ? nullptr : a->d_grad_weights,
                           a->d_grad_penetration, ctx->n_sm, s)) != cudaSuccess)
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("backward_kernel", e));
  int n_pn = 0;
  if (pointnet && (a->d_grad_weights || a->d_grad_penetration) &&
      (e = launch_backward_pointnet(ctx->m, io, a->d_grad_out, a->d_grad_weights, a->d_grad_penetration, ctx->n_sm, &n_pn, s)) != cudaSuccess)
    return fail(ctx, ETAC_ERR_CUDA, cuda_msg("pn_bwd_node_kernel", e));
  int n_pose = 0;
  if (g_ind_pose || g_patch_pose) {
    if (g_ind_pose && ctx->m.max_ind > 0 &&
        (e = cudaMemsetAsync(g_ind_pose, 0, sizeof(float) * 6 * (size_t)a->n_envs * ctx->m.max_ind, s)) != cudaSuccess)
      return fail(ctx, ETAC_ERR_CUDA, cuda_msg("memset", e));
    if ((e = launch_backward_pose(ctx->m, io, a->d_grad_penetration, g_ind_pose, g_patch_pose, s)) != cudaSuccess)
      return fail(ctx, ETAC_ERR_CUDA, cuda_msg("pose_grad_kernel", e));
    n_pose = 1;
  }
  ctx->last_launches = 1 + n_s1 + n_pn + n_pose;
  return ETAC_OK;
}

etac_status etac_time_steps(etac_ctx* ctx, void* cuda_stream, const etac_step_args* args, int32_t iters,
                            float* ms_per_step, float* ms_kernels) {
  if (!ctx || !ms_per_step || iters < 1) return ETAC_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  DeviceGuard guard(ctx->device);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, "cudaEventCreate");
  etac_status st = ETAC_OK;
  cudaStreamSynchronize(s);
  cudaEventRecord(e0, s);
  for (int i = 0; i < iters && st == ETAC_OK; ++i) st = step_impl(ctx, s, args, nullptr);
  cudaEventRecord(e1, s);
  cudaError_t e = cudaStreamSynchronize(s);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  *ms_per_step = ms / iters;
  cudaEventDestroy(e0), cudaEventDestroy(e1);
  if (st != ETAC_OK) return st;
  if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("etac_time_steps", e));
  if (ms_kernels) {
    // second pass with events between the kernels: [0] = S1 (incl. its memsets), [1] = fused S2-S4
    std::vector<cudaEvent_t> ev((size_t)iters * 3);
    for (auto& x : ev) cudaEventCreate(&x);
    for (int i = 0; i < iters && st == ETAC_OK; ++i) st = step_impl(ctx, s, args, &ev[(size_t)i * 3]);
    e = cudaStreamSynchronize(s);
    double a = 0, b = 0;
    if (st == ETAC_OK && e == cudaSuccess)
      for (int i = 0; i < iters; ++i) {
        float t;
        cudaEventElapsedTime(&t, ev[(size_t)i * 3], ev[(size_t)i * 3 + 1]), a += t;
        cudaEventElapsedTime(&t, ev[(size_t)i * 3 + 1], ev[(size_t)i * 3 + 2]), b += t;
      }
    for (auto& x : ev) cudaEventDestroy(x);
    ms_kernels[0] = (float)(a / iters), ms_kernels[1] = (float)(b / iters);
    if (st != ETAC_OK) return st;
    if (e != cudaSuccess) return fail(ctx, ETAC_ERR_CUDA, cuda_msg("etac_time_steps", e));
  }
  return ETAC_OK;
}

}  // extern "C"

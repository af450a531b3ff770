// etac_propagate_noalloc (include/etac_noalloc.h): the analytic propagation Omega U_a + mask of one patch
// for callers that must not allocate.  A variant of the gather form of S2
// (gather_fp32_kernel / the bf16 gather over S1's active-node lists) whose scratch -- the compact per-environment
// lists of active nodes -- is a file-scope __device__ array instead of a context workspace, and whose K is evaluated
// on the fly with the arithmetic of build_k_kernel.  Self-contained: shares no state with the context path.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/etac_noalloc.h"

namespace {

struct __align__(16) NaEntry {
  float ux, uy, uz;  // u^_j = -delta_j n_j
  int j;             // node
};
struct NaScratch {
  NaEntry list[ETAC_NOALLOC_MAX_ENTRIES];  // environment e: entries [e * n_nodes, e * n_nodes + count[e]), node order
  int count[ETAC_NOALLOC_MAX_ENVS];        // active nodes of environment e
};
// 4 MiB + 16 KiB per GPU that loads the library, until the process exits.  In HOST code `g_scratch` is only a
// stand-in for the symbol: its device address comes from cudaGetSymbolAddress (scratch_for_current_device).
static __device__ __align__(256) NaScratch g_scratch;

constexpr int kCompactThreads = 256, kRowThreads = 128;

// one CTA per environment: ordered compaction of the active nodes (delta > 0) into the environment's list
__global__ void __launch_bounds__(kCompactThreads) na_compact_kernel(NaScratch* __restrict__ sc, int n_nodes,
                                                                     const float* __restrict__ normal,
                                                                     const float* __restrict__ penetration) {
  __shared__ int s_wcnt[kCompactThreads / 32];
  const int e = blockIdx.x, t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const float* pen = penetration + (int64_t)e * n_nodes;
  NaEntry* list = sc->list + (int64_t)e * n_nodes;
  int base_slot = 0;
  for (int j0 = 0; j0 < n_nodes; j0 += kCompactThreads) {
    const int j = j0 + t;
    const float d = j < n_nodes ? fmaxf(pen[j], 0.0f) : 0.0f;  // negatives clamp (R19)
    const bool act = d > 0.0f;
    const unsigned bal = __ballot_sync(0xffffffffu, act);
    if (lane == 0) s_wcnt[warp] = __popc(bal);
    __syncthreads();
    int pre = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kCompactThreads / 32; ++w) {
      const int c = s_wcnt[w];
      pre += w < warp ? c : 0;
      total += c;
    }
    if (act) {
      NaEntry en;
      en.ux = -d * normal[3 * j], en.uy = -d * normal[3 * j + 1], en.uz = -d * normal[3 * j + 2], en.j = j;
      list[base_slot + pre + __popc(bal & ((1u << lane) - 1u))] = en;
    }
    base_slot += total;
    __syncthreads();  // s_wcnt is rewritten by the next sweep
  }
  if (t == 0) sc->count[e] = base_slot;  // overwritten by every call: nothing in the scratch has to start at zero
}

// thread = node i of environment e: Omega U_a over the environment's list, K_ij = exp(-alpha ||p_i - p_j||) as in
// build_k_kernel (row j, column i), sum in node order; active rows keep u^_i; environments without contact are 0
__global__ void __launch_bounds__(kRowThreads) na_rows_kernel(const NaScratch* __restrict__ sc, int n_nodes, int n_chunks, float alpha,
                                                              const float* __restrict__ pos, const float* __restrict__ normal,
                                                              const float* __restrict__ penetration, float* __restrict__ out) {
  __shared__ NaEntry s_en[kRowThreads];
  __shared__ float s_p[kRowThreads][3];
  const int e = blockIdx.x / n_chunks, i = (blockIdx.x - e * n_chunks) * kRowThreads + threadIdx.x;
  const bool valid = i < n_nodes;
  const int ic = valid ? i : 0;
  const int cnt = sc->count[e];
  const NaEntry* __restrict__ list = sc->list + (int64_t)e * n_nodes;
  const float px = pos[3 * ic], py = pos[3 * ic + 1], pz = pos[3 * ic + 2];
  float ax = 0.f, ay = 0.f, az = 0.f;
  for (int a0 = 0; a0 < cnt; a0 += kRowThreads) {
    const int nb = min(kRowThreads, cnt - a0);
    if ((int)threadIdx.x < nb) {
      const NaEntry en = list[a0 + threadIdx.x];
      s_en[threadIdx.x] = en;
      s_p[threadIdx.x][0] = pos[3 * en.j], s_p[threadIdx.x][1] = pos[3 * en.j + 1], s_p[threadIdx.x][2] = pos[3 * en.j + 2];
    }
    __syncthreads();
    for (int a = 0; a < nb; ++a) {
      const float dx = px - s_p[a][0], dy = py - s_p[a][1], dz = pz - s_p[a][2];
      const float k = expf(-alpha * sqrtf((dx * dx + dy * dy) + dz * dz));
      ax = fmaf(k, s_en[a].ux, ax), ay = fmaf(k, s_en[a].uy, ay), az = fmaf(k, s_en[a].uz, az);
    }
    __syncthreads();
  }
  if (!valid) return;
  const float d = fmaxf(penetration[(int64_t)e * n_nodes + i], 0.0f);
  if (d > 0.0f) ax = -d * normal[3 * i], ay = -d * normal[3 * i + 1], az = -d * normal[3 * i + 2];  // mask M_p
  float* o = out + ((int64_t)e * n_nodes + i) * 3;
  o[0] = ax, o[1] = ay, o[2] = az;
}

// device address of g_scratch on the current device: looked up once per device, with that device current
constexpr int kMaxDevices = 64;
std::mutex g_mu;
NaScratch* g_ptr[kMaxDevices] = {};

cudaError_t scratch_for_current_device(NaScratch** out, int* device) {
  cudaError_t e = cudaGetDevice(device);
  if (e != cudaSuccess) return e;
  if (*device < 0 || *device >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_ptr[*device]) {
    NaScratch* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_scratch);
    if (e != cudaSuccess) return e;
    g_ptr[*device] = p;
  }
  *out = g_ptr[*device];
  return cudaSuccess;
}

etac_status na_fail(etac_status st, char* err_msg, int32_t err_cap, const char* msg) {
  if (err_msg && err_cap > 0) snprintf(err_msg, (size_t)err_cap, "etac_propagate_noalloc: %s", msg);
  return st;
}

}  // namespace

extern "C" etac_status etac_propagate_noalloc(void* cuda_stream, int32_t n_envs, int32_t n_nodes, float alpha, const float* d_pos,
                                              const float* d_normal, const float* d_penetration, float* d_out, char* err_msg,
                                              int32_t err_cap) {
  if (err_msg && err_cap > 0) err_msg[0] = '\0';
  char buf[192];
  if (n_envs < 0 || n_nodes < 0) return na_fail(ETAC_ERR_INVALID_ARG, err_msg, err_cap, "n_envs and n_nodes must be >= 0");
  if (!(alpha > 0.0f) || !isfinite(alpha)) return na_fail(ETAC_ERR_INVALID_ARG, err_msg, err_cap, "alpha must be finite and > 0");
  if (n_envs == 0 || n_nodes == 0) return ETAC_OK;
  if (!d_pos || !d_normal || !d_penetration || !d_out) return na_fail(ETAC_ERR_INVALID_ARG, err_msg, err_cap, "NULL device pointer");
  if (n_envs > ETAC_NOALLOC_MAX_ENVS) {
    snprintf(buf, sizeof buf, "n_envs = %d exceeds ETAC_NOALLOC_MAX_ENVS = %d", n_envs, ETAC_NOALLOC_MAX_ENVS);
    return na_fail(ETAC_ERR_CAPACITY, err_msg, err_cap, buf);
  }
  if ((long long)n_envs * n_nodes > ETAC_NOALLOC_MAX_ENTRIES) {
    snprintf(buf, sizeof buf, "n_envs * n_nodes = %lld exceeds the static scratch of ETAC_NOALLOC_MAX_ENTRIES = %d entries",
             (long long)n_envs * n_nodes, ETAC_NOALLOC_MAX_ENTRIES);
    return na_fail(ETAC_ERR_CAPACITY, err_msg, err_cap, buf);
  }
  NaScratch* sc = nullptr;
  int device = 0;
  cudaError_t e = scratch_for_current_device(&sc, &device);
  if (e != cudaSuccess) {
    snprintf(buf, sizeof buf, "cudaGetSymbolAddress(scratch) on device %d: %s", device, cudaGetErrorString(e));
    return na_fail(ETAC_ERR_CUDA, err_msg, err_cap, buf);
  }
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int n_chunks = (n_nodes + kRowThreads - 1) / kRowThreads;
  na_compact_kernel<<<n_envs, kCompactThreads, 0, s>>>(sc, n_nodes, d_normal, d_penetration);
  na_rows_kernel<<<(unsigned)((int64_t)n_chunks * n_envs), kRowThreads, 0, s>>>(sc, n_nodes, n_chunks, alpha, d_pos, d_normal, d_penetration,
                                                                             d_out);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(buf, sizeof buf, "kernel launch: %s", cudaGetErrorString(e));
    return na_fail(ETAC_ERR_CUDA, err_msg, err_cap, buf);
  }
  return ETAC_OK;
}

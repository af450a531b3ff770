// S2+S3+S4, fp32 SIMT "sparse gather" path: Omega U_a literally -- every node of
// a contacting (env, patch) sums exp-decay contributions of the ACTIVE nodes only -- followed by
// the per-node residual MLP (fp32) and the mask/combine of Eq. (2).
// Used for ETAC_PREC_FP32 contexts and for ETAC_PATH_SPARSE.
//
// Work item = kGatherChunk (128) consecutive nodes of one patch in one environment; persistent CTAs of 256 threads.
// K is symmetric, so K[i][j] is read as K[j][i]: for a fixed active j the threads of a half read 128
// consecutive floats of row j (coalesced).  Active nodes are compacted in node order with
// ballots (deterministic summation order).
#include "etac_internal.h"

namespace etac {

constexpr int kWf32Floats = 64 * 3 + 64 * 64 + 64 + 3 * 64 + 3;  // W1u | W2 | b2 | W3 | b3

// silu(x) = x / (1 + e^-x) with the hardware exponential and reciprocal (MUFU.EX2, MUFU.RCP: relative error of a
// few 1e-7, far inside the 1e-4 bar of the fp32 path); the IEEE expf / division sequences cost five times the
// instructions and their slow-path branches serialise the 64 activations of a thread.  x << 0: e^-x = inf, x/inf = -0.
__device__ __forceinline__ float silu_f32(float x) { return __fdividef(x, 1.0f + __expf(-x)); }

// The residual MLP of the chunk's 128 nodes runs as CTA-level products through shared memory (256 threads):
//   layer 1  thread = (node, half of the hidden units): 32 units each, position / normal part precomputed (c1t)
//   layer 2  H2[64 x 128] = W2 H1 as 4 outputs x 8 nodes register tiles: 3 shared-memory loads per 32 FMAs
//            (a thread-per-node loop over W2 needs one load per 4 FMAs and is bound by shared-memory reads)
//   layer 3  thread = (node, half of the hidden units), partial sums combined through shared memory
// The grid is persistent: the weights (W2 transposed, so that a thread's four outputs are one 16-byte load) are
// staged once per CTA, not once per 128 nodes.
constexpr int kCtasPerSm = 3;            // 80 registers, 73 KB of shared memory: the phases of three items overlap on an SM
constexpr int kGT = 2 * kGatherChunk;   // threads per CTA
constexpr int kSub = 4, kSweep = kSub * kGT;  // nodes of a patch scanned per sweep: kSub per thread
constexpr int kCache = 1024;             // entries of the cached active-node list
constexpr int kMaxSeg = 64;              // sweeps of a patch whose list can be cached (patches of up to 65,536 nodes)
constexpr int kDepth = 16;              // K loads in flight per thread in the gather
constexpr int kHld = kGatherChunk + 4;  // row pitch of the [64][128] activation arrays (rows stay 16-byte aligned)
struct GatherSmem {
  float w2t[64 * 64];  // [k][k2]
  float w1u[64 * 3], b2[64], w3[3 * 64], b3[4];
  union {                          // the gather is over before the MLP starts
    float H[64 * kHld];            // hidden activations [k][node]: H1, then H2 in place
    struct {
      float u[kSweep][3];          // compacted active nodes of one sweep: u^_j and j
      int j[kSweep];
    };
  };
  float ulin[3][kGatherChunk];
  float part[2][3][kGatherChunk];  // per-half partial sums (gather: upper half; layer 3: upper half)
  int wcnt[kSub * (kGT / 32)];
  // (last: the one-chunk-per-item instantiation is launched without them)
  float cu[kCache][3];             // cached list of a patch's active nodes, shared by the chunks of an item
  int cj[kCache];
  int seg[kMaxSeg + 1];            // first entry of every sweep's part of the cached list (+ end)
};
constexpr size_t kGatherSmemNoCache = offsetof(GatherSmem, cu);
static_assert(sizeof(float) * (kSweep * 3 + kSweep) <= sizeof(float) * 64 * kHld, "sweep arrays inside H");

// Ordered compaction of the active nodes (delta > 0) among the nodes [base, base + kSweep) of a patch: entries
// (u^_j, j) are appended in node order at u[slot0 ..], jl[slot0 ..] as far as they fit below `cap`; returns the number
// of active nodes of the sweep.  Four delta loads in flight per thread: a sweep costs one L2 round trip and two barriers.
__device__ __forceinline__ int compact_sweep(GatherSmem& S, const float4* __restrict__ nrm4, int pn, const float* __restrict__ delta,
                                             int base, float (*__restrict__ u)[3], int* __restrict__ jl, int slot0, int cap) {
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  float d[kSub];
  unsigned bal[kSub];
#pragma unroll
  for (int q = 0; q < kSub; ++q) {
    const int j = base + q * kGT + t;
    d[q] = j < pn ? delta[j] : 0.0f;
  }
#pragma unroll
  for (int q = 0; q < kSub; ++q) {
    bal[q] = __ballot_sync(0xffffffffu, d[q] > 0.0f);
    if (lane == 0) S.wcnt[q * (kGT / 32) + warp] = __popc(bal[q]);
  }
  __syncthreads();
  int pre[kSub] = {0, 0, 0, 0}, total = 0;
#pragma unroll
  for (int w = 0; w < kSub * (kGT / 32); ++w) {
    const int c = S.wcnt[w];
#pragma unroll
    for (int q = 0; q < kSub; ++q) pre[q] += w < q * (kGT / 32) + warp ? c : 0;
    total += c;
  }
#pragma unroll
  for (int q = 0; q < kSub; ++q)
    if (d[q] > 0.0f) {
      const int j = base + q * kGT + t;
      const int slot = slot0 + pre[q] + __popc(bal[q] & ((1u << lane) - 1u));
      if (slot < cap) {
        const float4 n = nrm4[j];
        jl[slot] = j;
        u[slot][0] = -d[q] * n.x, u[slot][1] = -d[q] * n.y, u[slot][2] = -d[q] * n.z;
      }
    }
  __syncthreads();  // entries visible; wcnt free for the next sweep
  return total;
}

// a += sum over the list of K[j][li] u^_j: the two halves of the CTA take alternating groups of kDepth entries for
// their node, kDepth loads of K in flight per thread (the loop is bound by their latency); fixed order: deterministic
__device__ __forceinline__ void gather_list(const float (*__restrict__ u)[3], const int* __restrict__ jl, int total, const float* __restrict__ K, int n, int li,
                                            int half, float& ax, float& ay, float& az) {
  for (int a0 = half * kDepth; a0 < total; a0 += 2 * kDepth) {
    float kv[kDepth];
#pragma unroll
    for (int q = 0; q < kDepth; ++q) kv[q] = a0 + q < total ? K[(int64_t)jl[a0 + q] * n + li] : 0.0f;
#pragma unroll
    for (int q = 0; q < kDepth; ++q) {
      const int a = min(a0 + q, total - 1);  // (kv = 0 beyond the list)
      ax = fmaf(kv[q], u[a][0], ax);
      ay = fmaf(kv[q], u[a][1], ay);
      az = fmaf(kv[q], u[a][2], az);
    }
  }
}

// kShare: work items of several chunks with the shared list (cpg > 1); false: one chunk per item, no cache code
template <bool kShare>
__global__ void __launch_bounds__(kGT, kCtasPerSm) gather_fp32_kernel(DevModel m, StepIO io, int cpg) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  GatherSmem& S = *reinterpret_cast<GatherSmem*>(smem_raw);
  const int t = threadIdx.x;
  const int node = t & (kGatherChunk - 1), half = t >> 7;  // (warp-uniform)
  const bool mlp = m.resid != ETAC_RESID_NONE;
  if (mlp) {
    const float4* w2t = reinterpret_cast<const float4*>(m.wf32 + kWf32W2t);  // [k][k2], transposed at create
#pragma unroll
    for (int i = t; i < 1024; i += kGT) reinterpret_cast<float4*>(S.w2t)[i] = w2t[i];
    if (t < 192) S.w1u[t] = m.wf32[t], S.w3[t] = m.wf32[192 + 4096 + 64 + t];
    if (t < 64) S.b2[t] = m.wf32[192 + 4096 + t];
    if (t < 3) S.b3[t] = m.wf32[192 + 4096 + 64 + 192 + t];
  }
  __syncthreads();

  // Work item = `cpg` consecutive chunks of one environment (the host sizes cpg so that every CTA still gets several
  // items).  The chunks of one patch in an item share the patch's compacted active-node list if it fits the cache:
  // without it every chunk scans all delta of its patch, N / 128 scans per environment and patch.
  const int gpe = (m.n_chunks + cpg - 1) / cpg;  // items per environment
  const int64_t n_items = (int64_t)gpe * io.n_envs;
  for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
   const int e = (int)(item / gpe);
   const int c0 = (int)(item - (int64_t)e * gpe) * cpg, c1 = min(c0 + cpg, m.n_chunks);
   int cache_patch = -1, cache_total = -1, cache_nseg = 0;  // cache_total < 0: the list of cache_patch did not fit
   for (int c = c0; c < c1; ++c) {
    const ChunkInfo ch = m.chunk[c];
    if (!m.flags[(int64_t)e * m.n_patches + ch.patch]) continue;  // S1 zero-filled this patch (uniform over the CTA)
    const PatchInfo pi = m.patch[ch.patch];
    const bool valid = node < ch.count;
    const int g = ch.node0 + (valid ? node : 0);
    const int li = g - pi.off;
    const float* __restrict__ delta = m.delta + (int64_t)e * m.n_nodes + pi.off;
    const float* __restrict__ K = m.k32 + pi.k32_off;

    // ---- Omega U_a over the patch's active nodes in node order
    float ax = 0.f, ay = 0.f, az = 0.f;
    if (kShare && ch.patch != cache_patch && c + 1 < c1 && m.chunk[c + 1].patch == ch.patch) {  // more chunks of this patch follow
      // (the list is summed sweep by sweep, like the uncached form below: an environment's result then has the same
      //  bits whichever form the size of the launch selects)
      int total = 0, ns = 0;
      for (int base = 0; base < pi.n; base += kSweep, ++ns) {
        if (t == 0 && ns < kMaxSeg) S.seg[ns] = min(total, kCache);
        total += compact_sweep(S, m.nrm4 + pi.off, pi.n, delta, base, S.cu, S.cj, total, kCache);
      }
      if (t == 0 && ns <= kMaxSeg) S.seg[ns] = min(total, kCache);
      __syncthreads();
      cache_patch = ch.patch, cache_total = (total <= kCache && ns <= kMaxSeg) ? total : -1, cache_nseg = ns;
    }
    if (kShare && ch.patch == cache_patch && cache_total >= 0) {
      for (int sg = 0; sg < cache_nseg; ++sg) {
        const int b0 = S.seg[sg];
        gather_list(S.cu + b0, S.cj + b0, S.seg[sg + 1] - b0, K, pi.n, li, half, ax, ay, az);
      }
    } else {
      for (int base = 0; base < pi.n; base += kSweep) {  // (sweep arrays inside H: the previous chunk's MLP is over)
        const int total = compact_sweep(S, m.nrm4 + pi.off, pi.n, delta, base, S.u, S.j, 0, kSweep);
        gather_list(S.u, S.j, total, K, pi.n, li, half, ax, ay, az);
        __syncthreads();
      }
    }
    if (half) S.part[0][0][node] = ax, S.part[0][1][node] = ay, S.part[0][2][node] = az;
    __syncthreads();
    if (!half) {
      ax += S.part[0][0][node], ay += S.part[0][1][node], az += S.part[0][2][node];
      S.ulin[0][node] = ax, S.ulin[1][node] = ay, S.ulin[2][node] = az;
    }
    float r0 = 0.f, r1 = 0.f, r2 = 0.f;
    if (mlp) {
      __syncthreads();
      // ---- layer 1: 32 hidden units of this thread's node
      {
        const float ux = S.ulin[0][node], uy = S.ulin[1][node], uz = S.ulin[2][node];
        const float* __restrict__ c1 = m.c1t + (int64_t)(32 * half) * m.n_nodes + g;
#pragma unroll
        for (int q0 = 0; q0 < 32; q0 += 16) {  // 16 loads of the precomputed part in flight
          float z[16];
#pragma unroll
          for (int q = 0; q < 16; ++q) z[q] = c1[(int64_t)(q0 + q) * m.n_nodes];
#pragma unroll
          for (int q = 0; q < 16; ++q) {
            const int k = 32 * half + q0 + q;
            float zz = z[q];
            zz = fmaf(S.w1u[k * 3 + 0], ux, zz), zz = fmaf(S.w1u[k * 3 + 1], uy, zz), zz = fmaf(S.w1u[k * 3 + 2], uz, zz);
            S.H[k * kHld + node] = silu_f32(zz);
          }
        }
      }
      __syncthreads();
      // ---- layer 2: outputs 4 og .. 4 og + 3 of the nodes 4 ng .. 4 ng + 3 and 64 + 4 ng .. 64 + 4 ng + 3
      {
        const int ng = t & 15, og = t >> 4;
        float acc[4][8];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int c = 0; c < 8; ++c) acc[r][c] = S.b2[4 * og + r];
#pragma unroll 4
        for (int k = 0; k < 64; ++k) {
          const float4 a0 = *reinterpret_cast<const float4*>(&S.H[k * kHld + 4 * ng]);
          const float4 a1 = *reinterpret_cast<const float4*>(&S.H[k * kHld + 64 + 4 * ng]);
          const float4 w = *reinterpret_cast<const float4*>(&S.w2t[k * 64 + 4 * og]);
          const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
          const float wv[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
          for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int c = 0; c < 8; ++c) acc[r][c] = fmaf(wv[r], av[c], acc[r][c]);
        }
        __syncthreads();  // every thread has read H1: H2 goes in its place
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          float* row = &S.H[(4 * og + r) * kHld];
          *reinterpret_cast<float4*>(row + 4 * ng) =
              make_float4(silu_f32(acc[r][0]), silu_f32(acc[r][1]), silu_f32(acc[r][2]), silu_f32(acc[r][3]));
          *reinterpret_cast<float4*>(row + 64 + 4 * ng) =
              make_float4(silu_f32(acc[r][4]), silu_f32(acc[r][5]), silu_f32(acc[r][6]), silu_f32(acc[r][7]));
        }
      }
      __syncthreads();
      // ---- layer 3: this thread's half of the hidden units of its node
#pragma unroll 8
      for (int q = 0; q < 32; ++q) {
        const int k = 32 * half + q;
        const float h2 = S.H[k * kHld + node];
        r0 = fmaf(S.w3[k], h2, r0), r1 = fmaf(S.w3[64 + k], h2, r1), r2 = fmaf(S.w3[128 + k], h2, r2);
      }
      if (half) S.part[1][0][node] = r0, S.part[1][1][node] = r1, S.part[1][2][node] = r2;
      __syncthreads();
      if (!half) {
        r0 = (S.b3[0] + r0) + S.part[1][0][node];
        r1 = (S.b3[1] + r1) + S.part[1][1][node];
        r2 = (S.b3[2] + r2) + S.part[1][2][node];
      }
    }
    if (half || !valid) continue;  // (the next item's first barrier orders the reuse of the shared arrays)

    float ox = ax, oy = ay, oz = az;
    if (!mlp && m.residual_only) ox = oy = oz = 0.0f;  // Phi_p of a context without Phi
    if (mlp) {
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
  }
}

cudaError_t gather_fp32_configure() {
  cudaError_t e = cudaFuncSetAttribute(gather_fp32_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GatherSmem));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(gather_fp32_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GatherSmem));
  return e;
}

cudaError_t launch_gather_fp32(const DevModel& m, const StepIO& io, int n_sm, cudaStream_t s) {
  const int64_t slots = (int64_t)kCtasPerSm * n_sm, n_chunk_items = (int64_t)m.n_chunks * io.n_envs;
  // chunks per item: as many as leave every resident CTA about eight items (load balance), at most 16
  // (only for meshes with a patch of >= 8 chunks: on small patches the shared list saves less than the larger items cost)
  int cpg = (int)(n_chunk_items / (8 * slots) < 1 ? 1 : (n_chunk_items / (8 * slots) > 16 ? 16 : n_chunk_items / (8 * slots)));
  if (m.max_patch_nodes < 8 * kGatherChunk) cpg = 1;
  const int64_t n_items = (int64_t)((m.n_chunks + cpg - 1) / cpg) * io.n_envs;
  const unsigned grid = (unsigned)(n_items < slots ? n_items : slots);
  if (cpg > 1) gather_fp32_kernel<true><<<grid, kGT, sizeof(GatherSmem), s>>>(m, io, cpg);
  else gather_fp32_kernel<false><<<grid, kGT, kGatherSmemNoCache, s>>>(m, io, 1);
  return cudaGetLastError();
}

}  // namespace etac

// S1: contact detection and penalty displacement of the active nodes.
//
// One CTA per environment.  Every node of a non-culled patch is transformed into the world
// frame of the indenters, the union SDF phi = min_k sdf_k is evaluated, active <=> phi < 0,
// delta = -phi on active nodes.  The arithmetic of phi is single-rounded fp32 in a fixed order
// (no FMA contraction -> __fmul_rn/__fadd_rn/__fsub_rn/__fsqrt_rn) so that the
// contact decision is reproducible by an independent fp32 implementation.
//
// Outputs: delta workspace [E x N] (only where the patch was evaluated), per-(env,patch) contact
// flag, per-patch compact list of contacting environments (slot = position in that list), and,
// for the tensor-core path, the GEMM B operand U^ = -delta * n as bf16 rows uhat_t[slot*3+c][j].
// A patch with no active node gets its rows of the output zero-filled (R8) -- here for
// the gather path, by the idle warps of the fused kernel for the tensor-core path -- so the
// contraction kernels only ever compute contacting (env, patch) pairs.
#include "etac_internal.h"
#include "sdf_device.cuh"

namespace etac {


// Task of the two-kernel S1 (sdf_cull_kernel -> sdf_eval_kernel): a pair that survived the cull, with the rotations
// the cull computed
struct __align__(16) PairTask {
  float R[9], t[3];  // patch pose
  SInd ind;          // the environment's indenter (type NONE if it is this patch's own link)
  int pair;
  int evaluated;     // 0: culled -- only the contact-free outputs remain to be written
};
static_assert(sizeof(PairTask) == 128, "PairTask");


__device__ __forceinline__ void zero_fill(float* __restrict__ p, int count) {
  // p is 4-byte aligned; vectorise the 16-byte aligned body
  const int head = min(count, (int)(((16u - (uint32_t)((uintptr_t)p & 15u)) & 15u) >> 2));
  if ((int)threadIdx.x < head) p[threadIdx.x] = 0.0f;
  float4* body = reinterpret_cast<float4*>(p + head);
  const int nvec = (count - head) >> 2;
  for (int v = threadIdx.x; v < nvec; v += blockDim.x) body[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  const int tail0 = head + (nvec << 2);
  if (tail0 + (int)threadIdx.x < count) p[tail0 + threadIdx.x] = 0.0f;
}

constexpr int kPoseChunk = 32;
constexpr int kNodeChunk = 4;  // nodes per thread evaluated against one indenter held in registers
struct SPose {
  float R[9];
  float t[3];
  int evaluated;  // 0 = culled by the bounding-sphere test
};

// One CTA per environment.  Patches are handled kPoseChunk at a time in four block-wide phases
// (3 barriers per chunk, none per patch):
//   B  one thread per patch: pose -> rotation, conservative bounding-sphere cull
//   C  all threads: nodes of the non-culled patches -> phi, delta (workspace), per-patch "any"
//   D  one thread per patch: contact flag, slot in the patch's compact environment list
//   E  all threads: contact-free patches -> zero-fill of the output rows; contacting patches ->
//      U^ operand rows (bf16), optional delta / mask outputs
template <bool kIndenters, bool kGrid>
__global__ void __launch_bounds__(256, 4) sdf_penetration_kernel(DevModel m, StepIO io, int s1_flags) {
  // kS1Bucket: the slot of a contacting pair and its U^ rows are left to sdf_scatter_kernel (counting sort of the
  // environments by contact position); this kernel records the key and counts the environments per key
  const bool bucket = s1_flags & kS1Bucket;
  const bool write_uhat = (s1_flags & kS1WriteUhat) && !bucket, write_alist = s1_flags & kS1WriteAlist, fill_out = s1_flags & kS1FillOut;
  __shared__ int s_wcnt[8];
  __shared__ int s_key[kPoseChunk];  // first active node of the patch
  extern __shared__ uint8_t smem_raw[];
  SInd* sind = reinterpret_cast<SInd*>(smem_raw);
  float4* s_tb = reinterpret_cast<float4*>(smem_raw + (((size_t)(m.max_ind > 0 ? m.max_ind : 1) * sizeof(SInd) + 15) & ~(size_t)15));  // (t, rb2)
  __shared__ SPose s_pose[kPoseChunk];
  __shared__ int s_any[kPoseChunk];
  __shared__ int s_slot[kPoseChunk];
  __shared__ int s_off[kPoseChunk + 1];  // node offsets of the chunk's patches (+ end)
  __shared__ uint32_t s_kb[kKbWords];
  __shared__ int s_nind;  // indenters of the environment that are not empty slots

  const int e = blockIdx.x;
  const int lane = threadIdx.x & 31;
  const int words = (m.n_nodes + 31) >> 5;
  const bool posed = io.patch_pose != nullptr;
  if constexpr (kIndenters) {
    // the environment's indenters, empty slots dropped (slot order kept): every node pays a pre-test per entry
    if (threadIdx.x < 32) {
      int n_act = 0;
      for (int k0 = 0; k0 < m.max_ind; k0 += 32) {
        const int k = k0 + lane;
        SInd s;
        s.type = ETAC_IND_NONE;
        if (k < m.max_ind) s = load_indenter(io.ind + (int64_t)e * m.max_ind + k);
        const uint32_t bal = __ballot_sync(0xffffffffu, s.type != ETAC_IND_NONE);
        if (s.type != ETAC_IND_NONE) {
          const int pos = n_act + __popc(bal & ((1u << lane) - 1u));
          sind[pos] = s;
          s_tb[pos] = make_float4(s.t[0], s.t[1], s.t[2], s.rb2);
        }
        n_act += __popc(bal);
      }
      if (lane == 0) s_nind = n_act;
    }
  }
  for (int p0 = 0; p0 < m.n_patches; p0 += kPoseChunk) {
    const int np = min(kPoseChunk, m.n_patches - p0);
    __syncthreads();  // sind ready / previous chunk fully consumed
    const int n_ind = kIndenters ? s_nind : 0;
    // ---- phase B
    if ((int)threadIdx.x < np) {
      const int p = p0 + threadIdx.x;
      s_any[threadIdx.x] = 0;
      s_key[threadIdx.x] = 0x7fffffff;
      {
        const PatchInfo pi0 = m.patch[p];
        s_off[threadIdx.x] = pi0.off;
        if ((int)threadIdx.x == np - 1) s_off[np] = pi0.off + pi0.n;
      }
      if constexpr (kIndenters) {
        const PatchInfo pi = m.patch[p];
        SPose sp;
        float C0 = pi.bc[0], C1 = pi.bc[1], C2 = pi.bc[2];
        if (posed) {
          const float* pp = io.patch_pose + ((int64_t)e * m.n_patches + p) * 7;
          const float q[4] = {pp[3], pp[4], pp[5], pp[6]};
          sp.t[0] = pp[0], sp.t[1] = pp[1], sp.t[2] = pp[2];
          quat_to_rot(q, sp.R);
          const float x = C0, y = C1, z = C2;
          C0 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(sp.R[0], x), __fmul_rn(sp.R[1], y)), __fmul_rn(sp.R[2], z)), sp.t[0]);
          C1 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(sp.R[3], x), __fmul_rn(sp.R[4], y)), __fmul_rn(sp.R[5], z)), sp.t[1]);
          C2 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(sp.R[6], x), __fmul_rn(sp.R[7], y)), __fmul_rn(sp.R[8], z)), sp.t[2]);
        }
        // conservative cull: exact SDFs are 1-Lipschitz, so phi(x_i) >= phi(c) - brad
        const float phi_lo = union_sdf_lower<kGrid>(sind, n_ind, C0, C1, C2, pi.brad, m.grid, p + 1);
        // (phi_lo = +inf: no indenter applies to this patch -- all slots NONE, or only the patch's own link)
        sp.evaluated = phi_lo < __int_as_float(0x7f800000) && !(phi_lo > 0.01f + 1e-5f * (fabsf(phi_lo) + 3.0f * pi.brad));
        s_pose[threadIdx.x] = sp;
      }
    }
    __syncthreads();
    // ---- phase C
    for (int q = 0; q < np; ++q) {
      if constexpr (kIndenters) {
        if (!s_pose[q].evaluated) continue;
      }
      PatchInfo pi;
      pi.off = s_off[q], pi.n = s_off[q + 1] - s_off[q];
      const int64_t row0 = (int64_t)e * m.n_nodes + pi.off;
      float* delta = m.delta + row0;
      bool any = false;
      int nact = 0, first_act = 0x7fffffff;
      if constexpr (kIndenters) {
        const SPose& sp = s_pose[q];
        // kNodeChunk nodes per thread at a time with the indenter loop outside: an indenter's 17 words are
        // read from shared memory once per chunk instead of once per node; the union is still the min over
        // the slots in slot order, node by node
        for (int i0 = threadIdx.x; i0 < pi.n; i0 += blockDim.x * kNodeChunk) {
          float X[kNodeChunk][3], phi[kNodeChunk];
#pragma unroll
          for (int c = 0; c < kNodeChunk; ++c) {
            const int i = min(i0 + c * (int)blockDim.x, pi.n - 1);
            const float4 pos = m.pos4[pi.off + i];
            X[c][0] = pos.x, X[c][1] = pos.y, X[c][2] = pos.z;
            if (posed) {
              X[c][0] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(sp.R[0], pos.x), __fmul_rn(sp.R[1], pos.y)), __fmul_rn(sp.R[2], pos.z)), sp.t[0]);
              X[c][1] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(sp.R[3], pos.x), __fmul_rn(sp.R[4], pos.y)), __fmul_rn(sp.R[5], pos.z)), sp.t[1]);
              X[c][2] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(sp.R[6], pos.x), __fmul_rn(sp.R[7], pos.y)), __fmul_rn(sp.R[8], pos.z)), sp.t[2]);
            }
            phi[c] = __int_as_float(0x7f800000);
          }
          for (int k = 0; k < n_ind; ++k) {
            // A node further than the shape's bounding radius (+ margin) from its origin has phi > 0.05 whatever the
            // rounding: it stays passive (delta = 0) without the exact, single-rounded evaluation.  On a large patch
            // most nodes are far from every indenter (one 16-byte load and 7 instructions per slot and node instead
            // of the 18-word record and the two transforms).
            const float4 tb = s_tb[k];
            bool near[kNodeChunk], any_near = false;
#pragma unroll
            for (int c = 0; c < kNodeChunk; ++c) {
              const float dx = X[c][0] - tb.x, dy = X[c][1] - tb.y, dz = X[c][2] - tb.z;
              near[c] = !(fmaf(dx, dx, fmaf(dy, dy, dz * dz)) > tb.w);
              any_near |= near[c];
            }
            if (!any_near) continue;
            if (sind[k].skip1 == p0 + q + 1) continue;
            const SInd s = sind[k];
#pragma unroll
            for (int c = 0; c < kNodeChunk; ++c)
              if (near[c]) phi[c] = fminf(phi[c], sdf_one<kGrid>(s, X[c][0], X[c][1], X[c][2], m.grid));
          }
#pragma unroll
          for (int c = 0; c < kNodeChunk; ++c) {
            const int i = i0 + c * (int)blockDim.x;
            if (i < pi.n) {
              const float d = phi[c] < 0.0f ? -phi[c] : 0.0f;
              delta[i] = d;
              any |= d > 0.0f;
              nact += d > 0.0f;
              if (d > 0.0f) first_act = min(first_act, i);
            }
          }
        }
      } else {
        for (int i = threadIdx.x; i < pi.n; i += blockDim.x) {
          const float d = fmaxf(io.pen_in[row0 + i], 0.0f);
          delta[i] = d;
          any |= d > 0.0f;
          nact += d > 0.0f;
          if (d > 0.0f) first_act = min(first_act, i);
        }
      }
      if (__any_sync(0xffffffffu, any) && lane == 0) atomicOr(&s_any[q], 1);
      if (bucket) {
        first_act = __reduce_min_sync(0xffffffffu, first_act);
        if (lane == 0 && first_act != 0x7fffffff) atomicMin(&s_key[q], first_act);
      }
      if (io.nact_out) {
        nact = __reduce_add_sync(0xffffffffu, nact);
        if (lane == 0 && nact) atomicAdd(&io.nact_out[e], nact);
      }
    }
    __syncthreads();
    // ---- phase D
    if ((int)threadIdx.x < np) {
      const int p = p0 + threadIdx.x;
      const int hit = s_any[threadIdx.x];
      m.flags[(int64_t)e * m.n_patches + p] = (uint8_t)hit;
      if (io.contact_out) io.contact_out[(int64_t)e * m.n_patches + p] = (uint8_t)hit;
      if (hit && bucket) {
        const int n_p = s_off[threadIdx.x + 1] - s_off[threadIdx.x];
        const int key = (int)(((int64_t)s_key[threadIdx.x] << 8) / n_p);  // 0..255: position of the first active node
        m.keybuf[(int64_t)e * m.n_patches + p] = (uint8_t)key;
        atomicAdd(&m.khist[p * 256 + key], 1);
        s_slot[threadIdx.x] = 0;
      } else if (hit) {
        const int slot = atomicAdd(&m.count[p], 1);
        m.envlist[(int64_t)p * m.max_envs + slot] = e;
        s_slot[threadIdx.x] = slot;
      }
    }
    __syncthreads();
    // ---- phase E (runs of consecutive contact-free patches are zero-filled in one go)
    int run0 = -1;
    for (int q = 0; q <= np; ++q) {
      const bool hit = q < np && s_any[q];
      if (q < np && !hit) {
        if (run0 < 0) run0 = q;
        continue;
      }
      if (run0 >= 0) {
        const int64_t r0 = (int64_t)e * m.n_nodes + s_off[run0];
        const int cnt = s_off[q] - s_off[run0];
        if (fill_out) {  // (tensor-core paths: the fused kernel's issuer warps zero-fill these rows)
          zero_out_rows(io, e, s_off[run0], cnt, threadIdx.x, blockDim.x);
          if (io.analytic_out) zero_fill(io.analytic_out + r0 * 3, cnt * 3);
        }
        if (io.pen_out) zero_fill(io.pen_out + r0, cnt);
        run0 = -1;
      }
      if (q == np) break;
      const int off = s_off[q], n = s_off[q + 1] - off, uoff = m.patch[p0 + q].uoff;
      const int64_t row0 = (int64_t)e * m.n_nodes + off;
      const int slot = s_slot[q];
      const float* delta = m.delta + row0;
      if (write_alist) {
        // compact list of the patch's active nodes in node order (block-wide ordered compaction)
        ActiveEntry* al = m.alist + (int64_t)slot * m.ldu + off;
        int base = 0;
        for (int i0 = 0; i0 < n; i0 += blockDim.x) {
          const int i = i0 + threadIdx.x;
          const float d = i < n ? delta[i] : 0.0f;
          const uint32_t bal = __ballot_sync(0xffffffffu, d > 0.0f);
          if (lane == 0) s_wcnt[threadIdx.x >> 5] = __popc(bal);
          __syncthreads();
          int before = base, total = base;
          for (int w = 0; w < 8; ++w) {
            if (w < (int)(threadIdx.x >> 5)) before += s_wcnt[w];
            total += s_wcnt[w];
          }
          if (d > 0.0f) {
            const float4 nn = m.nrm4[off + i];
            ActiveEntry en;
            en.ux = -d * nn.x, en.uy = -d * nn.y, en.uz = -d * nn.z, en.j = i;
            al[before + __popc(bal & ((1u << lane) - 1u))] = en;
          }
          base = total;
          __syncthreads();
        }
        if (threadIdx.x == 0) m.acount[(int64_t)(p0 + q) * m.max_envs + slot] = base;
      }
      if (write_uhat) {  // bitmap of the 64-node k-blocks that hold an active node (the contraction skips the others)
        if (threadIdx.x < kKbWords) s_kb[threadIdx.x] = 0;
        __syncthreads();
      }
      for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const float d = delta[i];
        if (io.pen_out) io.pen_out[row0 + i] = d;
        if (io.mask_out && d > 0.0f) {
          const int g = off + i;
          atomicOr(&io.mask_out[(int64_t)e * words + (g >> 5)], 1u << (g & 31));
        }
        if (write_uhat) {
          const float4 nn = m.nrm4[off + i];
          __nv_bfloat16* u = m.uhat_t + (int64_t)(slot * 3) * m.ldu + uoff + i;
          u[0] = __float2bfloat16_rn(-d * nn.x);
          u[m.ldu] = __float2bfloat16_rn(-d * nn.y);
          u[2 * (int64_t)m.ldu] = __float2bfloat16_rn(-d * nn.z);
          const int kb = i >> 6;
          if (d > 0.0f && kb < 32 * kKbWords) atomicOr(&s_kb[kb >> 5], 1u << (kb & 31));
        }
      }
      if (write_uhat) {
        __syncthreads();
        if (threadIdx.x < kKbWords) m.kbmap[((int64_t)(p0 + q) * m.max_envs + slot) * kKbWords + threadIdx.x] = s_kb[threadIdx.x];
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// S1 for meshes of many small patches with SEVERAL indenter slots per environment (self-contact: the other
// links' shapes): one WARP per (env, patch) pair.  All lanes build the patch rotation and do the conservative
// bounding-sphere cull against the environment's indenters (warp-uniform, no divergence; the indenters are
// staged per warp in shared memory); a culled warp exits at once.  Otherwise the warp evaluates the nodes ->
// phi, delta (workspace), warp vote -> contact flag; on contact lane 0 takes a slot in the patch's compact
// environment list and the warp writes the U^ operand rows.  No block barrier.  (One slot per environment:
// sdf_cull_kernel / sdf_eval_kernel below.)
// Same single-rounded arithmetic in the same order as sdf_penetration_kernel.
constexpr int kPairWarps = 2;

template <bool kGrid>
__global__ void __launch_bounds__(kPairWarps * 32, 24) sdf_pairs_kernel(DevModel m, StepIO io, int s1_flags) {
  const bool write_uhat = s1_flags & kS1WriteUhat, write_alist = s1_flags & kS1WriteAlist, fill_out = s1_flags & kS1FillOut;
  extern __shared__ uint8_t smem_raw[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  SInd* sind = reinterpret_cast<SInd*>(smem_raw) + (size_t)wib * m.max_ind;  // per-warp staging
  const int P = m.n_patches;
  const int64_t pair = (int64_t)blockIdx.x * kPairWarps + wib;
  if (pair >= (int64_t)io.n_envs * P) return;
  const int e = (int)(pair / P), p = (int)(pair - (int64_t)e * P);
  const bool posed = io.patch_pose != nullptr;
  const PatchInfo pi = m.patch[p];
  const int off = pi.off, n = pi.n;
  const int64_t row0 = (int64_t)e * m.n_nodes + off;

  float R[9] = {1.f, 0.f, 0.f, 0.f, 1.f, 0.f, 0.f, 0.f, 1.f}, t[3] = {0.f, 0.f, 0.f};
  float C0 = pi.bc[0], C1 = pi.bc[1], C2 = pi.bc[2];
  if (posed) {
    const float* pp = io.patch_pose + pair * 7;
    const float q[4] = {pp[3], pp[4], pp[5], pp[6]};
    t[0] = pp[0], t[1] = pp[1], t[2] = pp[2];
    quat_to_rot(q, R);
    to_world(R, t, pi.bc[0], pi.bc[1], pi.bc[2], C0, C1, C2);
  }
  for (int k = lane; k < m.max_ind; k += 32) sind[k] = load_indenter(io.ind + (int64_t)e * m.max_ind + k);
  __syncwarp();
  const float phi_lo = union_sdf_lower<kGrid>(sind, m.max_ind, C0, C1, C2, pi.brad, m.grid, p + 1);
  // conservative cull: phi(x_i) >= phi(c) - L * brad on the patch's bounding sphere
  // (phi_lo = +inf: no indenter applies to this patch -- all slots NONE, or only the patch's own link)
  const bool evaluated = phi_lo < __int_as_float(0x7f800000) && !(phi_lo > 0.01f + 1e-5f * (fabsf(phi_lo) + 3.0f * pi.brad));
  bool any = false;
  int nact = 0;
  float* delta = m.delta + row0;
  if (evaluated) {
#pragma unroll 2
    for (int i = lane; i < n; i += 32) {
      const float4 pos = m.pos4[off + i];
      float X0 = pos.x, X1 = pos.y, X2 = pos.z;
      if (posed) to_world(R, t, pos.x, pos.y, pos.z, X0, X1, X2);
      const float phi = union_sdf<kGrid>(sind, m.max_ind, X0, X1, X2, m.grid, p + 1);
      const float d = phi < 0.0f ? -phi : 0.0f;
      delta[i] = d;
      any |= d > 0.0f;
      nact += d > 0.0f;
    }
    any = __any_sync(0xffffffffu, any);
  }
  if (io.nact_out && any) {
    nact = __reduce_add_sync(0xffffffffu, nact);
    if (lane == 0) atomicAdd(&io.nact_out[e], nact);
  }
  int slot = 0;
  if (lane == 0) {
    m.flags[pair] = (uint8_t)any;
    if (io.contact_out) io.contact_out[pair] = (uint8_t)any;
    if (any) {
      slot = atomicAdd(&m.count[p], 1);
      m.envlist[(int64_t)p * m.max_envs + slot] = e;
    }
  }
  if (any) {
    slot = __shfl_sync(0xffffffffu, slot, 0);
    const int words = (m.n_nodes + 31) >> 5;
    if (write_alist) {  // compact list of the patch's active nodes, in node order
      ActiveEntry* al = m.alist + (int64_t)slot * m.ldu + off;
      int base = 0;
      for (int i0 = 0; i0 < n; i0 += 32) {
        const int i = i0 + lane;
        const float d = i < n ? delta[i] : 0.0f;
        const uint32_t bal = __ballot_sync(0xffffffffu, d > 0.0f);
        if (d > 0.0f) {
          const float4 nn = m.nrm4[off + i];
          ActiveEntry en;
          en.ux = -d * nn.x, en.uy = -d * nn.y, en.uz = -d * nn.z, en.j = i;
          al[base + __popc(bal & ((1u << lane) - 1u))] = en;
        }
        base += __popc(bal);
      }
      if (lane == 0) m.acount[(int64_t)p * m.max_envs + slot] = base;
    }
    uint32_t kb0 = 0;  // bitmap of the 64-node k-blocks with an active node (n <= 2048: one word)
#pragma unroll 2
    for (int i = lane; i < n; i += 32) {
      const float d = delta[i];  // written by this thread above
      if (io.pen_out) io.pen_out[row0 + i] = d;
      if (io.mask_out && d > 0.0f) {
        const int g = off + i;
        atomicOr(&io.mask_out[(int64_t)e * words + (g >> 5)], 1u << (g & 31));
      }
      if (write_uhat) {
        const float4 nn = m.nrm4[off + i];
        __nv_bfloat16* u = m.uhat_t + (int64_t)(slot * 3) * m.ldu + pi.uoff + i;
        u[0] = __float2bfloat16_rn(-d * nn.x);
        u[m.ldu] = __float2bfloat16_rn(-d * nn.y);
        u[2 * (int64_t)m.ldu] = __float2bfloat16_rn(-d * nn.z);
        if (d > 0.0f) kb0 |= 1u << ((i >> 6) & 31);
      }
    }
    if (write_uhat) {
      kb0 = __reduce_or_sync(0xffffffffu, kb0);
      if (lane < kKbWords) m.kbmap[((int64_t)p * m.max_envs + slot) * kKbWords + lane] = lane == 0 ? kb0 : 0u;
    }
  } else {
    // contact-free pair: optional outputs are zero; for the fp32 gather kernel the output rows too
    // (the tensor-core kernel zero-fills them itself)
    if (fill_out) {
      zero_out_rows(io, e, off, n, lane, 32);
      if (io.analytic_out)
        for (int i = lane; i < n * 3; i += 32) io.analytic_out[row0 * 3 + i] = 0.0f;
    }
    if (io.pen_out)
      for (int i = lane; i < n; i += 32) io.pen_out[row0 + i] = 0.0f;
  }
}

// ---------------------------------------------------------------------------------------------
// S1 for meshes of many small patches with ONE indenter slot per environment (the dexterous hand of
// BASELINE.json configs[2]), as two kernels:
//   sdf_cull_kernel  one THREAD per (env, patch) pair: pose -> rotation, indenter -> rotation, conservative
//                    bounding-sphere cull.  Two thirds of the pairs of the hand workload end here after ~200
//                    instructions of one thread (in sdf_pairs_kernel every lane of a warp repeats them, 28 % of
//                    that kernel's instructions).  Survivors are appended, with their rotations, to a task list.
//   sdf_eval_kernel  one WARP per task: nodes -> phi, delta (workspace), warp vote -> contact flag, slot in the
//                    patch's compact environment list, then the U^ operand rows / active list / optional outputs.
//                    The grid is sized for the worst case (every pair a task); warps beyond the list exit at once.
// Same single-rounded arithmetic in the same order as the other S1 kernels.
constexpr int kCullThreads = 128, kEvalWarps = 4;

template <bool kGrid>
__global__ void __launch_bounds__(kCullThreads) sdf_cull_kernel(DevModel m, StepIO io, int s1_flags) {
  const bool fill_out = s1_flags & kS1FillOut;
  const int lane = threadIdx.x & 31;
  const int P = m.n_patches;
  const int64_t n_pairs = (int64_t)io.n_envs * P;
  const bool posed = io.patch_pose != nullptr;
  // a culled pair needs a warp only if rows have to be zero-filled for it
  const bool culled_needs_warp = fill_out || io.pen_out != nullptr;
  const int64_t pair = (int64_t)blockIdx.x * kCullThreads + threadIdx.x;
  bool task = false;
  PairTask tk;
  if (pair < n_pairs) {
    const int e = (int)(pair / P), p = (int)(pair - (int64_t)e * P);
    const PatchInfo pi = m.patch[p];
    tk.R[0] = tk.R[4] = tk.R[8] = 1.f, tk.R[1] = tk.R[2] = tk.R[3] = tk.R[5] = tk.R[6] = tk.R[7] = 0.f;
    tk.t[0] = tk.t[1] = tk.t[2] = 0.f;
    float C0 = pi.bc[0], C1 = pi.bc[1], C2 = pi.bc[2];
    if (posed) {
      const float* pp = io.patch_pose + pair * 7;
      const float q[4] = {pp[3], pp[4], pp[5], pp[6]};
      tk.t[0] = pp[0], tk.t[1] = pp[1], tk.t[2] = pp[2];
      quat_to_rot(q, tk.R);
      to_world(tk.R, tk.t, pi.bc[0], pi.bc[1], pi.bc[2], C0, C1, C2);
    }
    tk.ind = load_indenter(io.ind + e);
    if (tk.ind.skip1 == p + 1) tk.ind.type = ETAC_IND_NONE;  // the shape of this patch's own link
    const float phi_lo = union_sdf_lower<kGrid>(&tk.ind, 1, C0, C1, C2, pi.brad, m.grid, p + 1);
    // conservative cull: phi(x_i) >= phi(c) - L * brad on the patch's bounding sphere
    // (phi_lo = +inf: no indenter applies to this patch)
    tk.evaluated = phi_lo < __int_as_float(0x7f800000) && !(phi_lo > 0.01f + 1e-5f * (fabsf(phi_lo) + 3.0f * pi.brad));
    tk.pair = (int)pair;
    task = tk.evaluated || culled_needs_warp;
    if (!task) {
      m.flags[pair] = 0;
      if (io.contact_out) io.contact_out[pair] = 0;
    }
  }
  const uint32_t bal = __ballot_sync(0xffffffffu, task);
  int base = 0;
  if (lane == 0 && bal) base = atomicAdd(m.ntask, __popc(bal));
  base = __shfl_sync(0xffffffffu, base, 0);
  if (task) m.tasks[base + __popc(bal & ((1u << lane) - 1u))] = tk;
}

template <bool kGrid>
__global__ void __launch_bounds__(kEvalWarps * 32, 8) sdf_eval_kernel(DevModel m, StepIO io, int s1_flags) {
  const bool write_uhat = s1_flags & kS1WriteUhat, write_alist = s1_flags & kS1WriteAlist, fill_out = s1_flags & kS1FillOut;
  const int lane = threadIdx.x & 31;
  const int k = blockIdx.x * kEvalWarps + (threadIdx.x >> 5);
  if (k >= *m.ntask) return;
  const int P = m.n_patches;
  const bool posed = io.patch_pose != nullptr;
  const PairTask* __restrict__ tk = m.tasks + k;  // every lane reads the same words: broadcast loads
  const int64_t pair = tk->pair;
  const int e = (int)(pair / P), p = (int)(pair - (int64_t)e * P);
  const PatchInfo pi = m.patch[p];
  const int off = pi.off, n = pi.n;
  const int64_t row0 = (int64_t)e * m.n_nodes + off;
  float* delta = m.delta + row0;
  bool any = false;
  int nact = 0;
  if (tk->evaluated) {
    float R[9], t[3];
#pragma unroll
    for (int a = 0; a < 9; ++a) R[a] = tk->R[a];
    t[0] = tk->t[0], t[1] = tk->t[1], t[2] = tk->t[2];
    const SInd one = tk->ind;
#pragma unroll 2
    for (int i = lane; i < n; i += 32) {
      const float4 pos = m.pos4[off + i];
      float X0 = pos.x, X1 = pos.y, X2 = pos.z;
      if (posed) to_world(R, t, pos.x, pos.y, pos.z, X0, X1, X2);
      const float phi = fminf(__int_as_float(0x7f800000), sdf_one<kGrid>(one, X0, X1, X2, m.grid));
      const float d = phi < 0.0f ? -phi : 0.0f;
      delta[i] = d;
      any |= d > 0.0f;
      nact += d > 0.0f;
    }
    any = __any_sync(0xffffffffu, any);
  }
  if (io.nact_out && any) {
    nact = __reduce_add_sync(0xffffffffu, nact);
    if (lane == 0) atomicAdd(&io.nact_out[e], nact);
  }
  int slot = 0;
  if (lane == 0) {
    m.flags[pair] = (uint8_t)any;
    if (io.contact_out) io.contact_out[pair] = (uint8_t)any;
    if (any) {
      slot = atomicAdd(&m.count[p], 1);
      m.envlist[(int64_t)p * m.max_envs + slot] = e;
    }
  }
  if (any) {
    slot = __shfl_sync(0xffffffffu, slot, 0);
    const int words = (m.n_nodes + 31) >> 5;
    if (write_alist) {  // compact list of the patch's active nodes, in node order
      ActiveEntry* al = m.alist + (int64_t)slot * m.ldu + off;
      int base = 0;
      for (int i0 = 0; i0 < n; i0 += 32) {
        const int i = i0 + lane;
        const float d = i < n ? delta[i] : 0.0f;
        const uint32_t bal = __ballot_sync(0xffffffffu, d > 0.0f);
        if (d > 0.0f) {
          const float4 nn = m.nrm4[off + i];
          ActiveEntry en;
          en.ux = -d * nn.x, en.uy = -d * nn.y, en.uz = -d * nn.z, en.j = i;
          al[base + __popc(bal & ((1u << lane) - 1u))] = en;
        }
        base += __popc(bal);
      }
      if (lane == 0) m.acount[(int64_t)p * m.max_envs + slot] = base;
    }
    // second sweep: the U^ operand rows (bf16, all n columns: the rows are reused from step to step) and the
    // optional outputs.  A lane takes EIGHT consecutive nodes: delta comes back from L2 as two 16-byte loads
    // (written by this warp above), a group without an active node -- most of them: a tenth of the nodes of a
    // contacting patch is active -- costs three 16-byte zero stores, and normals are only loaded for active nodes.
    __nv_bfloat16* u0 = m.uhat_t + (int64_t)(slot * 3) * m.ldu + pi.uoff;
    const bool vec = (row0 & 3) == 0;  // 16-byte aligned groups (else node by node)
    __syncwarp();  // the lanes read delta values that other lanes of the warp wrote
    uint32_t kb0 = 0;  // bitmap of the 64-node k-blocks with an active node (n <= 2048: one word)
    if (write_uhat && vec) {
      for (int i0 = lane * 8; i0 < n; i0 += 256) {
        if (i0 + 8 > n) {  // ragged last group: node by node
          for (int i = i0; i < n; ++i) {
            const float dd = delta[i];
            const float4 nn = m.nrm4[off + i];
            u0[i] = __float2bfloat16_rn(-dd * nn.x);
            u0[m.ldu + i] = __float2bfloat16_rn(-dd * nn.y);
            u0[2 * (int64_t)m.ldu + i] = __float2bfloat16_rn(-dd * nn.z);
            if (dd > 0.0f) kb0 |= 1u << ((i >> 6) & 31);
          }
          continue;
        }
        const float4 da = *reinterpret_cast<const float4*>(delta + i0), db = *reinterpret_cast<const float4*>(delta + i0 + 4);
        const float d[8] = {da.x, da.y, da.z, da.w, db.x, db.y, db.z, db.w};
        uint32_t w[3][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
        bool some = false;
#pragma unroll
        for (int c = 0; c < 8; ++c) some |= d[c] > 0.0f;
        if (some) {
          kb0 |= 1u << ((i0 >> 6) & 31);
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            if (d[c] > 0.0f) {
              const float4 nn = m.nrm4[off + i0 + c];
              const uint32_t sh = (c & 1) * 16;
              w[0][c >> 1] |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(-d[c] * nn.x)) << sh;
              w[1][c >> 1] |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(-d[c] * nn.y)) << sh;
              w[2][c >> 1] |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(-d[c] * nn.z)) << sh;
            }
          }
        }
        // (columns past the patch end belong to the padding / the next patch's columns of this slot row, which
        //  only that patch's own contacting environments ever write: whole groups inside the patch only)
#pragma unroll
        for (int c = 0; c < 3; ++c)
          *reinterpret_cast<uint4*>(u0 + (int64_t)c * m.ldu + i0) = make_uint4(w[c][0], w[c][1], w[c][2], w[c][3]);
      }
    }
    if ((write_uhat && !vec) || io.pen_out || io.mask_out) {
      for (int i = lane; i < n; i += 32) {
        const float d = delta[i];
        if (io.pen_out) io.pen_out[row0 + i] = d;
        if (io.mask_out && d > 0.0f) {
          const int g = off + i;
          atomicOr(&io.mask_out[(int64_t)e * words + (g >> 5)], 1u << (g & 31));
        }
        if (write_uhat && !vec) {
          const float4 nn = m.nrm4[off + i];
          u0[i] = __float2bfloat16_rn(-d * nn.x);
          u0[m.ldu + i] = __float2bfloat16_rn(-d * nn.y);
          u0[2 * (int64_t)m.ldu + i] = __float2bfloat16_rn(-d * nn.z);
          if (d > 0.0f) kb0 |= 1u << ((i >> 6) & 31);
        }
      }
    }
    if (write_uhat) {
      kb0 = __reduce_or_sync(0xffffffffu, kb0);
      if (lane < kKbWords) m.kbmap[((int64_t)p * m.max_envs + slot) * kKbWords + lane] = lane == 0 ? kb0 : 0u;
    }
  } else {
    // contact-free pair: optional outputs are zero; for the fp32 gather kernel the output rows too
    // (the tensor-core kernel zero-fills them itself)
    if (fill_out) {
      zero_out_rows(io, e, off, n, lane, 32);
      if (io.analytic_out)
        for (int i = lane; i < n * 3; i += 32) io.analytic_out[row0 * 3 + i] = 0.0f;
    }
    if (io.pen_out)
      for (int i = lane; i < n; i += 32) io.pen_out[row0 + i] = 0.0f;
  }
}

// Second half of S1 with bucketing (kS1Bucket, large patches): one CTA per environment.  The slot of a contacting
// (env, patch) in the patch's environment list is its position in the counting sort by key (position of the first
// active node): environments of one tile of the contraction then share most of their active k-blocks, and the
// others are skipped (k_fused.cu).  Writes the list entry, the U^ operand rows and the k-block bitmap from delta.
__global__ void __launch_bounds__(256) sdf_scatter_kernel(DevModel m, StepIO io) {
  __shared__ int s_part[2][8];
  __shared__ int s_slot;
  __shared__ uint32_t s_kb[kKbWords];
  const int e = blockIdx.x, t = threadIdx.x, lane = t & 31;
  for (int p = 0; p < m.n_patches; ++p) {
    if (!m.flags[(int64_t)e * m.n_patches + p]) continue;  // (uniform over the CTA)
    const int key = m.keybuf[(int64_t)e * m.n_patches + p];
    const int h = m.khist[p * 256 + t];
    int below = __reduce_add_sync(0xffffffffu, t < key ? h : 0), total = __reduce_add_sync(0xffffffffu, h);
    __syncthreads();  // previous patch done with the shared words
    if (lane == 0) s_part[0][t >> 5] = below, s_part[1][t >> 5] = total;
    if (t < kKbWords) s_kb[t] = 0;
    __syncthreads();
    if (t == 0) {
      below = 0, total = 0;
      for (int w = 0; w < 8; ++w) below += s_part[0][w], total += s_part[1][w];
      const int slot = below + atomicAdd(&m.kcursor[p * 256 + key], 1);
      m.envlist[(int64_t)p * m.max_envs + slot] = e;
      m.count[p] = total;  // (every contacting environment writes the same value)
      s_slot = slot;
    }
    __syncthreads();
    const int slot = s_slot;
    const PatchInfo pi = m.patch[p];
    const int off = pi.off, n = pi.n;
    const int64_t row0 = (int64_t)e * m.n_nodes + off;
    const float* __restrict__ delta = m.delta + row0;
    __nv_bfloat16* u0 = m.uhat_t + (int64_t)(slot * 3) * m.ldu + pi.uoff;
    const bool vec = (row0 & 3) == 0;  // 16-byte aligned groups of eight nodes
    if (vec) {
      for (int i0 = t * 8; i0 < n; i0 += 2048) {
        float d[8];
        if (i0 + 8 <= n) {
          const float4 a = *reinterpret_cast<const float4*>(delta + i0), b = *reinterpret_cast<const float4*>(delta + i0 + 4);
          d[0] = a.x, d[1] = a.y, d[2] = a.z, d[3] = a.w, d[4] = b.x, d[5] = b.y, d[6] = b.z, d[7] = b.w;
        } else {
#pragma unroll
          for (int c = 0; c < 8; ++c) d[c] = i0 + c < n ? delta[i0 + c] : 0.0f;
        }
        uint32_t w[3][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
        bool some = false;
#pragma unroll
        for (int c = 0; c < 8; ++c) some |= d[c] > 0.0f;
        if (some) {
          const int kb = i0 >> 6;
          if (kb < 32 * kKbWords) atomicOr(&s_kb[kb >> 5], 1u << (kb & 31));
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            if (d[c] > 0.0f) {
              const float4 nn = m.nrm4[off + i0 + c];
              const uint32_t sh = (c & 1) * 16;
              w[0][c >> 1] |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(-d[c] * nn.x)) << sh;
              w[1][c >> 1] |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(-d[c] * nn.y)) << sh;
              w[2][c >> 1] |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(-d[c] * nn.z)) << sh;
            }
          }
        }
        if (i0 + 8 <= n) {
#pragma unroll
          for (int c = 0; c < 3; ++c)
            *reinterpret_cast<uint4*>(u0 + (int64_t)c * m.ldu + i0) = make_uint4(w[c][0], w[c][1], w[c][2], w[c][3]);
        } else {
          for (int c = 0; i0 + c < n; ++c)
            for (int a = 0; a < 3; ++a)
              u0[(int64_t)a * m.ldu + i0 + c] = __ushort_as_bfloat16((unsigned short)(w[a][c >> 1] >> ((c & 1) * 16)));
        }
      }
    } else {
      for (int i = t; i < n; i += 256) {
        const float d = delta[i];
        const float4 nn = m.nrm4[off + i];
        u0[i] = __float2bfloat16_rn(-d * nn.x);
        u0[m.ldu + i] = __float2bfloat16_rn(-d * nn.y);
        u0[2 * (int64_t)m.ldu + i] = __float2bfloat16_rn(-d * nn.z);
        const int kb = i >> 6;
        if (d > 0.0f && kb < 32 * kKbWords) atomicOr(&s_kb[kb >> 5], 1u << (kb & 31));
      }
    }
    __syncthreads();
    if (t < kKbWords) m.kbmap[((int64_t)p * m.max_envs + slot) * kKbWords + t] = s_kb[t];
  }
}

// ETAC_ABLATE_NO_PROPAGATION: U = U^, the penalty displacement -delta * n of the nodes in contact and 0
// elsewhere (no K, no Phi).  Reads S1's delta (valid for the contacting pairs) and pair flags.
__global__ void __launch_bounds__(256) penalty_only_kernel(DevModel m, StepIO io) {
  const int e = blockIdx.x, p = blockIdx.y;
  const PatchInfo pi = m.patch[p];
  const bool hit = m.flags[(int64_t)e * m.n_patches + p] != 0;
  for (int i = blockIdx.z * 256 + threadIdx.x; i < pi.n; i += gridDim.z * 256) {
    const int g = pi.off + i;
    const float d = hit ? m.delta[(int64_t)e * m.n_nodes + g] : 0.0f;
    const float4 nn = m.nrm4[g];
    const bool act = d > 0.0f;
    store_out3(io, e, g, act ? -d * nn.x : 0.0f, act ? -d * nn.y : 0.0f, act ? -d * nn.z : 0.0f);
    if (io.analytic_out) {
      float* a = io.analytic_out + ((int64_t)e * m.n_nodes + g) * 3;
      a[0] = 0.0f, a[1] = 0.0f, a[2] = 0.0f;
    }
  }
}

cudaError_t launch_penalty_only(const DevModel& m, const StepIO& io, cudaStream_t s) {
  const dim3 grid(io.n_envs, m.n_patches, min(64, (m.max_patch_nodes + 255) / 256));
  penalty_only_kernel<<<grid, 256, 0, s>>>(m, io);
  return cudaGetLastError();
}

cudaError_t launch_sdf(const DevModel& m, const StepIO& io, int s1_flags_in, int* launches, cudaStream_t s) {
  int s1_flags = s1_flags_in;
  *launches = 1;
  const unsigned grid = (unsigned)io.n_envs;
  bool grids = false;  // the sampled-SDF code is only in the variants launched once a grid is registered
  for (int k = 0; k < kMaxGrids; ++k) grids |= m.grid[k].v != nullptr;
  // many small patches with indenters: one warp per (env, patch) pair; otherwise one CTA per environment
  if (io.input_mode == ETAC_IN_INDENTERS && m.max_ind >= 1 && m.n_patches >= 4 && m.max_patch_nodes <= 2048) {
    s1_flags &= ~kS1Bucket;  // (slots are taken in arrival order by the pair kernels)
    const int64_t pairs = (int64_t)io.n_envs * m.n_patches;
    const unsigned pgrid = (unsigned)((pairs + kPairWarps - 1) / kPairWarps);
    const size_t smem = m.max_ind == 1 ? 0 : sizeof(SInd) * (size_t)m.max_ind * kPairWarps;
    if (m.max_ind == 1) {  // cull by threads, evaluate by warps (m.ntask is zeroed with the other per-step counters)
      const unsigned gc = (unsigned)((pairs + kCullThreads - 1) / kCullThreads), ge = (unsigned)((pairs + kEvalWarps - 1) / kEvalWarps);
      if (grids) sdf_cull_kernel<true><<<gc, kCullThreads, 0, s>>>(m, io, s1_flags), sdf_eval_kernel<true><<<ge, kEvalWarps * 32, 0, s>>>(m, io, s1_flags);
      else sdf_cull_kernel<false><<<gc, kCullThreads, 0, s>>>(m, io, s1_flags), sdf_eval_kernel<false><<<ge, kEvalWarps * 32, 0, s>>>(m, io, s1_flags);
      *launches = 2;
      return cudaGetLastError();
    }
    if (m.max_ind != 1 && !grids) sdf_pairs_kernel<false><<<pgrid, kPairWarps * 32, smem, s>>>(m, io, s1_flags);
    if (m.max_ind != 1 && grids) sdf_pairs_kernel<true><<<pgrid, kPairWarps * 32, smem, s>>>(m, io, s1_flags);
    return cudaGetLastError();
  }
  if (s1_flags & kS1Bucket) {
    cudaError_t e = cudaMemsetAsync(m.khist, 0, sizeof(int32_t) * 512 * (size_t)m.n_patches, s);  // histogram + cursors
    if (e != cudaSuccess) return e;
  }
  if (io.input_mode == ETAC_IN_INDENTERS) {
    const size_t smem = (sizeof(SInd) + sizeof(float4)) * (size_t)(m.max_ind > 0 ? m.max_ind : 1) + 16;  // + (t, rb2) per slot, aligned
    if (grids) sdf_penetration_kernel<true, true><<<grid, 256, smem, s>>>(m, io, s1_flags);
    else sdf_penetration_kernel<true, false><<<grid, 256, smem, s>>>(m, io, s1_flags);
  } else {
    sdf_penetration_kernel<false, false><<<grid, 256, 0, s>>>(m, io, s1_flags);
  }
  if (s1_flags & kS1Bucket) {
    sdf_scatter_kernel<<<grid, 256, 0, s>>>(m, io);
    *launches = 2;
  }
  return cudaGetLastError();
}

}  // namespace etac

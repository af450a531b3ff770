// S2+S3+S4 fused, tensor-core path (sm_100a: TMA + tcgen05.mma + TMEM).
//
//   S2  u_lin = K_p . U^  as a dense bf16 contraction with fp32 accumulation in TMEM
//       ("propagation matrix Omega ... computed as Omega U_a"; the zero rows of the
//       zero-padded U^ contribute nothing, R3),
//   S3  residual MLP 9 -> 64 -> 64 -> 3 (SiLU) on the accumulator tile, each layer one small
//       tcgen05.mma whose A operand is written to TMEM by the epilogue warps and whose B operand
//       (the weights, biases folded in as an extra K column) stays in shared memory,
//   S4  mask M_p + combine (Eq. 2) and the store of U[e][i][0..2]; the rows of
//       contact-free (env, patch) pairs are zero-filled by the MLP issuer warps (R8).
//
// Work item = (patch p, block of 128 nodes, tile of TE contacting environments of that patch).
// The grid is persistent (2 CTAs per SM); every CTA walks items blockIdx.x, +gridDim.x, ...
// 12 warps: 0 = TMA producer, 1 = propagation-GEMM MMA issuer (+ TMEM alloc), 2..5 and 6..9 = two
// epilogue warpgroups (thread = node), 10/11 = MLP MMA issuers of slot 0/1.
//
// TWO environments are in flight per CTA (slots 0/1, each with its own TMEM D/A regions, mbarrier
// pair and epilogue warpgroup): while the tensor core runs a layer of slot 0, warpgroup 1
// evaluates the SiLUs of slot 1 and vice versa; with 2 CTAs per SM every SM sub-partition has 4
// epilogue warps to hide the MMA round trips and TMEM load latency behind the MUFU pipe.
//
// TMEM columns (fp32 lanes = nodes):   [0,48)   u_lin accumulator, column 3*env+c
//   slot s at 48 + 104*s:              [+0,+64)   D: pre-activations of the current MLP layer
//                                      [+64,+104) A: bf16 layer input; layer 1 uses words 0..7
//                                                 [u_lin(3), p(3), n(3), 1, 0..], layers 2/3 use
//                                                 64 activations + a ones column (word 32)
#include "etac_internal.h"
#include "sm100_prims.cuh"

namespace etac {

constexpr int BM = 128, BK = 64, TE = kDenseTE, BN = kDenseBN, STAGES = 4;
constexpr int A_STAGE = BM * BK * 2, B_STAGE = BN * BK * 2;
constexpr int kDenseThreads = 384;
constexpr uint32_t kTmemCols = 256;
constexpr uint32_t COL_ACC = 0, COL_SLOT0 = 48, SLOT_STRIDE = 104, OFF_A = 64;

struct __align__(8) DenseBars {
  uint64_t full[STAGES], empty[STAGES];
  uint64_t acc_full, acc_empty, a_ready[2], d_ready[2];
  uint32_t tmem_base;
  uint32_t pad;
};

__host__ __device__ constexpr size_t dense_smem_bytes(int n_patches) {
  return 1024 /*align slack*/ + (size_t)STAGES * (A_STAGE + B_STAGE) + kWImgBytes + sizeof(DenseBars) +
         (size_t)(n_patches + 1) * 4 + 16;
}

#ifdef ETAC_TRACE
// timing experiment only: per-warp event log in shared memory (no global traffic while running)
__device__ unsigned long long g_trace[12 * 400];
__device__ unsigned int g_trace_n;
__shared__ unsigned long long s_trace[12 * 400];
__shared__ unsigned int s_trace_n[12];
#define TR(tag)                                                                       \
  do {                                                                                \
    if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) {                                 \
      unsigned int w_ = threadIdx.x >> 5, i_ = s_trace_n[w_];                         \
      if (i_ < 400) s_trace[w_ * 400 + i_] = ((unsigned long long)(tag) << 48) | ((unsigned long long)w_ << 40) | (clock64() & 0xFFFFFFFFFFull), s_trace_n[w_] = i_ + 1; \
    }                                                                                 \
  } while (0)
#else
#define TR(tag)
#endif

struct Item {
  int p, mb, tile, cnt;
};

// streaming zero-fill of `count` floats at a 4-byte aligned address by one warp
__device__ __forceinline__ void warp_zero_fill(float* __restrict__ p, int count, int lane) {
  const int head = min(count, (int)(((16u - (uint32_t)((uintptr_t)p & 15u)) & 15u) >> 2));
  if (lane < head) __stcs(p + lane, 0.0f);
  float4* body = reinterpret_cast<float4*>(p + head);
  const int nvec = (count - head) >> 2;
  for (int v = lane; v < nvec; v += 32) __stcs(body + v, make_float4(0.f, 0.f, 0.f, 0.f));
  const int tail0 = head + (nvec << 2);
  if (tail0 + lane < count) __stcs(p + tail0 + lane, 0.0f);
}

// Rows of (env, patch) pairs without contact are exactly 0 (R8).  Resumable sweep for one
// warp: warp `part` of `nparts` takes the pairs 32*part.., 32*(part+nparts)..; lane l looks at pair
// base+l; one step() zero-fills one run of consecutive contact-free patches of one environment,
// so that the sweep can be spread over the kernel instead of saturating HBM at its start.
struct ZeroFill {
  int64_t base, total, stride;
  uint32_t mask;
  __device__ __forceinline__ void init(const DevModel& m, const StepIO& io, int part, int nparts) {
    total = (int64_t)io.n_envs * m.n_patches, base = (int64_t)part * 32 - (int64_t)nparts * 32;
    stride = (int64_t)nparts * 32, mask = 0;
  }
  __device__ __forceinline__ bool step(const DevModel& m, const StepIO& io, int lane) {  // false: nothing left
    while (mask == 0) {
      base += stride;
      if (base >= total) return false;
      const int64_t idx = base + lane;
      mask = __ballot_sync(0xffffffffu, idx < total && m.flags[idx] == 0);
    }
    const int P = m.n_patches;
    const int b = __ffs(mask) - 1;
    const int64_t pair = base + b;
    const int e = (int)(pair / P), p = (int)(pair - (int64_t)e * P);
    int len = 1;
    while (b + len < 32 && p + len < P && ((mask >> (b + len)) & 1u)) ++len;
    mask &= ~(((len == 32) ? 0xffffffffu : ((1u << len) - 1u)) << b);
    const int off = m.patch[p].off;
    const int cnt = m.patch[p + len - 1].off + m.patch[p + len - 1].n - off;
    const int64_t r0 = ((int64_t)e * m.n_nodes + off) * 3;
    warp_zero_fill(io.out + r0, cnt * 3, lane);
    if (io.analytic_out) warp_zero_fill(io.analytic_out + r0, cnt * 3, lane);
    return true;
  }
};

__device__ __forceinline__ bool decode_item(const int* prefix, int n_patches, const DevModel& m, int w, int& pcur,
                                            Item& it) {
  if (w >= prefix[n_patches]) return false;
  while (prefix[pcur + 1] <= w) ++pcur;
  const int cnt = m.count[pcur];
  const int tiles = (cnt + TE - 1) / TE;
  const int r = w - prefix[pcur];
  it.p = pcur;
  it.mb = r / tiles;
  it.tile = r - it.mb * tiles;
  it.cnt = min(TE, cnt - it.tile * TE);
  return true;
}

template <bool kResid>
__global__ void __launch_bounds__(kDenseThreads, 2)
    dense_bf16_kernel(DevModel m, StepIO io, const __grid_constant__ CUtensorMap tmA,
                      const __grid_constant__ CUtensorMap tmB) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + STAGES * A_STAGE;
  uint8_t* sW = sB + STAGES * B_STAGE;
  DenseBars* bars = reinterpret_cast<DenseBars*>(sW + kWImgBytes);
  int* prefix = reinterpret_cast<int*>(bars + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#ifdef ETAC_TRACE
  if (threadIdx.x < 12) s_trace_n[threadIdx.x] = 0;
#endif

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) mbar_init(&bars->full[s], 1), mbar_init(&bars->empty[s], 1);
    mbar_init(&bars->acc_full, 1);
    mbar_init(&bars->acc_empty, 8);
    for (int s = 0; s < 2; ++s) mbar_init(&bars->a_ready[s], 4), mbar_init(&bars->d_ready[s], 1);
    fence_barrier_init();
    int acc = 0;
    prefix[0] = 0;
    for (int p = 0; p < m.n_patches; ++p) {
      const int cnt = m.count[p];
      acc += ((cnt + TE - 1) / TE) * ((m.patch[p].n + BM - 1) / BM);
      prefix[p + 1] = acc;
    }
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1) tmem_alloc<kTmemCols>(&bars->tmem_base);
  if constexpr (kResid) {
    const uint4* src = reinterpret_cast<const uint4*>(m.wimg);
    uint4* dst = reinterpret_cast<uint4*>(sW);
    for (int k = threadIdx.x; k < kWImgBytes / 16; k += kDenseThreads) dst[k] = src[k];
    fence_proxy_async_smem();  // generic-proxy writes -> visible to the tensor-core (async) proxy
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    // (the whole warp runs the loop so that every operand stays warp-uniform; one elected lane issues)
    {
      int pcur = 0, stage = 0;
      uint32_t ph = 0;
      Item it;
      for (int w = blockIdx.x; decode_item(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
        const PatchInfo pi = m.patch[it.p];
        const int nkb = (pi.n + BK - 1) / BK;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(&bars->empty[stage], ph ^ 1);
          if (elect_one()) {
            mbar_arrive_expect_tx(&bars->full[stage], A_STAGE + B_STAGE);
            tma_load_2d(sA + stage * A_STAGE, &tmA, &bars->full[stage], kb * BK, pi.off + it.mb * BM);
            tma_load_2d(sB + stage * B_STAGE, &tmB, &bars->full[stage], pi.off + kb * BK, it.tile * BN);
          }
          __syncwarp();
          if (++stage == STAGES) stage = 0, ph ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ MMA issuer
    // Warp-uniform control flow; tcgen05.mma / tcgen05.commit are issued by one elected lane.
    {
      constexpr uint32_t idesc_prop = make_idesc_bf16(BM, BN);
      constexpr uint32_t idesc_h = make_idesc_bf16(BM, 64);
      constexpr uint32_t idesc_o = make_idesc_bf16(BM, 16);
      const uint64_t dW1 = make_desc(smem_u32(sW), 1024, 128, kLayoutNone);
      const uint64_t dW2 = make_desc(smem_u32(sW + kW1ImgBytes), 1024, 128, kLayoutNone);
      const uint64_t dW3 = make_desc(smem_u32(sW + kW1ImgBytes + kW2ImgBytes), 256, 128, kLayoutNone);
      int pcur = 0, stage = 0;
      uint32_t ph = 0, acc_ph = 0, a_ph = 0;
      Item it;
      for (int w = blockIdx.x; decode_item(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
        const int nkb = (m.patch[it.p].n + BK - 1) / BK;
        mbar_wait(&bars->acc_empty, acc_ph ^ 1);
        acc_ph ^= 1;
        tc_fence_after();
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(&bars->full[stage], ph);
          tc_fence_after();
          const uint64_t dA = make_desc(smem_u32(sA + stage * A_STAGE), 16, 1024, kLayoutSw128);
          const uint64_t dB = make_desc(smem_u32(sB + stage * B_STAGE), 16, 1024, kLayoutSw128);
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < BK / 16; ++k)
              mma_ss(tmem + COL_ACC, dA + 2 * k, dB + 2 * k, idesc_prop, (kb | k) != 0);
            tc_commit(&bars->empty[stage]);
            if (kb == nkb - 1) tc_commit(&bars->acc_full);
          }
          __syncwarp();
          if (++stage == STAGES) stage = 0, ph ^= 1;
        }
      }
    }
  } else if (warp >= 10) {
    // ------------------------------------------------------------------ MLP MMA issuer of slot (warp - 10)
    // One dedicated issuer warp per slot: a tcgen05.mma round trip is ~450 cycles during which the
    // issuing warp makes no progress, so the two slots must not share an issuer.
    // Between requests the warp zero-fills its share of the output rows of contact-free (env, patch)
    // pairs, one run per request, so that these stores trickle out next to the MUFU-bound work.
    ZeroFill zf;
    zf.init(m, io, blockIdx.x * 2 + (warp - 10), gridDim.x * 2);
    if constexpr (kResid) {
      const int sl = warp - 10;
      constexpr uint32_t idesc_h = make_idesc_bf16(BM, 64);
      constexpr uint32_t idesc_o = make_idesc_bf16(BM, 16);
      const uint64_t dW1 = make_desc(smem_u32(sW), 1024, 128, kLayoutNone);
      const uint64_t dW2 = make_desc(smem_u32(sW + kW1ImgBytes), 1024, 128, kLayoutNone);
      const uint64_t dW3 = make_desc(smem_u32(sW + kW1ImgBytes + kW2ImgBytes), 256, 128, kLayoutNone);
      const uint32_t tD = tmem + COL_SLOT0 + SLOT_STRIDE * sl, tA = tD + OFF_A;
      uint64_t* a_ready = &bars->a_ready[sl];
      uint64_t* d_ready = &bars->d_ready[sl];
      int pcur = 0;
      uint32_t a_ph = 0;
      Item it;
      for (int w = blockIdx.x; decode_item(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
        for (int el = sl; el < it.cnt; el += 2) {
#pragma unroll 1
          for (int layer = 0; layer < 3; ++layer) {
            mbar_wait(a_ready, a_ph), a_ph ^= 1;
            TR(100 + sl * 10 + layer);
            tc_fence_after();
            if (elect_one()) {
#if defined(ETAC_ABLATE) && ETAC_ABLATE >= 4
              if (layer == 99) {
#else
              if (layer == 0) {
#endif
                mma_ts(tD, tA, dW1, idesc_h, 0);
#if defined(ETAC_ABLATE) && ETAC_ABLATE >= 4
              } else if (layer == 98) {
#else
              } else if (layer == 1) {
#endif
#pragma unroll
                for (int k = 0; k < 5; ++k) mma_ts(tD, tA + 8 * k, dW2 + (uint64_t)(k * (2048 >> 4)), idesc_h, k != 0);
#if defined(ETAC_ABLATE) && ETAC_ABLATE >= 4
              } else if (layer == 97) {
#else
              } else {
#endif
#pragma unroll
                for (int k = 0; k < 5; ++k) mma_ts(tD, tA + 8 * k, dW3 + (uint64_t)(k * (512 >> 4)), idesc_o, k != 0);
              }
              tc_commit(d_ready);
            }
            __syncwarp();
            TR(200 + sl * 10 + layer);
            zf.step(m, io, lane);
          }
        }
      }
    }
    while (zf.step(m, io, lane)) {
    }
  } else {
    // ------------------------------------------------------------------ epilogue (thread = node)
    // Two warpgroups; warpgroup s owns TMEM slot s and takes the environments el = s, s+2, ...
    const int sl = (warp - 2) >> 2;
    const uint32_t lane_base = (uint32_t)(warp & 3) * 32;
    const uint32_t trow = tmem + (lane_base << 16);
    const uint32_t tD = trow + COL_SLOT0 + SLOT_STRIDE * sl, tA = tD + OFF_A;
    const int row = lane_base + lane;
    uint64_t* a_ready = &bars->a_ready[sl];
    uint64_t* d_ready = &bars->d_ready[sl];
    if constexpr (kResid) {
      // bias ("ones") column of the layer-2/3 input: bf16 element 64 = 1.0, 65..79 = 0; written once
      const uint32_t ones[8] = {0x00003F80u, 0, 0, 0, 0, 0, 0, 0};
      tmem_st8(tA + 32, ones);
      tc_wait_st();
    }
    int pcur = 0;
    uint32_t acc_ph = 0, d_ph = 0;
    Item it;
    for (int w = blockIdx.x; decode_item(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
      const PatchInfo pi = m.patch[it.p];
      const int li = it.mb * BM + row;
      const bool valid = li < pi.n;
      const int g = pi.off + (valid ? li : 0);
      const float4 nrm = m.nrm4[g];
      uint32_t a1[8] = {0, 0, 0, 0, 0, 0, 0, 0};
      float px = 0.f;
      if constexpr (kResid) {
        const float4 pos = m.pos4[g];
        px = pos.x;
        a1[2] = pack_bf16(pos.y, pos.z);
        a1[3] = pack_bf16(nrm.x, nrm.y);
        a1[4] = pack_bf16(nrm.z, 1.0f);
      }
      // lane l prefetches the id of the item's l-th environment (broadcast by shuffle below)
      const int my_env = lane < it.cnt ? m.envlist[(int64_t)it.p * m.max_envs + it.tile * TE + lane] : 0;
      mbar_wait(&bars->acc_full, acc_ph), acc_ph ^= 1;
      tc_fence_after();
#ifdef ETAC_SKEW
      // De-phase the two warpgroups: both leave the accumulator barrier together and would then
      // alternate "both on the MUFU pipe" / "both waiting for the tensor core" in lock-step.
      if (sl == 1) {
        const long long t0 = clock64();
        while (clock64() - t0 < ETAC_SKEW) {
        }
      }
#endif
      for (int el = sl; el < it.cnt; el += 2) {
#if defined(ETAC_ABLATE) && ETAC_ABLATE >= 3
        const int env = it.tile * TE + el;
        const int64_t node = (int64_t)env * m.n_nodes + g;
        const float dl = 0.0f;
#else
        const int env = __shfl_sync(0xffffffffu, my_env, el);
        const int64_t node = (int64_t)env * m.n_nodes + g;
        const float dl = valid ? m.delta[node] : 0.0f;
#endif
        uint32_t ur[4];
        tmem_ld4(trow + COL_ACC + 3 * el, ur);
        tc_wait_ld();
        const float ux = __uint_as_float(ur[0]), uy = __uint_as_float(ur[1]), uz = __uint_as_float(ur[2]);
        float ox = ux, oy = uy, oz = uz;
        if constexpr (kResid) {
          a1[0] = pack_bf16(ux, uy);
          a1[1] = pack_bf16(uz, px);
          tmem_st8(tA, a1);
          tc_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(a_ready);
          TR(1);
#pragma unroll 1
          for (int layer = 0; layer < 2; ++layer) {
            mbar_wait(d_ready, d_ph), d_ph ^= 1;
            TR(2 + layer * 2);
            tc_fence_after();
            uint32_t h[32], packed[16];
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              tmem_ld32(tD + 32 * half, h);
              tc_wait_ld();
#pragma unroll
              for (int k = 0; k < 16; ++k) {
                // D holds x/2 (0.5 folded into the weights): silu(x) = x*sigmoid(x) = h + h*tanh(h)
                const float h0 = __uint_as_float(h[2 * k]), h1 = __uint_as_float(h[2 * k + 1]);
                packed[k] = pack_bf16(fmaf(h0, tanh_approx(h0), h0), fmaf(h1, tanh_approx(h1), h1));
              }
              tmem_st16(tA + 16 * half, packed);
            }
            tc_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(a_ready);
            TR(3 + layer * 2);
          }
          mbar_wait(d_ready, d_ph), d_ph ^= 1;
          TR(6);
          tc_fence_after();
          uint32_t rr[4];
          tmem_ld4(tD, rr);
          tc_wait_ld();
          ox += __uint_as_float(rr[0]), oy += __uint_as_float(rr[1]), oz += __uint_as_float(rr[2]);
        }
#if defined(ETAC_ABLATE) && ETAC_ABLATE >= 2
        if (valid && ox == 123.456f) {
#else
        if (valid) {
#endif
          if (dl > 0.0f && m.active_mode == ETAC_ACTIVE_PASSTHROUGH) ox = -dl * nrm.x, oy = -dl * nrm.y, oz = -dl * nrm.z;
          float* o = io.out + node * 3;
          o[0] = ox, o[1] = oy, o[2] = oz;
          if (io.analytic_out) {
            float* a = io.analytic_out + node * 3;
            a[0] = ux, a[1] = uy, a[2] = uz;
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->acc_empty);
    }
  }
  tc_fence_before();
  __syncthreads();
#ifdef ETAC_TRACE
  if (blockIdx.x == 0) {
    for (int k = threadIdx.x; k < 4800; k += blockDim.x) g_trace[k] = (k % 400) < s_trace_n[k / 400] ? s_trace[k] : 0ull;
    g_trace_n = 4800;
  }
#endif
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<kTmemCols>(tmem);
  }
}

cudaError_t dense_bf16_configure() {
  const int bytes = (int)dense_smem_bytes(kMaxPatches);
  cudaError_t e = cudaFuncSetAttribute(dense_bf16_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(dense_bf16_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

cudaError_t launch_dense_bf16(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB,
                              int n_sm, cudaStream_t s) {
  const size_t smem = dense_smem_bytes(m.n_patches);
  const int grid = 2 * n_sm;
  if (m.resid != ETAC_RESID_NONE)
    dense_bf16_kernel<true><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
  else
    dense_bf16_kernel<false><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
  return cudaGetLastError();
}

}  // namespace etac

#ifdef ETAC_TRACE
extern "C" void etac_debug_trace(unsigned long long* out, unsigned int* n) {
  cudaMemcpyFromSymbol(out, etac::g_trace, sizeof(unsigned long long) * 4800);
  cudaMemcpyFromSymbol(n, etac::g_trace_n, sizeof(unsigned int));
}
#endif

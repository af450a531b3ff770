// S2+S3+S4 fused, tensor-core path (sm_100a: TMA + tcgen05.mma + TMEM).
//
//   S2  u_lin = K_p . U^  as a dense bf16 contraction with fp32 accumulation in TMEM
//       ("propagation matrix Omega ... computed as Omega U_a"; the zero rows of the
//       zero-padded U^ contribute nothing, R3),
//   S3  residual MLP 9 -> 64 -> 64 -> 3 (SiLU) on the accumulator tile: the two hidden layers are
//       small tcgen05.mma's whose A operand is written to TMEM by the epilogue warps and whose B
//       operand (the weights, biases folded in as an extra K column) stays in shared memory; the
//       3 x 64 output layer is applied in fp32 by the epilogue to the SiLU outputs it holds in
//       registers (packed fma.rn.f32x2), which saves a tensor-core round trip per unit,
//   S4  mask M_p + combine (Eq. 2) and the store of U[e][i][0..2]; the rows of
//       contact-free (env, patch) pairs are zero-filled by the MLP issuer warps (R8).
//
// Work item = (patch p, block of 128 nodes, tile of TE contacting environments of that patch).
// The grid is persistent (2 CTAs per SM); every CTA walks items blockIdx.x, +gridDim.x, ...
// 12 warps: 0 = TMA producer, 1 = propagation-GEMM MMA issuer (+ TMEM alloc), 2/3 = MLP MMA issuers
// of slot 0/1, 4..7 and 8..11 = two epilogue warpgroups (thread = node).  setmaxnreg gives the
// epilogue warps 96 registers and the others 48.
//
// TWO environments are in flight per CTA (slots 0/1, each with its own TMEM D/A regions, mbarrier
// pair and epilogue warpgroup): while the tensor core runs a layer of slot 0, warpgroup 1
// evaluates the SiLUs of slot 1 and vice versa; with 2 CTAs per SM every SM sub-partition has 4
// epilogue warps to hide the MMA round trips and TMEM load latency behind the MUFU pipe.
//
// Within a slot the units of an item are software-pipelined (the next unit's u_lin is fetched behind
// the last layer's round trip, its layer-1 operand is requested before the current unit is stored)
// and the accumulator is released one unit before the item ends.
//
// Template variants (one source, see kMode / kGather below): per-node MLP or none; the PointNet form
// of Phi as an encoder pass with max-pool and a decoder pass; and the gather form of the propagation
// (Omega U_a over the active-node lists) instead of the dense contraction.
//
// TMEM columns (fp32 lanes = nodes):   [0,48)   u_lin accumulator, column 3*env+c
//   slot s at 48 + 104*s:              [+0,+64)   D: pre-activations of the current MLP layer
//                                      [+64,+104) A: bf16 layer input; layer 1 uses words 0..7
//                                                 [u_lin(3), p(3), n(3), 1, 0..], the K = 80 layers
//                                                 use 64 activations + a ones column (word 32)
#include "etac_internal.h"
#include "sm100_prims.cuh"

namespace etac {

constexpr int BM = 128, BK = 64, TE = kDenseTE, BN = kDenseBN, STAGES = 4;  // STAGES: upper bound (barrier arrays)
constexpr int A_STAGE = BM * BK * 2, B_STAGE = BN * BK * 2;
constexpr int kDenseThreads = 384;
// setmaxnreg moves registers inside the CTA's launch-time allocation: 12 warps x 80 registers
constexpr int kRegsCtrl = 48, kRegsEpi = 96;
static_assert(4 * kRegsCtrl + 8 * kRegsEpi <= 12 * 80, "register pool");
constexpr uint32_t kTmemCols = 256;
constexpr uint32_t COL_ACC = 0, COL_SLOT0 = 48, SLOT_STRIDE = 104, OFF_A = 64;

struct __align__(8) DenseBars {
  uint64_t full[STAGES], empty[STAGES];
  uint64_t acc_full, acc_empty, a_ready[2], d_ready[2];
  uint32_t tmem_base;
  uint32_t pad;
};

// Residual variants of the fused kernel (template parameter kMode).  The PointNet form of Phi
// needs the max-pool over all nodes of a patch before any node can be decoded,
// so it runs as two passes of this kernel with a tiny per-(env, patch) kernel in between:
//   kModePnEncode: [u^, p, n] -> E1 -> SiLU -> E2 -> SiLU = f_i, column max over the rows -> gmax
//   kModePnDecode: propagation as usual; f_i again; D1[:, :64] f_i + c_(e,p) -> SiLU -> D2 -> r
// where c_(e,p) = D1[:, 64:] silu(G1 g + g1) + d1 comes from pn_global_kernel.
constexpr int kModeNone = 0, kModePerNode = 1, kModePnEncode = 2, kModePnDecode = 3;
// layers that run as MMAs, each followed by a SiLU granule (the 3 x 64 output layer runs in the epilogue)
__host__ __device__ constexpr int mode_layers(int mode) { return mode == 1 ? 2 : mode == 2 ? 2 : mode == 3 ? 3 : 0; }
__host__ __device__ constexpr int mode_stages(int mode) { return mode == 3 ? 3 : 4; }  // shared memory: 2 CTAs per SM
__host__ __device__ constexpr int mode_img_bytes(int mode) {
  return mode == 1 ? kWImgBytes : mode == 2 ? kW1ImgBytes + kW2ImgBytes : mode == 3 ? kPnImgBytes : 0;
}

// The big-patch instantiation (kGrouped) keeps an item's u_lin in a per-thread shared-memory stash (24 fp32 per
// epilogue thread) and pays for it with one pipeline stage.
constexpr int kStashBytes = 8 * 3 * 256 * 4;
__host__ __device__ constexpr size_t dense_smem_bytes(int n_patches, int mode, bool big = false) {
  return 1024 /*align slack*/ + (size_t)(mode_stages(mode) - (big ? 1 : 0)) * (A_STAGE + B_STAGE) + (big ? kStashBytes : 0) +
         mode_img_bytes(mode) + sizeof(DenseBars) +
         (size_t)(5 * n_patches + 4) * 4 + 16 + 16 + 8 * 32 * 16;
}


struct Item {
  int p, mb, tile, cnt;
};

#ifndef ETAC_GATHER_DEPTH
#define ETAC_GATHER_DEPTH 16
#endif
constexpr int kGatherDepth = ETAC_GATHER_DEPTH;  // K loads in flight per thread in the gather form (divides 32)

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
    zero_out_rows(io, e, off, cnt, lane, 32);
    if (io.analytic_out) warp_zero_fill(io.analytic_out + ((int64_t)e * m.n_nodes + off) * 3, cnt * 3, lane);
    return true;
  }
};

// prefix[0..P]: first work index of every patch.  kGrouped: four more ints per patch behind it (contacting
// envs, env tiles, env tiles per group G, G x node blocks), written once by the prologue.
// Item order inside a patch.  Plain (kGrouped = false): node block mb = r / tiles, the env tile is the fast
// index.  Grouped: env tiles in groups of G whose U^ operand tiles (BN x n bf16 each) stay resident in L2
// together; a group sweeps all node blocks before the next group starts.  Without the groups a large single
// patch (cfg 4: 256 tiles x 786 KB = 201 MB > L2) re-reads every U^ tile from HBM once per node block.  The
// grouped decode is its own instantiation, launched only when a patch's operand can exceed ETAC_OPT_L2_GROUP_BYTES: the
// epilogue's schedule is sensitive to every instruction of the item set-up (cfg 3: 334 us plain, 336-345 us
// with the grouped decode in its three variants).
__host__ __device__ constexpr int kPrefixInts(int n_patches) { return n_patches + 1; }
template <bool kGrouped>
__device__ __forceinline__ bool decode_item(const int* prefix, int n_patches, const DevModel& m, int w, int& pcur,
                                            Item& it) {
  if (w >= prefix[n_patches]) return false;
  while (prefix[pcur + 1] <= w) ++pcur;
  const int r = w - prefix[pcur];
  it.p = pcur;
  if constexpr (!kGrouped) {
    const int cnt = m.count[pcur];
    const int tiles = (cnt + TE - 1) / TE;
    it.mb = r / tiles;
    it.tile = r - it.mb * tiles;
    it.cnt = min(TE, cnt - it.tile * TE);
  } else {
    const int* pinfo = prefix + kPrefixInts(n_patches) + 4 * pcur;
    const int cnt = pinfo[0], tiles = pinfo[1], G = pinfo[2], GN = pinfo[3];
    const int g = r / GN;
    const int rem = r - g * GN;
    const int gsz = min(G, tiles - g * G);
    it.mb = rem / gsz;
    it.tile = g * G + (rem - it.mb * gsz);
    it.cnt = min(TE, cnt - it.tile * TE);
  }
  return true;
}

#ifdef ETAC_PROFILE
// timing experiment only: per-epilogue-warp cycle accumulators [cta][warp 0..7][12]
__device__ long long g_prof[320 * 8 * 12];
#define PROF_MARK(i)                         \
  do {                                       \
    const long long now_ = clock64();        \
    prof[i] += now_ - plast, plast = now_;   \
  } while (0)
#else
#define PROF_MARK(i)
#endif

// kGather: the propagation is not the dense tensor-core contraction but Omega U_a literally
// (PAPER.md:L87): every epilogue thread sums K[i][j] u^_j over the ACTIVE nodes j of its unit,
// read from the compact lists S1 wrote (bf16 K row j, coalesced over i because K is symmetric;
// fp32 u^ and accumulation).  No TMA, no propagation MMA; the MLP part is unchanged.  It wins
// when few nodes are in contact (ETAC_PATH_SPARSE on a bf16 context).
template <int kMode, bool kGather, bool kOutBf16, bool kGrouped>
__global__ void __launch_bounds__(kDenseThreads, 2)
    dense_bf16_kernel(DevModel m, StepIO io, const __grid_constant__ CUtensorMap tmA,
                      const __grid_constant__ CUtensorMap tmB) {
  constexpr bool kResid = kMode != kModeNone;
  constexpr bool kPn = kMode == kModePnEncode || kMode == kModePnDecode;
  constexpr bool kProp = !kGather && kMode != kModePnEncode;  // TMA + propagation GEMM run
  constexpr bool kFill = kMode != kModePnEncode;              // the decode pass zero-fills
  constexpr int kLayers = mode_layers(kMode), kStages = mode_stages(kMode) - (kGrouped ? 1 : 0), kImgBytes = mode_img_bytes(kMode);
  constexpr bool kStash = kGrouped && kProp;  // u_lin of an item parked in shared memory, accumulator released at once
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + kStages * A_STAGE;
  uint8_t* sW = sB + kStages * B_STAGE;
  DenseBars* bars = reinterpret_cast<DenseBars*>(sW + kImgBytes);
  int* prefix = reinterpret_cast<int*>(bars + 1);
  uint8_t* sGather = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(prefix + kPrefixInts(m.n_patches) + 4 * m.n_patches) + 15) & ~uintptr_t(15));  // 8 warps x 32 entries
  float* sStash = reinterpret_cast<float*>(sGather + 8 * 32 * 16);  // kStash: [unit of the slot 0..7][component][epilogue thread]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&bars->full[s], 1), mbar_init(&bars->empty[s], 1);
    mbar_init(&bars->acc_full, 1);
    mbar_init(&bars->acc_empty, 8);
    for (int s = 0; s < 2; ++s) mbar_init(&bars->a_ready[s], 4), mbar_init(&bars->d_ready[s], 1);
    fence_barrier_init();
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 2) {
    // prefix[p] = first work index of patch p: warp scan, 32 patches per sweep (the per-patch counts
    // and sizes are global loads: issued in parallel instead of one dependent chain by one thread)
    int carry = 0;
    for (int p0 = 0; p0 < m.n_patches; p0 += 32) {
      const int p = p0 + lane;
      int v = 0;
      if (p < m.n_patches) {
        const int cnt = m.count[p], n = m.patch[p].n;
        const int tiles = (cnt + TE - 1) / TE, nmb = (n + BM - 1) / BM;
        if constexpr (kGrouped) {
          const int G = max(1, min(tiles, m.group_bytes / (BN * 2 * max(n, 1))));
          int* pinfo = prefix + kPrefixInts(m.n_patches) + 4 * p;
          pinfo[0] = cnt, pinfo[1] = tiles, pinfo[2] = G, pinfo[3] = max(G * nmb, 1);
        }
        v = tiles * nmb;
      }
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
      }
      if (p < m.n_patches) prefix[p + 1] = carry + v;
      carry += __shfl_sync(0xffffffffu, v, 31);
    }
    if (lane == 0) prefix[0] = 0;
  }
  if (warp == 1) tmem_alloc<kTmemCols>(&bars->tmem_base);
  if constexpr (kResid) {
    const uint4* src = reinterpret_cast<const uint4*>(kPn ? m.wimg_pn : m.wimg);
    uint4* dst = reinterpret_cast<uint4*>(sW);
    for (int k = threadIdx.x; k < kImgBytes / 16; k += kDenseThreads) dst[k] = src[k];
    fence_proxy_async_smem();  // generic-proxy writes -> visible to the tensor-core (async) proxy
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (warp == 0) {
    reg_dealloc<kRegsCtrl>();
    if constexpr (kProp)
    // ------------------------------------------------------------------ TMA producer
    // (the whole warp runs the loop so that every operand stays warp-uniform; one elected lane issues)
    {
      int pcur = 0, stage = 0;
      uint32_t ph = 0;
      Item it;
      for (int w = blockIdx.x; decode_item<kGrouped>(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
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
          if (++stage == kStages) stage = 0, ph ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    reg_dealloc<kRegsCtrl>();
    if constexpr (kProp)
    // ------------------------------------------------------------------ MMA issuer
    // Warp-uniform control flow; tcgen05.mma / tcgen05.commit are issued by one elected lane.
    {
      constexpr uint32_t idesc_prop = make_idesc_bf16(BM, BN);
      int pcur = 0, stage = 0;
      uint32_t ph = 0, acc_ph = 0;
      Item it;
      for (int w = blockIdx.x; decode_item<kGrouped>(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
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
          if (++stage == kStages) stage = 0, ph ^= 1;
        }
      }
    }
  } else if (warp < 4) {
    reg_dealloc<kRegsCtrl>();
    // ------------------------------------------------------------------ MLP MMA issuer of slot (warp - 2)
    // One dedicated issuer warp per slot: a tcgen05.mma round trip is ~450 cycles during which the
    // issuing warp makes no progress, so the two slots must not share an issuer.
    // Between requests the warp zero-fills its share of the output rows of contact-free (env, patch)
    // pairs, one run per request, so that these stores trickle out next to the MUFU-bound work.
    ZeroFill zf;
    zf.init(m, io, blockIdx.x * 2 + (warp - 2), gridDim.x * 2);
    if constexpr (kResid) {
      const int sl = warp - 2;
      constexpr uint32_t idesc_h = make_idesc_bf16(BM, 64);
      const uint64_t dW1 = make_desc(smem_u32(sW), 1024, 128, kLayoutNone);
      const uint64_t dW2 = make_desc(smem_u32(sW + kW1ImgBytes), 1024, 128, kLayoutNone);
      const uint64_t dW3h = make_desc(smem_u32(sW + kW1ImgBytes + kW2ImgBytes), 1024, 128, kLayoutNone);
      const uint32_t tD = tmem + COL_SLOT0 + SLOT_STRIDE * sl, tA = tD + OFF_A;
      uint64_t* a_ready = &bars->a_ready[sl];
      uint64_t* d_ready = &bars->d_ready[sl];
      int pcur = 0;
      uint32_t a_ph = 0;
      Item it;
      for (int w = blockIdx.x; decode_item<kGrouped>(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
        for (int el = sl; el < it.cnt; el += 2) {
#pragma unroll 1
          for (int layer = 0; layer < kLayers; ++layer) {
            mbar_wait(a_ready, a_ph), a_ph ^= 1;
            tc_fence_after();
            if (elect_one()) {
              // weight image: [64 x 16] | [64 x 80] | PointNet decoder: [64 x 80]
              if (layer == 0) {
                mma_ts(tD, tA, dW1, idesc_h, 0);
              } else {
                const uint64_t dWh = layer == 1 ? dW2 : dW3h;
#pragma unroll
                for (int k = 0; k < 5; ++k) mma_ts(tD, tA + 8 * k, dWh + (uint64_t)(k * (2048 >> 4)), idesc_h, k != 0);
              }
              tc_commit(d_ready);
            }
            __syncwarp();
            if constexpr (kFill) zf.step(m, io, lane);
          }
        }
      }
    }
    if constexpr (kFill) {
      while (zf.step(m, io, lane)) {
      }
    }
  } else {
    reg_alloc<kRegsEpi>();
    // ------------------------------------------------------------------ epilogue (thread = node)
    // Two warpgroups; warpgroup s owns TMEM slot s and takes the environments el = s, s+2, ...
    const int sl = (warp - 4) >> 2;
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
#ifdef ETAC_PROFILE
    long long prof[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    long long plast = clock64();
    const long long pstart = plast;
#endif
    for (int w = blockIdx.x; decode_item<kGrouped>(prefix, m.n_patches, m, w, pcur, it); w += gridDim.x) {
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
      PROF_MARK(0);  // item setup
      if constexpr (kProp) {
        mbar_wait(&bars->acc_full, acc_ph), acc_ph ^= 1;
        tc_fence_after();
      }
      PROF_MARK(1);  // acc_full wait
      if constexpr (kStash) {
        // Big patches: the propagation GEMM of an item is as long as its MLP work, and with one accumulator
        // the two would alternate.  Every epilogue thread parks the u_lin of its (up to 8) units of the item
        // in its own shared-memory words (nobody else reads them: no barrier) and the accumulator goes back
        // to the MMA warp at once, so the next item's GEMM runs under this item's MLP.
        float* st = sStash + (threadIdx.x - 128);
#pragma unroll
        for (int k0 = 0; k0 < 8; k0 += 4) {  // four units at a time: 16 registers in flight
          if (sl + 2 * k0 < it.cnt) {
            uint32_t q[4][4];
#pragma unroll
            for (int k = 0; k < 4; ++k) tmem_ld4(trow + COL_ACC + 3 * min(sl + 2 * (k0 + k), TE - 1), q[k]);
            tc_wait_ld();
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              st[(k0 + k) * 768] = __uint_as_float(q[k][0]);
              st[(k0 + k) * 768 + 256] = __uint_as_float(q[k][1]);
              st[(k0 + k) * 768 + 512] = __uint_as_float(q[k][2]);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->acc_empty);
      }
      // The units of an item are software-pipelined: while the tensor core runs the last MMA layer of unit
      // el, the u_lin of unit el+2 is already fetched from the accumulator, and its layer-1 operand
      // is written (and requested) before the output of unit el is combined and stored.  Every
      // TMEM access costs a few hundred cycles of latency; this takes two of them per unit off
      // the chain's critical path.
      struct Unit {
        int64_t node;
        float ux, uy, uz, dl;
        int slot;  // position of the unit's environment in the patch's contact list
      };
      auto fetch_unit = [&](Unit& u, const int el, uint32_t (&ur)[4]) {  // requests only; tc_wait_ld() follows
        const int env = __shfl_sync(0xffffffffu, my_env, el);
        u.node = (int64_t)env * m.n_nodes + g;
        u.dl = valid ? m.delta[u.node] : 0.0f;  // consumed when the unit is stored
        u.slot = it.tile * TE + el;
        if constexpr (kStash) {
          const float* st = sStash + ((el - sl) >> 1) * (3 * 256) + (threadIdx.x - 128);
          ur[0] = __float_as_uint(st[0]), ur[1] = __float_as_uint(st[256]), ur[2] = __float_as_uint(st[512]), ur[3] = 0;
        } else if constexpr (kProp) {
          tmem_ld4(trow + COL_ACC + 3 * el, ur);
        } else if constexpr (kMode == kModePnEncode) {
          ur[0] = ur[1] = ur[2] = ur[3] = 0;  // the encoder pass has no propagation
        } else {
          // Omega U_a: sum over the active nodes of this (env, patch); entry loads are warp-uniform
          // (broadcast), K row j is read coalesced over the rows i of the warp
          const int slot = it.tile * TE + el;
          const int cnt = m.acount[(int64_t)it.p * m.max_envs + slot];
          const ActiveEntry* __restrict__ al = m.alist + (int64_t)slot * m.ldu + pi.off;
          const __nv_bfloat16* __restrict__ kcol = m.k16 + (int64_t)pi.off * m.kw + (valid ? li : 0);
          float ax = 0.f, ay = 0.f, az = 0.f;
          // 32 entries per sweep: lane l loads entry k0+l (one coalesced 512-byte read) into the
          // warp's shared-memory staging row; the entries are then read back as broadcasts while
          // kGatherDepth K loads are in flight per thread
          float4* stage = reinterpret_cast<float4*>(sGather) + (warp - 4) * 32;
          for (int k0 = 0; k0 < cnt; k0 += 32) {
            float4 mine = make_float4(0.f, 0.f, 0.f, 0.f);  // padding entries: u^ = 0, j = 0
            if (k0 + lane < cnt) mine = __ldg(reinterpret_cast<const float4*>(al + k0 + lane));
            __syncwarp();
            stage[lane] = mine;
            __syncwarp();
            const int nb = min(32, cnt - k0);
            for (int q0 = 0; q0 < nb; q0 += kGatherDepth) {  // the loop is bound by loads in flight
              float kv[kGatherDepth];
#pragma unroll
              for (int q = 0; q < kGatherDepth; ++q)
                kv[q] = __bfloat162float(kcol[(int64_t)__float_as_int(stage[q0 + q].w) * m.kw]);
#pragma unroll
              for (int q = 0; q < kGatherDepth; ++q) {
                const float4 en = stage[q0 + q];
                ax = fmaf(kv[q], en.x, ax), ay = fmaf(kv[q], en.y, ay), az = fmaf(kv[q], en.z, az);
              }
            }
          }
          ur[0] = __float_as_uint(ax), ur[1] = __float_as_uint(ay), ur[2] = __float_as_uint(az), ur[3] = 0;
        }
      };
      auto request_layer1 = [&](Unit& u, const uint32_t (&ur)[4]) {
        u.ux = __uint_as_float(ur[0]), u.uy = __uint_as_float(ur[1]), u.uz = __uint_as_float(ur[2]);
        if constexpr (kResid) {
          if constexpr (kPn) {  // PointNet encoder input: u^ = -delta n of the node itself
            a1[0] = pack_bf16(-u.dl * nrm.x, -u.dl * nrm.y);
            a1[1] = pack_bf16(-u.dl * nrm.z, px);
          } else {
            a1[0] = pack_bf16(u.ux, u.uy);
            a1[1] = pack_bf16(u.uz, px);
          }
          tmem_st8(tA, a1);
          tc_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(a_ready);
        }
      };
      // the accumulator is released as soon as this warp has fetched its LAST u_lin of the item, a
      // whole unit before the item ends: the next item's propagation GEMM runs behind that unit's MLP
      auto release_acc = [&]() {
        if constexpr (kProp && !kStash) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&bars->acc_empty);
        }
      };
      Unit cur, nxt;
      {
        uint32_t ur[4];
        if (sl < it.cnt) {
          fetch_unit(cur, sl, ur);
          tc_wait_ld();
          if (sl + 2 >= it.cnt) release_acc();
          request_layer1(cur, ur);
        } else {
          release_acc();
        }
      }
      PROF_MARK(2);  // first unit of the item: u_lin, layer-1 operand
      for (int el = sl; el < it.cnt; el += 2) {
        const bool more = el + 2 < it.cnt;
        float rx = 0.f, ry = 0.f, rz = 0.f;
        uint32_t un[4] = {0, 0, 0, 0};
        // The next unit's layer-1 operand and request; the operand region is free once the last MMA layer
        // has been read.  Placement matters more than it should: issuing this (or the accumulator
        // release, or anything else with a warp-level sync) between the TMEM loads of the last
        // granule and its SiLUs costs 5-8 % (measured), so it sits after the granule.
        auto request_next = [&]() {
          if (more && el + 4 >= it.cnt) release_acc();
          if (more) request_layer1(nxt, un);
          PROF_MARK(3);  // next unit's layer-1 operand + arrive
        };
        if constexpr (kResid) {
          // One SiLU granule per MMA layer.  The inner granules write the next layer's bf16 operand
          // back to TMEM and request the layer; the last one keeps its fp32 outputs in registers and
          // applies the 3 x 64 output layer on the FMA pipe (per-node MLP / decoder) or max-pools
          // them over the rows (encoder).  The decoder's last layer adds the per-(env, patch)
          // vector c (halved like the weights).
          uint32_t ha[32], hb[32];
#pragma unroll 1
          for (int layer = 0; layer < kLayers - 1; ++layer) {
            mbar_wait(d_ready, d_ph), d_ph ^= 1;
            tc_fence_after();
            PROF_MARK(4);  // d_ready wait
            // both halves are requested at once: one TMEM load latency per layer instead of two
            uint32_t packed[16];
            tmem_ld32(tD, ha);
            tmem_ld32(tD + 32, hb);
            tc_wait_ld();
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              uint32_t(&h)[32] = half ? hb : ha;
#pragma unroll
              for (int k = 0; k < 16; ++k) {
                // D holds x/2 (0.5 folded into the weights): silu(x) = x*sigmoid(x) = h + h*tanh(h)
                float y0, y1;
                unpack_f32x2(silu_half_x2(__uint_as_float(h[2 * k]), __uint_as_float(h[2 * k + 1])), y0, y1);
                packed[k] = pack_bf16(y0, y1);
              }
              tmem_st16(tA + 16 * half, packed);
            }
            PROF_MARK(6);  // D load + SiLU + operand stores issued
            tc_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(a_ready);
            PROF_MARK(7);  // store wait + arrive
          }
          // ---- last granule
          if (more) fetch_unit(nxt, el + 2, un);  // overlaps the last layer's round trip
          mbar_wait(d_ready, d_ph), d_ph ^= 1;
          tc_fence_after();
          PROF_MARK(8);  // d_ready wait (last layer)
          tmem_ld32(tD, ha);
          tmem_ld32(tD + 32, hb);
          tc_wait_ld();
          PROF_MARK(9);  // D (and next u_lin) load
          if constexpr (kMode == kModePnEncode) {
            uint32_t pool0 = 0, pool1 = 0;  // lane l: max keys of hidden columns l and 32 + l
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              uint32_t(&h)[32] = half ? hb : ha;
#pragma unroll
              for (int k = 0; k < 32; ++k) {
                // column max over the warp's 32 rows.  silu >= -0.279, so 1 + silu is a positive
                // float whose bit pattern orders like the value; 0 = no row
                const float h0 = __uint_as_float(h[k]);
                const float y0 = fmaf(h0, tanh_approx(h0), h0);
                const uint32_t k0 = valid ? __float_as_uint(1.0f + y0) : 0u;
                const uint32_t m0 = __reduce_max_sync(0xffffffffu, k0);
                if (lane == k) (half ? pool1 : pool0) = m0;
              }
            }
            uint32_t* gm = m.gmax + ((int64_t)it.p * m.max_envs + cur.slot) * 64;
            atomicMax(gm + lane, pool0);
            atomicMax(gm + 32 + lane, pool1);
          } else {
            const float4* cv = nullptr;
            if constexpr (kMode == kModePnDecode)
              cv = reinterpret_cast<const float4*>(m.cvec + ((int64_t)it.p * m.max_envs + cur.slot) * 64);
            // even / odd hidden columns accumulate in the two halves of packed fp32x2 registers
            uint64_t ax = pack_f32x2(m.wout[192], 0.f), ay = pack_f32x2(m.wout[193], 0.f), az = pack_f32x2(m.wout[194], 0.f);
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              uint32_t(&h)[32] = half ? hb : ha;
#pragma unroll
              for (int k4 = 0; k4 < 8; ++k4) {
                float4 c4 = make_float4(0.f, 0.f, 0.f, 0.f);
                if constexpr (kMode == kModePnDecode) c4 = __ldg(cv + half * 8 + k4);
                const float cc[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
                for (int q = 0; q < 4; q += 2) {
                  const int k = 4 * k4 + q, col = 32 * half + k;
                  float h0 = __uint_as_float(h[k]), h1 = __uint_as_float(h[k + 1]);
                  if constexpr (kMode == kModePnDecode) h0 += cc[q], h1 += cc[q + 1];
                  const uint64_t y = silu_half_x2(h0, h1);
                  ax = fma_f32x2(y, pack_f32x2(m.wout[col], m.wout[col + 1]), ax);
                  ay = fma_f32x2(y, pack_f32x2(m.wout[64 + col], m.wout[65 + col]), ay);
                  az = fma_f32x2(y, pack_f32x2(m.wout[128 + col], m.wout[129 + col]), az);
                }
              }
            }
            float lo, hi;
            unpack_f32x2(ax, lo, hi), rx = lo + hi;
            unpack_f32x2(ay, lo, hi), ry = lo + hi;
            unpack_f32x2(az, lo, hi), rz = lo + hi;
          }
          request_next();
          PROF_MARK(5);  // last granule: SiLU + output layer / pool
        } else {
          if (more) {
            fetch_unit(nxt, el + 2, un);
            tc_wait_ld();
          }
          request_next();
        }
        // (the environment id is re-read from the prefetched list here rather than kept in a register
        // through the MLP: the register allocation of this loop is fragile)
        const int cur_env = __shfl_sync(0xffffffffu, my_env, el);
        if (valid && kMode != kModePnEncode) {  // S4: mask M_p + combine (Eq. 2); active rows keep u^ = -delta n in fp32
          const float lin = m.residual_only ? 0.0f : 1.0f;  // Table II ablation "Residual Network Only"
          float ox = fmaf(lin, cur.ux, rx), oy = fmaf(lin, cur.uy, ry), oz = fmaf(lin, cur.uz, rz);
          if (cur.dl > 0.0f && m.active_mode == ETAC_ACTIVE_PASSTHROUGH)
          {
            // (reloaded for the few active rows instead of held in three registers through the MLP)
            const float4 nn = kPn ? nrm : m.nrm4[g];
            ox = -cur.dl * nn.x, oy = -cur.dl * nn.y, oz = -cur.dl * nn.z;
          }
          store_out3<kOutBf16 ? ETAC_OUT_BF16 : ETAC_OUT_F32>(io, cur_env, g, ox, oy, oz);
          if (io.analytic_out) {
            float* a = io.analytic_out + cur.node * 3;
            __stcs(a, cur.ux), __stcs(a + 1, cur.uy), __stcs(a + 2, cur.uz);
          }
        }
        cur = nxt;
        PROF_MARK(10);  // mask, combine, store
      }
    }
#ifdef ETAC_PROFILE
    prof[11] = clock64() - pstart;
    if (lane == 0 && blockIdx.x < 320)
      for (int i = 0; i < 12; ++i) g_prof[(blockIdx.x * 8 + (warp - 4)) * 12 + i] = prof[i];
#endif
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<kTmemCols>(tmem);
  }
}

// c_(e,p) of the PointNet decoder: g = max-pooled features (keys = bits of 1 + f), g' = silu(G1 g + g1)
// ("further encoded by another MLP"), c = D1[:, 64:128] g' + d1, stored halved like
// the decoder weights.  A 64-thread CTA stages the two transposed 64 x 64 matrices in shared
// memory once and walks kPnSlots contact-list slots of one patch.
constexpr int kPnSlots = 16;
__global__ void __launch_bounds__(64) pn_global_kernel(DevModel m) {
  const int p = blockIdx.y, k = threadIdx.x;
  const int slot0 = blockIdx.x * kPnSlots, cnt = m.count[p];
  if (slot0 >= cnt) return;
  __shared__ float sG1[64 * 64], sD1[64 * 64], g[64], g2[64];
  const float* G1t = m.pn_f32, *g1 = G1t + 4096, *D1gt = g1 + 64, *d1 = D1gt + 4096;  // both matrices [in][out]
  for (int i = k; i < 4096; i += 64) sG1[i] = G1t[i], sD1[i] = D1gt[i];
  const float bg = g1[k], bd = d1[k];
  for (int slot = slot0; slot < min(cnt, slot0 + kPnSlots); ++slot) {
    const int64_t base = ((int64_t)p * m.max_envs + slot) * 64;
    const uint32_t key = m.gmax[base + k];
    __syncthreads();  // previous slot done with g / g2; first pass: weights staged
    g[k] = __uint_as_float(key) - 1.0f;  // keys are the bit patterns of 1 + f
    __syncthreads();
    float a = bg;
#pragma unroll 8
    for (int j = 0; j < 64; ++j) a = fmaf(sG1[j * 64 + k], g[j], a);
    g2[k] = a / (1.0f + expf(-a));
    __syncthreads();
    float c = bd;
#pragma unroll 8
    for (int j = 0; j < 64; ++j) c = fmaf(sD1[j * 64 + k], g2[j], c);
    m.cvec[base + k] = 0.5f * c;
  }
}

template <int kMode, bool kGather>
static cudaError_t configure_one() {
  const int bytes = (int)dense_smem_bytes(kMaxPatches, kMode), bytes_big = (int)dense_smem_bytes(kMaxPatches, kMode, true);
  cudaError_t e = cudaFuncSetAttribute(dense_bf16_kernel<kMode, kGather, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess && kMode != kModePnEncode)  // the encoder pass writes no displacement
    e = cudaFuncSetAttribute(dense_bf16_kernel<kMode, kGather, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if constexpr (!kGather && kMode != kModePnEncode) {  // grouped item order: dense propagation only
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dense_bf16_kernel<kMode, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes_big);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dense_bf16_kernel<kMode, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes_big);
  }
  return e;
}

cudaError_t dense_bf16_configure() {
  cudaError_t e = configure_one<kModeNone, false>();
  if (e == cudaSuccess) e = configure_one<kModeNone, true>();
  if (e == cudaSuccess) e = configure_one<kModePerNode, false>();
  if (e == cudaSuccess) e = configure_one<kModePerNode, true>();
  if (e == cudaSuccess) e = configure_one<kModePnEncode, false>();
  if (e == cudaSuccess) e = configure_one<kModePnDecode, false>();
  if (e == cudaSuccess) e = configure_one<kModePnDecode, true>();
  return e;
}

template <int kMode>
static void launch_one(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB, int grid,
                       bool gather, cudaStream_t s) {
  const size_t smem = dense_smem_bytes(m.n_patches, kMode);
  // big-patch instantiation (grouped item order + u_lin stash): where a patch's U^ operand (3 bf16 rows of n nodes
  // per env) can exceed the L2 share, or a patch is large enough for its propagation GEMM (2.75 n cycles per item)
  // to matter next to the MLP of the item's 16 units
  const bool grouped = !gather && ((size_t)io.n_envs * (size_t)m.max_patch_nodes * 6 > (size_t)m.group_bytes || m.max_patch_nodes >= 2048);
  if constexpr (kMode == kModePnEncode) {
    dense_bf16_kernel<kMode, false, false, false><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
  } else if (gather) {
    if (io.out_bf16) dense_bf16_kernel<kMode, true, true, false><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
    else dense_bf16_kernel<kMode, true, false, false><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
  } else if (grouped) {
    const size_t smem_big = dense_smem_bytes(m.n_patches, kMode, true);
    if (io.out_bf16) dense_bf16_kernel<kMode, false, true, true><<<grid, kDenseThreads, smem_big, s>>>(m, io, tmA, tmB);
    else dense_bf16_kernel<kMode, false, false, true><<<grid, kDenseThreads, smem_big, s>>>(m, io, tmA, tmB);
  } else {
    if (io.out_bf16) dense_bf16_kernel<kMode, false, true, false><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
    else dense_bf16_kernel<kMode, false, false, false><<<grid, kDenseThreads, smem, s>>>(m, io, tmA, tmB);
  }
}

// Launches S2-S4 for the context's residual form; *launches receives the number of kernels.
cudaError_t launch_dense_bf16(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB,
                              int n_sm, bool gather, int* launches, cudaStream_t s) {
  const int grid = 2 * n_sm;
  *launches = 1;
  if (m.resid == ETAC_RESID_NONE) {
    launch_one<kModeNone>(m, io, tmA, tmB, grid, gather, s);
  } else if (m.resid == ETAC_RESID_PERNODE_MLP) {
    launch_one<kModePerNode>(m, io, tmA, tmB, grid, gather, s);
  } else {  // ETAC_RESID_POINTNET: encode + max-pool, per-(env, patch) vector, decode
    cudaError_t e = cudaMemsetAsync(m.gmax, 0, sizeof(uint32_t) * 64 * (size_t)m.n_patches * m.max_envs, s);
    if (e != cudaSuccess) return e;
    launch_one<kModePnEncode>(m, io, tmA, tmB, grid, false, s);
    pn_global_kernel<<<dim3((unsigned)((io.n_envs + kPnSlots - 1) / kPnSlots), (unsigned)m.n_patches), 64, 0, s>>>(m);
    launch_one<kModePnDecode>(m, io, tmA, tmB, grid, gather, s);
    *launches = 3;
  }
  return cudaGetLastError();
}

}  // namespace etac

#ifdef ETAC_PROFILE
extern "C" void etac_debug_prof(long long* out) { cudaMemcpyFromSymbol(out, etac::g_prof, sizeof(long long) * 320 * 8 * 12); }
#endif


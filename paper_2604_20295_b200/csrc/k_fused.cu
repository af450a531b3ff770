// S2+S3+S4 fused, tensor-core path (sm_100a: TMA + tcgen05.mma + TMEM).
//
//   S2  u_lin = K_p . U^  as a dense bf16 contraction with fp32 accumulation in TMEM
//       ("propagation matrix Omega ... computed as Omega U_a"; the zero rows of the
//       zero-padded U^ contribute nothing, R3),
//   S3  residual MLP 9 -> 64 -> 64 -> 3 (SiLU) on the accumulator tile: the two hidden layers are
//       small tcgen05.mma's (SS form: the epilogue warps write the bf16 layer input into shared memory
//       in the UMMA core-matrix layout, the weights, with the biases as an extra K column against a
//       constant "ones" block, stay in shared memory); the 3 x 64 output layer is applied in fp32 by the
//       epilogue to the SiLU outputs it holds in registers (packed fma.rn.f32x2),
//   S4  mask M_p + combine (Eq. 2) and the store of U[e][i][0..2]; the rows of
//       contact-free (env, patch) pairs are zero-filled by two control warps (R8).
//
// Work item = (patch p, block of 128 nodes, tile of TE contacting environments of that patch); a UNIT is
// one environment of an item (128 nodes x 1 env: one M = 128 operand of the MLP).  Persistent grid,
// ONE CTA per SM; every CTA walks the items blockIdx.x, +gridDim.x, ...
//
// Warps: 0 = TMA producer, 1 = propagation-GEMM MMA issuer (+ TMEM alloc), 2/3 = zero-fill of the
// contact-free rows; then NC "chains" of four epilogue warps (thread = node = TMEM lane).  setmaxnreg
// gives the control warps 24 registers and the epilogue warps the rest of the pool.
//
// NC units are in flight per SM (6 for the 16-env tile, 5 for the 32-env tile): the kernel is bound by the
// special-function pipe (128 SiLUs per node-env), and a unit spends as much time in its two tcgen05.mma
// round trips (operand store -> chain barrier -> mma -> commit -> mbarrier -> TMEM load) as in its SiLUs, so the
// pipe only stays busy if enough independent units overlap.  A chain owns a 64-column D region of TMEM and
// 16 KB of shared memory for its layer operands; the units of the CTA's item stream are dealt to the chains
// round robin (unit q goes to chain q mod NC), independent of item boundaries.  The chain's own warps issue
// its MLP MMAs: three warps arrive on the chain's named barrier and go on, the fourth (warp c % 4 of chain c)
// waits on it and one of its lanes issues -- there is no issuer warp in between.  The next unit's layer 1 is
// requested as soon as the last layer's D is in registers.  The propagation accumulator is double-buffered,
// so the GEMM of item k+1 runs under the MLP of item k.
//
// Large patches (kGrouped, 32-env tile): the item order keeps the U^ tiles of a group of env tiles resident in
// L2, and the contraction is block-sparse -- the TMA and MMA warps skip the 64-node k-blocks in which no
// environment of the tile has an active node (S1 wrote the bitmaps and bucketed the environments by contact
// position; Omega is (n - m) x m).  The grid runs as clusters of two CTAs that take the two node
// blocks of a pair for the same env tile: each fetches half of the U^ tile and multicasts it into both shared
// memories, and a ring stage is released by the commits of both CTAs' MMAs.
//
// Template variants (one source, see kMode / kGather / TE below): per-node MLP or none; the PointNet form
// of Phi as an encoder pass with max-pool and a decoder pass; the gather form of the propagation
// (Omega U_a over the active-node lists) instead of the dense contraction.
//
// TMEM columns (fp32 lanes = nodes): [0, BN) and [BN, 2 BN): u_lin accumulators, column 3*env+c;
//                                    chain c at 2 BN + 64 c: D, the pre-activations of its current layer.
#include "etac_internal.h"
#include "sm100_prims.cuh"

namespace etac {

constexpr int BM = 128, BK = 64, kMaxStages = 4;
constexpr int A_STAGE = BM * BK * 2;
constexpr int kAop1Bytes = 128 * 16 * 2;   // layer-1 operand of a chain: [128 x 16] bf16, K-major core matrices
constexpr int kAop2Bytes = 128 * 64 * 2;   // hidden-layer operand: [128 x 64]
// The two share one region: the next unit's layer-1 operand is written when the last hidden layer's MMA, the last
// reader of the hidden operand, has completed (its D is in registers), and the hidden operand is written when the
// layer-1 MMA has completed.
constexpr int kAopBytes = kAop2Bytes;
static_assert(kAop1Bytes <= kAop2Bytes, "layer-1 operand inside the hidden operand");
constexpr int kOnesBytes = 128 * 16 * 2;   // [128 x 16]: column 0 = 1.0, the A operand of the bias k-step
constexpr uint32_t kAopLBO = 2048, kAopSBO = 128;   // 16 row groups x 128 B per k-octet

template <int TE>
struct Tile {
  static constexpr int BN = 3 * TE;
  static constexpr int NC = TE == 16 ? 6 : 5;                 // chains: 2 BN + 64 NC <= 512 TMEM columns
  static constexpr int kStages = TE == 16 ? 3 : 4;            // TMA ring (the pair's ring turns around more slowly)
  static constexpr int kThreads = 128 * (NC + 1);
  static constexpr int B_STAGE = BN * BK * 2;
  static constexpr uint32_t COL_D0 = 2 * BN;
  // register pool: kThreads x (65536 / kThreads rounded down to 8) = 4 warps x kRegsCtrl + 4 NC warps x kRegsEpi
  static constexpr int kRegsCtrl = TE == 16 ? 24 : 40;  // control warps (the 32-env tile's walk the k-block bitmaps)
  static constexpr int kRegsEpi = TE == 16 ? 80 : 88;
  static_assert(2 * BN + 64 * NC <= 512, "TMEM columns");
};

// The CTA's item stream.  Small patches (one CTA per item stream, dense propagation): the n-th item of a CTA is
// claimed from a global counter (DevModel::wq) instead of being blockIdx.x + n gridDim.x -- the SMs do not run at the
// same speed (end times of the static order spread over 9 % of the kernel), and a CTA that is ahead takes more
// items.  The TMA warp claims the next item when it has streamed the current one and publishes the sequence in
// shared memory.  The ring is longer than the pipeline is deep: the TMA warp is less than one item ahead of the
// MMA warp, which is at most two items (the two accumulators) ahead of the slowest chain.
constexpr int kSeqRing = 16;
constexpr int kNoWork = 0x7fffffff;

template <int NC>
struct __align__(8) FusedBars {
  uint64_t full[kMaxStages], empty[kMaxStages];
  uint64_t acc_full[2], acc_empty[2], d_ready[NC];
  uint32_t tmem_base;
  uint32_t pad;
  // dynamic item order (kDyn): entry n & (kSeqRing - 1) = (n << 32 | work index of the CTA's n-th item), written by
  // the TMA warp, read by the MMA warp and the chains
  unsigned long long seq[kSeqRing];
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
__host__ __device__ constexpr int mode_img_bytes(int mode) {
  return mode == 1 ? kWImgBytes : mode == 2 ? kW1ImgBytes + kW2ImgBytes : mode == 3 ? kPnImgBytes : 0;
}

// dynamic shared memory of one instantiation: TMA ring (dense propagation only), weight image, ones block, the
// chains' operand regions, barriers, the item prefix table (+ 4 ints per patch for the grouped order) and the
// per-warp staging rows of the gather form
constexpr int kMaxDynSmem = 232448;  // 227 KB opt-in limit of sm_100
template <int TE>
__host__ __device__ constexpr size_t fused_smem_bytes(int n_patches, int mode, bool gather, bool grouped) {
  const bool prop = !gather && mode != 2;
  return 1024 /*align slack*/ + (prop ? (size_t)Tile<TE>::kStages * (A_STAGE + Tile<TE>::B_STAGE) : 0) + mode_img_bytes(mode) + kOnesBytes +
         (size_t)Tile<TE>::NC * kAopBytes + sizeof(FusedBars<Tile<TE>::NC>) + (size_t)(8 * n_patches + 4) * 4 + 16 + 16 +
         (gather ? (size_t)Tile<TE>::NC * 4 * 32 * 16 : 0);
}

constexpr int kGatherDepth = 16;  // K loads in flight per thread in the gather form (divides 32)

__device__ __forceinline__ void named_bar_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ void named_bar_arrive(int id, int threads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ void st_shared_v4(uint32_t saddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(saddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

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

// prefix[0..P]: first work index of every patch, followed by one PTab per patch, both written once by the
// prologue into shared memory (an item decode on the epilogue's path must not wait for global memory).
// Item order inside a patch.  Plain (kGrouped = false): node block mb = r / tiles, the env tile is the fast
// index.  Grouped: env tiles in groups of G whose U^ operand tiles (BN x n bf16 each) stay resident in L2
// together; a group sweeps all node blocks before the next group starts.  Without the groups a large single
// patch (cfg 4: 201 MB of U^ tiles > L2) re-reads every U^ tile from HBM once per node block.
struct PTab {
  int cnt, tiles, off, n;  // contacting envs, env tiles, first node, nodes
  int G, GN;               // grouped order: env tiles per group, G x node blocks
  int uoff;                // first column of the patch in the U^ operand rows
};
__host__ __device__ constexpr int kTabInts(int n_patches) { return n_patches + 1 + 7 * n_patches; }
struct Item {
  int p, mb, tile, cnt, off, n, uoff;  // patch, node block, env tile, units; first node, node count, first U^ column of the patch
};
// Grouped order: the two CTAs of a cluster walk the same stream of (env tile, PAIR of node blocks) and CTA `rank`
// takes node block 2 mbp + rank, so that both want the same U^ tiles at the same time (TMA multicast, see the
// producer).  A patch with an odd number of node blocks leaves one CTA a block beyond the patch: it streams and
// multiplies along (the ring is shared) but has no units (cnt = 0).
template <bool kGrouped, int TE>
__device__ __forceinline__ bool decode_item(const int* prefix, int n_patches, int w, int rank, int& pcur, Item& it) {
  if (w >= prefix[n_patches]) return false;
  while (prefix[pcur + 1] <= w) ++pcur;
  const int r = w - prefix[pcur];
  const PTab t = reinterpret_cast<const PTab*>(prefix + n_patches + 1)[pcur];
  it.p = pcur, it.off = t.off, it.n = t.n, it.uoff = t.uoff;
  if constexpr (!kGrouped) {
    it.mb = r / t.tiles;
    it.tile = r - it.mb * t.tiles;
  } else {
    const int g = r / t.GN;
    const int rem = r - g * t.GN;
    const int gsz = min(t.G, t.tiles - g * t.G);
    const int mbp = rem / gsz;
    it.mb = 2 * mbp + rank;
    it.tile = g * t.G + (rem - mbp * gsz);
  }
  it.cnt = min(TE, t.cnt - it.tile * TE);
  if (kGrouped && it.mb * BM >= it.n) it.cnt = 0;
  return true;
}

// Block-sparse contraction (Omega is (n - m) x m, not n x n): a k-block of 64 nodes in which none of
// the item's environments has an active node contributes exact zeros to the accumulator and is skipped by the
// TMA and MMA warps alike (large patches only: the kGrouped instantiation).  S1 wrote one bitmap per contacting
// (patch, slot), kbtile_kernel ORs them per tile of TE slots, and the two warps read their item's 8 words one item
// ahead, so that the load is never waited for.
template <int TE>
__global__ void __launch_bounds__(32) kbtile_kernel(DevModel m) {
  const int p = blockIdx.y, tile = blockIdx.x, lane = threadIdx.x;
  const int cnt = min(TE, m.count[p] - tile * TE);
  if (cnt <= 0) return;
  const uint32_t* __restrict__ b = m.kbmap + ((int64_t)p * m.max_envs + tile * TE) * kKbWords + (lane & (kKbWords - 1));
  uint32_t v = 0;
#pragma unroll
  for (int s0 = 0; s0 < TE; s0 += 32 / kKbWords) {
    const int sidx = s0 + lane / kKbWords;
    if (sidx < cnt) v |= b[sidx * kKbWords];
  }
#pragma unroll
  for (int d = kKbWords; d < 32; d <<= 1) v |= __shfl_xor_sync(0xffffffffu, v, d);
  if (lane < kKbWords) m.kbtile[((int64_t)p * m.kbtile_stride + tile) * kKbWords + lane] = v;
}
__device__ __forceinline__ uint32_t load_tile_kbmask(const DevModel& m, const Item& it, int lane) {
  return lane < kKbWords ? __ldg(m.kbtile + ((int64_t)it.p * m.kbtile_stride + it.tile) * kKbWords + lane) : 0u;
}

// Walks the active k-blocks of an item in ascending order: next() returns the next k-block index or -1.  All lanes
// hold the same state (the words come from the lanes' union by shuffle); k-blocks beyond the bitmap are all active.
struct KbIter {
  uint32_t lane_word, bits;
  int word, nkb, tail;
  __device__ __forceinline__ void init(uint32_t mask_lane, int nkb_) {
    lane_word = mask_lane, nkb = nkb_, word = 0, tail = 32 * kKbWords;
    bits = __shfl_sync(0xffffffffu, lane_word, 0);
  }
  __device__ __forceinline__ int next() {
    while (word < kKbWords) {
      if (bits) {
        const int kb = word * 32 + __ffs(bits) - 1;
        bits &= bits - 1;
        if (kb < nkb) return kb;
        bits = 0;
      }
      if (++word < kKbWords) bits = __shfl_sync(0xffffffffu, lane_word, word);
    }
    return tail < nkb ? tail++ : -1;
  }
};

// kGather: the propagation is not the dense tensor-core contraction but Omega U_a literally
// (PAPER.md:L87): every epilogue thread sums K[i][j] u^_j over the ACTIVE nodes j of its unit,
// read from the compact lists S1 wrote (bf16 K row j, coalesced over i because K is symmetric;
// fp32 u^ and accumulation).  No TMA, no propagation MMA; the MLP part is unchanged.
template <int kMode, bool kGather, bool kOutBf16, bool kGrouped, int TE>
__global__ void __launch_bounds__(Tile<TE>::kThreads, 1)
    fused_mlp_kernel(DevModel m, StepIO io, const __grid_constant__ CUtensorMap tmA,
                     const __grid_constant__ CUtensorMap tmB) {
  using TL = Tile<TE>;
  constexpr int BN = TL::BN, NC = TL::NC, B_STAGE = TL::B_STAGE, kThreads = TL::kThreads, kStages = TL::kStages;
  constexpr bool kResid = kMode != kModeNone;
  constexpr bool kPn = kMode == kModePnEncode || kMode == kModePnDecode;
  constexpr bool kProp = !kGather && kMode != kModePnEncode;  // TMA + propagation GEMM run
  constexpr bool kFill = kMode != kModePnEncode;              // the decode pass zero-fills
  constexpr int kLayers = mode_layers(kMode), kImgBytes = mode_img_bytes(kMode);
  // Large patches run as clusters of two CTAs on the same env tile and adjacent node blocks: each CTA fetches half
  // of the U^ tile and multicasts it into both shared memories, which takes a fifth off the L2 -> SM traffic that
  // bounds the contraction (K tile 16 KB + 6 instead of 12 KB per k-block and SM).  A ring stage is refilled when
  // the MMAs of BOTH CTAs have read it: `empty` counts two commits, each CTA's commit arrives in both.
  constexpr bool kPair = kGrouped;
  constexpr uint16_t kPairMask = 3;
  constexpr bool kDyn = kProp && !kPair;  // item order claimed from DevModel::wq (see kSeqRing)
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + (kProp ? kStages * A_STAGE : 0);
  uint8_t* sW = sB + (kProp ? kStages * B_STAGE : 0);
  uint8_t* sOnes = sW + kImgBytes;
  uint8_t* sAop = sOnes + kOnesBytes;
  FusedBars<NC>* bars = reinterpret_cast<FusedBars<NC>*>(sAop + NC * kAopBytes);
  int* prefix = reinterpret_cast<int*>(bars + 1);
  uint8_t* sGather = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(prefix + kTabInts(m.n_patches)) + 15) & ~uintptr_t(15));  // 4 NC warps x 32 entries

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = kPair ? (int)cluster_ctarank() : 0;
  const int w_first = kPair ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, w_step = kPair ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  // kDyn: work index of the CTA's n-th item, n >= 1 (item 0 is w_first); waits until the TMA warp has published it
  auto seq_w = [&](const int n) -> int {
    volatile unsigned long long* slot = &bars->seq[n & (kSeqRing - 1)];
    unsigned long long v = *slot;
    uint32_t spins = 0;
    uint64_t t0 = 0;
    while ((int)(v >> 32) != n) {  // (bounded like mbar_wait: a protocol bug ends in a trap, not in a hung GPU)
      if ((++spins & 0x3fffu) == 0) {
        const uint64_t now = global_timer_ns();
        if (t0 == 0) t0 = now;
        else if (now - t0 > 10000000000ull) __trap();
      }
      v = *slot;
    }
    return (int)(uint32_t)v;
  };

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&bars->full[s], 1), mbar_init(&bars->empty[s], kPair ? 2 : 1);
    for (int b = 0; b < 2; ++b) mbar_init(&bars->acc_full[b], 1), mbar_init(&bars->acc_empty[b], 4 * NC);
    for (int c = 0; c < NC; ++c) mbar_init(&bars->d_ready[c], 1);
    for (int k = 0; k < kSeqRing; ++k) bars->seq[k] = ~0ull;
    fence_barrier_init();
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1) tmem_alloc<512>(&bars->tmem_base);
  if constexpr (kResid) {
    const uint4* src = reinterpret_cast<const uint4*>(kPn ? m.wimg_pn : m.wimg);
    uint4* dst = reinterpret_cast<uint4*>(sW);
    for (int k = threadIdx.x; k < kImgBytes / 16; k += kThreads) dst[k] = src[k];
    // "ones" operand of the bias k-step: row r, k-octet 0 = (1, 0, ..., 0); k-octet 1 = 0
    uint4* ones = reinterpret_cast<uint4*>(sOnes);
    for (int k = threadIdx.x; k < kOnesBytes / 16; k += kThreads) ones[k] = make_uint4(k < 128 ? 0x00003F80u : 0u, 0u, 0u, 0u);
    fence_proxy_async_smem();  // generic-proxy writes -> visible to the tensor-core (async) proxy
  }
  if (warp == 2) {
    // prefix[p] = first work index of patch p: warp scan, 32 patches per sweep (the per-patch counts
    // and sizes are global loads: issued in parallel instead of one dependent chain by one thread)
    int carry = 0;
    for (int p0 = 0; p0 < m.n_patches; p0 += 32) {
      const int p = p0 + lane;
      int v = 0;
      if (p < m.n_patches) {
        const PatchInfo pi = m.patch[p];
        PTab t;
        t.cnt = m.count[p], t.off = pi.off, t.n = pi.n, t.uoff = pi.uoff;
        t.tiles = (t.cnt + TE - 1) / TE;
        int nmb = (pi.n + BM - 1) / BM;
        if constexpr (kPair) nmb = (nmb + 1) / 2;  // pairs of node blocks
        t.G = max(1, min(t.tiles, m.group_bytes / (BN * 2 * max(pi.n, 1))));
        t.GN = max(t.G * nmb, 1);
        reinterpret_cast<PTab*>(prefix + m.n_patches + 1)[p] = t;
        v = t.tiles * nmb;
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
  tc_fence_before();
  __syncthreads();
  if constexpr (kPair) cluster_sync();  // the peer's barriers are initialised before anything is sent to them
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (warp == 0) {
    reg_dealloc<TL::kRegsCtrl>();
    if constexpr (kProp)
    // ------------------------------------------------------------------ TMA producer
    // (the whole warp runs the loop so that every operand stays warp-uniform; one elected lane issues)
    {
      int pcur = 0, stage = 0;
      uint32_t ph = 0;
      Item it, nx;
      int w = w_first, n_item = 0;
      bool have = decode_item<kGrouped, TE>(prefix, m.n_patches, w, rank, pcur, it);
      uint32_t km = 0;
      if constexpr (kGrouped) km = have ? load_tile_kbmask(m, it, lane) : 0u;
      while (have) {
        // static order: the next item and (large patches) its k-block mask, requested before this item's k-blocks
        // are streamed
        int wn = w + w_step;
        bool have_n = false;
        uint32_t kmn = 0;
        if constexpr (!kDyn) {
          have_n = decode_item<kGrouped, TE>(prefix, m.n_patches, wn, rank, pcur, nx);
          if constexpr (kGrouped) kmn = have_n ? load_tile_kbmask(m, nx, lane) : 0u;
        }
        const int nkb = (it.n + BK - 1) / BK;
        auto load_kb = [&](const int kb) {
          mbar_wait(&bars->empty[stage], ph ^ 1);
          if (elect_one()) {
            mbar_arrive_expect_tx(&bars->full[stage], A_STAGE + B_STAGE);
            tma_load_2d(sA + stage * A_STAGE, &tmA, &bars->full[stage], kb * BK, it.off + it.mb * BM);
            if constexpr (kPair)  // tmB's box is half a tile: rows [rank BN/2, +BN/2) of the tile, into both CTAs
              tma_load_2d_multicast(sB + stage * B_STAGE + rank * (B_STAGE / 2), &tmB, &bars->full[stage], it.uoff + kb * BK,
                                    it.tile * BN + rank * (BN / 2), kPairMask);
            else
              tma_load_2d(sB + stage * B_STAGE, &tmB, &bars->full[stage], it.uoff + kb * BK, it.tile * BN);
          }
          __syncwarp();
          if (++stage == kStages) stage = 0, ph ^= 1;
        };
        if constexpr (kGrouped) {
          KbIter ki;
          ki.init(km, nkb);
          for (int kb = ki.next(); kb >= 0; kb = ki.next()) load_kb(kb);
        } else {
          for (int kb = 0; kb < nkb; ++kb) load_kb(kb);
        }
        if constexpr (kDyn) {
          // dynamic order: the next item is claimed as late as possible -- when this one is streamed -- so that few
          // items are bound to a CTA when the counter runs out; this warp is an item ahead of the chains and can wait
          int claimed = 0;
          if (lane == 0) {
            claimed = (int)gridDim.x + atomicAdd(m.wq, 1);
            *reinterpret_cast<volatile unsigned long long*>(&bars->seq[(n_item + 1) & (kSeqRing - 1)]) =
                ((unsigned long long)(uint32_t)(n_item + 1) << 32) | (uint32_t)claimed;
          }
          wn = __shfl_sync(0xffffffffu, claimed, 0);
          have_n = decode_item<kGrouped, TE>(prefix, m.n_patches, wn, rank, pcur, nx);
        }
        it = nx, km = kmn, have = have_n, w = wn, ++n_item;
      }
    }
  } else if (warp == 1) {
    reg_dealloc<TL::kRegsCtrl>();
    if constexpr (kProp)
    // ------------------------------------------------------------------ MMA issuer
    // Warp-uniform control flow; tcgen05.mma / tcgen05.commit are issued by one elected lane.
    {
      constexpr uint32_t idesc_prop = make_idesc_bf16(BM, BN);
      int pcur = 0, stage = 0, k_item = 0;
      uint32_t ph = 0;
      Item it, nx;
      int w = w_first;
      bool have = decode_item<kGrouped, TE>(prefix, m.n_patches, w, rank, pcur, it);
      uint32_t km = 0;
      if constexpr (kGrouped) km = have ? load_tile_kbmask(m, it, lane) : 0u;
      while (have) {
        int wn = w + w_step;
        bool have_n = false;
        uint32_t kmn = 0;
        if constexpr (!kDyn) {
          have_n = decode_item<kGrouped, TE>(prefix, m.n_patches, wn, rank, pcur, nx);
          if constexpr (kGrouped) kmn = have_n ? load_tile_kbmask(m, nx, lane) : 0u;
        }
        const int nkb = (it.n + BK - 1) / BK;
        const int b = k_item & 1;
        mbar_wait(&bars->acc_empty[b], ((k_item >> 1) & 1) ^ 1);  // the epilogue has fetched item k_item - 2
        tc_fence_after();
        bool first = true;
        auto mma_kb = [&](const bool last) {
          mbar_wait(&bars->full[stage], ph);
          tc_fence_after();
          const uint64_t dA = make_desc(smem_u32(sA + stage * A_STAGE), 16, 1024, kLayoutSw128);
          const uint64_t dB = make_desc(smem_u32(sB + stage * B_STAGE), 16, 1024, kLayoutSw128);
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < BK / 16; ++k)
              mma_ss(tmem + b * BN, dA + 2 * k, dB + 2 * k, idesc_prop, (!first || k != 0) ? 1u : 0u);
            if constexpr (kPair) tc_commit_multicast(&bars->empty[stage], kPairMask);
            else tc_commit(&bars->empty[stage]);
            if (last) tc_commit(&bars->acc_full[b]);
          }
          __syncwarp();
          first = false;
          if (++stage == kStages) stage = 0, ph ^= 1;
        };
        if constexpr (kGrouped) {
          KbIter ki;  // (every slot of an item is a contacting pair: at least one k-block is active)
          ki.init(km, nkb);
          for (int kb = ki.next(), kb_next; kb >= 0; kb = kb_next) {
            kb_next = ki.next();
            mma_kb(kb_next < 0);
          }
        } else {
          for (int kb = 0; kb < nkb; ++kb) mma_kb(kb == nkb - 1);
        }
        if constexpr (kDyn) {  // (published once the TMA warp has streamed this item: not before the k-blocks are consumed)
          wn = seq_w(k_item + 1);
          have_n = decode_item<kGrouped, TE>(prefix, m.n_patches, wn, rank, pcur, nx);
        }
        it = nx, km = kmn, have = have_n, w = wn, ++k_item;
      }
    }
  } else if (warp < 4) {
    reg_dealloc<TL::kRegsCtrl>();
    // ------------------------------------------------------------------ zero-fill of the contact-free rows
    // Two warps per CTA walk the (env, patch) flags and zero-fill one run of contact-free patches at a time,
    // with a pause in between: 190 MB of stores (cfg 3) trickle out next to the MUFU-bound work instead of
    // saturating HBM for 30 us at the start of the kernel.
    if constexpr (kFill) {
      ZeroFill zf;
      zf.init(m, io, blockIdx.x * 2 + (warp - 2), gridDim.x * 2);
      while (zf.step(m, io, lane)) __nanosleep(1000);
    }
  } else {
    reg_alloc<TL::kRegsEpi>();
    // ------------------------------------------------------------------ epilogue (thread = node)
    const int c = (warp - 4) >> 2, q = warp & 3;  // chain, TMEM lane quarter (= warp % 4)
    const uint32_t lane_base = (uint32_t)q * 32;
    const uint32_t trow = tmem + (lane_base << 16);
    const uint32_t tD = trow + TL::COL_D0 + 64 * c;
    const int row = lane_base + lane;
    uint64_t* d_ready = &bars->d_ready[c];
    const uint32_t sA1 = smem_u32(sAop + c * kAopBytes), sA2 = sA1;  // (one region, see kAopBytes)
    const uint32_t sRow1 = sA1 + row * 16, sRow2 = sA2 + row * 16;  // this thread's 16-byte slot in k-octet 0
    uint32_t d_ph = 0;

    // ---- the chain's MMA issue: operand stores of all four warps -> async proxy, D reads done, then one lane
    auto issue_layer = [&](const int layer) {
      if constexpr (kResid) {
        fence_proxy_async_smem();
        tc_fence_before();
        // only the issuing warp has to wait for the chain; the other three arrive and go on (their next stop is the
        // layer's d_ready).  The issue costs its warp a few hundred cycles (the MMAs queue behind the MUFU traffic of
        // its sub-partition), so the role is spread over the sub-partitions: chain c issues from its warp c % 4.
        if (q != (c & 3)) {
          named_bar_arrive(1 + c, 128);
        } else {
          named_bar_sync(1 + c, 128);
          tc_fence_after();
          if (elect_one()) {
            constexpr uint32_t idesc_h = make_idesc_bf16(BM, 64);
            const uint32_t tDc = tmem + TL::COL_D0 + 64 * c;
            if (layer == 0) {
              mma_ss(tDc, make_desc(sA1, kAopLBO, kAopSBO, kLayoutNone), make_desc(smem_u32(sW), 1024, 128, kLayoutNone), idesc_h, 0);
            } else {
              // weight image: [64 x 16] | [64 x 80] | PointNet decoder: [64 x 80]
              const uint64_t dWl = make_desc(smem_u32(sW + kW1ImgBytes + (layer - 1) * kW2ImgBytes), 1024, 128, kLayoutNone);
              const uint64_t dA2 = make_desc(sA2, kAopLBO, kAopSBO, kLayoutNone);
#pragma unroll
              for (int k = 0; k < 4; ++k) mma_ss(tDc, dA2 + (uint64_t)(k * (4096 >> 4)), dWl + (uint64_t)(k * (2048 >> 4)), idesc_h, k != 0);
              mma_ss(tDc, make_desc(smem_u32(sOnes), kAopLBO, kAopSBO, kLayoutNone), dWl + (uint64_t)(4 * (2048 >> 4)), idesc_h, 1);
            }
            tc_commit(d_ready);
          }
          __syncwarp();
        }
      }
    };

    // ---- cursor over the units of this chain: unit q of the CTA's item stream belongs to chain q mod NC
    int cw = w_first, ck = 0, cel = c, pcur = 0;  // work index, item ordinal, unit within the item
    Item it;
    bool live = decode_item<kGrouped, TE>(prefix, m.n_patches, cw, rank, pcur, it);
    int it_g = 0;           // this thread's node of the item (row clamped into the patch) and whether the row is inside
    bool it_valid = false;
    auto item_setup = [&]() {
      const int li = it.mb * BM + row;
      it_valid = li < it.n;
      it_g = it.off + (it_valid ? li : 0);
    };
    if (live) item_setup();
    auto enter_item = [&]() {  // the propagation GEMM of item ck must have landed before its accumulator is touched
      if constexpr (kProp) {
        mbar_wait(&bars->acc_full[ck & 1], (ck >> 1) & 1);
        tc_fence_after();
      }
    };
    auto leave_item = [&]() {  // all of this warp's u_lin fetches from item ck are complete
      if constexpr (kProp) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->acc_empty[ck & 1]);
      }
    };
    auto skip_to_unit = [&]() {  // cel may point past the item: walk on until it names a unit (or the stream ends)
      while (live && cel >= it.cnt) {
        cel -= it.cnt;
        leave_item();
        ++ck;
        cw = kDyn ? seq_w(ck) : cw + w_step;
        live = decode_item<kGrouped, TE>(prefix, m.n_patches, cw, rank, pcur, it);
        if (live) item_setup(), enter_item();
      }
    };
    if (live) enter_item();
    skip_to_unit();

    struct Unit {
      int g, env, pslot;     // node (mesh index; row clamped into the patch), environment, patch * max_envs + position in the patch's contact list
      bool valid;            // row inside the patch
      float ux, uy, uz, dl;  // u_lin, delta
      uint4 a1c;             // constant part of the layer-1 operand of the node (bf16: px | py pz | nx ny | nz 1)
    };
    // requests only; tc_wait_ld() follows.  delta is loaded later (load_delta) so that no load waits on `env`.
    auto fetch_unit = [&](Unit& u, uint32_t (&ur)[4]) {
      u.valid = it_valid;
      u.g = it_g;
      const int slot = it.tile * TE + cel;
      u.pslot = it.p * m.max_envs + slot;
      u.env = __ldg(m.envlist + u.pslot);
      if constexpr (kResid) u.a1c = __ldg(m.a1c + u.g);
      if constexpr (kProp) {
        tmem_ld4(trow + (ck & 1) * BN + 3 * cel, ur);
      } else if constexpr (kMode == kModePnEncode) {
        ur[0] = ur[1] = ur[2] = ur[3] = 0;  // the encoder pass has no propagation
      } else {
        // Omega U_a: sum over the active nodes of this (env, patch); entry loads are warp-uniform
        // (broadcast), K row j is read coalesced over the rows i of the warp
        const int cnt = m.acount[u.pslot];
        const ActiveEntry* __restrict__ al = m.alist + (int64_t)slot * m.ldu + it.off;
        const __nv_bfloat16* __restrict__ kcol = m.k16 + (int64_t)it.off * m.kw + (u.g - it.off);
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
            for (int qq = 0; qq < kGatherDepth; ++qq)
              kv[qq] = __bfloat162float(kcol[(int64_t)__float_as_int(stage[q0 + qq].w) * m.kw]);
#pragma unroll
            for (int qq = 0; qq < kGatherDepth; ++qq) {
              const float4 en = stage[q0 + qq];
              ax = fmaf(kv[qq], en.x, ax), ay = fmaf(kv[qq], en.y, ay), az = fmaf(kv[qq], en.z, az);
            }
          }
        }
        ur[0] = __float_as_uint(ax), ur[1] = __float_as_uint(ay), ur[2] = __float_as_uint(az), ur[3] = 0;
      }
    };
    auto load_delta = [&](Unit& u) { u.dl = u.valid ? m.delta[(int64_t)u.env * m.n_nodes + u.g] : 0.0f; };
    // layer-1 operand [u_lin(3) | u^(3), p(3), n(3), 1, 0 x 6] of the unit -> shared memory, then the chain's MMA
    auto request_layer1 = [&](Unit& u, const uint32_t (&ur)[4]) {
      u.ux = __uint_as_float(ur[0]), u.uy = __uint_as_float(ur[1]), u.uz = __uint_as_float(ur[2]);
      if constexpr (kResid) {
        uint32_t w0, w1;
        if constexpr (kPn) {  // PointNet encoder input: u^ = -delta n of the node itself
          const float4 nn = m.nrm4[u.g];
          w0 = pack_bf16(-u.dl * nn.x, -u.dl * nn.y);
          w1 = (pack_bf16(-u.dl * nn.z, 0.0f) & 0x0000ffffu) | (u.a1c.x << 16);
        } else {
          w0 = pack_bf16(u.ux, u.uy);
          w1 = (pack_bf16(u.uz, 0.0f) & 0x0000ffffu) | (u.a1c.x << 16);
        }
        st_shared_v4(sRow1, w0, w1, u.a1c.y, u.a1c.z);
        st_shared_v4(sRow1 + kAopLBO, u.a1c.w, 0u, 0u, 0u);
        issue_layer(0);
      }
    };

    Unit cur, nxt;
    if (live) {
      uint32_t ur[4];
      fetch_unit(cur, ur);
      tc_wait_ld();
      if constexpr (kPn) load_delta(cur);
      request_layer1(cur, ur);
    }
    while (live) {
      float rx = 0.f, ry = 0.f, rz = 0.f;
      uint32_t un[4] = {0, 0, 0, 0};
      bool more = false;
      // the next unit of this chain: fetched behind the last layer's round trip; it may sit in a later item
      auto prefetch_next = [&]() {
        cel += NC;
        skip_to_unit();
        more = live;
        if (more) fetch_unit(nxt, un);
        if constexpr (!kPn) load_delta(cur);  // consumed when the unit is stored
      };
      if constexpr (kResid) {
        // One SiLU granule per MMA layer.  The inner granules write the next layer's bf16 operand to shared
        // memory (a thread's eight consecutive activations are one 16-byte row of a core matrix: a warp
        // stores 512 contiguous bytes) and request the layer; the last one keeps its fp32 outputs in
        // registers and applies the 3 x 64 output layer on the FMA pipe (per-node MLP / decoder) or
        // max-pools them over the rows (encoder).  The decoder's last layer adds the per-(env, patch)
        // vector c (halved like the weights).
        uint32_t h[32];
#pragma unroll 1
        for (int layer = 0; layer < kLayers - 1; ++layer) {
          mbar_wait(d_ready, d_ph), d_ph ^= 1;
          tc_fence_after();
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            tmem_ld32(tD + 32 * half, h);
            tc_wait_ld();
            uint32_t packed[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              // D holds x/2 (0.5 folded into the weights): silu(x) = x*sigmoid(x) = h + h*tanh(h)
              float y0, y1;
              unpack_f32x2(silu_half_x2(__uint_as_float(h[2 * k]), __uint_as_float(h[2 * k + 1])), y0, y1);
              packed[k] = pack_bf16(y0, y1);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j)
              st_shared_v4(sRow2 + (4 * half + j) * kAopLBO, packed[4 * j], packed[4 * j + 1], packed[4 * j + 2], packed[4 * j + 3]);
          }
          issue_layer(layer + 1);
        }
        // ---- last granule
        prefetch_next();  // overlaps the last layer's round trip
        mbar_wait(d_ready, d_ph), d_ph ^= 1;
        tc_fence_after();
        if constexpr (kMode == kModePnEncode) {
          uint32_t pool0 = 0, pool1 = 0;  // lane l: max keys of hidden columns l and 32 + l
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            tmem_ld32(tD + 32 * half, h);
            tc_wait_ld();
#pragma unroll
            for (int k = 0; k < 32; ++k) {
              // column max over the warp's 32 rows.  silu >= -0.279, so 1 + silu is a positive
              // float whose bit pattern orders like the value; 0 = no row
              const float h0 = __uint_as_float(h[k]);
              const float y0 = fmaf(h0, tanh_approx(h0), h0);
              const uint32_t k0 = cur.valid ? __float_as_uint(1.0f + y0) : 0u;
              const uint32_t m0 = __reduce_max_sync(0xffffffffu, k0);
              if (lane == k) (half ? pool1 : pool0) = m0;
            }
          }
          uint32_t* gm = m.gmax + (int64_t)cur.pslot * 64;
          atomicMax(gm + lane, pool0);
          atomicMax(gm + 32 + lane, pool1);
        } else {
          const float4* cv = nullptr;
          if constexpr (kMode == kModePnDecode)
            cv = reinterpret_cast<const float4*>(m.cvec + (int64_t)cur.pslot * 64);
          // even / odd hidden columns accumulate in the two halves of packed fp32x2 registers
          uint64_t ax = pack_f32x2(m.wout[192], 0.f), ay = pack_f32x2(m.wout[193], 0.f), az = pack_f32x2(m.wout[194], 0.f);
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            tmem_ld32(tD + 32 * half, h);
            tc_wait_ld();
            // D is in registers: the next unit's layer-1 operand and request go out now, its tensor-core round trip
            // runs under the second half's SiLUs and the output layer
            if (half == 1 && more) {
              if constexpr (kPn) load_delta(nxt);
              request_layer1(nxt, un);
            }
#pragma unroll
            for (int k4 = 0; k4 < 8; ++k4) {
              float4 c4 = make_float4(0.f, 0.f, 0.f, 0.f);
              if constexpr (kMode == kModePnDecode) c4 = __ldg(cv + half * 8 + k4);
              const float cc[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
              for (int qq = 0; qq < 4; qq += 2) {
                const int k = 4 * k4 + qq, col = 32 * half + k;
                float h0 = __uint_as_float(h[k]), h1 = __uint_as_float(h[k + 1]);
                if constexpr (kMode == kModePnDecode) h0 += cc[qq], h1 += cc[qq + 1];
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
      } else {
        prefetch_next();
        tc_wait_ld();
      }
      // the next unit's layer-1 operand and request: D is free once all four warps have read the last layer
      // (the chain barrier inside the request)
      if (more && (kMode == kModeNone || kMode == kModePnEncode)) {
        if constexpr (kPn) load_delta(nxt);
        request_layer1(nxt, un);
      }
      if (cur.valid && kMode != kModePnEncode) {  // S4: mask M_p + combine (Eq. 2); active rows keep u^ = -delta n in fp32
        const float lin = m.residual_only ? 0.0f : 1.0f;  // Table II ablation "Residual Network Only"
        float ox = fmaf(lin, cur.ux, rx), oy = fmaf(lin, cur.uy, ry), oz = fmaf(lin, cur.uz, rz);
        if (cur.dl > 0.0f && m.active_mode == ETAC_ACTIVE_PASSTHROUGH) {
          // (loaded for the few active rows instead of held in three registers through the MLP)
          const float4 nn = m.nrm4[cur.g];
          ox = -cur.dl * nn.x, oy = -cur.dl * nn.y, oz = -cur.dl * nn.z;
        }
        store_out3<kOutBf16 ? ETAC_OUT_BF16 : ETAC_OUT_F32>(io, cur.env, cur.g, ox, oy, oz);
        if (io.analytic_out) {
          float* a = io.analytic_out + ((int64_t)cur.env * m.n_nodes + cur.g) * 3;
          __stcs(a, cur.ux), __stcs(a + 1, cur.uy), __stcs(a + 2, cur.uz);
        }
      }
      cur = nxt;
      live = more;
    }
  }
  tc_fence_before();
  __syncthreads();
  if constexpr (kDyn) {
    // every claim of this CTA has returned; the last CTA to get here leaves the counters at zero for the next launch
    if (threadIdx.x == 0 && atomicAdd(m.wq + 1, 1) == (int)gridDim.x - 1) m.wq[0] = 0, m.wq[1] = 0;
  }
  if constexpr (kPair) cluster_sync();  // the peer's last commits arrive on this CTA's barriers
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<512>(tmem);
  }
}

// c_(e,p) of the PointNet decoder: g = max-pooled features (keys = bits of 1 + f), g' = silu(G1 g + g1)
// ("further encoded by another MLP"), c = D1[:, 64:128] g' + d1, stored halved like
// the decoder weights.  A 64-thread CTA stages the two transposed 64 x 64 matrices in shared
// memory once and walks kPnSlots contact-list slots of one patch.
constexpr int kPnSlots = 32, kPnGroups = 4, kPnPer = kPnSlots / kPnGroups;  // slots per CTA; groups of 64 threads; slots per group
__global__ void __launch_bounds__(64 * kPnGroups) pn_global_kernel(DevModel m) {
  // thread = output k of kPnPer slots held in registers: a weight read from shared memory serves kPnPer FMAs (one
  // output of one slot per thread would be bound by two shared-memory loads per FMA)
  const int p = blockIdx.y, k = threadIdx.x & 63, grp = threadIdx.x >> 6;
  const int slot0 = blockIdx.x * kPnSlots, cnt = m.count[p];
  if (slot0 >= cnt) return;
  __shared__ float sG1[64 * 64], sD1[64 * 64];
  __shared__ __align__(16) float g[64][kPnSlots], g2[64][kPnSlots];  // [input j][slot of the CTA]
  const float* G1t = m.pn_f32, *g1 = G1t + 4096, *D1gt = g1 + 64, *d1 = D1gt + 4096;  // both matrices [in][out]
#pragma unroll
  for (int i = 0; i < kPnPer; ++i) {
    const int sl = grp * kPnPer + i, slot = slot0 + sl;
    const uint32_t key = slot < cnt ? m.gmax[((int64_t)p * m.max_envs + slot) * 64 + k] : 0x3f800000u;
    g[k][sl] = __uint_as_float(key) - 1.0f;  // keys are the bit patterns of 1 + f
  }
  for (int i = threadIdx.x; i < 4096; i += 64 * kPnGroups) sG1[i] = G1t[i], sD1[i] = D1gt[i];
  const float bg = g1[k], bd = d1[k];
  __syncthreads();
  float acc[kPnPer];
#pragma unroll
  for (int i = 0; i < kPnPer; ++i) acc[i] = bg;
#pragma unroll 4
  for (int j = 0; j < 64; ++j) {
    const float w = sG1[j * 64 + k];
    const float4 x0 = *reinterpret_cast<const float4*>(&g[j][grp * kPnPer]), x1 = *reinterpret_cast<const float4*>(&g[j][grp * kPnPer + 4]);
    const float x[kPnPer] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
#pragma unroll
    for (int i = 0; i < kPnPer; ++i) acc[i] = fmaf(w, x[i], acc[i]);
  }
#pragma unroll
  for (int i = 0; i < kPnPer; ++i) g2[k][grp * kPnPer + i] = acc[i] / (1.0f + expf(-acc[i]));
  __syncthreads();
#pragma unroll
  for (int i = 0; i < kPnPer; ++i) acc[i] = bd;
#pragma unroll 4
  for (int j = 0; j < 64; ++j) {
    const float w = sD1[j * 64 + k];
    const float4 x0 = *reinterpret_cast<const float4*>(&g2[j][grp * kPnPer]), x1 = *reinterpret_cast<const float4*>(&g2[j][grp * kPnPer + 4]);
    const float x[kPnPer] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
#pragma unroll
    for (int i = 0; i < kPnPer; ++i) acc[i] = fmaf(w, x[i], acc[i]);
  }
#pragma unroll
  for (int i = 0; i < kPnPer; ++i) {
    const int slot = slot0 + grp * kPnPer + i;
    if (slot < cnt) m.cvec[((int64_t)p * m.max_envs + slot) * 64 + k] = 0.5f * acc[i];
  }
}
static_assert(kPnPer == 8, "pn_global_kernel reads a group's inputs as two float4");

template <int kMode, bool kGather, bool kOutBf16, bool kGrouped, int TE>
static cudaError_t set_smem() {
  return cudaFuncSetAttribute(fused_mlp_kernel<kMode, kGather, kOutBf16, kGrouped, TE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              kMaxDynSmem);
}
template <int kMode, bool kGather>
static cudaError_t configure_one() {
  cudaError_t e = set_smem<kMode, kGather, false, false, 16>();
  if (e == cudaSuccess && kMode != kModePnEncode) e = set_smem<kMode, kGather, true, false, 16>();  // the encoder pass writes no displacement
  if constexpr (!kGather && kMode != kModePnEncode) {  // large patches: 32-env tile, grouped item order; dense propagation only
    if (e == cudaSuccess) e = set_smem<kMode, false, false, true, 32>();
    if (e == cudaSuccess) e = set_smem<kMode, false, true, true, 32>();
  }
  return e;
}

cudaError_t fused_configure() {
  cudaError_t e = configure_one<kModeNone, false>();
  if (e == cudaSuccess) e = configure_one<kModeNone, true>();
  if (e == cudaSuccess) e = configure_one<kModePerNode, false>();
  if (e == cudaSuccess) e = configure_one<kModePerNode, true>();
  if (e == cudaSuccess) e = configure_one<kModePnEncode, false>();
  if (e == cudaSuccess) e = configure_one<kModePnDecode, false>();
  if (e == cudaSuccess) e = configure_one<kModePnDecode, true>();
  return e;
}

// the 32-env tile + grouped item order: where a patch's U^ operand (3 bf16 rows of n nodes per env) can exceed the
// L2 share, or a patch is large enough for its propagation GEMM to matter next to the MLP of the item's units
// false: the mesh has too many patches for the kernel's shared-memory tables (checked at create)
bool fused_fits(int n_patches) {
  return fused_smem_bytes<16>(n_patches, kModePnDecode, false, false) <= (size_t)kMaxDynSmem &&
         fused_smem_bytes<16>(n_patches, kModePnDecode, true, false) <= (size_t)kMaxDynSmem &&
         fused_smem_bytes<32>(n_patches, kModePnDecode, false, true) <= (size_t)kMaxDynSmem;
}

bool fused_uses_big_tile(const DevModel& m, int n_envs) {
  return (size_t)n_envs * (size_t)m.max_patch_nodes * 6 > (size_t)m.group_bytes || m.max_patch_nodes >= 2048;
}

// the 32-env instantiation: clusters of two CTAs (an even grid); tmB is the map with the half-tile box (48 rows)
template <int kMode, bool kOutBf16>
static cudaError_t launch_pairs(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB, int grid, size_t smem,
                                cudaStream_t s) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)(grid & ~1)), cfg.blockDim = dim3(Tile<32>::kThreads), cfg.dynamicSmemBytes = smem, cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2, at[0].val.clusterDim.y = 1, at[0].val.clusterDim.z = 1;
  cfg.attrs = at, cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, fused_mlp_kernel<kMode, false, kOutBf16, true, 32>, m, io, tmA, tmB);
}

template <int kMode>
static cudaError_t launch_one(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB, int grid, bool gather,
                              cudaStream_t s) {
  const size_t smem16 = fused_smem_bytes<16>(m.n_patches, kMode, gather, false), smem32 = fused_smem_bytes<32>(m.n_patches, kMode, false, true);
  constexpr int T16 = Tile<16>::kThreads;
  const bool big = !gather && fused_uses_big_tile(m, io.n_envs);
  if constexpr (kMode == kModePnEncode) {
    fused_mlp_kernel<kMode, false, false, false, 16><<<grid, T16, smem16, s>>>(m, io, tmA, tmB);
  } else if (gather) {
    if (io.out_bf16) fused_mlp_kernel<kMode, true, true, false, 16><<<grid, T16, smem16, s>>>(m, io, tmA, tmB);
    else fused_mlp_kernel<kMode, true, false, false, 16><<<grid, T16, smem16, s>>>(m, io, tmA, tmB);
  } else if (big) {
    kbtile_kernel<32><<<dim3((unsigned)((io.n_envs + 31) / 32), (unsigned)m.n_patches), 32, 0, s>>>(m);
    return io.out_bf16 ? launch_pairs<kMode, true>(m, io, tmA, tmB, grid, smem32, s) : launch_pairs<kMode, false>(m, io, tmA, tmB, grid, smem32, s);
  } else {
    if (io.out_bf16) fused_mlp_kernel<kMode, false, true, false, 16><<<grid, T16, smem16, s>>>(m, io, tmA, tmB);
    else fused_mlp_kernel<kMode, false, false, false, 16><<<grid, T16, smem16, s>>>(m, io, tmA, tmB);
  }
  return cudaSuccess;
}

// Launches S2-S4 for the context's residual form; *launches receives the number of kernels.
cudaError_t launch_fused_bf16(const DevModel& m, const StepIO& io, const CUtensorMap& tmA, const CUtensorMap& tmB, int n_sm, bool gather,
                              int* launches, cudaStream_t s) {
  const int grid = n_sm;
  const int n_big = (!gather && fused_uses_big_tile(m, io.n_envs)) ? 1 : 0;  // + kbtile_kernel
  *launches = 1 + n_big;
  cudaError_t e = cudaSuccess;
  if (m.resid == ETAC_RESID_NONE) {
    e = launch_one<kModeNone>(m, io, tmA, tmB, grid, gather, s);
  } else if (m.resid == ETAC_RESID_PERNODE_MLP) {
    e = launch_one<kModePerNode>(m, io, tmA, tmB, grid, gather, s);
  } else {  // ETAC_RESID_POINTNET: encode + max-pool, per-(env, patch) vector, decode
    e = cudaMemsetAsync(m.gmax, 0, sizeof(uint32_t) * 64 * (size_t)m.n_patches * m.max_envs, s);
    if (e != cudaSuccess) return e;
    launch_one<kModePnEncode>(m, io, tmA, tmB, grid, false, s);
    pn_global_kernel<<<dim3((unsigned)((io.n_envs + kPnSlots - 1) / kPnSlots), (unsigned)m.n_patches), 64 * kPnGroups, 0, s>>>(m);
    e = launch_one<kModePnDecode>(m, io, tmA, tmB, grid, gather, s);
    *launches = 3 + n_big;
  }
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace etac

// kernels.cuh — sm_100a device code of the hot path (BASELINE.json north_star subsystem (2)).
//
//   k_unpack   a1+a2 fused: raw word decode, calibration, STABLE digi/error compaction with a
//              single-pass decoupled look-back scan, modDigiStart, input-order check; TMA bulk
//              loads into a shared-memory ring, staged SoA output written by TMA bulk stores.
//   k_cluster  a3+a4 fused: per-module 8-connected components (one warp per pack of small modules:
//              all in registers; per module of 33..256 digis: hash look-up + label equivalence in
//              shared memory; CTA per large module: bitmap + rank look-up + min-index union-find),
//              exact cluster sums, cluster threshold, per-module numbering.
//   k_dense    the large-module path of k_cluster as a kernel of its own (larger shared-memory tiers), used
//              by launches whose modules are large on average.
//   k_finalize event-wide dense cluster numbering, cluster SoA, modClusStart, counters to the host.
//   k_export   exact-size copies of requested outputs into mapped pinned host memory.
//
// Kernels are batch-capable: a launch processes nEv independent events described by EvDesc
// records (one Run-3-like event is ~1000x too small to fill a B200).  The single-event path
// passes its descriptor as a __grid_constant__ kernel parameter (no descriptor upload).
//
// The paper describes no kernel; its only constraint on device code is "no
// assert() in kernel code" (L88): errors are reported through a status word, never trapped.
// Definitions of every quantity: DESIGN.md, readings A1-A14.  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace pixreco {

typedef uint16_t u16;
typedef uint32_t u32;
typedef uint64_t u64;
typedef long long i64;

constexpr u32 kInvalid = 0xFFFFFFFFu;

// ---- unpack kernel geometry ----
constexpr int kUnpackThreads = 256;
constexpr int kTileWords = 8 * kUnpackThreads;                       // 2048: warp w owns words [256w, 256w + 256), lane l word 32j + l of row j
constexpr int kLookBack = 8;                                         // predecessor states per lane and look-back round (256 per round)

// ---- cluster kernel geometry ----
constexpr int kClusterThreads = 256;
constexpr u32 kSmemDigis = 2048;      // modules with more digis use the global workspace tier
constexpr u32 kSmemClusters = 512;    // likewise for per-cluster accumulators
constexpr u32 kDenseDigis = 8192;     // the same tiers of k_dense (two CTAs per SM with their own, larger shared memory)
constexpr u32 kDenseClusters = 512;

// Per-event device counters (lives in the slot's control block, zeroed per acquire).
struct DevCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, pad;
};
// Per-launch control words (zeroed per acquire).
struct LaunchCtl {
  u32 modTicket, modDone;
  u64 tStart;                       // %globaltimer at the start of the acquire's first kernel
  u32 nBig, bigTicket;              // modules handed from k_cluster to k_dense, next one to take
  u32 pad[10];
};
// What the host reads after completion (mapped pinned memory, written by the last block).
struct HostCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, seq;
  u64 tStart, tEnd;                 // %globaltimer: first kernel of the acquire started, this event's counters published
};
__device__ __forceinline__ u64 global_timer() {
  u64 t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// One event of a launch.  The first 128 bytes are all that k_unpack reads: in a batch, one warp-wide
// load brings them into shared memory.
struct EvDesc {
  const u32* words; const u16* adc;
  u32 nWords, tileBase, nTiles, cap;
  // digi SoA [cap] (first six written by k_unpack)
  u16 *module, *row, *col, *adcOut; u32* wordIdx; float* charge;
  // error list [cap]
  u32 *errWord, *errIdx;
  u32* modDigiStart;                // [M+1]
  DevCounters* counters;
  u64* tileState;                   // k_unpack look-back states [nTiles]
  u64 unpackPad;                    // ---- 128 bytes up to here ----
  u32* label; int32_t* clus;
  u32* modClusStart;                // [M+1]
  // cluster SoA [cap]
  u32 *clLabel, *clSize; u16* clModule; float *clCharge, *clRow, *clCol;
  // global workspace tier for large modules [cap] each
  u32 *wsPerm, *wsParent, *wsRoot; int32_t* wsKnum; u32* wsSize; u64 *wsS, *wsSx, *wsSy;
  HostCounters* hostCounters;
  u32* modCount;                    // [M+1] kept clusters per module (k_cluster -> k_finalize)
  u32* grpCount;                    // [ceil(M / 32)] the same summed over groups of kFinMods modules (zeroed per acquire)
  // staged kept clusters: record k of the module with first digi s lives at index s + k [cap]
  double *stS, *stSx, *stSy; u32 *stLabel, *stSize;
};
static_assert(offsetof(EvDesc, label) == 128, "k_unpack's part of the descriptor is one 128-byte line");

struct Geom {
  u32 M, R, C;
  u32 stride;                       // bitmap words per padded row = ceil((C+2)/32)
  u32 bitmapWords;                  // (R+2)*stride + 1
  float pixThr;
  i64 clusThrFixed;                 // llrint(clusThr * 2^14)
  const float2* calib;              // device [M]: (gain, pedestal)
};

// ------------------------------------------------------------------ small helpers
__device__ __forceinline__ u64 ld_state(const u64* p) {
  u64 v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_state(u64* p, u64 v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// state word: [63:62] status (0 none, 1 aggregate, 2 inclusive) | [43:32] max(module)+1 | [31:0] count
constexpr u64 kStAgg = 1ull << 62, kStIncl = 2ull << 62;
__device__ __forceinline__ u64 pack_state(u64 st, u32 cnt, u32 mx1) { return st | ((u64)mx1 << 32) | cnt; }
__device__ __forceinline__ u32 st_status(u64 v) { return (u32)(v >> 62); }
__device__ __forceinline__ u32 st_count(u64 v) { return (u32)v; }
__device__ __forceinline__ u32 st_max1(u64 v) { return (u32)(v >> 32) & 0xFFFu; }

__device__ __forceinline__ u32 warp_incl_scan(u32 v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    u32 t = __shfl_up_sync(0xFFFFFFFFu, v, d);
    if (lane >= d) v += t;
  }
  return v;
}

// Block-wide exclusive scan of one value per thread (blockDim = 32 * kWarps); returns exclusive prefix,
// *total = block sum.  `sw` is kWarps words of shared scratch.  Contains two __syncthreads.
template <int kWarps = 8>
__device__ __forceinline__ u32 block_excl_scan(u32 v, u32* sw, u32* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  u32 incl = warp_incl_scan(v, lane);
  __syncthreads();                                   // protect sw against the previous use
  if (lane == 31) sw[warp] = incl;
  __syncthreads();
  u32 base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < kWarps; ++w) {
    u32 s = sw[w];
    if (w < warp) base += s;
    tot += s;
  }
  *total = tot;
  return base + incl - v;
}

// Decoupled look-back by ONE warp, split in two so that its latency hides behind other work:
// lookback_issue puts the first round's state loads in flight (lane l reads kLookBack predecessors,
// 32 * kLookBack tiles per round); lookback_resolve consumes them, spins on predecessors that had
// not published yet, and goes further back if no inclusive state was among them.  Returns in all
// lanes the combined (count, max module + 1) of all predecessors in [0, self).
__device__ __forceinline__ void lookback_issue(const u64* state, int self, u32 lane, u64 (&v)[kLookBack]) {
#pragma unroll
  for (int k = 0; k < kLookBack; ++k) {
    const int idx = self - 1 - 32 * k - (int)lane;
    v[k] = idx >= 0 ? ld_state(state + idx) : kStIncl;     // virtual zero inclusive before tile 0
  }
}
__device__ __forceinline__ void lookback_resolve(const u64* state, int self, u32 lane, u64 (&v)[kLookBack], u32* cnt, u32* mx1) {
  u32 c = 0, m = 0;
  int look = self - 1;
  for (;;) {                                               // warp-uniform
    bool found = false;
#pragma unroll
    for (int k = 0; k < kLookBack; ++k) {
      if (!found) {
        const int idx = look - 32 * k - (int)lane;
        while (st_status(v[k]) == 0) v[k] = ld_state(state + idx);   // predecessor has not published yet
        const u32 inclMask = __ballot_sync(0xFFFFFFFFu, st_status(v[k]) == 2);
        const u32 upto = inclMask ? (u32)__ffs((int)inclMask) - 1u : 31u;
        c += __reduce_add_sync(0xFFFFFFFFu, lane <= upto ? st_count(v[k]) : 0u);
        m = max(m, __reduce_max_sync(0xFFFFFFFFu, lane <= upto ? st_max1(v[k]) : 0u));
        found = inclMask != 0u;
      }
    }
    if (found) break;
    look -= 32 * kLookBack;
#pragma unroll
    for (int k = 0; k < kLookBack; ++k) {
      const int idx = look - 32 * k - (int)lane;
      v[k] = idx >= 0 ? ld_state(state + idx) : kStIncl;
    }
  }
  *cnt = c; *mx1 = m;
}

// ================================================================== k_unpack (a1 + a2)
// Persistent CTAs; CTA b takes tiles b, b + gridDim.x, ... of the launch (a tile = kTileWords
// consecutive words of one event; the grid never exceeds what is co-resident, because the
// look-back reads states published by CTAs that must be running).  "Local tile k" below is the
// k-th tile of this CTA.  Per iteration i the CTA does, with two barriers:
//   load    (end of iteration i)  one thread issues TMA bulk copies (cp.async.bulk, completion on an
//           mbarrier) of tile i + kRawSlots into the ring slot tile i just vacated: raw words and
//           ADC values reach shared memory without passing through registers
//   count   tile i + kCountAhead: validity (A2, A3) of every word, one ballot per 32 words kept in
//           shared memory, per-warp digi counts; the tile's aggregate (count, max module + 1) is
//           PUBLISHED kCountAhead iterations before the tile is written, so when a successor looks
//           back, the aggregate has long been there: no CTA waits for the progress of another one
//   scatter tile i: its event-global digi offset g0 is known (look-back resolved in iteration
//           i - 1).  Warp w owns words [256w, 256w + 256) of the tile, lane l word 32j + l of row j:
//           position = g0 + warp prefix + row prefix + popc(ballot below lane).  The digi is stored
//           in FINAL form (module,row,col,adc u16; wordIdx u32; charge f32 = fmaf, A7) into six
//           shared-memory arrays at index 8 + (g0 & 7) + position, i.e. with the 16-byte phase of
//           its global destination; error words (rare) go straight to global memory
//   look-back (warp 0) for tile i + 1: loads issued before the scatter, resolved after it
//   store   one thread issues six TMA bulk stores of the 16-byte-aligned middle of the staged
//           arrays; sixteen lanes store the up-to-7 head and tail elements; all threads scan the
//           staged module array for module boundaries (modDigiStart) and order violations (A5)
// Algorithmic HBM bytes per event: 6W read + 16D (digi SoA incl. charge) + 8E written.
constexpr int kUnpackCtasPerSM = 2;
constexpr int kRawSlots = 4;                      // raw tiles in the shared-memory ring
constexpr int kCountAhead = 2;                    // a tile is counted this many iterations before it is written
constexpr int kDescRing = 8;                      // descriptor ring (batch), power of two >= kRawSlots + 2
constexpr u32 kStageElems = kTileWords + 32;      // 8 front pad + phase (< 8) + tile, multiple of 8
static_assert(kCountAhead >= 1 && kCountAhead <= kRawSlots - 2, "a raw tile needs a full iteration to arrive before it is counted");
static_assert(kRawSlots + 2 <= kDescRing, "descriptor ring too small");

struct __align__(128) UnpackShared {
  u32 words[kRawSlots][kTileWords];               // raw ring (TMA destination)
  u16 adc[kRawSlots][kTileWords];
  u16 sModule[kStageElems], sRow[kStageElems], sCol[kStageElems], sAdc[kStageElems];   // staging (TMA source)
  u32 sWordIdx[kStageElems];
  float sCharge[kStageElems];
  u64 full[kRawSlots];                            // mbarriers: raw slot filled
  u32 bal[kRawSlots][8][8];                       // [slot][warp][row] validity ballots
  u32 wcnt[kRawSlots][8], wmax[kRawSlots][8];     // per warp: digis, max(module)+1
  u32 g0[2], carry1[2];                           // look-back result of local tile k at [k & 1]
  u32 desc[kDescRing][32];                        // batch: first 128 bytes of the tiles' event descriptors
};

__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* bar, u32 count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, u32 bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, u32 parity) {
  u32 ok;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void bulk_load(void* dstSmem, const void* srcGlobal, u32 bytes, u64* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dstSmem)), "l"(__cvta_generic_to_global(srcGlobal)), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dstGlobal, const void* srcSmem, u32 bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               ::"l"(__cvta_generic_to_global(dstGlobal)), "r"(smem_u32(srcSmem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

#ifdef PIXRECO_TRACE
__device__ unsigned long long g_trace[1024 * 32];
#define TR_T(v) long long v; asm volatile("mov.u64 %0, %%clock64;" : "=l"(v) :: "memory")
#define TR_ADD(slot, t0) do { long long t1_; asm volatile("mov.u64 %0, %%clock64;" : "=l"(t1_) :: "memory"); trAcc[slot] += (unsigned long long)(t1_ - (t0)); } while (0)
#else
#define TR_T(v)
#define TR_ADD(slot, t0)
#endif
template <bool kSingle>
__global__ void __launch_bounds__(kUnpackThreads + 64, kUnpackCtasPerSM)
k_unpack(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, const u16* __restrict__ tileEvent,
         u32 totalTiles, LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  extern __shared__ __align__(128) unsigned char unpackSmem[];
  UnpackShared& sh = *reinterpret_cast<UnpackShared*>(unpackSmem);
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, lt = (1u << lane) - 1u, G = gridDim.x;
  const bool ctl = warp == 8u, scn = warp == 9u;             // warps 0..7 work on words; warp 8 drives the TMA; warp 9 publishes and looks back
  const u32 first = blockIdx.x;
  if (first >= totalTiles) return;
  if (first == 0 && tid == 0) lc->tStart = global_timer();
#ifdef PIXRECO_TRACE
  unsigned long long trAcc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long trStart = clock64();
#endif
  const int nLocal = (int)((totalTiles - first + G - 1u) / G);
  const u32 limM = g.M, limR = g.R << 12, limC = g.C << 3;
  auto desc_of = [&](int k) -> const EvDesc& {
    return kSingle ? single : *reinterpret_cast<const EvDesc*>(sh.desc[k & (kDescRing - 1)]);
  };
  // ---- load of local tile k into its ring slot, by the control warp: TMA for the 16-byte multiple, lanes for the tail
  auto issue_load = [&](int k) {
    const EvDesc& e = desc_of(k);
    const u32 T0 = (first + (u32)k * G - e.tileBase) * (u32)kTileWords, W = e.nWords;
    const u32 nIn = W > T0 ? min(W - T0, (u32)kTileWords) : 0u, slot = (u32)k % kRawSlots;
    const u32 n4 = nIn & ~3u, n8 = nIn & ~7u;
    if (lane == 0) {
      mbar_expect_tx(&sh.full[slot], n4 * 4u + n8 * 2u);
      if (n4) bulk_load(sh.words[slot], e.words + T0, n4 * 4u, &sh.full[slot]);
      if (n8) bulk_load(sh.adc[slot], e.adc + T0, n8 * 2u, &sh.full[slot]);
    }
    if (lane < nIn - n4) sh.words[slot][n4 + lane] = __ldcs(e.words + T0 + n4 + lane);
    if (lane < nIn - n8) sh.adc[slot][n8 + lane] = __ldcs(e.adc + T0 + n8 + lane);
  };

  // ---- prologue: barriers, the first descriptors, the first loads
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kRawSlots; ++s) mbar_init(&sh.full[s], 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  u32 eNext = 0;                                               // batch, control warp: event of local tile i + kRawSlots + 1
  if (!kSingle) {
    if ((int)warp <= kRawSlots && (int)warp < nLocal)
      sh.desc[warp][lane] = __ldg(reinterpret_cast<const u32*>(batch + tileEvent[first + warp * G]) + lane);
    if (ctl && kRawSlots + 1 < nLocal) eNext = tileEvent[first + (u32)(kRawSlots + 1) * G];
  }
  __syncthreads();
  if (ctl)
    for (int k = 0; k < kRawSlots && k < nLocal; ++k) issue_load(k);
  __syncthreads();

  for (int i = -kCountAhead; i < nLocal; ++i) {
    const int kc = i + kCountAhead, kl = i + 1, kd = i + kRawSlots + 1;
    u32 dword = 0, eN2 = 0, tl = 0;
    u64 lb[kLookBack];
    if (ctl) {
      // batch: descriptor of local tile i + kRawSlots + 1 in flight until the end of the iteration
      if (!kSingle && i >= 0) {
        if (kd < nLocal) dword = __ldg(reinterpret_cast<const u32*>(batch + eNext) + lane);
        if (kd + 1 < nLocal) eN2 = tileEvent[first + (u32)(kd + 1) * G];
      }
      { TR_T(t0); if (lane == 0 && i > 0) bulk_wait_read(); TR_ADD(0, t0); }   // the staging arrays are free again
    } else if (!scn && kc < nLocal) {
      // ---- count: local tile i + kCountAhead
      const EvDesc& e = desc_of(kc);
      const u32 T0 = (first + (u32)kc * G - e.tileBase) * (u32)kTileWords, W = e.nWords;
      const u32 nIn = W > T0 ? min(W - T0, (u32)kTileWords) : 0u, slot = (u32)kc % kRawSlots;
      { TR_T(t0); mbar_wait(&sh.full[slot], ((u32)kc / kRawSlots) & 1u); if (warp == 0) TR_ADD(1, t0); }
      const u32* wseg = sh.words[slot] + 256u * warp + lane;
      u32 cnt = 0, mx = 0, myb = 0;
      const u32 inWarp = nIn > 256u * warp ? nIn - 256u * warp : 0u;      // words of this warp's segment that exist
      if (inWarp >= 256u) {                                    // the common case: no range test per word
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const u32 x = wseg[32 * j];
          const bool ok = (x >> 20) < limM && (x & 0xFF000u) < limR && (x & 0xFF8u) < limC;
          const u32 b = __ballot_sync(0xFFFFFFFFu, ok);
          cnt += (u32)__popc(b);
          if (ok) mx = max(mx, x);                             // a digi's word has bit 31 clear: max word = max module
          if ((int)lane == j) myb = b;
        }
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const u32 x = wseg[32 * j];
          const bool ok = (x >> 20) < limM && (x & 0xFF000u) < limR && (x & 0xFF8u) < limC && 32u * j + lane < inWarp;
          const u32 b = __ballot_sync(0xFFFFFFFFu, ok);
          cnt += (u32)__popc(b);
          if (ok) mx = max(mx, x);
          if ((int)lane == j) myb = b;
        }
      }
      if (lane < 8u) sh.bal[slot][warp][lane] = myb;
      mx = __reduce_max_sync(0xFFFFFFFFu, mx);
      if (lane == 0) { sh.wcnt[slot][warp] = cnt; sh.wmax[slot][warp] = cnt ? (mx >> 20) + 1u : 0u; }
    }
    { TR_T(t0); __syncthreads(); { volatile u32* vp = sh.g0; u32 dummy = vp[0]; asm volatile("" :: "r"(dummy) : "memory"); } TR_ADD(2, t0); }                                                         // #1
    if (scn) {
      // ---- publish the aggregate of tile i + kCountAhead, issue the look-back loads of tile i + 1
      if (kc < nLocal) {
        const EvDesc& e = desc_of(kc);
        const u32 tile = first + (u32)kc * G - e.tileBase, slot = (u32)kc % kRawSlots;
        const u32 n = __reduce_add_sync(0xFFFFFFFFu, lane < 8u ? sh.wcnt[slot][lane] : 0u);
        const u32 mx1 = __reduce_max_sync(0xFFFFFFFFu, lane < 8u ? sh.wmax[slot][lane] : 0u);
        if (lane == 0) st_state(e.tileState + tile, pack_state(tile ? kStAgg : kStIncl, n, mx1));
      }
      if (kl >= 0 && kl < nLocal) {
        const EvDesc& e = desc_of(kl);
        tl = first + (u32)kl * G - e.tileBase;
        if (tl) lookback_issue(e.tileState, (int)tl, lane, lb);
      }
    } else if (!ctl && i >= 0) {
      // ---- scatter: local tile i
      const EvDesc& e = desc_of(i);
      const u32 T0 = (first + (u32)i * G - e.tileBase) * (u32)kTileWords, W = e.nWords;
      const u32 nIn = W > T0 ? min(W - T0, (u32)kTileWords) : 0u, slot = (u32)i % kRawSlots;
      const u32 g0 = sh.g0[i & 1], ph = g0 & 7u;
      const u32 c8 = lane < 8u ? sh.wcnt[slot][lane] : 0u;
      const u32 wbase = __reduce_add_sync(0xFFFFFFFFu, lane < warp ? c8 : 0u);
      const u32 myb = lane < 8u ? sh.bal[slot][warp][lane] : 0u;
      const u32* wseg = sh.words[slot] + 256u * warp + lane;
      const u16* aseg = sh.adc[slot] + 256u * warp + lane;
      u32 ebase = 8u + ph + wbase;                             // staging element of the warp's next digi
      const u32 wi0 = T0 + 256u * warp + lane;                 // event-local index of this lane's word of row 0
      if (tid == 0) {                                          // "the digi before the tile" for the order check (module 0 if none)
        const u32 c1 = sh.carry1[i & 1];
        sh.sModule[8u + ph - 1u] = (u16)(c1 ? c1 - 1u : 0u);
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const u32 b = __shfl_sync(0xFFFFFFFFu, myb, j);
        const u32 x = wseg[32 * j], a = aseg[32 * j];
        const u32 el = ebase + (u32)__popc(b & lt);
        if (b >> lane & 1u) {
          const u32 mod = x >> 20;
          const float2 gp = __ldg(g.calib + mod);
          sh.sModule[el] = (u16)mod; sh.sRow[el] = (u16)((x >> 12) & 0xFFu); sh.sCol[el] = (u16)((x >> 3) & 0x1FFu);
          sh.sAdc[el] = (u16)a; sh.sWordIdx[el] = wi0 + 32u * j;
          sh.sCharge[el] = __fmaf_rn((float)a, gp.x, gp.y);
        } else if (256u * warp + 32u * j + lane < nIn) {
          // error word (A2-A4): errors before it = words before it - digis before it
          const u32 ei = (wi0 + 32u * j) - (g0 + (el - 8u - ph));
          e.errWord[ei] = x; e.errIdx[ei] = wi0 + 32u * j;
        }
        ebase += (u32)__popc(b);
      }
      fence_async_smem();                                      // staged digis -> visible to the TMA store
    }
    { TR_T(t0); __syncthreads(); { volatile u32* vp = sh.g0; u32 dummy = vp[0]; asm volatile("" :: "r"(dummy) : "memory"); } TR_ADD(3, t0); }                                                         // #2
    if (ctl) {
      if (i >= 0) {
        const EvDesc& e = desc_of(i);
        const u32 slot = (u32)i % kRawSlots, g0 = sh.g0[i & 1], ph = g0 & 7u;
        const u32 n = __reduce_add_sync(0xFFFFFFFFu, lane < 8u ? sh.wcnt[slot][lane] : 0u);
        const u32 midLo = (g0 + 7u) & ~7u, midHi = (g0 + n) & ~7u;
        if (lane == 0) {
          if (midHi > midLo) {
            const u32 cnt = midHi - midLo, se = 8u + ph + (midLo - g0);
            bulk_store(e.module + midLo, sh.sModule + se, cnt * 2u); bulk_store(e.row + midLo, sh.sRow + se, cnt * 2u);
            bulk_store(e.col + midLo, sh.sCol + se, cnt * 2u); bulk_store(e.adcOut + midLo, sh.sAdc + se, cnt * 2u);
            bulk_store(e.wordIdx + midLo, sh.sWordIdx + se, cnt * 4u); bulk_store(e.charge + midLo, sh.sCharge + se, cnt * 4u);
          }
          bulk_commit();
        }
        if (i + kRawSlots < nLocal) issue_load(i + kRawSlots);   // into the slot this tile vacated
        if (lane < 16u) {
          // head (k < 8) and tail (k >= n - 8) digis outside the 16-byte-aligned middle
          const u32 lo = 8u + ph, k = lane < 8u ? lane : n - 16u + lane, p = g0 + k;
          if (k < n && (lane < 8u || k >= 8u) && !(p >= midLo && p < midHi)) {
            const u32 se = lo + k;
            e.module[p] = sh.sModule[se]; e.row[p] = sh.sRow[se]; e.col[p] = sh.sCol[se]; e.adcOut[p] = sh.sAdc[se];
            e.wordIdx[p] = sh.sWordIdx[se]; e.charge[p] = sh.sCharge[se];
          }
        }
      }
      if (!kSingle && i >= 0) {
        if (kd < nLocal) sh.desc[kd & (kDescRing - 1)][lane] = dword;
        eNext = eN2;
      }
    } else if (scn) {
      // ---- resolve the look-back of tile i + 1 (its loads flew during the scatter), publish its inclusive state
      if (kl >= 0 && kl < nLocal) {
        const EvDesc& e = desc_of(kl);
        const u32 slot = (u32)kl % kRawSlots;
        u32 c = 0, m = 0;
        if (tl) {
          { TR_T(t0); lookback_resolve(e.tileState, (int)tl, lane, lb, &c, &m); TR_ADD(6, t0); }
          const u32 n = __reduce_add_sync(0xFFFFFFFFu, lane < 8u ? sh.wcnt[slot][lane] : 0u);
          const u32 mx1 = __reduce_max_sync(0xFFFFFFFFu, lane < 8u ? sh.wmax[slot][lane] : 0u);
          if (lane == 0) st_state(e.tileState + tl, pack_state(kStIncl, c + n, max(m, mx1)));
        }
        if (lane == 0) { sh.g0[kl & 1] = c; sh.carry1[kl & 1] = m; }
      }
    } else if (i >= 0) {
      const EvDesc& e = desc_of(i);
      const u32 tile = first + (u32)i * G - e.tileBase, slot = (u32)i % kRawSlots;
      const u32 g0 = sh.g0[i & 1], ph = g0 & 7u, carry1 = sh.carry1[i & 1];
      const u32 c8 = lane < 8u ? sh.wcnt[slot][lane] : 0u, m8 = lane < 8u ? sh.wmax[slot][lane] : 0u;
      const u32 n = __reduce_add_sync(0xFFFFFFFFu, c8), tileMax1 = __reduce_max_sync(0xFFFFFFFFu, m8);
      const u32 lo = 8u + ph, hi = lo + n;
      // order check (A5): no digi's module is below that of the digi before it.  Eight digis per thread;
      // per halfword, bit 15 of (m | 0x8000) - p stays set iff m >= p (modules are below 2^11).
      {
        u32 bad = 0;
        for (u32 c = 1u + tid; 8u * c < hi; c += kUnpackThreads) {
          const uint4 v = *reinterpret_cast<const uint4*>(sh.sModule + 8u * c);
          const u32 prev = sh.sModule[8u * c - 1u];
          if (8u * c >= lo && 8u * c + 8u <= hi) {
            const u32 s0 = v.x << 16 | prev, s1 = __funnelshift_l(v.x, v.y, 16), s2 = __funnelshift_l(v.y, v.z, 16), s3 = __funnelshift_l(v.z, v.w, 16);
            const u32 t = ((v.x | 0x80008000u) - s0) & ((v.y | 0x80008000u) - s1) & ((v.z | 0x80008000u) - s2) & ((v.w | 0x80008000u) - s3);
            bad |= ~t & 0x80008000u;
          } else {                                             // the tile's first and last chunk may be partial
            const u32 w4[4] = {v.x, v.y, v.z, v.w};
            u32 p = prev;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              const u32 m = (q & 1) ? w4[q >> 1] >> 16 : w4[q >> 1] & 0xFFFFu, idx = 8u * c + (u32)q;
              if (idx >= lo && idx < hi && m < p) bad = 1u;
              p = m;
            }
          }
        }
        if (bad) atomicOr(&e.counters->status, 1u);            // PR_STATUS_INPUT_ORDER
      }
      // modDigiStart[m] for the modules that begin in this tile (or are skipped by it): the number of staged
      // digis with module < m (the staged modules ascend unless the order check fired).  Warp w resolves the
      // modules that are new in its own 256-word segment, [max module + 1 before it, max module + 1 in it), by a
      // 4-ary search inside the segment: every warp gets its share.
      if (n) {
        const u32 prev1 = max(carry1, __reduce_max_sync(0xFFFFFFFFu, lane < warp ? m8 : 0u));
        const u32 wbase = __reduce_add_sync(0xFFFFFFFFu, lane < warp ? c8 : 0u);
        const u32 cntW = __shfl_sync(0xFFFFFFFFu, c8, warp), mx1W = __shfl_sync(0xFFFFFFFFu, m8, warp);
        const u16* base = sh.sModule + lo + wbase;
        for (u32 m = prev1 + lane; m < mx1W; m += 32u) {
          u32 pos = 0, len = cntW;                             // digis [0, pos) of the segment are < m; the answer is < pos + len
#pragma unroll
          for (u32 q = 64u; q; q >>= 2) {                      // len <= 256: quarters of 64, 16, 4, 1
            u32 adv = 0;
#pragma unroll
            for (u32 r = 1; r <= 3u; ++r)
              if (r * q <= len && base[pos + r * q - 1u] < m) adv = r;
            pos += adv * q;
            len = min(len - adv * q, q);
          }
          e.modDigiStart[m] = g0 + wbase + pos;
        }
      }
      // the event's last tile closes modDigiStart and the counters
      if (tile == e.nTiles - 1u) {
        const u32 D = g0 + n, mx1 = max(carry1, tileMax1), W = e.nWords;
        for (u32 m = mx1 + tid; m <= g.M; m += kUnpackThreads) e.modDigiStart[m] = D;
        if (tid == 0) { e.counters->nWords = W; e.counters->nDigis = D; e.counters->nErrors = W - D; }
      }
    }
  }
  if (ctl && lane == 0) bulk_wait_all();
#ifdef PIXRECO_TRACE
  if (lane == 0 && blockIdx.x < 1024) {
    unsigned long long* o = g_trace + blockIdx.x * 32;
    o[warp * 2] = trAcc[2]; o[warp * 2 + 1] = trAcc[3];
    if (ctl) { o[20] = trAcc[0]; o[22] = (unsigned long long)(clock64() - trStart); }
    if (scn) o[21] = trAcc[6];
    if (warp == 0) o[23] = trAcc[1];
  }
#endif
}

// ================================================================== k_cluster (a3 + a4)
// Every module is an independent problem.  No unit of work waits for another one:
//   warp path    consecutive modules with at most 32 digis together are clustered in one pass by ONE
//                warp, in registers (warp_pack).  A module of 33..kWarpCap digis is clustered by ONE warp with
//                only __syncwarp between its phases: warp-private hash table (row,col) -> digi for the
//                backward-neighbour look-ups (each found edge is recorded on both ends),
//                label-equivalence rounds (min over neighbours, hook the old representative with
//                atomicMin, pointer jumping) until stable, then per-cluster sums accumulated in
//                shared memory as binary64 (exact: at most 256 terms below 2^43).  Warps take
//                batches of kModBatch consecutive modules from a global ticket.
//   dense path   a module with more than kWarpCap digis is clustered by a whole CTA: occupancy
//                bitmap + popcount ranks, union-find and per-cluster atomics (shared-memory tiers,
//                global workspace beyond).  Every CTA first scans its residue class of the
//                launch's modules for such modules, then joins the warp path.
// Both paths write label[] (final), clus[] = rank of the digi's cluster among the module's kept
// clusters (or -1), the module's kept-cluster count, and stage the kept clusters' sums at index
// (first digi of the module + rank).  k_finalize turns the ranks into the event-wide dense
// numbering (ascending label order, A12) and writes the cluster SoA.
constexpr u32 kWarpCap = 256;                    // warp path: modules with at most this many digis
constexpr u32 kWarpTab = 2 * kWarpCap;           // hash slots per warp (load <= 1/4 up to 128 digis, <= 1/2 beyond)
constexpr u32 kAccRoots = 96;                    // clusters accumulated per pass over a module
constexpr u32 kModBatch = 4;                     // most modules per warp ticket (small tickets: a short tail; 8 was 6 % slower, 16 17 %);
                                                 // small launches use 2 or 1 so that every warp gets work (modBatch, a power of two)
constexpr u32 kEmpty = 0xFFFFFFFFu;
constexpr u32 kNoKey = 0xFFFFFFFFu;
constexpr u32 kNoRank = 0xFFFFu;

struct WarpRegion {                 // 5 KB of shared memory per warp
  u32 tab[kWarpTab];                // hash table; afterwards L[256] then the head of the accumulators
  uint2 nb[kWarpCap];               // 8 neighbour digi indices, one byte each (self = none); afterwards accumulators
  u32 key[kWarpCap];                // row << 9 | col of kept digis, kNoKey otherwise
};
static_assert(sizeof(u32) * (kWarpTab - kWarpCap) + sizeof(uint2) * kWarpCap >= kAccRoots * 28, "accumulators must fit");

__host__ __device__ inline size_t dense_smem_bytes(u32 bitmapWords, u32 capDigis = kSmemDigis, u32 capClusters = kSmemClusters) {
  size_t w = (bitmapWords + 3) & ~3u;
  return (size_t)w * 4 * 2 + (size_t)capDigis * 4 * 2 + (size_t)capClusters * (4 + 4 + 4 + 8 * 3);
}
__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t dense = dense_smem_bytes(bitmapWords), warp = sizeof(WarpRegion) * (kClusterThreads / 32);
  return ((dense > warp ? dense : warp) + 15) & ~(size_t)15;
}

// Root of x, halving the path on the way (a node's parent only ever moves to another ancestor in its set, so
// concurrent finds and hooks stay consistent).  Only while unions are running: see uf_root.
__device__ __forceinline__ u32 uf_find(volatile u32* parent, u32 x) {
  u32 p = parent[x];
  while (p != x) {
    const u32 gp = parent[p];
    if (gp != p) parent[x] = gp;
    x = p; p = gp;
  }
  return x;
}
// Root of x without touching the forest: for the flattening pass, where a late halving store could
// overwrite another thread's final root.
__device__ __forceinline__ u32 uf_root(const volatile u32* parent, u32 x) {
  u32 p;
  while ((p = parent[x]) != x) x = p;
  return x;
}
// Hook the larger root under the smaller one (atomicMin), so the final root of every set is its
// minimum digi index = the canonical label (A10).
__device__ __forceinline__ void uf_union(u32* parent, u32 a, u32 b) {
  for (;;) {
    a = uf_find(parent, a); b = uf_find(parent, b);
    if (a == b) return;
    if (a < b) { u32 t = a; a = b; b = t; }
    const u32 old = atomicMin(parent + a, b);
    if (old == a) return;
    a = old;
  }
}

struct ClusterShared {
  u32 scan[16];
  u32 nBig, big[kClusterThreads];
};

__device__ __forceinline__ u32 wm_slot(u32 key, u32 shift) { return (key * 0x9E3779B1u) >> shift; }
// First digi on pixel `key` (a module without duplicate pixels), kEmpty if none.
__device__ __forceinline__ u32 wm_find(const u32* tab, u32 pmask, u32 shift, u32 key) {
  u32 h = wm_slot(key, shift);
  for (;;) {
    const u32 v = tab[h];
    if (v == kEmpty) return kEmpty;
    if ((v >> 8) == key) return v & 0xFFu;
    h = (h + 1) & pmask;
  }
}
// Minimum digi index on pixel `key` (duplicate pixels present: owner = min index, A6).
__device__ __forceinline__ u32 wm_find_min(const u32* tab, u32 pmask, u32 shift, u32 key) {
  u32 h = wm_slot(key, shift), best = kEmpty;
  for (;;) {
    const u32 v = tab[h];
    if (v == kEmpty) return best;
    if ((v >> 8) == key) best = min(best, v & 0xFFu);
    h = (h + 1) & pmask;
  }
}

// ---- warp path, one digi per lane: a PACK of consecutive modules with at most 32 digis together, digis
// [s, s+n).  Everything lives in registers: lane i learns its neighbours by comparing its (module, row,
// col) with every other lane's (n shuffles, no table; two digis on one pixel are simply adjacent, A6),
// adjacency and reachability are 32-bit lane masks (Warshall closure with shuffles), a cluster's
// minimum lane is its root, sums run along each cluster's lane list.  mIdx/mStart: the lane's module
// (index within the pack) and that module's first digi.  Returns the ballots of kept digis, of roots
// and of roots of kept clusters.
__device__ __forceinline__ void warp_pack(const EvDesc& ev, const Geom& g, u32 s, u32 n, float q0, u32 rc0, u32 mIdx, u32 mStart,
                                          u32* keptDigis, u32* roots, u32* keptRoots) {
  const u32 lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  const float q = lane < n ? q0 : 0.f;
  const bool kept = lane < n && q >= g.pixThr;                                  // A8
  // K = col | row << 10 | module << 19 with a guard bit above col and row: K_i - K_j + (1 | 1 << 10) has both
  // fields in {0, 1, 2} and nothing else set iff same module, |d row| <= 1 and |d col| <= 1.  A digi that is
  // not kept gets a module of its own.
  const u32 K = kept ? ((rc0 & 511u) | (rc0 >> 9) << 10 | mIdx << 19) : (0x1000u + lane) << 19;
  const u32 Kb = K + 0x401u;
  u32 adj = 0;
#pragma unroll 4
  for (u32 j = 0; j < n; ++j) {
    const u32 t = Kb - __shfl_sync(0xFFFFFFFFu, K, j);
    const u32 bad = (t & ~0xC03u) | (t & (t >> 1) & 0x401u);
    adj |= (bad == 0u ? 1u : 0u) << j;
  }
  adj |= 1u << lane;
  // transitive closure (Warshall): after step j every lane that reaches j also reaches all of j's set
  u32 reach = adj;
  for (u32 j = 0; j < n; ++j) {
    const u32 rj = __shfl_sync(0xFFFFFFFFu, reach, j);
    if (reach & (1u << j)) reach |= rj;
  }
  const u32 root = (u32)__ffs((int)reach) - 1u;
  const bool isRoot = kept && root == lane;
  // sums of qf = q * 2^14 (A9) in binary64 (exact: at most 32 terms below 2^43), suffix sums along the lane list
  double qf = 0.0, qx = 0.0, qy = 0.0;
  if (kept) { qf = (double)(q * 16384.0f); qx = qf * (double)(rc0 >> 9); qy = qf * (double)(rc0 & 511u); }
  const u32 most = __reduce_max_sync(0xFFFFFFFFu, (u32)__popc(reach));
  const u32 above = reach & (0xFFFFFFFEu << lane);
  u32 nxt = above ? (u32)__ffs((int)above) - 1u : 32u;
  for (u32 span = 1; span < most; span <<= 1) {
    const u32 src = nxt & 31u;
    const double a = __shfl_sync(0xFFFFFFFFu, qf, src), b = __shfl_sync(0xFFFFFFFFu, qx, src), c = __shfl_sync(0xFFFFFFFFu, qy, src);
    const u32 nn = __shfl_sync(0xFFFFFFFFu, nxt, src);
    if (nxt < 32u) { qf += a; qx += b; qy += c; nxt = nn; }
  }
  const bool keptC = isRoot && __double2ll_rz(qf) >= g.clusThrFixed;
  const u32 kb = __ballot_sync(0xFFFFFFFFu, keptC);
  const u32 kr = (u32)__popc(kb & lt & ~((1u << (mStart - s)) - 1u));           // rank among the module's kept clusters
  if (keptC) {
    const u32 o = mStart + kr;
    ev.stS[o] = qf; ev.stSx[o] = qx; ev.stSy[o] = qy;
    ev.stLabel[o] = s + lane; ev.stSize[o] = (u32)__popc(reach);
  }
  const u32 krRoot = __shfl_sync(0xFFFFFFFFu, keptC ? kr : kNoRank, root);
  if (lane < n) {
    ev.label[s + lane] = kept ? s + root : kInvalid;
    ev.clus[s + lane] = (kept && krRoot != kNoRank) ? (int32_t)krRoot : -1;
  }
  *keptDigis = __ballot_sync(0xFFFFFFFFu, kept); *roots = __ballot_sync(0xFFFFFFFFu, isRoot); *keptRoots = kb;
}

// ---- warp path: one module = digis [s, s+n), 0 < n <= kWarpCap, processed by the calling warp.
// Returns (kept digis, clusters, kept clusters) in all lanes.
__device__ __forceinline__ void warp_module(const EvDesc& ev, const Geom& g, u32 s, u32 n, WarpRegion& wr, float q0, u32 rc0,
                                            u32* nKeptDigis, u32* nRootsOut, u32* nKeptClusters) {
  const u32 lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  const u32 nPad = (n + 31u) & ~31u;
  const u32 lg = min(32u - (u32)__clz((int)(max(4u * n, 128u) - 1u)), 9u);   // log2 table size: >= 4n up to 128 digis, 512 beyond
  const u32 pmask = (1u << lg) - 1u, shift = 32u - lg;
  u32* tab = wr.tab;
  unsigned char* nbB = reinterpret_cast<unsigned char*>(wr.nb);

  // A: clear the table
  for (u32 i = lane * 4u; i <= pmask; i += 128u) *reinterpret_cast<uint4*>(tab + i) = make_uint4(kEmpty, kEmpty, kEmpty, kEmpty);
  __syncwarp();
  // B: load, kept flag (A8), insert; every digi starts with no neighbours (all bytes = self)
  // The loads run one chunk ahead (the first chunk came with the call): charge, row and col together.
  u32 nKept = 0; bool dup = false;
  float qc = q0; u32 rcc = rc0;
  for (u32 i = lane; i < nPad; i += 32u) {
    float qn = 0.f; u32 rcn = 0;
    if (i + 32u < n) { qn = ev.charge[s + i + 32u]; rcn = (u32)ev.row[s + i + 32u] << 9 | (u32)ev.col[s + i + 32u]; }
    const u32 key = (i < n && qc >= g.pixThr) ? rcc : kNoKey;                  // A8
    qc = qn; rcc = rcn;
    wr.key[i] = key;
    wr.nb[i] = make_uint2(i * 0x01010101u, i * 0x01010101u);
    if (key != kNoKey) {
      const u32 ent = key << 8 | i;
      u32 h = wm_slot(key, shift);
      for (;;) {
        const u32 old = atomicCAS(tab + h, kEmpty, ent);
        if (old == kEmpty) break;
        if ((old >> 8) == key) dup = true;
        h = (h + 1) & pmask;
      }
    }
    nKept += __popc(__ballot_sync(0xFFFFFFFFu, key != kNoKey));
  }
  dup = __any_sync(0xFFFFFFFFu, dup);
  __syncwarp();
  // C: backward neighbours W, NW, N, NE of every kept digi; an edge found is recorded on both
  // ends (slot d of i, slot d+4 of the neighbour: one writer per slot).  A duplicate only follows
  // its pixel's owner (A6).
  for (u32 i = lane; i < nPad; i += 32u) {
    const u32 key = wr.key[i];
    if (key == kNoKey) continue;
    const u32 row = key >> 9, col = key & 511u;
    if (dup) {
      const u32 owner = wm_find_min(tab, pmask, shift, key);
      if (owner != i) { nbB[i * 8u] = (unsigned char)owner; continue; }
    }
    const bool up = row > 0, left = col > 0, right = col + 1 < g.C;
#define WM_NB(cond, delta, d)                                                                      \
    if (cond) {                                                                                    \
      const u32 j = dup ? wm_find_min(tab, pmask, shift, key - (delta)) : wm_find(tab, pmask, shift, key - (delta)); \
      if (j != kEmpty) { nbB[i * 8u + (d)] = (unsigned char)j; nbB[j * 8u + (d) + 4u] = (unsigned char)i; }          \
    }
    WM_NB(left, 1u, 0u)
    WM_NB(up && left, 513u, 1u)
    WM_NB(up, 512u, 2u)
    WM_NB(up && right, 511u, 3u)
#undef WM_NB
  }
  __syncwarp();
  // D: label equivalence.  L[i] only decreases and always names a digi of i's component; a round
  // takes the minimum over the neighbours, hooks the old representative under it, then flattens.
  // The first round needs no look-ups: with L = identity the minimum over the neighbours is the minimum
  // neighbour index.
  u32* L = tab;
  for (u32 i = lane; i < nPad; i += 32u) {
    const uint2 nb = wr.nb[i];
    u32 v = __vminu4(nb.x, nb.y);
    v = __vminu4(v, v >> 16); v = __vminu4(v, v >> 8);
    L[i] = min(i, v & 0xFFu);
  }
  __syncwarp();
  for (u32 i = lane; i < nPad; i += 32u) {
    u32 l = L[i], p;
    while ((p = L[l]) != l) l = p;
    L[i] = l;
  }
  __syncwarp();
  for (;;) {
    bool changed = false;
    for (u32 i = lane; i < nPad; i += 32u) {
      const uint2 nb = wr.nb[i];
      const u32 li = L[i];
      u32 m = li;
      m = min(m, L[nb.x & 0xFFu]); m = min(m, L[(nb.x >> 8) & 0xFFu]); m = min(m, L[(nb.x >> 16) & 0xFFu]); m = min(m, L[nb.x >> 24]);
      m = min(m, L[nb.y & 0xFFu]); m = min(m, L[(nb.y >> 8) & 0xFFu]); m = min(m, L[(nb.y >> 16) & 0xFFu]); m = min(m, L[nb.y >> 24]);
      if (m < li) {
        atomicMin(L + li, m);
        if (li != i) atomicMin(L + i, m);
        changed = true;
      }
    }
    if (!__any_sync(0xFFFFFFFFu, changed)) break;
    __syncwarp();
    for (u32 i = lane; i < nPad; i += 32u) {
      u32 l = L[i], p;
      while ((p = L[l]) != l) l = p;
      L[i] = l;
    }
    __syncwarp();
  }
  // E: rank of every root among the module's clusters (ascending index): L[root] |= rank << 8
  u32 nR = 0;
  for (u32 i = lane; i < nPad; i += 32u) {
    const bool isRoot = wr.key[i] != kNoKey && L[i] == i;
    const u32 rb = __ballot_sync(0xFFFFFFFFu, isRoot);
    if (isRoot) L[i] = i | (nR + __popc(rb & lt)) << 8 | kNoRank << 16;
    nR += __popc(rb);
  }
  __syncwarp();
  // F: per-cluster sums S, Sx, Sy of qf = q * 2^14 (A9) as binary64 in shared memory, kAccRoots
  // clusters per pass.  The lanes of one 32-digi chunk that share a cluster are reduced with
  // shuffles, their first lane owns the read-modify-write; then the roots apply the cluster
  // threshold (A8), number the kept clusters and stage their sums.
  double* acc = reinterpret_cast<double*>(tab + kWarpCap);
  u32* cnt = reinterpret_cast<u32*>(acc + kAccRoots * 3u);
  u32 nK = 0;
  for (u32 p0 = 0; p0 < nR; p0 += kAccRoots) {
    const u32 nAcc = min(nR - p0, kAccRoots);
    for (u32 i = lane; i < nAcc * 3u; i += 32u) acc[i] = 0.0;
    for (u32 i = lane; i < nAcc; i += 32u) cnt[i] = 0u;
    __syncwarp();
    for (u32 i = lane; i < nPad; i += 32u) {
      const u32 key = wr.key[i];
      u32 rk = 0; bool in = false;
      u32 r = 256u + lane;
      if (key != kNoKey) {
        r = L[i] & 0xFFu;
        rk = ((L[r] >> 8) & 0xFFu) - p0;
        in = rk < nAcc;
        if (!in) r = 256u + lane;
      }
      const u32 peers = __match_any_sync(0xFFFFFFFFu, r);
      const u32 most = __reduce_max_sync(0xFFFFFFFFu, in ? (u32)__popc(peers) : 0u);
      double qf = 0.0, qx = 0.0, qy = 0.0;
      if (in) {
        qf = (double)(ev.charge[s + i] * 16384.0f);
        qx = qf * (double)(key >> 9); qy = qf * (double)(key & 511u);
      }
      // suffix sums along each cluster's lane list by pointer jumping: the first lane ends with the total
      const u32 above = peers & (0xFFFFFFFEu << lane);
      u32 nxt = above ? (u32)__ffs((int)above) - 1u : 32u;
      for (u32 span = 1; span < most; span <<= 1) {
        const u32 src = nxt & 31u;
        const double a = __shfl_sync(0xFFFFFFFFu, qf, src), b = __shfl_sync(0xFFFFFFFFu, qx, src), c = __shfl_sync(0xFFFFFFFFu, qy, src);
        const u32 nn = __shfl_sync(0xFFFFFFFFu, nxt, src);
        if (nxt < 32u) { qf += a; qx += b; qy += c; nxt = nn; }
      }
      if (in && (peers & lt) == 0u) {                 // one owner per cluster and chunk
        double* a = acc + rk * 3u;
        a[0] += qf; a[1] += qx; a[2] += qy;
        cnt[rk] += (u32)__popc(peers);
      }
      __syncwarp();
    }
    for (u32 i = lane; i < nPad; i += 32u) {
      const u32 w = wr.key[i] != kNoKey ? L[i] : 0u;
      const u32 rk = ((w >> 8) & 0xFFu) - p0;
      const bool mine = wr.key[i] != kNoKey && (w & 0xFFu) == i && rk < nAcc;
      double S = 0.0;
      if (mine) S = acc[rk * 3u];
      const bool keptC = mine && __double2ll_rz(S) >= g.clusThrFixed;
      const u32 kb = __ballot_sync(0xFFFFFFFFu, keptC);
      if (keptC) {
        const u32 kr = nK + __popc(kb & lt), o = s + kr;
        ev.stS[o] = S; ev.stSx[o] = acc[rk * 3u + 1u]; ev.stSy[o] = acc[rk * 3u + 2u];
        ev.stLabel[o] = s + i; ev.stSize[o] = cnt[rk];
        L[i] = (w & 0xFFFFu) | kr << 16;
      }
      nK += __popc(kb);
    }
    __syncwarp();
  }
  // G: per-digi outputs: label (final), cluster rank within the module
  for (u32 i = lane; i < n; i += 32u) {
    const bool kept = wr.key[i] != kNoKey;
    u32 lab = kInvalid; int32_t cl = -1;
    if (kept) {
      const u32 r = L[i] & 0xFFu, kr = L[r] >> 16;
      lab = s + r;
      if (kr != kNoRank) cl = (int32_t)kr;
    }
    ev.label[s + i] = lab; ev.clus[s + i] = cl;
  }
  *nKeptDigis = nKept; *nRootsOut = nR; *nKeptClusters = nK;
}

// ---- dense path: one module = digis [s, s+nn), nn > kWarpCap, processed by the whole CTA.
// dense_count clusters and sums (shared-memory tiers, global workspace beyond); dense_stage writes
// label[], clus[] = rank among the module's kept clusters, and stages the kept clusters' sums.
struct DenseCtx {
  u32 *perm, *parent, *root, *csize; int32_t* knum; u64 *S, *Sx, *Sy;
  u32 nAll, nKept;
};

template <u32 kT = kClusterThreads>
__device__ __forceinline__ void dense_count(const EvDesc& ev, const Geom& g, u32 s, u32 nn,
                                            unsigned char* smemRaw, ClusterShared& sh, DenseCtx& cx,
                                            u32 capDigis = kSmemDigis, u32 capClusters = kSmemClusters) {
  const int tid = threadIdx.x, lane = tid & 31;
  const u32 bwPad = (g.bitmapWords + 3) & ~3u;
  u64* smS = reinterpret_cast<u64*>(smemRaw);
  u64* smSx = smS + capClusters;
  u64* smSy = smSx + capClusters;
  u32* smBitmap = reinterpret_cast<u32*>(smSy + capClusters);
  u32* smPrefix = smBitmap + bwPad;
  u32* smPerm = smPrefix + bwPad;
  u32* smParent = smPerm + capDigis;
  u32* smRoot = smParent + capDigis;
  u32* smSize = smRoot + capClusters;
  int32_t* smKnum = reinterpret_cast<int32_t*>(smSize + capClusters);
  u32* sScan = sh.scan;
  const u32 stride = g.stride;

  const bool digiInSmem = nn <= capDigis;
  u32* perm = digiInSmem ? smPerm : ev.wsPerm + s;
  u32* parent = digiInSmem ? smParent : ev.wsParent + s;
  cx.perm = perm; cx.parent = parent;
  cx.root = smRoot; cx.csize = smSize; cx.knum = smKnum; cx.S = smS; cx.Sx = smSx; cx.Sy = smSy;

  // P0: clear the occupancy bitmap, init perm
  for (u32 i = tid; i < g.bitmapWords; i += kT) smBitmap[i] = 0;
  for (u32 i = tid; i < nn; i += kT) perm[i] = kInvalid;
  __syncthreads();
  // P1: kept flag (A8: q >= pixThr) and occupancy bits at padded coordinates (row+1, col+1)
  u32 myKept = 0;
  for (u32 i = tid; i < nn; i += kT) {
    const float q = ev.charge[s + i];
    const bool kept = q >= g.pixThr;
    parent[i] = kept ? i : kInvalid;
    if (kept) {
      const u32 b = ev.col[s + i] + 1u, wd = (ev.row[s + i] + 1u) * stride + (b >> 5);
      atomicOr(smBitmap + wd, 1u << (b & 31));
      ++myKept;
    }
  }
  myKept = __reduce_add_sync(0xFFFFFFFFu, myKept);
  __syncthreads();
  // P2: exclusive popcount prefix per bitmap word (contiguous chunk per thread)
  {
    const u32 per = (g.bitmapWords + kT - 1) / kT;
    const u32 lo = min(tid * per, g.bitmapWords), hi = min(lo + per, g.bitmapWords);
    u32 sum = 0;
    for (u32 i = lo; i < hi; ++i) sum += __popc(smBitmap[i]);
    u32 tot;
    u32 run = block_excl_scan<kT / 32>(sum, sScan, &tot);
    for (u32 i = lo; i < hi; ++i) { smPrefix[i] = run; run += __popc(smBitmap[i]); }
  }
  if (lane == 0 && myKept) atomicAdd(&ev.counters->nKept, myKept);
  __syncthreads();
  // P3: owner of each occupied pixel = the minimum digi index on it (duplicates, A6)
  for (u32 i = tid; i < nn; i += kT) {
    if (parent[i] == kInvalid) continue;
    const u32 b = ev.col[s + i] + 1u, wd = (ev.row[s + i] + 1u) * stride + (b >> 5);
    const u32 r = smPrefix[wd] + __popc(smBitmap[wd] & ((1u << (b & 31)) - 1u));
    atomicMin(perm + r, i);
  }
  __syncthreads();
  // P4: unions with the backward neighbours (W, NW, N, NE), decision tree:
  //     N ? {N} : { NE?, W ? {W} : NW? }   — spans every 8-adjacency once all pixels did it.
  for (u32 i = tid; i < nn; i += kT) {
    if (parent[i] == kInvalid) continue;
    const u32 prow = ev.row[s + i] + 1u, b = ev.col[s + i] + 1u;
    const u32 wd = prow * stride + (b >> 5);
    const u32 r = smPrefix[wd] + __popc(smBitmap[wd] & ((1u << (b & 31)) - 1u));
    const u32 owner = perm[r];
    if (owner != i) { uf_union(parent, i, owner); continue; }
    const u32 pos = b - 1u, w0 = pos >> 5, shf = pos & 31u;
    const u32 rowAbove = (prow - 1u) * stride, rowSelf = prow * stride;
    const u32 nb = __funnelshift_r(smBitmap[rowAbove + w0], smBitmap[rowAbove + w0 + 1], shf) & 7u;
    const u32 cb = __funnelshift_r(smBitmap[rowSelf + w0], smBitmap[rowSelf + w0 + 1], shf) & 7u;
    auto owner_at = [&](u32 rowBase, u32 bb) -> u32 {
      const u32 ww = rowBase + (bb >> 5);
      return perm[smPrefix[ww] + __popc(smBitmap[ww] & ((1u << (bb & 31)) - 1u))];
    };
    if (nb & 2u) {
      uf_union(parent, i, owner_at(rowAbove, b));
    } else {
      if (nb & 4u) uf_union(parent, i, owner_at(rowAbove, b + 1u));
      if (cb & 1u) uf_union(parent, i, owner_at(rowSelf, b - 1u));
      else if (nb & 1u) uf_union(parent, i, owner_at(rowAbove, b - 1u));
    }
  }
  __syncthreads();
  // P5: flatten (roots are stable now)
  for (u32 i = tid; i < nn; i += kT) {
    if (parent[i] == kInvalid) continue;
    const u32 rt = uf_root(parent, i);
    if (rt != i) parent[i] = rt;
  }
  __syncthreads();
  // P6: ordinal of every root in ascending index (= ascending label) order -> perm[root]
  {
    const u32 per = (nn + kT - 1) / kT;
    const u32 lo = min(tid * per, nn), hi = min(lo + per, nn);
    u32 c = 0;
    for (u32 i = lo; i < hi; ++i) c += (parent[i] == i);
    u32 run = block_excl_scan<kT / 32>(c, sScan, &cx.nAll);
    if (cx.nAll > capClusters) {
      cx.root = ev.wsRoot + s; cx.csize = ev.wsSize + s; cx.knum = ev.wsKnum + s;
      cx.S = ev.wsS + s; cx.Sx = ev.wsSx + s; cx.Sy = ev.wsSy + s;
    }
    for (u32 i = lo; i < hi; ++i)
      if (parent[i] == i) { perm[i] = run; cx.root[run] = i; ++run; }
  }
  // P7: zero the accumulators
  for (u32 c = tid; c < cx.nAll; c += kT) { cx.S[c] = 0; cx.Sx[c] = 0; cx.Sy[c] = 0; cx.csize[c] = 0; }
  __syncthreads();
  // P8: exact fixed-point sums (A9): qf = q * 2^14 is an integer for every kept digi
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = parent[i];
    if (p == kInvalid) continue;
    const u32 c = perm[p];
    const u64 qf = (u64)__float2ll_rz(ev.charge[s + i] * 16384.0f);
    atomicAdd(reinterpret_cast<unsigned long long*>(cx.S + c), (unsigned long long)qf);
    atomicAdd(reinterpret_cast<unsigned long long*>(cx.Sx + c), (unsigned long long)(qf * ev.row[s + i]));
    atomicAdd(reinterpret_cast<unsigned long long*>(cx.Sy + c), (unsigned long long)(qf * ev.col[s + i]));
    atomicAdd(cx.csize + c, 1u);
  }
  __syncthreads();
  // P9: cluster threshold (A8, A9) and local numbering of kept clusters
  {
    const u32 per = (cx.nAll + kT - 1) / kT;
    const u32 lo = min(tid * per, cx.nAll), hi = min(lo + per, cx.nAll);
    u32 c = 0;
    for (u32 k = lo; k < hi; ++k) c += ((i64)cx.S[k] >= g.clusThrFixed);
    u32 run = block_excl_scan<kT / 32>(c, sScan, &cx.nKept);
    for (u32 k = lo; k < hi; ++k) cx.knum[k] = ((i64)cx.S[k] >= g.clusThrFixed) ? (int32_t)run++ : -1;
  }
  __syncthreads();
}

template <u32 kT = kClusterThreads>
__device__ __forceinline__ void dense_stage(const EvDesc& ev, u32 m, u32 s, u32 nn, const DenseCtx& cx) {
  const int tid = threadIdx.x;
  for (u32 k = tid; k < cx.nAll; k += kT) {
    const int32_t kn = cx.knum[k];
    if (kn < 0) continue;
    const u32 o = s + (u32)kn;                       // kn <= k < nn: inside the module's own range
    ev.stS[o] = __ll2double_rn((i64)cx.S[k]); ev.stSx[o] = __ll2double_rn((i64)cx.Sx[k]); ev.stSy[o] = __ll2double_rn((i64)cx.Sy[k]);
    ev.stLabel[o] = s + cx.root[k]; ev.stSize[o] = cx.csize[k];
  }
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = cx.parent[i];
    u32 lab = kInvalid; int32_t cl = -1;
    if (p != kInvalid) { lab = s + p; cl = cx.knum[cx.perm[p]]; }
    ev.label[s + i] = lab;
    ev.clus[s + i] = cl;
  }
  if (tid == 0) {
    ev.modCount[m] = cx.nKept;
    if (cx.nKept) atomicAdd(&ev.grpCount[m / 32u], cx.nKept);
    if (cx.nAll) atomicAdd(&ev.counters->nClustersAll, cx.nAll);
  }
}

template <bool kSingle>
__global__ void __launch_bounds__(kClusterThreads, 4)
k_cluster(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv,
          LaunchCtl* __restrict__ lc, u32* __restrict__ bigList, u32 modBatch, const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ ClusterShared sh;
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const u32 M = g.M, total = nEv * M;

  // ---- phase 1: dense path.  Module (e, m) has index e * M + m; CTA b looks at the indices
  // congruent to b modulo the grid size (neighbouring hot modules go to different CTAs).
  for (u32 base = 0; base < total; base += gridDim.x * kClusterThreads) {
    const u32 gi = base + tid * gridDim.x + blockIdx.x;
    bool big = false;
    if (gi < total) {
      const u32 e = gi / M, m = gi - e * M;
      const EvDesc& ev = kSingle ? single : batch[e];
      if (!(ev.counters->status & 1u)) {              // A5 violated: modDigiStart is undefined, no per-digi work
        const u32 s = ev.modDigiStart[m], t = ev.modDigiStart[m + 1];
        big = t >= s && t <= ev.cap && t - s > kWarpCap;
      }
    }
    if (bigList) {                                      // a launch full of large modules: k_dense takes them (larger tiers)
      if (big) bigList[atomicAdd(&lc->nBig, 1u)] = gi;
      continue;
    }
    if (tid == 0) sh.nBig = 0;
    __syncthreads();
    if (big) sh.big[atomicAdd(&sh.nBig, 1u)] = gi;
    __syncthreads();
    const u32 nBig = sh.nBig;
    for (u32 k = 0; k < nBig; ++k) {
      const u32 gk = sh.big[k], e = gk / M, m = gk - e * M;
      const EvDesc& ev = kSingle ? single : batch[e];
      const u32 s = ev.modDigiStart[m], nn = ev.modDigiStart[m + 1] - s;
      DenseCtx cx;
      dense_count(ev, g, s, nn, smemRaw, sh, cx);
      dense_stage(ev, m, s, nn, cx);
      __syncthreads();
    }
    __syncthreads();
  }

  // ---- phase 2: warp path.  A ticket is a batch of modBatch (1, 2 or 4) consecutive modules of one event.
  WarpRegion& wr = reinterpret_cast<WarpRegion*>(smemRaw)[warp];
  // Tickets shrink towards the end of a large launch (modBatch 4): the first nEvA events are handed out four
  // modules at a time, the next nEvB events two at a time, the rest one by one, so that the last tickets are short.
  const u32 bpe = (M + modBatch - 1) / modBatch, bpeB = (M + 1u) / 2u;
  const u32 nEvA = modBatch == 4u ? nEv - nEv / 4u : nEv, nEvB = modBatch == 4u ? (nEv - nEvA + 1u) / 2u : 0u;
  const u32 tA = nEvA * bpe, tB = tA + nEvB * bpeB, nTickets = tB + (nEv - nEvA - nEvB) * M;
  for (;;) {
    u32 t = 0;
    if (lane == 0) t = atomicAdd(&lc->modTicket, 1u);
    t = __shfl_sync(0xFFFFFFFFu, t, 0);
    if (t >= nTickets) break;
    u32 e, m0, nm;
    if (t < tA) { e = t / bpe; m0 = (t - e * bpe) * modBatch; nm = min(modBatch, M - m0); }
    else if (t < tB) { const u32 u = t - tA; e = u / bpeB; m0 = (u - e * bpeB) * 2u; nm = min(2u, M - m0); e += nEvA; }
    else { const u32 u = t - tB; e = u / M; m0 = u - e * M; nm = 1u; e += nEvA + nEvB; }
    const EvDesc& ev = kSingle ? single : batch[e];
    if (ev.counters->status & 1u) continue;
    const u32 st = lane <= nm ? ev.modDigiStart[m0 + lane] : 0u;
    u32 accK = 0, accA = 0, accG = 0;
    // The ticket's digis are contiguous.  The next unit's first chunk (32 digis) is loaded while the current unit
    // (a pack of small modules, or one module of 33..kWarpCap digis) is processed.
    const u32 sEnd = min(__shfl_sync(0xFFFFFFFFu, st, nm), ev.cap);
    auto preload = [&](u32 s, float* q, u32* rc) {
      *q = 0.f; *rc = 0u;
      if (s + lane < sEnd) { *q = ev.charge[s + lane]; *rc = (u32)ev.row[s + lane] << 9 | (u32)ev.col[s + lane]; }
    };
    float qNext; u32 rcNext;
    preload(__shfl_sync(0xFFFFFFFFu, st, 0), &qNext, &rcNext);
    for (u32 k = 0; k < nm;) {
      const u32 s = __shfl_sync(0xFFFFFFFFu, st, k), t1 = __shfl_sync(0xFFFFFFFFu, st, k + 1);
      if (t1 < s || t1 > ev.cap) {                           // inconsistent module table
        if (lane == 0) { atomicOr(&ev.counters->status, 2u); ev.modCount[m0 + k] = 0u; }   // PR_STATUS_CAPACITY
        preload(t1 <= ev.cap ? t1 : sEnd, &qNext, &rcNext);
        ++k;
        continue;
      }
      const float q0 = qNext; const u32 rc0 = rcNext;
      if (t1 - s > 32u) {                                    // one module of its own
        const u32 n = t1 - s;
        preload(t1, &qNext, &rcNext);
        if (n <= kWarpCap) {                                 // else: the dense path wrote this module
          u32 nk, nr, cnt;
          warp_module(ev, g, s, n, wr, q0, rc0, &nk, &nr, &cnt);
          accK += nk; accA += nr; accG += cnt;
          if (lane == 0) ev.modCount[m0 + k] = cnt;
        }
        ++k;
        continue;
      }
      // pack: modules k .. k2-1, consecutive, consistent, at most 32 digis together
      u32 k2 = k + 1u, e2 = t1, mIdx = 0, mStart = s;
      while (k2 < nm) {
        const u32 en = __shfl_sync(0xFFFFFFFFu, st, k2 + 1u);
        if (en < e2 || en > ev.cap || en - s > 32u) break;
        if (e2 - s <= lane) { mIdx = k2 - k; mStart = e2; }   // module k2 starts at e2
        e2 = en; ++k2;
      }
      preload(e2, &qNext, &rcNext);
      const u32 n = e2 - s;
      u32 kd = 0, rb = 0, kb = 0;
      if (n) warp_pack(ev, g, s, n, q0, rc0, mIdx, mStart, &kd, &rb, &kb);
      accK += (u32)__popc(kd); accA += (u32)__popc(rb); accG += (u32)__popc(kb);
      // kept clusters per module of the pack: lane j - k writes module j's
      {
        const u32 j = k + lane;
        const u32 lo = __shfl_sync(0xFFFFFFFFu, st, min(j, nm)) - s, hi = __shfl_sync(0xFFFFFFFFu, st, min(j + 1u, nm)) - s;
        if (j < k2) {
          const u32 mask = (hi >= 32u ? 0xFFFFFFFFu : (1u << hi) - 1u) & ~(lo >= 32u ? 0xFFFFFFFFu : (1u << lo) - 1u);
          ev.modCount[m0 + j] = (u32)__popc(kb & mask);
        }
      }
      k = k2;
    }
    if (lane == 0 && accG) atomicAdd(&ev.grpCount[m0 / 32u], accG);     // modBatch divides 32: one group per ticket
    if (lane == 0) {
      if (accK) atomicAdd(&ev.counters->nKept, accK);
      if (accA) atomicAdd(&ev.counters->nClustersAll, accA);
    }
  }
}

// ================================================================== k_dense (a3 + a4 for launches full of large modules)
// The dense path of k_cluster as a kernel of its own, for launches whose modules are large on average
// (BASELINE.json configs[4]: 6.7k digis per module): two CTAs per SM with 8192 digis / 512 clusters
// per module in shared memory instead of 2048 / 512, so the union-find of such a module never leaves
// the SM.  k_cluster only collects the large modules in that case (bigList); CTAs take them by ticket.
constexpr u32 kDenseThreads = 512;
template <bool kSingle>
__global__ void __launch_bounds__(kDenseThreads, 2)
k_dense(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, LaunchCtl* __restrict__ lc,
        const u32* __restrict__ bigList, const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ ClusterShared sh;
  const u32 M = g.M, nBig = lc->nBig;
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) sh.nBig = atomicAdd(&lc->bigTicket, 1u);
    __syncthreads();
    const u32 t = sh.nBig;
    if (t >= nBig) break;
    const u32 gk = bigList[t], e = gk / M, m = gk - e * M;
    const EvDesc& ev = kSingle ? single : batch[e];
    const u32 s = ev.modDigiStart[m], nn = ev.modDigiStart[m + 1] - s;
    DenseCtx cx;
    dense_count<kDenseThreads>(ev, g, s, nn, smemRaw, sh, cx, kDenseDigis, kDenseClusters);
    dense_stage<kDenseThreads>(ev, m, s, nn, cx);
  }
}

// ================================================================== k_finalize (numbering of a4)
// One CTA per (event, group of kFinMods consecutive modules): the group's first dense cluster
// number is the sum of the kept-cluster counts of all earlier modules (at most 2048 values), so
// no CTA depends on another.  Turns clus[] ranks into event-wide cluster numbers, converts the
// staged sums into the cluster SoA (A9: binary64 division, one rounding to binary32), writes
// modClusStart[]; the CTA of an event's last module group publishes that event's counters to mapped pinned host memory.
constexpr u32 kFinMods = 32;
static_assert(kFinMods == 32 && 32 % kModBatch == 0, "grpCount groups are 32 modules and hold whole warp tickets");
template <bool kSingle>
__global__ void __launch_bounds__(256)
k_finalize(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv, u32 unitsPerEvent, u32 splits,
           LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  __shared__ u32 sStart[kFinMods + 1], sDigi[kFinMods + 1], sScan[8];
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, M = g.M;
  // `splits` CTAs share one (event, group) when events are huge: slice sp of the group's digis and clusters
  const u32 unit = blockIdx.x / splits, sp = blockIdx.x - unit * splits;
  const u32 e = unit / unitsPerEvent, u = unit - e * unitsPerEvent;
  const EvDesc& ev = kSingle ? single : batch[e];
  const u32 m0 = u * kFinMods, m1 = min(m0 + kFinMods, M);
  if (!(ev.counters->status & 1u)) {
    u32 sum = 0, base;
    for (u32 k = tid; k < u; k += 256) sum += ev.grpCount[k];      // groups of kFinMods modules before this one
    block_excl_scan(sum, sScan, &base);
    if (warp == 0) {
      const u32 c = m0 + lane < m1 ? ev.modCount[m0 + lane] : 0u;
      const u32 incl = warp_incl_scan(c, lane);
      sStart[lane] = base + incl - c;
      if (lane == 31) sStart[32] = base + incl;
      sDigi[lane] = ev.modDigiStart[min(m0 + lane, M)];
      if (lane == 31) sDigi[32] = ev.modDigiStart[min(m0 + 32u, M)];
    }
    __syncthreads();
    if (sp == 0) {
      for (u32 m = m0 + tid; m < m1; m += 256) ev.modClusStart[m] = sStart[m - m0];
      if (m1 == M && tid == 0) { ev.modClusStart[M] = sStart[32]; ev.counters->nClusters = sStart[32]; }
    }
    const u32 d0 = sDigi[0], d1 = sDigi[m1 - m0];
    if (d0 <= d1 && d1 <= ev.cap) {
      for (u32 dd = d0 + sp * 1024u + tid; dd < d1; dd += splits * 1024u) {     // four independent digis per thread and trip
        int32_t c[4]; u32 md[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const u32 d = dd + 256u * k;
          c[k] = d < d1 ? ev.clus[d] : -1;
          md[k] = d < d1 ? (u32)ev.module[d] : m0;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (c[k] >= 0) ev.clus[dd + 256u * k] = (int32_t)(sStart[min(md[k] - m0, kFinMods - 1)] + (u32)c[k]);
      }
      for (u32 o = sStart[0] + sp * 256u + tid; o < sStart[32]; o += splits * 256u) {
        u32 li = 0;
#pragma unroll
        for (u32 step = 16; step > 0; step >>= 1)
          if (li + step < kFinMods + 1 && sStart[li + step] <= o) li += step;   // last module with start <= o and a cluster there
        const u32 src = sDigi[li] + (o - sStart[li]);
        if (o < ev.cap && src < ev.cap) {
          const double S = ev.stS[src];
          ev.clLabel[o] = ev.stLabel[src]; ev.clModule[o] = (u16)(m0 + li); ev.clSize[o] = ev.stSize[src];
          ev.clCharge[o] = __double2float_rn(S * (1.0 / 16384.0));
          ev.clRow[o] = __double2float_rn(__ddiv_rn(ev.stSx[src], S));
          ev.clCol[o] = __double2float_rn(__ddiv_rn(ev.stSy[src], S));
        }
      }
    }
  }
  // The CTA of the event's last module group publishes the event's counters to mapped pinned host memory: all
  // the others were final when this kernel started, nClusters is this CTA's own result.
  if (m1 == M && sp == 0 && tid == 0) {
    const DevCounters* c = ev.counters;
    const u32 status = c->status;
    HostCounters h;
    h.nWords = c->nWords; h.nDigis = c->nDigis; h.nErrors = c->nErrors; h.nKept = c->nKept;
    h.nClustersAll = c->nClustersAll; h.nClusters = (status & 1u) ? 0u : sStart[32]; h.status = status; h.seq = 1;
    h.tStart = lc->tStart; h.tEnd = global_timer();
    *ev.hostCounters = h;
  }
}

// ================================================================== k_export
// Exact-size copies of requested outputs to mapped pinned host memory (transfers only
// when asked).  Element counts are read from the device counters, so no host round trip.
struct ExportItem { const void* src; void* dst; u32 elemBytes; u32 countSel; u32 fixedCount; u32 ev; };
// countSel: 0 = nDigis, 1 = nErrors, 2 = nClusters, 3 = fixedCount
__global__ void __launch_bounds__(256)
k_export(const ExportItem* __restrict__ items, u32 nItems, const DevCounters* __restrict__ counters) {
  for (u32 it = blockIdx.y; it < nItems; it += gridDim.y) {
    const ExportItem x = items[it];
    const DevCounters& c = counters[x.ev];
    const u32 cnt = x.countSel == 0 ? c.nDigis : x.countSel == 1 ? c.nErrors : x.countSel == 2 ? c.nClusters : x.fixedCount;
    const size_t bytes = (size_t)cnt * x.elemBytes;
    const size_t nVec = (bytes + 15) >> 4;                 // buffers are padded to 16 B
    const uint4* s = reinterpret_cast<const uint4*>(x.src);
    uint4* d = reinterpret_cast<uint4*>(x.dst);
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < nVec; v += (size_t)gridDim.x * blockDim.x) d[v] = s[v];
  }
}

}  // namespace pixreco

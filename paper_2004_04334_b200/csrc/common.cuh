// common.cuh — types, per-event descriptors, launch control blocks and the decoupled look-back shared by the
// kernels of the hot path.  Part of kernels.cuh (include that, not this file).
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
constexpr u32 kSmemClusters = 384;    // likewise for per-cluster accumulators
constexpr u32 kDenseDigis = 8192;     // the same tiers of k_dense (two CTAs per SM with their own, larger shared memory)
constexpr u32 kDenseClusters = 512;
constexpr u32 kMaxModuleDigis = (1u << 17) - 1u;   // A9: the exact sums are overflow-free up to 2^17 digis per module; more -> PR_STATUS_CAPACITY

// Per-event device counters (lives in the slot's control block, zeroed per acquire).
struct DevCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, pad;
};
// Per-launch control words.  The first two and unpackStarted are put back to zero by the last CTA of k_unpack (with the
// look-back states); the rest is zeroed per acquire together with the counters.
struct LaunchCtl {
  u32 tileTicket, unpackExited;     // k_unpack: next tile of the launch, CTAs that have left
  u32 modTicket, modDone;           // k_cluster: next warp ticket
  u64 tStart;                       // %globaltimer at the start of the acquire's first kernel
  u32 nBig, bigTicket;              // modules handed from k_cluster to k_dense, next one to take
  u32 unpackStarted;                // k_unpack: CTAs that have started (put back to zero with the ticket)
  u32 pad[7];
};
// What the host reads after completion (mapped pinned memory, written by the CTA that finishes the event).
struct HostCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, seq;
  u64 tStart, tEnd;                 // %globaltimer: first kernel of the acquire started, this event's counters published
};
__device__ __forceinline__ u64 global_timer() {
  u64 t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// A kept cluster as the clustering kernels stage it for k_finalize: exact sums (A9), label, size, bounding box (A28:
// max(255 - row) << 16 | max(row), max(511 - col) << 16 | max(col)).  ONE 48-byte record per cluster (three 16-byte
// accesses): a module's kept clusters are one contiguous run in memory.  (Seven separate arrays, as until capture Q of
// round 2, made seven sparse runs per module: k_finalize read 2.5 times the bytes it used.)
struct __align__(16) StagedCluster { double S, Sx, Sy; u32 label, size, boxR, boxC, pad0, pad1; };
static_assert(sizeof(StagedCluster) == 48, "three 16-byte vectors");
__device__ __forceinline__ void stage_store(StagedCluster* p, double S, double Sx, double Sy, u32 label, u32 size, u32 boxR, u32 boxC) {
  uint4* q = reinterpret_cast<uint4*>(p);
  q[0] = make_uint4((u32)__double2loint(S), (u32)__double2hiint(S), (u32)__double2loint(Sx), (u32)__double2hiint(Sx));
  q[1] = make_uint4((u32)__double2loint(Sy), (u32)__double2hiint(Sy), label, size);
  q[2] = make_uint4(boxR, boxC, 0u, 0u);
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
  // hit SoA [cap], hit k belongs to cluster k (A26-A30)
  float *htX, *htY, *htXerr, *htYerr; u32 *htRows, *htCols; u16* htFlags;
  // global workspace tier for large modules [cap] each (wsBox: 4 per digi slot)
  u32 *wsPerm, *wsParent, *wsRoot; int32_t* wsKnum; u32* wsSize; u64 *wsS, *wsSx, *wsSy; u32* wsBox;
  HostCounters* hostCounters;
  DevCounters* result;              // device copy of the event's final counters (per acquire; k_export reads its sizes there)
  u32* modCount;                    // [M+1] kept clusters per module (k_cluster -> k_finalize)
  u32* grpCount;                    // [ceil(M / 32)] the same summed over groups of kFinMods modules (zeroed per acquire)
  StagedCluster* staged;            // staged kept clusters: record k of the module with first digi s lives at index s + k [cap]
};
static_assert(offsetof(EvDesc, label) == 128, "k_unpack's part of the descriptor is one 128-byte line");

struct Geom {
  u32 M, R, C;
  u32 stride;                       // bitmap words per padded row = ceil((C+2)/32)
  u32 bitmapWords;                  // (R+2)*stride + 1
  float pixThr;
  i64 clusThrFixed;                 // llrint(clusThr * 2^14)
  double pitchRow, pitchCol;        // um per row index (local x) / col index (local y), A26
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

}  // namespace pixreco

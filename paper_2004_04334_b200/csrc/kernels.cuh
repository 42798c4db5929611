// kernels.cuh — sm_100a device code of the hot path (BASELINE.json north_star subsystem (2)).
//
//   k_unpack   a1+a2 fused: raw word decode, calibration, STABLE digi/error compaction with a
//              single-pass decoupled look-back scan, modDigiStart, input-order check.
//   k_cluster  a3+a4 fused: per-module 8-connected components (bitmap + rank lookup + min-index
//              union-find in shared memory), exact int64 fixed-point cluster sums, cluster
//              threshold, dense numbering through a cross-module decoupled look-back.
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
#include <stdint.h>

namespace pixreco {

typedef uint16_t u16;
typedef uint32_t u32;
typedef uint64_t u64;
typedef long long i64;

constexpr u32 kInvalid = 0xFFFFFFFFu;

// ---- unpack kernel geometry ----
constexpr int kUnpackThreads = 256;
constexpr int kWordsPerThread = 8;
constexpr int kTileWords = kUnpackThreads * kWordsPerThread;   // 2048

// ---- cluster kernel geometry ----
constexpr int kClusterThreads = 256;
constexpr u32 kWindowLog2 = 9;
constexpr u32 kWindow = 1u << kWindowLog2;       // a cluster work unit = 512 consecutive digi indices
constexpr u32 kSmemDigis = 2048;      // modules with more digis use the global workspace tier
constexpr u32 kSmemClusters = 512;    // likewise for per-cluster accumulators

// Per-event device counters (lives in the slot's control block, zeroed per acquire).
struct DevCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, pad;
};
// Per-launch control words (zeroed per acquire).
struct LaunchCtl {
  u32 tileTicket, modTicket, modDone, pad[13];
};
// What the host reads after completion (mapped pinned memory, written by the last block).
struct HostCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, seq;
};

// One event of a launch.
struct EvDesc {
  const u32* words; const u16* adc;
  u32 nWords, tileBase, nTiles, cap;
  // digi SoA [cap]
  u16 *module, *row, *col, *adcOut; u32* wordIdx; float* charge; u32* label; int32_t* clus;
  // error list [cap]
  u32 *errWord, *errIdx;
  // [M+1]
  u32 *modDigiStart, *modClusStart;
  // cluster SoA [cap]
  u32 *clLabel, *clSize; u16* clModule; float *clCharge, *clRow, *clCol;
  // global workspace tier for large modules [cap] each
  u32 *wsPerm, *wsParent, *wsRoot; int32_t* wsKnum; u32* wsSize; u64 *wsS, *wsSx, *wsSy;
  DevCounters* counters; HostCounters* hostCounters;
  u64 *tileState, *winState;        // look-back states: [nTiles], [nWin]
  u32* winInv;                      // [nWin]: M - (first module starting in the window), 0 = none
  u32 winBase, nWin;                // this event's windows in the launch's flattened unit space
};

struct Geom {
  u32 M, R, C;
  u32 stride;                       // bitmap words per padded row = ceil((C+2)/32)
  u32 bitmapWords;                  // (R+2)*stride + 1
  float pixThr;
  i64 clusThrFixed;                 // llrint(clusThr * 2^14)
  const float *gain, *ped;          // device [M]
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

// Block-wide exclusive scan of one value per thread (blockDim = 256); returns exclusive prefix,
// *total = block sum.  `sw` is 8 words of shared scratch.  Contains two __syncthreads.
__device__ __forceinline__ u32 block_excl_scan(u32 v, u32* sw, u32* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  u32 incl = warp_incl_scan(v, lane);
  __syncthreads();                                   // protect sw against the previous use
  if (lane == 31) sw[warp] = incl;
  __syncthreads();
  u32 base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    u32 s = sw[w];
    if (w < warp) base += s;
    tot += s;
  }
  *total = tot;
  return base + incl - v;
}

// Decoupled look-back over states [first, self): returns the combined (count, max1) of all
// predecessors.  Called by one full warp.
__device__ __forceinline__ void lookback(const u64* state, int first, int self, int lane, u32* cnt, u32* mx1) {
  u32 c = 0, m = 0;
  int look = self - 1;
  while (look >= first) {
    int idx = look - lane;
    u64 v;
    bool real = idx >= first;
    do {
      v = real ? ld_state(state + idx) : kStIncl;    // virtual zero inclusive before the event start
    } while (__any_sync(0xFFFFFFFFu, st_status(v) == 0));
    u32 inclMask = __ballot_sync(0xFFFFFFFFu, st_status(v) == 2);
    int upto = inclMask ? (__ffs(inclMask) - 1) : 31;
    u32 cc = lane <= upto ? st_count(v) : 0, mm = lane <= upto ? st_max1(v) : 0;
    c += __reduce_add_sync(0xFFFFFFFFu, cc);
    m = max(m, __reduce_max_sync(0xFFFFFFFFu, mm));
    if (inclMask) break;
    look -= 32;
  }
  *cnt = c; *mx1 = m;
}


// CTA-wide decoupled look-back (blockDim = 256): thread j reads the state of unit (self-1-j), so
// one round covers 256 predecessors.  With hundreds of units in flight, a 32-wide window needed
// one serial L2 round trip per 32 predecessors and dominated the kernels.  Every thread returns
// the combined (count, max1) of all predecessors in [0, self).  Contains __syncthreads.
struct LbShared { u32 cnt[8], mx[8]; };
__device__ __forceinline__ void lookback_cta(const u64* state, int self, LbShared& lb, u32* cnt, u32* mx1) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  u32 c = 0, m = 0;
  int look = self - 1;
  while (look >= 0) {                                  // block-uniform
    const int idx = look - tid;
    u64 v = kStIncl;                                   // virtual zero inclusive before unit 0
    if (idx >= 0) do { v = ld_state(state + idx); } while (st_status(v) == 0);
    const u32 inclMask = __ballot_sync(0xFFFFFFFFu, st_status(v) == 2);
    const int upto = inclMask ? (__ffs(inclMask) - 1) : 31;
    const u32 cc = lane <= upto ? st_count(v) : 0, mm = lane <= upto ? st_max1(v) : 0;
    const u32 wc = __reduce_add_sync(0xFFFFFFFFu, cc), wm = __reduce_max_sync(0xFFFFFFFFu, mm);
    __syncthreads();                                   // previous readers of lb are done
    if (lane == 0) { lb.cnt[warp] = wc; lb.mx[warp] = wm | (inclMask ? 0x80000000u : 0u); }
    __syncthreads();
    bool found = false;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (!found) {
        c += lb.cnt[k];
        const u32 x = lb.mx[k];
        m = max(m, x & 0xFFFu);
        found = (x >> 31) != 0;
      }
    }
    if (found) break;
    look -= 256;
  }
  *cnt = c; *mx1 = m;
}

template <bool kSingle>
__device__ __forceinline__ const EvDesc& pick_event_by_tile(const EvDesc& single, const EvDesc* batch, u32 nEv, u32 t, u32* e) {
  if (kSingle) { *e = 0; return single; }
  u32 lo = 0, hi = nEv - 1;                          // last event with tileBase <= t
  while (lo < hi) {
    u32 mid = (lo + hi + 1) >> 1;
    if (batch[mid].tileBase <= t) lo = mid; else hi = mid - 1;
  }
  *e = lo;
  return batch[lo];
}

// ================================================================== k_unpack (a1 + a2)
// One CTA per tile of 2048 words, 8 consecutive words per thread (2 x LDG.128 words + 1 x LDG.128
// adc).  Algorithmic HBM bytes per event: 6W read + 16D (digi SoA incl. charge) + 8E written.
template <bool kSingle>
__global__ void __launch_bounds__(kUnpackThreads, 4)
k_unpack(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv,
         LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  __shared__ __align__(16) u32 sWord[kTileWords + 8];
  __shared__ __align__(16) u16 sAdc[kTileWords + 8];
  __shared__ __align__(16) u16 sOff[kTileWords + 8];
  __shared__ u32 sWsum[8], sWmax[8];
  __shared__ LbShared sLb;
  __shared__ u32 sTicket;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) sTicket = atomicAdd(&lc->tileTicket, 1u);
  __syncthreads();
  const u32 t = sTicket;
  u32 e;
  const EvDesc& ev = pick_event_by_tile<kSingle>(single, batch, nEv, t, &e);
  const u32 tile = t - ev.tileBase, W = ev.nWords;
  const u32 i0 = tile * kTileWords + tid * kWordsPerThread;

  // ---- load 8 words + 8 adc
  u32 w[8]; u16 a[8];
  if (i0 + 8 <= W) {
    const uint4 w0 = __ldg(reinterpret_cast<const uint4*>(ev.words + i0));
    const uint4 w1 = __ldg(reinterpret_cast<const uint4*>(ev.words + i0) + 1);
    const uint4 aa = __ldg(reinterpret_cast<const uint4*>(ev.adc + i0));
    w[0] = w0.x; w[1] = w0.y; w[2] = w0.z; w[3] = w0.w; w[4] = w1.x; w[5] = w1.y; w[6] = w1.z; w[7] = w1.w;
    a[0] = (u16)aa.x; a[1] = (u16)(aa.x >> 16); a[2] = (u16)aa.y; a[3] = (u16)(aa.y >> 16);
    a[4] = (u16)aa.z; a[5] = (u16)(aa.z >> 16); a[6] = (u16)aa.w; a[7] = (u16)(aa.w >> 16);
  } else {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const bool in = i0 + j < W;
      w[j] = in ? __ldg(ev.words + i0 + j) : 0u;
      a[j] = in ? __ldg(ev.adc + i0 + j) : (u16)0;
    }
  }
  // ---- decode validity (A2, A3): digi iff !bit31 and module<M and row<R and col<C
  u32 vmask = 0, inmask = 0, max1 = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const u32 x = w[j];
    const u32 mod = (x >> 20) & 0x7FFu, row = (x >> 12) & 0xFFu, col = (x >> 3) & 0x1FFu;
    const bool in = i0 + j < W;
    const bool ok = in && !(x >> 31) && mod < g.M && row < g.R && col < g.C;
    inmask |= (u32)in << j;
    vmask |= (u32)ok << j;
    if (ok) max1 = max(max1, mod + 1);
  }
  const u32 cnt = __popc(vmask);
  const u32 incl = warp_incl_scan(cnt, lane);
  const u32 wmax = __reduce_max_sync(0xFFFFFFFFu, max1);
  if (lane == 31) { sWsum[warp] = incl; sWmax[warp] = wmax; }
  __syncthreads();
  u32 wbase = 0, tileCnt = 0, tileMax1 = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const u32 s = sWsum[k];
    if (k < warp) wbase += s;
    tileCnt += s;
    tileMax1 = max(tileMax1, sWmax[k]);
  }
  const u32 r0 = wbase + incl - cnt;                 // tile-local rank of this thread's first digi

  // ---- decoupled look-back for the event-global digi offset and running max(module)+1
  u32 g0 = 0, carryMax1 = 0;
  {
    u64* state = ev.tileState;
    if (tile > 0) {
      if (tid == 0) st_state(state + tile, pack_state(kStAgg, tileCnt, tileMax1));
      lookback_cta(state, (int)tile, sLb, &g0, &carryMax1);
    }
    if (tid == 0) st_state(state + tile, pack_state(kStIncl, g0 + tileCnt, max(carryMax1, tileMax1)));
  }
  const u32 ph = g0 & 7u;                            // smem phase = global 16-byte phase of u16 arrays

  // ---- compact into shared memory; errors straight to global (rare)
  {
    u32 p = ph + r0, before = g0 + r0;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (vmask >> j & 1) {
        sWord[p] = w[j]; sAdc[p] = a[j]; sOff[p] = (u16)(tid * kWordsPerThread + j);
        ++p; ++before;
      } else if (inmask >> j & 1) {
        const u32 i = i0 + j, ei = i - before;       // errors before i = i - digis before i
        ev.errWord[ei] = w[j]; ev.errIdx[ei] = i;
      }
    }
  }
  __syncthreads();

  // ---- write out: chunk c covers global digis [ga + 8c, ga + 8c + 8), ga = g0 & ~7
  const u32 ga = g0 - ph, end = ph + tileCnt;
  const u32 nChunks = (end + 7) >> 3;
  const u32 wordBase = tile * kTileWords;
  u32 violation = 0;
  for (u32 c = tid; c < nChunks; c += kUnpackThreads) {
    const u32 sb = c << 3, gb = ga + sb;
    const uint4 x0 = *reinterpret_cast<const uint4*>(sWord + sb);
    const uint4 x1 = *reinterpret_cast<const uint4*>(sWord + sb + 4);
    const uint4 av = *reinterpret_cast<const uint4*>(sAdc + sb);
    const uint4 ov = *reinterpret_cast<const uint4*>(sOff + sb);
    const u32 xs[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
    const u32 a2[4] = {av.x, av.y, av.z, av.w}, o2[4] = {ov.x, ov.y, ov.z, ov.w};
    int prev = (sb > ph) ? (int)((sWord[sb - 1] >> 20) & 0x7FFu) : (int)carryMax1 - 1;
    u32 modv[4], rowv[4], colv[4], widx[8]; float q[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const u32 s = sb + j;
      const bool in = s >= ph && s < end;
      const u32 x = xs[j];
      const u32 mod = in ? (x >> 20) & 0x7FFu : 0u, row = (x >> 12) & 0xFFu, col = (x >> 3) & 0x1FFu;
      const u32 ad = (a2[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu, off = (o2[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu;
      q[j] = __fmaf_rn((float)ad, __ldg(g.gain + mod), __ldg(g.ped + mod));     // A7: one rounding
      widx[j] = wordBase + off;
      if (j & 1) { modv[j >> 1] |= mod << 16; rowv[j >> 1] |= row << 16; colv[j >> 1] |= col << 16; }
      else { modv[j >> 1] = mod; rowv[j >> 1] = row; colv[j >> 1] = col; }
      if (in) {
        if ((int)mod > prev) {
          for (int m = prev + 1; m <= (int)mod; ++m) ev.modDigiStart[m] = gb + j;
          atomicMax(ev.winInv + ((gb + j) >> kWindowLog2), g.M - (u32)(prev + 1));   // first module starting in this digi window
        }
        if ((int)mod < prev) violation = 1;
        prev = (int)mod;
      }
    }
    if (sb >= ph && sb + 8 <= end) {
      *reinterpret_cast<uint4*>(ev.module + gb) = make_uint4(modv[0], modv[1], modv[2], modv[3]);
      *reinterpret_cast<uint4*>(ev.row + gb) = make_uint4(rowv[0], rowv[1], rowv[2], rowv[3]);
      *reinterpret_cast<uint4*>(ev.col + gb) = make_uint4(colv[0], colv[1], colv[2], colv[3]);
      *reinterpret_cast<uint4*>(ev.adcOut + gb) = av;
      *reinterpret_cast<uint4*>(ev.wordIdx + gb) = make_uint4(widx[0], widx[1], widx[2], widx[3]);
      *reinterpret_cast<uint4*>(ev.wordIdx + gb + 4) = make_uint4(widx[4], widx[5], widx[6], widx[7]);
      *reinterpret_cast<float4*>(ev.charge + gb) = make_float4(q[0], q[1], q[2], q[3]);
      *reinterpret_cast<float4*>(ev.charge + gb + 4) = make_float4(q[4], q[5], q[6], q[7]);
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const u32 s = sb + j;
        if (s >= ph && s < end) {
          ev.module[gb + j] = (u16)(modv[j >> 1] >> ((j & 1) * 16));
          ev.row[gb + j] = (u16)(rowv[j >> 1] >> ((j & 1) * 16));
          ev.col[gb + j] = (u16)(colv[j >> 1] >> ((j & 1) * 16));
          ev.adcOut[gb + j] = (u16)(a2[j >> 1] >> ((j & 1) * 16));
          ev.wordIdx[gb + j] = widx[j];
          ev.charge[gb + j] = q[j];
        }
      }
    }
  }
  if (violation) atomicOr(&ev.counters->status, 1u);  // PR_STATUS_INPUT_ORDER (A5)

  // ---- the event's last tile closes modDigiStart and the counters
  if (tile == ev.nTiles - 1) {
    const u32 D = g0 + tileCnt, mx1 = max(carryMax1, tileMax1);
    for (u32 m = mx1 + tid; m <= g.M; m += kUnpackThreads) ev.modDigiStart[m] = D;
    if (tid == 0 && mx1 < g.M) atomicMax(ev.winInv + (D >> kWindowLog2), g.M - mx1);   // trailing empty modules start at D
    if (tid == 0) { ev.counters->nWords = W; ev.counters->nDigis = D; ev.counters->nErrors = W - D; }
  }
}

// ================================================================== k_cluster (a3 + a4)
// Work unit = one "window" of kWindow consecutive digi indices of one event: the CTA owns every
// module whose first digi index falls into the window (k_unpack leaves the first such module in
// winInv[]).  Because a module with more than kWindow digis reaches past the window's end, only
// the LAST module of a window can be that large; all others ("smalls") together hold fewer than
// 2*kWindow = kRangeCap digis.  Units are independent, so no CTA waits on another CTA's progress
// before it has published all of its own counts:
//   sparse path  the smalls of the window are clustered at once: shared-memory hash
//                (module,row,col) -> digi, min-index union-find over the backward neighbours,
//                per-root member lists walked by the root's thread for the exact int64 sums.
//                O(1) work per digi, ~9 block barriers per ~19 modules (Run-3-like occupancy).
//   dense path   a module with more than kWindow digis: occupancy bitmap + popcount ranks,
//                union-find and per-cluster atomics (shared-memory tiers, global workspace beyond).
// Dense numbering of kept clusters: decoupled look-back over per-module states.
constexpr u32 kRangeCap = 2 * kWindow;           // > digis of a window's smalls; local index fits 10 bits
constexpr u32 kHashSlots = 2048;
constexpr u32 kEmpty = 0xFFFFFFFFu;
constexpr int kPerThread = kRangeCap / kClusterThreads;   // 4

__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t w = (bitmapWords + 3) & ~3u;
  size_t dense = (size_t)w * 4 * 2 + (size_t)kSmemDigis * 4 * 2 + (size_t)kSmemClusters * (4 + 4 + 4 + 8 * 3);
  size_t sparse = (size_t)kHashSlots * 4 * 2 + (size_t)kRangeCap * 4 * 5;
  return (dense > sparse ? dense : sparse) + 64;
}

__device__ __forceinline__ u32 uf_find(const volatile u32* parent, u32 x) {
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

// Open-addressing hash: tabKey[h] = module << 17 | row << 9 | col (28 bits), tabVal[h] = minimum
// local digi index on that pixel (duplicates: owner = min index, A6).
__device__ __forceinline__ u32 hash_slot(u32 key) { return (key * 0x9E3779B1u) >> 21; }
__device__ __forceinline__ void hash_insert(u32* tabKey, u32* tabVal, u32 key, u32 idx) {
  u32 h = hash_slot(key);
  for (;;) {
    const u32 old = atomicCAS(tabKey + h, kEmpty, key);
    if (old == kEmpty || old == key) { atomicMin(tabVal + h, idx); return; }
    h = (h + 1) & (kHashSlots - 1);
  }
}
__device__ __forceinline__ u32 hash_find(const u32* tabKey, const u32* tabVal, u32 key) {
  u32 h = hash_slot(key);
  for (;;) {
    const u32 v = tabKey[h];
    if (v == kEmpty) return kInvalid;
    if (v == key) return tabVal[h];
    h = (h + 1) & (kHashSlots - 1);
  }
}

struct ClusterShared {
  u32 scan[8];
  u32 cnt[2][kPerThread * 8];       // per (k, warp): kept roots / all roots
  u32 kb[kPerThread * 8];           // per (k, warp): ballot of kept roots
  u32 offs[kPerThread * 8 + 1];
  u32 ticket, base, last, first;
  LbShared lb;
};

// Number of kept roots with local index < b (b in [0, n]); valid after the scan of the sparse path.
__device__ __forceinline__ u32 kept_prefix(const ClusterShared& sh, u32 b, u32 total) {
  if (b >= kRangeCap) return total;
  const u32 k = b / kClusterThreads, r = b % kClusterThreads, w = r >> 5, l = r & 31;
  return sh.offs[k * 8 + w] + __popc(sh.kb[k * 8 + w] & ((1u << l) - 1u));
}

// Publish this unit's kept-cluster count, look back over the event's earlier windows, publish the
// inclusive prefix.  Returns the dense number of the unit's first kept cluster (all threads).
__device__ __forceinline__ u32 unit_lookback(const EvDesc& ev, u32 j, u32 total, ClusterShared& sh) {
  u32 ec = 0, em = 0;
  if (j > 0) {
    if (threadIdx.x == 0) st_state(ev.winState + j, pack_state(kStAgg, total, 0));
    lookback_cta(ev.winState, (int)j, sh.lb, &ec, &em);
  }
  if (threadIdx.x == 0) st_state(ev.winState + j, pack_state(kStIncl, ec + total, 0));
  return ec;
}

// ---- sparse path: modules [m0, m1) of event ev (m1 > m0), digis [s, s+n), n < kRangeCap, all
// starting in window j.  `extra` = kept clusters of the window's big module (numbered after these).
// Returns the number of kept clusters; *baseOut = dense number of its first kept cluster.
__device__ __forceinline__ u32 cluster_range_sparse(const EvDesc& ev, const Geom& g, u32 j, u32 extra, u32 m0, u32 m1, u32 s, u32 n,
                                                    unsigned char* smemRaw, ClusterShared& sh, u32* baseOut) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  u32* tabKey = reinterpret_cast<u32*>(smemRaw);
  u32* tabVal = tabKey + kHashSlots;
  u32* key = tabVal + kHashSlots;
  u32* parent = key + kRangeCap;
  u32* head = parent + kRangeCap;
  u32* next = head + kRangeCap;
  float* qs = reinterpret_cast<float*>(next + kRangeCap);

  u32 total = 0, nAll = 0;
  u32 kb[kPerThread];
  float cq[kPerThread], cr[kPerThread], cc[kPerThread]; u32 csz[kPerThread]; u32 keptMask = 0;
  if (n > 0) {
    // A: init
    for (u32 i = tid; i < kHashSlots; i += kClusterThreads) { tabKey[i] = kEmpty; tabVal[i] = kInvalid; }
    __syncthreads();
    // B: load, kept flag (A8), hash insert
    u32 myKept = 0;
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      const u32 i = k * kClusterThreads + tid;
      if (i < n) {
        const float q = ev.charge[s + i];
        const bool kept = q >= g.pixThr;
        u32 kk = kInvalid;
        if (kept) {
          kk = (u32)ev.module[s + i] << 17 | (u32)ev.row[s + i] << 9 | (u32)ev.col[s + i];
          hash_insert(tabKey, tabVal, kk, i);
          ++myKept;
        }
        key[i] = kk; qs[i] = q; parent[i] = kept ? i : kInvalid; head[i] = kInvalid;
      }
    }
    myKept = __reduce_add_sync(0xFFFFFFFFu, myKept);
    if (lane == 0 && myKept) atomicAdd(&ev.counters->nKept, myKept);
    __syncthreads();
    // C: unions with backward neighbours: N ? {N} : { NE?, W ? {W} : NW? }; duplicates join their owner
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      const u32 i = k * kClusterThreads + tid;
      if (i >= n) continue;
      const u32 kk = key[i];
      if (kk == kInvalid) continue;
      const u32 owner = hash_find(tabKey, tabVal, kk);
      if (owner != i) { uf_union(parent, i, owner); continue; }
      const u32 row = (kk >> 9) & 0xFFu, col = kk & 0x1FFu;
      u32 j = row ? hash_find(tabKey, tabVal, kk - 512u) : kInvalid;
      if (j != kInvalid) { uf_union(parent, i, j); continue; }
      if (row && col + 1 < g.C) { j = hash_find(tabKey, tabVal, kk - 511u); if (j != kInvalid) uf_union(parent, i, j); }
      j = col ? hash_find(tabKey, tabVal, kk - 1u) : kInvalid;
      if (j != kInvalid) uf_union(parent, i, j);
      else if (row && col) { j = hash_find(tabKey, tabVal, kk - 513u); if (j != kInvalid) uf_union(parent, i, j); }
    }
    __syncthreads();
    // D: flatten and push every kept digi on its root's member list
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      const u32 i = k * kClusterThreads + tid;
      if (i >= n || parent[i] == kInvalid) continue;
      const u32 rt = uf_find(parent, i);
      if (rt != i) parent[i] = rt;
      next[i] = atomicExch(head + rt, i);
    }
    __syncthreads();
    // E: each root walks its list: exact fixed-point sums (A9), cluster threshold
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      const u32 i = k * kClusterThreads + tid;
      const bool isRoot = i < n && parent[i] == i;
      bool keptC = false;
      csz[k] = 0; cq[k] = cr[k] = cc[k] = 0.f;
      if (isRoot) {
        u64 S = 0, Sx = 0, Sy = 0; u32 sz = 0;
        for (u32 j = head[i]; j != kInvalid; j = next[j]) {
          const u32 kj = key[j];
          const u64 qf = (u64)__float2ll_rz(qs[j] * 16384.0f);
          S += qf; Sx += qf * ((kj >> 9) & 0xFFu); Sy += qf * (kj & 0x1FFu); ++sz;
        }
        keptC = (i64)S >= g.clusThrFixed;
        if (keptC) {
          const double dS = __ll2double_rn((i64)S);
          cq[k] = __double2float_rn(dS * (1.0 / 16384.0));
          cr[k] = __double2float_rn(__ddiv_rn(__ll2double_rn((i64)Sx), dS));
          cc[k] = __double2float_rn(__ddiv_rn(__ll2double_rn((i64)Sy), dS));
          csz[k] = sz;
        }
      }
      kb[k] = __ballot_sync(0xFFFFFFFFu, keptC);
      const u32 rb = __ballot_sync(0xFFFFFFFFu, isRoot);
      keptMask |= (u32)keptC << k;
      if (lane == 0) { sh.cnt[0][k * 8 + warp] = __popc(kb[k]); sh.cnt[1][k * 8 + warp] = __popc(rb); sh.kb[k * 8 + warp] = kb[k]; }
    }
    __syncthreads();
    if (warp == 0) {
      const u32 c0 = sh.cnt[0][lane], c1 = sh.cnt[1][lane];
      const u32 inc = warp_incl_scan(c0, lane);
      const u32 t1 = __reduce_add_sync(0xFFFFFFFFu, c1);
      sh.offs[lane] = inc - c0;
      if (lane == 31) { sh.offs[32] = inc; sh.scan[0] = t1; }
    }
    __syncthreads();
    total = sh.offs[32]; nAll = sh.scan[0];
    // local number of every kept root goes to head[root] (lists are no longer needed)
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      const u32 i = k * kClusterThreads + tid;
      if (i < n && parent[i] == i)
        head[i] = (keptMask >> k & 1) ? sh.offs[k * 8 + warp] + __popc(kb[k] & ((1u << lane) - 1u)) : kInvalid;
    }
  }
  // F: numbering base of this window through the cross-window look-back
  __syncthreads();
  const u32 base = unit_lookback(ev, j, total + extra, sh);
  __syncthreads();
  // G: outputs
  if (n > 0) {
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      const u32 i = k * kClusterThreads + tid;
      if (i >= n) continue;
      const u32 p = parent[i];
      u32 lab = kInvalid; int32_t cl = -1;
      if (p != kInvalid) {
        lab = s + p;
        const u32 kn = head[p];
        cl = kn == kInvalid ? -1 : (int32_t)(base + kn);
      }
      ev.label[s + i] = lab; ev.clus[s + i] = cl;
      if (keptMask >> k & 1) {
        const u32 o = base + head[i];
        if (o < ev.cap) {
          ev.clLabel[o] = s + i; ev.clModule[o] = (u16)(key[i] >> 17); ev.clSize[o] = csz[k];
          ev.clCharge[o] = cq[k]; ev.clRow[o] = cr[k]; ev.clCol[o] = cc[k];
        }
      }
    }
  }
  // modClusStart[m] = base + kept clusters rooted before the module's first digi
  for (u32 m = m0 + tid; m < m1; m += kClusterThreads)
    ev.modClusStart[m] = base + (n > 0 ? kept_prefix(sh, ev.modDigiStart[m] - s, total) : 0u);
  if (tid == 0 && nAll) atomicAdd(&ev.counters->nClustersAll, nAll);
  *baseOut = base;
  return total;
}

// ---- dense path: one module m with digis [s, s+nn), in two halves so that the caller can publish
// the module's count before it waits for anything (count) and write outputs later (output).
// `deferred`: shared memory will be reused in between, so every array that must survive lives in
// the global workspace tier.
struct DenseCtx {
  u32 *perm, *parent, *root, *csize; int32_t* knum; u64 *S, *Sx, *Sy;
  u32 nAll, nKept;
};

__device__ __forceinline__ void dense_count(const EvDesc& ev, const Geom& g, u32 s, u32 nn, bool deferred,
                                            unsigned char* smemRaw, ClusterShared& sh, DenseCtx& cx) {
  const int tid = threadIdx.x, lane = tid & 31;
  const u32 bwPad = (g.bitmapWords + 3) & ~3u;
  u64* smS = reinterpret_cast<u64*>(smemRaw);
  u64* smSx = smS + kSmemClusters;
  u64* smSy = smSx + kSmemClusters;
  u32* smBitmap = reinterpret_cast<u32*>(smSy + kSmemClusters);
  u32* smPrefix = smBitmap + bwPad;
  u32* smPerm = smPrefix + bwPad;
  u32* smParent = smPerm + kSmemDigis;
  u32* smRoot = smParent + kSmemDigis;
  u32* smSize = smRoot + kSmemClusters;
  int32_t* smKnum = reinterpret_cast<int32_t*>(smSize + kSmemClusters);
  u32* sScan = sh.scan;
  const u32 stride = g.stride;

  const bool digiInSmem = !deferred && nn <= kSmemDigis;
  u32* perm = digiInSmem ? smPerm : ev.wsPerm + s;
  u32* parent = digiInSmem ? smParent : ev.wsParent + s;
  cx.perm = perm; cx.parent = parent;
  cx.root = smRoot; cx.csize = smSize; cx.knum = smKnum; cx.S = smS; cx.Sx = smSx; cx.Sy = smSy;

  // P0: clear the occupancy bitmap, init perm
  for (u32 i = tid; i < g.bitmapWords; i += kClusterThreads) smBitmap[i] = 0;
  for (u32 i = tid; i < nn; i += kClusterThreads) perm[i] = kInvalid;
  __syncthreads();
  // P1: kept flag (A8: q >= pixThr) and occupancy bits at padded coordinates (row+1, col+1)
  u32 myKept = 0;
  for (u32 i = tid; i < nn; i += kClusterThreads) {
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
    const u32 per = (g.bitmapWords + kClusterThreads - 1) / kClusterThreads;
    const u32 lo = min(tid * per, g.bitmapWords), hi = min(lo + per, g.bitmapWords);
    u32 sum = 0;
    for (u32 i = lo; i < hi; ++i) sum += __popc(smBitmap[i]);
    u32 tot;
    u32 run = block_excl_scan(sum, sScan, &tot);
    for (u32 i = lo; i < hi; ++i) { smPrefix[i] = run; run += __popc(smBitmap[i]); }
  }
  if (lane == 0 && myKept) atomicAdd(&ev.counters->nKept, myKept);
  __syncthreads();
  // P3: owner of each occupied pixel = the minimum digi index on it (duplicates, A6)
  for (u32 i = tid; i < nn; i += kClusterThreads) {
    if (parent[i] == kInvalid) continue;
    const u32 b = ev.col[s + i] + 1u, wd = (ev.row[s + i] + 1u) * stride + (b >> 5);
    const u32 r = smPrefix[wd] + __popc(smBitmap[wd] & ((1u << (b & 31)) - 1u));
    atomicMin(perm + r, i);
  }
  __syncthreads();
  // P4: unions with the backward neighbours (W, NW, N, NE), decision tree:
  //     N ? {N} : { NE?, W ? {W} : NW? }   — spans every 8-adjacency once all pixels did it.
  for (u32 i = tid; i < nn; i += kClusterThreads) {
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
  for (u32 i = tid; i < nn; i += kClusterThreads) {
    if (parent[i] == kInvalid) continue;
    const u32 rt = uf_find(parent, i);
    if (rt != i) parent[i] = rt;
  }
  __syncthreads();
  // P6: ordinal of every root in ascending index (= ascending label) order -> perm[root]
  {
    const u32 per = (nn + kClusterThreads - 1) / kClusterThreads;
    const u32 lo = min(tid * per, nn), hi = min(lo + per, nn);
    u32 c = 0;
    for (u32 i = lo; i < hi; ++i) c += (parent[i] == i);
    u32 run = block_excl_scan(c, sScan, &cx.nAll);
    if (deferred || cx.nAll > kSmemClusters) {
      cx.root = ev.wsRoot + s; cx.csize = ev.wsSize + s; cx.knum = ev.wsKnum + s;
      cx.S = ev.wsS + s; cx.Sx = ev.wsSx + s; cx.Sy = ev.wsSy + s;
    }
    for (u32 i = lo; i < hi; ++i)
      if (parent[i] == i) { perm[i] = run; cx.root[run] = i; ++run; }
  }
  // P7: zero the accumulators
  for (u32 c = tid; c < cx.nAll; c += kClusterThreads) { cx.S[c] = 0; cx.Sx[c] = 0; cx.Sy[c] = 0; cx.csize[c] = 0; }
  __syncthreads();
  // P8: exact fixed-point sums (A9): qf = q * 2^14 is an integer for every kept digi
  for (u32 i = tid; i < nn; i += kClusterThreads) {
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
    const u32 per = (cx.nAll + kClusterThreads - 1) / kClusterThreads;
    const u32 lo = min(tid * per, cx.nAll), hi = min(lo + per, cx.nAll);
    u32 c = 0;
    for (u32 k = lo; k < hi; ++k) c += ((i64)cx.S[k] >= g.clusThrFixed);
    u32 run = block_excl_scan(c, sScan, &cx.nKept);
    for (u32 k = lo; k < hi; ++k) cx.knum[k] = ((i64)cx.S[k] >= g.clusThrFixed) ? (int32_t)run++ : -1;
  }
  __syncthreads();
}

__device__ __forceinline__ void dense_output(const EvDesc& ev, u32 m, u32 s, u32 nn, u32 base, const DenseCtx& cx) {
  const int tid = threadIdx.x;
  for (u32 k = tid; k < cx.nAll; k += kClusterThreads) {
    const int32_t kn = cx.knum[k];
    if (kn < 0) continue;
    const u32 o = base + (u32)kn;
    if (o >= ev.cap) continue;                      // cannot happen (N <= D <= cap); stay in bounds
    const double dS = __ll2double_rn((i64)cx.S[k]);
    ev.clLabel[o] = s + cx.root[k];
    ev.clModule[o] = (u16)m;
    ev.clSize[o] = cx.csize[k];
    ev.clCharge[o] = __double2float_rn(dS * (1.0 / 16384.0));
    ev.clRow[o] = __double2float_rn(__ddiv_rn(__ll2double_rn((i64)cx.Sx[k]), dS));
    ev.clCol[o] = __double2float_rn(__ddiv_rn(__ll2double_rn((i64)cx.Sy[k]), dS));
  }
  for (u32 i = tid; i < nn; i += kClusterThreads) {
    const u32 p = cx.parent[i];
    u32 lab = kInvalid; int32_t cl = -1;
    if (p != kInvalid) {
      lab = s + p;
      const int32_t kn = cx.knum[cx.perm[p]];
      cl = kn < 0 ? -1 : (int32_t)(base + (u32)kn);
    }
    ev.label[s + i] = lab;
    ev.clus[s + i] = cl;
  }
  if (tid == 0) {
    ev.modClusStart[m] = base;
    if (cx.nAll) atomicAdd(&ev.counters->nClustersAll, cx.nAll);
  }
}

template <bool kSingle>
__device__ __forceinline__ const EvDesc& pick_event_by_window(const EvDesc& single, const EvDesc* batch, u32 nEv, u32 t) {
  if (kSingle) return single;
  u32 lo = 0, hi = nEv - 1;                          // last event with winBase <= t
  while (lo < hi) {
    u32 mid = (lo + hi + 1) >> 1;
    if (batch[mid].winBase <= t) lo = mid; else hi = mid - 1;
  }
  return batch[lo];
}

template <bool kSingle>
__global__ void __launch_bounds__(kClusterThreads)
k_cluster(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv, u32 totalWindows,
          LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ ClusterShared sh;
  const int tid = threadIdx.x;

  for (;;) {
    __syncthreads();
    if (tid == 0) sh.ticket = atomicAdd(&lc->modTicket, 1u);
    __syncthreads();
    const u32 ticket = sh.ticket;
    if (ticket >= totalWindows) break;
    const EvDesc& ev = pick_event_by_window<kSingle>(single, batch, nEv, ticket);
    const u32 j = ticket - ev.winBase;
    const u32 wi = ev.winInv[j];
    // An event that violated the input contract (A5) has undefined modDigiStart: no per-digi work.
    const bool bad = (ev.counters->status & 1u) != 0;
    if (wi != 0 && !bad) {
      const u32 first = g.M - wi, hi = (j + 1) << kWindowLog2;
      // modules whose first digi lies in this window: [first, mEnd)
      u32 mEnd = first;
      for (;;) {
        const u32 m = mEnd + tid;
        const int c = __syncthreads_count(m < g.M && ev.modDigiStart[m] < hi);
        mEnd += (u32)c;
        if (c < kClusterThreads) break;
      }
      const u32 s = ev.modDigiStart[first];
      const u32 sLastMod = ev.modDigiStart[mEnd - 1], sEnd = ev.modDigiStart[mEnd];
      const bool bigLast = sEnd - sLastMod > kWindow;
      const u32 smallEnd = bigLast ? mEnd - 1 : mEnd;
      const bool haveSmall = smallEnd > first;
      const bool sane = s <= sLastMod && sLastMod <= sEnd && sEnd <= ev.cap && (!haveSmall || ev.modDigiStart[smallEnd] - s < kRangeCap);
      if (sane) {
        DenseCtx cx;
        const u32 mBig = mEnd - 1, nBig = sEnd - sLastMod;
        if (bigLast) dense_count(ev, g, sLastMod, nBig, haveSmall, smemRaw, sh, cx);   // count first: nobody waits on us
        const u32 nBigKept = bigLast ? cx.nKept : 0u;
        u32 base = 0;
        if (haveSmall) {
          const u32 total = cluster_range_sparse(ev, g, j, nBigKept, first, smallEnd, s, ev.modDigiStart[smallEnd] - s, smemRaw, sh, &base);
          base += total;
        } else {
          base = unit_lookback(ev, j, nBigKept, sh);
        }
        if (bigLast) {
          dense_output(ev, mBig, sLastMod, nBig, base, cx);
          base += nBigKept;
        }
        if (mEnd == g.M && tid == 0) { ev.modClusStart[g.M] = base; ev.counters->nClusters = base; }
      } else {
        if (tid == 0) atomicOr(&ev.counters->status, 2u);   // PR_STATUS_CAPACITY: inconsistent module table
        unit_lookback(ev, j, 0, sh);
      }
    } else {
      // empty window (or bad event): transparent to its successors, no look-back of its own
      if (tid == 0) st_state(ev.winState + j, pack_state(j > 0 ? kStAgg : kStIncl, 0, 0));
    }
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      sh.last = (atomicAdd(&lc->modDone, 1u) == totalWindows - 1);
    }
    __syncthreads();
    if (sh.last) {
      // the launch's last unit: publish every event's counters to mapped pinned host memory
      __threadfence();
      for (u32 k = tid; k < nEv; k += kClusterThreads) {
        const EvDesc& d = kSingle ? single : batch[k];
        const volatile DevCounters* c = d.counters;
        HostCounters h;
        h.nWords = c->nWords; h.nDigis = c->nDigis; h.nErrors = c->nErrors; h.nKept = c->nKept;
        h.nClustersAll = c->nClustersAll; h.nClusters = c->nClusters; h.status = c->status; h.seq = 1;
        *d.hostCounters = h;
      }
    }
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

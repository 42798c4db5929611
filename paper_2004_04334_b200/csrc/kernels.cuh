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
  u64 *tileState, *modState;        // look-back states: [nTiles], [M]
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
__global__ void __launch_bounds__(kUnpackThreads)
k_unpack(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv,
         LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  __shared__ __align__(16) u32 sWord[kTileWords + 8];
  __shared__ __align__(16) u16 sAdc[kTileWords + 8];
  __shared__ __align__(16) u16 sOff[kTileWords + 8];
  __shared__ u32 sWsum[8], sWmax[8];
  __shared__ u32 sTicket, sExclCnt, sExclMax;

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
  if (warp == 0) {
    u64* state = ev.tileState;
    u32 ec = 0, em = 0;
    if (tile > 0) {
      if (lane == 0) st_state(state + tile, pack_state(kStAgg, tileCnt, tileMax1));
      lookback(state, 0, (int)tile, lane, &ec, &em);
    }
    if (lane == 0) {
      st_state(state + tile, pack_state(kStIncl, ec + tileCnt, max(em, tileMax1)));
      sExclCnt = ec; sExclMax = em;
    }
  }
  __syncthreads();
  const u32 g0 = sExclCnt, carryMax1 = sExclMax;
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
        if ((int)mod > prev) for (int m = prev + 1; m <= (int)mod; ++m) ev.modDigiStart[m] = gb + j;
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
    if (tid == 0) { ev.counters->nWords = W; ev.counters->nDigis = D; ev.counters->nErrors = W - D; }
  }
}

// ================================================================== k_cluster (a3 + a4)
struct ClusterSmem {           // carved from dynamic shared memory by the kernel
  u32 *bitmap, *prefix, *perm, *parent, *root, *size;
  int32_t* knum;
  u64 *S, *Sx, *Sy;
};
__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t w = (bitmapWords + 3) & ~3u;
  return (size_t)w * 4 * 2 + (size_t)kSmemDigis * 4 * 2 + (size_t)kSmemClusters * (4 + 4 + 4 + 8 * 3) + 64;
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

template <bool kSingle>
__global__ void __launch_bounds__(kClusterThreads)
k_cluster(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv,
          LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ u32 sScan[8];
  __shared__ u32 sTicket, sBase, sLast;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
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

  const u32 totalModules = nEv * g.M;
  const u32 stride = g.stride;

  for (;;) {
    __syncthreads();
    if (tid == 0) sTicket = atomicAdd(&lc->modTicket, 1u);
    __syncthreads();
    const u32 ticket = sTicket;
    if (ticket >= totalModules) break;
    const u32 e = kSingle ? 0u : ticket / g.M, m = kSingle ? ticket : ticket - e * g.M;
    const EvDesc& ev = kSingle ? single : batch[e];
    const u32 s = ev.modDigiStart[m], n = ev.modDigiStart[m + 1] - s;
    const bool order_bad = (ev.counters->status & 1u) != 0;   // outputs undefined then; stay in bounds
    const u32 nn = (order_bad || s + n > ev.cap || s > ev.cap) ? 0u : n;

    u32 nKeptDigis = 0, nAll = 0, nKeptClusters = 0;
    const bool digiInSmem = nn <= kSmemDigis;
    u32* perm = digiInSmem ? smPerm : ev.wsPerm + s;
    u32* parent = digiInSmem ? smParent : ev.wsParent + s;
    bool clInSmem = true;
    u32* root = smRoot; u32* csize = smSize; int32_t* knum = smKnum; u64 *S = smS, *Sx = smSx, *Sy = smSy;

    if (nn > 0) {
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
      nKeptDigis = 1;   // (only used as "did work" marker below)
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
        const u32 pos = b - 1u, w0 = pos >> 5, sh = pos & 31u;
        const u32 rowAbove = (prow - 1u) * stride, rowSelf = prow * stride;
        const u32 nb = __funnelshift_r(smBitmap[rowAbove + w0], smBitmap[rowAbove + w0 + 1], sh) & 7u;
        const u32 cb = __funnelshift_r(smBitmap[rowSelf + w0], smBitmap[rowSelf + w0 + 1], sh) & 7u;
        // rank of a pixel at padded (rowBase, bit position bb)
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
        u32 run = block_excl_scan(c, sScan, &nAll);
        clInSmem = nAll <= kSmemClusters;
        if (!clInSmem) {
          root = ev.wsRoot + s; csize = ev.wsSize + s; knum = ev.wsKnum + s;
          S = ev.wsS + s; Sx = ev.wsSx + s; Sy = ev.wsSy + s;
        }
        for (u32 i = lo; i < hi; ++i)
          if (parent[i] == i) { perm[i] = run; root[run] = i; ++run; }
      }
      // P7: zero the accumulators
      for (u32 c = tid; c < nAll; c += kClusterThreads) { S[c] = 0; Sx[c] = 0; Sy[c] = 0; csize[c] = 0; }
      __syncthreads();
      // P8: exact fixed-point sums (A9): qf = q * 2^14 is an integer for every kept digi
      for (u32 i = tid; i < nn; i += kClusterThreads) {
        const u32 p = parent[i];
        if (p == kInvalid) continue;
        const u32 c = perm[p];
        const u64 qf = (u64)__float2ll_rz(ev.charge[s + i] * 16384.0f);
        atomicAdd(reinterpret_cast<unsigned long long*>(S + c), (unsigned long long)qf);
        atomicAdd(reinterpret_cast<unsigned long long*>(Sx + c), (unsigned long long)(qf * ev.row[s + i]));
        atomicAdd(reinterpret_cast<unsigned long long*>(Sy + c), (unsigned long long)(qf * ev.col[s + i]));
        atomicAdd(csize + c, 1u);
      }
      __syncthreads();
      // P9: cluster threshold (A8, A9) and local numbering of kept clusters
      {
        const u32 per = (nAll + kClusterThreads - 1) / kClusterThreads;
        const u32 lo = min(tid * per, nAll), hi = min(lo + per, nAll);
        u32 c = 0;
        for (u32 k = lo; k < hi; ++k) c += ((i64)S[k] >= g.clusThrFixed);
        u32 run = block_excl_scan(c, sScan, &nKeptClusters);
        for (u32 k = lo; k < hi; ++k) knum[k] = ((i64)S[k] >= g.clusThrFixed) ? (int32_t)run++ : -1;
      }
    }
    // P10: dense numbering across modules: decoupled look-back over the event's modules
    if (warp == 0) {
      u32 ec = 0, em = 0;
      if (m > 0) {
        if (lane == 0) st_state(ev.modState + m, pack_state(kStAgg, nKeptClusters, 0));
        lookback(ev.modState, 0, (int)m, lane, &ec, &em);
      }
      if (lane == 0) {
        st_state(ev.modState + m, pack_state(kStIncl, ec + nKeptClusters, 0));
        sBase = ec;
      }
    }
    __syncthreads();
    const u32 base = sBase;
    // P11: outputs
    if (nn > 0) {
      for (u32 k = tid; k < nAll; k += kClusterThreads) {
        const int32_t kn = knum[k];
        if (kn < 0) continue;
        const u32 o = base + (u32)kn;
        if (o >= ev.cap) continue;                      // cannot happen (N <= D <= cap); stay in bounds
        const double dS = __ll2double_rn((i64)S[k]);
        ev.clLabel[o] = s + root[k];
        ev.clModule[o] = (u16)m;
        ev.clSize[o] = csize[k];
        ev.clCharge[o] = __double2float_rn(dS * (1.0 / 16384.0));
        ev.clRow[o] = __double2float_rn(__ddiv_rn(__ll2double_rn((i64)Sx[k]), dS));
        ev.clCol[o] = __double2float_rn(__ddiv_rn(__ll2double_rn((i64)Sy[k]), dS));
      }
      for (u32 i = tid; i < nn; i += kClusterThreads) {
        const u32 p = parent[i];
        u32 lab = kInvalid; int32_t cl = -1;
        if (p != kInvalid) {
          lab = s + p;
          const int32_t kn = knum[perm[p]];
          cl = kn < 0 ? -1 : (int32_t)(base + (u32)kn);
        }
        ev.label[s + i] = lab;
        ev.clus[s + i] = cl;
      }
    } else if (order_bad) {
      // undefined-but-initialised outputs for an event that violated the input contract
      for (u32 i = tid; i < n && s + i < ev.cap; i += kClusterThreads) { ev.label[s + i] = kInvalid; ev.clus[s + i] = -1; }
    }
    if (tid == 0) {
      ev.modClusStart[m] = base;
      if (nAll) atomicAdd(&ev.counters->nClustersAll, nAll);
      if (m == g.M - 1) { ev.modClusStart[g.M] = base + nKeptClusters; ev.counters->nClusters = base + nKeptClusters; }
      __threadfence();
      sLast = (atomicAdd(&lc->modDone, 1u) == totalModules - 1);
    }
    (void)nKeptDigis;
    __syncthreads();
    if (sLast) {
      // the launch's last module: publish every event's counters to mapped pinned host memory
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

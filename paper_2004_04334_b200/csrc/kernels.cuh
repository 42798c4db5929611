// kernels.cuh — sm_100a device code of the hot path (BASELINE.json north_star subsystem (2)).
//
//   k_unpack   a1+a2 fused: raw word decode, calibration, STABLE digi/error compaction with a
//              single-pass decoupled look-back scan, modDigiStart, input-order check.
//   k_cluster  a3+a4 fused: per-module 8-connected components (warp per module: hash look-up +
//              label equivalence in shared memory; CTA per large module: bitmap + rank look-up +
//              min-index union-find), exact cluster sums, cluster threshold, per-module numbering.
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
constexpr int kTileWords = 8 * kUnpackThreads;                       // 2048: each thread owns two runs of 4 consecutive words
constexpr int kLookBack = 8;                                         // predecessor states per lane and look-back round (256 per round)

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
  u32 modTicket, modDone, pad[14];
};
// What the host reads after completion (mapped pinned memory, written by the last block).
struct HostCounters {
  u32 nWords, nDigis, nErrors, nKept, nClustersAll, nClusters, status, seq;
};

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
// consecutive words of one event; the grid never exceeds what is co-resident).  Thread t owns words
// [4t, 4t+4) and [1024 + 4t, 1024 + 4t + 4) of the tile: one LDG.128 + one LDG.64 per run.
// The loop is software-pipelined over tiles so that no phase waits for another CTA:
//   A(i)  decode + validity (A2, A3), packed warp scan of the two runs' counts, publish the tile
//         aggregate, stage every word in shared memory (digis at their position in the tile,
//         error words behind them), issue the loads of tile i+1, issue the look-back loads of tile i
//   B(i-1) write the previous tile from shared memory: its event-global digi offset g0 is known by
//         now; a quad of 4 consecutive digis aligned to the OUTPUT position becomes one 8- or
//         16-byte store per array (module,row,col,adc u16; wordIdx u32; charge f32 = fmaf, A7);
//         module boundaries (modDigiStart) and order violations (A5) come from comparing each
//         digi with the one before it; error words (rare) are copied out behind
//   R(i)  warp 0 resolves tile i's look-back (its loads flew during B) and publishes the
//         inclusive state
// The stage is kept in four planes (slot s lives at plane s & 3, index s >> 2), so that both the
// scattered staging stores and the output-aligned quad reads are free of bank conflicts whatever
// g0 mod 4 is.
// Algorithmic HBM bytes per event: 6W read + 16D (digi SoA incl. charge) + 8E written.
constexpr u32 kStagePlane = kTileWords / 4 + 4;
__device__ __forceinline__ u32 stage_idx(u32 s) { return (s & 3u) * kStagePlane + (s >> 2); }

struct UnpackStage { u32 x[4 * kStagePlane], a[4 * kStagePlane]; };   // raw word; adc | (word offset in tile) << 16
struct UnpackShared {
  UnpackStage st[2];                // tile i is staged in st[i & 1]; slot = 4 + position
  uint2 wagg[8];                    // per warp: packed counts of the two runs, max(module)+1
  u32 g0, carry1;                   // look-back result of the tile just resolved
  u32 desc[4][32];                  // batch: descriptors of the previous, this, the next tile and the one after
};

struct RawTile { uint4 xa, xb; uint2 aa, ab; };   // aa/ab: four u16 adc values each

__device__ __forceinline__ void unpack_load(const u32* __restrict__ words, const u16* __restrict__ adc, u32 W, u32 tileInEv,
                                            u32 tid, RawTile& r) {
  const u32 T0 = tileInEv * (u32)kTileWords;
  if (T0 + (u32)kTileWords <= W) {
    r.xa = __ldcs(reinterpret_cast<const uint4*>(words + T0) + tid);
    r.xb = __ldcs(reinterpret_cast<const uint4*>(words + T0 + kTileWords / 2) + tid);
    r.aa = __ldcs(reinterpret_cast<const uint2*>(adc + T0) + tid);
    r.ab = __ldcs(reinterpret_cast<const uint2*>(adc + T0 + kTileWords / 2) + tid);
  } else {                                             // the event's ragged last tile: words beyond W read as invalid
    u32 x[8], a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const u32 i = T0 + (j < 4 ? 0u : (u32)kTileWords / 2) + 4u * tid + (u32)(j & 3);
      const bool in = i < W;
      x[j] = in ? __ldcs(words + i) : 0xFFFFFFFFu;
      a[j] = in ? (u32)__ldcs(adc + i) : 0u;
    }
    r.xa = make_uint4(x[0], x[1], x[2], x[3]); r.xb = make_uint4(x[4], x[5], x[6], x[7]);
    r.aa = make_uint2(a[0] | a[1] << 16, a[2] | a[3] << 16); r.ab = make_uint2(a[4] | a[5] << 16, a[6] | a[7] << 16);
  }
}

// B: write one staged tile.  n digis at event positions [g0, g0 + n); carry1 = module + 1 of the
// digi before the tile (0 if none); the tile's in-range words are [wordBase, wordBase + inRange).
__device__ __forceinline__ void unpack_write(const EvDesc& ev, const Geom& g, const UnpackStage& st, u32 tid, u32 tile, u32 n,
                                             u32 tileMax1, u32 g0, u32 carry1) {
  const u32 ph = g0 & 3u, base4 = g0 & ~3u, nQ = (ph + n + 3u) >> 2, wordBase = tile * (u32)kTileWords, W = ev.nWords;
  const u32 fake = ((carry1 - 1u) & 0xFFFu) << 20;       // stands for "the digi before this tile"
  u32 violation = 0;
  for (u32 q = tid; q < nQ; q += kUnpackThreads) {
    const u32 p0 = base4 + 4u * q, s0 = 4u * q + 4u - ph;  // output element p0 + j <- stage slot s0 + j
    if (4u * q >= ph && 4u * q + 4u <= ph + n) {
      u32 xs[5], as[4];
      xs[0] = s0 == 4u ? fake : st.x[stage_idx(s0 - 1u)];
#pragma unroll
      for (int j = 0; j < 4; ++j) { xs[j + 1] = st.x[stage_idx(s0 + (u32)j)]; as[j] = st.a[stage_idx(s0 + (u32)j)]; }
      const u32 d = (xs[1] ^ xs[0]) | (xs[2] ^ xs[1]) | (xs[3] ^ xs[2]) | (xs[4] ^ xs[3]);
      float4 ch;
      if ((d >> 20) == 0u) {                             // one module, same as the digi before: the common case
        const float2 gp = __ldg(g.calib + (xs[1] >> 20));
        ch.x = __fmaf_rn((float)(as[0] & 0xFFFFu), gp.x, gp.y); ch.y = __fmaf_rn((float)(as[1] & 0xFFFFu), gp.x, gp.y);
        ch.z = __fmaf_rn((float)(as[2] & 0xFFFFu), gp.x, gp.y); ch.w = __fmaf_rn((float)(as[3] & 0xFFFFu), gp.x, gp.y);
      } else {
        float c4[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const u32 mod = xs[j + 1] >> 20, prev1 = ((xs[j] >> 20) + 1u) & 0xFFFu;
          const float2 gp = __ldg(g.calib + mod);
          c4[j] = __fmaf_rn((float)(as[j] & 0xFFFFu), gp.x, gp.y);
          if (mod + 1u > prev1) {
            for (u32 m = prev1; m <= mod; ++m) ev.modDigiStart[m] = p0 + (u32)j;
          } else if (mod + 1u < prev1) violation = 1;
        }
        ch = make_float4(c4[0], c4[1], c4[2], c4[3]);
      }
      *reinterpret_cast<uint2*>(ev.module + p0) = make_uint2((xs[1] >> 20) | (xs[2] >> 20) << 16, (xs[3] >> 20) | (xs[4] >> 20) << 16);
      *reinterpret_cast<uint2*>(ev.row + p0) = make_uint2(((xs[1] >> 12) & 0xFFu) | ((xs[2] >> 12) & 0xFFu) << 16,
                                                          ((xs[3] >> 12) & 0xFFu) | ((xs[4] >> 12) & 0xFFu) << 16);
      *reinterpret_cast<uint2*>(ev.col + p0) = make_uint2(((xs[1] >> 3) & 0x1FFu) | ((xs[2] >> 3) & 0x1FFu) << 16,
                                                          ((xs[3] >> 3) & 0x1FFu) | ((xs[4] >> 3) & 0x1FFu) << 16);
      *reinterpret_cast<uint2*>(ev.adcOut + p0) = make_uint2(__byte_perm(as[0], as[1], 0x5410), __byte_perm(as[2], as[3], 0x5410));
      *reinterpret_cast<uint4*>(ev.wordIdx + p0) = make_uint4(wordBase + (as[0] >> 16), wordBase + (as[1] >> 16),
                                                              wordBase + (as[2] >> 16), wordBase + (as[3] >> 16));
      *reinterpret_cast<float4*>(ev.charge + p0) = ch;
    } else {                                              // the tile's first and last quad may be partial
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const u32 pos = 4u * q + (u32)j - ph;             // position in the tile (wraps below 0)
        if (pos >= n) continue;
        const u32 xx = st.x[stage_idx(pos + 4u)], aa = st.a[stage_idx(pos + 4u)];
        const u32 xp = pos ? st.x[stage_idx(pos + 3u)] : fake;
        const u32 mod = xx >> 20, prev1 = ((xp >> 20) + 1u) & 0xFFFu, p = p0 + (u32)j;
        const float2 gp = __ldg(g.calib + mod);
        ev.module[p] = (u16)mod; ev.row[p] = (u16)((xx >> 12) & 0xFFu); ev.col[p] = (u16)((xx >> 3) & 0x1FFu);
        ev.adcOut[p] = (u16)(aa & 0xFFFFu); ev.wordIdx[p] = wordBase + (aa >> 16);
        ev.charge[p] = __fmaf_rn((float)(aa & 0xFFFFu), gp.x, gp.y);
        if (mod + 1u > prev1) {
          for (u32 m = prev1; m <= mod; ++m) ev.modDigiStart[m] = p;
        } else if (mod + 1u < prev1) violation = 1;
      }
    }
  }
  if (violation) atomicOr(&ev.counters->status, 1u);     // PR_STATUS_INPUT_ORDER (A5)
  // ---- error words (A2-A4): staged behind the digis in word order; errors before the tile = words - digis before it
  {
    const u32 inRange = W > wordBase ? min(W - wordBase, (u32)kTileWords) : 0u, nErr = inRange - n, e0 = wordBase - g0;
    for (u32 e = tid; e < nErr; e += kUnpackThreads) {
      const u32 s = stage_idx(n + e + 4u);
      ev.errWord[e0 + e] = st.x[s]; ev.errIdx[e0 + e] = wordBase + (st.a[s] >> 16);
    }
  }
  // ---- the event's last tile closes modDigiStart and the counters
  if (tile == ev.nTiles - 1u) {
    const u32 D = g0 + n, mx1 = max(carry1, tileMax1);
    for (u32 m = mx1 + tid; m <= g.M; m += kUnpackThreads) ev.modDigiStart[m] = D;
    if (tid == 0) { ev.counters->nWords = W; ev.counters->nDigis = D; ev.counters->nErrors = W - D; }
  }
}

template <bool kSingle>
__global__ void __launch_bounds__(kUnpackThreads, 4)
k_unpack(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, const u16* __restrict__ tileEvent,
         u32 totalTiles, const __grid_constant__ Geom g) {
  __shared__ __align__(16) UnpackShared sh;
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, G = gridDim.x;
  u32 t = blockIdx.x;
  if (t >= totalTiles) return;
  u32 prv = 3, cur = 0, nxt = 1, nn = 2, eNN = 0;      // descriptor ring (batch)
  if (!kSingle) {
    if (warp < 2) {
      const u32 tt = min(t + warp * G, totalTiles - 1u);
      sh.desc[warp][lane] = __ldg(reinterpret_cast<const u32*>(batch + tileEvent[tt]) + lane);
      if (warp == 1 && t + 2u * G < totalTiles) eNN = tileEvent[t + 2u * G];
    }
    __syncthreads();
  }
  RawTile raw;
  {
    const EvDesc& ev = kSingle ? single : *reinterpret_cast<const EvDesc*>(sh.desc[0]);
    unpack_load(ev.words, ev.adc, ev.nWords, t - ev.tileBase, tid, raw);
  }
  const u32 limM = g.M, limR = g.R << 12, limC = g.C << 3;
  bool haveA = true, haveB = false;
  u32 pTile = 0, pN = 0, pMax1 = 0, pG0 = 0, pCarry1 = 0;          // the previous tile, for B

  for (u32 it = 0;; ++it) {
    const EvDesc& ev = kSingle ? single : *reinterpret_cast<const EvDesc*>(sh.desc[cur]);
    UnpackStage& st = sh.st[it & 1u];
    u32 tile = 0, n = 0, tileMax1 = 0, dword = 0, eN3 = 0;
    u32 x[8], ap[4], vmask = 0, packed = 0, incl = 0;
    RawTile rawNext;
    u64 lb[kLookBack];
    if (haveA) {
      tile = t - ev.tileBase;
      // batch: descriptor of tile t + 2G and event of tile t + 3G, in flight until the end of the iteration
      if (!kSingle && warp == 1) {
        if (t + 2u * G < totalTiles) dword = __ldg(reinterpret_cast<const u32*>(batch + eNN) + lane);
        if (t + 3u * G < totalTiles) eN3 = tileEvent[t + 3u * G];
      }
      // ---- validity (A2, A3): digi iff module < M (bit 31 set makes it >= 2048), row < R, col < C
      x[0] = raw.xa.x; x[1] = raw.xa.y; x[2] = raw.xa.z; x[3] = raw.xa.w; x[4] = raw.xb.x; x[5] = raw.xb.y; x[6] = raw.xb.z; x[7] = raw.xb.w;
      ap[0] = raw.aa.x; ap[1] = raw.aa.y; ap[2] = raw.ab.x; ap[3] = raw.ab.y;
      int mmax = -1;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const u32 mod = x[j] >> 20;
        const bool ok = mod < limM && (x[j] & 0xFF000u) < limR && (x[j] & 0xFF8u) < limC;
        if (ok) { vmask |= 1u << j; mmax = max(mmax, (int)mod); }
      }
      packed = (u32)__popc(vmask & 15u) | (u32)__popc(vmask >> 4) << 16;
      incl = warp_incl_scan(packed, (int)lane);
      const u32 wmax1 = __reduce_max_sync(0xFFFFFFFFu, (u32)(mmax + 1));
      if (lane == 31) sh.wagg[warp] = make_uint2(incl, wmax1);
    }
    __syncthreads();                                                         // #1
    if (haveA) {
      u32 base = 0, tot = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint2 s = sh.wagg[k];
        if (k < (int)warp) base += s.x;
        tot += s.x;
        tileMax1 = max(tileMax1, s.y);
      }
      const u32 tileA = tot & 0xFFFFu;
      n = tileA + (tot >> 16);
      u64* state = ev.tileState;
      if (tid == 0) st_state(state + tile, pack_state(tile ? kStAgg : kStIncl, n, tileMax1));
      // ---- the next tile's loads are issued now and consumed in the next iteration
      if (t + G < totalTiles) {
        const EvDesc& en = kSingle ? single : *reinterpret_cast<const EvDesc*>(sh.desc[nxt]);
        unpack_load(en.words, en.adc, en.nWords, t + G - en.tileBase, tid, rawNext);
      }
      if (warp == 0 && tile) lookback_issue(state, (int)tile, lane, lb);
      // ---- stage: digi k of the tile at slot 4 + k, error word e of the tile at slot 4 + n + e
      const u32 ex = base + incl - packed;
      u32 posA = ex & 0xFFFFu, posB = tileA + (ex >> 16);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const u32 off = (j < 4 ? 0u : (u32)kTileWords / 2) + 4u * tid + (u32)(j & 3);
        const u32 a16 = (j & 1) ? ap[j >> 1] >> 16 : ap[j >> 1] & 0xFFFFu;
        u32& pos = j < 4 ? posA : posB;
        u32 s;
        if (vmask >> j & 1u) { s = 4u + pos; ++pos; }
        else s = 4u + n + (off - pos);                    // words beyond W of a ragged tile land beyond the used slots
        if (s < 4u + (u32)kTileWords) {
          s = stage_idx(s);
          st.x[s] = x[j]; st.a[s] = a16 | off << 16;
        }
      }
    }
    if (haveB) {
      const EvDesc& ep = kSingle ? single : *reinterpret_cast<const EvDesc*>(sh.desc[prv]);
      unpack_write(ep, g, sh.st[(it & 1u) ^ 1u], tid, pTile, pN, pMax1, pG0, pCarry1);
    }
    if (haveA && warp == 0) {
      u32 c = 0, m = 0;
      if (tile) {
        lookback_resolve(ev.tileState, (int)tile, lane, lb, &c, &m);
        if (lane == 0) st_state(ev.tileState + tile, pack_state(kStIncl, c + n, max(m, tileMax1)));
      }
      if (lane == 0) { sh.g0 = c; sh.carry1 = m; }
    }
    __syncthreads();                                                         // #2
    if (!haveA) break;
    haveB = true; pTile = tile; pN = n; pMax1 = tileMax1; pG0 = sh.g0; pCarry1 = sh.carry1;
    if (!kSingle && warp == 1) { sh.desc[nn][lane] = dword; eNN = eN3; }
    t += G; haveA = t < totalTiles; raw = rawNext;
    const u32 r = prv; prv = cur; cur = nxt; nxt = nn; nn = r;
  }
}

// ================================================================== k_cluster (a3 + a4)
// Every module is an independent problem.  No unit of work waits for another one:
//   warp path    a module with at most kWarpCap digis is clustered by ONE warp, with only
//                __syncwarp between its phases: warp-private hash table (row,col) -> digi for the
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
constexpr u32 kModBatch = 8;                     // modules per warp ticket
constexpr u32 kEmpty = 0xFFFFFFFFu;
constexpr u32 kNoKey = 0xFFFFFFFFu;
constexpr u32 kNoRank = 0xFFFFu;

struct WarpRegion {                 // 5 KB of shared memory per warp
  u32 tab[kWarpTab];                // hash table; afterwards L[256] then the head of the accumulators
  uint2 nb[kWarpCap];               // 8 neighbour digi indices, one byte each (self = none); afterwards accumulators
  u32 key[kWarpCap];                // row << 9 | col of kept digis, kNoKey otherwise
};
static_assert(sizeof(u32) * (kWarpTab - kWarpCap) + sizeof(uint2) * kWarpCap >= kAccRoots * 28, "accumulators must fit");

__host__ __device__ inline size_t dense_smem_bytes(u32 bitmapWords) {
  size_t w = (bitmapWords + 3) & ~3u;
  return (size_t)w * 4 * 2 + (size_t)kSmemDigis * 4 * 2 + (size_t)kSmemClusters * (4 + 4 + 4 + 8 * 3);
}
__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t dense = dense_smem_bytes(bitmapWords), warp = sizeof(WarpRegion) * (kClusterThreads / 32);
  return ((dense > warp ? dense : warp) + 15) & ~(size_t)15;
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

struct ClusterShared {
  u32 scan[8];
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

// ---- warp path, one digi per lane: module = digis [s, s+n), 0 < n <= 32.  Everything lives in
// registers: adjacency and reachability are 32-bit lane masks (Warshall closure with shuffles),
// the cluster's minimum lane is its root, sums run along each cluster's lane list.
__device__ __forceinline__ void warp_module_small(const EvDesc& ev, const Geom& g, u32 s, u32 n, WarpRegion& wr,
                                                  u32* nKeptDigis, u32* nRootsOut, u32* nKeptClusters) {
  const u32 lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  constexpr u32 pmask = 127u, shift = 25u;          // 128 slots: load <= 1/4
  u32* tab = wr.tab;
  u32* fw = wr.tab + 128;                           // forward edges: lane mask per digi
  *reinterpret_cast<uint4*>(tab + lane * 4u) = make_uint4(kEmpty, kEmpty, kEmpty, kEmpty);
  fw[lane] = 0u;
  __syncwarp();
  float q = 0.f; u32 key = kNoKey;
  if (lane < n) {
    q = ev.charge[s + lane];
    if (q >= g.pixThr) key = (u32)ev.row[s + lane] << 9 | (u32)ev.col[s + lane];
  }
  const bool kept = key != kNoKey;
  bool dup = false;
  if (kept) {
    const u32 ent = key << 8 | lane;
    u32 h = wm_slot(key, shift);
    for (;;) {
      const u32 old = atomicCAS(tab + h, kEmpty, ent);
      if (old == kEmpty) break;
      if ((old >> 8) == key) dup = true;
      h = (h + 1) & pmask;
    }
  }
  const u32 keptMask = __ballot_sync(0xFFFFFFFFu, kept);
  dup = __any_sync(0xFFFFFFFFu, dup);
  __syncwarp();
  // backward neighbours W, NW, N, NE; each edge is recorded on both ends
  u32 adj = 1u << lane;
  if (kept) {
    const u32 row = key >> 9, col = key & 511u;
    u32 owner = lane;
    if (dup) owner = wm_find_min(tab, pmask, shift, key);
    if (owner != lane) {                              // a duplicate only joins its pixel's owner (A6)
      adj |= 1u << owner; atomicOr(fw + owner, 1u << lane);
    } else {
      const bool up = row > 0, left = col > 0, right = col + 1 < g.C;
#define WM_NB(cond, delta)                                                                          \
      if (cond) {                                                                                   \
        const u32 j = dup ? wm_find_min(tab, pmask, shift, key - (delta)) : wm_find(tab, pmask, shift, key - (delta)); \
        if (j != kEmpty) { adj |= 1u << j; atomicOr(fw + j, 1u << lane); }                          \
      }
      WM_NB(left, 1u)
      WM_NB(up && left, 513u)
      WM_NB(up, 512u)
      WM_NB(up && right, 511u)
#undef WM_NB
    }
  }
  __syncwarp();
  u32 reach = adj | fw[lane];
  // transitive closure (Warshall): after step j every lane that reaches j also reaches all of j's set
  for (u32 j = 0; j < n; ++j) {
    const u32 rj = __shfl_sync(0xFFFFFFFFu, reach, j);
    if (reach & (1u << j)) reach |= rj;
  }
  const u32 root = (u32)__ffs((int)reach) - 1u;
  const bool isRoot = kept && root == lane;
  const u32 nR = (u32)__popc(__ballot_sync(0xFFFFFFFFu, isRoot));
  // sums of qf = q * 2^14 (A9) in binary64 (exact: at most 32 terms below 2^43), suffix sums along the lane list
  double qf = 0.0, qx = 0.0, qy = 0.0;
  if (kept) { qf = (double)(q * 16384.0f); qx = qf * (double)(key >> 9); qy = qf * (double)(key & 511u); }
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
  const u32 kr = (u32)__popc(kb & lt);
  if (keptC) {
    const u32 o = s + kr;
    ev.stS[o] = qf; ev.stSx[o] = qx; ev.stSy[o] = qy;
    ev.stLabel[o] = s + lane; ev.stSize[o] = (u32)__popc(reach);
  }
  const u32 krRoot = __shfl_sync(0xFFFFFFFFu, keptC ? kr : kNoRank, root);
  if (lane < n) {
    ev.label[s + lane] = kept ? s + root : kInvalid;
    ev.clus[s + lane] = (kept && krRoot != kNoRank) ? (int32_t)krRoot : -1;
  }
  __syncwarp();
  *nKeptDigis = (u32)__popc(keptMask); *nRootsOut = nR; *nKeptClusters = (u32)__popc(kb);
}

// ---- warp path: one module = digis [s, s+n), 0 < n <= kWarpCap, processed by the calling warp.
// Returns (kept digis, clusters, kept clusters) in all lanes.
__device__ __forceinline__ void warp_module(const EvDesc& ev, const Geom& g, u32 s, u32 n, WarpRegion& wr,
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
  u32 nKept = 0; bool dup = false;
  for (u32 i = lane; i < nPad; i += 32u) {
    u32 key = kNoKey;
    if (i < n && ev.charge[s + i] >= g.pixThr) key = (u32)ev.row[s + i] << 9 | (u32)ev.col[s + i];
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
  u32* L = tab;
  for (u32 i = lane; i < nPad; i += 32u) L[i] = i;
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

__device__ __forceinline__ void dense_count(const EvDesc& ev, const Geom& g, u32 s, u32 nn,
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

  const bool digiInSmem = nn <= kSmemDigis;
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
    if (cx.nAll > kSmemClusters) {
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

__device__ __forceinline__ void dense_stage(const EvDesc& ev, u32 m, u32 s, u32 nn, const DenseCtx& cx) {
  const int tid = threadIdx.x;
  for (u32 k = tid; k < cx.nAll; k += kClusterThreads) {
    const int32_t kn = cx.knum[k];
    if (kn < 0) continue;
    const u32 o = s + (u32)kn;                       // kn <= k < nn: inside the module's own range
    ev.stS[o] = __ll2double_rn((i64)cx.S[k]); ev.stSx[o] = __ll2double_rn((i64)cx.Sx[k]); ev.stSy[o] = __ll2double_rn((i64)cx.Sy[k]);
    ev.stLabel[o] = s + cx.root[k]; ev.stSize[o] = cx.csize[k];
  }
  for (u32 i = tid; i < nn; i += kClusterThreads) {
    const u32 p = cx.parent[i];
    u32 lab = kInvalid; int32_t cl = -1;
    if (p != kInvalid) { lab = s + p; cl = cx.knum[cx.perm[p]]; }
    ev.label[s + i] = lab;
    ev.clus[s + i] = cl;
  }
  if (tid == 0) {
    ev.modCount[m] = cx.nKept;
    if (cx.nAll) atomicAdd(&ev.counters->nClustersAll, cx.nAll);
  }
}

template <bool kSingle>
__global__ void __launch_bounds__(kClusterThreads, 4)
k_cluster(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv,
          LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
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

  // ---- phase 2: warp path.  A ticket is a batch of kModBatch consecutive modules of one event.
  WarpRegion& wr = reinterpret_cast<WarpRegion*>(smemRaw)[warp];
  const u32 bpe = (M + kModBatch - 1) / kModBatch, nTickets = nEv * bpe;
  for (;;) {
    u32 t = 0;
    if (lane == 0) t = atomicAdd(&lc->modTicket, 1u);
    t = __shfl_sync(0xFFFFFFFFu, t, 0);
    if (t >= nTickets) break;
    const u32 e = t / bpe, m0 = (t - e * bpe) * kModBatch, nm = min(kModBatch, M - m0);
    const EvDesc& ev = kSingle ? single : batch[e];
    if (ev.counters->status & 1u) continue;
    const u32 st = lane <= nm ? ev.modDigiStart[m0 + lane] : 0u;
    u32 accK = 0, accA = 0;
    for (u32 k = 0; k < nm; ++k) {
      const u32 s = __shfl_sync(0xFFFFFFFFu, st, k), t1 = __shfl_sync(0xFFFFFFFFu, st, k + 1);
      u32 cnt = 0;
      if (t1 < s || t1 > ev.cap) {
        if (lane == 0) atomicOr(&ev.counters->status, 2u);   // PR_STATUS_CAPACITY: inconsistent module table
      } else {
        const u32 n = t1 - s;
        if (n > kWarpCap) continue;                          // dense path wrote this module
        if (n > 0) {
          u32 nk, nr;
          if (n <= 32u) warp_module_small(ev, g, s, n, wr, &nk, &nr, &cnt);
          else warp_module(ev, g, s, n, wr, &nk, &nr, &cnt);
          accK += nk; accA += nr;
        }
      }
      if (lane == 0) ev.modCount[m0 + k] = cnt;
    }
    if (lane == 0) {
      if (accK) atomicAdd(&ev.counters->nKept, accK);
      if (accA) atomicAdd(&ev.counters->nClustersAll, accA);
    }
  }
}

// ================================================================== k_finalize (numbering of a4)
// One CTA per (event, group of kFinMods consecutive modules): the group's first dense cluster
// number is the sum of the kept-cluster counts of all earlier modules (at most 2048 values), so
// no CTA depends on another.  Turns clus[] ranks into event-wide cluster numbers, converts the
// staged sums into the cluster SoA (A9: binary64 division, one rounding to binary32), writes
// modClusStart[]; the launch's last CTA publishes all counters to mapped pinned host memory.
constexpr u32 kFinMods = 32;
template <bool kSingle>
__global__ void __launch_bounds__(256)
k_finalize(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv, u32 unitsPerEvent,
           LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g) {
  __shared__ u32 sStart[kFinMods + 1], sDigi[kFinMods + 1], sScan[8], sLast;
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, M = g.M;
  const u32 e = blockIdx.x / unitsPerEvent, u = blockIdx.x - e * unitsPerEvent;
  const EvDesc& ev = kSingle ? single : batch[e];
  const u32 m0 = u * kFinMods, m1 = min(m0 + kFinMods, M);
  if (!(ev.counters->status & 1u)) {
    u32 sum = 0, base;
    for (u32 m = tid; m < m0; m += 256) sum += ev.modCount[m];
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
    for (u32 m = m0 + tid; m < m1; m += 256) ev.modClusStart[m] = sStart[m - m0];
    if (m1 == M && tid == 0) { ev.modClusStart[M] = sStart[32]; ev.counters->nClusters = sStart[32]; }
    const u32 d0 = sDigi[0], d1 = sDigi[m1 - m0];
    if (d0 <= d1 && d1 <= ev.cap) {
      for (u32 d = d0 + tid; d < d1; d += 256) {
        const int32_t c = ev.clus[d];
        if (c >= 0) ev.clus[d] = (int32_t)(sStart[min((u32)ev.module[d] - m0, kFinMods - 1)] + (u32)c);
      }
      for (u32 o = sStart[0] + tid; o < sStart[32]; o += 256) {
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
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    sLast = (atomicAdd(&lc->modDone, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (sLast) {
    __threadfence();
    for (u32 k = tid; k < nEv; k += 256) {
      const EvDesc& d = kSingle ? single : batch[k];
      const volatile DevCounters* c = d.counters;
      HostCounters h;
      h.nWords = c->nWords; h.nDigis = c->nDigis; h.nErrors = c->nErrors; h.nKept = c->nKept;
      h.nClustersAll = c->nClustersAll; h.nClusters = c->nClusters; h.status = c->status; h.seq = 1;
      *d.hostCounters = h;
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

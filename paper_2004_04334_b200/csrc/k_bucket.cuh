// k_bucket.cuh — the step before the decode for words in ARBITRARY order (reading A31): a stable
// bucket sort of an event's words by module on the device.  Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

// Key of a word = its module if it is a digi word (the validity test of k_unpack: A2, A3), else M: error and
// out-of-range words form one last bucket.  Equal keys keep their input order.  One counting sort with M + 1 bins over
// tiles of kTileWords words:
//   k_bucket<false>  per tile: the number of words per bin -> hist[bin * nTiles + tile]
//   k_bucket_scan    per event: exclusive prefix sum over hist in that (bin-major) order = where a tile's words of a bin go
//   k_bucket<true>   per tile: every word's rank among the tile's words of its bin, in input order, and its move
//   k_unbucket_idx   after k_unpack: wordIdx[] and errIdx[] (positions in the bucketed stream) -> positions in the input
// Inside a tile, warp w owns words [256 w, 256 w + 256), lane l word 32 j + l of row j (input order = warp, row, lane).  A
// word's rank = words of its bin in earlier warps + in earlier rows of its warp + in lower lanes of its row
// (__match_any_sync); the per-warp, per-bin counts live in shared memory as halfwords (at most 256 each).
struct BucketDesc {
  const u32* srcW; const u16* srcA;       // the event's words as they came (device memory; the H2D copy of host input)
  u32* dstW; u16* dstA;                   // bucketed stream: what k_unpack reads
  u32* orig;                              // [nWords] input position of the word now at position p
  u32* hist;                              // [(M + 1) * nTiles]
  u32 *wordIdx, *errIdx;                  // the event's index arrays, rewritten by k_unbucket_idx
  const DevCounters* counters;
  u32 nWords, nTiles, tileBase, pad;
};
constexpr u32 kBucketThreads = 256;
constexpr u32 kBucketMaxBins = 2048 + 1;
constexpr u32 kBucketBinPad = (kBucketMaxBins + 3) & ~3u;

template <bool kScatter>
__global__ void __launch_bounds__(kBucketThreads)
k_bucket(const BucketDesc* __restrict__ descs, const u16* __restrict__ tileEvent, const __grid_constant__ Geom g) {
  __shared__ u16 wh[kBucketThreads / 32][kBucketBinPad];
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, lt = (1u << lane) - 1u;
  const BucketDesc bd = descs[tileEvent[blockIdx.x]];
  const u32 tile = blockIdx.x - bd.tileBase, T0 = tile * (u32)kTileWords;
  const u32 nIn = bd.nWords > T0 ? min(bd.nWords - T0, (u32)kTileWords) : 0u;
  const u32 bins = g.M + 1u, limR = g.R << 12, limC = g.C << 3;
  for (u32 i = tid; i < (kBucketThreads / 32) * kBucketBinPad / 2; i += kBucketThreads) reinterpret_cast<u32*>(&wh[0][0])[i] = 0u;
  __syncthreads();
  u32 x[8], key[8], rank[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const u32 idx = 256u * warp + 32u * j + lane;
    const bool in = idx < nIn;
    x[j] = in ? bd.srcW[T0 + idx] : 0u;
    const bool digi = (x[j] >> 20) < g.M && (x[j] & 0xFF000u) < limR && (x[j] & 0xFF8u) < limC;   // bit 31 set -> module field >= 2048 > M - 1
    key[j] = in ? (digi ? x[j] >> 20 : g.M) : 0xFFFFu + lane;                                      // words past the end: a key of their own
    const u32 peers = __match_any_sync(0xFFFFFFFFu, key[j]);
    const u32 before = in ? wh[warp][key[j]] : 0u;
    __syncwarp();
    if (in && (peers & lt) == 0u) wh[warp][key[j]] = (u16)(before + __popc(peers));
    __syncwarp();
    rank[j] = before + __popc(peers & lt);
  }
  __syncthreads();
  for (u32 b = tid; b < bins; b += kBucketThreads) {
    u32 run = 0;
#pragma unroll
    for (u32 w = 0; w < kBucketThreads / 32; ++w) { const u32 c = wh[w][b]; wh[w][b] = (u16)run; run += c; }
    if (!kScatter) bd.hist[(size_t)b * bd.nTiles + tile] = run;
  }
  if (kScatter) {
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const u32 idx = 256u * warp + 32u * j + lane;
      if (idx < nIn) {
        const u32 p = bd.hist[(size_t)key[j] * bd.nTiles + tile] + wh[warp][key[j]] + rank[j];
        bd.dstW[p] = x[j]; bd.dstA[p] = bd.srcA[T0 + idx]; bd.orig[p] = T0 + idx;
      }
    }
  }
}

// One CTA per event: hist[] <- its exclusive prefix sum (bin-major, tile-minor).
__global__ void __launch_bounds__(1024)
k_bucket_scan(const BucketDesc* __restrict__ descs, const __grid_constant__ Geom g) {
  __shared__ u32 sw[32];
  const BucketDesc bd = descs[blockIdx.x];
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const size_t L = (size_t)(g.M + 1u) * bd.nTiles, per = (L + 1023) / 1024;
  const size_t lo = min((size_t)tid * per, L), hi = min(lo + per, L);
  u32 sum = 0;
  for (size_t i = lo; i < hi; ++i) sum += bd.hist[i];
  const u32 incl = warp_incl_scan(sum, (int)lane);
  if (lane == 31u) sw[warp] = incl;
  __syncthreads();
  if (warp == 0) { const u32 v = sw[lane], s = warp_incl_scan(v, (int)lane); sw[lane] = s - v; }
  __syncthreads();
  u32 run = sw[warp] + incl - sum;
  for (size_t i = lo; i < hi; ++i) { const u32 c = bd.hist[i]; bd.hist[i] = run; run += c; }
}

// After k_unpack: index arrays from positions in the bucketed stream to positions in the input.  grid (x, events).
__global__ void __launch_bounds__(256)
k_unbucket_idx(const BucketDesc* __restrict__ descs) {
  const BucketDesc bd = descs[blockIdx.y];
  const u32 D = min(bd.counters->nDigis, bd.nWords), E = min(bd.counters->nErrors, bd.nWords);
  for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < D + E; i += gridDim.x * blockDim.x) {
    u32* p = i < D ? bd.wordIdx + i : bd.errIdx + (i - D);
    const u32 v = *p;
    if (v < bd.nWords) *p = bd.orig[v];
  }
}

}  // namespace pixreco

// k_chain.cuh — the small kernels of the CHAINED modules (section 4.2: a module's product is
// consumed by the next module without a host wait): closing a digi product, opening a consumer on it, and a second
// consumer on a parallel branch (per-module occupancy).  Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

// Module "raw -> digis" ends here: the event's digi counters go to the host (mapped pinned memory) and into `result`,
// the device copy that consumers and k_export read.  One thread.
__global__ void k_publish_digis(const __grid_constant__ EvDesc ev, const LaunchCtl* __restrict__ lc) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const DevCounters* c = ev.counters;
  HostCounters h;
  h.nWords = c->nWords; h.nDigis = c->nDigis; h.nErrors = c->nErrors; h.nKept = 0; h.nClustersAll = 0; h.nClusters = 0;
  h.status = c->status; h.seq = 1;
  h.tStart = lc->tStart; h.tEnd = global_timer();
  *ev.hostCounters = h;
  DevCounters r;
  r.nWords = h.nWords; r.nDigis = h.nDigis; r.nErrors = h.nErrors; r.nKept = 0; r.nClustersAll = 0; r.nClusters = 0;
  r.status = h.status; r.pad = 0;
  *ev.result = r;
}

// A consumer of a digi product starts here: what the producer found out about the event (sizes, the input-order
// status bit that makes modDigiStart undefined) becomes the start of the consumer's own counters.  One thread; also
// stamps the start time of the consumer's chain.
__global__ void k_import_digis(DevCounters* __restrict__ dst, const DevCounters* __restrict__ src, LaunchCtl* __restrict__ lc) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  dst->nWords = src->nWords; dst->nDigis = src->nDigis; dst->nErrors = src->nErrors; dst->status = src->status;
  lc->tStart = global_timer();
}

// Second consumer of a digi product (a parallel branch of the module graph): per module the number of kept digis
// (charge >= pixel threshold, A8) and the sum of their ADC values.  One warp per module; nothing if the input order was
// violated (modDigiStart is undefined then).  The last block publishes the counters of this small module.
__global__ void __launch_bounds__(256)
k_occupancy(const __grid_constant__ EvDesc ev, const DevCounters* __restrict__ src, u32* __restrict__ occCount, u32* __restrict__ occAdcSum,
            HostCounters* __restrict__ hostCounters, const __grid_constant__ Geom g) {
  const u32 lane = threadIdx.x & 31u, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nWarps = (gridDim.x * blockDim.x) >> 5;
  const u32 status = src->status;
  for (u32 m = warp; m < g.M; m += nWarps) {
    u32 cnt = 0, sum = 0;
    if (!(status & 1u)) {
      const u32 s = ev.modDigiStart[m], t = min(ev.modDigiStart[m + 1], ev.cap);
      for (u32 i = s + lane; i < t; i += 32u)
        if (ev.charge[i] >= g.pixThr) { ++cnt; sum += ev.adcOut[i]; }
    }
    cnt = __reduce_add_sync(0xFFFFFFFFu, cnt); sum = __reduce_add_sync(0xFFFFFFFFu, sum);
    if (lane == 0) { occCount[m] = cnt; occAdcSum[m] = sum; }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    HostCounters h;
    h.nWords = src->nWords; h.nDigis = src->nDigis; h.nErrors = src->nErrors; h.nKept = 0; h.nClustersAll = 0; h.nClusters = 0;
    h.status = status; h.seq = 1; h.tStart = global_timer(); h.tEnd = h.tStart;
    *hostCounters = h;
  }
}

}  // namespace pixreco

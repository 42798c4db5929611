// k_finalize.cuh — numbering of a4, cluster table, counters to the host (k_finalize); exact-size gathers (k_export)
// Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

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
        int32_t c[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const u32 d = dd + 256u * k;
          c[k] = d < d1 ? ev.clus[d] : -1;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (c[k] < 0) continue;
          // the digi's module within the group: the last one that starts at or before the digi (no read of module[])
          const u32 d = dd + 256u * k;
          u32 li = 0;
#pragma unroll
          for (u32 step = 16; step > 0; step >>= 1)
            if (li + step < m1 - m0 && sDigi[li + step] <= d) li += step;
          ev.clus[d] = (int32_t)(sStart[li] + (u32)c[k]);
        }
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

// k_finalize.cuh — numbering of a4, cluster table, hit table, counters to the host (k_finalize); exact-size gathers (k_export)
// Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

// ================================================================== k_finalize (numbering of a4)
// One CTA per (event, group of kFinMods consecutive modules): the group's first dense cluster
// number is the sum of the kept-cluster counts of all earlier modules (at most 2048 values), so
// no CTA depends on another.  Turns clus[] ranks (clus_ranked) into event-wide cluster numbers, converts the
// staged sums into the cluster SoA (A9: binary64 division, one rounding to binary32) and the hit SoA (the step after
// clustering in the paper's Fig. 1; A26-A30: position from the same exact sums, bounding box, border flags, error
// estimate), writes modClusStart[]; the CTA of an event's last module group publishes that event's counters to mapped
// pinned host memory.
// The event's counters to mapped pinned host memory and, for k_export, to their device copy.  With `flag` the host polls
// seq instead of the completion event: the other fields and every earlier write of the launch are fenced before it.
__device__ __forceinline__ void publish_counters(const EvDesc& ev, const LaunchCtl* lc, u32 nClusters, bool flag) {
  const DevCounters* c = ev.counters;
  const u32 status = __ldcg(&c->status);
  HostCounters h;
  h.nWords = __ldcg(&c->nWords); h.nDigis = __ldcg(&c->nDigis); h.nErrors = __ldcg(&c->nErrors); h.nKept = __ldcg(&c->nKept);
  h.nClustersAll = __ldcg(&c->nClustersAll); h.nClusters = (status & 1u) ? 0u : nClusters; h.status = status; h.seq = flag ? 0u : 1u;
  h.tStart = lc->tStart; h.tEnd = global_timer();
  *ev.hostCounters = h;
  DevCounters r;                                   // device copy of the final counters: k_export takes its sizes from it
  r.nWords = h.nWords; r.nDigis = h.nDigis; r.nErrors = h.nErrors; r.nKept = h.nKept; r.nClustersAll = h.nClustersAll;
  r.nClusters = h.nClusters; r.status = status; r.pad = 0;
  *ev.result = r;
  if (flag) {
    __threadfence_system();
    *reinterpret_cast<volatile u32*>(&ev.hostCounters->seq) = 1u;
  }
}

constexpr u32 kFinMods = 32;                     // modules per group of grpCount[] (k_cluster adds whole tickets to one group)
constexpr u32 kFinMaxGroups = 4;                 // a CTA takes 1, 2 or 4 consecutive groups (launches with many units: less set-up per digi)
static_assert(kFinMods == 32 && 32 % kModBatch == 0, "grpCount groups are 32 modules and hold whole warp tickets");
template <bool kSingle>
__global__ void __launch_bounds__(256, 8)
k_finalize(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv, u32 unitsPerEvent, u32 splits,
           u32 groupsPerUnit, LaunchCtl* __restrict__ lc, const __grid_constant__ Geom g, u32 selfClean) {
  __shared__ u32 sStart[kFinMods * kFinMaxGroups + 1], sDigi[kFinMods * kFinMaxGroups + 1], sScan[8], sTot[kFinMaxGroups];
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, M = g.M;
  // `splits` CTAs share one unit when events are huge: slice sp of the unit's digis and clusters
  const u32 unit = blockIdx.x / splits, sp = blockIdx.x - unit * splits;
  const u32 e = unit / unitsPerEvent, u = unit - e * unitsPerEvent;
  const EvDesc& ev = kSingle ? single : batch[e];
  const u32 nMods = kFinMods * groupsPerUnit;
  const u32 m0 = u * nMods, m1 = min(m0 + nMods, M), nm = m1 - m0;
  // (the tables are read beside the status word, not after it: they are there whatever the status says)
  u32 sum = 0, cLoad = 0, dLoad = 0;
  for (u32 k = tid; k < u * groupsPerUnit; k += 256) sum += ev.grpCount[k];        // the groups before this unit
  if (warp < groupsPerUnit && m0 + tid < m1) cLoad = ev.modCount[m0 + tid];
  if (tid <= nMods) dLoad = ev.modDigiStart[min(m0 + tid, M)];
  if (!(ev.counters->status & 1u)) {
    u32 base;
    u32 c = 0, incl = 0;
    if (warp < groupsPerUnit) {                       // warp w scans the unit's group w
      c = cLoad;
      incl = warp_incl_scan(c, lane);
      if (lane == 31) sTot[warp] = incl;
    }
    if (tid <= nMods) sDigi[tid] = dLoad;
    block_excl_scan(sum, sScan, &base);               // (two barriers: sTot is visible after it)
    if (warp < groupsPerUnit) {
      u32 off = base;
      for (u32 w = 0; w < warp; ++w) off += sTot[w];
      sStart[tid] = off + incl - c;
      if (tid == nMods - 1u) sStart[nMods] = off + incl;
    }
    __syncthreads();
    if (sp == 0) {
      for (u32 m = m0 + tid; m < m1; m += 256) ev.modClusStart[m] = sStart[m - m0];
      if (m1 == M && tid == 0) { ev.modClusStart[M] = sStart[nMods]; ev.counters->nClusters = sStart[nMods]; }
    }
    const u32 d0 = sDigi[0], d1 = sDigi[nm];
    if (d0 <= d1 && d1 <= ev.cap) {
      for (u32 dd = d0 + sp * 2048u + tid; dd < d1; dd += splits * 2048u) {     // eight independent digis per thread and trip
        int32_t c[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const u32 d = dd + 256u * k;
          c[k] = d < d1 ? ev.clus[d] : -1;
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          if (c[k] < 0) continue;
          // clus_ranked: rank among the module's kept clusters | the module's position among 128 << 20
          const u32 d = dd + 256u * k, li = ((u32)c[k] >> 20) & (nMods - 1u);
          ev.clus[d] = (int32_t)(sStart[li] + ((u32)c[k] & 0xFFFFFu));
        }
      }
      for (u32 o = sStart[0] + sp * 256u + tid; o < sStart[nMods]; o += splits * 256u) {
        u32 li = 0;
#pragma unroll
        for (u32 step = kFinMods * kFinMaxGroups / 2; step > 0; step >>= 1)
          if (li + step < nMods + 1 && sStart[li + step] <= o) li += step;       // last module with start <= o and a cluster there
        const u32 src = sDigi[li] + (o - sStart[li]);
        if (o < ev.cap && src < ev.cap) {
          const uint4* rec = reinterpret_cast<const uint4*>(ev.staged + src);                              // StagedCluster
          const uint4 r0 = rec[0], r1 = rec[1], r2 = rec[2];
          const double S = __hiloint2double((int)r0.y, (int)r0.x), Sx = __hiloint2double((int)r0.w, (int)r0.z), Sy = __hiloint2double((int)r1.y, (int)r1.x);
          ev.clLabel[o] = r1.z; ev.clModule[o] = (u16)(m0 + li); ev.clSize[o] = r1.w;
          ev.clCharge[o] = __double2float_rn(S * (1.0 / 16384.0));
          const double rc = __ddiv_rn(Sx, S), cc = __ddiv_rn(Sy, S);                                       // A9
          ev.clRow[o] = __double2float_rn(rc);
          ev.clCol[o] = __double2float_rn(cc);
          // the hit of this cluster.  A27: divide, add 0.5, subtract half the module, multiply by the pitch — binary64, in
          // this order, one cast; A28 box; A29 border flags; A30 error = pitch/sqrt(12) * {span at a border, 1 for span 1, else 0.5}
          const u32 bR = r2.x, bC = r2.y;
          const u32 rmin = 255u - (bR >> 16), rmax = bR & 0xFFFFu, cmin = 511u - (bC >> 16), cmax = bC & 0xFFFFu;
          const bool er = rmin == 0u || rmax == g.R - 1u, ec = cmin == 0u || cmax == g.C - 1u;
          const u32 sr = rmax - rmin + 1u, sc = cmax - cmin + 1u;
          const double fr = er ? (double)sr : (sr == 1u ? 1.0 : 0.5), fc = ec ? (double)sc : (sc == 1u ? 1.0 : 0.5);
          ev.htX[o] = __double2float_rn(__dmul_rn(__dsub_rn(__dadd_rn(rc, 0.5), 0.5 * (double)g.R), g.pitchRow));
          ev.htY[o] = __double2float_rn(__dmul_rn(__dsub_rn(__dadd_rn(cc, 0.5), 0.5 * (double)g.C), g.pitchCol));
          ev.htXerr[o] = __double2float_rn(__dmul_rn(__dmul_rn(g.pitchRow, 0.28867513459481287), fr));
          ev.htYerr[o] = __double2float_rn(__dmul_rn(__dmul_rn(g.pitchCol, 0.28867513459481287), fc));
          ev.htRows[o] = rmin | rmax << 16; ev.htCols[o] = cmin | cmax << 16;
          ev.htFlags[o] = (u16)((er ? 1u : 0u) | (ec ? 2u : 0u));
        }
      }
    }
  }
  // The CTA of the event's last module group publishes the event's counters to mapped pinned host memory: all
  // the others were final when this kernel started, nClusters is this CTA's own result.
  if (!selfClean && m1 == M && sp == 0 && tid == 0) publish_counters(ev, lc, sStart[nMods], false);
  // selfClean (a slot's graph, one event): the last CTA to leave publishes the counters instead — every other CTA's
  // results are visible by then, so the host may take seq != 0 in the mapped counters as the completion of the whole
  // acquire, without a driver call — and puts the zeros back into the words that the next launch of the graph expects
  // cleared — the module ticket, the event's counters and group counts — so that the graph needs no memset node
  // (k_unpack does the same for its ticket and its look-back states).
  if (selfClean) {
    __shared__ u32 sLast;
    __syncthreads();
    if (tid == 0) { __threadfence(); sLast = atomicAdd(&lc->modDone, 1u) == gridDim.x - 1u ? 1u : 0u; }
    __syncthreads();
    if (sLast) {
      __threadfence();
      if (tid == 0) publish_counters(ev, lc, __ldcg(&ev.counters->nClusters), true);
      __syncthreads();
      u32* c = reinterpret_cast<u32*>(ev.counters);
      if (tid < sizeof(DevCounters) / 4u) c[tid] = 0u;
      for (u32 k = tid; k < (M + kFinMods - 1u) / kFinMods; k += 256u) ev.grpCount[k] = 0u;
      if (tid == 0) { lc->modTicket = 0u; lc->modDone = 0u; }
    }
  }
}


// ================================================================== k_export
// Exact-size copies of requested outputs to mapped pinned host memory (transfers only
// when asked).  Element counts are read from the device counters, so no host round trip.
struct ExportItem { const void* src; void* dst; const DevCounters* cnt; u32 elemBytes; u32 countSel; u32 fixedCount; u32 pad; };
// countSel: 0 = nDigis, 1 = nErrors, 2 = nClusters of *cnt (the event's final counters), 3 = fixedCount
__global__ void __launch_bounds__(256)
k_export(const ExportItem* __restrict__ items, u32 nItems) {
  for (u32 it = blockIdx.y; it < nItems; it += gridDim.y) {
    const ExportItem x = items[it];
    u32 cnt = x.fixedCount;
    if (x.countSel < 3u) { const DevCounters c = *x.cnt; cnt = x.countSel == 0 ? c.nDigis : x.countSel == 1 ? c.nErrors : c.nClusters; }
    const size_t bytes = (size_t)cnt * x.elemBytes;
    const size_t nVec = (bytes + 15) >> 4;                 // buffers are padded to 16 B
    const uint4* s = reinterpret_cast<const uint4*>(x.src);
    uint4* d = reinterpret_cast<uint4*>(x.dst);
    const size_t step = (size_t)gridDim.x * blockDim.x;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < nVec; v += 4 * step) {     // four loads, then four stores
      uint4 r[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) if (v + k * step < nVec) r[k] = s[v + k * step];
#pragma unroll
      for (int k = 0; k < 4; ++k) if (v + k * step < nVec) d[v + k * step] = r[k];
    }
  }
}

}  // namespace pixreco

// k_export.cuh — exact-size gathers of requested outputs into pinned host memory (k_export)
// Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

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
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < nVec; v += (size_t)gridDim.x * blockDim.x) d[v] = s[v];
  }
}

}  // namespace pixreco

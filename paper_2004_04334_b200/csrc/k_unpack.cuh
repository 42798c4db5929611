// k_unpack.cuh — a1 + a2: raw words -> digis with calibration, stable compaction (TMA ring, count-ahead, look-back)
// Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

// ================================================================== k_unpack (a1 + a2)
// Persistent CTAs; a tile = kTileWords consecutive words of one event.  Tiles are handed out by an ATOMIC TICKET
// (LaunchCtl::tileTicket) in launch order, drawn by the control warp six tiles ahead of the scatter: a tile is only
// ever owned by a CTA that is running, and a CTA works through its tiles in ascending order, so the look-back (which
// reads states published by the owners of earlier tiles) makes progress whatever the order or the moment in which the
// hardware starts the CTAs — also beside other kernels that fill part of the GPU.  `pro` (1..7) bounds the tiles a CTA
// holds at a time (7 = a full pipeline): small launches spread one tile per CTA (the pipeline then runs with bubbles), large ones keep the
// pipeline full.  "Local tile k" below is the k-th slot of this CTA's pipeline (a tile, a bubble, or the end mark).
// The last CTA to leave puts the zeros back into the ticket and the look-back states (the control block is all zero
// between acquires: no per-acquire memset).  Per iteration i the CTA does, with two barriers:
//   load    (end of iteration i)  one thread issues TMA bulk copies (cp.async.bulk, completion on an
//           mbarrier) of tile i + kRawSlots into the ring slot tile i just vacated: raw words and
//           ADC values reach shared memory without passing through registers
//   count   tile i + kCountAhead: validity (A2, A3) of every word, one ballot per 32 words kept in
//           shared memory, per-warp digi counts; the tile's aggregate (count, max module + 1) is
//           PUBLISHED kCountAhead iterations before the tile is written, so when a successor looks
//           back, the aggregate has long been there: no CTA waits for the progress of another one
//   scatter tile i: its event-global digi offset g0 is known (look-back resolved in iteration
//           i - 1).  Warp w owns words [256w, 256w + 256) of the tile, lane l word 32j + l of row j:
//           position = g0 + warp prefix + row prefix + popc(ballot below lane).  The digi's four
//           16-bit fields (module,row,col,adc) are stored in FINAL form into four shared-memory
//           arrays at index 8 + (g0 & 7) + position, i.e. with the 16-byte phase of their global
//           destination; its two 32-bit fields (wordIdx; charge = fmaf, A7) go straight to global
//           memory — consecutive lanes hold consecutive digis, so a warp's row is one contiguous
//           run of 4-byte stores — which keeps the CTA at 69 KB of shared memory and 64 registers:
//           three CTAs per SM with the full four-slot ring; error words (rare) go straight to
//           global memory too
//   look-back (warp 0) for tile i + 1: loads issued before the scatter, resolved after it
//   store   one thread issues four TMA bulk stores of the 16-byte-aligned middle of the staged
//           arrays; sixteen lanes store the up-to-7 head and tail elements; all threads scan the
//           staged module array for module boundaries (modDigiStart) and order violations (A5)
// Algorithmic HBM bytes per event: 6W read + 16D (digi SoA incl. charge) + 8E written.
constexpr int kUnpackCtasPerSM = 3;
constexpr int kRawSlots = 4;                      // raw tiles in the shared-memory ring
constexpr int kCountAhead = 2;                    // a tile is counted this many iterations before it is written
constexpr int kDescRing = 8;                      // descriptor / tile-index ring, power of two >= kRawSlots + 4
constexpr int kDrawAhead = 6;                     // a ticket drawn in iteration i becomes local tile i + kDrawAhead
constexpr u32 kTilesFromDesc = 0xFFFFFFFDu;       // totalTiles argument of a graph launch: take nTiles of the (one) event
constexpr u32 kStartWaitGrid = 128;               // launches with at least this many CTAs wait for one another at the start
constexpr u64 kStartWaitNs = 20000;               // upper bound of the wait for the rest of the grid at the start of a CTA
constexpr u32 kTileSkip = 0xFFFFFFFEu, kTileEnd = 0xFFFFFFFFu;   // pipeline slot without a tile: a bubble / no more tiles
constexpr u32 kStageElems = kTileWords + 32;      // 8 front pad + phase (< 8) + tile, multiple of 8
static_assert(kCountAhead >= 1 && kCountAhead <= kRawSlots - 2, "a raw tile needs a full iteration to arrive before it is counted");
static_assert(kRawSlots + 4 <= kDescRing && kDrawAhead == kRawSlots + 2, "rings too small for the draw-ahead");

struct __align__(128) UnpackShared {
  u32 words[kRawSlots][kTileWords];               // raw ring (TMA destination)
  u16 adc[kRawSlots][kTileWords];
  u16 sModule[kStageElems], sRow[kStageElems], sCol[kStageElems], sAdc[kStageElems];   // staging (TMA source)
  u64 full[kRawSlots];                            // mbarriers: raw slot filled
  u32 bal[kRawSlots][8][8];                       // [slot][warp][row] validity ballots
  u32 wcnt[kRawSlots][8], wmax[kRawSlots][8];     // per warp: digis, max(module)+1
  u32 g0[2], carry1[2];                           // look-back result of local tile k at [k & 1]
  u32 desc[kDescRing][32];                        // batch: first 128 bytes of the tiles' event descriptors
  u32 tile[kDescRing];                            // tile index (ticket) of local tile k at [k & 7], or kTileSkip / kTileEnd
  u32 last;                                       // this CTA is the last one to leave
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

template <bool kSingle>
__global__ void __launch_bounds__(kUnpackThreads + 64, kUnpackCtasPerSM)
k_unpack(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, const u16* __restrict__ tileEvent,
         u32 totalTiles, u32 pro, LaunchCtl* __restrict__ lc, u64* __restrict__ tileStateAll, const __grid_constant__ Geom g,
         const EvDesc* __restrict__ hostDesc) {
  extern __shared__ __align__(128) unsigned char unpackSmem[];
  UnpackShared& sh = *reinterpret_cast<UnpackShared*>(unpackSmem);
  const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, lt = (1u << lane) - 1u;
  // a launch replayed from a CUDA graph does not know its size when it is recorded: a one-event launch then reads it
  // from the event's descriptor
  // hostDesc (a slot's graph): the one event's descriptor lies in mapped pinned HOST memory and is read from there (no
  // copy node in the graph); the CTA that draws ticket 0 leaves a device copy in batch[0] for the kernels that follow
  const EvDesc* descs = (!kSingle && hostDesc) ? hostDesc : batch;
  if (!kSingle && totalTiles == kTilesFromDesc) totalTiles = descs[0].nTiles;
  const bool ctl = warp == 8u, scn = warp == 9u;             // warps 0..7 work on words; warp 8 drives the TMA and draws the tickets; warp 9 publishes and looks back
  const u32 limM = g.M, limR = g.R << 12, limC = g.C << 3;
  auto desc_of = [&](int k) -> const EvDesc& {
    return kSingle ? single : *reinterpret_cast<const EvDesc*>(sh.desc[k & (kDescRing - 1)]);
  };
  auto tile_of = [&](int k) -> u32 { return sh.tile[k & (kDescRing - 1)]; };   // < totalTiles iff local tile k is a tile
  // ---- load of local tile k into its ring slot, by the control warp: TMA for the 16-byte multiple, lanes for the tail.
  // A slot without a tile still completes its barrier phase (0 bytes), so phase parity follows the local index.
  auto issue_load = [&](int k) {
    const u32 t = tile_of(k), slot = (u32)k % kRawSlots;
    if (t >= totalTiles) {
      if (lane == 0) mbar_expect_tx(&sh.full[slot], 0u);
      return;
    }
    const EvDesc& e = desc_of(k);
    const u32 T0 = (t - e.tileBase) * (u32)kTileWords, W = e.nWords;
    const u32 nIn = W > T0 ? min(W - T0, (u32)kTileWords) : 0u;
    const u32 n4 = nIn & ~3u, n8 = nIn & ~7u;
    if (lane == 0) {
      mbar_expect_tx(&sh.full[slot], n4 * 4u + n8 * 2u);
      if (n4) bulk_load(sh.words[slot], e.words + T0, n4 * 4u, &sh.full[slot]);
      if (n8) bulk_load(sh.adc[slot], e.adc + T0, n8 * 2u, &sh.full[slot]);
    }
    if (lane < nIn - n4) sh.words[slot][n4 + lane] = __ldcs(e.words + T0 + n4 + lane);
    if (lane < nIn - n8) sh.adc[slot][n8 + lane] = __ldcs(e.adc + T0 + n8 + lane);
  };

  // ---- prologue: barriers, the first block of tickets (local tiles 0 .. kDrawAhead - 1), their descriptors and loads
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kRawSlots; ++s) mbar_init(&sh.full[s], 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    // ONE ticket now, the next ones one per iteration: consecutive tiles go to different CTAs, which count (and
    // publish) them at about the same time — a block of consecutive tiles per CTA would make every CTA's first
    // look-back wait for its predecessor's third iteration, a chain through the whole grid
    const u32 t0 = atomicAdd(&lc->tileTicket, 1u);
    if (t0 == 0u) lc->tStart = global_timer();
#pragma unroll
    for (u32 j = 0; j < (u32)kDescRing; ++j) sh.tile[j] = j == 0u ? (t0 < totalTiles ? t0 : kTileEnd) : (j < (u32)kDrawAhead && t0 < totalTiles ? kTileSkip : kTileEnd);
    sh.last = 0u;
    // The CTAs of the launch start their pipelines together.  A CTA that starts alone — the grid arrives piecemeal when
    // it follows another stream's kernel whose CTAs retire one by one — runs through its empty pipeline slots in no
    // time and draws a BLOCK of consecutive tickets; its successors' first look-backs then wait for its later
    // iterations, a chain through the whole grid (measured: 0.49-0.54 ms instead of 0.30 ms for the 256-event batch
    // behind a k_cluster of the other stream).  The wait is bounded: nothing depends on it, and a grid that is not
    // co-resident (beside other kernels, or oversubscribed on purpose) goes on after kStartWaitNs.
    // (a small launch — a single event — has no chain worth the wait)
    if (gridDim.x >= kStartWaitGrid) {
      atomicAdd(&lc->unpackStarted, 1u);
      const u64 tw = global_timer();
      while (*reinterpret_cast<volatile u32*>(&lc->unpackStarted) < gridDim.x && global_timer() - tw < kStartWaitNs) {}
    }
  }
  __syncthreads();
  if (!kSingle && (int)warp < kDrawAhead && tile_of((int)warp) < totalTiles)
    sh.desc[warp][lane] = __ldg(reinterpret_cast<const u32*>(descs + tileEvent[tile_of((int)warp)]) + lane);
  if (!kSingle && hostDesc && tile_of(0) == 0u && tid < sizeof(EvDesc) / 4u)
    reinterpret_cast<u32*>(const_cast<EvDesc*>(batch))[tid] = reinterpret_cast<const u32*>(hostDesc)[tid];
  // control warp: tiles in flight, whether a draw came back empty, the ticket drawn in the previous iteration and its event
  u32 inflight = 0, tktP = kTileSkip, eP = 0;
  bool ended = gridDim.x >= totalTiles;        // one ticket per CTA covers the launch: the draws of the prologues were the last ones
  if (ctl) {
    for (int j = 0; j < kDrawAhead; ++j) { inflight += tile_of(j) < totalTiles ? 1u : 0u; ended = ended || tile_of(j) == kTileEnd; }
  }
  __syncthreads();
  if (ctl)
    for (int k = 0; k < kRawSlots; ++k) issue_load(k);
  __syncthreads();

  for (int i = -kCountAhead;; ++i) {
    const int kc = i + kCountAhead, kl = i + 1, kd = i + kDrawAhead - 1;
    const u32 ti = i >= 0 ? tile_of(i) : kTileSkip;            // this iteration's tile to scatter and store
    if (ti == kTileEnd) break;
    const bool vi = ti < totalTiles, vc = tile_of(kc) < totalTiles, vl = tile_of(kl) < totalTiles;
    u32 dword = 0, tkt = kTileSkip, tl = 0;
    u64 lb[kLookBack];
    if (ctl) {
      // a new ticket (it becomes local tile i + kDrawAhead); the descriptor of the one drawn an iteration ago
      if (!ended && inflight < pro && lane == 0) tkt = atomicAdd(&lc->tileTicket, 1u);
      if (!kSingle && tktP < totalTiles) dword = __ldg(reinterpret_cast<const u32*>(descs + eP) + lane);
      if (lane == 0 && i > 0) bulk_wait_read();               // the staging arrays are free again
    } else if (!scn && vc) {
      // ---- count: local tile i + kCountAhead
      const EvDesc& e = desc_of(kc);
      const u32 T0 = (tile_of(kc) - e.tileBase) * (u32)kTileWords, W = e.nWords;
      const u32 nIn = W > T0 ? min(W - T0, (u32)kTileWords) : 0u, slot = (u32)kc % kRawSlots;
      mbar_wait(&sh.full[slot], ((u32)kc / kRawSlots) & 1u);
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
    __syncthreads();                                                                                           // #1
    if (sh.last) break;                                        // the control warp saw the end with nothing in flight (written before this barrier)
    if (scn) {
      // ---- publish the aggregate of tile i + kCountAhead, issue the look-back loads of tile i + 1
      if (vc) {
        const EvDesc& e = desc_of(kc);
        const u32 tile = tile_of(kc) - e.tileBase, slot = (u32)kc % kRawSlots;
        const u32 n = __reduce_add_sync(0xFFFFFFFFu, lane < 8u ? sh.wcnt[slot][lane] : 0u);
        const u32 mx1 = __reduce_max_sync(0xFFFFFFFFu, lane < 8u ? sh.wmax[slot][lane] : 0u);
        if (lane == 0) st_state(e.tileState + tile, pack_state(tile ? kStAgg : kStIncl, n, mx1));
      }
      if (kl >= 0 && vl) {
        const EvDesc& e = desc_of(kl);
        tl = tile_of(kl) - e.tileBase;
        if (tl) lookback_issue(e.tileState, (int)tl, lane, lb);
      }
    } else if (!ctl && vi) {
      // ---- scatter: local tile i
      const EvDesc& e = desc_of(i);
      const u32 T0 = (ti - e.tileBase) * (u32)kTileWords, W = e.nWords;
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
          sh.sAdc[el] = (u16)a;
          // (the two 4-byte arrays go straight to global memory: consecutive lanes hold consecutive digis)
          const u32 p = g0 + (el - 8u - ph);
          e.wordIdx[p] = wi0 + 32u * j; e.charge[p] = __fmaf_rn((float)a, gp.x, gp.y);
        } else if (256u * warp + 32u * j + lane < nIn) {
          // error word (A2-A4): errors before it = words before it - digis before it
          const u32 ei = (wi0 + 32u * j) - (g0 + (el - 8u - ph));
          e.errWord[ei] = x; e.errIdx[ei] = wi0 + 32u * j;
        }
        ebase += (u32)__popc(b);
      }
      fence_async_smem();                                      // staged digis -> visible to the TMA store
    }
    __syncthreads();                                                                                           // #2
    if (ctl) {
      if (vi) {
        const EvDesc& e = desc_of(i);
        const u32 slot = (u32)i % kRawSlots, g0 = sh.g0[i & 1], ph = g0 & 7u;
        const u32 n = __reduce_add_sync(0xFFFFFFFFu, lane < 8u ? sh.wcnt[slot][lane] : 0u);
        const u32 midLo = (g0 + 7u) & ~7u, midHi = (g0 + n) & ~7u;
        if (lane == 0) {
          if (midHi > midLo) {
            const u32 cnt = midHi - midLo, se = 8u + ph + (midLo - g0);
            bulk_store(e.module + midLo, sh.sModule + se, cnt * 2u); bulk_store(e.row + midLo, sh.sRow + se, cnt * 2u);
            bulk_store(e.col + midLo, sh.sCol + se, cnt * 2u); bulk_store(e.adcOut + midLo, sh.sAdc + se, cnt * 2u);
          }
          bulk_commit();
        }
        if (lane < 16u) {
          // head (k < 8) and tail (k >= n - 8) digis outside the 16-byte-aligned middle
          const u32 lo = 8u + ph, k = lane < 8u ? lane : n - 16u + lane, p = g0 + k;
          if (k < n && (lane < 8u || k >= 8u) && !(p >= midLo && p < midHi)) {
            const u32 se = lo + k;
            e.module[p] = sh.sModule[se]; e.row[p] = sh.sRow[se]; e.col[p] = sh.sCol[se]; e.adcOut[p] = sh.sAdc[se];
          }
        }
        --inflight;
      }
      if (i >= 0) issue_load(i + kRawSlots);                   // into the slot this tile vacated (its ring entry was written an iteration ago)
      if (i >= 1 - kCountAhead) {
        // ring entry of local tile i + kDrawAhead - 1: the ticket drawn in the previous iteration
        if (!kSingle && tktP < totalTiles) sh.desc[kd & (kDescRing - 1)][lane] = dword;
        if (lane == 0) sh.tile[kd & (kDescRing - 1)] = tktP < totalTiles ? tktP : (ended ? kTileEnd : kTileSkip);
      }
      {
        // this iteration's draw: its event now, its descriptor in the next iteration
        tkt = __shfl_sync(0xFFFFFFFFu, tkt, 0);
        if (tkt < totalTiles) { ++inflight; if (!kSingle) eP = tileEvent[tkt]; }
        else if (tkt != kTileSkip) ended = true;               // the launch has no more tiles
        tktP = tkt;
        if (ended && inflight == 0u && lane == 0) sh.last = 1u;  // nothing left to do: everybody leaves at the next iteration
      }
      __syncwarp();
    } else if (scn) {
      // ---- resolve the look-back of tile i + 1 (its loads flew during the scatter), publish its inclusive state
      if (kl >= 0 && vl) {
        const EvDesc& e = desc_of(kl);
        const u32 slot = (u32)kl % kRawSlots;
        u32 c = 0, m = 0;
        if (tl) {
          lookback_resolve(e.tileState, (int)tl, lane, lb, &c, &m);
          const u32 n = __reduce_add_sync(0xFFFFFFFFu, lane < 8u ? sh.wcnt[slot][lane] : 0u);
          const u32 mx1 = __reduce_max_sync(0xFFFFFFFFu, lane < 8u ? sh.wmax[slot][lane] : 0u);
          if (lane == 0) st_state(e.tileState + tl, pack_state(kStIncl, c + n, max(m, mx1)));
        }
        if (lane == 0) { sh.g0[kl & 1] = c; sh.carry1[kl & 1] = m; }
      }
    } else if (vi) {
      const EvDesc& e = desc_of(i);
      const u32 tile = ti - e.tileBase, slot = (u32)i % kRawSlots;
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
  // ---- the last CTA to leave puts the zeros back: look-back states and ticket words
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    sh.last = atomicAdd(&lc->unpackExited, 1u) == gridDim.x - 1u ? 1u : 0u;     // (sh.last is reused: now "last CTA to leave")
  }
  __syncthreads();
  if (sh.last) {
    __threadfence();
    for (u32 t = tid; t < totalTiles; t += kUnpackThreads + 64) tileStateAll[t] = 0ull;
    if (tid == 0) { lc->tileTicket = 0u; lc->unpackExited = 0u; lc->unpackStarted = 0u; }
  }
}

}  // namespace pixreco

// k_cluster.cuh — a3 + a4: per-module connected components and exact cluster sums (k_cluster, k_dense)
// Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

// ================================================================== k_cluster (a3 + a4)
// Every module is an independent problem.  No unit of work waits for another one:
//   warp path    consecutive modules with at most 32 digis together are clustered in one pass by ONE
//                warp, in registers (warp_pack).  A module of 33..kWarpCap digis is clustered by ONE warp with
//                only __syncwarp between its phases: warp-private hash table (row,col) -> digi for the
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
constexpr u32 kAccRoots = 84;                    // clusters accumulated per pass over a module
constexpr u32 kModBatch = 4;                     // most modules per warp ticket (small tickets: a short tail; 8 was 6 % slower, 16 17 %);
                                                 // small launches use 2 or 1 so that every warp gets work (modBatch, a power of two)
constexpr u32 kEmpty = 0xFFFFFFFFu;
constexpr u32 kNoKey = 0xFFFFFFFFu;
constexpr u32 kNoRank = 0xFFFFu;

struct WarpRegion {                 // 5 KB of shared memory per warp
  u32 tab[kWarpTab];                // hash table; afterwards L[256] then the head of the accumulators
  uint2 nb[kWarpCap];               // 8 neighbour digi indices, one byte each (self = none); afterwards accumulators
  u32 key[kWarpCap];                // row << 9 | col of kept digis, kNoKey otherwise
};
static_assert(sizeof(u32) * (kWarpTab - kWarpCap) + sizeof(uint2) * kWarpCap >= kAccRoots * 36, "accumulators must fit");

__host__ __device__ inline size_t dense_smem_bytes(u32 bitmapWords, u32 capDigis = kSmemDigis, u32 capClusters = kSmemClusters) {
  size_t w = (bitmapWords + 3) & ~3u;
  return (size_t)w * 4 * 2 + (size_t)capDigis * 4 * 2 + (size_t)capClusters * (4 + 4 + 4 + 8 * 3 + 4 * 4);
}
__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t dense = dense_smem_bytes(bitmapWords), warp = sizeof(WarpRegion) * (kClusterThreads / 32);
  return ((dense > warp ? dense : warp) + 15) & ~(size_t)15;
}

// Root of x, halving the path on the way (a node's parent only ever moves to another ancestor in its set, so
// concurrent finds and hooks stay consistent).  Only while unions are running: see uf_root.
__device__ __forceinline__ u32 uf_find(volatile u32* parent, u32 x) {
  u32 p = parent[x];
  while (p != x) {
    const u32 gp = parent[p];
    if (gp != p) parent[x] = gp;
    x = p; p = gp;
  }
  return x;
}
// Root of x without touching the forest: for the flattening pass, where a late halving store could
// overwrite another thread's final root.
__device__ __forceinline__ u32 uf_root(const volatile u32* parent, u32 x) {
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
  u32 scan[16];
  u32 nBig, big[kClusterThreads];
};

// Bounding box (A28) as two words of two halfword maxima each: rows max(255 - row) << 16 | max(row), cols
// max(511 - col) << 16 | max(col); __vmaxu2 combines two boxes.
__device__ __forceinline__ u32 box_rows(u32 row) { return (255u - row) << 16 | row; }
__device__ __forceinline__ u32 box_cols(u32 col) { return (511u - col) << 16 | col; }

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

// ---- warp path, one digi per lane: a PACK of consecutive modules with at most 32 digis together, digis
// [s, s+n).  Everything lives in registers: lane i learns its neighbours by comparing its (module, row,
// col) with every other lane's (n shuffles, no table; two digis on one pixel are simply adjacent, A6),
// adjacency and reachability are 32-bit lane masks (Warshall closure with shuffles), a cluster's
// minimum lane is its root, sums run along each cluster's lane list.  mIdx/mStart: the lane's module
// (index within the pack) and that module's first digi.  Returns the ballots of kept digis, of roots
// and of roots of kept clusters.
__device__ __forceinline__ void warp_pack(const EvDesc& ev, const Geom& g, u32 s, u32 n, float q0, u32 rc0, u32 mIdx, u32 mStart,
                                          u32* keptDigis, u32* roots, u32* keptRoots) {
  const u32 lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  const float q = lane < n ? q0 : 0.f;
  const bool kept = lane < n && q >= g.pixThr;                                  // A8
  // K = col | row << 10 | module << 19 with a guard bit above col and row: K_i - K_j + (1 | 1 << 10) has both
  // fields in {0, 1, 2} and nothing else set iff same module, |d row| <= 1 and |d col| <= 1.  A digi that is
  // not kept gets a module of its own.
  const u32 K = kept ? ((rc0 & 511u) | (rc0 >> 9) << 10 | mIdx << 19) : (0x1000u + lane) << 19;
  const u32 Kb = K + 0x401u;
  u32 adj = 0;
#pragma unroll 4
  for (u32 j = 0; j < n; ++j) {
    const u32 t = Kb - __shfl_sync(0xFFFFFFFFu, K, j);
    const u32 bad = (t & ~0xC03u) | (t & (t >> 1) & 0x401u);
    adj |= (bad == 0u ? 1u : 0u) << j;
  }
  adj |= 1u << lane;
  // transitive closure (Warshall): after step j every lane that reaches j also reaches all of j's set
  u32 reach = adj;
  for (u32 j = 0; j < n; ++j) {
    const u32 rj = __shfl_sync(0xFFFFFFFFu, reach, j);
    if (reach & (1u << j)) reach |= rj;
  }
  const u32 root = (u32)__ffs((int)reach) - 1u;
  const bool isRoot = kept && root == lane;
  // sums of qf = q * 2^14 (A9) in binary64 (exact: at most 32 terms below 2^43), suffix sums along the lane list
  double qf = 0.0, qx = 0.0, qy = 0.0;
  u32 bR = 0, bC = 0;
  if (kept) { qf = (double)(q * 16384.0f); qx = qf * (double)(rc0 >> 9); qy = qf * (double)(rc0 & 511u); bR = box_rows(rc0 >> 9); bC = box_cols(rc0 & 511u); }
  const u32 most = __reduce_max_sync(0xFFFFFFFFu, (u32)__popc(reach));
  const u32 above = reach & (0xFFFFFFFEu << lane);
  u32 nxt = above ? (u32)__ffs((int)above) - 1u : 32u;
  for (u32 span = 1; span < most; span <<= 1) {
    const u32 src = nxt & 31u;
    const double a = __shfl_sync(0xFFFFFFFFu, qf, src), b = __shfl_sync(0xFFFFFFFFu, qx, src), c = __shfl_sync(0xFFFFFFFFu, qy, src);
    const u32 nn = __shfl_sync(0xFFFFFFFFu, nxt, src);
    const u32 r2 = __shfl_sync(0xFFFFFFFFu, bR, src), c2 = __shfl_sync(0xFFFFFFFFu, bC, src);
    if (nxt < 32u) { qf += a; qx += b; qy += c; bR = __vmaxu2(bR, r2); bC = __vmaxu2(bC, c2); nxt = nn; }
  }
  const bool keptC = isRoot && __double2ll_rz(qf) >= g.clusThrFixed;
  const u32 kb = __ballot_sync(0xFFFFFFFFu, keptC);
  const u32 kr = (u32)__popc(kb & lt & ~((1u << (mStart - s)) - 1u));           // rank among the module's kept clusters
  if (keptC) {
    const u32 o = mStart + kr;
    ev.stS[o] = qf; ev.stSx[o] = qx; ev.stSy[o] = qy;
    ev.stLabel[o] = s + lane; ev.stSize[o] = (u32)__popc(reach);
    ev.stBoxR[o] = bR; ev.stBoxC[o] = bC;
  }
  const u32 krRoot = __shfl_sync(0xFFFFFFFFu, keptC ? kr : kNoRank, root);
  if (lane < n) {
    ev.label[s + lane] = kept ? s + root : kInvalid;
    ev.clus[s + lane] = (kept && krRoot != kNoRank) ? (int32_t)krRoot : -1;
  }
  *keptDigis = __ballot_sync(0xFFFFFFFFu, kept); *roots = __ballot_sync(0xFFFFFFFFu, isRoot); *keptRoots = kb;
}

// ---- warp path: one module = digis [s, s+n), 0 < n <= kWarpCap, processed by the calling warp.
// Returns (kept digis, clusters, kept clusters) in all lanes.
__device__ __forceinline__ void warp_module(const EvDesc& ev, const Geom& g, u32 s, u32 n, WarpRegion& wr, float q0, u32 rc0,
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
  // The loads run one chunk ahead (the first chunk came with the call): charge, row and col together.
  u32 nKept = 0; bool dup = false;
  float qc = q0; u32 rcc = rc0;
  for (u32 i = lane; i < nPad; i += 32u) {
    float qn = 0.f; u32 rcn = 0;
    if (i + 32u < n) { qn = ev.charge[s + i + 32u]; rcn = (u32)ev.row[s + i + 32u] << 9 | (u32)ev.col[s + i + 32u]; }
    const u32 key = (i < n && qc >= g.pixThr) ? rcc : kNoKey;                  // A8
    qc = qn; rcc = rcn;
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
  // The first round needs no look-ups: with L = identity the minimum over the neighbours is the minimum
  // neighbour index.
  u32* L = tab;
  for (u32 i = lane; i < nPad; i += 32u) {
    const uint2 nb = wr.nb[i];
    u32 v = __vminu4(nb.x, nb.y);
    v = __vminu4(v, v >> 16); v = __vminu4(v, v >> 8);
    L[i] = min(i, v & 0xFFu);
  }
  __syncwarp();
  for (u32 i = lane; i < nPad; i += 32u) {
    u32 l = L[i], p;
    while ((p = L[l]) != l) l = p;
    L[i] = l;
  }
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
  u32* box = cnt + kAccRoots;                      // two words per cluster: rows, cols
  u32 nK = 0;
  for (u32 p0 = 0; p0 < nR; p0 += kAccRoots) {
    const u32 nAcc = min(nR - p0, kAccRoots);
    for (u32 i = lane; i < nAcc * 3u; i += 32u) acc[i] = 0.0;
    for (u32 i = lane; i < nAcc; i += 32u) { cnt[i] = 0u; box[2u * i] = 0u; box[2u * i + 1u] = 0u; }
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
      u32 bR = 0, bC = 0;
      if (in) {
        qf = (double)(ev.charge[s + i] * 16384.0f);
        qx = qf * (double)(key >> 9); qy = qf * (double)(key & 511u);
        bR = box_rows(key >> 9); bC = box_cols(key & 511u);
      }
      // suffix sums along each cluster's lane list by pointer jumping: the first lane ends with the total
      const u32 above = peers & (0xFFFFFFFEu << lane);
      u32 nxt = above ? (u32)__ffs((int)above) - 1u : 32u;
      for (u32 span = 1; span < most; span <<= 1) {
        const u32 src = nxt & 31u;
        const double a = __shfl_sync(0xFFFFFFFFu, qf, src), b = __shfl_sync(0xFFFFFFFFu, qx, src), c = __shfl_sync(0xFFFFFFFFu, qy, src);
        const u32 nn = __shfl_sync(0xFFFFFFFFu, nxt, src);
        const u32 r2 = __shfl_sync(0xFFFFFFFFu, bR, src), c2 = __shfl_sync(0xFFFFFFFFu, bC, src);
        if (nxt < 32u) { qf += a; qx += b; qy += c; bR = __vmaxu2(bR, r2); bC = __vmaxu2(bC, c2); nxt = nn; }
      }
      if (in && (peers & lt) == 0u) {                 // one owner per cluster and chunk
        double* a = acc + rk * 3u;
        a[0] += qf; a[1] += qx; a[2] += qy;
        cnt[rk] += (u32)__popc(peers);
        box[2u * rk] = __vmaxu2(box[2u * rk], bR); box[2u * rk + 1u] = __vmaxu2(box[2u * rk + 1u], bC);
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
        ev.stBoxR[o] = box[2u * rk]; ev.stBoxC[o] = box[2u * rk + 1u];
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
  u32 *perm, *parent, *root, *csize, *box; int32_t* knum; u64 *S, *Sx, *Sy;
  u32 nAll, nKept;
};

template <u32 kT = kClusterThreads>
__device__ __forceinline__ void dense_count(const EvDesc& ev, const Geom& g, u32 s, u32 nn,
                                            unsigned char* smemRaw, ClusterShared& sh, DenseCtx& cx,
                                            u32 capDigis = kSmemDigis, u32 capClusters = kSmemClusters) {
  const int tid = threadIdx.x, lane = tid & 31;
  const u32 bwPad = (g.bitmapWords + 3) & ~3u;
  u64* smS = reinterpret_cast<u64*>(smemRaw);
  u64* smSx = smS + capClusters;
  u64* smSy = smSx + capClusters;
  u32* smBox = reinterpret_cast<u32*>(smSy + capClusters);        // four maxima per cluster
  u32* smBitmap = smBox + 4u * capClusters;
  u32* smPrefix = smBitmap + bwPad;
  u32* smPerm = smPrefix + bwPad;
  u32* smParent = smPerm + capDigis;
  u32* smRoot = smParent + capDigis;
  u32* smSize = smRoot + capClusters;
  int32_t* smKnum = reinterpret_cast<int32_t*>(smSize + capClusters);
  u32* sScan = sh.scan;
  const u32 stride = g.stride;

  const bool digiInSmem = nn <= capDigis;
  u32* perm = digiInSmem ? smPerm : ev.wsPerm + s;
  u32* parent = digiInSmem ? smParent : ev.wsParent + s;
  cx.perm = perm; cx.parent = parent;
  cx.root = smRoot; cx.csize = smSize; cx.knum = smKnum; cx.S = smS; cx.Sx = smSx; cx.Sy = smSy; cx.box = smBox;

  // P0: clear the occupancy bitmap, init perm
  for (u32 i = tid; i < g.bitmapWords; i += kT) smBitmap[i] = 0;
  for (u32 i = tid; i < nn; i += kT) perm[i] = kInvalid;
  __syncthreads();
  // P1: kept flag (A8: q >= pixThr) and occupancy bits at padded coordinates (row+1, col+1)
  u32 myKept = 0;
  for (u32 i = tid; i < nn; i += kT) {
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
    const u32 per = (g.bitmapWords + kT - 1) / kT;
    const u32 lo = min(tid * per, g.bitmapWords), hi = min(lo + per, g.bitmapWords);
    u32 sum = 0;
    for (u32 i = lo; i < hi; ++i) sum += __popc(smBitmap[i]);
    u32 tot;
    u32 run = block_excl_scan<kT / 32>(sum, sScan, &tot);
    for (u32 i = lo; i < hi; ++i) { smPrefix[i] = run; run += __popc(smBitmap[i]); }
  }
  if (lane == 0 && myKept) atomicAdd(&ev.counters->nKept, myKept);
  __syncthreads();
  // P3: owner of each occupied pixel = the minimum digi index on it (duplicates, A6)
  for (u32 i = tid; i < nn; i += kT) {
    if (parent[i] == kInvalid) continue;
    const u32 b = ev.col[s + i] + 1u, wd = (ev.row[s + i] + 1u) * stride + (b >> 5);
    const u32 r = smPrefix[wd] + __popc(smBitmap[wd] & ((1u << (b & 31)) - 1u));
    atomicMin(perm + r, i);
  }
  __syncthreads();
  // P4: unions with the backward neighbours (W, NW, N, NE), decision tree:
  //     N ? {N} : { NE?, W ? {W} : NW? }   — spans every 8-adjacency once all pixels did it.
  for (u32 i = tid; i < nn; i += kT) {
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
  for (u32 i = tid; i < nn; i += kT) {
    if (parent[i] == kInvalid) continue;
    const u32 rt = uf_root(parent, i);
    if (rt != i) parent[i] = rt;
  }
  __syncthreads();
  // P6: ordinal of every root in ascending index (= ascending label) order -> perm[root]
  {
    const u32 per = (nn + kT - 1) / kT;
    const u32 lo = min(tid * per, nn), hi = min(lo + per, nn);
    u32 c = 0;
    for (u32 i = lo; i < hi; ++i) c += (parent[i] == i);
    u32 run = block_excl_scan<kT / 32>(c, sScan, &cx.nAll);
    if (cx.nAll > capClusters) {
      cx.root = ev.wsRoot + s; cx.csize = ev.wsSize + s; cx.knum = ev.wsKnum + s;
      cx.S = ev.wsS + s; cx.Sx = ev.wsSx + s; cx.Sy = ev.wsSy + s; cx.box = ev.wsBox + 4u * (size_t)s;
    }
    for (u32 i = lo; i < hi; ++i)
      if (parent[i] == i) { perm[i] = run; cx.root[run] = i; ++run; }
  }
  // P7: zero the accumulators
  for (u32 c = tid; c < cx.nAll; c += kT) { cx.S[c] = 0; cx.Sx[c] = 0; cx.Sy[c] = 0; cx.csize[c] = 0; cx.box[4u * c] = 0; cx.box[4u * c + 1u] = 0; cx.box[4u * c + 2u] = 0; cx.box[4u * c + 3u] = 0; }
  __syncthreads();
  // P8: exact fixed-point sums (A9): qf = q * 2^14 is an integer for every kept digi
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = parent[i];
    if (p == kInvalid) continue;
    const u32 c = perm[p];
    const u64 qf = (u64)__float2ll_rz(ev.charge[s + i] * 16384.0f);
    atomicAdd(reinterpret_cast<unsigned long long*>(cx.S + c), (unsigned long long)qf);
    atomicAdd(reinterpret_cast<unsigned long long*>(cx.Sx + c), (unsigned long long)(qf * ev.row[s + i]));
    atomicAdd(reinterpret_cast<unsigned long long*>(cx.Sy + c), (unsigned long long)(qf * ev.col[s + i]));
    atomicAdd(cx.csize + c, 1u);
    atomicMax(cx.box + 4u * c, 255u - (u32)ev.row[s + i]); atomicMax(cx.box + 4u * c + 1u, (u32)ev.row[s + i]);
    atomicMax(cx.box + 4u * c + 2u, 511u - (u32)ev.col[s + i]); atomicMax(cx.box + 4u * c + 3u, (u32)ev.col[s + i]);
  }
  __syncthreads();
  // P9: cluster threshold (A8, A9) and local numbering of kept clusters
  {
    const u32 per = (cx.nAll + kT - 1) / kT;
    const u32 lo = min(tid * per, cx.nAll), hi = min(lo + per, cx.nAll);
    u32 c = 0;
    for (u32 k = lo; k < hi; ++k) c += ((i64)cx.S[k] >= g.clusThrFixed);
    u32 run = block_excl_scan<kT / 32>(c, sScan, &cx.nKept);
    for (u32 k = lo; k < hi; ++k) cx.knum[k] = ((i64)cx.S[k] >= g.clusThrFixed) ? (int32_t)run++ : -1;
  }
  __syncthreads();
}

template <u32 kT = kClusterThreads>
__device__ __forceinline__ void dense_stage(const EvDesc& ev, u32 m, u32 s, u32 nn, const DenseCtx& cx) {
  const int tid = threadIdx.x;
  for (u32 k = tid; k < cx.nAll; k += kT) {
    const int32_t kn = cx.knum[k];
    if (kn < 0) continue;
    const u32 o = s + (u32)kn;                       // kn <= k < nn: inside the module's own range
    ev.stS[o] = __ll2double_rn((i64)cx.S[k]); ev.stSx[o] = __ll2double_rn((i64)cx.Sx[k]); ev.stSy[o] = __ll2double_rn((i64)cx.Sy[k]);
    ev.stLabel[o] = s + cx.root[k]; ev.stSize[o] = cx.csize[k];
    ev.stBoxR[o] = cx.box[4u * k] << 16 | cx.box[4u * k + 1u]; ev.stBoxC[o] = cx.box[4u * k + 2u] << 16 | cx.box[4u * k + 3u];
  }
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = cx.parent[i];
    u32 lab = kInvalid; int32_t cl = -1;
    if (p != kInvalid) { lab = s + p; cl = cx.knum[cx.perm[p]]; }
    ev.label[s + i] = lab;
    ev.clus[s + i] = cl;
  }
  if (tid == 0) {
    ev.modCount[m] = cx.nKept;
    if (cx.nKept) atomicAdd(&ev.grpCount[m / 32u], cx.nKept);
    if (cx.nAll) atomicAdd(&ev.counters->nClustersAll, cx.nAll);
  }
}

template <bool kSingle>
__global__ void __launch_bounds__(kClusterThreads, 4)
k_cluster(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv,
          LaunchCtl* __restrict__ lc, u32* __restrict__ bigList, u32 modBatch, const __grid_constant__ Geom g) {
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
        if (big && t - s > kMaxModuleDigis) { big = false; atomicOr(&ev.counters->status, 2u); ev.modCount[m] = 0u; }   // A9's own limit: PR_STATUS_CAPACITY, the module stays unclustered
      }
    }
    if (bigList) {                                      // a launch full of large modules: k_dense takes them (larger tiers)
      if (big) bigList[atomicAdd(&lc->nBig, 1u)] = gi;
      continue;
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

  // ---- phase 2: warp path.  A ticket is a batch of modBatch (1, 2 or 4) consecutive modules of one event.
  WarpRegion& wr = reinterpret_cast<WarpRegion*>(smemRaw)[warp];
  // Tickets shrink towards the end of a large launch (modBatch 4): the first nEvA events are handed out four
  // modules at a time, the next nEvB events two at a time, the rest one by one, so that the last tickets are short.
  const u32 bpe = (M + modBatch - 1) / modBatch, bpeB = (M + 1u) / 2u;
  const u32 nEvA = modBatch == 4u ? nEv - nEv / 4u : nEv, nEvB = modBatch == 4u ? (nEv - nEvA + 1u) / 2u : 0u;
  const u32 tA = nEvA * bpe, tB = tA + nEvB * bpeB, nTickets = tB + (nEv - nEvA - nEvB) * M;
  for (;;) {
    u32 t = 0;
    if (lane == 0) t = atomicAdd(&lc->modTicket, 1u);
    t = __shfl_sync(0xFFFFFFFFu, t, 0);
    if (t >= nTickets) break;
    u32 e, m0, nm;
    if (t < tA) { e = t / bpe; m0 = (t - e * bpe) * modBatch; nm = min(modBatch, M - m0); }
    else if (t < tB) { const u32 u = t - tA; e = u / bpeB; m0 = (u - e * bpeB) * 2u; nm = min(2u, M - m0); e += nEvA; }
    else { const u32 u = t - tB; e = u / M; m0 = u - e * M; nm = 1u; e += nEvA + nEvB; }
    const EvDesc& ev = kSingle ? single : batch[e];
    if (ev.counters->status & 1u) continue;
    const u32 st = lane <= nm ? ev.modDigiStart[m0 + lane] : 0u;
    u32 accK = 0, accA = 0, accG = 0;
    // The ticket's digis are contiguous.  The next unit's first chunk (32 digis) is loaded while the current unit
    // (a pack of small modules, or one module of 33..kWarpCap digis) is processed.
    const u32 sEnd = min(__shfl_sync(0xFFFFFFFFu, st, nm), ev.cap);
    auto preload = [&](u32 s, float* q, u32* rc) {
      *q = 0.f; *rc = 0u;
      if (s + lane < sEnd) { *q = ev.charge[s + lane]; *rc = (u32)ev.row[s + lane] << 9 | (u32)ev.col[s + lane]; }
    };
    float qNext; u32 rcNext;
    preload(__shfl_sync(0xFFFFFFFFu, st, 0), &qNext, &rcNext);
    for (u32 k = 0; k < nm;) {
      const u32 s = __shfl_sync(0xFFFFFFFFu, st, k), t1 = __shfl_sync(0xFFFFFFFFu, st, k + 1);
      if (t1 < s || t1 > ev.cap) {                           // inconsistent module table
        if (lane == 0) { atomicOr(&ev.counters->status, 2u); ev.modCount[m0 + k] = 0u; }   // PR_STATUS_CAPACITY
        preload(t1 <= ev.cap ? t1 : sEnd, &qNext, &rcNext);
        ++k;
        continue;
      }
      const float q0 = qNext; const u32 rc0 = rcNext;
      if (t1 - s > 32u) {                                    // one module of its own
        const u32 n = t1 - s;
        preload(t1, &qNext, &rcNext);
        if (n <= kWarpCap) {                                 // else: the dense path wrote this module
          u32 nk, nr, cnt;
          warp_module(ev, g, s, n, wr, q0, rc0, &nk, &nr, &cnt);
          accK += nk; accA += nr; accG += cnt;
          if (lane == 0) ev.modCount[m0 + k] = cnt;
        }
        ++k;
        continue;
      }
      // pack: modules k .. k2-1, consecutive, consistent, at most 32 digis together
      u32 k2 = k + 1u, e2 = t1, mIdx = 0, mStart = s;
      while (k2 < nm) {
        const u32 en = __shfl_sync(0xFFFFFFFFu, st, k2 + 1u);
        if (en < e2 || en > ev.cap || en - s > 32u) break;
        if (e2 - s <= lane) { mIdx = k2 - k; mStart = e2; }   // module k2 starts at e2
        e2 = en; ++k2;
      }
      preload(e2, &qNext, &rcNext);
      const u32 n = e2 - s;
      u32 kd = 0, rb = 0, kb = 0;
      if (n) warp_pack(ev, g, s, n, q0, rc0, mIdx, mStart, &kd, &rb, &kb);
      accK += (u32)__popc(kd); accA += (u32)__popc(rb); accG += (u32)__popc(kb);
      // kept clusters per module of the pack: lane j - k writes module j's
      {
        const u32 j = k + lane;
        const u32 lo = __shfl_sync(0xFFFFFFFFu, st, min(j, nm)) - s, hi = __shfl_sync(0xFFFFFFFFu, st, min(j + 1u, nm)) - s;
        if (j < k2) {
          const u32 mask = (hi >= 32u ? 0xFFFFFFFFu : (1u << hi) - 1u) & ~(lo >= 32u ? 0xFFFFFFFFu : (1u << lo) - 1u);
          ev.modCount[m0 + j] = (u32)__popc(kb & mask);
        }
      }
      k = k2;
    }
    if (lane == 0 && accG) atomicAdd(&ev.grpCount[m0 / 32u], accG);     // modBatch divides 32: one group per ticket
    if (lane == 0) {
      if (accK) atomicAdd(&ev.counters->nKept, accK);
      if (accA) atomicAdd(&ev.counters->nClustersAll, accA);
    }
  }
}

// ================================================================== k_dense (a3 + a4 for launches full of large modules)
// The dense path of k_cluster as a kernel of its own, for launches whose modules are large on average
// (BASELINE.json configs[4]: 6.7k digis per module): two CTAs per SM with 8192 digis / 512 clusters
// per module in shared memory instead of 2048 / 512, so the union-find of such a module never leaves
// the SM.  k_cluster only collects the large modules in that case (bigList); CTAs take them by ticket.
constexpr u32 kDenseThreads = 512;
template <bool kSingle>
__global__ void __launch_bounds__(kDenseThreads, 2)
k_dense(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, LaunchCtl* __restrict__ lc,
        const u32* __restrict__ bigList, const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ ClusterShared sh;
  const u32 M = g.M, nBig = lc->nBig;
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) sh.nBig = atomicAdd(&lc->bigTicket, 1u);
    __syncthreads();
    const u32 t = sh.nBig;
    if (t >= nBig) break;
    const u32 gk = bigList[t], e = gk / M, m = gk - e * M;
    const EvDesc& ev = kSingle ? single : batch[e];
    const u32 s = ev.modDigiStart[m], nn = ev.modDigiStart[m + 1] - s;
    DenseCtx cx;
    dense_count<kDenseThreads>(ev, g, s, nn, smemRaw, sh, cx, kDenseDigis, kDenseClusters);
    dense_stage<kDenseThreads>(ev, m, s, nn, cx);
  }
}

}  // namespace pixreco

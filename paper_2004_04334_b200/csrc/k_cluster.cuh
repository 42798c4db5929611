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
constexpr u32 kMediumCap = 1024;                 // one warp with its large arrays in the global workspace: up to this many digis
constexpr u32 kWarpRegion = 6784;                 // bytes of shared memory per warp: eight of them are what the CTA path needs anyway
constexpr u32 kWarpScratch = kWarpRegion - kWarpCap * (4 + 4 + 4 + 1 + 1);   // 3200 bytes
constexpr u32 kAccRoots = kWarpScratch / 44;      // 72 clusters accumulated per pass over a module (kAccWords = 11 words each)
constexpr u32 kModBatch = 8;                     // most modules per warp ticket (two units of four Run-3-like modules; tickets of 4: 3 % slower there, 1 % on the high pile-up batch);
                                                 // small launches use 2 or 1 so that every warp gets work (modBatch, a power of two)
constexpr u32 kNoKey = 0xFFFFFFFFu;
constexpr u32 kNoRank = 0xFFFFu;

struct WarpRegion {                 // kWarpRegion bytes of shared memory per warp
  u32 info[kWarpCap];               // col | row' << 9 | next digi of the column << 20 (kNoIdx: none); kNoKey for a digi below the pixel threshold
  float q[kWarpCap];                // charge
  u32 L[kWarpCap];                  // union-find forest (a word per digi: hooks are atomicMin), finally the root = minimum digi index of the
                                    // cluster in the low half; at a root the high half then takes the rank among the module's kept clusters
  unsigned char rk[kWarpCap];       // at a root: rank of its cluster among the module's clusters (ascending label)
  unsigned char rootAt[kWarpCap];   // root of the cluster with that rank
  __align__(16) unsigned char scratch[kWarpScratch];   // column heads, then the accumulators
};
static_assert(kWarpScratch >= kAccRoots * 44 && kWarpScratch >= 4 * (512 + 2), "scratch holds the accumulators and the column heads");
static_assert(sizeof(WarpRegion) == kWarpRegion, "the warp's region");

__host__ __device__ inline size_t dense_smem_bytes(u32 bitmapWords, u32 capDigis = kSmemDigis, u32 capClusters = kSmemClusters) {
  size_t w = (bitmapWords + 3) & ~3u;
  return (size_t)w * 4 * 2 + (size_t)capDigis * 4 * 2 + (size_t)capClusters * (4 + 4 + 4 + 8 * 3 + 4 * 4);
}
__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t dense = dense_smem_bytes(bitmapWords), warp = sizeof(WarpRegion) * (kClusterThreads / 32);
  return ((dense > warp ? dense : warp) + 15) & ~(size_t)15;
}

// The union-find forest of the dense path lives in shared memory (modules up to the shared tier) or in the global
// workspace.  ParentRef names it with its address space known at compile time: volatile loads and stores of shared
// memory proper (a generic volatile load goes through the global-memory path and waits on the long scoreboard).
template <bool kShared> struct ParentRef {
  u32* p;
  __device__ __forceinline__ u32 ld(u32 i) const {
    u32 v;
    if (kShared) asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"((u32)__cvta_generic_to_shared(p + i)) : "memory");
    else v = *reinterpret_cast<volatile u32*>(p + i);
    return v;
  }
  __device__ __forceinline__ void st(u32 i, u32 v) const {
    if (kShared) asm volatile("st.volatile.shared.u32 [%0], %1;" ::"r"((u32)__cvta_generic_to_shared(p + i)), "r"(v) : "memory");
    else *reinterpret_cast<volatile u32*>(p + i) = v;
  }
};
// Root of x, halving the path on the way (a node's parent only ever moves to another ancestor in its set, so
// concurrent finds and hooks stay consistent).  Only while unions are running: see uf_root.
template <bool kShared>
__device__ __forceinline__ u32 uf_find(ParentRef<kShared> parent, u32 x) {
  u32 p = parent.ld(x);
  while (p != x) {
    const u32 gp = parent.ld(p);
    if (gp != p) parent.st(x, gp);
    x = p; p = gp;
  }
  return x;
}
// Root of x without touching the forest: for the flattening pass, where a late halving store could
// overwrite another thread's final root.
template <bool kShared>
__device__ __forceinline__ u32 uf_root(ParentRef<kShared> parent, u32 x) {
  u32 p;
  while ((p = parent.ld(x)) != x) x = p;
  return x;
}
// Hook the larger root under the smaller one (atomicMin), so the final root of every set is its
// minimum digi index = the canonical label (A10).
template <bool kShared>
__device__ __forceinline__ void uf_union(ParentRef<kShared> parent, u32 a, u32 b) {
  for (;;) {
    a = uf_find(parent, a); b = uf_find(parent, b);
    if (a == b) return;
    if (a < b) { u32 t = a; a = b; b = t; }
    const u32 old = atomicMin(parent.p + a, b);
    if (old == a) return;
    a = old;
  }
}

// What k_cluster / k_dense leave in clus[] for k_finalize: the digi's cluster as its rank among the kept clusters of
// its module (below 2^17, A9) with the module's position among 128 consecutive modules above it, so that k_finalize
// adds the module's first event-wide cluster number without looking the module up.
__device__ __forceinline__ u32 clus_ranked(u32 rank, u32 module) { return rank | (module & 127u) << 20; }

struct ClusterShared {
  u32 scan[16];
  u32 nBig, big[kClusterThreads];
};

// Bounding box (A28) as two words of two halfword maxima each: rows max(255 - row) << 16 | max(row), cols
// max(511 - col) << 16 | max(col); __vmaxu2 combines two boxes.
__device__ __forceinline__ u32 box_rows(u32 row) { return (255u - row) << 16 | row; }
__device__ __forceinline__ u32 box_cols(u32 col) { return (511u - col) << 16 | col; }

// ---- warp path, one digi per lane: a PACK of consecutive modules with at most 32 digis together, digis
// [s, s+n).  Everything lives in registers: lane i learns its neighbours by comparing its (module, row,
// col) with every other lane's (n shuffles, no table; two digis on one pixel are simply adjacent, A6),
// adjacency and reachability are 32-bit lane masks (Warshall closure with shuffles), a cluster's
// minimum lane is its root, sums run along each cluster's lane list.  mIdx/mStart: the lane's module
// (index within the pack) and that module's first digi.  Returns the ballots of kept digis, of roots
// and of roots of kept clusters.
__device__ __forceinline__ void warp_pack(const EvDesc& ev, const Geom& g, u32 s, u32 n, float q0, u32 rc0, u32 mFirst, u32 mIdx, u32 mStart,
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
    stage_store(ev.staged + o, qf, qx, qy, s + lane, (u32)__popc(reach), bR, bC);
  }
  const u32 krRoot = __shfl_sync(0xFFFFFFFFu, keptC ? kr : kNoRank, root);
  if (lane < n) {
    ev.label[s + lane] = kept ? s + root : kInvalid;
    ev.clus[s + lane] = (kept && krRoot != kNoRank) ? (int32_t)clus_ranked(krRoot, mFirst + mIdx) : -1;
  }
  *keptDigis = __ballot_sync(0xFFFFFFFFu, kept); *roots = __ballot_sync(0xFFFFFFFFu, isRoot); *keptRoots = kb;
}

// ---- warp path: one module = digis [s, s+n), 32 < n <= kWarpCap, processed by the calling warp with only __syncwarp
// between its passes.  Returns (kept digis, clusters, kept clusters) in all lanes.
//   P1  load; kept flag (A8); every kept digi is pushed on the list of its COLUMN (head per column, `next` inside the
//       digi's info word) with one atomicExch on the head.
//   P2  neighbours: a walk over the digi's own column list (N = row - 1; a second digi on the same pixel, A6) and over
//       the list of the column before (NW, W, SW).  Of these backward neighbours (column-major order) at most two
//       edges are kept:  W ? {W} : { N ? N : NW,  SW }  — the dropped ones are adjacent to a kept one and are found from
//       there, so the kept edges span every 8-adjacency.  A digi that shares its pixel with one of lower index keeps
//       only the edge to that one.
//   P3  (inside P2's loop) union of the two ends of every kept edge on the forest L[] (one word per digi, L[i] <= i, a
//       digi of i's component; a root has L[i] == i): both roots by plain loads, then atomicMin(L[larger root],
//       smaller root).  If the larger one was a root it now hangs under the smaller one; if another lane had hooked it
//       meanwhile, atomicMin left it under the smaller of the two candidates and the union goes on with the other pair
//       (wm_union).  No edge list, no rounds: an edge is resolved when its lane leaves the loop.  Roots only ever go
//       under smaller digis: the final root of a component is its minimum digi index = the canonical label (A10).
//   P4  flatten; rank of every root in ascending index (= label) order.
//   P5  per-cluster sums S, Sx, Sy of qf = q * 2^14 (A9) as 64-bit integers in shared memory, size and bounding box,
//       accRoots clusters per pass: every digi adds to its cluster's eleven words with native 32-bit atomics (a 64-bit
//       add is the add on the low word, whose return value tells this thread whether ITS add carried, and an add of
//       high word + carry when that is not zero: acc_add64).
//   P6  the roots apply the cluster threshold (A8), number the kept clusters and stage their sums; the rank among the
//       module's kept clusters goes into the free high half of the root's own word L[root].
//   P7  per-digi outputs: label (final), cluster rank within the module.
// Where warp_module keeps its arrays.  A module of at most kWarpCap digis lives in the warp's own region of shared
// memory with one-byte digi indices; a module of up to kMediumCap digis (kMedium) keeps the forest L[], the column
// heads and the accumulators there and, while they fit, the info words and the cluster ranks too (wm_store_medium);
// the rest lies in the event's global workspace at the module's own digi range (cached in L1/L2; the module belongs
// to this warp alone).
template <bool kMedium> struct WmStore;
template <> struct WmStore<false> {
  typedef unsigned char idx_t;
  static constexpr u32 kNoIdx = 0x7FFu;
  u32* info; float* q; u32* L; idx_t *rk, *rootAt; unsigned char* scratch; u32 accRoots;
};
template <> struct WmStore<true> {
  typedef u16 idx_t;
  static constexpr u32 kNoIdx = 0x7FFu;
  u32* info; float* q; u32* L; idx_t *rk, *rootAt; unsigned char* scratch; u32 accRoots;
};
__device__ __forceinline__ WmStore<false> wm_store_small(WarpRegion& r) {
  WmStore<false> st;
  st.info = r.info; st.q = r.q; st.L = r.L; st.rk = r.rk; st.rootAt = r.rootAt; st.scratch = r.scratch; st.accRoots = kAccRoots;
  return st;
}
// Medium module = digis [s, s + n), 256 < n <= kMediumCap: the warp's region always holds the forest L (a word per digi),
// the column heads and then the accumulators.  While eight bytes per digi leave room for the column heads (some 600
// digis: the hot modules of a high pile-up event) the info words sit beside L too: the neighbour walk of P2 then stays
// in shared memory; with ten bytes per digi (some 480 digis) the cluster ranks as well.  What does not fit lies in the
// event's global workspace at the module's own digi range.
__device__ __forceinline__ u32 wm_head_bytes(const Geom& g) { return ((g.C + 2u + 3u) & ~3u) * 4u; }
__device__ __forceinline__ WmStore<true> wm_store_medium(WarpRegion& r, const EvDesc& ev, const Geom& g, u32 s, u32 n) {
  WmStore<true> st;
  unsigned char* base = reinterpret_cast<unsigned char*>(&r);
  const u32 nCap = (n + 31u) & ~31u, room = kWarpRegion - wm_head_bytes(g);
  st.L = reinterpret_cast<u32*>(base);
  st.info = ev.wsPerm + s; st.rk = reinterpret_cast<u16*>(ev.wsRoot + s);
  u32 used = 4u * nCap;
  if (8u * nCap <= room) { st.info = reinterpret_cast<u32*>(base + used); used += 4u * nCap; }
  if (10u * nCap <= room) { st.rk = reinterpret_cast<u16*>(base + used); used += 2u * nCap; }
  used = (used + 15u) & ~15u;
  st.scratch = base + used; st.accRoots = (kWarpRegion - used) / 44u;
  st.q = nullptr; st.rootAt = reinterpret_cast<u16*>(ev.wsSize + s);
  return st;
}
static_assert(kWarpRegion - 4u * kMediumCap >= 4u * (512u + 4u), "L of the largest medium module leaves room for the column heads");

template <typename idx_t>
__device__ __forceinline__ u32 wm_find(const idx_t* L, u32 x) {
  u32 l = L[x];
  for (;;) {
    const u32 p = L[l];
    if (p == l) return l;
    l = p;
  }
}
// acc[0..1] += v as a 64-bit integer with native 32-bit shared-memory atomics: the add on the low word returns what was
// there, so this thread knows whether ITS add carried, and takes the carry along with its high word.
constexpr u32 kAccWords = 11;
constexpr u32 kMomentOff = 8;                     // Sx, Sy are accumulated relative to (root row - 8, root col - 8)
__device__ __forceinline__ void acc_add64(u32* a, u64 v) {
  const u32 lo = (u32)v;
  u32 hi = (u32)(v >> 32);
  const u32 old = atomicAdd(a, lo);
  hi += old > ~lo ? 1u : 0u;
  if (hi) atomicAdd(a + 1, hi);
}

// Union of the sets of a and b on a forest of words (L[x] <= x): roots by plain loads, then the larger root goes under
// the smaller one with atomicMin; if it was no root any more (another lane hooked it meanwhile) its former parent and the
// smaller root are merged next.  Lanes of one warp may run this side by side on one forest.
__device__ __forceinline__ void wm_union(u32* L, u32 a, u32 b) {
  a = wm_find(L, a); b = wm_find(L, b);
  while (a != b) {
    const u32 hi = max(a, b), lo = min(a, b);
    const u32 old = atomicMin(L + hi, lo);
    if (old == hi) break;
    a = old; b = lo;
  }
}

// Union of the sets of i, e1 and e2 (e2 == i: none): the three roots in one loop (independent loads), then the larger
// roots under the smallest one; a root that another lane had hooked meanwhile takes the slow way (wm_union).
__device__ __forceinline__ void wm_union3(u32* L, u32 i, u32 e1, u32 e2) {
  u32 a = L[i], b = L[e1], c = L[e2];
  for (;;) {
    const u32 pa = L[a], pb = L[b], pc = L[c];
    if (pa == a && pb == b && pc == c) break;
    a = pa; b = pb; c = pc;
  }
  const u32 m = min(a, min(b, c));
  u32 oa = a, ob = b, oc = c;
  if (a != m) oa = atomicMin(L + a, m);
  if (b != m) ob = atomicMin(L + b, m);
  if (c != m && c != a && c != b) oc = atomicMin(L + c, m);
  if (oa != a) wm_union(L, oa, m);
  if (ob != b) wm_union(L, ob, m);
  if (oc != c) wm_union(L, oc, m);
}

// A UNIT may hold up to four consecutive modules (digis [s, s + n); module j + 1 of the unit starts at digi s + bnd.b[j],
// kNoBnd if the unit has no such module): their pixels are stacked along the row index, 512 rows apart
// (row' = row | j << 9: bits 18-19 of the info word are the module, and rows of two modules are never adjacent), so that
// one pass clusters them all and no edge crosses a module border.  Kept clusters are ranked per module; cntOut[j] receives module j's number of kept clusters.
constexpr u32 kNoBnd = 0xFFFFFFFFu;
struct UnitBounds { u32 b[3]; };
__device__ __forceinline__ u32 unit_module(const UnitBounds& bnd, u32 i) { return (i >= bnd.b[0] ? 1u : 0u) + (i >= bnd.b[1] ? 1u : 0u) + (i >= bnd.b[2] ? 1u : 0u); }

template <bool kMedium>
__device__ __forceinline__ void warp_module(const EvDesc& ev, const Geom& g, u32 s, u32 n, const WmStore<kMedium>& wr, float q0, u32 rc0,
                                            u32 mFirst, const UnitBounds& bnd, u32* nKeptDigis, u32* nRootsOut, u32 (&cntOut)[4]) {
  typedef typename WmStore<kMedium>::idx_t idx_t;
  constexpr u32 kNoIdx = WmStore<kMedium>::kNoIdx;
  const u32 kAccRoots = wr.accRoots;
  const u32 lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  const u32 nPad = (n + 31u) & ~31u;
  u32* head = reinterpret_cast<u32*>(wr.scratch);            // [C + 2]: head[c + 1] = last digi pushed on column c, head[0] stays empty
  const u16* rootOf = reinterpret_cast<const u16*>(wr.L);   // after P4: low half of L[i] = root of i ...
  u16* krAt = reinterpret_cast<u16*>(wr.L) + 1;             // ... after P6: high half of L[root] = rank among the module's KEPT clusters

  // P1
  // The lists are per (column, parity of the module within the unit): the odd modules' columns start `off` heads
  // further on, in what the accumulators do not need yet (a unit's four modules would otherwise share every column's
  // list, and a digi walks the whole list).  Where the two ranges overlap a list holds digis of two columns; the
  // walks compare the whole (column, row') key.  A medium module is alone: one list per column.
  const u32 nHead = kMedium ? g.C + 2u : kWarpScratch / 4u, off = kMedium ? 0u : nHead - (g.C + 2u);
  for (u32 i = lane; i < nHead; i += 32u) head[i] = 0xFFFFFFFFu;
  __syncwarp();
  u32 nKept = 0;
  float qc = q0; u32 rcc = rc0;
  for (u32 i = lane; i < nPad; i += 32u) {
    float qn = 0.f; u32 rcn = 0;
    if (i + 32u < n) { qn = ev.charge[s + i + 32u]; rcn = (u32)ev.row[s + i + 32u] << 9 | (u32)ev.col[s + i + 32u]; }
    const bool kept = i < n && qc >= g.pixThr;                                   // A8
    if (!kMedium) wr.q[i] = qc;
    wr.L[i] = i;
    u32 next = kNoIdx;
    const u32 mu = unit_module(bnd, i);
    if (kept) next = atomicExch(head + (rcc & 511u) + 1u + (mu & 1u) * off, i) & kNoIdx;
    if (!kMedium || i < n) wr.info[i] = kept ? (rcc | mu << 18 | next << 20) : kNoKey;   // (the global workspace ends at n)
    nKept += __popc(__ballot_sync(0xFFFFFFFFu, kept));
    qc = qn; rcc = rcn;
  }
  __syncwarp();
  // P2
  for (u32 i = lane; i < nPad; i += 32u) {
    const u32 x = (!kMedium || i < n) ? wr.info[i] : kNoKey;
    u32 e1 = i, e2 = i;
    if (x != kNoKey) {
      const u32 key = x & 0xFFFFFu, c = x & 511u, hb = c + ((x >> 18) & 1u) * off;   // key = col | row' << 9 (row' holds the module)
      u32 W = kNoIdx, N = kNoIdx, NW = kNoIdx, SW = kNoIdx, own = i;
      for (u32 j = head[hb + 1u]; j < kNoIdx;) {   // the digi's own column (never empty): N, and the lowest digi on the same pixel
        const u32 y = wr.info[j], ky = y & 0xFFFFFu;
        if (ky == key) own = min(own, j);
        if (ky + 512u == key) N = j;
        j = y >> 20;
      }
      for (u32 j = c ? head[hb] : kNoIdx; j < kNoIdx;) {   // the column before: NW, W, SW
        const u32 y = wr.info[j], d = (y & 0xFFFFFu) - (key - 1u);
        if (d == 0u) W = j;
        if (d == 0u - 512u) NW = j;
        if (d == 512u) SW = j;
        j = y >> 20;
      }
      if (own != i) e1 = own;
      else if (W != kNoIdx) e1 = W;
      else {
        e1 = N != kNoIdx ? N : NW;
        if (e1 == kNoIdx) { e1 = SW != kNoIdx ? SW : i; }
        else if (SW != kNoIdx) e2 = SW;
      }
    }
    // P3: the unions of the kept edges, at once
    if (e1 != i) wm_union3(wr.L, i, e1, e2);
  }
  __syncwarp();
  // P4
  u32 nR = 0;
  for (u32 i = lane; i < nPad; i += 32u) {
    const bool kept = (!kMedium || i < n) && wr.info[i] != kNoKey;
    u32 l = i;
    if (kept) { l = wm_find(wr.L, i); wr.L[i] = l; }
    const bool isRoot = kept && l == i;
    const u32 rb = __ballot_sync(0xFFFFFFFFu, isRoot);
    if (isRoot) { const u32 k = nR + __popc(rb & lt); wr.rk[i] = (idx_t)k; wr.rootAt[k] = (idx_t)i; }
    nR += __popc(rb);
  }
  __syncwarp();
  // P5, P6
  u32* acc = reinterpret_cast<u32*>(wr.scratch);             // kAccWords per cluster: S, Sx, Sy as (low, high) words, size, four box maxima
  cntOut[0] = cntOut[1] = cntOut[2] = cntOut[3] = 0u;
  for (u32 p0 = 0; p0 < nR; p0 += kAccRoots) {
    const u32 nAcc = min(nR - p0, kAccRoots);
    for (u32 i = lane; i < nAcc * kAccWords; i += 32u) acc[i] = 0u;
    __syncwarp();
    // Lane l takes the digis [l c, (l + 1) c) (c = chunks of the unit), not every 32nd one: neighbouring digis mostly
    // share their cluster, and 32 lanes that add to the same few words in one instruction are served one after the
    // other.  The lanes start at different offsets inside their blocks (rotated by l / (32 / gcd(c, 32))), which
    // puts the 32 loads of an instruction in 32 different banks.
    const u32 cN = nPad >> 5, aN = min((u32)__ffs((int)cN) - 1u, 5u), offN = lane >> (5u - aN);
    for (u32 kk = 0; kk < cN; ++kk) {
      u32 t = kk + offN;
      if (t >= cN) t -= cN;
      const u32 i = lane * cN + t;
      const u32 x = (!kMedium || i < n) ? wr.info[i] : kNoKey;
      if (x != kNoKey) {
        const u32 r = rootOf[2u * i], rk = (u32)wr.rk[r] - p0;
        if (rk < nAcc) {
          const u32 row = (x >> 9) & 0x1FFu, col = x & 511u;
          const i64 qf = __float2ll_rz((kMedium ? ev.charge[s + i] : wr.q[i]) * 16384.0f);
          // Sx and Sy are taken relative to the cluster's root pixel (kMomentOff rows / columns before it): the products
          // then stay below 2^32 as a rule and their high words are zero, i.e. one atomic instead of two (any other
          // value is still added exactly, as a 64-bit integer modulo 2^64; P6 adds the root's share back)
          const u32 x0 = wr.info[r];
          const int dr = (int)(row + kMomentOff) - (int)((x0 >> 9) & 0x1FFu), dc = (int)(col + kMomentOff) - (int)(x0 & 511u);
          u32* a = acc + rk * kAccWords;
          acc_add64(a, (u64)qf); acc_add64(a + 2, (u64)(qf * dr)); acc_add64(a + 4, (u64)(qf * dc));
          atomicAdd(a + 6, 1u);
          atomicMax(a + 7, 255u - row); atomicMax(a + 8, row); atomicMax(a + 9, 511u - col); atomicMax(a + 10, col);
        }
      }
    }
    __syncwarp();
    for (u32 k = lane; k < ((nAcc + 31u) & ~31u); k += 32u) {
      i64 S = 0;
      u32 root = 0, mr = 4u;
      const u32* a = acc + k * kAccWords;
      if (k < nAcc) { S = (i64)((u64)a[0] | (u64)a[1] << 32); root = wr.rootAt[p0 + k]; mr = unit_module(bnd, root); }
      const bool keptC = k < nAcc && S >= g.clusThrFixed;
      const u32 kb = __ballot_sync(0xFFFFFFFFu, keptC);
      u32 mine = 0;                                  // the kept roots of this chunk in my module; the roots come in ascending order
#pragma unroll
      for (u32 j = 0; j < 4u; ++j) {
        const u32 mj = __ballot_sync(0xFFFFFFFFu, mr == j) & kb;
        if (mr == j) mine = mj;
        cntOut[j] += (u32)__popc(mj);
      }
      if (k < nAcc) {
        u32 kr = kNoRank;
        if (keptC) {
          // rank among the kept clusters of the root's own module: those of earlier chunks + those before me in this one
          const u32 before = mr == 0u ? cntOut[0] : mr == 1u ? cntOut[1] : mr == 2u ? cntOut[2] : cntOut[3];
          kr = before - (u32)__popc(mine) + (u32)__popc(mine & lt);
          const u32 o = s + (mr ? bnd.b[mr - 1u] : 0u) + kr;
          const u32 x0 = wr.info[root];
          const i64 Sx = (i64)((u64)a[2] | (u64)a[3] << 32) + ((i64)((x0 >> 9) & 0x1FFu) - (i64)kMomentOff) * S;
          const i64 Sy = (i64)((u64)a[4] | (u64)a[5] << 32) + ((i64)(x0 & 511u) - (i64)kMomentOff) * S;
          stage_store(ev.staged + o, __ll2double_rn(S), __ll2double_rn(Sx), __ll2double_rn(Sy), s + root, a[6], a[7] << 16 | a[8], a[9] << 16 | a[10]);
        }
        krAt[2u * root] = (u16)kr;
      }
    }
    __syncwarp();
  }
  // P7
  for (u32 i = lane; i < n; i += 32u) {
    u32 lab = kInvalid; int32_t cl = -1;
    const u32 x = wr.info[i];
    if (x != kNoKey) {
      const u32 r = rootOf[2u * i], kr = krAt[2u * r];
      lab = s + r;
      if (kr != kNoRank) cl = (int32_t)clus_ranked(kr, mFirst + ((x >> 18) & 3u));
    }
    ev.label[s + i] = lab; ev.clus[s + i] = cl;
  }
  *nKeptDigis = nKept; *nRootsOut = nR;
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
  // A thread first finds its (at most two) partners — where to look is a different place in every branch of the tree, what
  // to do with them is not: the unions then run with all the threads that have one side by side.
  for (u32 i0 = 0; i0 < nn; i0 += kT) {
    const u32 i = i0 + tid;
    u32 e1 = kInvalid, e2 = kInvalid;
    if (i < nn && parent[i] != kInvalid) {
      const u32 prow = ev.row[s + i] + 1u, b = ev.col[s + i] + 1u;
      const u32 wd = prow * stride + (b >> 5);
      const u32 r = smPrefix[wd] + __popc(smBitmap[wd] & ((1u << (b & 31)) - 1u));
      const u32 owner = perm[r];
      if (owner != i) e1 = owner;
      else {
        const u32 pos = b - 1u, w0 = pos >> 5, shf = pos & 31u;
        const u32 rowAbove = (prow - 1u) * stride, rowSelf = prow * stride;
        const u32 nb = __funnelshift_r(smBitmap[rowAbove + w0], smBitmap[rowAbove + w0 + 1], shf) & 7u;
        const u32 cb = __funnelshift_r(smBitmap[rowSelf + w0], smBitmap[rowSelf + w0 + 1], shf) & 7u;
        // pixel 1 (bit offset from b - 1 in the row above: 0 = NW, 1 = N, 2 = NE; in the own row: 0 = W) and pixel 2
        u32 p1 = kInvalid, p2 = kInvalid;               // rowBase << 16 | padded column
        if (nb & 2u) p1 = rowAbove << 16 | b;
        else {
          if (nb & 4u) p1 = rowAbove << 16 | (b + 1u);
          if (cb & 1u) p2 = rowSelf << 16 | (b - 1u);
          else if (nb & 1u) p2 = rowAbove << 16 | (b - 1u);
        }
        if (p1 == kInvalid) { p1 = p2; p2 = kInvalid; }
        auto owner_at = [&](u32 p) -> u32 {
          const u32 bb = p & 0xFFFFu, ww = (p >> 16) + (bb >> 5);
          return perm[smPrefix[ww] + __popc(smBitmap[ww] & ((1u << (bb & 31)) - 1u))];
        };
        if (p1 != kInvalid) e1 = owner_at(p1);
        if (p2 != kInvalid) e2 = owner_at(p2);
      }
    }
    if (digiInSmem) {
      if (e1 != kInvalid) uf_union(ParentRef<true>{parent}, i, e1);
      if (e2 != kInvalid) uf_union(ParentRef<true>{parent}, i, e2);
    } else {
      if (e1 != kInvalid) uf_union(ParentRef<false>{parent}, i, e1);
      if (e2 != kInvalid) uf_union(ParentRef<false>{parent}, i, e2);
    }
  }
  __syncthreads();
  // P5: flatten (roots are stable now)
  for (u32 i = tid; i < nn; i += kT) {
    if (parent[i] == kInvalid) continue;
    const u32 rt = digiInSmem ? uf_root(ParentRef<true>{parent}, i) : uf_root(ParentRef<false>{parent}, i);
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
    stage_store(ev.staged + o, __ll2double_rn((i64)cx.S[k]), __ll2double_rn((i64)cx.Sx[k]), __ll2double_rn((i64)cx.Sy[k]), s + cx.root[k], cx.csize[k],
                cx.box[4u * k] << 16 | cx.box[4u * k + 1u], cx.box[4u * k + 2u] << 16 | cx.box[4u * k + 3u]);
  }
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = cx.parent[i];
    u32 lab = kInvalid; int32_t cl = -1;
    if (p != kInvalid) { lab = s + p; cl = cx.knum[cx.perm[p]]; if (cl >= 0) cl = (int32_t)clus_ranked((u32)cl, m); }
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

  // ---- phase 1: modules with more than kWarpCap digis.  Module (e, m) has index e * M + m; lane l of warp w of the
  // launch looks at the indices congruent to l * (number of warps) + w, one per trip (neighbouring hot modules go to
  // different warps).  More than kMediumCap digis (with a bigList: more than kWarpCap, handed to k_dense): the whole
  // CTA on one module at a time (dense path).  kWarpCap + 1 .. kMediumCap digis: remembered (one bit per trip) and
  // clustered afterwards by ONE warp each (the warp path with its large arrays in the global workspace): no warp
  // waits for another one there, and these heavy modules are done before the tickets of phase 2.
  WarpRegion& wr = reinterpret_cast<WarpRegion*>(smemRaw)[warp];
  const u32 nWarps = gridDim.x * (kClusterThreads / 32u), gw = blockIdx.x * (kClusterThreads / 32u) + warp;
  const u32 bigAbove = bigList ? kWarpCap : kMediumCap;
  auto medium_modules = [&](u32 base0, u32 bits) {
    for (u32 it = 0; it < 32u; ++it) {
      const u32 gi = base0 + it * 32u * nWarps + lane * nWarps + gw;
      for (u32 todo = __ballot_sync(0xFFFFFFFFu, (bits >> it) & 1u); todo; todo &= todo - 1u) {
        const u32 gk = __shfl_sync(0xFFFFFFFFu, gi, __ffs((int)todo) - 1), e = gk / M, m = gk - e * M;
        const EvDesc& ev = kSingle ? single : batch[e];
        const u32 s = ev.modDigiStart[m], nn = ev.modDigiStart[m + 1] - s;
        const float q0 = ev.charge[s + lane]; const u32 rc0 = (u32)ev.row[s + lane] << 9 | (u32)ev.col[s + lane];
        u32 nk, nr, cnts[4];
        const UnitBounds one = {{kNoBnd, kNoBnd, kNoBnd}};
        warp_module<true>(ev, g, s, nn, wm_store_medium(wr, ev, g, s, nn), q0, rc0, m, one, &nk, &nr, cnts);
        const u32 cnt = cnts[0];
        if (lane == 0) {
          ev.modCount[m] = cnt;
          if (cnt) atomicAdd(&ev.grpCount[m / 32u], cnt);
          if (nk) atomicAdd(&ev.counters->nKept, nk);
          if (nr) atomicAdd(&ev.counters->nClustersAll, nr);
        }
        __syncwarp();
      }
    }
  };
  u32 medBits = 0, trip = 0, base0 = 0;
  for (u32 base = 0; base < total; base += 32u * nWarps, ++trip) {
    if (trip == 32u) { if (__any_sync(0xFFFFFFFFu, medBits != 0u)) medium_modules(base0, medBits); medBits = 0; trip = 0; base0 = base; }
    const u32 gi = base + lane * nWarps + gw;
    bool big = false;
    if (gi < total) {
      const u32 e = gi / M, m = gi - e * M;
      const EvDesc& ev = kSingle ? single : batch[e];
      const u32 s = ev.modDigiStart[m], t = ev.modDigiStart[m + 1];   // (asked for beside the status word: one round trip)
      if (!(ev.counters->status & 1u)) {              // A5 violated: modDigiStart is undefined, no per-digi work
        const bool ok = t >= s && t <= ev.cap;
        big = ok && t - s > bigAbove;
        if (ok && !big && t - s > kWarpCap) medBits |= 1u << trip;
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
  if (__any_sync(0xFFFFFFFFu, medBits != 0u)) medium_modules(base0, medBits);

  // ---- phase 2: warp path.  A ticket is a batch of modBatch (1, 2 or kModBatch = 8) consecutive modules of one event.
  // Tickets shrink towards the end of a large launch (modBatch 8): the first nEvA events are handed out eight
  // modules at a time, the next nEvB events two at a time, the rest one by one, so that the last tickets are short.
  const u32 bpe = (M + modBatch - 1) / modBatch, bpeB = (M + 1u) / 2u;
  const u32 nEvA = modBatch == kModBatch ? nEv - nEv / 4u : nEv, nEvB = modBatch == kModBatch ? (nEv - nEvA + 1u) / 2u : 0u;
  const u32 tA = nEvA * bpe, tB = tA + nEvB * bpeB, nTickets = tB + (nEv - nEvA - nEvB) * M;
  // Warp w's first ticket is ticket w, without a trip to the counter (all the warps of a launch would meet there at its
  // start: some thousand atomics on one word); the counter hands out the tickets from nWarps on.  A launch with a warp
  // for every ticket — a single event — never goes there: the trip after the work is done is off the event's latency too.
  const bool oneEach = nTickets <= nWarps;
  for (u32 trip = 0;; ++trip) {
    u32 t = gw;
    if (trip) {
      if (oneEach) break;
      if (lane == 0) t = nWarps + atomicAdd(&lc->modTicket, 1u);
      t = __shfl_sync(0xFFFFFFFFu, t, 0);
    }
    if (t >= nTickets) break;
    u32 e, m0, nm;
    if (t < tA) { e = t / bpe; m0 = (t - e * bpe) * modBatch; nm = min(modBatch, M - m0); }
    else if (t < tB) { const u32 u = t - tA; e = u / bpeB; m0 = (u - e * bpeB) * 2u; nm = min(2u, M - m0); e += nEvA; }
    else { const u32 u = t - tB; e = u / M; m0 = u - e * M; nm = 1u; e += nEvA + nEvB; }
    const EvDesc& ev = kSingle ? single : batch[e];
    const u32 st = lane <= nm ? ev.modDigiStart[m0 + lane] : 0u;      // (asked for together with the status: one round trip)
    if (ev.counters->status & 1u) continue;
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
      if (t1 - s > kWarpCap) {                               // phase 1 wrote this module
        preload(t1, &qNext, &rcNext);
        ++k;
        continue;
      }
      // unit: modules k .. k2-1, consecutive, consistent, at most kWarpCap digis together
      u32 k2 = k + 1u, e2 = t1, mIdx = 0, mStart = s;
      while (k2 < nm) {
        const u32 en = __shfl_sync(0xFFFFFFFFu, st, k2 + 1u);
        if (en < e2 || en > ev.cap || en - s > kWarpCap) break;
        if (k2 - k >= 4u && en - s > 32u) break;              // at most four modules in a unit of the shared-memory path (eight: spills, 5 % slower)
        if (e2 - s <= lane) { mIdx = k2 - k; mStart = e2; }   // module k2 starts at e2 (what a pack of at most 32 digis needs)
        e2 = en; ++k2;
      }
      preload(e2, &qNext, &rcNext);
      const u32 n = e2 - s;
      if (n > 32u) {                                         // shared-memory path, all modules of the unit in one pass
        UnitBounds bnd;
#pragma unroll
        for (u32 j = 0; j < 3u; ++j) {
          const u32 v = __shfl_sync(0xFFFFFFFFu, st, min(k + 1u + j, nm));
          bnd.b[j] = k + 1u + j < k2 ? v - s : kNoBnd;
        }
        u32 nk, nr, cnts[4];
        warp_module<false>(ev, g, s, n, wm_store_small(wr), q0, rc0, m0 + k, bnd, &nk, &nr, cnts);
        accK += nk; accA += nr; accG += cnts[0] + cnts[1] + cnts[2] + cnts[3];
        if (lane < k2 - k) ev.modCount[m0 + k + lane] = lane == 0u ? cnts[0] : lane == 1u ? cnts[1] : lane == 2u ? cnts[2] : cnts[3];
        k = k2;
        continue;
      }
      u32 kd = 0, rb = 0, kb = 0;
      if (n) warp_pack(ev, g, s, n, q0, rc0, m0 + k, mIdx, mStart, &kd, &rb, &kb);
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

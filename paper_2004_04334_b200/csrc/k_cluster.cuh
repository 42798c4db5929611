// k_cluster.cuh — a3 + a4 + hits: per-module connected components, exact cluster sums, cluster threshold, EVENT-WIDE
// numbering, cluster table and hit table in ONE kernel (k_cluster; k_dense for launches full of large modules).
// Part of kernels.cuh (include that, not this file).
#pragma once
#include "common.cuh"

namespace pixreco {

// ================================================================== the unit of work
// A UNIT is a run of G consecutive modules of one event (G a power of two <= kMaxGroup chosen per launch so that a unit
// holds a few hundred digis; G = 1 in k_dense).  Units are handed out by an atomic ticket in (event, group) order, one
// CTA per unit, so every unit with a smaller ticket is running or done: a unit may wait for its predecessors.
//
// Fast path (a unit of at most kUnitCap digis), one THREAD per digi, everything in shared memory:
//   P1 insert    key = (module in unit, row, col) of every kept digi (A8) into an open-addressing hash table
//   P2 union     backward neighbours by the decision tree  N ? {N} : { NE?, W ? {W} : NW? }  (spans every 8-adjacency once
//                every digi did it); union-find with the LARGER root hooked under the smaller one (atomicMin), so a set's
//                root is its minimum digi index = the canonical label (A10).  Two digis on one pixel: the later ones only
//                follow the first of their probe chain (A6)
//   P3 flatten   root of every digi; roots numbered in ascending index order by ballots + a 64-entry prefix
//   P4 sums      per cluster, 14 u32 accumulators fed by NATIVE 32-bit shared-memory reductions: the exact fixed-point
//                sums of A9 (qf = q * 2^14; S, Sx = sum qf*row, Sy = sum qf*col) as three 15-bit limbs each (a 64-bit
//                shared-memory atomicAdd is a compare-and-swap loop on sm_100: 6x slower, measured), the size, and the
//                bounding box (A28) as four maxima
//   P5 finish    one thread per cluster: limbs -> int64, cluster threshold (A8/A9), centroid (binary64 divide, one
//                rounding, A9), hit position / flags / errors (A26-A30); kept clusters ranked by ballots
//   numbering    the unit publishes its kept-cluster count; its first cluster number is the sum of the counts of the
//                event's earlier units (read directly: at most 1856 of them; spin only on units still running)
//   emit         label[], clus[] with the FINAL event-wide number, cluster table, hit table, modClusStart — written once
// Units beyond the caps (more than kUnitCap digis, or more than kAccCap clusters) go module run by module run (or pass by
// pass) with their finished records STAGED in global memory and a fix-up after the numbering; a single module above
// kUnitCap digis takes the dense path (occupancy bitmap + popcount ranks + union-find, global workspace tiers).  No
// capacity limit except A9's own 2^17 digis per module (PR_STATUS_CAPACITY).
// The CTA that completes an event's last unit publishes the event's counters to mapped pinned host memory and puts the
// zeros back into the control block.
constexpr u32 kTabSlots = 4096;                       // hash slots (load <= 1/2); afterwards the cluster accumulators
constexpr u32 kAccCap = kTabSlots / kAccWords;        // clusters per accumulation pass (292)
constexpr u32 kNoKey = 0xFFFFFFFFu, kEmpty = 0xFFFFFFFFu, kNoRank = 0xFFFFFFFFu;
constexpr u32 kAggReady = 0x80000000u;
static_assert(kAccCap <= 320, "ordRoot / keptBal sizes");

struct UnitShared {
  u32 rootBal[64], chunkBase[64];     // per 32 digis: ballot of roots, number of roots before the chunk
  u32 keptBal[16];                    // per 32 clusters of a pass: ballot of kept clusters
  u16 ordRoot[320];                   // local digi index of the root of each cluster of the pass
  u32 modStart[kMaxGroup + 1], modKept[kMaxGroup + 1];
  u32 nKeptDigis, nRoots, dup, base, ticket, K, fin, nAllClusters;
  u32 scan[16];                       // block_excl_scan scratch (dense path)
};
__host__ __device__ inline size_t dense_smem_bytes(u32 bitmapWords, u32 capDigis, u32 capClusters) {
  size_t w = (bitmapWords + 3) & ~3u;
  return (size_t)w * 4 * 2 + (size_t)capDigis * 4 * 2 + (size_t)capClusters * (kAccWords * 4 + 8);
}
__host__ __device__ inline size_t cluster_smem_bytes(u32 bitmapWords) {
  size_t fast = (size_t)(kTabSlots + 2 * (kUnitCap + 1)) * 4, dense = dense_smem_bytes(bitmapWords, 0, 0);
  return ((dense > fast ? dense : fast) + 15) & ~(size_t)15;
}

// ------------------------------------------------------------------ union-find (local digi indices)
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

// ------------------------------------------------------------------ per-cluster accumulators and records
// Accumulator words (reductions):  0-2 S, 3-5 Sx, 6-8 Sy as limbs of 15, 15 and the remaining bits (every term is below
// 2^15 and a module has at most 2^17 - 1 digis: no limb sum overflows 32 bits); 9 size; 10 max(255 - row), 11 max(row),
// 12 max(511 - col), 13 max(col).  All start at zero.
template <typename P>
__device__ __forceinline__ void acc_add(P* a, u64 qf, u32 row, u32 col) {
  const u64 px = qf * row, py = qf * col;
  atomicAdd(a + 0, (u32)qf & 0x7FFFu); atomicAdd(a + 1, (u32)(qf >> 15) & 0x7FFFu); atomicAdd(a + 2, (u32)(qf >> 30));
  atomicAdd(a + 3, (u32)px & 0x7FFFu); atomicAdd(a + 4, (u32)(px >> 15) & 0x7FFFu); atomicAdd(a + 5, (u32)(px >> 30));
  atomicAdd(a + 6, (u32)py & 0x7FFFu); atomicAdd(a + 7, (u32)(py >> 15) & 0x7FFFu); atomicAdd(a + 8, (u32)(py >> 30));
  atomicAdd(a + 9, 1u);
  atomicMax(a + 10, 255u - row); atomicMax(a + 11, row); atomicMax(a + 12, 511u - col); atomicMax(a + 13, col);
}
// Record words (what acc_finish leaves in place of the accumulators of a KEPT cluster):
// 0 label, 1 size, 2 charge, 3 rowC, 4 colC, 5 x, 6 y, 7 xerr, 8 yerr (binary32 bits), 9 rows, 10 cols, 11 flags | module << 16,
// 12 rank among the kept clusters (set by the caller), 13 unused.
// Returns whether the cluster is kept (A8/A9: on the exact int64 sum).
__device__ __forceinline__ bool acc_finish(u32* a, const Geom& g, u32 label, u32 module) {
  const u64 S = (u64)a[0] + ((u64)a[1] << 15) + ((u64)a[2] << 30);
  if ((i64)S < g.clusThrFixed) return false;
  const u64 Sx = (u64)a[3] + ((u64)a[4] << 15) + ((u64)a[5] << 30);
  const u64 Sy = (u64)a[6] + ((u64)a[7] << 15) + ((u64)a[8] << 30);
  const u32 size = a[9], rmin = 255u - a[10], rmax = a[11], cmin = 511u - a[12], cmax = a[13];
  const double dS = __ll2double_rn((i64)S);
  const double rc = __ddiv_rn(__ll2double_rn((i64)Sx), dS), cc = __ddiv_rn(__ll2double_rn((i64)Sy), dS);   // A9
  // A27: divide, add 0.5, subtract half the module, multiply by the pitch — binary64, this order, then one cast
  const double x = __dmul_rn(__dsub_rn(__dadd_rn(rc, 0.5), 0.5 * (double)g.R), g.pitchRow);
  const double y = __dmul_rn(__dsub_rn(__dadd_rn(cc, 0.5), 0.5 * (double)g.C), g.pitchCol);
  const bool er = rmin == 0u || rmax == g.R - 1u, ec = cmin == 0u || cmax == g.C - 1u;                      // A29
  const u32 sr = rmax - rmin + 1u, sc = cmax - cmin + 1u;
  const double fr = er ? (double)sr : (sr == 1u ? 1.0 : 0.5), fc = ec ? (double)sc : (sc == 1u ? 1.0 : 0.5);   // A30
  const double xe = __dmul_rn(__dmul_rn(g.pitchRow, 0.28867513459481287), fr);
  const double ye = __dmul_rn(__dmul_rn(g.pitchCol, 0.28867513459481287), fc);
  a[0] = label; a[1] = size;
  a[2] = __float_as_uint(__double2float_rn(dS * (1.0 / 16384.0)));
  a[3] = __float_as_uint(__double2float_rn(rc)); a[4] = __float_as_uint(__double2float_rn(cc));
  a[5] = __float_as_uint(__double2float_rn(x)); a[6] = __float_as_uint(__double2float_rn(y));
  a[7] = __float_as_uint(__double2float_rn(xe)); a[8] = __float_as_uint(__double2float_rn(ye));
  a[9] = rmin | rmax << 16; a[10] = cmin | cmax << 16;
  a[11] = (er ? 1u : 0u) | (ec ? 2u : 0u) | module << 16;
  return true;
}
// Cluster `pos` of the event's cluster and hit tables from a finished record.
__device__ __forceinline__ void write_record(const EvDesc& ev, u32 pos, const u32* r) {
  if (pos >= ev.cap) return;
  ev.clLabel[pos] = r[0]; ev.clSize[pos] = r[1];
  ev.clCharge[pos] = __uint_as_float(r[2]); ev.clRow[pos] = __uint_as_float(r[3]); ev.clCol[pos] = __uint_as_float(r[4]);
  ev.htX[pos] = __uint_as_float(r[5]); ev.htY[pos] = __uint_as_float(r[6]);
  ev.htXerr[pos] = __uint_as_float(r[7]); ev.htYerr[pos] = __uint_as_float(r[8]);
  ev.htRows[pos] = r[9]; ev.htCols[pos] = r[10];
  const u32 fm = r[11];
  ev.clModule[pos] = (u16)(fm >> 16); ev.htFlags[pos] = (u16)(fm & 0xFFFFu);
}

// ------------------------------------------------------------------ fast path
__device__ __forceinline__ u32 h_slot(u32 key, u32 shift) { return (key * 0x9E3779B1u) >> shift; }
// Local index of the first digi on pixel `key` in probe order, kEmpty if none.
__device__ __forceinline__ u32 tab_find(const u32* tab, u32 pmask, u32 shift, u32 key) {
  u32 h = h_slot(key, shift);
  for (;;) {
    const u32 v = tab[h];
    if (v == kEmpty) return kEmpty;
    if ((v >> 11) == key) return v & 0x7FFu;
    h = (h + 1) & pmask;
  }
}

// Digis [s, s+n), 0 < n <= kUnitCap, of the modules from mRun on (at most kMaxGroup of them), clustered by the whole CTA.
// `direct`: the caller wants the finished records left in shared memory (tab) for an in-place emit; that works if all the
// clusters fit one accumulation pass.  Otherwise (or if the caller asks for it) the records are staged in global memory at
// (sUnit + kept rank within the unit) and clus[] gets the unit-relative rank.  Returns true if the records are in shared
// memory.  sh.K (kept clusters of the unit so far), sh.modKept, sh.nKeptDigis, sh.nAllClusters are advanced.
template <u32 kT>
__device__ __forceinline__ bool fast_cluster(const EvDesc& ev, const Geom& g, UnitShared& sh, u32* tab, u32* key, u32* par,
                                             u32 s, u32 n, u32 mRun, u32 mUnit, u32 sUnit, bool direct) {
  const u32 tid = threadIdx.x, lane = tid & 31u, lt = (1u << lane) - 1u;
  const u32 nPad = (n + 31u) & ~31u;
  const u32 lg = max(32u - (u32)__clz((int)(2u * n - 1u)), 6u);          // table size: a power of two >= 2n
  const u32 pmask = (1u << lg) - 1u, shift = 32u - lg;
  // P0
  for (u32 i = tid * 4u; i <= pmask; i += kT * 4u) *reinterpret_cast<uint4*>(tab + i) = make_uint4(kEmpty, kEmpty, kEmpty, kEmpty);
  if (tid == 0) sh.dup = 0u;
  __syncthreads();
  // P1: kept flag (A8), key, insert
  {
    u32 myKept = 0;
    for (u32 i = tid; i < nPad; i += kT) {
      u32 k = kNoKey;
      if (i < n) {
        const float q = ev.charge[s + i];
        if (q >= g.pixThr) k = ((u32)ev.module[s + i] - mRun) << 17 | (u32)ev.row[s + i] << 9 | (u32)ev.col[s + i];
      }
      key[i] = k; par[i] = i;
      if (k != kNoKey) {
        const u32 ent = k << 11 | i;
        u32 h = h_slot(k, shift);
        for (;;) {
          const u32 old = atomicCAS(tab + h, kEmpty, ent);
          if (old == kEmpty) break;
          if ((old >> 11) == k) sh.dup = 1u;
          h = (h + 1) & pmask;
        }
      }
      myKept += (u32)__popc(__ballot_sync(0xFFFFFFFFu, k != kNoKey));
    }
    if (lane == 0 && myKept) atomicAdd(&sh.nKeptDigis, myKept);
  }
  __syncthreads();
  // P2: unions with the backward neighbours
  {
    const bool dup = sh.dup != 0u;
    for (u32 i = tid; i < n; i += kT) {
      const u32 k = key[i];
      if (k == kNoKey) continue;
      if (dup) {
        const u32 o = tab_find(tab, pmask, shift, k);
        if (o != i) { uf_union(par, i, o); continue; }
      }
      const u32 row = (k >> 9) & 0xFFu, col = k & 0x1FFu;
      const bool up = row > 0u, left = col > 0u, right = col + 1u < g.C;
      u32 j = up ? tab_find(tab, pmask, shift, k - 512u) : kEmpty;
      if (j != kEmpty) uf_union(par, i, j);
      else {
        if (up && right) { j = tab_find(tab, pmask, shift, k - 511u); if (j != kEmpty) uf_union(par, i, j); }
        j = left ? tab_find(tab, pmask, shift, k - 1u) : kEmpty;
        if (j != kEmpty) uf_union(par, i, j);
        else if (up && left) { j = tab_find(tab, pmask, shift, k - 513u); if (j != kEmpty) uf_union(par, i, j); }
      }
    }
  }
  __syncthreads();
  // P3: flatten; ballots of roots; the table becomes the accumulators
  for (u32 i = tid * 4u; i < kTabSlots; i += kT * 4u) *reinterpret_cast<uint4*>(tab + i) = make_uint4(0u, 0u, 0u, 0u);
  for (u32 i = tid; i < nPad; i += kT) {
    bool isRoot = false;
    if (key[i] != kNoKey) {
      const u32 r = uf_root(par, i);
      isRoot = r == i;
      if (!isRoot) par[i] = r;
    }
    const u32 b = __ballot_sync(0xFFFFFFFFu, isRoot);
    if (lane == 0) sh.rootBal[i >> 5] = b;
  }
  __syncthreads();
  if (tid < 32u) {
    const u32 nCh = nPad >> 5;
    const u32 c0 = 2u * lane < nCh ? (u32)__popc(sh.rootBal[2u * lane]) : 0u, c1 = 2u * lane + 1u < nCh ? (u32)__popc(sh.rootBal[2u * lane + 1u]) : 0u;
    const u32 incl = warp_incl_scan(c0 + c1, lane);
    sh.chunkBase[2u * lane] = incl - c0 - c1; sh.chunkBase[2u * lane + 1u] = incl - c1;
    if (lane == 31u) sh.nRoots = incl;
  }
  __syncthreads();
  const u32 nR = sh.nRoots;
  const bool inSmem = direct && nR <= kAccCap;
  // every root notes its ordinal (ascending index = ascending label order) in the free bits of its key
  for (u32 i = tid; i < n; i += kT)
    if (key[i] != kNoKey && par[i] == i) key[i] |= (sh.chunkBase[i >> 5] + (u32)__popc(sh.rootBal[i >> 5] & lt)) << 21;
  u32 Kb = sh.K;                                                          // kept clusters of the unit before this pass
  for (u32 p0 = 0; p0 == 0u || p0 < nR; p0 += kAccCap) {
    const u32 nAcc = min(nR - p0, kAccCap), nAccPad = (nAcc + 31u) & ~31u;
    if (p0) {
      __syncthreads();
      for (u32 i = tid * 4u; i < kTabSlots; i += kT * 4u) *reinterpret_cast<uint4*>(tab + i) = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();                                                      // ordinals (and zeros) visible
    // P4: sums
    for (u32 i = tid; i < n; i += kT) {
      const u32 k = key[i];
      if (k == kNoKey) continue;
      const u32 r = par[i], o = (key[r] >> 21) - p0;
      if (o >= nAcc) continue;
      if (r == i) sh.ordRoot[o] = (u16)i;
      const u64 qf = (u64)__float2ll_rz(ev.charge[s + i] * 16384.0f);    // A9: exact, q is a multiple of 2^-14
      acc_add(tab + o * kAccWords, qf, (k >> 9) & 0xFFu, k & 0x1FFu);
    }
    __syncthreads();
    // P5: finish, one thread per cluster; ballots of the kept ones
    for (u32 o = tid; o < nAccPad; o += kT) {
      bool kept = false;
      if (o < nAcc) {
        const u32 r = sh.ordRoot[o];
        kept = acc_finish(tab + o * kAccWords, g, s + r, mRun + ((key[r] >> 17) & 15u));
      }
      const u32 b = __ballot_sync(0xFFFFFFFFu, kept);
      if (lane == 0) sh.keptBal[o >> 5] = b;
    }
    __syncthreads();
    u32 passKept = 0;
    for (u32 c = 0; c < (nAccPad >> 5); ++c) passKept += (u32)__popc(sh.keptBal[c]);
    for (u32 o = tid; o < nAcc; o += kT) {
      const u32 b = sh.keptBal[o >> 5];
      u32 kr = kNoRank;
      if (b >> lane & 1u) {
        kr = Kb + (u32)__popc(b & lt);
        for (u32 c = 0; c < (o >> 5); ++c) kr += (u32)__popc(sh.keptBal[c]);
        atomicAdd(&sh.modKept[(tab[o * kAccWords + 11u] >> 16) - mUnit], 1u);
        if (!inSmem) {                                                    // stage the finished record
          u32* dst = ev.stage + (size_t)(sUnit + kr) * kAccWords;
#pragma unroll
          for (u32 w = 0; w < 12u; ++w) dst[w] = tab[o * kAccWords + w];
        }
      }
      tab[o * kAccWords + 12u] = kr;
    }
    if (!inSmem) {
      __syncthreads();
      for (u32 i = tid; i < n; i += kT) {
        const u32 k = key[i];
        if (k == kNoKey) { if (p0 == 0u) { ev.label[s + i] = kInvalid; ev.clus[s + i] = -1; } continue; }
        const u32 r = par[i], o = (key[r] >> 21) - p0;
        if (o >= nAcc) continue;
        const u32 kr = tab[o * kAccWords + 12u];
        ev.label[s + i] = s + r; ev.clus[s + i] = kr == kNoRank ? -1 : (int32_t)kr;
      }
    }
    Kb += passKept;
  }
  __syncthreads();
  if (tid == 0) { sh.K = Kb; sh.nAllClusters += nR; }
  __syncthreads();
  return inSmem;
}

// ------------------------------------------------------------------ dense path: one module = digis [s, s+nn), whole CTA
// Occupancy bitmap + popcount-prefix ranks for the neighbour look-up, union-find over the digis, per-cluster
// accumulators; shared-memory tiers of capDigis digis / capClusters clusters, the global workspace beyond.
// Leaves in cx: parent[] (root of every kept digi, kInvalid otherwise), perm[root] = cluster ordinal, acc (finished
// records of the kept clusters), knum[ordinal] = rank among the module's kept clusters or -1, root[ordinal].
struct DenseCtx {
  u32 *perm, *parent, *root, *acc; int32_t* knum;
  u32 nAll, nKept, nKeptDigis;
};

template <u32 kT>
__device__ __forceinline__ void dense_count(const EvDesc& ev, const Geom& g, u32 m, u32 s, u32 nn, unsigned char* smemRaw, u32* sScan,
                                            DenseCtx& cx, u32 capDigis, u32 capClusters) {
  const u32 tid = threadIdx.x, lane = tid & 31u;
  const u32 bwPad = (g.bitmapWords + 3) & ~3u;
  u32* smAcc = reinterpret_cast<u32*>(smemRaw);
  u32* smRoot = smAcc + capClusters * kAccWords;
  int32_t* smKnum = reinterpret_cast<int32_t*>(smRoot + capClusters);
  u32* smBitmap = reinterpret_cast<u32*>(smKnum + capClusters);
  u32* smPrefix = smBitmap + bwPad;
  u32* smPerm = smPrefix + bwPad;
  u32* smParent = smPerm + capDigis;
  const u32 stride = g.stride;

  const bool digiInSmem = nn <= capDigis;
  u32* perm = digiInSmem ? smPerm : ev.wsPerm + s;
  u32* parent = digiInSmem ? smParent : ev.wsParent + s;
  cx.perm = perm; cx.parent = parent;
  cx.root = smRoot; cx.knum = smKnum; cx.acc = smAcc;

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
  __syncthreads();
  // P2: exclusive popcount prefix per bitmap word (contiguous chunk per thread); kept digis of the module
  {
    const u32 per = (g.bitmapWords + kT - 1) / kT;
    const u32 lo = min(tid * per, g.bitmapWords), hi = min(lo + per, g.bitmapWords);
    u32 sum = 0;
    for (u32 i = lo; i < hi; ++i) sum += __popc(smBitmap[i]);
    u32 tot;
    u32 run = block_excl_scan<kT / 32>(sum, sScan, &tot);
    for (u32 i = lo; i < hi; ++i) { smPrefix[i] = run; run += __popc(smBitmap[i]); }
    u32 totK;
    block_excl_scan<kT / 32>(myKept, sScan, &totK);
    cx.nKeptDigis = totK;
  }
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
    if (cx.nAll > capClusters) { cx.root = ev.wsRoot + s; cx.knum = ev.wsKnum + s; cx.acc = ev.wsAcc + (size_t)s * kAccWords; }
    for (u32 i = lo; i < hi; ++i)
      if (parent[i] == i) { perm[i] = run; cx.root[run] = i; ++run; }
  }
  // P7: zero the accumulators
  for (u32 c = tid; c < cx.nAll * kAccWords; c += kT) cx.acc[c] = 0u;
  __syncthreads();
  // P8: exact fixed-point sums (A9), size and bounding box by 32-bit reductions
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = parent[i];
    if (p == kInvalid) continue;
    const u64 qf = (u64)__float2ll_rz(ev.charge[s + i] * 16384.0f);
    acc_add(cx.acc + (size_t)perm[p] * kAccWords, qf, ev.row[s + i], ev.col[s + i]);
  }
  __syncthreads();
  // P9: finish every cluster (threshold A8/A9, centroid, hit) and number the kept ones within the module
  {
    const u32 per = (cx.nAll + kT - 1) / kT;
    const u32 lo = min(tid * per, cx.nAll), hi = min(lo + per, cx.nAll);
    u32 c = 0;
    for (u32 k = lo; k < hi; ++k) {
      const bool kept = acc_finish(cx.acc + (size_t)k * kAccWords, g, s + cx.root[k], m);
      cx.knum[k] = kept ? 0 : -1;
      c += kept;
    }
    u32 run = block_excl_scan<kT / 32>(c, sScan, &cx.nKept);
    for (u32 k = lo; k < hi; ++k) if (cx.knum[k] == 0) cx.knum[k] = (int32_t)run++;
  }
  __syncthreads();
}

// label[], clus[] = clusOff + rank within the module, and the records of the kept clusters at index recOff + rank of
// the event's tables, or of the staging area if `staged`.
template <u32 kT>
__device__ __forceinline__ void dense_emit(const EvDesc& ev, u32 s, u32 nn, const DenseCtx& cx, u32 recOff, u32 clusOff, bool staged) {
  const u32 tid = threadIdx.x;
  for (u32 k = tid; k < cx.nAll; k += kT) {
    const int32_t kn = cx.knum[k];
    if (kn < 0) continue;
    const u32* rec = cx.acc + (size_t)k * kAccWords;
    if (staged) {
      u32* dst = ev.stage + (size_t)(recOff + (u32)kn) * kAccWords;
#pragma unroll
      for (u32 w = 0; w < 12u; ++w) dst[w] = rec[w];
    } else write_record(ev, recOff + (u32)kn, rec);
  }
  for (u32 i = tid; i < nn; i += kT) {
    const u32 p = cx.parent[i];
    u32 lab = kInvalid; int32_t cl = -1;
    if (p != kInvalid) {
      lab = s + p;
      const int32_t kn = cx.knum[cx.perm[p]];
      if (kn >= 0) cl = (int32_t)(clusOff + (u32)kn);
    }
    ev.label[s + i] = lab;
    ev.clus[s + i] = cl;
  }
}

// ------------------------------------------------------------------ numbering across the units of an event, completion
// Publish this unit's kept-cluster count and return (in all threads) the sum over the event's earlier units.  Those hold
// smaller tickets, so they are running or done: the spin ends.
template <u32 kT>
__device__ __forceinline__ u32 publish_and_look_back(u32* agg, u32 grp, u32 K, u32* shBase) {
  const u32 tid = threadIdx.x, lane = tid & 31u;
  if (tid == 0) asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(agg + grp), "r"(K | kAggReady) : "memory");
  if (tid < 32u) {
    u32 sum = 0;
    for (u32 j = lane; j < grp; j += 32u) {
      u32 v;
      for (;;) {
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(agg + j) : "memory");
        if (v & kAggReady) break;
        __nanosleep(40);
      }
      sum += v & ~kAggReady;
    }
    sum = __reduce_add_sync(0xFFFFFFFFu, sum);
    if (lane == 0) *shBase = sum;
  }
  __syncthreads();
  return *shBase;
}

// After the unit's last store: count it; the CTA that completes the event's last unit publishes the counters to the
// host (mapped pinned memory) and puts the zeros back into the event's part of the control block.
template <u32 kT>
__device__ __forceinline__ void unit_complete(const EvDesc& ev, const LaunchCtl* lc, u32 nGroups, u32* shFin) {
  const u32 tid = threadIdx.x;
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    *shFin = atomicAdd(&ev.counters->unitsDone, 1u) == nGroups - 1u ? 1u : 0u;
  }
  __syncthreads();
  if (*shFin) {
    __threadfence();
    for (u32 j = tid; j < nGroups; j += kT) ev.grpAgg[j] = 0u;
    if (tid == 0) {
      volatile DevCounters* c = ev.counters;
      const u32 status = c->status;
      HostCounters h;
      h.nWords = c->nWords; h.nDigis = c->nDigis; h.nErrors = c->nErrors; h.nKept = c->nKept;
      h.nClustersAll = c->nClustersAll; h.nClusters = (status & 1u) ? 0u : c->nClusters; h.status = status; h.seq = 1;
      h.tStart = *reinterpret_cast<const volatile u64*>(&lc->tStart); h.tEnd = global_timer();
      *ev.hostCounters = h;
      DevCounters r;
      r.nWords = h.nWords; r.nDigis = h.nDigis; r.nErrors = h.nErrors; r.nKept = h.nKept; r.nClustersAll = h.nClustersAll;
      r.nClusters = h.nClusters; r.status = status; r.unitsDone = nGroups;
      *ev.result = r;
      c->nWords = 0; c->nDigis = 0; c->nErrors = 0; c->nKept = 0; c->nClustersAll = 0; c->nClusters = 0; c->status = 0; c->unitsDone = 0;
    }
  }
}
// A CTA leaves the kernel: the last one puts the ticket words back to zero.
__device__ __forceinline__ void cta_exit(u32* ticket, u32* exited) {
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(exited, 1u) == gridDim.x - 1u) { *ticket = 0u; __threadfence(); *exited = 0u; }
  }
}
// modClusStart of the unit's modules; the event's last unit closes the table and the cluster counter.
template <u32 kT>
__device__ __forceinline__ void write_mod_clus_start(const EvDesc& ev, const UnitShared& sh, u32 m0, u32 nm, u32 M, u32 base, bool ok) {
  const u32 tid = threadIdx.x;
  if (tid < nm) {
    u32 b = base;
    for (u32 j = 0; j < tid; ++j) b += sh.modKept[j];
    ev.modClusStart[m0 + tid] = b;
  }
  if (tid == 0 && m0 + nm == M) {
    u32 b = base;
    for (u32 j = 0; j < nm; ++j) b += sh.modKept[j];
    ev.modClusStart[M] = b;
    if (ok) ev.counters->nClusters = b;
  }
}

// ================================================================== k_cluster
template <bool kSingle>
__global__ void __launch_bounds__(kClusterThreads, 5)
k_cluster(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv, LaunchCtl* __restrict__ lc,
          u32 G, u32 nGroups, const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ UnitShared sh;
  constexpr u32 kT = kClusterThreads;
  u32* tab = reinterpret_cast<u32*>(smemRaw);
  u32* key = tab + kTabSlots;
  u32* par = key + kUnitCap + 1u;
  const u32 tid = threadIdx.x, M = g.M, total = nEv * nGroups;

  for (;;) {
    __syncthreads();
    if (tid == 0) {
      sh.ticket = atomicAdd(&lc->unitTicket, 1u);
      sh.nKeptDigis = 0u; sh.K = 0u; sh.nAllClusters = 0u;
    }
    if (tid <= kMaxGroup) sh.modKept[tid] = 0u;
    __syncthreads();
    const u32 t = sh.ticket;
    if (t >= total) break;
    const u32 e = t / nGroups, grp = t - e * nGroups;
    const EvDesc& ev = kSingle ? single : batch[e];
    const u32 m0 = grp * G, nm = min(G, M - m0);
    const bool ok = !(__ldcg(&ev.counters->status) & 1u);      // A5 violated: modDigiStart is undefined, no per-digi work
    if (ok && tid <= nm) sh.modStart[tid] = ev.modDigiStart[m0 + tid];
    __syncthreads();
    u32 s0 = 0, n = 0;
    bool sane = ok;
    if (ok) {
      s0 = sh.modStart[0];
      const u32 s1 = sh.modStart[nm];
      sane = s0 <= s1 && s1 <= ev.cap;
      for (u32 j = 0; j < nm; ++j) sane = sane && sh.modStart[j] <= sh.modStart[j + 1];
      n = sane ? s1 - s0 : 0u;
      if (!sane && tid == 0) atomicOr(&ev.counters->status, 2u);   // inconsistent module table: PR_STATUS_CAPACITY
    }
    bool inSmem = false;
    if (n && n <= kUnitCap) {
      inSmem = fast_cluster<kT>(ev, g, sh, tab, key, par, s0, n, m0, m0, s0, true);
    } else if (n) {
      // a unit above the cap: maximal runs of whole modules with at most kUnitCap digis, a larger module alone (dense path)
      u32 mi = 0;
      while (mi < nm) {
        const u32 a = sh.modStart[mi];
        u32 mj = mi + 1u;
        while (mj < nm && sh.modStart[mj + 1u] - a <= kUnitCap) ++mj;
        const u32 cnt = sh.modStart[mj] - a;
        if (cnt > kMaxModuleDigis) {
          if (tid == 0) atomicOr(&ev.counters->status, 2u);        // A9's own limit: PR_STATUS_CAPACITY, the module stays unclustered
        } else if (cnt > kUnitCap) {
          DenseCtx cx;
          dense_count<kT>(ev, g, m0 + mi, a, cnt, smemRaw, sh.scan, cx, 0u, 0u);
          dense_emit<kT>(ev, a, cnt, cx, s0 + sh.K, sh.K, true);   // staged: unit-relative ranks, fixed up after the numbering
          __syncthreads();
          if (tid == 0) { sh.modKept[mi] = cx.nKept; sh.K += cx.nKept; sh.nKeptDigis += cx.nKeptDigis; sh.nAllClusters += cx.nAll; }
          __syncthreads();
        } else if (cnt) {
          fast_cluster<kT>(ev, g, sh, tab, key, par, a, cnt, m0 + mi, m0, s0, false);
        }
        mi = mj;
      }
    }
    // ---- numbering: this unit's first cluster number
    const u32 K = sh.K;
    if (tid == 0) {
      if (sh.nKeptDigis) atomicAdd(&ev.counters->nKept, sh.nKeptDigis);
      if (sh.nAllClusters) atomicAdd(&ev.counters->nClustersAll, sh.nAllClusters);
    }
    if (inSmem) {                                               // label[] does not depend on the numbering: before the wait
      for (u32 i = tid; i < n; i += kT) ev.label[s0 + i] = key[i] != kNoKey ? s0 + par[i] : kInvalid;
    }
    const u32 base = publish_and_look_back<kT>(ev.grpAgg, grp, K, &sh.base);
    if (inSmem) {
      for (u32 i = tid; i < n; i += kT) {
        int32_t cl = -1;
        if (key[i] != kNoKey) {
          const u32 kr = tab[(key[par[i]] >> 21) * kAccWords + 12u];
          if (kr != kNoRank) cl = (int32_t)(base + kr);
        }
        ev.clus[s0 + i] = cl;
      }
      const u32 nR = sh.nRoots;
      for (u32 o = tid; o < nR; o += kT) {
        const u32* rec = tab + o * kAccWords;
        if (rec[12] != kNoRank) write_record(ev, base + rec[12], rec);
      }
    } else if (n) {                                             // staged: fix up clus[], move the records
      for (u32 i = tid; i < n; i += kT) { const int32_t c = ev.clus[s0 + i]; if (c >= 0) ev.clus[s0 + i] = c + (int32_t)base; }
      for (u32 k = tid; k < K; k += kT) write_record(ev, base + k, ev.stage + (size_t)(s0 + k) * kAccWords);
    }
    if (ok) write_mod_clus_start<kT>(ev, sh, m0, nm, M, base, ok);
    unit_complete<kT>(ev, lc, nGroups, &sh.fin);
  }
  cta_exit(&lc->unitTicket, &lc->clusterExited);
}

// ================================================================== k_dense (launches full of large modules)
// One module per unit, the dense path with its own, larger shared-memory tiers (kDenseDigis digis / kDenseClusters
// clusters per module, two CTAs of 512 threads per SM), same numbering and completion (BASELINE.json configs[4]).
constexpr u32 kDenseThreads = 512;
template <bool kSingle>
__global__ void __launch_bounds__(kDenseThreads, 2)
k_dense(const __grid_constant__ EvDesc single, const EvDesc* __restrict__ batch, u32 nEv, LaunchCtl* __restrict__ lc,
        const __grid_constant__ Geom g) {
  extern __shared__ __align__(16) unsigned char smemRaw[];
  __shared__ UnitShared sh;
  constexpr u32 kT = kDenseThreads;
  const u32 tid = threadIdx.x, M = g.M, total = nEv * M;
  for (;;) {
    __syncthreads();
    if (tid == 0) sh.ticket = atomicAdd(&lc->unitTicket, 1u);
    __syncthreads();
    const u32 t = sh.ticket;
    if (t >= total) break;
    const u32 e = t / M, m = t - e * M;
    const EvDesc& ev = kSingle ? single : batch[e];
    const bool ok = !(__ldcg(&ev.counters->status) & 1u);
    u32 s = 0, nn = 0;
    if (ok) {
      s = ev.modDigiStart[m];
      const u32 s1 = ev.modDigiStart[m + 1];
      if (s <= s1 && s1 <= ev.cap && s1 - s <= kMaxModuleDigis) nn = s1 - s;
      else if (tid == 0) atomicOr(&ev.counters->status, 2u);
    }
    DenseCtx cx;
    cx.nAll = 0; cx.nKept = 0; cx.nKeptDigis = 0;
    if (nn) dense_count<kT>(ev, g, m, s, nn, smemRaw, sh.scan, cx, kDenseDigis, kDenseClusters);
    if (tid == 0) {
      if (cx.nKeptDigis) atomicAdd(&ev.counters->nKept, cx.nKeptDigis);
      if (cx.nAll) atomicAdd(&ev.counters->nClustersAll, cx.nAll);
      sh.modKept[0] = cx.nKept;
    }
    const u32 base = publish_and_look_back<kT>(ev.grpAgg, m, cx.nKept, &sh.base);
    if (nn) dense_emit<kT>(ev, s, nn, cx, base, base, false);
    if (ok) write_mod_clus_start<kT>(ev, sh, m, 1u, M, base, ok);
    unit_complete<kT>(ev, lc, M, &sh.fin);
  }
  cta_exit(&lc->unitTicket, &lc->clusterExited);
}

}  // namespace pixreco

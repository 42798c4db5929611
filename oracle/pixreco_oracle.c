/* pixreco_oracle.c — THE ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, single-threaded CPU implementation of what the hot path computes:
 * raw-word decode with stable digi/error compaction -> per-module ADC-to-charge calibration with
 * pixel threshold -> per-module 8-connected connected components with canonical label = minimum
 * digi index -> exact cluster charge sums, charge-weighted centroids, cluster threshold and dense
 * numbering -> hits (bounding box, local position, error estimate) of the kept clusters.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call anything in oracle/.  It shares no code, header, table or helper with the
 * CUDA path (paper_2004_04334_b200/csrc) and neither includes the other.
 *
 * What defines the computation: the paper describes only the offload boundary and
 * defers the offloaded application to its ref. [8] (section 5), so every step below
 * follows BASELINE.json `north_star` subsystems (2)-(3) and `configs[0]` (word format, calibration,
 * thresholds) under the readings A1-A14 listed in DESIGN.md (= SURVEY.md section 8(c)).  Each
 * function cites the reading it implements.  Each step is the plain definition written out:
 * no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py, `-m "not gpu"`): hand-computed word encodings, exhaustive codec
 * round trip, closed-form calibration values and the float64 single-rounding identity, exhaustive
 * 4x4 occupancy patterns against an O(n^2) transitive closure, scipy.ndimage.label /
 * sum_labels / center_of_mass, networkx components for duplicate pixels, special shapes,
 * permutation invariance, worked reduce example; for the bucket step: a worked example, numpy's stable argsort,
 * identity on grouped input; for hits: worked values, closed forms (single
 * pixel, strips, centred and translated clusters), numpy min/max and scipy.ndimage.center_of_mass.  Against the PAPER there is nothing to pin:
 * it prints no value for this path ("parity unpinned" with respect to the paper).
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fPIC -shared pixreco_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PO_INVALID 0xFFFFFFFFu

/* ---- O1 decode (BASELINE.json configs[0] word format; readings A1-A5, A20) ----
 * For i ascending: bit31 set, or module >= M, or row >= R, or col >= C  -> error list (word, i);
 * else digi (module,row,col,adc[i],i).  Both lists keep the original order (A4).
 * mod_digi_start[m] = number of digis with module < m, m = 0..M (defined for any order).
 * *sorted_ok = 1 iff the digis' module sequence is non-decreasing (A5).                          */
void po_decode(const uint32_t *words, const uint16_t *adc, uint32_t W,
               uint32_t M, uint32_t R, uint32_t C,
               uint16_t *d_module, uint16_t *d_row, uint16_t *d_col, uint16_t *d_adc, uint32_t *d_word_idx,
               uint32_t *e_word, uint32_t *e_idx,
               uint32_t *mod_digi_start /* [M+1] */,
               uint32_t *n_digis, uint32_t *n_errors, uint32_t *sorted_ok) {
  uint32_t D = 0, E = 0, ok = 1;
  for (uint32_t m = 0; m <= M; ++m) mod_digi_start[m] = 0;
  for (uint32_t i = 0; i < W; ++i) {
    uint32_t w = words[i];
    uint32_t err = w >> 31, mod = (w >> 20) & 0x7FFu, row = (w >> 12) & 0xFFu, col = (w >> 3) & 0x1FFu;
    if (err || mod >= M || row >= R || col >= C) {
      e_word[E] = w; e_idx[E] = i; ++E;
    } else {
      if (D > 0 && mod < d_module[D - 1]) ok = 0;
      d_module[D] = (uint16_t)mod; d_row[D] = (uint16_t)row; d_col[D] = (uint16_t)col;
      d_adc[D] = adc[i]; d_word_idx[D] = i; ++D;
      mod_digi_start[mod + 1] += 1;           /* histogram, turned into "count below m" next */
    }
  }
  for (uint32_t m = 0; m < M; ++m) mod_digi_start[m + 1] += mod_digi_start[m];
  *n_digis = D; *n_errors = E; *sorted_ok = ok;
}

/* ---- O2 calibrate (A7, A8): q = fmaf((float)adc, gain[module], ped[module]), one binary32
 * rounding; kept = q >= pixThr.                                                                 */
void po_calibrate(uint32_t D, const uint16_t *d_adc, const uint16_t *d_module,
                  const float *gain, const float *ped, float pix_thr,
                  float *charge, uint8_t *kept, uint32_t *n_kept) {
  uint32_t k = 0;
  for (uint32_t d = 0; d < D; ++d) {
    float q = fmaf((float)d_adc[d], gain[d_module[d]], ped[d_module[d]]);
    charge[d] = q;
    kept[d] = (q >= pix_thr) ? 1 : 0;
    k += kept[d];
  }
  *n_kept = k;
}

/* ---- O3 cluster (A6, A10, A11; BASELINE.json north_star "8-connected ... canonical label =
 * minimum digi index").  Per module, over kept digis: a,b adjacent <=> |drow|<=1 and |dcol|<=1
 * (a != b; equal coordinates count, A6); label = minimum digi index of the component;
 * not-kept digis get PO_INVALID and do not bridge (A11).
 * Implementation (i): dense R x C grid holding the head of a chain of digi indices per cell
 * (chains only matter for duplicate pixels); digis of a module visited in ascending index; an
 * unlabelled kept digi starts a breadth-first search over the 3x3 neighbourhood, and everything
 * reached gets the start index, which is the component minimum by construction.
 * Order-agnostic: modules need not be grouped in the input.                                      */
int po_cluster(uint32_t D, uint32_t M, uint32_t R, uint32_t C,
               const uint16_t *d_module, const uint16_t *d_row, const uint16_t *d_col,
               const uint8_t *kept, uint32_t *label) {
  uint32_t *grid = (uint32_t *)malloc((size_t)R * C * sizeof(uint32_t));  /* head digi per cell   */
  uint32_t *next = (uint32_t *)malloc((size_t)(D ? D : 1) * sizeof(uint32_t)); /* chain in a cell */
  uint32_t *order = (uint32_t *)malloc((size_t)(D ? D : 1) * sizeof(uint32_t)); /* digis by module */
  uint32_t *start = (uint32_t *)calloc((size_t)M + 2, sizeof(uint32_t));
  uint32_t *queue = (uint32_t *)malloc((size_t)(D ? D : 1) * sizeof(uint32_t));
  if (!grid || !next || !order || !start || !queue) { free(grid); free(next); free(order); free(start); free(queue); return -1; }
  for (size_t c = 0; c < (size_t)R * C; ++c) grid[c] = PO_INVALID;
  /* stable bucket of digi indices by module (ascending index inside each module) */
  for (uint32_t d = 0; d < D; ++d) start[d_module[d] + 2] += 1;
  for (uint32_t m = 0; m < M; ++m) start[m + 2] += start[m + 1];
  for (uint32_t d = 0; d < D; ++d) order[start[d_module[d] + 1]++] = d;   /* start[m+1] ends as end of m */
  for (uint32_t d = 0; d < D; ++d) label[d] = PO_INVALID;

  for (uint32_t m = 0; m < M; ++m) {
    uint32_t lo = start[m], hi = start[m + 1];
    /* fill the grid; insert in DESCENDING index so each chain reads in ascending index */
    for (uint32_t k = hi; k-- > lo;) {
      uint32_t d = order[k];
      if (!kept[d]) continue;
      size_t cell = (size_t)d_row[d] * C + d_col[d];
      next[d] = grid[cell]; grid[cell] = d;
    }
    for (uint32_t k = lo; k < hi; ++k) {
      uint32_t s = order[k];
      if (!kept[s] || label[s] != PO_INVALID) continue;
      uint32_t qh = 0, qt = 0;
      label[s] = s; queue[qt++] = s;
      while (qh < qt) {
        uint32_t a = queue[qh++];
        int ar = d_row[a], ac = d_col[a];
        for (int dr = -1; dr <= 1; ++dr)
          for (int dc = -1; dc <= 1; ++dc) {
            int rr = ar + dr, cc = ac + dc;
            if (rr < 0 || cc < 0 || rr >= (int)R || cc >= (int)C) continue;   /* no wrap-around */
            for (uint32_t b = grid[(size_t)rr * C + cc]; b != PO_INVALID; b = next[b])
              if (label[b] == PO_INVALID) { label[b] = s; queue[qt++] = b; }
          }
      }
    }
    for (uint32_t k = lo; k < hi; ++k) {           /* clear only the cells this module touched */
      uint32_t d = order[k];
      if (kept[d]) grid[(size_t)d_row[d] * C + d_col[d]] = PO_INVALID;
    }
  }
  free(grid); free(next); free(order); free(start); free(queue);
  return 0;
}

/* ---- O4 reduce (A9, A12, A13).  For each distinct label L (ascending):
 *   qf[d] = (int64)(q[d] * 2^14)   exact: every kept q >= pixThr >= 512 is a multiple of 2^-14
 *   size = |members|, S = sum qf, Sx = sum qf*row, Sy = sum qf*col          (int64, order-free)
 *   kept cluster <=> S >= llrint(clusThr * 2^14)
 * kept clusters numbered k = 0..N-1 in ascending L:
 *   label=L, module=module[L], size, charge=(float)((double)S / 2^14),
 *   rowC=(float)((double)Sx/(double)S), colC=(float)((double)Sy/(double)S)   (binary64 ops, RN)
 * clus[d] = k or -1;  mod_clus_start[m] = number of kept clusters with module < m.
 * Returns 0, or -2 if some kept q*2^14 is not integral (contract pixThr >= 512 violated).        */
int po_reduce(uint32_t D, uint32_t M,
              const uint32_t *label, const float *charge,
              const uint16_t *d_module, const uint16_t *d_row, const uint16_t *d_col,
              float clus_thr,
              uint32_t *cl_label, uint16_t *cl_module, uint32_t *cl_size,
              float *cl_charge, float *cl_row, float *cl_col,
              int32_t *clus, uint32_t *mod_clus_start /* [M+1] */,
              uint32_t *n_clusters_all, uint32_t *n_clusters) {
  uint32_t *ord = (uint32_t *)malloc((size_t)(D ? D : 1) * sizeof(uint32_t));
  uint32_t nall = 0;
  for (uint32_t d = 0; d < D; ++d)               /* distinct labels in ascending order */
    if (label[d] == d) ord[d] = nall++;
  int64_t *S = (int64_t *)calloc((size_t)(nall ? nall : 1), sizeof(int64_t));
  int64_t *Sx = (int64_t *)calloc((size_t)(nall ? nall : 1), sizeof(int64_t));
  int64_t *Sy = (int64_t *)calloc((size_t)(nall ? nall : 1), sizeof(int64_t));
  uint32_t *sz = (uint32_t *)calloc((size_t)(nall ? nall : 1), sizeof(uint32_t));
  int32_t *knum = (int32_t *)malloc((size_t)(nall ? nall : 1) * sizeof(int32_t));
  int rc = 0;
  for (uint32_t d = 0; d < D; ++d) {
    if (label[d] == PO_INVALID) continue;
    float scaled = charge[d] * 16384.0f;          /* power-of-two scale: exact */
    int64_t qf = (int64_t)scaled;
    if ((float)qf != scaled) rc = -2;
    uint32_t c = ord[label[d]];
    sz[c] += 1; S[c] += qf; Sx[c] += qf * (int64_t)d_row[d]; Sy[c] += qf * (int64_t)d_col[d];
  }
  const int64_t thr = (int64_t)llrint((double)clus_thr * 16384.0);
  for (uint32_t m = 0; m <= M; ++m) mod_clus_start[m] = 0;
  uint32_t N = 0;
  for (uint32_t d = 0; d < D; ++d) {
    if (label[d] != d) continue;
    uint32_t c = ord[d];
    if (S[c] >= thr) {
      cl_label[N] = d; cl_module[N] = d_module[d]; cl_size[N] = sz[c];
      cl_charge[N] = (float)((double)S[c] / 16384.0);
      cl_row[N] = (float)((double)Sx[c] / (double)S[c]);
      cl_col[N] = (float)((double)Sy[c] / (double)S[c]);
      mod_clus_start[d_module[d] + 1] += 1;
      knum[c] = (int32_t)N++;
    } else knum[c] = -1;
  }
  for (uint32_t m = 0; m < M; ++m) mod_clus_start[m + 1] += mod_clus_start[m];
  for (uint32_t d = 0; d < D; ++d) clus[d] = (label[d] == PO_INVALID) ? -1 : knum[ord[label[d]]];
  *n_clusters_all = nall; *n_clusters = N;
  free(ord); free(S); free(Sx); free(Sy); free(sz); free(knum);
  return rc;
}

/* ---- O5 hits (the step after clustering in the paper's Fig. 1: raw -> clusters
 * -> hits).  The paper defines no hit arithmetic (L118); readings A26-A30 of
 * DESIGN.md fix it.  For every KEPT cluster k (dense number of O4), over its member digis
 * {d : clus[d] == k} (duplicates included, A6):
 *   bounding box   minRow, maxRow, minCol, maxCol                                        (A28)
 *   exact sums     S, Sx, Sy as in O4 (int64, scale 2^14)                                (A9)
 *   local position x = ((double)Sx/(double)S + 0.5 - R/2) * pitch_row   [um]  (row index -> local x)
 *                  y = ((double)Sy/(double)S + 0.5 - C/2) * pitch_col   [um]  (col index -> local y)
 *                  pixel centres sit at index + 0.5, origin at the module centre, uniform pitch, no
 *                  big-pixel correction (A13, A26); binary64 operations in exactly this order
 *                  (divide, add 0.5, subtract R/2, multiply), each rounded to nearest, then ONE
 *                  cast to binary32 (A27)
 *   edge flags     bit0: minRow == 0 or maxRow == R-1;  bit1: minCol == 0 or maxCol == C-1   (A29)
 *   error estimate per coordinate, span = max - min + 1, c = 1/sqrt(12) (binary64 literal):
 *                  touching that border: pitch*c*span; else span == 1: pitch*c; else pitch*c*0.5
 *                  evaluated as (pitch*c)*factor in binary64, cast to binary32               (A30)
 * ht_rows = minRow | maxRow << 16, ht_cols = minCol | maxCol << 16.  Returns 0, -1 on allocation failure. */
int po_hits(uint32_t D, uint32_t N, uint32_t R, uint32_t C,
            const int32_t *clus, const float *charge, const uint16_t *d_row, const uint16_t *d_col,
            double pitch_row_um, double pitch_col_um,
            float *ht_x, float *ht_y, float *ht_xerr, float *ht_yerr,
            uint32_t *ht_rows, uint32_t *ht_cols, uint16_t *ht_flags) {
  const double inv_sqrt12 = 0.28867513459481287;   /* 1/sqrt(12) rounded to binary64 */
  size_t n = N ? N : 1;
  int64_t *S = (int64_t *)calloc(n, sizeof(int64_t)), *Sx = (int64_t *)calloc(n, sizeof(int64_t)), *Sy = (int64_t *)calloc(n, sizeof(int64_t));
  uint32_t *rmin = (uint32_t *)malloc(n * sizeof(uint32_t)), *rmax = (uint32_t *)malloc(n * sizeof(uint32_t));
  uint32_t *cmin = (uint32_t *)malloc(n * sizeof(uint32_t)), *cmax = (uint32_t *)malloc(n * sizeof(uint32_t));
  if (!S || !Sx || !Sy || !rmin || !rmax || !cmin || !cmax) { free(S); free(Sx); free(Sy); free(rmin); free(rmax); free(cmin); free(cmax); return -1; }
  for (uint32_t k = 0; k < N; ++k) { rmin[k] = 0xFFFFFFFFu; cmin[k] = 0xFFFFFFFFu; rmax[k] = 0; cmax[k] = 0; }
  for (uint32_t d = 0; d < D; ++d) {
    if (clus[d] < 0) continue;
    uint32_t k = (uint32_t)clus[d];
    int64_t qf = (int64_t)(charge[d] * 16384.0f);
    S[k] += qf; Sx[k] += qf * (int64_t)d_row[d]; Sy[k] += qf * (int64_t)d_col[d];
    if (d_row[d] < rmin[k]) rmin[k] = d_row[d];
    if (d_row[d] > rmax[k]) rmax[k] = d_row[d];
    if (d_col[d] < cmin[k]) cmin[k] = d_col[d];
    if (d_col[d] > cmax[k]) cmax[k] = d_col[d];
  }
  for (uint32_t k = 0; k < N; ++k) {
    double x = (double)Sx[k] / (double)S[k];
    x = x + 0.5; x = x - 0.5 * (double)R; x = x * pitch_row_um;
    double y = (double)Sy[k] / (double)S[k];
    y = y + 0.5; y = y - 0.5 * (double)C; y = y * pitch_col_um;
    ht_x[k] = (float)x; ht_y[k] = (float)y;
    uint32_t span_r = rmax[k] - rmin[k] + 1, span_c = cmax[k] - cmin[k] + 1;
    int edge_r = (rmin[k] == 0 || rmax[k] == R - 1), edge_c = (cmin[k] == 0 || cmax[k] == C - 1);
    double fr = edge_r ? (double)span_r : (span_r == 1 ? 1.0 : 0.5);
    double fc = edge_c ? (double)span_c : (span_c == 1 ? 1.0 : 0.5);
    double er = pitch_row_um * inv_sqrt12; er = er * fr;
    double ec = pitch_col_um * inv_sqrt12; ec = ec * fc;
    ht_xerr[k] = (float)er; ht_yerr[k] = (float)ec;
    ht_rows[k] = rmin[k] | (rmax[k] << 16); ht_cols[k] = cmin[k] | (cmax[k] << 16);
    ht_flags[k] = (uint16_t)((edge_r ? 1 : 0) | (edge_c ? 2 : 0));
  }
  free(S); free(Sx); free(Sy); free(rmin); free(rmax); free(cmin); free(cmax);
  return 0;
}

/* ---- occupancy (a second consumer of the digis on a parallel branch; the paper's Fig. 1 and
 * section 4.2, only say that several modules may consume one product).  Per module m: the number of
 * kept digis (charge >= pixThr, A8) and the sum of their ADC values (uint32, exact).                                   */
void po_occupancy(uint32_t D, uint32_t M, const uint16_t *d_module, const uint16_t *d_adc, const uint8_t *kept,
                  uint32_t *occ_count /* [M] */, uint32_t *occ_adc_sum /* [M] */) {
  for (uint32_t m = 0; m < M; ++m) { occ_count[m] = 0; occ_adc_sum[m] = 0; }
  for (uint32_t d = 0; d < D; ++d)
    if (kept[d]) { occ_count[d_module[d]] += 1; occ_adc_sum[d_module[d]] += d_adc[d]; }
}

/* ---- O0 bucket by module (reading A31; arbitrary word order) ----
 * The step BEFORE decode when the words of an event come in arbitrary order: a STABLE bucket sort of the words by
 * module.  Key of word i = its module if it is a digi word (bit 31 clear, module < M, row < R, col < C: the test of
 * O1), else M (error and invalid words form one last bucket).  out_* receive the words and ADC values in key order,
 * equal keys in their input order; orig[p] = input index of the word now at position p.  Decoding the bucketed
 * stream (O1) then yields the digi list "by module, input order inside a module" and the error list in input order;
 * word indices are mapped back to input positions through orig[] by the caller (oracle.run_unordered).
 * Plain counting sort: count, prefix, place.                                                                       */
void po_bucket(const uint32_t *words, const uint16_t *adc, uint32_t W, uint32_t M, uint32_t R, uint32_t C,
               uint32_t *out_words, uint16_t *out_adc, uint32_t *orig) {
  uint32_t *start = (uint32_t *)calloc((size_t)M + 2, sizeof(uint32_t));
  if (!start) return;
  for (uint32_t i = 0; i < W; ++i) {
    uint32_t w = words[i], mod = (w >> 20) & 0x7FFu, row = (w >> 12) & 0xFFu, col = (w >> 3) & 0x1FFu;
    uint32_t key = ((w >> 31) || mod >= M || row >= R || col >= C) ? M : mod;
    start[key + 1] += 1;
  }
  for (uint32_t k = 0; k <= M; ++k) start[k + 1] += start[k];     /* start[k] = number of words with key < k */
  for (uint32_t i = 0; i < W; ++i) {
    uint32_t w = words[i], mod = (w >> 20) & 0x7FFu, row = (w >> 12) & 0xFFu, col = (w >> 3) & 0x1FFu;
    uint32_t key = ((w >> 31) || mod >= M || row >= R || col >= C) ? M : mod;
    uint32_t p = start[key]++;
    out_words[p] = w; out_adc[p] = adc[i]; orig[p] = i;
  }
  free(start);
}

/* ---- the whole chain, in order O1..O5 (what bench.py's cpu_baseline times) ----
 * All output arrays have capacity W (mod_* arrays M+1) and are owned by the caller.
 * Hit arrays have capacity W too.
 * counters[0..6] = n_digis, n_errors, n_kept_digis, n_clusters_all, n_clusters, sorted_ok, rc.   */
int po_run(const uint32_t *words, const uint16_t *adc, uint32_t W,
           uint32_t M, uint32_t R, uint32_t C,
           const float *gain, const float *ped, float pix_thr, float clus_thr,
           uint16_t *d_module, uint16_t *d_row, uint16_t *d_col, uint16_t *d_adc, uint32_t *d_word_idx,
           uint32_t *e_word, uint32_t *e_idx, uint32_t *mod_digi_start,
           float *charge, uint8_t *kept, uint32_t *label,
           uint32_t *cl_label, uint16_t *cl_module, uint32_t *cl_size,
           float *cl_charge, float *cl_row, float *cl_col,
           int32_t *clus, uint32_t *mod_clus_start,
           double pitch_row_um, double pitch_col_um,
           float *ht_x, float *ht_y, float *ht_xerr, float *ht_yerr,
           uint32_t *ht_rows, uint32_t *ht_cols, uint16_t *ht_flags, uint32_t *counters) {
  uint32_t D, E, ok, nk, nall, N;
  po_decode(words, adc, W, M, R, C, d_module, d_row, d_col, d_adc, d_word_idx, e_word, e_idx,
            mod_digi_start, &D, &E, &ok);
  po_calibrate(D, d_adc, d_module, gain, ped, pix_thr, charge, kept, &nk);
  int rc = po_cluster(D, M, R, C, d_module, d_row, d_col, kept, label);
  if (rc == 0)
    rc = po_reduce(D, M, label, charge, d_module, d_row, d_col, clus_thr, cl_label, cl_module, cl_size,
                   cl_charge, cl_row, cl_col, clus, mod_clus_start, &nall, &N);
  else { nall = 0; N = 0; }
  if (rc == 0 && po_hits(D, N, R, C, clus, charge, d_row, d_col, pitch_row_um, pitch_col_um, ht_x, ht_y, ht_xerr, ht_yerr,
                         ht_rows, ht_cols, ht_flags) != 0) rc = -1;
  counters[0] = D; counters[1] = E; counters[2] = nk; counters[3] = nall; counters[4] = N;
  counters[5] = ok; counters[6] = (uint32_t)rc;
  return rc;
}

/* ---- O6 exact-sum self-check (A9), paranoid mode, never timed.  Verifies for one event's
 * decoded/calibrated/labelled data that (a) q*2^14 is integral for every kept digi, (b) int64
 * sums equal an __int128 accumulation, (c) where the sums stay below 2^53 a plain binary64 sum
 * in index order and in reversed order both equal S*2^-14.  Returns 0 if all hold, else the
 * number of the first failed check.                                                             */
int po_check_exact_sums(uint32_t D, const uint32_t *label, const float *charge, const uint16_t *d_col) {
  for (uint32_t L = 0; L < D; ++L) {
    if (label[L] != L) continue;
    int64_t S = 0, Sy = 0; __int128 S128 = 0, Sy128 = 0; double fwd = 0.0, bwd = 0.0;
    for (uint32_t d = 0; d < D; ++d) {
      if (label[d] != L) continue;
      float scaled = charge[d] * 16384.0f; int64_t qf = (int64_t)scaled;
      if ((float)qf != scaled) return 1;
      S += qf; Sy += qf * (int64_t)d_col[d]; S128 += qf; Sy128 += (__int128)qf * d_col[d];
      fwd += (double)charge[d];
    }
    for (uint32_t d = D; d-- > 0;) if (label[d] == L) bwd += (double)charge[d];
    if ((__int128)S != S128 || (__int128)Sy != Sy128) return 2;
    if (S < ((int64_t)1 << 53)) {
      double exact = (double)S / 16384.0;
      if (fwd != exact || bwd != exact) return 3;
    }
  }
  return 0;
}

/* pixgen.c — seeded synthetic pixel-detector events (the five workloads of BASELINE.json `configs`).
 *
 * This is the ONE input generator that both the CUDA path's tests/bench and the oracle's tests
 * use.  It holds none of the method's arithmetic: it only draws cluster shapes and ADC values,
 * ENCODES them into raw words (the inverse of what the method decodes) and draws calibration
 * tables.  It never decodes, calibrates, clusters or reduces anything.
 *
 * Recipe: DESIGN.md "Input recipe" (readings A15-A19, A21 of SURVEY.md section 8(c)/(d)).
 * The paper itself gives no workload (PAPER.md L118 defers performance to its ref. [8]).
 *
 * Plain C99, single thread, deterministic: every (config, event, module) has its own PRNG stream,
 * so an event does not depend on which other events were generated before it.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---------------- PRNG: SplitMix64 mixer seeding a xoshiro256** state ---------------- */
typedef struct { uint64_t s[4]; } rng_t;

static uint64_t mix64(uint64_t *x) {
  uint64_t z = (*x += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
static void rng_seed(rng_t *r, uint64_t base, uint64_t a, uint64_t b, uint64_t c) {
  uint64_t x = base;
  x ^= mix64(&x) + a * 0xD6E8FEB86659FD93ull;
  x ^= mix64(&x) + b * 0xA0761D6478BD642Full;
  x ^= mix64(&x) + c * 0xE7037ED1A0B428DBull;
  for (int i = 0; i < 4; ++i) r->s[i] = mix64(&x);
}
static inline uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static inline uint64_t rng_u64(rng_t *r) {
  uint64_t *s = r->s, res = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
  s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45);
  return res;
}
static inline double rng_unit(rng_t *r) { return (double)(rng_u64(r) >> 11) * (1.0 / 9007199254740992.0); }
/* uniform integer in [0, n) */
static inline uint32_t rng_below(rng_t *r, uint32_t n) {
  return (uint32_t)(((rng_u64(r) >> 32) * (uint64_t)n) >> 32);
}
static double rng_normal(rng_t *r) { /* Box-Muller, one value per call */
  double u1 = rng_unit(r), u2 = rng_unit(r);
  if (u1 < 1e-300) u1 = 1e-300;
  return sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
}
static uint32_t rng_poisson(rng_t *r, double lam) { /* Knuth product method, lam < ~500 */
  double L = exp(-lam), p = 1.0; uint32_t k = 0;
  do { ++k; p *= rng_unit(r); } while (p > L);
  return k - 1;
}
/* Geometric on {1,2,...} with the given mean (success probability 1/mean). */
static uint32_t rng_geometric(rng_t *r, double mean) {
  if (mean <= 1.0) return 1;
  double p = 1.0 / mean, u = rng_unit(r);
  if (u < 1e-300) u = 1e-300;
  double k = floor(log(u) / log(1.0 - p));
  if (k > 1e6) k = 1e6;
  return 1u + (uint32_t)k;
}

/* ---------------- workload parameters ---------------- */
typedef struct {
  uint32_t n_modules, n_rows, n_cols;
  double   lambda;          /* mean seeded clusters per module (Poisson); unused if fill_pixels>0  */
  uint32_t hot_modules;     /* first `hot_modules` modules get lambda*hot_factor                   */
  double   hot_factor;
  double   compact_mean;    /* Geometric mean size of compact clusters                             */
  double   frac_elongated;  /* fraction of clusters grown along col                                */
  double   elongated_mean;  /* their size is 1 + Geometric(elongated_mean - 1)                     */
  double   frac_strip;      /* fraction of 1-pixel-wide strips (configs[4])                        */
  uint32_t strip_min, strip_max;
  double   p_touch;         /* probability that a cluster starts 8-adjacent to the previous one    */
  uint32_t fill_pixels;     /* if >0: add clusters until the module holds >= this many pixels      */
  double   err_frac;        /* fraction of all words that are error words                          */
  uint32_t adc_law;         /* 0 = uniform 10..255, 1 = Landau-like (Moyal), A17                   */
} pixgen_params;

typedef struct {
  uint64_t n_words, n_digis, n_errors, n_seeded_clusters, max_digis_per_module;
} pixgen_stats;

int pixgen_default_params(uint32_t config, pixgen_params *p) {
  memset(p, 0, sizeof *p);
  p->n_rows = 160; p->n_cols = 416; p->hot_factor = 1.0; p->compact_mean = 3.0;
  p->strip_min = 20; p->strip_max = 100;
  switch (config) {
    case 0: p->n_modules = 64;   p->lambda = 10.4; p->err_frac = 0.01;  p->adc_law = 0; break;
    case 1: /* fallthrough: configs[2] is 64 events of the configs[1] law */
    case 2: p->n_modules = 1856; p->lambda = 4.31; p->err_frac = 0.005; p->adc_law = 1;
            p->frac_elongated = 0.2; p->elongated_mean = 20.75; break;
    case 3: p->n_modules = 1856; p->lambda = 14.0; p->err_frac = 0.005; p->adc_law = 1;
            p->frac_elongated = 0.2; p->elongated_mean = 23.05; p->hot_modules = 96; p->hot_factor = 4.0; break;
    case 4: p->n_modules = 1856; p->err_frac = 0.005; p->adc_law = 1; p->compact_mean = 13.0;
            p->frac_strip = 0.15; p->p_touch = 0.15; p->fill_pixels = 6656; break;
    default: return -1;
  }
  return 0;
}

/* Calibration tables (A21): gain ~ N(80,5) in (0,128), pedestal ~ N(0,200), stored as binary32. */
int pixgen_calib(uint64_t seed, uint32_t config, uint32_t n_modules, float *gain, float *ped) {
  rng_t r; rng_seed(&r, seed, config, 0xCA11Bull, 0);
  for (uint32_t m = 0; m < n_modules; ++m) {
    float g, p;
    do { g = (float)(80.0 + 5.0 * rng_normal(&r)); } while (!(g > 0.0f && g < 128.0f));
    do { p = (float)(200.0 * rng_normal(&r)); } while (p != 0.0f && fabsf(p) < 9.5367431640625e-07f);
    gain[m] = g; ped[m] = p;
  }
  return 0;
}

/* ---------------- per-module pixel drawing ---------------- */
typedef struct { uint16_t row, col; } pix_t;

typedef struct {
  uint32_t R, C;
  uint8_t *occ;           /* R*C occupancy flags                                  */
  pix_t   *pix;           /* all pixels of the module, in creation order          */
  uint32_t n, cap;
  uint32_t prev_start, prev_n;   /* the previous cluster = pix[prev_start .. +prev_n) */
} modbuf_t;

static inline int mb_free(const modbuf_t *mb, int r, int c) {
  return r >= 0 && c >= 0 && (uint32_t)r < mb->R && (uint32_t)c < mb->C && !mb->occ[(uint32_t)r * mb->C + (uint32_t)c];
}
static inline void mb_add(modbuf_t *mb, int r, int c) {
  if (mb->n == mb->cap) { mb->cap = mb->cap ? mb->cap * 2 : 1024; mb->pix = (pix_t *)realloc(mb->pix, mb->cap * sizeof(pix_t)); }
  mb->occ[(uint32_t)r * mb->C + (uint32_t)c] = 1;
  mb->pix[mb->n].row = (uint16_t)r; mb->pix[mb->n].col = (uint16_t)c; mb->n++;
}
static const int DR[8] = {-1, -1, -1, 0, 0, 1, 1, 1};
static const int DC[8] = {-1, 0, 1, -1, 1, -1, 0, 1};

/* Pick the start pixel: uniform, or (touching rule) a free pixel 8-adjacent to a random pixel of
 * the previous cluster.  Returns 0 if none found after a bounded number of tries. */
static int pick_start(modbuf_t *mb, rng_t *r, double p_touch, int *pr, int *pc) {
  if (p_touch > 0.0 && mb->prev_n > 0 && rng_unit(r) < p_touch) {
    for (int t = 0; t < 32; ++t) {
      pix_t q = mb->pix[mb->prev_start + rng_below(r, mb->prev_n)];
      int k = (int)rng_below(r, 8), rr = q.row + DR[k], cc = q.col + DC[k];
      if (mb_free(mb, rr, cc)) { *pr = rr; *pc = cc; return 1; }
    }
  }
  for (int t = 0; t < 64; ++t) {
    int rr = (int)rng_below(r, mb->R), cc = (int)rng_below(r, mb->C);
    if (mb_free(mb, rr, cc)) { *pr = rr; *pc = cc; return 1; }
  }
  return 0;
}

static void grow_compact(modbuf_t *mb, rng_t *r, uint32_t size, int r0, int c0) {
  uint32_t start = mb->n, rejects = 0;
  mb_add(mb, r0, c0);
  while (mb->n - start < size && rejects < 16u * size) {
    pix_t q = mb->pix[start + rng_below(r, mb->n - start)];
    int k = (int)rng_below(r, 8), rr = q.row + DR[k], cc = q.col + DC[k];
    if (mb_free(mb, rr, cc)) mb_add(mb, rr, cc); else ++rejects;
  }
}
/* grown from the last pixel: dcol = s, drow in {-1,0,+1} w.p. {p_side, 1-2 p_side, p_side} */
static void grow_line(modbuf_t *mb, rng_t *r, uint32_t size, int r0, int c0, int s, double p_side) {
  uint32_t start = mb->n; int rr = r0, cc = c0;
  mb_add(mb, r0, c0);
  while (mb->n - start < size) {
    double u = rng_unit(r);
    int dr = (u < p_side) ? -1 : (u < 2.0 * p_side ? 1 : 0);
    int nr = rr + dr, nc = cc + s;
    if (!mb_free(mb, nr, nc)) break;
    mb_add(mb, nr, nc); rr = nr; cc = nc;
  }
}

static uint16_t draw_adc(rng_t *r, uint32_t law) {
  if (law == 0) return (uint16_t)(10u + rng_below(r, 246));
  double z = rng_normal(r), y = z * z;
  if (y < 1e-300) y = 1e-300;
  double v = floor(40.0 + 10.0 * (-log(y)) + 0.5);
  if (v < 10.0) v = 10.0;
  if (v > 255.0) v = 255.0;
  return (uint16_t)v;
}

/* ---------------- one event ---------------- */
/* Output buffers are malloc'ed here; release with pixgen_free.  Returns 0 on success. */
int pixgen_event(uint64_t seed, uint32_t config, uint32_t event, const pixgen_params *P,
                 uint32_t **words_out, uint16_t **adc_out, pixgen_stats *st) {
  const uint32_t M = P->n_modules, R = P->n_rows, C = P->n_cols;
  if (M == 0 || M > 2048 || R == 0 || R > 256 || C == 0 || C > 512) return -1;
  modbuf_t mb; memset(&mb, 0, sizeof mb);
  mb.R = R; mb.C = C; mb.occ = (uint8_t *)calloc((size_t)R * C, 1);

  size_t cap = 1u << 16, D = 0;
  uint32_t *dw = (uint32_t *)malloc(cap * sizeof(uint32_t));   /* digi words, module-grouped */
  uint16_t *da = (uint16_t *)malloc(cap * sizeof(uint16_t));
  uint64_t n_clusters = 0, max_pm = 0;

  for (uint32_t m = 0; m < M; ++m) {
    rng_t r; rng_seed(&r, seed, config, event, m);
    mb.n = 0; mb.prev_n = 0; mb.prev_start = 0;
    uint32_t target_clusters = 0;
    if (!P->fill_pixels) {
      double lam = P->lambda * (m < P->hot_modules ? P->hot_factor : 1.0);
      target_clusters = rng_poisson(&r, lam);
    }
    uint32_t made = 0, stalls = 0;
    while (P->fill_pixels ? (mb.n < P->fill_pixels && stalls < 1000) : (made < target_clusters)) {
      int r0, c0;
      if (!pick_start(&mb, &r, P->p_touch, &r0, &c0)) { ++stalls; ++made; continue; }
      uint32_t start = mb.n;
      double u = rng_unit(&r);
      if (u < P->frac_strip) {
        uint32_t len = P->strip_min + rng_below(&r, P->strip_max - P->strip_min + 1);
        grow_line(&mb, &r, len, r0, c0, +1, 0.0);
      } else if (u < P->frac_strip + P->frac_elongated) {
        uint32_t size = 1u + rng_geometric(&r, P->elongated_mean - 1.0);
        int s = (rng_u64(&r) & 1) ? 1 : -1;
        grow_line(&mb, &r, size, r0, c0, s, 0.1);
      } else {
        grow_compact(&mb, &r, rng_geometric(&r, P->compact_mean), r0, c0);
      }
      mb.prev_start = start; mb.prev_n = mb.n - start;
      ++made; ++n_clusters;
    }
    /* Fisher-Yates shuffle of this module's pixels: nothing may rely on pixel order (A5) */
    for (uint32_t i = mb.n; i > 1; --i) {
      uint32_t j = rng_below(&r, i); pix_t t = mb.pix[i - 1]; mb.pix[i - 1] = mb.pix[j]; mb.pix[j] = t;
    }
    if (D + mb.n > cap) {
      while (D + mb.n > cap) cap *= 2;
      dw = (uint32_t *)realloc(dw, cap * sizeof(uint32_t)); da = (uint16_t *)realloc(da, cap * sizeof(uint16_t));
    }
    for (uint32_t i = 0; i < mb.n; ++i) {
      dw[D] = (m << 20) | ((uint32_t)mb.pix[i].row << 12) | ((uint32_t)mb.pix[i].col << 3);
      da[D] = draw_adc(&r, P->adc_law);
      mb.occ[(uint32_t)mb.pix[i].row * C + mb.pix[i].col] = 0;
      ++D;
    }
    if (mb.n > max_pm) max_pm = mb.n;
  }

  /* error words (A19): E = round(f*D/(1-f)) at uniform positions of the final stream */
  rng_t re; rng_seed(&re, seed, config, event, 0xE7707ull);
  size_t E = (P->err_frac > 0.0 && P->err_frac < 1.0) ? (size_t)floor(P->err_frac * (double)D / (1.0 - P->err_frac) + 0.5) : 0;
  size_t W = D + E;
  uint32_t *w = (uint32_t *)malloc((W ? W : 1) * sizeof(uint32_t));
  uint16_t *a = (uint16_t *)malloc((W ? W : 1) * sizeof(uint16_t));
  /* choose which of the W positions are errors: selection sampling (Knuth 3.4.2 S), in order */
  size_t need = E, di = D; /* fill from the back so "module of the following word" is known */
  uint32_t following_module = M ? M - 1 : 0;
  for (size_t pos = W; pos-- > 0;) {
    size_t remaining = pos + 1;
    int is_err = need > 0 && (rng_unit(&re) * (double)remaining < (double)need);
    if (is_err || di == 0) {
      if (!is_err && di == 0) is_err = 1; /* cannot happen: need == remaining then */
      uint32_t junk = (uint32_t)(rng_u64(&re) & 0x1FFFFu), code = 1u + rng_below(&re, 7);
      w[pos] = 0x80000000u | (following_module << 20) | (junk << 3) | code;
      a[pos] = 0; --need;
    } else {
      --di; w[pos] = dw[di]; a[pos] = da[di]; following_module = dw[di] >> 20;
    }
  }
  free(dw); free(da); free(mb.occ); free(mb.pix);
  *words_out = w; *adc_out = a;
  if (st) { st->n_words = W; st->n_digis = D; st->n_errors = E; st->n_seeded_clusters = n_clusters; st->max_digis_per_module = max_pm; }
  return 0;
}

void pixgen_free(void *p) { free(p); }

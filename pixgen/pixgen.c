/* pixgen.c -- seeded synthetic inputs for the pixel Clusters path (tables + raw-word events).
 *
 * This module serves BOTH the oracle tests and the CUDA tests/bench.  It produces input bytes
 * only: the cabling map, the gain/pedestal table, and per-event raw 32-bit words with their FED
 * offsets.  It holds none of the method's arithmetic (no decode, no calibration, no clustering);
 * it ENCODES (module,row,col,adc) into words through the cabling it built itself, which is the
 * inverse direction of the path.  The clusters it draws are not ground truth: drawn clusters may
 * touch and merge, only the oracle defines the answer.
 *
 * Recipe: DESIGN.md "Input recipe" (G1-G8), after BASELINE.json configs[0..4] and PAPER.md:41
 * (1000 events ~ 250 MB => ~62.5k words/event at <PU>=50).  Integer-only PRNG (splitmix64-seeded
 * xoshiro256**), no libm, so bytes are identical on every box.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include "adc_cdf.h"

#define ROWS 160
#define COLS 416
#define ROC_ROWS 80
#define ROC_COLS 52
#define OCC_WORDS ((ROWS * COLS) / 32) /* 2080 */

/* ---------------------------------------------------------------- PRNG */
typedef struct { uint64_t s[4]; } rng_t;

static uint64_t splitmix64(uint64_t* x) {
  uint64_t z = (*x += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
static void rng_seed(rng_t* r, uint64_t seed) {
  uint64_t x = seed;
  for (int i = 0; i < 4; ++i) r->s[i] = splitmix64(&x);
}
static inline uint64_t rotl64(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static inline uint64_t rng_next(rng_t* r) {
  uint64_t* s = r->s;
  uint64_t result = rotl64(s[1] * 5, 7) * 9;
  uint64_t t = s[1] << 17;
  s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3];
  s[2] ^= t; s[3] = rotl64(s[3], 45);
  return result;
}
static inline uint32_t rng_u32(rng_t* r) { return (uint32_t)(rng_next(r) >> 32); }
/* uniform in [0,n): multiply-shift (bias < 2^-32 * n, irrelevant here, and deterministic) */
static inline uint32_t rng_below(rng_t* r, uint32_t n) { return (uint32_t)(((uint64_t)rng_u32(r) * n) >> 32); }

static void shuffle_u32(rng_t* r, uint32_t* a, uint32_t n) {
  for (uint32_t i = n; i > 1; --i) {
    uint32_t j = rng_below(r, i);
    uint32_t t = a[i - 1]; a[i - 1] = a[j]; a[j] = t;
  }
}

/* ---------------------------------------------------------------- tables */
/* Cabling entry packing (S3): bit0 link_mapped, bit1 roc_valid, bits2-17 module,
 * bits18-20 rocx (0..7), bit21 rocy, bit22 flip_r, bit23 flip_c.  Index (fed*64+link)*32+roc. */
static inline uint32_t pack_entry(uint32_t roc_valid, uint32_t module, uint32_t rocx, uint32_t rocy,
                                  uint32_t flip_r, uint32_t flip_c) {
  return 1u | (roc_valid << 1) | (module << 2) | (rocx << 18) | (rocy << 21) | (flip_r << 22) | (flip_c << 23);
}

/* n_feds * links_per_fed must equal n_modules; links_per_fed <= 64. Returns 0 on success. */
int pixgen_cabling(uint32_t n_feds, uint32_t links_per_fed, uint32_t n_modules, uint64_t seed, uint32_t* entry) {
  if (links_per_fed > 64 || n_feds * links_per_fed != n_modules || n_modules > 65534) return -1;
  rng_t r; rng_seed(&r, seed);
  memset(entry, 0, (size_t)n_feds * 64 * 32 * sizeof(uint32_t));
  uint32_t* modperm = (uint32_t*)malloc(sizeof(uint32_t) * n_modules);
  for (uint32_t i = 0; i < n_modules; ++i) modperm[i] = i;
  shuffle_u32(&r, modperm, n_modules);
  uint32_t k = 0;
  for (uint32_t fed = 0; fed < n_feds; ++fed) {
    uint32_t links[64];
    for (uint32_t i = 0; i < 64; ++i) links[i] = i;
    shuffle_u32(&r, links, 64); /* first links_per_fed entries = mapped links of this FED */
    uint8_t mapped[64]; memset(mapped, 0, sizeof mapped);
    for (uint32_t i = 0; i < links_per_fed; ++i) mapped[links[i]] = 1;
    for (uint32_t link = 0; link < 64; ++link) {
      if (!mapped[link]) continue;
      uint32_t module = modperm[k++];
      uint32_t place[16];
      for (uint32_t i = 0; i < 16; ++i) place[i] = i;
      shuffle_u32(&r, place, 16);
      uint32_t* e = entry + ((size_t)fed * 64 + link) * 32;
      for (uint32_t roc = 0; roc < 32; ++roc) {
        if (roc < 16) {
          uint32_t p = place[roc];
          uint32_t bits = rng_u32(&r);
          e[roc] = pack_entry(1, module, p & 7, p >> 3, bits & 1, (bits >> 1) & 1);
        } else {
          e[roc] = pack_entry(0, module, 0, 0, 0, 0);
        }
      }
    }
  }
  free(modperm);
  return 0;
}

/* gain ~ N(3.0, 0.1), pedestal ~ N(20, 2) per (module, col), float32.  The normal variate is the
 * sum of 12 uniforms minus 6 (Irwin-Hall), built from integers so no libm is involved. */
static double normal12(rng_t* r) {
  uint64_t acc = 0;
  for (int i = 0; i < 12; ++i) acc += rng_u32(r);
  return ((double)acc - 6.0 * 4294967296.0) / 4294967296.0;
}
void pixgen_gains(uint32_t n_modules, uint64_t seed, float* gain, float* pedestal) {
  rng_t r; rng_seed(&r, seed);
  for (size_t i = 0; i < (size_t)n_modules * COLS; ++i) {
    gain[i] = (float)(3.0 + 0.1 * normal12(&r));
    pedestal[i] = (float)(20.0 + 2.0 * normal12(&r));
  }
}

/* ---------------------------------------------------------------- event generation */
typedef struct {
  uint32_t clusters_per_module; /* >0: exactly this many short clusters in every module (cfg0) */
  uint32_t n_clusters;          /* else: this many clusters, module drawn per cluster (cfg1/3) */
  uint32_t inner_modules;       /* module ids [0, inner_modules) get weight inner_weight (BJ cfg1: 96, 4) */
  uint32_t inner_weight;
  uint32_t long_permille;       /* per-mille of clusters that are long 50-500 px tracks (cfg3: 20) */
  uint32_t shuffle_order;       /* 1: words of a module in seeded random order; 0: read-out order */
  uint32_t edge_class;          /* 0 none; 1 dense(a) 2 duplicates(b) 3 invalid words(c) 4 edges(d) 5 degenerate(e) */
  uint32_t edge_sub;            /* sub-case selector for class 5 (0..4) */
} pixgen_cfg;

typedef struct {
  uint32_t n_feds, n_modules;
  const uint32_t* entry;
  /* inverse cabling */
  uint16_t* mod_fed; uint16_t* mod_link;  /* [M] */
  uint8_t* mod_roc;                       /* [M*16] roc id at placement p */
  uint8_t* mod_flip;                      /* [M*16] bit0 flip_r bit1 flip_c at placement p */
  uint8_t* link_unmapped;                 /* [F*8]: up to 8 unmapped link ids per FED, count in [F*8+...]*/
  uint8_t* n_unmapped;                    /* [F] */
  uint32_t* occ;                          /* [M*OCC_WORDS] occupancy bitmap, all-zero between events */
  /* pixel buffer */
  uint32_t cap, n;
  uint16_t* pm; uint8_t* pr; uint16_t* pc; uint8_t* pa;
  /* per-module word lists */
  uint32_t* mstart;                       /* [M+1] */
  uint32_t* wbuf; uint32_t* wbuf2;
} ctx_t;

static void ctx_free(ctx_t* c) {
  free(c->mod_fed); free(c->mod_link); free(c->mod_roc); free(c->mod_flip); free(c->link_unmapped);
  free(c->n_unmapped); free(c->occ); free(c->pm); free(c->pr); free(c->pc); free(c->pa);
  free(c->mstart); free(c->wbuf); free(c->wbuf2);
}

static int ctx_init(ctx_t* c, uint32_t n_feds, uint32_t n_modules, const uint32_t* entry, uint32_t cap) {
  memset(c, 0, sizeof *c);
  c->n_feds = n_feds; c->n_modules = n_modules; c->entry = entry; c->cap = cap;
  c->mod_fed = (uint16_t*)malloc(2 * (size_t)n_modules);
  c->mod_link = (uint16_t*)malloc(2 * (size_t)n_modules);
  c->mod_roc = (uint8_t*)malloc(16 * (size_t)n_modules);
  c->mod_flip = (uint8_t*)malloc(16 * (size_t)n_modules);
  c->link_unmapped = (uint8_t*)calloc(64 * (size_t)n_feds, 1);
  c->n_unmapped = (uint8_t*)calloc(n_feds, 1);
  c->occ = (uint32_t*)calloc((size_t)n_modules * OCC_WORDS, sizeof(uint32_t));
  c->pm = (uint16_t*)malloc(2 * (size_t)cap); c->pr = (uint8_t*)malloc(cap);
  c->pc = (uint16_t*)malloc(2 * (size_t)cap); c->pa = (uint8_t*)malloc(cap);
  c->mstart = (uint32_t*)malloc(sizeof(uint32_t) * ((size_t)n_modules + 1));
  c->wbuf = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)cap);
  c->wbuf2 = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)cap);
  if (!c->occ || !c->wbuf || !c->wbuf2 || !c->pm) return -1;
  memset(c->mod_fed, 0xFF, 2 * (size_t)n_modules);
  for (uint32_t fed = 0; fed < n_feds; ++fed)
    for (uint32_t link = 0; link < 64; ++link) {
      const uint32_t* e = entry + ((size_t)fed * 64 + link) * 32;
      if (!(e[0] & 1u)) { c->link_unmapped[fed * 64 + c->n_unmapped[fed]++] = (uint8_t)link; continue; }
      for (uint32_t roc = 0; roc < 32; ++roc) {
        if (!(e[roc] & 2u)) continue;
        uint32_t m = (e[roc] >> 2) & 0xFFFF, rocx = (e[roc] >> 18) & 7, rocy = (e[roc] >> 21) & 1;
        c->mod_fed[m] = (uint16_t)fed; c->mod_link[m] = (uint16_t)link;
        c->mod_roc[m * 16 + rocy * 8 + rocx] = (uint8_t)roc;
        c->mod_flip[m * 16 + rocy * 8 + rocx] = (uint8_t)((e[roc] >> 22) & 3);
      }
    }
  return 0;
}

static inline uint32_t draw_adc(rng_t* r) {
  uint32_t u = rng_u32(r);
  /* adc = 1 + #{i : u >= T[i]}; T is non-decreasing -> binary search for the first T[i] > u */
  uint32_t lo = 0, hi = 254;
  while (lo < hi) { uint32_t mid = (lo + hi) >> 1; if (PIXGEN_ADC_CDF[mid] > u) hi = mid; else lo = mid + 1; }
  return 1 + lo;
}

static inline int occ_get(const ctx_t* c, uint32_t m, int r, int col) {
  uint32_t b = (uint32_t)r * COLS + (uint32_t)col;
  return (c->occ[(size_t)m * OCC_WORDS + (b >> 5)] >> (b & 31)) & 1u;
}
static inline void occ_set(ctx_t* c, uint32_t m, int r, int col) {
  uint32_t b = (uint32_t)r * COLS + (uint32_t)col;
  c->occ[(size_t)m * OCC_WORDS + (b >> 5)] |= 1u << (b & 31);
}
static inline void occ_clear(ctx_t* c, uint32_t m, int r, int col) {
  uint32_t b = (uint32_t)r * COLS + (uint32_t)col;
  c->occ[(size_t)m * OCC_WORDS + (b >> 5)] &= ~(1u << (b & 31));
}

/* add pixel if free; returns 1 when added */
static int add_pixel(ctx_t* c, rng_t* r, uint32_t m, int row, int col) {
  if (row < 0 || row >= ROWS || col < 0 || col >= COLS) return 0;
  if (c->n >= c->cap) return 0;
  if (occ_get(c, m, row, col)) return 0;
  occ_set(c, m, row, col);
  c->pm[c->n] = (uint16_t)m; c->pr[c->n] = (uint8_t)row; c->pc[c->n] = (uint16_t)col;
  c->pa[c->n] = (uint8_t)draw_adc(r);
  c->n++;
  return 1;
}

/* G1/G2: short cluster, n = min(Geometric(1/4), 30), 8-neighbour random walk, longer along col */
static void short_cluster(ctx_t* c, rng_t* r, uint32_t m, int r0, int c0) {
  uint32_t n = 1;
  while (n < 30 && rng_u32(r) >= 0x40000000u) ++n;
  int row = r0, col = c0;
  uint32_t got = (uint32_t)add_pixel(c, r, m, row, col);
  for (uint32_t step = 0; got < n && step < 20 * n + 50; ++step) {
    int dc, dr;
    do {
      dc = (int)rng_below(r, 3) - 1;
      uint32_t u = rng_below(r, 10);
      dr = u < 2 ? -1 : (u < 8 ? 0 : 1);
    } while (dc == 0 && dr == 0);
    row += dr; col += dc;
    if (row < 0) row = 0;
    if (row >= ROWS) row = ROWS - 1;
    if (col < 0) col = 0;
    if (col >= COLS) col = COLS - 1;
    got += (uint32_t)add_pixel(c, r, m, row, col);
  }
}

/* 2^(2^-k), k = 1..16 */
static const double POW2_FRAC[16] = {
  1.4142135623730951, 1.189207115002721, 1.0905077326652577, 1.0442737824274138,
  1.0218971486541166, 1.0108892860517005, 1.0054299011128027, 1.0027112750502025,
  1.0013547198921082, 1.0006771306930664, 1.0003385080526823, 1.0001692397053021,
  1.0000846162726944, 1.0000423072413958, 1.0000211533969647, 1.0000105766425498};

/* G6: long cluster = staircase track, length log-uniform in [50,500], slope k/64 with k in [6,64] */
static void long_cluster(ctx_t* c, rng_t* r, uint32_t m, int r0, int c0) {
  uint32_t xi = (uint32_t)(((uint64_t)rng_below(r, 65536) * 217706u) >> 16); /* 16.16 fixed in [0, log2 10) */
  double v = (double)(1u << (xi >> 16));
  for (int k = 0; k < 16; ++k) if (xi & (0x8000u >> k)) v *= POW2_FRAC[k];
  uint32_t len = (uint32_t)(50.0 * v);
  if (len > 500) len = 500;
  uint32_t k = 6 + rng_below(r, 59);
  int sc = (rng_u32(r) & 1) ? 1 : -1, sr = (rng_u32(r) & 1) ? 1 : -1;
  int row = r0, col = c0; uint32_t err = 0, got = 0;
  got += (uint32_t)add_pixel(c, r, m, row, col);
  while (got < len) {
    col += sc;
    if (col < 0 || col >= COLS) break;
    err += k;
    if (err >= 64) {
      err -= 64;
      got += (uint32_t)add_pixel(c, r, m, row, col); /* the row-step pixel */
      row += sr;
      if (row < 0 || row >= ROWS) break;
    }
    got += (uint32_t)add_pixel(c, r, m, row, col);
  }
}

static uint32_t draw_module(const pixgen_cfg* cfg, rng_t* r, uint32_t M) {
  uint32_t inner = cfg->inner_modules < M ? cfg->inner_modules : M;
  uint32_t w = cfg->inner_weight ? cfg->inner_weight : 1;
  uint32_t total = inner * w + (M - inner);
  uint32_t u = rng_below(r, total);
  if (u < inner * w) return u / w;
  return inner + (u - inner * w);
}

static inline uint32_t encode(const ctx_t* c, uint32_t m, uint32_t row, uint32_t col, uint32_t adc) {
  uint32_t rocy = row / ROC_ROWS, rloc = row % ROC_ROWS, rocx = col / ROC_COLS, cloc = col % ROC_COLS;
  uint32_t p = rocy * 8 + rocx;
  uint32_t roc = c->mod_roc[m * 16 + p], flip = c->mod_flip[m * 16 + p];
  uint32_t rr = (flip & 1) ? (ROC_ROWS - 1 - rloc) : rloc;
  uint32_t cc = (flip & 2) ? (ROC_COLS - 1 - cloc) : cloc;
  uint32_t dcol = cc >> 1, pxid = rr * 2 + (cc & 1);
  return ((uint32_t)c->mod_link[m] << 26) | (roc << 21) | (dcol << 16) | (pxid << 8) | adc;
}

static int cmp_u32(const void* a, const void* b) {
  uint32_t x = *(const uint32_t*)a, y = *(const uint32_t*)b;
  return x < y ? -1 : (x > y ? 1 : 0);
}

/* class (d): clusters on the module edges, wrap trap and cross-module trap */
static void edge_clusters(ctx_t* c, rng_t* r, uint32_t M) {
  uint32_t nmod = M < 200 ? M : 200;
  for (uint32_t i = 0; i < nmod; ++i) {
    uint32_t m = rng_below(r, M);
    short_cluster(c, r, m, 0, (int)rng_below(r, COLS));
    short_cluster(c, r, m, ROWS - 1, (int)rng_below(r, COLS));
    short_cluster(c, r, m, (int)rng_below(r, ROWS), 0);
    short_cluster(c, r, m, (int)rng_below(r, ROWS), COLS - 1);
    add_pixel(c, r, m, 0, 0); add_pixel(c, r, m, 0, COLS - 1);
    add_pixel(c, r, m, ROWS - 1, 0); add_pixel(c, r, m, ROWS - 1, COLS - 1);
    int rw = (int)rng_below(r, ROWS - 1);
    add_pixel(c, r, m, rw, COLS - 1); add_pixel(c, r, m, rw + 1, 0);            /* wrap trap */
    uint32_t m2 = (m + 1) % M; int rx = (int)rng_below(r, ROWS);
    add_pixel(c, r, m, rx, COLS - 1); add_pixel(c, r, m2, rx, 0);               /* cross-module trap */
  }
}

/* Generates one event.  words: capacity cap.  fed_offsets: [F+1].  tally: [5] = injected
 * n_empty, n_err_link, n_err_roc, n_err_dcol, n_err_pxid.  Returns n_words, or -1 on overflow. */
static int64_t gen_event(ctx_t* c, const pixgen_cfg* cfg, uint64_t seed, uint32_t* words, uint32_t* fed_offsets,
                         uint32_t* tally) {
  const uint32_t M = c->n_modules, F = c->n_feds;
  rng_t rs; rng_seed(&rs, seed ^ 0x5EEDC0DE12345678ull);
  rng_t* r = &rs;
  c->n = 0;
  memset(tally, 0, 5 * sizeof(uint32_t));

  const int degenerate = (cfg->edge_class == 5);
  uint32_t only_modules = 0; /* class e sub 3: data in only 3 modules */
  if (!(degenerate && (cfg->edge_sub == 0 || cfg->edge_sub == 1 || cfg->edge_sub == 2))) {
    if (degenerate && cfg->edge_sub == 3) only_modules = 3;
    if (cfg->clusters_per_module) {
      for (uint32_t m = 0; m < M; ++m)
        for (uint32_t k = 0; k < cfg->clusters_per_module; ++k)
          short_cluster(c, r, m, (int)rng_below(r, ROWS), (int)rng_below(r, COLS));
    } else {
      for (uint32_t k = 0; k < cfg->n_clusters; ++k) {
        uint32_t m = draw_module(cfg, r, M);
        if (only_modules) m = (m % only_modules) * (M / only_modules);
        int r0 = (int)rng_below(r, ROWS), c0 = (int)rng_below(r, COLS);
        if (cfg->long_permille && rng_below(r, 1000) < cfg->long_permille) long_cluster(c, r, m, r0, c0);
        else short_cluster(c, r, m, r0, c0);
      }
    }
    if (cfg->edge_class == 4) edge_clusters(c, r, M);
    /* G4: 1% isolated noise pixels */
    uint32_t n_noise = (c->n + 50) / 100;
    for (uint32_t k = 0; k < n_noise; ++k) {
      for (int attempt = 0; attempt < 100; ++attempt) {
        uint32_t m = rng_below(r, M);
        if (only_modules) m = (m % only_modules) * (M / only_modules);
        int row = (int)rng_below(r, ROWS), col = (int)rng_below(r, COLS), busy = 0;
        for (int dr = -1; dr <= 1 && !busy; ++dr)
          for (int dc = -1; dc <= 1; ++dc) {
            int rr = row + dr, cc = col + dc;
            if (rr < 0 || rr >= ROWS || cc < 0 || cc >= COLS) continue;
            if (occ_get(c, m, rr, cc)) { busy = 1; break; }
          }
        if (!busy) { add_pixel(c, r, m, row, col); break; }
      }
    }
    /* G7 class (a): 8 seeded modules filled with independent p = 0.10 */
    if (cfg->edge_class == 1) {
      for (int k = 0; k < 8; ++k) {
        uint32_t m = rng_below(r, M);
        for (int row = 0; row < ROWS; ++row)
          for (int col = 0; col < COLS; ++col)
            if (rng_below(r, 10) == 0) add_pixel(c, r, m, row, col);
      }
    }
  }
  if (c->n >= c->cap) { /* overflow: clean the bitmap and bail out */
    for (uint32_t i = 0; i < c->n; ++i) occ_clear(c, c->pm[i], c->pr[i], c->pc[i]);
    return -1;
  }

  /* counting sort of encoded words by module */
  memset(c->mstart, 0, sizeof(uint32_t) * ((size_t)M + 1));
  for (uint32_t i = 0; i < c->n; ++i) c->mstart[c->pm[i] + 1]++;
  for (uint32_t m = 0; m < M; ++m) c->mstart[m + 1] += c->mstart[m];
  {
    uint32_t* cursor = (uint32_t*)malloc(sizeof(uint32_t) * M);
    memcpy(cursor, c->mstart, sizeof(uint32_t) * M);
    for (uint32_t i = 0; i < c->n; ++i)
      c->wbuf[cursor[c->pm[i]]++] = encode(c, c->pm[i], c->pr[i], c->pc[i], c->pa[i]);
    free(cursor);
  }
  for (uint32_t i = 0; i < c->n; ++i) occ_clear(c, c->pm[i], c->pr[i], c->pc[i]); /* sparse clear */

  for (uint32_t m = 0; m < M; ++m) {
    uint32_t* w = c->wbuf + c->mstart[m]; uint32_t nm = c->mstart[m + 1] - c->mstart[m];
    qsort(w, nm, sizeof(uint32_t), cmp_u32);     /* read-out order: (roc, dcol, pxid) ascending */
    if (cfg->shuffle_order) shuffle_u32(r, w, nm);
  }

  /* emission: FED blocks ascending, links ascending inside a FED */
  uint32_t nw = 0; const uint32_t cap = c->cap;
  int fed_empty = (degenerate && cfg->edge_sub == 4) ? (int)rng_below(r, F) : -1;
  for (uint32_t fed = 0; fed < F; ++fed) {
    fed_offsets[fed] = nw;
    if ((int)fed == fed_empty) continue;
    for (uint32_t link = 0; link < 64; ++link) {
      const uint32_t e0 = c->entry[((size_t)fed * 64 + link) * 32];
      if (!(e0 & 1u)) continue;
      uint32_t m = (e0 >> 2) & 0xFFFF;
      const uint32_t* w = c->wbuf + c->mstart[m]; uint32_t nm = c->mstart[m + 1] - c->mstart[m];
      if (nm == 0) continue;
      uint32_t start = nw;
      if (nw + nm > cap) return -1;
      memcpy(words + nw, w, sizeof(uint32_t) * nm); nw += nm;
      if (cfg->edge_class == 2) {
        /* class (b): 2% of the run's words re-emitted verbatim and 1% re-emitted with another ADC,
         * each at a random LATER place in the same run.  c->wbuf2[p] = 1 marks inserted copies. */
        uint32_t* run = words + start; uint32_t* is_copy = c->wbuf2;
        memset(is_copy, 0, sizeof(uint32_t) * nm);
        uint32_t run_len = nm;
        for (uint32_t i = 0; i < nm; ++i) {
          uint32_t u = rng_below(r, 100);
          if (u >= 3) continue;
          if (nw + 1 > cap) return -1;
          uint32_t word = w[i];
          if (u == 2) { uint32_t a; do { a = draw_adc(r); } while (a == (word & 255u)); word = (word & ~255u) | a; }
          uint32_t pos = 0, seen = 0;            /* current position of original i */
          for (uint32_t p = 0; p < run_len; ++p) if (!is_copy[p]) { if (seen == i) { pos = p; break; } ++seen; }
          uint32_t ins = pos + 1 + rng_below(r, run_len - pos);
          memmove(run + ins + 1, run + ins, sizeof(uint32_t) * (run_len - ins));
          memmove(is_copy + ins + 1, is_copy + ins, sizeof(uint32_t) * (run_len - ins));
          run[ins] = word; is_copy[ins] = 1; ++run_len; ++nw;
        }
      }
    }
  }
  fed_offsets[F] = nw;

  if (degenerate && cfg->edge_sub == 1) { /* exactly one word */
    uint32_t m = rng_below(r, M);
    uint32_t f = c->mod_fed[m];
    words[0] = encode(c, m, rng_below(r, ROWS), rng_below(r, COLS), 200);
    nw = 1;
    for (uint32_t fed = 0; fed <= F; ++fed) fed_offsets[fed] = fed <= f ? 0 : 1;
  }

  /* class (c) and class (e) sub 2: invalid words */
  if (cfg->edge_class == 3 || (degenerate && cfg->edge_sub == 2)) {
    if (degenerate) { /* only undecodable words: 500 of them spread over the FEDs */
      nw = 0;
      for (uint32_t fed = 0; fed < F; ++fed) { fed_offsets[fed] = nw; for (int k = 0; k < 16 && nw < cap; ++k) words[nw++] = 1; }
      fed_offsets[F] = nw;
    }
    uint32_t fed = 0;
    for (uint32_t i = 0; i < nw; ++i) {
      while (fed + 1 <= F && i >= fed_offsets[fed + 1]) ++fed;
      uint32_t u = degenerate ? rng_below(r, 35) : rng_below(r, 1000);
      if (u >= 35) continue;
      /* a mapped link of this FED, for the classes that need one */
      uint32_t mapped_link = 0;
      for (uint32_t tries = 0; tries < 64; ++tries) { mapped_link = rng_below(r, 64); if (c->entry[((size_t)fed * 64 + mapped_link) * 32] & 1u) break; }
      if (!(c->entry[((size_t)fed * 64 + mapped_link) * 32] & 1u)) for (mapped_link = 0; mapped_link < 64; ++mapped_link) if (c->entry[((size_t)fed * 64 + mapped_link) * 32] & 1u) break;
      uint32_t cls = u < 30 ? (u & 3) : 4; /* 3%: four error classes in equal shares; 0.5%: zero word */
      if (cls == 0 && c->n_unmapped[fed] == 0) cls = 1;
      uint32_t w = 0;
      switch (cls) {
        case 0: w = ((uint32_t)c->link_unmapped[fed * 64 + rng_below(r, c->n_unmapped[fed])] << 26) | (rng_u32(r) & 0x03FFFFFFu); if (w == 0) w = 1; tally[1]++; break;
        case 1: w = (mapped_link << 26) | ((16 + rng_below(r, 16)) << 21) | (rng_u32(r) & 0x001FFFFFu); tally[2]++; break;
        case 2: w = (mapped_link << 26) | (rng_below(r, 16) << 21) | ((26 + rng_below(r, 6)) << 16) | (rng_u32(r) & 0xFFFFu); tally[3]++; break;
        case 3: w = (mapped_link << 26) | (rng_below(r, 16) << 21) | (rng_below(r, 26) << 16) | ((160 + rng_below(r, 96)) << 8) | (rng_u32(r) & 0xFFu); tally[4]++; break;
        default: w = 0; tally[0]++; break;
      }
      words[i] = w;
    }
  }
  return (int64_t)nw;
}

/* ---------------------------------------------------------------- C API */
/* Upper bound on words per event used for the internal pixel buffer. */
#define PIXGEN_EVENT_CAP (1u << 20)

/* One event.  Returns n_words (<= cap) or a negative code. */
int64_t pixgen_event(const pixgen_cfg* cfg, uint32_t n_feds, uint32_t n_modules, const uint32_t* entry,
                     uint64_t seed, uint32_t* words, uint32_t cap, uint32_t* fed_offsets, uint32_t* tally) {
  ctx_t c;
  if (ctx_init(&c, n_feds, n_modules, entry, PIXGEN_EVENT_CAP) != 0) { ctx_free(&c); return -2; }
  uint32_t* tmp = (uint32_t*)malloc(sizeof(uint32_t) * PIXGEN_EVENT_CAP);
  int64_t n = gen_event(&c, cfg, seed, tmp, fed_offsets, tally);
  if (n > (int64_t)cap) n = -1;
  if (n > 0) memcpy(words, tmp, sizeof(uint32_t) * (size_t)n);
  free(tmp); ctx_free(&c);
  return n;
}

/* A batch of events, one per (cfgs[e], seeds[e]), generated in parallel (OpenMP), concatenated.
 * words: capacity cap_total.  event_offsets: [E+1].  fed_offsets: [E*(F+1)] event-relative.
 * tally: [E*5].  Returns total words or a negative code. */
int64_t pixgen_batch(const pixgen_cfg* cfgs, const uint64_t* seeds, uint32_t n_events, uint32_t n_feds,
                     uint32_t n_modules, const uint32_t* entry, uint32_t* words, uint64_t cap_total,
                     uint32_t* event_offsets, uint32_t* fed_offsets, uint32_t* tally) {
  uint32_t** bufs = (uint32_t**)calloc(n_events, sizeof(uint32_t*));
  int64_t* ns = (int64_t*)calloc(n_events, sizeof(int64_t));
  int fail = 0;
#pragma omp parallel
  {
    ctx_t c; int ok = ctx_init(&c, n_feds, n_modules, entry, PIXGEN_EVENT_CAP) == 0;
    uint32_t* tmp = (uint32_t*)malloc(sizeof(uint32_t) * PIXGEN_EVENT_CAP);
#pragma omp for schedule(dynamic, 1)
    for (uint32_t e = 0; e < n_events; ++e) {
      if (!ok || !tmp) { ns[e] = -2; continue; }
      int64_t n = gen_event(&c, &cfgs[e], seeds[e], tmp, fed_offsets + (size_t)e * (n_feds + 1), tally + (size_t)e * 5);
      ns[e] = n;
      if (n > 0) { bufs[e] = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)n); if (bufs[e]) memcpy(bufs[e], tmp, sizeof(uint32_t) * (size_t)n); else ns[e] = -2; }
    }
    free(tmp); ctx_free(&c);
  }
  uint64_t total = 0;
  for (uint32_t e = 0; e < n_events; ++e) { if (ns[e] < 0) fail = 1; else total += (uint64_t)ns[e]; }
  int64_t ret;
  if (fail) ret = -2;
  else if (total > cap_total || total > 0xFFFFFFFFull) ret = -1;
  else {
    uint64_t off = 0;
    for (uint32_t e = 0; e < n_events; ++e) {
      event_offsets[e] = (uint32_t)off;
      if (ns[e] > 0) memcpy(words + off, bufs[e], sizeof(uint32_t) * (size_t)ns[e]);
      off += (uint64_t)ns[e];
    }
    event_offsets[n_events] = (uint32_t)off;
    ret = (int64_t)total;
  }
  for (uint32_t e = 0; e < n_events; ++e) free(bufs[e]);
  free(bufs); free(ns);
  return ret;
}

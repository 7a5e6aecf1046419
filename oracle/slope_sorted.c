/* INDEPENDENT SECOND CPU IMPLEMENTATION -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A pin for oracle/cbm_oracle.c ("agreement with an independent slope-binned CPU
 * count", BASELINE.json north_star).  It reaches the same
 * integers by a different route, so that a mistake in either shows up as a
 * disagreement:
 *   - layers 0 and 2 of a station are SORTED by x (within one layer z is constant,
 *     so x order is slope order), and the x-window of a hit is located by binary
 *     search instead of being tested pair by pair;
 *   - the window test uses the per-layer-pair integer threshold
 *     T_AB = floor(a*z_A*z_B / b) and |D| <= T_AB (reading R4) instead of
 *     the oracle's b*|D| <= a*z_A*z_B;
 *   - the search is centred on the middle-layer hit, and linking runs over distinct
 *     middle hits with multiplicities m_s[h1] (reading R8) instead of over
 *     one list entry per triplet.
 * It also returns N_eval, the number of algorithmic window evaluations of this
 * canonical sorted search, used for the integer-pipe roofline:
 * one per (h0,h1) pair inside the x-band, two per h2 inside the x-band of both hits of a
 * pair that passed in y, two per pair of middle hits with triplets of consecutive
 * stations.  (Reading: the canonical search links distinct middle hits,
 * so the link term counts middle hits, not triplets.)  Pinned by hand counts in
 * tests/test_oracle_pins.py::test_n_eval_hand_counts.
 *
 * Follows PAPER.md:73-76, 88 (section 3.2 steps 1-3) with the north_star's window and
 * linking; shares no code with the oracle or with the CUDA path.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define SS_MAX_LAYERS 24
#define SS_SAT 0xFFFFFFFFULL

typedef struct {
  uint32_t n_stations;
  int32_t  layer_z[SS_MAX_LAYERS];
  uint32_t win_in_num, win_in_den;
  uint32_t win_link_num, win_link_den;
  uint32_t min_candidates;
} ss_geometry_t;

typedef struct { int32_t x, y; } hit_t;

static int cmp_hit_x(const void* p, const void* q) {
  const hit_t* a = (const hit_t*)p; const hit_t* b = (const hit_t*)q;
  return (a->x > b->x) - (a->x < b->x);
}

/* first index i in sorted h[0..n) with h[i].x * zo - xr * zs >= lo_bound */
static uint32_t lower_idx(const hit_t* h, uint32_t n, int64_t zs, int64_t xr, int64_t zo, int64_t bound) {
  /* D(i) = h[i].x*zo - xr*zs is non-decreasing in i; find first i with D(i) >= bound */
  uint32_t lo = 0, hi = n;
  while (lo < hi) {
    uint32_t mid = lo + (hi - lo) / 2;
    int64_t D = (int64_t)h[mid].x * zo - xr * zs;
    if (D >= bound) hi = mid; else lo = mid + 1;
  }
  return lo;
}

static inline int64_t absd(int64_t v) { return v < 0 ? -v : v; }
static inline uint64_t clampsat(uint64_t v) { return v > SS_SAT ? SS_SAT : v; }

typedef struct { int32_t x, y; uint64_t m, c; } mid_t;

static int ss_event(const ss_geometry_t* G, const int32_t* x, const int32_t* y, const uint32_t* off_ev,
                    uint32_t* n_triplets, uint32_t* n_candidates, uint8_t* accept, uint64_t* n_eval) {
  const uint32_t S = G->n_stations;
  mid_t* prev = NULL; size_t n_prev = 0;
  uint64_t evals = 0;
  int dead = 0; /* some station had no triplet: candidates = 0, but triplet counts still needed */
  for (uint32_t s = 0; s < S; ++s) {
    const int64_t z0 = G->layer_z[3 * s], z1 = G->layer_z[3 * s + 1], z2 = G->layer_z[3 * s + 2];
    const uint32_t b0 = off_ev[3 * s], b1 = off_ev[3 * s + 1], b2 = off_ev[3 * s + 2], b3 = off_ev[3 * s + 3];
    const uint32_t n0 = b1 - b0, n1 = b2 - b1, n2 = b3 - b2;
    const int64_t a = G->win_in_num, b = G->win_in_den;
    const int64_t T01 = (a * z0 * z1) / b, T02 = (a * z0 * z2) / b, T12 = (a * z1 * z2) / b;
    hit_t* h0 = (hit_t*)malloc((n0 + 1) * sizeof(hit_t));
    hit_t* h2 = (hit_t*)malloc((n2 + 1) * sizeof(hit_t));
    mid_t* cur = (mid_t*)malloc((n1 + 1) * sizeof(mid_t));
    if (!h0 || !h2 || !cur) { free(h0); free(h2); free(cur); free(prev); return -2; }
    for (uint32_t i = 0; i < n0; ++i) { h0[i].x = x[b0 + i]; h0[i].y = y[b0 + i]; }
    for (uint32_t i = 0; i < n2; ++i) { h2[i].x = x[b2 + i]; h2[i].y = y[b2 + i]; }
    qsort(h0, n0, sizeof(hit_t), cmp_hit_x);
    qsort(h2, n2, sizeof(hit_t), cmp_hit_x);
    size_t n_cur = 0;
    uint64_t station_total = 0;
    for (uint32_t i1 = b1; i1 < b2; ++i1) {
      const int64_t x1 = x[i1], y1 = y[i1];
      /* h0 with |x0*z1 - x1*z0| <= T01 : contiguous range of the sorted layer */
      uint32_t lo0 = lower_idx(h0, n0, z0, x1, z1, -T01);
      uint32_t hi0 = lower_idx(h0, n0, z0, x1, z1, T01 + 1);
      /* h2 with |x2*z1 - x1*z2| <= T12 */
      uint32_t lo2 = lower_idx(h2, n2, z2, x1, z1, -T12);
      uint32_t hi2 = lower_idx(h2, n2, z2, x1, z1, T12 + 1);
      uint64_t m = 0;
      for (uint32_t i = lo0; i < hi0; ++i) {
        ++evals; /* y evaluation of the (h0,h1) pair */
        if (absd((int64_t)h0[i].y * z1 - y1 * z0) > T01) continue;
        /* h2 in the x-band of both h1 (above) and h0 */
        uint32_t lo = lower_idx(h2, n2, z2, h0[i].x, z0, -T02);
        uint32_t hi = lower_idx(h2, n2, z2, h0[i].x, z0, T02 + 1);
        if (lo < lo2) lo = lo2;
        if (hi > hi2) hi = hi2;
        for (uint32_t k = lo; k < hi; ++k) {
          evals += 2;
          if (absd((int64_t)h2[k].y * z1 - y1 * z2) <= T12 &&
              absd((int64_t)h2[k].y * z0 - (int64_t)h0[i].y * z2) <= T02) ++m;
        }
      }
      if (m) { cur[n_cur].x = (int32_t)x1; cur[n_cur].y = (int32_t)y1; cur[n_cur].m = m; cur[n_cur].c = 0; ++n_cur; }
      station_total += m; /* m <= n0*n2 < 2^64 / n1 for any batch with < 2^32 hits */
    }
    n_triplets[s] = (uint32_t)clampsat(station_total);
    /* chain counts over distinct middle hits with multiplicity */
    if (s == 0) {
      for (size_t u = 0; u < n_cur; ++u) cur[u].c = clampsat(cur[u].m);
    } else if (!dead) {
      const int64_t zA = G->layer_z[3 * (s - 1) + 1], zB = z1;
      const int64_t TL = ((int64_t)G->win_link_num * zA * zB) / (int64_t)G->win_link_den;
      for (size_t u = 0; u < n_cur; ++u) {
        uint64_t acc = 0;
        for (size_t t = 0; t < n_prev; ++t) {
          evals += 2;
          if (absd((int64_t)prev[t].x * zB - (int64_t)cur[u].x * zA) <= TL &&
              absd((int64_t)prev[t].y * zB - (int64_t)cur[u].y * zA) <= TL)
            acc = clampsat(acc + prev[t].c);
        }
        cur[u].c = clampsat(clampsat(cur[u].m) * acc); /* both factors <= 2^32-1: no overflow */
      }
    }
    if (n_cur == 0) dead = 1;
    free(h0); free(h2); free(prev);
    prev = cur; n_prev = n_cur;
  }
  uint64_t total = 0;
  if (!dead) for (size_t u = 0; u < n_prev; ++u) total = clampsat(total + prev[u].c);
  free(prev);
  *n_candidates = (uint32_t)total;
  *accept = total >= G->min_candidates ? 1 : 0;
  *n_eval += evals;
  return 0;
}

/* Events [e_begin, e_end); outputs relative to e_begin; *n_eval accumulates window evaluations. */
int cbm_slope_sorted_run(const ss_geometry_t* G, const int32_t* x, const int32_t* y, const uint32_t* off,
                         uint64_t e_begin, uint64_t e_end,
                         uint32_t* n_triplets, uint32_t* n_candidates, uint8_t* accept, uint64_t* n_eval) {
  if (!G || !off || !n_triplets || !n_candidates || !accept || !n_eval) return -1;
  if (G->n_stations < 1 || G->n_stations > SS_MAX_LAYERS / 3) return -1;
  if (G->win_in_den == 0 || G->win_link_den == 0) return -1;
  const uint32_t S = G->n_stations, L = 3 * S;
  *n_eval = 0;
  for (uint64_t e = e_begin; e < e_end; ++e) {
    int rc = ss_event(G, x, y, off + e * L, n_triplets + (e - e_begin) * S, n_candidates + (e - e_begin),
                      accept + (e - e_begin), n_eval);
    if (rc) return rc;
  }
  return 0;
}

/* Seeded synthetic MUCH-hit generator (input generator ONLY).
 *
 * This file holds none of the trigger's arithmetic: no window test, no triplet
 * search, no linking.  It only draws hits.  It is the one module that both the
 * CUDA path's tests/bench and the CPU oracle's tests consume (through its
 * outputs: x[], y[], off[]).
 *
 * What it stands in for: the paper's simulated samples D1-D3 (PLUTO J/psi,
 * UrQMD central Au+Au, GEANT transport; section 3.3), which do
 * not exist in this repository.  Shapes follow BASELINE.json `configs` and the
 * readings R13-R18 of SURVEY.md section 8(c); the recipe is restated in
 * DESIGN.md section "Input recipe".
 *
 * Output layout (one CSR-SoA record per batch):
 *   off[e*L + l]  = index of the first hit of event e, layer l (L = 3*S)
 *   off[E*L]      = total number of hits
 *   x[i], y[i]    = int32 coordinates in 10-um units (1 cm = 1000 units)
 *
 * Reproducibility: every event k owns a private splitmix64 stream keyed by
 * (seed, first_event + k), so any chunking / thread count gives identical data.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define CBM_GEN_MAX_LAYERS 24

typedef struct {
  uint32_t struct_size;
  uint32_t n_stations;          /* S, layers = 3*S                                  */
  int32_t  layer_z[CBM_GEN_MAX_LAYERS]; /* 10-um units                              */
  uint32_t occupancy_mode;      /* 0: fixed mean_a; 1: log-normal(median mean_a, sigma mean_b);
                                   2: mixture: frac_b of events use mean_b, others mean_a */
  uint32_t max_bg_per_layer;    /* hard clamp of the background count per layer      */
  double   mean_a;
  double   mean_b;
  double   frac_b;
  double   mean_clamp;          /* clamp of the per-event mean in mode 1 (R14)       */
  double   half_aperture;       /* background uniform in |x|,|y| <= half_aperture*z  */
  double   signal_fraction;     /* Bernoulli per event                               */
  double   vertex_sigma_cm;     /* one vertex per event, shared by both muons (R16)  */
  double   signal_slope_max;    /* |tx|,|ty| <= this, uniform                        */
  double   smear_sigma_cm;      /* per-layer Gaussian smear                          */
  double   layer_efficiency;    /* per-layer hit probability of a signal track       */
} cbm_gen_params_t;

/* ---- counter-based RNG: splitmix64 stream per event ---------------------- */
typedef struct { uint64_t s; } rng_t;

static inline uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
static inline void rng_seed(rng_t* r, uint64_t seed, uint64_t event) {
  r->s = mix64(mix64(seed + 0x9E3779B97F4A7C15ULL) ^ (event * 0xD1342543DE82EF95ULL + 0x2545F4914F6CDD1DULL));
}
static inline uint64_t rng_next(rng_t* r) {
  r->s += 0x9E3779B97F4A7C15ULL;
  return mix64(r->s);
}
static inline double rng_uniform(rng_t* r) { /* [0,1) with 53 bits */
  return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0);
}
static inline double rng_gauss(rng_t* r) { /* Box-Muller, one value per call */
  double u1 = 1.0 - rng_uniform(r); /* (0,1] */
  double u2 = rng_uniform(r);
  return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925 * u2);
}
static uint32_t rng_poisson(rng_t* r, double lambda) {
  /* exact: sum of k independent Poisson(lambda/k), lambda/k <= 64, each by CDF inversion */
  if (!(lambda > 0.0)) return 0;
  uint32_t k = (uint32_t)ceil(lambda / 64.0);
  double lc = lambda / (double)k;
  double p0 = exp(-lc);
  uint32_t total = 0;
  for (uint32_t c = 0; c < k; ++c) {
    double u = rng_uniform(r);
    double p = p0, F = p0;
    uint32_t n = 0;
    while (u > F && n < 2000) {
      ++n;
      p *= lc / (double)n;
      F += p;
    }
    total += n;
  }
  return total;
}

/* ---- per-event header: everything that fixes the hit counts -------------- */
typedef struct {
  uint32_t n_bg[CBM_GEN_MAX_LAYERS];
  uint32_t n_sig[CBM_GEN_MAX_LAYERS];
  int32_t  sig_x[CBM_GEN_MAX_LAYERS][2];
  int32_t  sig_y[CBM_GEN_MAX_LAYERS][2];
  uint8_t  truth; /* bit0: signal pair planted; bit1: both tracks hit every layer; bit2: mode-2 class b */
} header_t;

static inline int32_t to_units(double cm) { return (int32_t)nearbyint(cm * 1000.0); }

static void gen_header(const cbm_gen_params_t* P, rng_t* r, header_t* H) {
  const uint32_t L = 3 * P->n_stations;
  /* fixed draw order, independent of the configuration */
  double u_class = rng_uniform(r);
  double g_occ   = rng_gauss(r);
  double u_sig   = rng_uniform(r);
  double lambda  = P->mean_a;
  H->truth = 0;
  if (P->occupancy_mode == 1) {
    lambda = exp(log(P->mean_a) + P->mean_b * g_occ);
    if (lambda > P->mean_clamp) lambda = P->mean_clamp;
  } else if (P->occupancy_mode == 2) {
    if (u_class < P->frac_b) { lambda = P->mean_b; H->truth |= 4; }
  }
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t n = rng_poisson(r, lambda);
    if (n > P->max_bg_per_layer) n = P->max_bg_per_layer;
    H->n_bg[l] = n;
    H->n_sig[l] = 0;
  }
  int planted = (u_sig < P->signal_fraction);
  if (planted) {
    H->truth |= 1;
    double vx = P->vertex_sigma_cm * rng_gauss(r);
    double vy = P->vertex_sigma_cm * rng_gauss(r);
    int all_layers = 1;
    for (int t = 0; t < 2; ++t) {
      double tx = (2.0 * rng_uniform(r) - 1.0) * P->signal_slope_max;
      double ty = (2.0 * rng_uniform(r) - 1.0) * P->signal_slope_max;
      for (uint32_t l = 0; l < L; ++l) {
        double u_eff = rng_uniform(r);
        double gx = rng_gauss(r), gy = rng_gauss(r);
        if (u_eff < P->layer_efficiency) {
          double z_cm = (double)P->layer_z[l] / 1000.0;
          uint32_t k = H->n_sig[l]++;
          H->sig_x[l][k] = to_units(vx + tx * z_cm + P->smear_sigma_cm * gx);
          H->sig_y[l][k] = to_units(vy + ty * z_cm + P->smear_sigma_cm * gy);
        } else {
          all_layers = 0;
        }
      }
    }
    if (all_layers) H->truth |= 2;
  }
}

static void gen_body(const cbm_gen_params_t* P, rng_t* r, const header_t* H,
                     const uint32_t* off_ev, int32_t* x, int32_t* y) {
  const uint32_t L = 3 * P->n_stations;
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t base = off_ev[l];
    double half = P->half_aperture * (double)P->layer_z[l]; /* in units */
    uint32_t n = H->n_bg[l];
    for (uint32_t i = 0; i < n; ++i) {
      double ux = rng_uniform(r), uy = rng_uniform(r);
      x[base + i] = (int32_t)nearbyint((2.0 * ux - 1.0) * half);
      y[base + i] = (int32_t)nearbyint((2.0 * uy - 1.0) * half);
    }
    /* signal hits: append, then move to a uniformly random position (background hits
       are exchangeable, so this equals a full Fisher-Yates shuffle in distribution) */
    for (uint32_t k = 0; k < H->n_sig[l]; ++k) {
      uint32_t pos = n + k;
      uint32_t j = (uint32_t)(rng_uniform(r) * (double)(pos + 1));
      if (j > pos) j = pos;
      x[base + pos] = x[base + j];
      y[base + pos] = y[base + j];
      x[base + j] = H->sig_x[l][k];
      y[base + j] = H->sig_y[l][k];
    }
  }
}

/* ---- threaded drivers ---------------------------------------------------- */
typedef struct {
  const cbm_gen_params_t* P;
  uint64_t seed, first_event;
  uint32_t e0, e1;
  uint32_t* off;      /* pass 1: counts written to off[e*L+l+1]; pass 2: read-only offsets */
  int32_t *x, *y;
  uint8_t* truth;
  int pass;
} job_t;

static void* worker(void* arg) {
  job_t* J = (job_t*)arg;
  const uint32_t L = 3 * J->P->n_stations;
  header_t H;
  rng_t r;
  for (uint32_t e = J->e0; e < J->e1; ++e) {
    rng_seed(&r, J->seed, J->first_event + e);
    gen_header(J->P, &r, &H);
    if (J->pass == 1) {
      for (uint32_t l = 0; l < L; ++l) J->off[(size_t)e * L + l + 1] = H.n_bg[l] + H.n_sig[l];
      if (J->truth) J->truth[e] = H.truth;
    } else {
      gen_body(J->P, &r, &H, J->off + (size_t)e * L, J->x, J->y);
    }
  }
  return NULL;
}

static int run_jobs(const cbm_gen_params_t* P, uint64_t seed, uint64_t first_event, uint32_t n_events,
                    uint32_t* off, int32_t* x, int32_t* y, uint8_t* truth, int pass, int n_threads) {
  if (n_threads < 1) n_threads = 1;
  if (n_threads > 256) n_threads = 256;
  if ((uint32_t)n_threads > n_events) n_threads = n_events ? (int)n_events : 1;
  pthread_t th[256];
  job_t jobs[256];
  /* many small contiguous chunks per thread would balance better, but events are iid */
  for (int t = 0; t < n_threads; ++t) {
    jobs[t].P = P; jobs[t].seed = seed; jobs[t].first_event = first_event;
    jobs[t].e0 = (uint32_t)((uint64_t)n_events * t / n_threads);
    jobs[t].e1 = (uint32_t)((uint64_t)n_events * (t + 1) / n_threads);
    jobs[t].off = off; jobs[t].x = x; jobs[t].y = y; jobs[t].truth = truth; jobs[t].pass = pass;
  }
  if (n_threads == 1) { worker(&jobs[0]); return 0; }
  for (int t = 0; t < n_threads; ++t)
    if (pthread_create(&th[t], NULL, worker, &jobs[t]) != 0) return -1;
  for (int t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
  return 0;
}

static int check_params(const cbm_gen_params_t* P) {
  if (!P || P->struct_size != sizeof(cbm_gen_params_t)) return -1;
  if (P->n_stations < 1 || P->n_stations > 8) return -1;
  return 0;
}

/* Pass 1: fills off[0 .. n_events*L] (prefix sums) and optional truth[n_events].
 * Returns the total number of hits, or UINT64_MAX on error. */
uint64_t cbm_gen_offsets(const cbm_gen_params_t* P, uint64_t seed, uint64_t first_event,
                         uint32_t n_events, uint32_t* off, uint8_t* truth, int n_threads) {
  if (check_params(P) || !off) return UINT64_MAX;
  const uint32_t L = 3 * P->n_stations;
  off[0] = 0;
  if (run_jobs(P, seed, first_event, n_events, off, NULL, NULL, truth, 1, n_threads)) return UINT64_MAX;
  uint64_t acc = 0;
  const size_t n = (size_t)n_events * L;
  for (size_t i = 1; i <= n; ++i) {
    acc += off[i];
    if (acc > 0xFFFFFFFFULL) return UINT64_MAX;
    off[i] = (uint32_t)acc;
  }
  return acc;
}

/* Pass 2: fills x[], y[] (each off[n_events*L] entries) for the offsets of pass 1. */
int cbm_gen_hits(const cbm_gen_params_t* P, uint64_t seed, uint64_t first_event, uint32_t n_events,
                 const uint32_t* off, int32_t* x, int32_t* y, int n_threads) {
  if (check_params(P) || !off || !x || !y) return -1;
  return run_jobs(P, seed, first_event, n_events, (uint32_t*)off, x, y, NULL, 2, n_threads);
}

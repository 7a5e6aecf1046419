/* ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * The paper's own selection, literally (section 3.2):
 *   step 1  "Create all possible triplets of hits in the trigger station, with one hit from
 *           each layer."
 *   step 2a  "Fit the hits of the triplet plus the event vertex (0, 0) by a straight line in both
 *           the x-z (bending) plane and the y-z (non-bending) plane, i.e., x = m0 z and y = m1 z."
 *   step 2b  "Compute the Mean Square Deviation (MSD) of the triplet fit.  A triplet is rejected
 *           if the MSD (per degree of freedom) is above a threshold (0.03 for MSD_xz, 0.025 for MSD_yz)."
 *   step 3  "Select the event if it contains at least two triplets passing the MSD cut."
 *
 * Written out: the least-squares line through the origin has m0 = Sxz / Szz with Sxz = sum x_i z_i and
 * Szz = sum z_i^2 over the three hits (the vertex (0,0) lies on every such line and adds nothing to either sum),
 * the sum of squared residuals is  sum (x_i - m0 z_i)^2 = Sxx - Sxz^2 / Szz,  and the cut
 *       (Sxx - Sxz^2/Szz) / ndf  <=  thr
 * is, multiplied by Szz > 0 and with thr = num/den cm^2 = num * 10^6 / den in squared 10-um units,
 *       den * (Szz*Sxx - Sxz^2)  <=  num * 1000000 * ndf * Szz                       (exact, 128-bit integers).
 * Readings (R2, B8): residuals in cm (thresholds in cm^2), ndf = 2 (three hits, one fitted slope; the
 * vertex is a constraint) unless the caller says 3; the cut is closed (<=); the trigger station is the last one
 * unless the caller names another.  The paper's implementation is floating point with unstated precision; this
 * oracle evaluates the same inequality exactly, so exactly one answer is right.
 *
 * Pins (tests/test_msd_mode.py): hand-computed residuals (z = k, 2k, 3k; x = 0, 0, d: SSR = 5 d^2 / 14, so with
 * ndf 2 and 0.03 cm^2 d = 409 passes and d = 410 fails), exact lines (SSR = 0), an independent evaluation with
 * Python fractions on tiny events, float64 numpy least squares on random triplets away from the threshold,
 * permutation invariance, and the n0*n1*n2 closed form when every triplet passes.
 */
#include <stdint.h>

#define ORACLE_MAX_LAYERS 24
#define ORACLE_SAT 0xFFFFFFFFULL

typedef struct {
  uint32_t n_stations;
  int32_t  layer_z[ORACLE_MAX_LAYERS];
  uint32_t station;                 /* the trigger station */
  uint32_t thr_x_num, thr_x_den;    /* MSD_xz threshold in cm^2 as a rational */
  uint32_t thr_y_num, thr_y_den;    /* MSD_yz threshold */
  uint32_t ndf;                     /* degrees of freedom the sum of squares is divided by */
  uint32_t min_triplets;            /* select iff this many triplets pass (2) */
} msd_params_t;

typedef unsigned __int128 u128;

/* den * (Szz*Svv - Svz^2) <= num * 10^6 * ndf * Szz */
static int msd_ok(const int64_t v[3], const int64_t z[3], uint32_t num, uint32_t den, uint32_t ndf) {
  int64_t svz = 0, szz = 0, svv = 0;
  for (int i = 0; i < 3; ++i) {
    svz += v[i] * z[i];
    szz += z[i] * z[i];
    svv += v[i] * v[i];
  }
  const u128 a = (u128)(uint64_t)szz * (u128)(uint64_t)svv;
  const u128 b = (u128)(uint64_t)(svz < 0 ? -svz : svz) * (u128)(uint64_t)(svz < 0 ? -svz : svz);
  const u128 lhs = (u128)den * (a - b);                              /* a >= b (Cauchy-Schwarz) */
  const u128 rhs = (u128)num * (u128)1000000u * (u128)ndf * (u128)(uint64_t)szz;
  return lhs <= rhs;
}

/* events [e_begin, e_end): n_passing[e - e_begin] = min(2^32-1, passing triplets), accept = n_passing >= min */
int cbm_msd_oracle_run(const msd_params_t* p, const int32_t* x, const int32_t* y, const uint32_t* off,
                       uint64_t e_begin, uint64_t e_end, uint32_t* n_passing, uint8_t* accept) {
  if (!p || p->n_stations < 1 || 3 * p->n_stations > ORACLE_MAX_LAYERS || p->station >= p->n_stations ||
      p->thr_x_den == 0 || p->thr_y_den == 0 || p->ndf == 0)
    return -1;
  const uint64_t L = 3ull * p->n_stations;
  const int64_t z[3] = {p->layer_z[3 * p->station], p->layer_z[3 * p->station + 1], p->layer_z[3 * p->station + 2]};
  for (uint64_t e = e_begin; e < e_end; ++e) {
    const uint32_t* o = off + e * L + 3ull * p->station;
    uint64_t n = 0;
    for (uint32_t i0 = o[0]; i0 < o[1]; ++i0)
      for (uint32_t i1 = o[1]; i1 < o[2]; ++i1)
        for (uint32_t i2 = o[2]; i2 < o[3]; ++i2) {
          const int64_t vx[3] = {x[i0], x[i1], x[i2]}, vy[3] = {y[i0], y[i1], y[i2]};
          if (msd_ok(vx, z, p->thr_x_num, p->thr_x_den, p->ndf) && msd_ok(vy, z, p->thr_y_num, p->thr_y_den, p->ndf)) ++n;
        }
    const uint32_t c = n > ORACLE_SAT ? (uint32_t)ORACLE_SAT : (uint32_t)n;
    n_passing[e - e_begin] = c;
    accept[e - e_begin] = c >= p->min_triplets ? 1 : 0;
  }
  return 0;
}

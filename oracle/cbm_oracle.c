/* ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU statement of what the hot path computes:
 * the first-level J/psi event selection in the CBM muon chambers, as nested
 * loops over hit combinations.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call it.  It shares no
 * code with the CUDA path (paper_1810_11966_b200/csrc) and never will.
 *
 * What it follows
 *   PAPER.md:73      (section 3.2 step 1)  "Create all possible triplets of hits
 *                    ..., with one hit from each layer."
 *   PAPER.md:75-76   (step 2)  each triplet plus the event vertex (0,0) must lie
 *                    on a straight line through the target in the x-z and the
 *                    y-z plane.  The paper's floating-point MSD cut is replaced,
 *                    as BASELINE.json's north_star fixes, by an exact integer
 *                    slope window (readings R2-R5).
 *   PAPER.md:88      (step 3)  "Select the event if it contains at least two
 *                    triplets passing the ... cut" -- generalised by north_star
 *                    to >= 2 candidates linked across all stations (R1, R8, R9).
 *
 * Definition:
 *   compat(h in layer A, g in layer B; a/b)
 *        :=  b*|x_h*z_B - x_g*z_A| <= a*z_A*z_B  and  b*|y_h*z_B - y_g*z_A| <= a*z_A*z_B
 *   T_s  := { (h0,h1,h2) in H_{s,0} x H_{s,1} x H_{s,2} : all three pairs compat under w_in }
 *   link(t in T_s, u in T_{s+1}) := compat(t.h1, u.h1; w_link)          (middle-layer hits)
 *   candidates := number of tuples (t_0..t_{S-1}), t_s in T_s, consecutive ones linked
 *   outputs: n_triplets[e*S+s] = min(2^32-1, |T_s|), n_candidates[e] = min(2^32-1, candidates),
 *            accept[e] = n_candidates[e] >= min_candidates
 *
 * All arithmetic is integer (int64 / uint64, the window products in 128 bits); there is no floating point, no sorting, no
 * blocking.  The only shortcut is the (h0,h1) short-circuit before the h2 loop.
 *
 * Pins (tests/test_oracle_pins.py): brute force without any short-circuit and with
 * explicit S-tuple enumeration (oracle/brute_force.py) on tiny events; hand-computed
 * boundary-equality cases; planted exact lines; narrow-cone closed form
 * (|T_s| = n0*n1*n2, candidates = prod |T_s|, saturation); permutation invariance;
 * zero on constructed non-collinear noise; the independent slope-sorted counter
 * (oracle/slope_sorted.c); the closed-form uniform-background triplet rate.
 * The paper's literal MSD cut is a separate oracle: oracle/msd_oracle.c.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_MAX_LAYERS 24
#define ORACLE_SAT 0xFFFFFFFFULL

typedef struct {
  uint32_t n_stations;                     /* S */
  int32_t  layer_z[ORACLE_MAX_LAYERS];     /* z of layer 3*s+l, 10-um units */
  uint32_t win_in_num, win_in_den;         /* a/b of the in-station window  */
  uint32_t win_link_num, win_link_den;     /* a/b of the cross-station window */
  uint32_t min_candidates;
} oracle_geometry_t;

static int64_t iabs64(int64_t v) { return v < 0 ? -v : v; }

/* compat(): |x_h/z_A - x_g/z_B| <= a/b and the same in y, cross-multiplied (z > 0).
 * The products b*|D| are formed in 128 bits so that the definition holds for every int32 coordinate
 * (|D| < 2^56, b <= 2^12; reading B2), not only for |x|, |y| <= 2^23. */
static int compat(int64_t xh, int64_t yh, int64_t zA, int64_t xg, int64_t yg, int64_t zB,
                  int64_t a, int64_t b) {
  __int128 rhs = (__int128)a * zA * zB;
  if ((__int128)b * iabs64(xh * zB - xg * zA) > rhs) return 0;
  if ((__int128)b * iabs64(yh * zB - yg * zA) > rhs) return 0;
  return 1;
}

static uint64_t sat_add(uint64_t p, uint64_t q) {
  uint64_t r = p + q;
  return r > ORACLE_SAT ? ORACLE_SAT : r;
}

typedef struct { uint32_t* v; size_t n, cap; } list_t;

static int list_push(list_t* l, uint32_t v, size_t max_entries) {
  if (l->n == l->cap) {
    size_t nc = l->cap ? 2 * l->cap : 64;
    if (nc > max_entries) nc = max_entries;
    if (l->n >= nc) return -1;
    uint32_t* p = (uint32_t*)realloc(l->v, nc * sizeof(uint32_t));
    if (!p) return -1;
    l->v = p; l->cap = nc;
  }
  l->v[l->n++] = v;
  return 0;
}

/* One event.  off_ev points at the event's L+1 offsets (off_ev[l] .. off_ev[l+1]).
 * Returns 0, or -2 if a triplet list would exceed max_list_entries (oracle limit). */
static int oracle_event(const oracle_geometry_t* G, const int32_t* x, const int32_t* y,
                        const uint32_t* off_ev, size_t max_list_entries,
                        uint32_t* n_triplets, uint32_t* n_candidates, uint8_t* accept) {
  const uint32_t S = G->n_stations;
  list_t T[ORACLE_MAX_LAYERS / 3];
  memset(T, 0, sizeof(T));
  int rc = 0;

  /* steps 1+2: every triplet of every station, window test on all three pairs */
  for (uint32_t s = 0; s < S && rc == 0; ++s) {
    const int64_t z0 = G->layer_z[3 * s], z1 = G->layer_z[3 * s + 1], z2 = G->layer_z[3 * s + 2];
    const uint32_t b0 = off_ev[3 * s], b1 = off_ev[3 * s + 1], b2 = off_ev[3 * s + 2], b3 = off_ev[3 * s + 3];
    const int64_t a = G->win_in_num, b = G->win_in_den;
    uint64_t count = 0;
    for (uint32_t i0 = b0; i0 < b1 && rc == 0; ++i0) {
      for (uint32_t i1 = b1; i1 < b2 && rc == 0; ++i1) {
        if (!compat(x[i0], y[i0], z0, x[i1], y[i1], z1, a, b)) continue;
        for (uint32_t i2 = b2; i2 < b3; ++i2) {
          if (compat(x[i0], y[i0], z0, x[i2], y[i2], z2, a, b) &&
              compat(x[i1], y[i1], z1, x[i2], y[i2], z2, a, b)) {
            ++count;
            if (list_push(&T[s], i1, max_list_entries)) { rc = -2; break; }
          }
        }
      }
    }
    n_triplets[s] = (uint32_t)(count > ORACLE_SAT ? ORACLE_SAT : count);
  }

  /* linking: chain count over stations, c_0[t] = 1, c_s[u] = sum over linked t of c_{s-1}[t] */
  if (rc == 0) {
    uint64_t *c_prev = NULL, *c_cur = NULL;
    size_t nmax = 0;
    for (uint32_t s = 0; s < S; ++s) if (T[s].n > nmax) nmax = T[s].n;
    c_prev = (uint64_t*)malloc((nmax + 1) * sizeof(uint64_t));
    c_cur = (uint64_t*)malloc((nmax + 1) * sizeof(uint64_t));
    if (!c_prev || !c_cur) rc = -2;
    if (rc == 0) {
      for (size_t t = 0; t < T[0].n; ++t) c_prev[t] = 1;
      for (uint32_t s = 1; s < S; ++s) {
        const int64_t zA = G->layer_z[3 * (s - 1) + 1], zB = G->layer_z[3 * s + 1];
        for (size_t u = 0; u < T[s].n; ++u) {
          const uint32_t iu = T[s].v[u];
          uint64_t acc = 0;
          for (size_t t = 0; t < T[s - 1].n; ++t) {
            const uint32_t it = T[s - 1].v[t];
            if (compat(x[it], y[it], zA, x[iu], y[iu], zB, G->win_link_num, G->win_link_den))
              acc = sat_add(acc, c_prev[t]);
          }
          c_cur[u] = acc;
        }
        uint64_t* tmp = c_prev; c_prev = c_cur; c_cur = tmp;
      }
      uint64_t total = 0;
      for (size_t u = 0; u < T[S - 1].n; ++u) total = sat_add(total, c_prev[u]);
      *n_candidates = (uint32_t)total;
      /* step 3 */
      *accept = (total >= G->min_candidates) ? 1 : 0;
    }
    free(c_prev); free(c_cur);
  }
  for (uint32_t s = 0; s < S; ++s) free(T[s].v);
  return rc;
}

/* Events [e_begin, e_end) of a CSR-SoA batch (off has n_events*L+1 entries, absolute indices).
 * Outputs are indexed relative to e_begin: n_triplets[(e-e_begin)*S+s], n_candidates[e-e_begin],
 * accept[e-e_begin].  Returns 0, -1 on bad arguments, -2 if an event exceeds the list limit. */
int cbm_oracle_run(const oracle_geometry_t* G, const int32_t* x, const int32_t* y, const uint32_t* off,
                   uint64_t e_begin, uint64_t e_end, uint64_t max_list_entries,
                   uint32_t* n_triplets, uint32_t* n_candidates, uint8_t* accept) {
  if (!G || !off || !n_triplets || !n_candidates || !accept) return -1;
  if (G->n_stations < 1 || G->n_stations > ORACLE_MAX_LAYERS / 3) return -1;
  if (G->win_in_den == 0 || G->win_link_den == 0) return -1;
  const uint32_t S = G->n_stations, L = 3 * S;
  if (max_list_entries == 0) max_list_entries = (uint64_t)1 << 27;
  for (uint64_t e = e_begin; e < e_end; ++e) {
    int rc = oracle_event(G, x, y, off + e * L, (size_t)max_list_entries,
                          n_triplets + (e - e_begin) * S, n_candidates + (e - e_begin), accept + (e - e_begin));
    if (rc) return rc;
  }
  return 0;
}

/* A list of event ids (for sampled parity at full batch size).  Outputs indexed by position. */
int cbm_oracle_run_list(const oracle_geometry_t* G, const int32_t* x, const int32_t* y, const uint32_t* off,
                        const uint64_t* event_ids, uint64_t n_ids, uint64_t max_list_entries,
                        uint32_t* n_triplets, uint32_t* n_candidates, uint8_t* accept) {
  if (!G || !off || !event_ids || !n_triplets || !n_candidates || !accept) return -1;
  if (G->n_stations < 1 || G->n_stations > ORACLE_MAX_LAYERS / 3) return -1;
  if (G->win_in_den == 0 || G->win_link_den == 0) return -1;
  const uint32_t S = G->n_stations, L = 3 * S;
  if (max_list_entries == 0) max_list_entries = (uint64_t)1 << 27;
  for (uint64_t k = 0; k < n_ids; ++k) {
    int rc = oracle_event(G, x, y, off + event_ids[k] * L, (size_t)max_list_entries,
                          n_triplets + k * S, n_candidates + k, accept + k);
    if (rc) return rc;
  }
  return 0;
}

// params.h -- plain-old-data shared by the host side (cbm_trigger.cu) and the kernels.
//
// Everything the kernels need about the geometry and the windows is precomputed once on the host at
// cbm_trigger_create() and passed to every launch by value (__grid_constant__).
#pragma once
#include <stdint.h>

namespace cbm {

constexpr int kMaxStations = 8;
constexpr int kMaxLayers = 24;
constexpr uint32_t kSat = 0xFFFFFFFFu;       // outputs are min(2^32-1, exact)  (R9, R12)
constexpr uint32_t kNotTiny = 0xFFFFFFFFu;

// Event classes of the scheduler: tiny events are finished by the tile kernel,
// the others are queued for a team kernel with a team size and a shared-memory budget that fits them.
// List X ("extra") collects the few events a kernel hands on because one of its fixed-size shared-memory
// tables overflowed; they are redone, after all other kernels, by the class-G kernel, whose tables hold anything.
constexpr int kNumTeamClasses = 3;           // M, H, G
constexpr int kClsM = 0, kClsH = 1, kClsG = 2, kClsX = 3;
constexpr int kNumLists = 4;

struct Params {
  uint32_t S, L;
  int32_t z[kMaxLayers];               // layer z, 10-um units
  // window thresholds, R4: |x_h*z_B - x_g*z_A| <= T_AB = floor(a*z_A*z_B / b)  (left side is an integer)
  int64_t thr_in[kMaxStations][3];     // [s][0] = T01, [1] = T02, [2] = T12
  int64_t thr_link[kMaxStations];      // [s], s >= 1: middle layers of stations s-1 and s
  // the same thresholds doubled: the test is evaluated as (uint64)(a*z_B + T - b*z_A) <= 2*T
  uint64_t thr2_in[kMaxStations][3];
  uint64_t thr2_link[kMaxStations];
  // Slope keys, used ONLY to choose which pairs get the exact test (never to accept or reject a pair):
  // key(x, l) = mulhi(x, key_mul[l]) = floor(x * key_mul[l] / 2^32) ~ K * x / z_l, with |key - K*x/z_l| < 1.25,
  // so two hits compatible under win_in have |key_h - key_g| <= key_R in x and in y.
  int32_t key_mul[kMaxLayers];
  int32_t key_R;                       // <= 254
  // packed test of both projections at once: P = (key_x mod 2^16) | (key_y mod 2^16) << 16;
  // |dkey_x| <= R and |dkey_y| <= R  =>  ((P_a + key_add - P_b) & key_mask) == 0
  uint32_t key_add, key_mask;
  int32_t cell_sh;                     // filter cell = floor(key / 2^cell_sh) mod 64 per axis, key_R <= 2^cell_sh
  uint32_t cls_max[kNumTeamClasses];   // fullest layer an event of this class may have
  uint32_t min_candidates;
  uint32_t max_hits_per_layer;
  uint32_t tiny_max_layer;             // 0 disables the tiny path
  uint32_t tiny_max_total;
};

// Device-resident scheduler state of one run; zero-initialised by cudaMemsetAsync before the first kernel.
struct Ctrl {
  uint32_t count[kNumLists];           // list lengths (M, H, G written by the classify kernel; X by the others)
  uint32_t work[kNumLists];            // work-fetch cursors of the persistent team kernels
  uint32_t n_invalid;
  uint32_t first_invalid_inv;          // max over invalid events of ~event  (0 = none)
  uint32_t n_tiny;                     // events the tile kernel finishes
  uint32_t pad[5];
};
static_assert(sizeof(Ctrl) == 64, "Ctrl is copied as one 64-byte record");

// tile kernel geometry
constexpr int kTileEvents = 32;              // events per tile = lanes of the planning warp
constexpr uint32_t kTinyMaxTotal = 96;       // a tiny event holds at most this many hits ...
constexpr uint32_t kTinySlack = 6;           // ... plus at most 3 + 3 hits of 16-byte alignment around its run
// Hits a tile stages in shared memory.  Tiny events are admitted in order while their sizes (+ slack) fit; the
// few that do not (a tile of 32 events near the 96-hit limit) go to class M.  2304 = 32 x (66 + 6): the load-
// imbalance workload's minimum-bias events hold 60 +- 8 hits.
constexpr uint32_t kTileHitCap = 2304;
constexpr uint32_t kTinyMaxLayerLimit = 32;
constexpr int kTileFound = 64;               // (h0,h1) pairs with triplets a tile links itself; more: list X

}  // namespace cbm

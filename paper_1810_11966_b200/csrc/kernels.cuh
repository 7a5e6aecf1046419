// kernels.cuh -- the sm_100a kernels of the CBM-MUCH first-level J/psi selection.
//
// Steps a3..a8 of DESIGN.md:
//   tile_kernel   a3 classify every event (reads off[] once), queue the non-tiny ones by class;
//                 a4 stage the tiny events of a 32-event tile into shared memory with 1-D TMA bulk copies;
//                 a5 thread-per-(event,station) triplet search on the staged hits; a8 result write.
//   team_kernel   persistent, one team (1, 4 or 16 warps) per queued event:
//                 a4/a5 2-D slope-binned triplet search anchored on the middle layer, a6 ballot/popc
//                 compaction of compatible (h0,h1) pairs, a7 cross-station chain count, a8 result write.
//
// The window test is always the exact int64 inequality (PAPER.md:75-76 with the north_star's window):
//   |x_h*z_B - x_g*z_A| <= T_AB,  evaluated as  (uint64)(x_h*z_B + T_AB - x_g*z_A) <= 2*T_AB.
// Slope keys / bins only decide WHERE to look; the bins searched are a proven superset (params.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "params.h"

namespace cbm {

// ---------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
// dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---------------------------------------------------------------------------------------------- window test
// P = a*z_other + T (hoisted per anchor hit);  pass  <=>  |a*z_other - b*z_a| <= T
__device__ __forceinline__ bool win(int64_t P, int32_t b, int32_t za, uint64_t T2) {
  return (uint64_t)(P - (int64_t)b * (int64_t)za) <= T2;
}
__device__ __forceinline__ uint32_t sat32(unsigned long long v) { return v > (unsigned long long)kSat ? kSat : (uint32_t)v; }

__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// ================================================================================================ tile kernel
// One CTA = kTileEvents (32) consecutive events, blockDim.x = 32*S threads: thread t <-> (event t/S, station t%S).
struct TileSmem {
  alignas(16) int32_t sx[kTileHitCap];
  alignas(16) int32_t sy[kTileHitCap];
  uint32_t off[kTileEvents * kMaxLayers + 1];
  uint32_t ev_max[kTileEvents];
  uint32_t ev_dst[kTileEvents];
  uint32_t st_cnt[kTileEvents * kMaxStations];
  alignas(8) uint64_t bar;
};

__global__ void __launch_bounds__(kTileEvents* kMaxStations)
    tile_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                const uint32_t* __restrict__ off, uint32_t n_events, uint32_t n_hits, uint32_t* __restrict__ n_triplets,
                uint32_t* __restrict__ n_candidates, uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl,
                uint32_t* __restrict__ list_M, uint32_t* __restrict__ list_H, uint32_t* __restrict__ list_G) {
  __shared__ TileSmem sm;
  const uint32_t tid = threadIdx.x, nthr = blockDim.x;
  const uint32_t S = p.S, L = p.L;
  const uint32_t e0 = blockIdx.x * kTileEvents;
  const uint32_t ne = min((uint32_t)kTileEvents, n_events - e0);

  // ---- a3: offsets of the tile, read once, coalesced
  {
    const uint32_t n_off = ne * L + 1;
    const uint32_t* src = off + (size_t)e0 * L;
    for (uint32_t i = tid; i < n_off; i += nthr) sm.off[i] = __ldg(src + i);
  }
  if (tid < kTileEvents) sm.ev_max[tid] = 0;
  if (tid == 0) {
    mbar_init(&sm.bar, 1);
    fence_mbar_init();
  }
  __syncthreads();

  const uint32_t el = tid / S, s = tid - el * S;
  const bool active = el < ne;
  uint32_t o0 = 0, o1 = 0, o2 = 0, o3 = 0;
  if (active) {
    const uint32_t* o = &sm.off[el * L + 3 * s];
    o0 = o[0]; o1 = o[1]; o2 = o[2]; o3 = o[3];
    const bool valid = (o0 <= o1) & (o1 <= o2) & (o2 <= o3) & (o3 <= n_hits);
    uint32_t mx = max(max(o1 - o0, o2 - o1), o3 - o2);
    if (!valid || mx > p.max_hits_per_layer) mx = 0xFFFFFFFFu;
    atomicMax(&sm.ev_max[el], mx);
  }
  __syncthreads();

  // ---- planning warp: lane <-> event.  Classes, queues, shared-memory placement, TMA issue.
  if (tid < 32) {
    const uint32_t lane = tid;
    const bool in = lane < ne;
    const uint32_t mx = in ? sm.ev_max[lane] : 0u;
    const uint32_t ob = in ? sm.off[lane * L] : 0u, oe = in ? sm.off[(lane + 1) * L] : 0u;
    const bool invalid = in && mx == 0xFFFFFFFFu;
    const uint32_t tot = oe - ob;
    const bool tiny = in && !invalid && p.tiny_max_total != 0 && mx <= p.tiny_max_layer && tot <= p.tiny_max_total;
    const uint32_t tmask = __ballot_sync(0xFFFFFFFFu, tiny);
    // my run = maximal block of consecutive tiny events around me; runs are contiguous in x[] / y[]
    const uint32_t nz_below = (~tmask) & ((1u << lane) - 1u);
    const uint32_t rs = nz_below ? (32u - __clz(nz_below)) : 0u;  // first lane of my run
    const uint32_t nz_above = (~tmask) >> lane;                   // bit k: lane+k is not tiny
    const uint32_t re = nz_above ? (lane + __ffs(nz_above) - 2u) & 31u : 31u;  // last lane of my run
    const bool start = tiny && rs == lane;
    const uint32_t run_src = __shfl_sync(0xFFFFFFFFu, ob, rs) & ~3u;  // 16-byte aligned source
    const uint32_t run_oe = __shfl_sync(0xFFFFFFFFu, oe, re);
    const uint32_t run_len = start ? (((run_oe + 3u) & ~3u) - run_src) : 0u;  // multiple of 4 hits
    uint32_t incl = run_len;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
      if (lane >= (uint32_t)d) incl += v;
    }
    const uint32_t excl = incl - run_len;
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);  // <= kTileHitCap by construction (params.h)
    const uint32_t run_dst = __shfl_sync(0xFFFFFFFFu, excl, rs);
    sm.ev_dst[lane] = tiny ? run_dst + (ob - run_src) : kNotTiny;
    if (lane == 0) mbar_arrive_expect_tx(&sm.bar, total * 8u);
    __syncwarp();
    if (start && run_len) {  // a4: one bulk copy per run and coordinate
      bulk_g2s(&sm.sx[excl], x + run_src, run_len * 4u, &sm.bar);
      bulk_g2s(&sm.sy[excl], y + run_src, run_len * 4u, &sm.bar);
    }
    // queue the rest by class (order inside a list is irrelevant: results are indexed by event)
    int cls = -1;
    if (in && !invalid && !tiny) cls = mx <= p.cls_max[kClsM] ? kClsM : (mx <= p.cls_max[kClsH] ? kClsH : kClsG);
    uint32_t* const lists[kNumTeamClasses] = {list_M, list_H, list_G};
#pragma unroll
    for (int c = 0; c < kNumTeamClasses; ++c) {
      const uint32_t m = __ballot_sync(0xFFFFFFFFu, cls == c);
      if (m) {
        const int leader = __ffs(m) - 1;
        uint32_t base = 0;
        if ((int)lane == leader) base = atomicAdd(&ctrl->count[c], __popc(m));
        base = __shfl_sync(0xFFFFFFFFu, base, leader);
        if (cls == c) lists[c][base + __popc(m & lanemask_lt())] = e0 + lane;
      }
    }
    if (invalid) {  // rejected on the device: outputs 0, reported by fetch_results / device_status
      const uint32_t e = e0 + lane;
      for (uint32_t k = 0; k < S; ++k) n_triplets[(size_t)e * S + k] = 0;
      n_candidates[e] = 0;
      accept[e] = 0;
      atomicAdd(&ctrl->n_invalid, 1u);
      atomicMax(&ctrl->first_invalid_inv, ~e);
    }
  }
  __syncthreads();
  while (!mbar_try_wait(&sm.bar, 0)) {
  }

  // ---- a5: brute-force triplet search of one station of one tiny event per thread (5 x 5 pairs typical)
  const uint32_t dst = active ? sm.ev_dst[el] : kNotTiny;
  const bool mine = dst != kNotTiny;
  uint32_t cnt = 0;
  if (mine) {
    const uint32_t shift = dst - sm.off[el * L];  // shared index = global index + shift (mod 2^32)
    const int32_t z0 = p.z[3 * s], z1 = p.z[3 * s + 1], z2 = p.z[3 * s + 2];
    const int64_t T01 = p.thr_in[s][0], T02 = p.thr_in[s][1], T12 = p.thr_in[s][2];
    const uint32_t b0 = o0 + shift, b1 = o1 + shift, b2 = o2 + shift, b3 = o3 + shift;
    // one flat loop over the n0*n1 (h0,h1) pairs: lanes of a warp run max(n0*n1) iterations instead of
    // max(n0)*max(n1) (nested loops diverge twice)
    const uint32_t n_pairs = (b2 != b3) ? (b1 - b0) * (b2 - b1) : 0u;
    if (n_pairs) {
      uint32_t i0 = b0, i1 = b1;
      int32_t x0 = sm.sx[i0], y0 = sm.sy[i0];
      int64_t Px = (int64_t)x0 * z1 + T01, Py = (int64_t)y0 * z1 + T01;
      for (uint32_t pr = 0; pr < n_pairs; ++pr) {
        const int32_t x1 = sm.sx[i1];
        if (win(Px, x1, z0, 2 * (uint64_t)T01)) {
          const int32_t y1 = sm.sy[i1];
          if (win(Py, y1, z0, 2 * (uint64_t)T01)) {
            const int64_t Qx0 = (int64_t)x0 * z2 + T02, Qy0 = (int64_t)y0 * z2 + T02;
            const int64_t Qx1 = (int64_t)x1 * z2 + T12, Qy1 = (int64_t)y1 * z2 + T12;
            for (uint32_t i2 = b2; i2 < b3; ++i2) {
              const int32_t x2 = sm.sx[i2], y2 = sm.sy[i2];
              const bool ok = win(Qx0, x2, z0, 2 * (uint64_t)T02) & win(Qy0, y2, z0, 2 * (uint64_t)T02) &
                              win(Qx1, x2, z1, 2 * (uint64_t)T12) & win(Qy1, y2, z1, 2 * (uint64_t)T12);
              cnt += ok ? 1u : 0u;
            }
          }
        }
        if (++i1 == b2) {
          i1 = b1;
          if (++i0 < b1) {
            x0 = sm.sx[i0]; y0 = sm.sy[i0];
            Px = (int64_t)x0 * z1 + T01; Py = (int64_t)y0 * z1 + T01;
          }
        }
      }
    }
    sm.st_cnt[tid] = cnt;
    n_triplets[(size_t)e0 * S + tid] = cnt;  // a8: consecutive threads, consecutive addresses
  }
  __syncthreads();
  // ---- a7/a8: a chain needs a triplet in every station.  If some station has none: 0 candidates, done.
  // Otherwise (rare: essentially only planted tracks) the event is re-queued to class M, whose kernel
  // recomputes it with the full chain count and overwrites these outputs.
  if (mine && s == 0) {
    const uint32_t e = e0 + el;
    bool all = true;
    for (uint32_t k = 0; k < S; ++k) all &= sm.st_cnt[el * S + k] != 0;
    if (!all) {
      n_candidates[e] = 0;
      accept[e] = p.min_candidates == 0 ? 1 : 0;
    } else if (S == 1) {
      n_candidates[e] = cnt;
      accept[e] = cnt >= p.min_candidates ? 1 : 0;
    } else {
      const uint32_t pos = atomicAdd(&ctrl->count[kClsM], 1u);
      list_M[pos] = e;
      atomicAdd(&ctrl->n_escalated, 1u);
    }
  }
}

// ================================================================================================ team kernel
// One team = one CTA of W warps works on one event at a time (persistent: events are fetched from the class
// list with an atomic cursor, two fetches ahead so that the next event can be prefetched into L2).
// CAP = fullest layer the class admits; NCV = uint4 vectors of bin counters (both binned layers of a station);
// LISTCAP = middle hits with triplets kept in shared memory per station (more spill to a global scratch).
template <int W>
__device__ __forceinline__ void team_sync() {
  if (W == 1) __syncwarp(); else __syncthreads();
}

template <int W, int CAP, int NCV, int LISTCAP>
struct TeamSmem {
  alignas(16) uint32_t cellraw[4 + 4 * NCV];  // cell = cellraw + 4: cell[k] = end of bin k after the scatter, cell[-1] = 0
  int32_t sx[2 * CAP], sy[2 * CAP];           // layer 0 then layer 2 of the station, bin-sorted
  uint32_t m[CAP];                            // m[i1] = number of triplets with middle hit i1   (R8)
  int32_t ux[2][LISTCAP], uy[2][LISTCAP];     // distinct middle hits with m > 0 of the previous / current station
  uint32_t uc[2][LISTCAP];                    // their saturated chain counts c_s[u]
  uint32_t queue[W][64];                      // per-warp queue of compatible (h0,h1) pairs: (j_sorted << 16) | i1
  uint16_t cid[2 * CAP];                      // bin of every hit of layers 0 and 2 (count pass -> scatter pass)
  uint32_t off[kMaxLayers + 1];
  uint32_t wsum[32];
  unsigned long long acc;                     // block-wide u64 accumulator (triplet total / candidate total)
  uint32_t ucount;
  uint32_t li[3];                             // ring of fetched work indices
};

// in-place exclusive scan of cell[0 .. 4*nvec) by the whole team, 128-bit shared-memory accesses
template <int W>
__device__ __forceinline__ void team_exclusive_scan(uint32_t* cell, uint32_t nvec, uint32_t* wsum) {
  constexpr uint32_t T = 32 * W;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t chunk = (nvec + T - 1) / T;
  const uint32_t lo = min(tid * chunk, nvec), hi = min(lo + chunk, nvec);
  uint4* const v = reinterpret_cast<uint4*>(cell);
  uint32_t sum = 0;
  for (uint32_t i = lo; i < hi; ++i) {
    const uint4 c = v[i];
    sum += c.x + c.y + c.z + c.w;
  }
  uint32_t incl = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= (uint32_t)d) incl += u;
  }
  uint32_t base = incl - sum;
  if (W > 1) {
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t wv = (lane < (uint32_t)W && lane < warp) ? wsum[lane] : 0u;
    wv = __reduce_add_sync(0xFFFFFFFFu, wv);
    base += wv;
  }
  for (uint32_t i = lo; i < hi; ++i) {
    const uint4 c = v[i];
    uint4 o;
    o.x = base; o.y = o.x + c.x; o.z = o.y + c.y; o.w = o.z + c.z;
    base = o.w + c.w;
    v[i] = o;
  }
}

__device__ __forceinline__ int bin_of(int key, int kmin, int sh, int nbm1) {
  return min(max((key - kmin) >> sh, 0), nbm1);
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// exact window test with the anchor side hoisted: Q = T - b*z_a (int64), pass <=> (uint64)(a*z_o + Q) <= 2T
__device__ __forceinline__ int64_t anchor_q(int32_t b, int32_t neg_za, int64_t T) { return (int64_t)b * neg_za + T; }
__device__ __forceinline__ bool win_q(int32_t a, int32_t zo, int64_t Q, uint64_t T2) {
  return (uint64_t)((int64_t)a * zo + Q) <= T2;
}

// The bins that can hold a hit compatible with a hit of slope keys (kx, ky): at most two rows (bx) of
// consecutive bins, because 2*R <= 2^shift.  Rows as index ranges [a0, a0+n0), [a1, a1+n1) of the bin-sorted
// layer whose bins start at cell[base].
struct Rows { uint32_t a0, n0, a1, n1; };
__device__ __forceinline__ Rows rows_of(const uint32_t* cell, int base, int kx, int ky, int kmin, int R, int sh, int nb) {
  const int tx = kx - R - kmin, ty = ky - R - kmin;
  const int bxl = min(max(tx >> sh, 0), nb - 1), bxh = min(max((tx + 2 * R) >> sh, 0), nb - 1);
  const int byl = min(max(ty >> sh, 0), nb - 1), byh = min(max((ty + 2 * R) >> sh, 0), nb - 1);
  const int r0 = base + bxl * nb, r1 = base + bxh * nb;
  Rows r;
  r.a0 = cell[r0 + byl - 1];
  r.n0 = cell[r0 + byh] - r.a0;
  r.a1 = cell[r1 + byl - 1];
  r.n1 = bxh != bxl ? cell[r1 + byh] - r.a1 : 0u;
  return r;
}

// per-station constants, loaded once per station
struct StationConst {
  int32_t z0, z1, z2, nz0, nz1, nz2;  // nz = -z
  int32_t M0, M1, M2;
  int64_t T01, T02, T12;
  uint64_t T01x2, T02x2, T12x2;
};

// Phase 2 (a5): for one compatible (h0,h1) pair, count the h2 of layer 2 compatible with both.
// Looks only at the 2-D bins around h1's slope (superset of its window), tests exactly.
template <class SM>
__device__ __forceinline__ uint32_t count_h2(const SM& sm, const uint32_t* cell, int ncell, const StationConst& c,
                                             int32_t x0, int32_t y0, int32_t x1, int32_t y1, int kmin, int R, int sh,
                                             int nb) {
  const Rows r = rows_of(cell, ncell, __mulhi(x1, c.M1), __mulhi(y1, c.M1), kmin, R, sh, nb);
  const uint32_t n = r.n0 + r.n1;
  if (n == 0) return 0;
  // |x2*z1 - x1*z2| <= T12 and |x2*z0 - x0*z2| <= T02 (and the same in y)
  const int64_t Qx1 = anchor_q(x1, c.nz2, c.T12), Qy1 = anchor_q(y1, c.nz2, c.T12);
  const int64_t Qx0 = anchor_q(x0, c.nz2, c.T02), Qy0 = anchor_q(y0, c.nz2, c.T02);
  uint32_t cnt = 0;
  for (uint32_t k = 0; k < n; ++k) {
    const uint32_t j = k < r.n0 ? r.a0 + k : r.a1 + (k - r.n0);
    const int32_t x2 = sm.sx[j], y2 = sm.sy[j];
    const bool ok = win_q(x2, c.z1, Qx1, c.T12x2) & win_q(y2, c.z1, Qy1, c.T12x2) & win_q(x2, c.z0, Qx0, c.T02x2) &
                    win_q(y2, c.z0, Qy0, c.T02x2);
    cnt += ok ? 1u : 0u;
  }
  return cnt;
}

template <int W, int CAP, int NCV, int LISTCAP, int CLS, int MINB, bool STATIC_SMEM>
__global__ void __launch_bounds__(32 * W, MINB)
    team_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                const uint32_t* __restrict__ off, uint32_t* __restrict__ n_triplets, uint32_t* __restrict__ n_candidates,
                uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ list,
                uint32_t* __restrict__ spill) {
  using SM = TeamSmem<W, CAP, NCV, LISTCAP>;
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  __shared__ __align__(16) unsigned char smem_static[STATIC_SMEM ? sizeof(SM) : 16];
  SM& sm = *reinterpret_cast<SM*>(STATIC_SMEM ? smem_static : smem_dyn);
  constexpr uint32_t T = 32 * W;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t S = p.S, L = p.L;
  const uint32_t n_list = ctrl->count[CLS];
  const int kmin = p.key_min, R = p.key_R, sh = p.cls_shift[CLS], nb = (int)p.cls_nb[CLS];
  const int ncell = nb * nb;
  const uint32_t nvec = (uint32_t)(2 * ncell + 3) >> 2;
  uint32_t* const cell = sm.cellraw + 4;
  // spill area of this CTA: list entries beyond LISTCAP, [2 lists][x, y, c][CAP] words
  uint32_t* const spill_cta = spill + (size_t)blockIdx.x * 6 * CAP;
  int32_t* const spill_i = reinterpret_cast<int32_t*>(spill_cta);

  if (tid == 0) {
    sm.li[0] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.li[1] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.cellraw[3] = 0;
  }
  team_sync<W>();

  for (uint32_t it3 = 0;; it3 = it3 == 2 ? 0 : it3 + 1) {
    const uint32_t li = sm.li[it3];
    if (li >= n_list) break;
    const uint32_t nxt = sm.li[it3 == 2 ? 0 : it3 + 1];
    if (tid == 0) sm.li[it3 == 0 ? 2 : it3 - 1] = atomicAdd(&ctrl->work[CLS], 1u);
    const uint32_t e = __ldg(list + li);
    // extent of the NEXT event: loaded now, used for its L2 prefetch after station 0 (latency hidden)
    uint32_t pf_a = 0, pf_b = 0;
    if (nxt < n_list) {
      const uint32_t e2 = __ldg(list + nxt);
      pf_a = __ldg(off + (size_t)e2 * L);
      pf_b = __ldg(off + (size_t)e2 * L + L);
    }
    for (uint32_t i = tid; i <= L; i += T) sm.off[i] = __ldg(off + (size_t)e * L + i);
    team_sync<W>();

    uint32_t nprev = 0;
    bool dead = false;  // some station so far has no triplet => no chain; triplet counts are still needed
    int cur = 0;
    for (uint32_t s = 0; s < S; ++s) {
      const uint32_t b0 = sm.off[3 * s], b1 = sm.off[3 * s + 1], b2 = sm.off[3 * s + 2], b3 = sm.off[3 * s + 3];
      const uint32_t n0 = b1 - b0, n1 = b2 - b1, n2 = b3 - b2;
      StationConst c;
      c.z0 = p.z[3 * s]; c.z1 = p.z[3 * s + 1]; c.z2 = p.z[3 * s + 2];
      c.nz0 = -c.z0; c.nz1 = -c.z1; c.nz2 = -c.z2;
      c.M0 = p.key_mul[3 * s]; c.M1 = p.key_mul[3 * s + 1]; c.M2 = p.key_mul[3 * s + 2];
      c.T01 = p.thr_in[s][0]; c.T02 = p.thr_in[s][1]; c.T12 = p.thr_in[s][2];
      c.T01x2 = p.thr2_in[s][0]; c.T02x2 = p.thr2_in[s][1]; c.T12x2 = p.thr2_in[s][2];
      if (tid == 0) { sm.acc = 0; sm.ucount = 0; }
      const bool search = (n0 != 0) & (n1 != 0) & (n2 != 0);
      if (search) {
        // ---- a4: bin layers 0 and 2 on a 2-D slope grid: count, one scan over both grids, scatter
        {
          uint4* const v = reinterpret_cast<uint4*>(cell);
          for (uint32_t i = tid; i < nvec; i += T) v[i] = make_uint4(0, 0, 0, 0);
          for (uint32_t i = tid; i < n1; i += T) sm.m[i] = 0;
        }
        team_sync<W>();
        for (uint32_t i = tid; i < n0 + n2; i += T) {
          const bool l2 = i >= n0;
          const uint32_t g = l2 ? b2 + (i - n0) : b0 + i;
          const int32_t hx = __ldg(x + g), hy = __ldg(y + g);
          const int32_t M = l2 ? c.M2 : c.M0;
          const int cc = (l2 ? ncell : 0) + bin_of(__mulhi(hx, M), kmin, sh, nb - 1) * nb +
                         bin_of(__mulhi(hy, M), kmin, sh, nb - 1);
          sm.cid[i] = (uint16_t)cc;
          atomicAdd(&cell[cc], 1u);
        }
        team_sync<W>();
        team_exclusive_scan<W>(cell, nvec, sm.wsum);
        team_sync<W>();
        for (uint32_t i = tid; i < n0 + n2; i += T) {
          const uint32_t g = i >= n0 ? b2 + (i - n0) : b0 + i;
          const int32_t hx = __ldg(x + g), hy = __ldg(y + g);  // L1 hit
          const uint32_t pos = atomicAdd(&cell[sm.cid[i]], 1u);
          sm.sx[pos] = hx;
          sm.sy[pos] = hy;
        }
        team_sync<W>();

        // ---- a5/a6: anchors = middle-layer hits, one per lane; compatible (h0,h1) pairs are compacted
        // into the warp's queue with ballot/popc and drained 32 at a time by phase 2.
        uint32_t qn = 0;
        uint32_t* const q = sm.queue[warp];
        for (uint32_t base = warp * 32; base < n1; base += T) {
          const uint32_t i1 = base + lane;
          const bool act = i1 < n1;
          int32_t x1 = 0, y1 = 0;
          Rows r = {0, 0, 0, 0};
          if (act) {
            x1 = __ldg(x + b1 + i1);
            y1 = __ldg(y + b1 + i1);
            r = rows_of(cell, 0, __mulhi(x1, c.M1), __mulhi(y1, c.M1), kmin, R, sh, nb);
          }
          const uint32_t nc = r.n0 + r.n1;
          const uint32_t ncmax = __reduce_max_sync(0xFFFFFFFFu, nc);
          // |x0*z1 - x1*z0| <= T01  <=>  (uint64)(x0*z1 + (T01 - x1*z0)) <= 2*T01
          const int64_t Qx = anchor_q(x1, c.nz0, c.T01), Qy = anchor_q(y1, c.nz0, c.T01);
          // test loop: no cross-lane traffic, each lane records its passing candidates as bits of `mask`
          for (uint32_t k0 = 0; k0 < ncmax; k0 += 32) {
            const uint32_t kend = min(ncmax - k0, 32u);
            uint32_t mask = 0;
            for (uint32_t kk = 0; kk < kend; ++kk) {
              const uint32_t k = k0 + kk;
              if (k < nc) {
                const uint32_t j = k < r.n0 ? r.a0 + k : r.a1 + (k - r.n0);
                const bool pass = win_q(sm.sx[j], c.z1, Qx, c.T01x2) & win_q(sm.sy[j], c.z1, Qy, c.T01x2);
                mask |= (pass ? 1u : 0u) << kk;
              }
            }
            // a6: rounds of ballot/popc compaction, one pair per lane and round, drained 32 at a time
            for (uint32_t pm = __ballot_sync(0xFFFFFFFFu, mask != 0); pm; pm = __ballot_sync(0xFFFFFFFFu, mask != 0)) {
              if (mask) {
                const uint32_t k = k0 + (uint32_t)__ffs(mask) - 1u;
                const uint32_t j = k < r.n0 ? r.a0 + k : r.a1 + (k - r.n0);
                q[qn + __popc(pm & lanemask_lt())] = (j << 16) | i1;
                mask &= mask - 1u;
              }
              qn += __popc(pm);
              if (qn >= 32) {
                __syncwarp();
                qn -= 32;
                const uint32_t ent = q[qn + lane];
                const uint32_t j0 = ent >> 16, k1 = ent & 0xFFFFu;
                const uint32_t t = count_h2(sm, cell, ncell, c, sm.sx[j0], sm.sy[j0], __ldg(x + b1 + k1),
                                            __ldg(y + b1 + k1), kmin, R, sh, nb);
                if (t) atomicAdd(&sm.m[k1], t);
                __syncwarp();
              }
            }
          }
        }
        __syncwarp();
        if (lane < qn) {
          const uint32_t ent = q[lane];
          const uint32_t j0 = ent >> 16, k1 = ent & 0xFFFFu;
          const uint32_t t = count_h2(sm, cell, ncell, c, sm.sx[j0], sm.sy[j0], __ldg(x + b1 + k1), __ldg(y + b1 + k1),
                                      kmin, R, sh, nb);
          if (t) atomicAdd(&sm.m[k1], t);
        }
      }
      if (s == 0 && pf_b > pf_a) {  // pull the next event of this team into L2 while this one is being searched
        const uint32_t la = pf_a >> 5, lb = (pf_b + 31) >> 5;  // 128-byte lines
        for (uint32_t l = la + tid; l < lb; l += T) {
          prefetch_l2(x + (size_t)l * 32);
          prefetch_l2(y + (size_t)l * 32);
        }
      }
      team_sync<W>();

      // ---- station total, list of distinct middle hits with triplets (R8)
      if (search) {
        constexpr bool kSmallSum = (CAP + T - 1) / T < 8;  // 32 lanes * 7 hits * 2^24 < 2^32
        uint32_t part32 = 0;
        unsigned long long part64 = 0;
        for (uint32_t i = tid; i < n1; i += T) {
          const uint32_t mm = sm.m[i];
          if (kSmallSum) part32 += mm; else part64 += mm;
          if (mm && !dead) {
            const uint32_t pos = atomicAdd(&sm.ucount, 1u);
            const int32_t hx = __ldg(x + b1 + i), hy = __ldg(y + b1 + i);
            if (pos < (uint32_t)LISTCAP) {
              sm.ux[cur][pos] = hx; sm.uy[cur][pos] = hy; sm.uc[cur][pos] = mm;
            } else {
              const uint32_t o = pos - LISTCAP;
              spill_i[(cur * 3 + 0) * CAP + o] = hx; spill_i[(cur * 3 + 1) * CAP + o] = hy;
              spill_cta[(cur * 3 + 2) * CAP + o] = mm;
            }
          }
        }
        if (kSmallSum) {
          part32 = __reduce_add_sync(0xFFFFFFFFu, part32);
          if (lane == 0 && part32) atomicAdd(&sm.acc, (unsigned long long)part32);
        } else {
#pragma unroll
          for (int d = 16; d >= 1; d >>= 1) part64 += __shfl_xor_sync(0xFFFFFFFFu, part64, d);
          if (lane == 0 && part64) atomicAdd(&sm.acc, part64);
        }
      }
      team_sync<W>();
      const uint32_t ncur = dead ? 0u : sm.ucount;
      if (tid == 0) n_triplets[(size_t)e * S + s] = sat32(sm.acc);
      // ---- a7: chain counts c_s[u] = m_u * sum over linked t of c_{s-1}[t], saturating (R9)
      if (s > 0 && !dead && ncur) {
        const int32_t nzA = -p.z[3 * (s - 1) + 1], zB = c.z1;
        const int64_t TL = p.thr_link[s];
        const uint64_t TLx2 = p.thr2_link[s];
        if (ncur <= (uint32_t)LISTCAP && nprev <= (uint32_t)LISTCAP) {  // everything in shared memory
          for (uint32_t u = tid; u < ncur; u += T) {
            // |x_t*zB - x_u*zA| <= TL
            const int64_t Qx = anchor_q(sm.ux[cur][u], nzA, TL), Qy = anchor_q(sm.uy[cur][u], nzA, TL);
            unsigned long long a = 0;
            for (uint32_t t = 0; t < nprev; ++t) {
              const bool ok = win_q(sm.ux[cur ^ 1][t], zB, Qx, TLx2) & win_q(sm.uy[cur ^ 1][t], zB, Qy, TLx2);
              if (ok) a += sm.uc[cur ^ 1][t];  // < 4096 * 2^32
            }
            sm.uc[cur][u] = sat32((unsigned long long)sat32(a) * sm.uc[cur][u]);  // m_u <= 2^24: no overflow
          }
        } else {  // rare: some entries live in the global spill area
          auto LX = [&](int w, uint32_t i) { return i < (uint32_t)LISTCAP ? sm.ux[w][i] : spill_i[(w * 3 + 0) * CAP + i - LISTCAP]; };
          auto LY = [&](int w, uint32_t i) { return i < (uint32_t)LISTCAP ? sm.uy[w][i] : spill_i[(w * 3 + 1) * CAP + i - LISTCAP]; };
          auto LC = [&](int w, uint32_t i) { return i < (uint32_t)LISTCAP ? sm.uc[w][i] : spill_cta[(w * 3 + 2) * CAP + i - LISTCAP]; };
          for (uint32_t u = tid; u < ncur; u += T) {
            const int64_t Qx = anchor_q(LX(cur, u), nzA, TL), Qy = anchor_q(LY(cur, u), nzA, TL);
            unsigned long long a = 0;
            for (uint32_t t = 0; t < nprev; ++t) {
              const bool ok = win_q(LX(cur ^ 1, t), zB, Qx, TLx2) & win_q(LY(cur ^ 1, t), zB, Qy, TLx2);
              if (ok) a += LC(cur ^ 1, t);
            }
            const uint32_t v = sat32((unsigned long long)sat32(a) * LC(cur, u));
            if (u < (uint32_t)LISTCAP) sm.uc[cur][u] = v; else spill_cta[(cur * 3 + 2) * CAP + u - LISTCAP] = v;
          }
        }
      }
      if (ncur == 0) dead = true;
      nprev = ncur;
      cur ^= 1;
      team_sync<W>();
    }

    // ---- candidates = sum over the last station's middle hits; a8: one writer per event
    if (tid == 0) sm.acc = 0;
    team_sync<W>();
    if (!dead) {
      unsigned long long part = 0;
      for (uint32_t u = tid; u < nprev; u += T)
        part += u < (uint32_t)LISTCAP ? sm.uc[cur ^ 1][u] : spill_cta[((cur ^ 1) * 3 + 2) * CAP + u - LISTCAP];
      if (__any_sync(0xFFFFFFFFu, part != 0)) {
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(0xFFFFFFFFu, part, d);
        if (lane == 0) atomicAdd(&sm.acc, part);
      }
    }
    team_sync<W>();
    if (tid == 0) {
      const uint32_t cand = sat32(sm.acc);
      n_candidates[e] = cand;
      accept[e] = cand >= p.min_candidates ? 1 : 0;
    }
    team_sync<W>();
  }
}

}  // namespace cbm

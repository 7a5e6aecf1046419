// msd.cuh -- the paper's own selection, literally (section 3.2):
// all triplets of the trigger station, least-squares line through the event vertex (0,0) in x-z and y-z
// (x = m0 z, y = m1 z), mean square deviation per degree of freedom against 0.03 / 0.025, event selected with
// at least two passing triplets.
//
// Exact form of the cut (the paper's floating-point precision is unstated; B8): with Svz = sum v_i z_i,
// Szz = sum z_i^2, Svv = sum v_i^2 over the three hits, the sum of squared residuals of the fitted line is
// Svv - Svz^2/Szz, and  MSD/ndf <= num/den cm^2  <=>  den*(Szz*Svv - Svz^2) <= num*10^6*ndf*Szz  in 10-um units:
// 128-bit integers; exact for any int32 coordinates and 0 < z <= 2^23 (Svz < 2^56 in int64, Svv < 2^64 in uint64,
// Szz*Svv < 2^112, left side < 2^124, right side < 2^92).
//
// Sixteen lanes per event (two events per warp); lane <-> hit of layer 0, loop over layer 1.  A passing triplet has every residual |r_i| <= delta = sqrt(thr*ndf),
// hence |v1*z0 - v0*z1| = |r1*z0 - r0*z1| <= delta*(z0+z1): an exact 64-bit necessary condition on the pair that
// keeps the 128-bit test and the h2 loop for the few pairs that can belong to a passing triplet.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cbm {

struct MsdDev {
  uint32_t L, first_layer;       // layers per event, first layer of the trigger station
  int32_t z0, z1, z2;
  uint32_t num_x, den_x, num_y, den_y, ndf, min_triplets;
  int64_t pre_x, pre_y;          // delta_x * (z0 + z1), delta_y * (z0 + z1), delta = floor(sqrt(thr*ndf)) + 1
};

constexpr int kMsdWarps = 4;
constexpr int kMsdLanes = 16;  // lanes per event: the paper's trigger station holds about 15 hits per layer

__device__ __forceinline__ bool msd_ok(int64_t v0, int64_t v1, int64_t v2, int64_t z0, int64_t z1, int64_t z2, int64_t szz,
                                       uint32_t num, uint32_t den, uint32_t ndf) {
  const int64_t svz = v0 * z0 + v1 * z1 + v2 * z2;
  const uint64_t svv = (uint64_t)(v0 * v0) + (uint64_t)(v1 * v1) + (uint64_t)(v2 * v2);  // < 3 * 2^62
  const uint64_t asvz = (uint64_t)(svz < 0 ? -svz : svz);
  const unsigned __int128 ssr_szz = (unsigned __int128)(uint64_t)szz * svv - (unsigned __int128)asvz * asvz;  // >= 0
  const unsigned __int128 lhs = ssr_szz * den;
  const unsigned __int128 rhs = (unsigned __int128)((uint64_t)num * 1000000ull * ndf) * (uint64_t)szz;
  return lhs <= rhs;
}

__global__ void __launch_bounds__(32 * kMsdWarps)
    msd_kernel(const MsdDev p, const int32_t* __restrict__ x, const int32_t* __restrict__ y, const uint32_t* __restrict__ off,
               uint32_t n_events, uint32_t n_hits, uint32_t* __restrict__ n_passing, uint8_t* __restrict__ accept) {
  const uint32_t lane = threadIdx.x & (kMsdLanes - 1);
  const uint32_t e = blockIdx.x * (kMsdWarps * 32 / kMsdLanes) + threadIdx.x / kMsdLanes;
  if (e >= n_events) return;  // whole groups of kMsdLanes lanes leave: the shuffles below stay inside a group
  const uint32_t* o = off + (size_t)e * p.L + p.first_layer;
  const uint32_t o0 = __ldg(o), o1 = __ldg(o + 1), o2 = __ldg(o + 2), o3 = __ldg(o + 3);
  unsigned long long cnt = 0;
  const bool well_formed = (o0 <= o1) & (o1 <= o2) & (o2 <= o3) & (o3 <= n_hits);
  if (well_formed) {  // a malformed event selects nothing and is never accepted
    const int64_t z0 = p.z0, z1 = p.z1, z2 = p.z2;
    const int64_t szz = z0 * z0 + z1 * z1 + z2 * z2;
    // lane <-> hit of layer 0; the hits of layers 1 and 2 are read at addresses uniform in the group (one transaction each)
    for (uint32_t i0 = o0 + lane; i0 < o1; i0 += kMsdLanes) {
      const int64_t x0 = __ldg(x + i0), y0 = __ldg(y + i0);
      const int64_t ax = x0 * z1, ay = y0 * z1;
      for (uint32_t i1 = o1; i1 < o2; ++i1) {
        const int64_t x1 = __ldg(x + i1);
        const int64_t dx = x1 * z0 - ax;
        if ((dx < 0 ? -dx : dx) > p.pre_x) continue;  // exact necessary condition on the pair (h0, h1)
        const int64_t y1 = __ldg(y + i1);
        const int64_t dy = y1 * z0 - ay;
        if ((dy < 0 ? -dy : dy) > p.pre_y) continue;
        for (uint32_t i2 = o2; i2 < o3; ++i2) {
          const int64_t x2 = __ldg(x + i2), y2 = __ldg(y + i2);
          if (msd_ok(x0, x1, x2, z0, z1, z2, szz, p.num_x, p.den_x, p.ndf) &&
              msd_ok(y0, y1, y2, z0, z1, z2, szz, p.num_y, p.den_y, p.ndf))
            ++cnt;
        }
      }
    }
  }
  const uint32_t gmask = kMsdLanes == 32 ? 0xFFFFFFFFu : (((1u << kMsdLanes) - 1u) << ((threadIdx.x & 31u) & ~(uint32_t)(kMsdLanes - 1)));
#pragma unroll
  for (int d = kMsdLanes / 2; d >= 1; d >>= 1) cnt += __shfl_xor_sync(gmask, cnt, d);
  if (lane == 0) {
    const uint32_t c = cnt > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)cnt;
    n_passing[e] = c;
    accept[e] = (well_formed && c >= p.min_triplets) ? 1 : 0;
  }
}

}  // namespace cbm

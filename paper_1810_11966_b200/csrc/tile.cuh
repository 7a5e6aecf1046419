// tile.cuh -- tile_kernel: the tiny events (a4, a5, a7, a8 of DESIGN.md / SURVEY.md section 8(a)).
//
// One CTA = one tile of 32 consecutive events.  The classes were decided by classify_kernel; this kernel takes
// the same decision again from the same offsets (tile_admit) and finishes the tile's tiny events:
//   a4 stage the tiny events of the tile into shared memory with 1-D TMA bulk copies (one per run of
//      consecutive tiny events and coordinate);
//   a5 one thread per search unit (a layer-0 hit): exact (h0,h1) x test over the station's layer 1, the y test
//      and the h2 loop only for a pair that passes;
//   a7 in-tile chain count over the remembered pairs, a8 result write.
//
// The window test is always the exact int64 inequality (PAPER.md:75-76 with the north_star's window):
//   |x_h*z_B - x_g*z_A| <= T_AB,  evaluated as  (uint64)(x_h*z_B + T_AB - x_g*z_A) <= 2*T_AB.
#pragma once
#include <stddef.h>

#include "classify.cuh"

namespace cbm {

// ================================================================================================ tile kernel
// One CTA = kTileEvents (32) consecutive events, blockDim.x = 32*S threads: thread t <-> (station t/32, event t%32),
// so a warp handles one station of the tile's 32 events.
struct TileStation {  // constants of one station, read from shared memory (lanes of a warp may differ in station)
  int32_t z0, z1, z2, pad;
  int64_t T01, T02, T12;
};
template <int MS>  // MS: stations the tables are sized for (4 or 8)
struct TileSmem {
  alignas(16) int32_t sx[kTileHitCap];
  alignas(16) int32_t sy[kTileHitCap];
  alignas(16) TileStation sc[MS];
  uint32_t off[kTileEvents * 3 * MS + 1];
  uint32_t ev_max[kTileEvents];
  uint32_t ev_dst[kTileEvents];
  uint32_t st_cnt[kTileEvents * MS];            // triplets of (event el, station s) at [el*S + s]
  uint32_t pre[kTileEvents * MS];               // first search unit of (station, event) thread t
  alignas(8) uint2 desc[kTileEvents * MS];      // its layer boundaries in sx/sy: (b0 | b1<<16, b2 | b3<<16)
  uint32_t wsum[MS];
  uint32_t f_key[kTileFound];                   // found (h0,h1) pairs with triplets: owner thread << 16 | index of h1
  uint32_t f_t[kTileFound];                     // number of h2 completing the pair
  uint32_t f_c[kTileFound];                     // chain count of the entry (a7)
  uint32_t nfound;
  uint8_t owner[kTileHitCap];                   // search unit (one layer-0 hit) -> owner thread
  alignas(8) uint64_t bar;
};

template <int MS>
__global__ void __launch_bounds__(kTileEvents* MS)
    tile_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                const uint32_t* __restrict__ off, uint32_t n_events, uint32_t n_hits, uint32_t* __restrict__ n_triplets,
                uint32_t* __restrict__ n_candidates, uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl,
                uint32_t* __restrict__ list_x) {
  __shared__ TileSmem<MS> sm;
  constexpr uint32_t FULL = 0xFFFFFFFFu;
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
  if (tid < S) {
    TileStation k;
    k.z0 = p.z[3 * tid]; k.z1 = p.z[3 * tid + 1]; k.z2 = p.z[3 * tid + 2]; k.pad = 0;
    k.T01 = p.thr_in[tid][0]; k.T02 = p.thr_in[tid][1]; k.T12 = p.thr_in[tid][2];
    sm.sc[tid] = k;
  }
  if (tid == 0) {
    sm.nfound = 0;
    mbar_init(&sm.bar, 1);
    fence_mbar_init();
  }
  __syncthreads();

  const uint32_t s = tid >> 5, el = tid & 31;
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

  // ---- planning warp: lane <-> event.  Admission, shared-memory placement, TMA issue.
  if (tid < 32) {
    const uint32_t lane = tid;
    const bool in = lane < ne;
    const uint32_t mx = in ? sm.ev_max[lane] : 0u;
    const uint32_t ob = in ? sm.off[lane * L] : 0u, oe = in ? sm.off[(lane + 1) * L] : 0u;
    const bool invalid = in && mx == 0xFFFFFFFFu;
    const uint32_t tot = oe - ob;
    const bool tiny = tile_admit(p, lane, in, invalid, mx, tot);  // the decision classify_kernel took
    const uint32_t tmask = __ballot_sync(FULL, tiny);
    // my run = maximal block of consecutive tiny events around me; runs are contiguous in x[] / y[]
    const uint32_t nz_below = (~tmask) & ((1u << lane) - 1u);
    const uint32_t rs = nz_below ? (32u - __clz(nz_below)) : 0u;  // first lane of my run
    const uint32_t nz_above = (~tmask) >> lane;                   // bit k: lane+k is not tiny
    const uint32_t re = nz_above ? (lane + __ffs(nz_above) - 2u) & 31u : 31u;  // last lane of my run
    const bool start = tiny && rs == lane;
    const uint32_t run_src = __shfl_sync(FULL, ob, rs) & ~3u;  // 16-byte aligned source
    const uint32_t run_oe = __shfl_sync(FULL, oe, re);
    const uint32_t run_len = start ? (((run_oe + 3u) & ~3u) - run_src) : 0u;  // multiple of 4 hits
    uint32_t incl = run_len;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t v = __shfl_up_sync(FULL, incl, d);
      if (lane >= (uint32_t)d) incl += v;
    }
    const uint32_t excl = incl - run_len;
    const uint32_t total = __shfl_sync(FULL, incl, 31);  // <= kTileHitCap: every run is shorter than its events + slack
    const uint32_t run_dst = __shfl_sync(FULL, excl, rs);
    sm.ev_dst[lane] = tiny ? run_dst + (ob - run_src) : kNotTiny;
    if (lane == 0) mbar_arrive_expect_tx(&sm.bar, total * 8u);
    __syncwarp();
    if (start && run_len) {  // a4: one bulk copy per run and coordinate
      bulk_g2s(&sm.sx[excl], x + run_src, run_len * 4u, &sm.bar);
      bulk_g2s(&sm.sy[excl], y + run_src, run_len * 4u, &sm.bar);
    }
  }
  __syncthreads();

  // ---- search units: one per layer-0 hit of a (tiny event, station) with three non-empty layers.  Block-wide
  // exclusive scan of the unit counts, then every thread names itself owner of its units; the staging copies
  // are in flight meanwhile.
  const uint32_t dst = active ? sm.ev_dst[el] : kNotTiny;
  const bool mine = dst != kNotTiny;
  const uint32_t lane = tid & 31;
  uint32_t nu = 0;
  if (mine) {
    const uint32_t shift = dst - sm.off[el * L];  // shared index = global index + shift (mod 2^32)
    sm.desc[tid] = make_uint2(((o0 + shift) & 0xFFFFu) | ((o1 + shift) << 16), ((o2 + shift) & 0xFFFFu) | ((o3 + shift) << 16));
    nu = (o1 != o2 && o2 != o3) ? o1 - o0 : 0u;
    sm.st_cnt[el * S + s] = 0;
  }
  uint32_t incl = nu;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t v = __shfl_up_sync(FULL, incl, d);
    if (lane >= (uint32_t)d) incl += v;
  }
  if (lane == 31) sm.wsum[s] = incl;
  __syncthreads();
  uint32_t first = incl - nu, n_units = 0;
  for (uint32_t w = 0; w < S; ++w) {
    const uint32_t v = sm.wsum[w];
    first += w < s ? v : 0u;
    n_units += v;
  }
  sm.pre[tid] = first;
  for (uint32_t k = 0; k < nu; ++k) sm.owner[first + k] = (uint8_t)tid;
  __syncthreads();
  while (!mbar_try_wait(&sm.bar, 0)) {
  }

  // ---- a5: unit u = layer-0 hit i0 of its owner's station: all its (h0,h1) pairs, x test first; the h2 loop
  // runs only for a compatible pair.  Pairs with triplets are remembered for the linking (a6).
  for (uint32_t u = tid; u < n_units; u += nthr) {
    const uint32_t ow = sm.owner[u];
    const uint32_t i0 = u - sm.pre[ow];
    const uint2 dsc = sm.desc[ow];
    const uint32_t b0 = dsc.x & 0xFFFFu, b1 = dsc.x >> 16, b2 = dsc.y & 0xFFFFu, b3 = dsc.y >> 16;
    const TileStation& k = sm.sc[ow >> 5];
    const int32_t z0 = k.z0, z1 = k.z1, nz0 = -z0;
    const int64_t T01 = k.T01;
    const uint64_t T01x2 = 2 * (uint64_t)T01;
    constexpr int kDY = (int)(offsetof(TileSmem<MS>, sy) - offsetof(TileSmem<MS>, sx));
    const uint32_t ax = smem_u32(sm.sx);
    const int32_t x0 = lds_s32(ax + 4 * (b0 + i0)), y0 = lds_s32<kDY>(ax + 4 * (b0 + i0));
    // |x0*z1 - x1*z0| <= T01  <=>  (uint64)(x1*(-z0) + (x0*z1 + T01)) <= 2*T01
    const int64_t Px = (int64_t)x0 * z1 + T01, Py = (int64_t)y0 * z1 + T01;
    uint32_t cnt = 0;
    const uint32_t a_end = ax + 4 * b2;
    // the rare continuation of a pair that passed the x test: y test, then the h2 loop
    auto pair_passed_x = [&](uint32_t a1, int32_t x1) {
      const int32_t y1 = lds_s32<kDY>(a1);
      if ((uint64_t)((int64_t)y1 * nz0 + Py) <= T01x2) {
        const int32_t z2 = k.z2;
        const int64_t T02 = k.T02, T12 = k.T12;
        const int64_t Qx0 = (int64_t)x0 * z2 + T02, Qy0 = (int64_t)y0 * z2 + T02;
        const int64_t Qx1 = (int64_t)x1 * z2 + T12, Qy1 = (int64_t)y1 * z2 + T12;
        uint32_t t = 0;
        for (uint32_t i2 = b2; i2 < b3; ++i2) {
          const int32_t x2 = sm.sx[i2], y2 = sm.sy[i2];
          const bool ok = win(Qx0, x2, z0, 2 * (uint64_t)T02) & win(Qy0, y2, z0, 2 * (uint64_t)T02) &
                          win(Qx1, x2, z1, 2 * (uint64_t)T12) & win(Qy1, y2, z1, 2 * (uint64_t)T12);
          t += ok ? 1u : 0u;
        }
        if (t) {
          cnt += t;
          const uint32_t slot = atomicAdd(&sm.nfound, 1u);
          if (slot < (uint32_t)kTileFound) {
            sm.f_key[slot] = (ow << 16) | ((a1 - ax) >> 2);
            sm.f_t[slot] = t;
          }
        }
      }
    };
    // two pairs per trip: two independent load/test chains, half the loop overhead (the second load of an odd
    // last trip reads the next layer's first hit; its result is masked)
    for (uint32_t a1 = ax + 4 * b1; a1 < a_end; a1 += 8) {
      const int32_t xa = lds_s32(a1), xb = lds_s32<4>(a1);
      const bool pa = (uint64_t)((int64_t)xa * nz0 + Px) <= T01x2;
      const bool pb = ((uint64_t)((int64_t)xb * nz0 + Px) <= T01x2) & (a1 + 4 < a_end);
      if (pa | pb) {
        if (pa) pair_passed_x(a1, xa);
        if (pb) pair_passed_x(a1 + 4, xb);
      }
    }
    if (cnt) atomicAdd(&sm.st_cnt[(ow & 31u) * S + (ow >> 5)], cnt);
  }
  __syncthreads();

  // ---- a8: triplet counts, coalesced (tiny events only; the others are written by their team)
  {
    const uint32_t oe = tid / S;  // event of output element tid
    if (oe < ne && sm.ev_dst[oe] != kNotTiny) n_triplets[(size_t)e0 * S + tid] = sm.st_cnt[tid];
  }
  // ---- a7/a8: a chain needs a triplet in every station.  If some station has none: 0 candidates, done.
  // Otherwise (rare: essentially only planted tracks) the event's thread of station 0 counts the chains over
  // the remembered pairs: an entry (h0,h1) with t triplets stands for t triplets with middle hit h1 (R8), so
  // c_0 = t, c_s[u] = t_u * sum over linked entries v of station s-1 of c_{s-1}[v], saturating (R9).
  if (mine && s == 0) {
    const uint32_t e = e0 + el;
    bool all = true;
    for (uint32_t q = 0; q < S; ++q) all &= sm.st_cnt[el * S + q] != 0;
    const uint32_t nf = sm.nfound;
    if (!all) {
      n_candidates[e] = 0;
      accept[e] = p.min_candidates == 0 ? 1 : 0;
    } else if (S == 1) {
      const uint32_t cand = sm.st_cnt[el];
      n_candidates[e] = cand;
      accept[e] = cand >= p.min_candidates ? 1 : 0;
    } else if (nf <= (uint32_t)kTileFound) {
      unsigned long long cand = 0;
      for (uint32_t q = 0; q < S; ++q) {
        const uint32_t me = (q << 5) | el, prev = ((q - 1u) << 5) | el;
        const int32_t nzA = q ? -p.z[3 * (q - 1) + 1] : 0, zB = p.z[3 * q + 1];
        const int64_t TL = p.thr_link[q];
        const uint64_t TLx2 = p.thr2_link[q];
        for (uint32_t u = 0; u < nf; ++u) {
          const uint32_t ku = sm.f_key[u];
          if ((ku >> 16) != me) continue;
          unsigned long long a = 1;
          if (q) {
            // |x_v*zB - x_u*zA| <= TL  <=>  (uint64)(x_v*zB + (TL - x_u*zA)) <= 2*TL
            const int64_t Qx = (int64_t)sm.sx[ku & 0xFFFFu] * nzA + TL, Qy = (int64_t)sm.sy[ku & 0xFFFFu] * nzA + TL;
            a = 0;
            for (uint32_t v = 0; v < nf; ++v) {
              const uint32_t kv = sm.f_key[v];
              if ((kv >> 16) != prev) continue;
              const bool ok = (uint64_t)((int64_t)sm.sx[kv & 0xFFFFu] * zB + Qx) <= TLx2 &&
                              (uint64_t)((int64_t)sm.sy[kv & 0xFFFFu] * zB + Qy) <= TLx2;
              if (ok) a += sm.f_c[v];
            }
          }
          const uint32_t cu = sat32((unsigned long long)sat32(a) * sm.f_t[u]);
          sm.f_c[u] = cu;
          if (q == S - 1) cand += cu;
        }
      }
      const uint32_t c32 = sat32(cand);
      n_candidates[e] = c32;
      accept[e] = c32 >= p.min_candidates ? 1 : 0;
    } else {  // too many pairs with triplets in this tile: list X (redone after all other kernels; its outputs are overwritten)
      list_x[atomicAdd(&ctrl->count[kClsX], 1u)] = e;
    }
  }
}

}  // namespace cbm

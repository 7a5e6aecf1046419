// team.cuh -- team_kernel: steps a4..a8 for the events of classes M, H, G.
//
// One team = one CTA of W warps works on one event at a time (persistent: events are fetched from the class
// list with an atomic cursor).  Per station, with the middle layer as anchor (R8: linking needs only the
// middle hit):
//
//   stage  six 1-D TMA bulk copies (three layers x two coordinates) bring the station into shared memory.
//   A      every hit gets its filter cell (fx, fy) on a cyclic 64 x 64 grid of its slope keys
//          (cell = floor(key / 2^cell_sh) mod 64, 2^cell_sh >= key_R) and sets its bit in its layer's
//          occupancy bitmap (RED.OR); the cell is kept (16 bits per hit).
//   B      Three hits that are pairwise compatible have keys within key_R <= one cell width of each other in
//          x and in y, so they lie in ONE 2 x 2 block of cells.  T = blocks that hold a hit of every layer
//          (bit-parallel: 64-bit rows), J = cells covered by a block of T.  One warp, two rows per lane.
//   C      a hit whose cell is not in J cannot belong to a triplet.  The others (20 % at 300 hits per layer)
//          are kept: middle hits in a list, hits of layers 0 and 2 with their packed slope key
//          P = (key_x mod 2^16) | (key_y mod 2^16) << 16 in per-band tables (band = a few cell columns).
//   D      one lane per kept middle hit h1: it scans the kept hits of layer 0 in the <= 3 bands its window
//          touches with the packed test ((P1 + key_add - P0) & key_mask) == 0 (both projections in two
//          integer instructions; it never rejects a compatible pair) and runs the exact int64 test on the few
//          that pass; lanes that found an h0 scan layer 2 the same way, with exact tests against h1 and the
//          recorded h0.  (x1, y1, number of triplets with this middle hit) goes to the station's list.
//   F      chain counts against the previous station's list (a7), result write (a8).
//
// Accept/reject never uses a key, a cell or a bitmap: those only decide which pairs get the exact test, and
// the pairs tested are a proven superset of the compatible ones.
#pragma once
#include "ptx.cuh"

namespace cbm {

template <int W>
__device__ __forceinline__ void team_sync() {
  if (W == 1) __syncwarp(); else __syncthreads();
}

// W warps; CAP_ = fullest layer of the class; S1CAP_ = kept middle hits; bands of 2^BSH_ cell columns with
// BCAP_ kept hits each, OCAP_ more in an overflow band that every middle hit scans; LISTCAP_ = middle hits
// with triplets kept per station in shared memory.
template <int W_, int CAP_, int S1CAP_, int BSH_, int BCAP_, int OCAP_, int LISTCAP_>
struct TeamSmem {
  static constexpr int W = W_, CAP = CAP_, S1CAP = S1CAP_, BSH = BSH_, BCAP = BCAP_, OCAP = OCAP_, LISTCAP = LISTCAP_;
  static constexpr int NB = 64 >> BSH;
  static constexpr int SLOTS = NB * BCAP + OCAP;
  static constexpr int LCAP = CAP + 8;          // a layer as it lies in x[], from the 16-byte boundary below it
  static_assert(CAP % 8 == 0 && BCAP % 4 == 0 && OCAP % 4 == 0 && S1CAP % 2 == 0, "vector accesses");
  alignas(16) int32_t sx[3][LCAP];
  alignas(16) int32_t sy[3][LCAP];
  alignas(16) uint16_t sc[3][LCAP];             // filter cell (fx << 6 | fy) of every staged element
  alignas(16) uint32_t occ[3][128];             // occupancy bitmaps: row fx = 64 bits, bit fy
  alignas(16) uint32_t J[128];                  // cells covered by a 2 x 2 block that holds all three layers
  alignas(16) uint32_t bP[2][SLOTS];            // packed keys of the kept hits of layers 0 and 2, by band
  uint16_t bI[2][SLOTS];                        // ... and their element index in sx / sy
  uint16_t s1[S1CAP];                           // kept middle hits (element index)
  uint32_t bcnt[2][2][NB + 1];                  // [parity][layer 0 / 2][band]; [NB] = overflow band
  uint32_t n1s[2];                              // [parity]
  int32_t ux[2][LISTCAP], uy[2][LISTCAP];       // middle hits with triplets of the previous / current station
  uint32_t uc[2][LISTCAP];                      // their multiplicities, then saturated chain counts c_s[u]
  uint32_t off[kMaxLayers + 1];
  alignas(8) unsigned long long acc[2];         // triplets of the station (parity-buffered with ucount)
  uint32_t ucount[2];
  uint32_t li[3];                               // ring of fetched work indices
  uint32_t fail;                                // a table overflowed: the event goes to list X
  alignas(8) uint64_t bar;                      // completion of the station's bulk copies
};

// per-station constants of the exact tests, read from the kernel parameters (constant bank) where they are used:
// the exact tests are rare (only pairs that pass the packed key test get one)
struct StationConst {
  const Params& p;
  uint32_t s;
  __device__ __forceinline__ int32_t z0() const { return p.z[3 * s]; }
  __device__ __forceinline__ int32_t z1() const { return p.z[3 * s + 1]; }
  __device__ __forceinline__ int32_t z2() const { return p.z[3 * s + 2]; }
  __device__ __forceinline__ int64_t T01() const { return p.thr_in[s][0]; }
  __device__ __forceinline__ int64_t T02() const { return p.thr_in[s][1]; }
  __device__ __forceinline__ int64_t T12() const { return p.thr_in[s][2]; }
  __device__ __forceinline__ uint64_t T01x2() const { return p.thr2_in[s][0]; }
  __device__ __forceinline__ uint64_t T02x2() const { return p.thr2_in[s][1]; }
  __device__ __forceinline__ uint64_t T12x2() const { return p.thr2_in[s][2]; }
};

// Scan of the kept hits of layer li (0: layer 0, 1: layer 2) in bands blo .. blo+nb-1 (cyclic) and in the
// overflow band: f(slot) for every entry that passes the packed key test against A1 = P1 + key_add.
// Per-lane loops, no warp-level operation inside.
template <class SM, class F>
__device__ __forceinline__ void scan_bands(const SM& sm, int li, const uint32_t* __restrict__ cnt, uint32_t A1, uint32_t mask,
                                           uint32_t blo, uint32_t nb, F&& f) {
  for (uint32_t i = 0; i <= nb; ++i) {
    const bool ovf = i == nb;
    const uint32_t b = ovf ? (uint32_t)SM::NB : ((blo + i) & (uint32_t)(SM::NB - 1));
    const uint32_t n = min(cnt[b], ovf ? (uint32_t)SM::OCAP : (uint32_t)SM::BCAP);
    const uint32_t base = b * SM::BCAP;
    for (uint32_t t0 = 0; t0 < n; t0 += 4) {
      const uint4 P = *reinterpret_cast<const uint4*>(&sm.bP[li][base + t0]);
      uint32_t mm = (((A1 - P.x) & mask) == 0 ? 1u : 0u) | (((A1 - P.y) & mask) == 0 ? 2u : 0u) |
                    (((A1 - P.z) & mask) == 0 ? 4u : 0u) | (((A1 - P.w) & mask) == 0 ? 8u : 0u);
      while (mm) {  // rare
        const uint32_t k = (uint32_t)__ffs((int)mm) - 1u;
        mm &= mm - 1u;
        if (t0 + k < n) f(base + t0 + k);
      }
    }
  }
}

// Rare path of phase D (a middle hit with more than two compatible h0): number of kept h0 compatible with both
// h1 (anchors Qx, Qy) and h2 (x2, y2).
template <class SM>
__device__ __noinline__ uint32_t count_h0_slow(const SM& sm, const uint32_t* cnt0, uint32_t A1, uint32_t mask, uint32_t blo,
                                               uint32_t nb, const Params& p, uint32_t s, int64_t Qx, int64_t Qy, int32_t x2,
                                               int32_t y2) {
  const StationConst c{p, s};
  uint32_t n = 0;
  scan_bands(sm, 0, cnt0, A1, mask, blo, nb, [&](uint32_t slot) {
    const uint32_t e0 = sm.bI[0][slot];
    const int32_t x0 = sm.sx[0][e0], y0 = sm.sy[0][e0];
    const bool ok = win_q(x0, c.z1(), Qx, c.T01x2()) & win_q(y0, c.z1(), Qy, c.T01x2()) &
                    win_q(x2, c.z0(), anchor_q(x0, -c.z2(), c.T02()), c.T02x2()) &
                    win_q(y2, c.z0(), anchor_q(y0, -c.z2(), c.T02()), c.T02x2());
    n += ok ? 1u : 0u;
  });
  return n;
}

// CLS: the list this kernel works on.  SPILL: station lists beyond LISTCAP go to a per-CTA global scratch and no
// table can overflow (S1CAP = OCAP = CAP), so the kernel never hands an event on (class G and list X); without
// it an overflowing event is appended to list X.
template <class SM, int CLS, int MINB, bool SPILL, bool STATIC_SMEM>
__global__ void __launch_bounds__(32 * SM::W, MINB)
    team_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                const uint32_t* __restrict__ off, uint32_t* __restrict__ n_triplets, uint32_t* __restrict__ n_candidates,
                uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ list,
                uint32_t* __restrict__ list_x, uint32_t* __restrict__ spill) {
  constexpr int W = SM::W, CAP = SM::CAP, S1CAP = SM::S1CAP, BSH = SM::BSH, BCAP = SM::BCAP, OCAP = SM::OCAP;
  constexpr int LISTCAP = SM::LISTCAP, NB = SM::NB;
  static_assert(!SPILL || (S1CAP >= CAP && OCAP >= CAP), "a spilling kernel must hold any station");
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  __shared__ __align__(16) unsigned char smem_static[STATIC_SMEM ? sizeof(SM) : 16];
  SM& sm = *reinterpret_cast<SM*>(STATIC_SMEM ? smem_static : smem_dyn);
  constexpr uint32_t T = 32 * W;
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t S = p.S, L = p.L;
  const uint32_t n_list = ctrl->count[CLS];
  const int fsh = p.cell_sh;
  const uint32_t kmask = p.key_mask, kadd = p.key_add;
  // spill area of this CTA: list entries beyond LISTCAP, [2 lists][x, y, c][CAP] words
  uint32_t* const spill_cta = SPILL ? spill + (size_t)blockIdx.x * 6 * CAP : nullptr;
  int32_t* const spill_i = reinterpret_cast<int32_t*>(spill_cta);

  for (uint32_t i = tid; i < 3 * 128; i += T) (&sm.occ[0][0])[i] = 0;
  for (uint32_t i = tid; i < 2 * 2 * (NB + 1); i += T) (&sm.bcnt[0][0][0])[i] = 0;
  if (tid == 0) {
    sm.li[0] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.li[1] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.acc[0] = sm.acc[1] = 0;
    sm.ucount[0] = sm.ucount[1] = 0;
    sm.n1s[0] = sm.n1s[1] = 0;
    sm.fail = 0;
    mbar_init(&sm.bar, 1);
    fence_mbar_init();
  }
  team_sync<W>();
  uint32_t par = 0;  // phase parity of the staging barrier
  uint32_t sp = 0;   // parity of the per-station list counters
  uint32_t cp = 0;   // parity of the per-station filter counters

  auto searchable = [&](uint32_t s) {
    return (sm.off[3 * s] != sm.off[3 * s + 1]) & (sm.off[3 * s + 1] != sm.off[3 * s + 2]) & (sm.off[3 * s + 2] != sm.off[3 * s + 3]);
  };
  // a4: thread 0 starts the bulk copies of station s of the event whose offsets are in sm.off: every layer from
  // the 16-byte boundary below its first hit to the one above its last
  auto issue_stage = [&](uint32_t s) {
    uint32_t a[3], bytes[3];
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      a[l] = sm.off[3 * s + l] & ~3u;
      bytes[l] = (((sm.off[3 * s + l + 1] + 3u) & ~3u) - a[l]) * 4u;  // <= (CAP + 4) * 4
    }
    mbar_arrive_expect_tx(&sm.bar, 2u * (bytes[0] + bytes[1] + bytes[2]));
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      bulk_g2s(sm.sx[l], x + a[l], bytes[l], &sm.bar);
      bulk_g2s(sm.sy[l], y + a[l], bytes[l], &sm.bar);
    }
  };

  for (uint32_t it3 = 0;; it3 = it3 == 2 ? 0 : it3 + 1) {
    const uint32_t li = sm.li[it3];
    if (li >= n_list) break;
    if (tid == 0) sm.li[it3 == 0 ? 2 : it3 - 1] = atomicAdd(&ctrl->work[CLS], 1u);
    const uint32_t e = __ldg(list + li);
    for (uint32_t i = tid; i <= L; i += T) sm.off[i] = __ldg(off + (size_t)e * L + i);
    team_sync<W>();
    if (tid == 0 && searchable(0)) issue_stage(0);

    uint32_t nprev = 0;
    bool dead = false;    // some station so far has no triplet => no chain; triplet counts are still needed
    bool failed = false;  // the event was handed on to list X
    int cur = 0;
    for (uint32_t s = 0; s < S; ++s) {
      const uint32_t b0 = sm.off[3 * s], b1 = sm.off[3 * s + 1], b2 = sm.off[3 * s + 2], b3 = sm.off[3 * s + 3];
      const uint32_t n0 = b1 - b0, n1 = b2 - b1, n2 = b3 - b2;
      const bool search = (n0 != 0) & (n1 != 0) & (n2 != 0);
      if (search) {
        // quads (4 staged elements) of the three layers: layer l starts at element b_l & 3 of its region
        const uint32_t st0 = b0 & 3u, st1 = b1 & 3u, st2 = b2 & 3u;
        const uint32_t nq0 = (st0 + n0 + 3u) >> 2, nq01 = nq0 + ((st1 + n1 + 3u) >> 2), nqt = nq01 + ((st2 + n2 + 3u) >> 2);
        const int32_t M0 = p.key_mul[3 * s], M1 = p.key_mul[3 * s + 1], M2 = p.key_mul[3 * s + 2];
        while (!mbar_try_wait(&sm.bar, par)) {
        }
        par ^= 1u;
        // ---- A: filter cells and occupancy bitmaps.  Elements of a quad outside the layer (<= 3 at either
        // end: hits of the neighbouring layers) only add bits, which keeps the filter a superset.
        for (uint32_t qi = tid; qi < nqt; qi += T) {
          const uint32_t l = (qi >= nq0 ? 1u : 0u) + (qi >= nq01 ? 1u : 0u);
          const uint32_t q = qi - (l == 0 ? 0u : (l == 1 ? nq0 : nq01));
          const int32_t M = l == 0 ? M0 : (l == 1 ? M1 : M2);
          const int4 xv = *reinterpret_cast<const int4*>(&sm.sx[l][4 * q]);
          const int4 yv = *reinterpret_cast<const int4*>(&sm.sy[l][4 * q]);
          uint32_t* const occ = sm.occ[l];
          auto cell = [&](int32_t xx, int32_t yy) {
            const uint32_t c = (((uint32_t)(__mulhi(xx, M) >> fsh) & 63u) << 6) | ((uint32_t)(__mulhi(yy, M) >> fsh) & 63u);
            reds_or(&occ[c >> 5], 1u << (c & 31u));
            return c;
          };
          const uint32_t c0 = cell(xv.x, yv.x), c1 = cell(xv.y, yv.y), c2 = cell(xv.z, yv.z), c3 = cell(xv.w, yv.w);
          *reinterpret_cast<uint2*>(&sm.sc[l][4 * q]) = make_uint2(c0 | (c1 << 16), c2 | (c3 << 16));
        }
        team_sync<W>();
        // ---- B: block (i, j) = cells {i, i+1} x {j, j+1} (cyclic).  T[i] bit j = the block holds a hit of every
        // layer; J[i] bit j = cell (i, j) lies in some block of T.  One warp; lane <-> rows 2*lane, 2*lane+1.
        if (warp == s % W) {
          unsigned long long t0 = ~0ull, t1 = ~0ull;
#pragma unroll
          for (int l = 0; l < 3; ++l) {
            const unsigned long long* rows = reinterpret_cast<const unsigned long long*>(sm.occ[l]);
            const unsigned long long ra = rows[2 * lane], rb = rows[2 * lane + 1], rc = rows[(2 * lane + 2) & 63];
            const unsigned long long va = ra | rb, vb = rb | rc;
            t0 &= va | (va >> 1) | (va << 63);
            t1 &= vb | (vb >> 1) | (vb << 63);
          }
          const unsigned long long tm = __shfl_sync(FULL, t1, (lane + 31) & 31);  // T of row 2*lane - 1
          const unsigned long long ja = t0 | tm, jb = t1 | t0;
          const unsigned long long j0 = ja | (ja << 1) | (ja >> 63), j1 = jb | (jb << 1) | (jb >> 63);
          *reinterpret_cast<ulonglong2*>(&sm.J[4 * lane]) = make_ulonglong2(j0, j1);
        }
        team_sync<W>();
        // ---- C (a6): keep the hits whose cell is in J
        {
          uint32_t* const cnt0 = sm.bcnt[cp][0];
          uint32_t* const cnt2 = sm.bcnt[cp][1];
          for (uint32_t qi = tid; qi < nqt; qi += T) {
            const uint32_t l = (qi >= nq0 ? 1u : 0u) + (qi >= nq01 ? 1u : 0u);
            const uint32_t q = qi - (l == 0 ? 0u : (l == 1 ? nq0 : nq01));
            const uint32_t st = l == 0 ? st0 : (l == 1 ? st1 : st2), nl = l == 0 ? n0 : (l == 1 ? n1 : n2);
            const uint2 cc = *reinterpret_cast<const uint2*>(&sm.sc[l][4 * q]);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const uint32_t c = ((k & 2) ? cc.y : cc.x) >> ((k & 1) * 16) & 0xFFFFu;
              const uint32_t el = 4 * q + k;
              const bool keep = (el - st < nl) && ((sm.J[c >> 5] >> (c & 31u)) & 1u);
              if (keep) {
                if (l == 1) {
                  const uint32_t pos = atoms_add(&sm.n1s[cp], 1u);
                  if (pos < (uint32_t)S1CAP) sm.s1[pos] = (uint16_t)el; else sm.fail = 1;
                } else {
                  const int li2 = (int)(l >> 1);
                  const uint32_t P = packed_key(sm.sx[l][el], sm.sy[l][el], l == 0 ? M0 : M2);
                  uint32_t* const cnt = li2 ? cnt2 : cnt0;
                  const uint32_t band = c >> (6 + BSH);
                  uint32_t slot = atoms_add(&cnt[band], 1u);
                  if (slot < (uint32_t)BCAP) {
                    slot += band * BCAP;
                  } else {
                    slot = atoms_add(&cnt[NB], 1u);
                    if (slot >= (uint32_t)OCAP) { sm.fail = 1; slot = 0xFFFFFFFFu; } else slot += NB * BCAP;
                  }
                  if (slot != 0xFFFFFFFFu) { sm.bP[li2][slot] = P; sm.bI[li2][slot] = (uint16_t)el; }
                }
              }
            }
          }
        }
        team_sync<W>();
        // ---- D (a5): one lane per kept middle hit
        {
          for (uint32_t i = tid; i < 3 * 128; i += T) (&sm.occ[0][0])[i] = 0;                    // free since B
          for (uint32_t i = tid; i < 2 * (NB + 1); i += T) (&sm.bcnt[cp ^ 1u][0][0])[i] = 0;      // the next station's
          if (tid == 0) sm.n1s[cp ^ 1u] = 0;
          const StationConst c{p, s};
          const uint32_t n1k = min(sm.n1s[cp], (uint32_t)S1CAP);
          const uint32_t* const cnt0 = sm.bcnt[cp][0];
          const uint32_t* const cnt2 = sm.bcnt[cp][1];
          unsigned long long trip = 0;
          for (uint32_t base = warp * 32; base < n1k; base += T) {
            const uint32_t j = base + lane;
            uint32_t t = 0;  // triplets with this middle hit
            int32_t x1 = 0, y1 = 0;
            if (j < n1k) {
              const uint32_t e1 = sm.s1[j];
              x1 = sm.sx[1][e1];
              y1 = sm.sy[1][e1];
              const int32_t kx = __mulhi(x1, M1), ky = __mulhi(y1, M1);
              const uint32_t A1 = __byte_perm((uint32_t)kx, (uint32_t)ky, 0x5410) + kadd;
              const uint32_t fx = (uint32_t)(kx >> fsh) & 63u;
              const uint32_t blo = ((fx - 1u) & 63u) >> BSH, bhi = ((fx + 1u) & 63u) >> BSH;
              const uint32_t nb = ((bhi - blo) & (uint32_t)(NB - 1)) + 1u;  // bands a compatible hit can lie in
              // h0 compatible with h1:  |x0*z1 - x1*z0| <= T01  <=>  (uint64)(x0*z1 + (T01 - x1*z0)) <= 2*T01
              const int64_t Qx = anchor_q(x1, -c.z0(), c.T01()), Qy = anchor_q(y1, -c.z0(), c.T01());
              uint32_t np = 0, pk = 0;  // number of compatible h0; the first two (element index, 16 bits each)
              scan_bands(sm, 0, cnt0, A1, kmask, blo, nb, [&](uint32_t slot) {
                const uint32_t e0 = sm.bI[0][slot];
                if (win_q(sm.sx[0][e0], c.z1(), Qx, c.T01x2()) & win_q(sm.sy[0][e0], c.z1(), Qy, c.T01x2())) {
                  if (np < 2) pk |= e0 << (np << 4);
                  ++np;
                }
              });
              if (np) {
                // h2 compatible with h1:  |x2*z1 - x1*z2| <= T12;  with h0:  |x2*z0 - x0*z2| <= T02
                const int64_t Rx = anchor_q(x1, -c.z2(), c.T12()), Ry = anchor_q(y1, -c.z2(), c.T12());
                scan_bands(sm, 1, cnt2, A1, kmask, blo, nb, [&](uint32_t slot) {
                  const uint32_t e2 = sm.bI[1][slot];
                  const int32_t x2 = sm.sx[2][e2], y2 = sm.sy[2][e2];
                  if (win_q(x2, c.z1(), Rx, c.T12x2()) & win_q(y2, c.z1(), Ry, c.T12x2())) {
                    if (np <= 2) {
                      uint32_t q = pk, n = np;
                      do {
                        const int32_t x0 = sm.sx[0][q & 0xFFFFu], y0 = sm.sy[0][q & 0xFFFFu];
                        const bool ok = win_q(x2, c.z0(), anchor_q(x0, -c.z2(), c.T02()), c.T02x2()) &
                                        win_q(y2, c.z0(), anchor_q(y0, -c.z2(), c.T02()), c.T02x2());
                        t += ok ? 1u : 0u;
                        q >>= 16;
                      } while (--n);
                    } else {
                      t += count_h0_slow(sm, cnt0, A1, kmask, blo, nb, p, s, Qx, Qy, x2, y2);
                    }
                  }
                });
              }
            }
            trip += t;
            // a6: middle hits with triplets -> the station's list (distinct hits: every h1 has one lane)
            const uint32_t am = __ballot_sync(FULL, t != 0);
            if (am && !dead) {
              const int leader = __ffs(am) - 1;
              uint32_t pos = 0;
              if ((int)lane == leader) pos = atoms_add(&sm.ucount[sp], (uint32_t)__popc(am));
              pos = __shfl_sync(FULL, pos, leader) + __popc(am & lanemask_lt());
              if (t) {
                if (pos < (uint32_t)LISTCAP) {
                  sm.ux[cur][pos] = x1; sm.uy[cur][pos] = y1; sm.uc[cur][pos] = t;
                } else if (SPILL) {
                  const uint32_t o = pos - LISTCAP;
                  spill_i[(cur * 3 + 0) * CAP + o] = x1; spill_i[(cur * 3 + 1) * CAP + o] = y1;
                  spill_cta[(cur * 3 + 2) * CAP + o] = t;
                } else {
                  sm.fail = 1;
                }
              }
            }
          }
          if (__any_sync(FULL, trip != 0)) {
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) trip += __shfl_xor_sync(FULL, trip, d);
            if (lane == 0) atomicAdd(&sm.acc[sp], trip);
          }
        }
        cp ^= 1u;
      }
      team_sync<W>();

      // ---- F: the search is over: the staging buffer is free
      if (!SPILL && sm.fail) { failed = true; break; }
      const uint32_t ncur = dead ? 0u : sm.ucount[sp];
      if (tid == 0) {
        n_triplets[(size_t)e * S + s] = sat32(sm.acc[sp]);
        sm.acc[sp ^ 1u] = 0;
        sm.ucount[sp ^ 1u] = 0;
        if (s + 1 < S && searchable(s + 1)) issue_stage(s + 1);
      }
      // ---- a7: chain counts c_s[u] = m_u * sum over linked t of c_{s-1}[t], saturating (R9).  Small teams: warp
      // 0 alone, while the others already wait for the next station's copies.
      if (s > 0 && ncur && (SPILL || warp == 0)) {
        const int32_t nzA = -p.z[3 * (s - 1) + 1], zB = p.z[3 * s + 1];
        const int64_t TL = p.thr_link[s];
        const uint64_t TLx2 = p.thr2_link[s];
        auto LX = [&](int w, uint32_t i) { return (!SPILL || i < (uint32_t)LISTCAP) ? sm.ux[w][i] : spill_i[(w * 3 + 0) * CAP + i - LISTCAP]; };
        auto LY = [&](int w, uint32_t i) { return (!SPILL || i < (uint32_t)LISTCAP) ? sm.uy[w][i] : spill_i[(w * 3 + 1) * CAP + i - LISTCAP]; };
        auto LC = [&](int w, uint32_t i) { return (!SPILL || i < (uint32_t)LISTCAP) ? sm.uc[w][i] : spill_cta[(w * 3 + 2) * CAP + i - LISTCAP]; };
        for (uint32_t u = SPILL ? tid : lane; u < ncur; u += SPILL ? T : 32u) {
          // |x_t*zB - x_u*zA| <= TL
          const int64_t Qx = anchor_q(LX(cur, u), nzA, TL), Qy = anchor_q(LY(cur, u), nzA, TL);
          unsigned long long a = 0;
          for (uint32_t t = 0; t < nprev; ++t) {
            const bool ok = win_q(LX(cur ^ 1, t), zB, Qx, TLx2) & win_q(LY(cur ^ 1, t), zB, Qy, TLx2);
            if (ok) a += LC(cur ^ 1, t);  // < 4096 * 2^32
          }
          const uint32_t v = sat32((unsigned long long)sat32(a) * LC(cur, u));  // m_u <= 2^24
          if (!SPILL || u < (uint32_t)LISTCAP) sm.uc[cur][u] = v; else spill_cta[(cur * 3 + 2) * CAP + u - LISTCAP] = v;
        }
      }
      if (SPILL) team_sync<W>();  // the whole team linked
      if (ncur == 0) dead = true;
      nprev = ncur;
      cur ^= 1;
      sp ^= 1u;
    }

    if (failed) {  // hand the event on: list X is redone by the spilling kernel after all others
      team_sync<W>();
      if (tid == 0) {
        list_x[atomicAdd(&ctrl->count[kClsX], 1u)] = e;
        sm.fail = 0;
        sm.acc[0] = sm.acc[1] = 0;
        sm.ucount[0] = sm.ucount[1] = 0;
      }
      team_sync<W>();
      continue;
    }
    // ---- candidates = sum over the last station's middle hits; a8: one writer per event
    if (warp == 0) {
      __syncwarp();
      unsigned long long part = 0;
      if (!dead)
        for (uint32_t u = lane; u < nprev; u += 32)
          part += (!SPILL || u < (uint32_t)LISTCAP) ? sm.uc[cur ^ 1][u] : spill_cta[((cur ^ 1) * 3 + 2) * CAP + u - LISTCAP];
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(FULL, part, d);
      if (lane == 0) {
        const uint32_t cand = sat32(part);
        n_candidates[e] = cand;
        accept[e] = cand >= p.min_candidates ? 1 : 0;
      }
    }
    team_sync<W>();
  }
}

}  // namespace cbm

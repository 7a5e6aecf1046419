// team.cuh -- team_kernel: steps a4..a8 for the events of classes M, H, G.
//
// One team = one CTA of W warps works on one event at a time (persistent: events are fetched from the class
// list with an atomic cursor).  Per station, with the middle layer as anchor (R8: linking needs only the
// middle hit):
//
//   A      the station's hits are read from global memory once, four consecutive hits per thread and coordinate
//          (128-bit coalesced loads; the lines were pulled into L2 one station ahead, prefetch.global.L2).
//          Every hit gets its packed slope key P = (key_x mod 2^16) | (key_y mod 2^16) << 16 (kept in shared
//          memory) and sets the bit of its filter cell (fx, fy) -- cell = floor(key / 2^cell_sh) mod 64,
//          2^cell_sh >= key_R -- in its layer's 64 x 64 occupancy bitmap (RED.OR); hits of layers 0 and 2 are
//          pushed on the chain of their coarse cell (atomicExch on the cell's head, 16-bit link per hit).
//   B      Three hits that are pairwise compatible have keys within key_R <= one cell width of each other in
//          x and in y, so they lie in ONE 2 x 2 block of cells.  T = blocks that hold a hit of every layer
//          (bit-parallel: 64-bit rows), J = cells covered by a block of T.  One warp, two rows per lane.
//   C      a middle hit whose cell is not in J cannot belong to a triplet; the others (20 % at 300 hits per
//          layer) are compacted (ballot/popc) into a list.
//   D      two lanes per kept middle hit h1, one for layer 0 and one for layer 2: each walks the chains of the
//          <= 2 x 2 coarse cells the window of h1 touches in its layer, collects the hits that pass the packed
//          test ((P1 + key_add - P) & key_mask) == 0 (both projections in two integer instructions; it never
//          rejects a compatible pair) and runs the exact int64 test against h1 on those; the two lanes then
//          swap what they found and test the (h0, h2) pairs.  (x1, y1, number of triplets with this middle
//          hit) goes to the station's list.
//   F      chain counts against the previous station's list (a7), result write (a8).
//
// Accept/reject never uses a key, a cell or a bitmap: those only decide which pairs get the exact test, and
// the pairs tested are a proven superset of the compatible ones.  The exact tests read
// the coordinates from global memory again (L1 / L2 hits: the station has just been read).
#pragma once
#include "ptx.cuh"

namespace cbm {

template <int W>
__device__ __forceinline__ void team_sync() {
  if (W == 1) __syncwarp(); else __syncthreads();
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// W warps; CAP_ = fullest layer of the class; K1CAP_ = kept middle hits; coarse table of 2^TXB_ x 2^TYB_ cells
// (TXB_, TYB_ <= 5: a coarse cell spans at least two filter cells, so a window touches at most 2 x 2 of them);
// LISTCAP_ = middle hits with triplets kept per station in shared memory.
template <int W_, int CAP_, int K1CAP_, int TXB_, int TYB_, int LISTCAP_>
struct TeamSmem {
  static constexpr int W = W_, CAP = CAP_, K1CAP = K1CAP_, TXB = TXB_, TYB = TYB_, LISTCAP = LISTCAP_;
  static constexpr int LCAP = CAP + 8;          // a layer as it lies in x[], from the 16-byte boundary below it
  static constexpr int NHEAD = 2 << (TXB + TYB);
  static_assert(CAP % 8 == 0 && K1CAP % 2 == 0 && TXB <= 5 && TYB <= 5 && LCAP < 65535, "layout");
  alignas(16) uint32_t P[3][LCAP];              // packed slope keys
  alignas(16) uint32_t occ[3][128];             // occupancy bitmaps: row fy = 64 bits, bit fx
  alignas(16) uint32_t J[128];                  // cells covered by a 2 x 2 block that holds all three layers
  uint32_t head[NHEAD];                         // chain heads of layers 0 and 2: epoch << 16 | (element + 1); an
                                                // entry of another epoch (= station) counts as empty: no zeroing
  uint16_t nx[2][LCAP];                         // chain links (element + 1; 0 = end)
  uint16_t k1[K1CAP];                           // kept middle hits (element index)
  uint32_t n1k[2];                              // [parity] number of kept middle hits
  int32_t ux[2][LISTCAP], uy[2][LISTCAP];       // middle hits with triplets of the previous / current station
  uint32_t uc[2][LISTCAP];                      // their multiplicities, then saturated chain counts c_s[u]
  uint32_t off[2][kMaxLayers + 1];              // offsets of this event and of the next one
  uint32_t ntr[kMaxStations];                   // triplets per station of this event
  alignas(8) unsigned long long acc[2];         // triplets of the station (parity-buffered with ucount)
  uint32_t ucount[2];
  uint32_t li[4];                               // ring of fetched work indices
  uint32_t fail;                                // a table overflowed: the event goes to list X
  uint32_t trash;                               // chain head of the elements that are not hits of the layer
};

// stations of an event with three non-empty layers, as a bit mask (o: the event's L + 1 offsets)
__device__ __forceinline__ uint32_t searchable_mask(const uint32_t* o, uint32_t S) {
  uint32_t m = 0;
  for (uint32_t s = 0; s < S; ++s)
    if ((o[3 * s] != o[3 * s + 1]) & (o[3 * s + 1] != o[3 * s + 2]) & (o[3 * s + 2] != o[3 * s + 3])) m |= 1u << s;
  return m;
}

// Walk of the chains of layer li (0: layer 0, 1: layer 2) in the <= 2 x 2 coarse cells a hit compatible with a
// hit of keys (kx, ky) (mod 2^16) can lie in: f(el) for every hit whose packed key passes the test against
// A1 = P1 + key_add.  Per-lane loop, no warp-level operation inside.
template <class SM, class F>
__device__ __forceinline__ void walk_chains(const SM& sm, uint32_t li, uint32_t ep, uint32_t kx, uint32_t ky, int R, int fsh,
                                            uint32_t A1, uint32_t mask, F&& f) {
  constexpr int XS = 6 - SM::TXB, YS = 6 - SM::TYB;  // filter cells per coarse cell (log2), >= 1
  constexpr uint32_t MX = (1u << SM::TXB) - 1u, MY = (1u << SM::TYB) - 1u;
  // key_R <= 2^cell_sh and a coarse cell is >= 2^(cell_sh+1) wide: at most two columns and two rows (cyclic)
  const uint32_t lox = ((kx - R) >> (fsh + XS)) & MX, hix = ((kx + R) >> (fsh + XS)) & MX;
  const uint32_t loy = ((ky - R) >> (fsh + YS)) & MY, hiy = ((ky + R) >> (fsh + YS)) & MY;
  const uint32_t* hd = sm.head + li * (SM::NHEAD / 2);
  unsigned long long hq = 0;  // non-empty chain heads of this epoch, 16 bits each
  {
    uint32_t v = hd[(lox << SM::TYB) | loy];
    if ((v >> 16) == ep) hq = v & 0xFFFFu;
    if (hiy != loy) { v = hd[(lox << SM::TYB) | hiy]; if ((v >> 16) == ep) hq = (hq << 16) | (v & 0xFFFFu); }
    if (hix != lox) {
      v = hd[(hix << SM::TYB) | loy]; if ((v >> 16) == ep) hq = (hq << 16) | (v & 0xFFFFu);
      if (hiy != loy) { v = hd[(hix << SM::TYB) | hiy]; if ((v >> 16) == ep) hq = (hq << 16) | (v & 0xFFFFu); }
    }
  }
  const uint32_t* Pl = sm.P[2 * li];
  const uint16_t* nx = sm.nx[li];
  uint32_t v = (uint32_t)hq & 0xFFFFu;
  hq >>= 16;
  while (v) {
    const uint32_t el = v - 1u;
    v = nx[el];
    if (!v) { v = (uint32_t)hq & 0xFFFFu; hq >>= 16; }
    if (((A1 - Pl[el]) & mask) == 0) f(el);
  }
}

// Where the three layers of the station start in x[] / y[] (element 0 = the 16-byte boundary below the layer's
// first hit), for the exact tests.  z and the thresholds come from the constant bank.
struct StationCtx {
  const int32_t* x;
  const int32_t* y;
  uint32_t g0, g1, g2;
};

// Rare path of phase D: a middle hit with more candidates than the fast path holds in a layer, or more than
// two hits compatible with it in a layer.  Everything exact, no limits: the number of (h0, h2) with h0-h1,
// h2-h1 and h0-h2 compatible (R5).
template <class SM>
__device__ __noinline__ uint32_t triplets_of_h1_slow(const SM& sm, const Params& p, uint32_t s, uint32_t ep, const StationCtx c,
                                                     int32_t x1, int32_t y1, uint32_t kx, uint32_t ky, uint32_t A1) {
  const int R = p.key_R, fsh = p.cell_sh;
  const uint32_t mask = p.key_mask;
  const int32_t z0 = p.z[3 * s], z1 = p.z[3 * s + 1], z2 = p.z[3 * s + 2];
  const int64_t T01 = p.thr_in[s][0], T02 = p.thr_in[s][1], T12 = p.thr_in[s][2];
  const uint64_t T01x2 = p.thr2_in[s][0], T02x2 = p.thr2_in[s][1], T12x2 = p.thr2_in[s][2];
  uint32_t t = 0;
  walk_chains(sm, 1, ep, kx, ky, R, fsh, A1, mask, [&](uint32_t e2) {
    const int32_t x2 = __ldg(c.x + c.g2 + e2), y2 = __ldg(c.y + c.g2 + e2);
    // |x2*z1 - x1*z2| <= T12
    if (win_q(x2, z1, anchor_q(x1, -z2, T12), T12x2) & win_q(y2, z1, anchor_q(y1, -z2, T12), T12x2))
      walk_chains(sm, 0, ep, kx, ky, R, fsh, A1, mask, [&](uint32_t e0) {
        const int32_t x0 = __ldg(c.x + c.g0 + e0), y0 = __ldg(c.y + c.g0 + e0);
        // |x0*z1 - x1*z0| <= T01 and |x2*z0 - x0*z2| <= T02
        const bool ok = win_q(x0, z1, anchor_q(x1, -z0, T01), T01x2) & win_q(y0, z1, anchor_q(y1, -z0, T01), T01x2) &
                        win_q(x2, z0, anchor_q(x0, -z2, T02), T02x2) & win_q(y2, z0, anchor_q(y0, -z2, T02), T02x2);
        t += ok ? 1u : 0u;
      });
  });
  return t;
}

// CLS: the list this kernel works on.  SPILL: station lists beyond LISTCAP go to a per-CTA global scratch and no
// table can overflow (K1CAP >= CAP + 8), so the kernel never hands an event on (class G and list X); without it
// an overflowing event is appended to list X.
template <class SM, int CLS, int MINB, bool SPILL, bool STATIC_SMEM>
__global__ void __launch_bounds__(32 * SM::W, MINB)
    team_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                const uint32_t* __restrict__ off, uint32_t* __restrict__ n_triplets, uint32_t* __restrict__ n_candidates,
                uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ list,
                uint32_t* __restrict__ list_x, uint32_t* __restrict__ spill) {
  constexpr int W = SM::W, CAP = SM::CAP, K1CAP = SM::K1CAP, LISTCAP = SM::LISTCAP, NHEAD = SM::NHEAD;
  constexpr uint32_t kCand = 4;  // candidates per middle hit and layer the fast path of phase D holds
  static_assert(!SPILL || K1CAP >= CAP + 8, "a spilling kernel must hold any station");
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  __shared__ __align__(16) unsigned char smem_static[STATIC_SMEM ? sizeof(SM) : 16];
  SM& sm = *reinterpret_cast<SM*>(STATIC_SMEM ? smem_static : smem_dyn);
  constexpr uint32_t T = 32 * W;
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t S = p.S, L = p.L;
  const uint32_t n_list = ctrl->count[CLS];
  const int fsh = p.cell_sh, R = p.key_R;
  const uint32_t kmask = p.key_mask, kadd = p.key_add;
  // spill area of this CTA: list entries beyond LISTCAP, [2 lists][x, y, c][CAP] words
  uint32_t* const spill_cta = SPILL ? spill + (size_t)blockIdx.x * 6 * CAP : nullptr;
  int32_t* const spill_i = reinterpret_cast<int32_t*>(spill_cta);

  // pulls station s of the event with offsets o[] into L2 (all threads; one 128-byte line per thread and trip)
  auto prefetch_station = [&](const uint32_t* o, uint32_t s) {
    const uint32_t la = o[3 * s] >> 5, lb = (o[3 * s + 3] + 31u) >> 5;  // 128-byte lines of x[] and of y[]
    for (uint32_t l = la + tid; l < lb; l += T) {
      prefetch_l2(x + (size_t)l * 32);
      prefetch_l2(y + (size_t)l * 32);
    }
  };

  for (uint32_t i = tid; i < 3 * 128; i += T) (&sm.occ[0][0])[i] = 0;
  for (uint32_t i = tid; i < (uint32_t)NHEAD; i += T) sm.head[i] = 0;
  if (tid == 0) {
    sm.li[0] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.li[1] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.acc[0] = sm.acc[1] = 0;
    sm.ucount[0] = sm.ucount[1] = 0;
    sm.n1k[0] = sm.n1k[1] = 0;
    sm.fail = 0;
  }
  team_sync<W>();
  if (sm.li[0] >= n_list) return;
  {  // offsets of the first event
    const uint32_t e = __ldg(list + sm.li[0]);
    for (uint32_t i = tid; i <= L; i += T) sm.off[0][i] = __ldg(off + (size_t)e * L + i);
  }
  team_sync<W>();
  uint32_t sp = 0;   // parity of the per-station list counters
  uint32_t kp = 0;   // parity of the kept-hit counter
  uint32_t ob = 0;   // which of sm.off[] holds this event
  uint32_t ep = 0;   // epoch of the chain heads: one per searched station

  for (uint32_t it4 = 0;; it4 = (it4 + 1) & 3u, ob ^= 1u) {
    const uint32_t li = sm.li[it4];
    if (li >= n_list) break;
    const uint32_t li_next = sm.li[(it4 + 1) & 3u];
    if (tid == 0) sm.li[(it4 + 2) & 3u] = atomicAdd(&ctrl->work[CLS], 1u);
    const uint32_t e = __ldg(list + li);
    const uint32_t* const o = sm.off[ob];
    const bool has_next = li_next < n_list;
    if (has_next) {  // offsets of the next event: visible after this event's first barrier
      const uint32_t e2 = __ldg(list + li_next);
      for (uint32_t i = tid; i <= L; i += T) sm.off[ob ^ 1u][i] = __ldg(off + (size_t)e2 * L + i);
    }
    if (tid < S) sm.ntr[tid] = 0;
    uint32_t todo = searchable_mask(o, S);  // stations still to search
    uint32_t nprev = 0;
    bool dead = todo != (S >= 32 ? FULL : ((1u << S) - 1u));  // a chain needs a triplet in every station
    bool failed = false;                                       // the event was handed on to list X
    int cur = 0;
    while (todo) {
      const uint32_t s = (uint32_t)__ffs((int)todo) - 1u;
      todo &= todo - 1u;
      const uint32_t b0 = o[3 * s], b1 = o[3 * s + 1], b2 = o[3 * s + 2], b3 = o[3 * s + 3];
      const uint32_t n0 = b1 - b0, n1 = b2 - b1, n2 = b3 - b2;
      // quads (4 consecutive elements from a 16-byte boundary) of the three layers: layer l starts at element
      // b_l & 3 of its first quad
      const uint32_t st0 = b0 & 3u, st1 = b1 & 3u, st2 = b2 & 3u;
      const uint32_t nq0 = (st0 + n0 + 3u) >> 2, nq1 = (st1 + n1 + 3u) >> 2, nq01 = nq0 + nq1, nqt = nq01 + ((st2 + n2 + 3u) >> 2);
      const uint32_t g0 = b0 & ~3u, g1 = b1 & ~3u, g2 = b2 & ~3u;
      if (++ep == 0x10000u) {  // the epoch tag wrapped: start over with an empty table
        team_sync<W>();
        for (uint32_t i = tid; i < (uint32_t)NHEAD; i += T) sm.head[i] = 0;
        team_sync<W>();
        ep = 1;
      }
      // ---- A: packed keys, occupancy bitmaps, chains of layers 0 and 2.  Elements of a quad outside the layer
      // (<= 3 at either end: hits of the neighbouring layers) only add bits to the bitmap, which keeps the filter
      // a superset; their chain push goes to a head nobody walks.
      {
        constexpr int XS = 6 - SM::TXB, YS = 6 - SM::TYB;
        constexpr uint32_t MX = (1u << SM::TXB) - 1u, MY = (1u << SM::TYB) - 1u;
        const uint32_t tag = ep << 16;
        // layers 0 and 2: quads [0, nq0) and [nq0, nq0 + nq2)
        const uint32_t nq2 = nqt - nq01, nq02 = nq0 + nq2;
#pragma unroll 1
        for (uint32_t qi = tid; qi < nq02; qi += T) {
          const bool l2 = qi >= nq0;
          const uint32_t q = l2 ? qi - nq0 : qi;
          const int32_t M = p.key_mul[3 * s + (l2 ? 2 : 0)];
          const uint32_t g = l2 ? g2 : g0, st = l2 ? st2 : st0, nl = l2 ? n2 : n0;
          const int4 xv = __ldg(reinterpret_cast<const int4*>(x + g) + q);
          const int4 yv = __ldg(reinterpret_cast<const int4*>(y + g) + q);
          const int32_t xs[4] = {xv.x, xv.y, xv.z, xv.w}, ys[4] = {yv.x, yv.y, yv.z, yv.w};
          uint32_t* const occ = sm.occ[l2 ? 2 : 0];
          uint32_t* const hd = sm.head + (l2 ? NHEAD / 2 : 0);
          uint16_t* const nx = sm.nx[l2 ? 1 : 0] + 4 * q;
          uint32_t Pk[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            Pk[k] = packed_key(xs[k], ys[k], M);
            const uint32_t c2 = (Pk[k] >> fsh) & 0x003F003Fu;  // fx | fy << 16
            atomicOr(&occ[((c2 >> 15) & 0x7Eu) | ((c2 >> 5) & 1u)], 1u << (c2 & 31u));
            const uint32_t cc = (((c2 >> XS) & MX) << SM::TYB) | ((c2 >> (16 + YS)) & MY);
            const uint32_t old = atomicExch((4 * q + k - st < nl) ? &hd[cc] : &sm.trash, tag | (4 * q + k + 1u));
            nx[k] = (old >> 16) == ep ? (uint16_t)old : (uint16_t)0;
          }
          *reinterpret_cast<uint4*>(&sm.P[l2 ? 2 : 0][4 * q]) = make_uint4(Pk[0], Pk[1], Pk[2], Pk[3]);
        }
        // layer 1: keys and bitmap only
        {
          const int32_t M = p.key_mul[3 * s + 1];
#pragma unroll 1
          for (uint32_t q = tid; q < nq1; q += T) {
            const int4 xv = __ldg(reinterpret_cast<const int4*>(x + g1) + q);
            const int4 yv = __ldg(reinterpret_cast<const int4*>(y + g1) + q);
            const int32_t xs[4] = {xv.x, xv.y, xv.z, xv.w}, ys[4] = {yv.x, yv.y, yv.z, yv.w};
            uint32_t Pk[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              Pk[k] = packed_key(xs[k], ys[k], M);
              const uint32_t c2 = (Pk[k] >> fsh) & 0x003F003Fu;
              atomicOr(&sm.occ[1][((c2 >> 15) & 0x7Eu) | ((c2 >> 5) & 1u)], 1u << (c2 & 31u));
            }
            *reinterpret_cast<uint4*>(&sm.P[1][4 * q]) = make_uint4(Pk[0], Pk[1], Pk[2], Pk[3]);
          }
        }
        // the next station to search (of this event, else the first of the next event) -> L2
        if (todo) {
          prefetch_station(o, (uint32_t)__ffs((int)todo) - 1u);
        } else if (has_next) {
          const uint32_t m2 = searchable_mask(sm.off[ob ^ 1u], S);
          if (m2) prefetch_station(sm.off[ob ^ 1u], (uint32_t)__ffs((int)m2) - 1u);
        }
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
      // ---- C (a6): keep the middle hits whose cell is in J (ballot/popc; one atomic per warp pass)
#pragma unroll 1
      for (uint32_t q0 = warp * 32u; q0 < nq1; q0 += T) {
        const uint32_t q = q0 + lane;
        uint4 Pq = make_uint4(0, 0, 0, 0);
        if (q < nq1) Pq = *reinterpret_cast<const uint4*>(&sm.P[1][4 * q]);
        const uint32_t Pk[4] = {Pq.x, Pq.y, Pq.z, Pq.w};
        uint32_t km[4], tot = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint32_t c2 = (Pk[k] >> fsh) & 0x003F003Fu;
          const bool keep = q < nq1 && (4 * q + k - st1 < n1) && ((sm.J[((c2 >> 15) & 0x7Eu) | ((c2 >> 5) & 1u)] >> (c2 & 31u)) & 1u);
          km[k] = __ballot_sync(FULL, keep);
          tot += __popc(km[k]);
        }
        if (tot) {
          uint32_t pos = 0;
          if (lane == 0) pos = atoms_add(&sm.n1k[kp], tot);
          pos = __shfl_sync(FULL, pos, 0);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            if ((km[k] >> lane) & 1u) {
              const uint32_t w = pos + __popc(km[k] & lanemask_lt());
              if (w < (uint32_t)K1CAP) sm.k1[w] = (uint16_t)(4 * q + k); else sm.fail = 1;
            }
            pos += __popc(km[k]);
          }
        }
      }
      team_sync<W>();
      // ---- D (a5): two lanes per kept middle hit (side 0: layer 0, side 1: layer 2); the rows of 16 middle hits
      // go round the warps, starting at warp s
      {
        for (uint32_t i = tid; i < 3 * 128; i += T) (&sm.occ[0][0])[i] = 0;  // free since B
        if (tid == 0) sm.n1k[kp ^ 1u] = 0;                                     // the next station's counter
        const uint32_t n1kept = min(sm.n1k[kp], (uint32_t)K1CAP);
        const uint32_t side = lane & 1u;
        const int32_t z0 = p.z[3 * s], z1 = p.z[3 * s + 1], z2 = p.z[3 * s + 2];
        // this lane tests hits of layer 2*side (z_c) against h1:  |x_c*z1 - x1*z_c| <= T_c1
        const int32_t zc = side ? z2 : z0;
        const int64_t Tc1 = p.thr_in[s][2 * side];
        const uint64_t Tc1x2 = p.thr2_in[s][2 * side];
        const uint32_t gc = side ? g2 : g0;
        unsigned long long trip = 0;
#pragma unroll 1
        for (uint32_t base = ((warp - s) & (W - 1)) * 16u; base < n1kept; base += T / 2) {
          const uint32_t j = base + (lane >> 1);
          uint32_t t = 0;           // triplets with this middle hit
          int32_t x1 = 0, y1 = 0;
          uint32_t np = 0, pk = 0;  // hits of my layer compatible with h1: number, the first two (element, 16 bits each)
          uint32_t P1 = 0;
          bool slow = false;
          if (j < n1kept) {
            const uint32_t e1 = sm.k1[j];
            P1 = sm.P[1][e1];
            x1 = __ldg(x + g1 + e1);
            y1 = __ldg(y + g1 + e1);
            // candidates of my layer: hits on the chains that pass the packed test
            unsigned long long cd = 0;
            uint32_t nc = 0;
            walk_chains(sm, side, ep, P1 & 0xFFFFu, P1 >> 16, R, fsh, P1 + kadd, kmask, [&](uint32_t el) {
              if (nc < kCand) cd |= (unsigned long long)el << (16 * nc);
              ++nc;
            });
            slow = nc > kCand;
            if (!slow && nc) {
              const int64_t Qx = anchor_q(x1, -zc, Tc1), Qy = anchor_q(y1, -zc, Tc1);
              for (; nc; --nc, cd >>= 16) {
                const uint32_t ec = (uint32_t)cd & 0xFFFFu;
                if (win_q(__ldg(x + gc + ec), z1, Qx, Tc1x2) & win_q(__ldg(y + gc + ec), z1, Qy, Tc1x2)) {
                  if (np < 2) pk |= ec << (16 * np);
                  ++np;
                }
              }
              slow = np > 2;
            }
          }
          // the two lanes of a middle hit swap what they found
          const uint32_t np_o = __shfl_xor_sync(FULL, np, 1), pk_o = __shfl_xor_sync(FULL, pk, 1);
          slow |= __shfl_xor_sync(FULL, (int)slow, 1) != 0;
          if (slow) {
            if (side == 0)
              t = triplets_of_h1_slow(sm, p, s, ep, StationCtx{x, y, g0, g1, g2}, x1, y1, P1 & 0xFFFFu, P1 >> 16, P1 + kadd);
          } else if (np && np_o) {
            // (h0, h2) pairs: the lane of side i takes h0 number i against all h2   (|x2*z0 - x0*z2| <= T02)
            const uint32_t np0 = side ? np_o : np, pk0 = side ? pk_o : pk, np2 = side ? np : np_o;
            uint32_t q2 = side ? pk : pk_o;
            if (side < np0) {
              const uint32_t e0 = (pk0 >> (16 * side)) & 0xFFFFu;
              const int64_t T02 = p.thr_in[s][1];
              const uint64_t T02x2 = p.thr2_in[s][1];
              const int64_t Qx = anchor_q(__ldg(x + g0 + e0), -z2, T02), Qy = anchor_q(__ldg(y + g0 + e0), -z2, T02);
              for (uint32_t n = np2; n; --n, q2 >>= 16)
                t += (win_q(__ldg(x + g2 + (q2 & 0xFFFFu)), z0, Qx, T02x2) & win_q(__ldg(y + g2 + (q2 & 0xFFFFu)), z0, Qy, T02x2)) ? 1u : 0u;
            }
          }
          t += __shfl_xor_sync(FULL, t, 1);  // both lanes now hold the middle hit's triplet count
          if (side) t = 0;
          trip += t;
          // a6: middle hits with triplets -> the station's list (distinct hits: every h1 has one side-0 lane)
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
                const uint32_t o2 = pos - LISTCAP;
                spill_i[(cur * 3 + 0) * CAP + o2] = x1; spill_i[(cur * 3 + 1) * CAP + o2] = y1;
                spill_cta[(cur * 3 + 2) * CAP + o2] = t;
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
      kp ^= 1u;
      team_sync<W>();

      // ---- F: the search is over: the chains are free
      if (!SPILL && sm.fail) { failed = true; break; }
      const uint32_t ncur = dead ? 0u : sm.ucount[sp];
      if (tid == 0) {
        sm.ntr[s] = sat32(sm.acc[sp]);
        sm.acc[sp ^ 1u] = 0;
        sm.ucount[sp ^ 1u] = 0;
      }
      // ---- a7: chain counts c_s[u] = m_u * sum over linked t of c_{s-1}[t], saturating (R9).  Small teams: warp
      // 0 alone, while the others go on.
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
    // ---- candidates = sum over the last station's middle hits; a8: one writer per output
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
      if (lane < S) n_triplets[(size_t)e * S + lane] = sm.ntr[lane];
    }
    team_sync<W>();
  }
}

}  // namespace cbm

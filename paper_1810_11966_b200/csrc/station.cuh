// station.cuh -- station_kernel: steps a4..a8 for the events of class H, one WARP per (event, station).
//
// Work item = one station of one event of the class list (item = list position * S + station), fetched by the
// warps of a persistent grid with an atomic cursor.  A warp owns its tables in shared memory and never meets a
// CTA barrier; the stations of an event are searched by whichever warps fetch them and the warp that finishes
// an event's last station links the stations' lists (a7) and writes the event's results (a8).
//
// Per station, with the middle layer as anchor (R8: linking needs only the middle hit):
//   A   layers 0 and 2 are read from global memory once, four consecutive hits per lane and coordinate (128-bit
//       loads; the lines were pulled into L2 one item ahead).  Every hit gets its slope keys (kx, ky), sets the bit
//       of its fine cell in its layer's 64 x 64 occupancy bitmap and is pushed on the chain of its coarse cell in
//       ONE table for both layers (atomicExch on the head; node word = 11 + 11 key bits | link).
//   B   J = dilate3x3(occ0) & dilate3x3(occ2) (64-bit rows in registers, neighbours by shuffle).
//   C   layer 1 is read, two hits per lane; a middle hit whose fine cell is not in J cannot have both a compatible
//       h0 and a compatible h2; the others are compacted (ballot/popc).
//   D   dense work lists instead of per-lane chain walks:
//       D1  lane <-> kept middle hit: the heads of the <= 2 x 2 coarse cells its window touches; the head element
//           gets the packed key test of both projections against the middle hit (it never rejects a compatible
//           pair); a passing element is recorded in the middle hit's slot of its layer (count and the first three
//           elements); the element's chain link becomes an item (middle hit, element);
//       D2  lane <-> item: the same test, record (shared-memory atomics) and link for the chains' further elements;
//       D4  lane <-> middle hit with candidates in both layers: exact int64 window tests h0-h1, h2-h1, h0-h2
//           -> number of triplets with this middle hit; (index, count) goes to the station's list in global memory.
//   F   n_triplets of the station; the last station of the event to finish runs the chain count over the lists.
//
// Accept/reject never uses a key, a cell or a bitmap: those only decide which pairs get the exact test, and the
// pairs tested are a proven superset of the compatible ones.
#pragma once
#include "ptx.cuh"
#include "team.cuh"

namespace cbm {

constexpr int kStEnt = 32;  // middle hits with triplets a station list holds; an event with more goes to list X

template <int CAP_, int TXB_, int TYB_>
struct StationSmem {
  static constexpr int CAP = CAP_, TXB = TXB_, TYB = TYB_;
  static constexpr int LCAP = CAP + 8;            // a layer as it lies in x[], from the 16-byte boundary below it
  static constexpr int NHEAD = 1 << (TXB + TYB);
  static constexpr int KCAP = 128;                // kept middle hits per round of phases C and D
  static constexpr int ICAP = 32 + 4 * 32;
  static_assert(2 * LCAP + 1 < 1024 && LCAP < 512 && KCAP <= 128 && KCAP % 64 == 0, "field widths");
  static_assert((long long)CAP * CAP < (1 << 18), "entry = index | triplets << 9");
  alignas(16) uint32_t node[2 * LCAP];            // layers 0 and 2: link | (kx mod 2^11) << 10 | (ky mod 2^11) << 21
  alignas(16) uint32_t head[NHEAD];               // chains of both layers: element + 1; 0 = empty
  alignas(16) uint32_t occ[2][128];               // occupancy bitmaps, row fy = 64 bits, bit fx; after B: slots
  alignas(16) uint32_t J[128];
  uint32_t kP[KCAP];                              // kept middle hits: packed key (kx mod 2^16 | ky mod 2^16 << 16),
                                                  // after D1 the anchor word of the packed test
  uint32_t items[ICAP];                           // survivor | (element + 1) << 8
  uint16_t kI[KCAP];                              // kept middle hits: hit index in layer 1
  uint32_t trash;                                 // chain head of the elements of a quad that are not hits of the layer
};

struct StationGeo {
  const int32_t* x;
  const int32_t* y;
  uint32_t b0, b1, b2, n0, n1, n2;  // first hit and size of the three layers
  int32_t z0, z1, z2;
  int64_t T01, T02, T12;
};

// Rare path of phase D: a middle hit with more than two compatible hits in a layer.  Warp-cooperative, exact,
// no limits: the number of (h0, h2) with h0-h1, h2-h1 and h0-h2 compatible (R5).
__device__ __noinline__ uint32_t station_triplets_slow(const StationGeo g, int32_t x1, int32_t y1) {
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  const uint32_t lane = threadIdx.x & 31;
  const int64_t Q12x = anchor_q(x1, -g.z2, g.T12), Q12y = anchor_q(y1, -g.z2, g.T12);
  const int64_t Q01x = anchor_q(x1, -g.z0, g.T01), Q01y = anchor_q(y1, -g.z0, g.T01);
  uint32_t t = 0;
  for (uint32_t j2 = lane; j2 < ((g.n2 + 31u) & ~31u); j2 += 32) {
    int32_t x2 = 0, y2 = 0;
    bool ok2 = false;
    if (j2 < g.n2) {
      x2 = __ldg(g.x + g.b2 + j2); y2 = __ldg(g.y + g.b2 + j2);
      ok2 = win_q(x2, g.z1, Q12x, 2 * (uint64_t)g.T12) & win_q(y2, g.z1, Q12y, 2 * (uint64_t)g.T12);
    }
    uint32_t m = __ballot_sync(FULL, ok2);
    while (m) {
      const int src = __ffs((int)m) - 1;
      m &= m - 1;
      const int32_t xs = __shfl_sync(FULL, x2, src), ys = __shfl_sync(FULL, y2, src);
      for (uint32_t j0 = lane; j0 < g.n0; j0 += 32) {
        const int32_t x0 = __ldg(g.x + g.b0 + j0), y0 = __ldg(g.y + g.b0 + j0);
        const bool ok = win_q(x0, g.z1, Q01x, 2 * (uint64_t)g.T01) & win_q(y0, g.z1, Q01y, 2 * (uint64_t)g.T01) &
                        win_q(xs, g.z0, anchor_q(x0, -g.z2, g.T02), 2 * (uint64_t)g.T02) &
                        win_q(ys, g.z0, anchor_q(y0, -g.z2, g.T02), 2 * (uint64_t)g.T02);
        t += ok ? 1u : 0u;
      }
    }
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) t += __shfl_xor_sync(FULL, t, d);
  return t;
}

// a7, a8 for one event whose S station lists are complete (called by one whole warp).
// st_cnt / st_ent: entries of item li * S + s.  Returns false if a list overflowed (the event goes to list X).
__device__ __noinline__ bool station_link(const Params& p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                                          const uint32_t* __restrict__ off, uint32_t e, uint32_t li,
                                          const uint32_t* st_cnt, const uint32_t* st_ent, uint32_t* __restrict__ n_candidates,
                                          uint8_t* __restrict__ accept) {
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t S = p.S, L = p.L;
  uint32_t cnt = 1, b1 = 0;
  if (lane < S) {
    cnt = __ldcg(st_cnt + (size_t)li * S + lane);
    b1 = __ldg(off + (size_t)e * L + 3 * lane + 1);
  }
  if (__any_sync(FULL, cnt > (uint32_t)kStEnt)) return false;
  unsigned long long total = 0;
  if (!__any_sync(FULL, cnt == 0)) {
    int32_t xp = 0, yp = 0;
    uint32_t cp = 0, nprev = 0;
    bool alive = true;
    for (uint32_t s = 0; s < S && alive; ++s) {
      const uint32_t n = __shfl_sync(FULL, cnt, s), base = __shfl_sync(FULL, b1, s);
      int32_t xu = 0, yu = 0;
      uint32_t tu = 0;
      if (lane < n) {
        const uint32_t ent = __ldcg(st_ent + ((size_t)li * S + s) * kStEnt + lane);
        tu = ent >> 9;
        xu = __ldg(x + base + (ent & 511u));
        yu = __ldg(y + base + (ent & 511u));
      }
      uint32_t cu = tu;
      if (s > 0) {
        // |x_t*zB - x_u*zA| <= TL, t in station s-1 (zA), u in station s (zB)
        const int32_t nzA = -p.z[3 * (s - 1) + 1], zB = p.z[3 * s + 1];
        const int64_t TL = p.thr_link[s];
        const uint64_t TLx2 = p.thr2_link[s];
        const int64_t Qx = anchor_q(xu, nzA, TL), Qy = anchor_q(yu, nzA, TL);
        unsigned long long a = 0;
        for (uint32_t v = 0; v < nprev; ++v) {
          const int32_t xv = __shfl_sync(FULL, xp, v), yv = __shfl_sync(FULL, yp, v);
          const uint32_t cv = __shfl_sync(FULL, cp, v);
          if (win_q(xv, zB, Qx, TLx2) & win_q(yv, zB, Qy, TLx2)) a += cv;
        }
        cu = lane < n ? sat32((unsigned long long)sat32(a) * tu) : 0u;
      }
      alive = __any_sync(FULL, cu != 0);
      xp = xu; yp = yu; cp = cu; nprev = n;
    }
    if (alive) {
      total = cp;
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) total += __shfl_xor_sync(FULL, total, d);
    }
  }
  if (lane == 0) {
    const uint32_t cand = sat32(total);
    n_candidates[e] = cand;
    accept[e] = cand >= p.min_candidates ? 1 : 0;
  }
  return true;
}

__device__ __forceinline__ uint32_t atoms_exch_addr(uint32_t addr, uint32_t v) {
  uint32_t old;
  asm volatile("atom.shared.exch.b32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(v) : "memory");
  return old;
}
__device__ __forceinline__ void reds_or_addr(uint32_t addr, uint32_t v) {
  asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lds_addr(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t atoms_add_addr(uint32_t addr, uint32_t v) {
  uint32_t old;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(v) : "memory");
  return old;
}

#ifdef ST_DEBUG
__device__ unsigned long long g_st_dbg[16];
#define ST_DBG(i, v) do { const unsigned long long v_ = (unsigned long long)(v); if (lane == 0) atomicAdd(&g_st_dbg[i], v_); } while (0)
#else
#define ST_DBG(i, v) do { } while (0)
#endif
constexpr uint32_t kSlotCap = 3;  // elements a slot records: count << 27 | e2 << 18 | e1 << 9 | e0  (element + 1)

template <class SM, int WPC, int CLS, int MINB>
__global__ void __launch_bounds__(32 * WPC, MINB)
    station_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                   const uint32_t* __restrict__ off, uint32_t* __restrict__ n_triplets, uint32_t* __restrict__ n_candidates,
                   uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ list,
                   uint32_t* __restrict__ list_x, uint32_t* __restrict__ st_cnt, uint32_t* __restrict__ st_ent,
                   uint32_t* __restrict__ done) {
  constexpr int LCAP = SM::LCAP, KCAP = SM::KCAP, NHEAD = SM::NHEAD;
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  constexpr int XS = 6 - SM::TXB, YS = 6 - SM::TYB;  // fine cells per coarse cell (log2), >= 1
  constexpr uint32_t MX = (1u << SM::TXB) - 1u, MY = (1u << SM::TYB) - 1u;
  static_assert(XS >= 1 && YS >= 1, "a coarse cell spans at least two fine cells");
  static_assert(KCAP * 2 <= 256, "the slots live in the bitmaps");
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  SM& sm = reinterpret_cast<SM*>(smem_dyn)[warp];
  const uint32_t a_node = smem_u32(sm.node), a_head = smem_u32(sm.head), a_occ = smem_u32(sm.occ), a_J = smem_u32(sm.J);
  const uint32_t a_slot = a_occ;
  const uint32_t S = p.S, L = p.L;
  const uint32_t n_items = ctrl->count[CLS] * S;
  const int fsh = p.cell_sh, R = p.key_R;
  // packed test on the node words (fields of 11 bits at bits 10 and 21, link in bits 0..9):
  // |dkx|, |dky| <= R  =>  ((A - node) & nmask) == 0 with A = fields(h1) + nadd, low 10 bits all ones (no borrow)
  const uint32_t nhalf = p.key_mask & 0x7FFu;  // bits >= m of a field, 2^m >= 2R + 3
  const uint32_t nmask = (nhalf << 10) | (nhalf << 21);
  const uint32_t nadd = ((uint32_t)R << 10) | ((uint32_t)(R + 1) << 21);
  const uint32_t lt = lanemask_lt();

  auto fetch = [&]() {
    uint32_t w = 0;
    if (lane == 0) w = atomicAdd(&ctrl->work[CLS], 1u);
    return __shfl_sync(FULL, w, 0);
  };
  // the item's event and the four offsets of its station (lanes 0..3 load, every lane gets all four)
  auto load_item = [&](uint32_t w, uint32_t& e, uint32_t& s, uint32_t& b0, uint32_t& b1, uint32_t& b2, uint32_t& b3) {
    const uint32_t li = w / S;
    s = w - li * S;
    e = __ldg(list + li);
    uint32_t o = 0;
    if (lane < 4) o = __ldg(off + (size_t)e * L + 3 * s + lane);
    b0 = __shfl_sync(FULL, o, 0); b1 = __shfl_sync(FULL, o, 1); b2 = __shfl_sync(FULL, o, 2); b3 = __shfl_sync(FULL, o, 3);
  };

  // Three items in flight per warp: w0 is searched, w1's offsets are known and its hits are on their way into L2,
  // w2's event and offsets are being loaded; the cursor fetch of the item after those is pending in lane 0.
  uint32_t w0 = fetch(), w1 = fetch(), w2 = fetch();
  uint32_t e = 0, s = 0, b0 = 0, b1 = 0, b2 = 0, b3 = 0;
  uint32_t e_n = 0, s_n = 0, nb0 = 0, nb1 = 0, nb2 = 0, nb3 = 0;
  if (w0 < n_items) load_item(w0, e, s, b0, b1, b2, b3);
  if (w1 < n_items) load_item(w1, e_n, s_n, nb0, nb1, nb2, nb3);

  while (w0 < n_items) {
    uint32_t wp = 0;
    if (lane == 0) wp = atomicAdd(&ctrl->work[CLS], 1u);
    const bool v2 = w2 < n_items;
    uint32_t e2 = 0, s2 = 0, o2 = 0;
    if (v2) {
      const uint32_t li2 = w2 / S;
      s2 = w2 - li2 * S;
      e2 = __ldg(list + li2);
    }
    const uint32_t n0 = b1 - b0, n1 = b2 - b1, n2 = b3 - b2;
    const bool search = (n0 != 0) & (n1 != 0) & (n2 != 0);
    uint32_t trip = 0;  // triplets found by this lane
    uint32_t ne = 0;    // entries of the station's list (warp-uniform)
    if (search) {
      const uint32_t st0 = b0 & 3u, st2 = b2 & 3u;
      const uint32_t g0 = b0 & ~3u, g2 = b2 & ~3u;
      const uint32_t nq0 = (st0 + n0 + 3u) >> 2, nq02 = nq0 + ((st2 + n2 + 3u) >> 2);
      const int32_t M0 = p.key_mul[3 * s], M2 = p.key_mul[3 * s + 2];
      // quad qi of layers 0 and 2 (layer 2 follows layer 0): its address in x[] (y[] at the same index)
      auto quad_index = [&](uint32_t qi) { return qi >= nq0 ? (g2 >> 2) + (qi - nq0) : (g0 >> 2) + qi; };
      int4 xv = make_int4(0, 0, 0, 0), yv = xv;
      if (lane < nq02) {  // first trip of phase A: in flight while the tables are cleared
        const uint32_t gi = quad_index(lane);
        xv = __ldg(reinterpret_cast<const int4*>(x) + gi);
        yv = __ldg(reinterpret_cast<const int4*>(y) + gi);
      }
      // ---- tables empty
      {
        uint4* const hv = reinterpret_cast<uint4*>(sm.head);
#pragma unroll
        for (uint32_t i = 0; i < NHEAD / 4 / 32; ++i) hv[lane + 32 * i] = make_uint4(0, 0, 0, 0);
        uint4* const ov = reinterpret_cast<uint4*>(&sm.occ[0][0]);
        ov[lane] = make_uint4(0, 0, 0, 0);
        ov[lane + 32] = make_uint4(0, 0, 0, 0);
      }
      __syncwarp();
      // ---- A: layers 0 and 2.  Quads (4 consecutive elements from a 16-byte boundary); elements of a quad outside
      // the layer (<= 3 at either end: hits of the neighbouring layers) only add bits to the bitmap, which keeps the
      // filter a superset; they are not pushed on a chain.
      const uint32_t a_trash = smem_u32(&sm.trash);
      auto quad = [&](uint32_t qi, const int4& xq, const int4& yq) {
        const bool l2 = qi >= nq0;
        const uint32_t q = l2 ? qi - nq0 : qi;
        const int32_t M = l2 ? M2 : M0;
        const uint32_t nl = l2 ? n2 : n0;
        const uint32_t i0 = 4 * q - (l2 ? st2 : st0);                   // hit index in its layer of the quad's first element
        const uint32_t el1 = (l2 ? (uint32_t)LCAP : 0u) + 4 * q + 1u;   // element number + 1 of the quad's first element
        const uint32_t a_oc = a_occ + (l2 ? 512u : 0u);
        const int32_t xs[4] = {xq.x, xq.y, xq.z, xq.w}, ys[4] = {yq.x, yq.y, yq.z, yq.w};
        uint32_t nd[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const int kx = __mulhi(xs[k], M), ky = __mulhi(ys[k], M);
          const uint32_t fx = (uint32_t)(kx >> fsh), ty = (uint32_t)(ky >> (fsh - 1));  // ty = fy << 1 | .
          // bitmap: row fy = two words, word fx / 32, bit fx % 32
          reds_or_addr(a_oc + (((ty << 2) & 0x1F8u) | ((fx >> 3) & 4u)), 1u << (fx & 31u));
          // coarse cell (fx >> XS, fy >> YS)
          const uint32_t a_hd = a_head + (((fx >> XS) & MX) << (SM::TYB + 2)) + (((ty >> (YS + 1)) & MY) << 2);
          const uint32_t old = atoms_exch_addr((i0 + k < nl) ? a_hd : a_trash, el1 + k);
          nd[k] = (old + ((uint32_t)ky << 21)) | (((uint32_t)kx << 10) & 0x1FFC00u);  // old < 2^10: a sum is an or
        }
        *reinterpret_cast<uint4*>(&sm.node[el1 - 1u]) = make_uint4(nd[0], nd[1], nd[2], nd[3]);
      };
      auto load_quad = [&](uint32_t qi, int4& xq, int4& yq) {
        if (qi < nq02) {
          const uint32_t gi = quad_index(qi);
          xq = __ldg(reinterpret_cast<const int4*>(x) + gi);
          yq = __ldg(reinterpret_cast<const int4*>(y) + gi);
        }
      };
#pragma unroll 1
      for (uint32_t qi = lane; qi < nq02; qi += 64) {  // two trips per turn: the loads of the next trip fly
        int4 xn = make_int4(0, 0, 0, 0), yn = xn;
        load_quad(qi + 32, xn, yn);
        quad(qi, xv, yv);
        load_quad(qi + 64, xv, yv);
        if (qi + 32 < nq02) quad(qi + 32, xn, yn);
      }
      if (v2 && lane < 4) o2 = __ldg(off + (size_t)e2 * L + 3 * s2 + lane);  // used at the end of this item
      // layer 1 in pairs from an 8-byte boundary: the first trip's loads fly during phase B
      const int32_t M1 = p.key_mul[3 * s + 1];
      const uint32_t sp1 = b1 & 1u, h1 = b1 & ~1u;
      const uint32_t npair1 = (sp1 + n1 + 1u) >> 1;
      const int2* const x1p = reinterpret_cast<const int2*>(x + h1);
      const int2* const y1p = reinterpret_cast<const int2*>(y + h1);
      int2 xc = make_int2(0, 0), yc = xc;
      if (lane < npair1) { xc = __ldg(x1p + lane); yc = __ldg(y1p + lane); }
      __syncwarp();
      // ---- B: J = dilate(occ0) & dilate(occ2) on the cyclic grid; lane <-> rows 2*lane, 2*lane + 1
      {
        unsigned long long j0 = ~0ull, j1 = ~0ull;
#pragma unroll
        for (int l = 0; l < 2; ++l) {
          const uint4 r4 = reinterpret_cast<const uint4*>(sm.occ[l])[lane];
          const unsigned long long ra = ((unsigned long long)r4.y << 32) | r4.x, rb = ((unsigned long long)r4.w << 32) | r4.z;
          const unsigned long long rm = __shfl_sync(FULL, rb, (lane + 31) & 31);  // row 2*lane - 1
          const unsigned long long rp = __shfl_sync(FULL, ra, (lane + 1) & 31);   // row 2*lane + 2
          const unsigned long long va = rm | ra | rb, vb = ra | rb | rp;
          j0 &= va | (va << 1) | (va >> 63) | (va >> 1) | (va << 63);
          j1 &= vb | (vb << 1) | (vb >> 63) | (vb >> 1) | (vb << 63);
        }
        reinterpret_cast<uint4*>(sm.J)[lane] = make_uint4((uint32_t)j0, (uint32_t)(j0 >> 32), (uint32_t)j1, (uint32_t)(j1 >> 32));
      }
      __syncwarp();  // from here on the bitmaps are the slots of phase D: [survivor][layer]

      const int32_t z0 = p.z[3 * s], z1 = p.z[3 * s + 1], z2 = p.z[3 * s + 2];
      uint32_t pr0 = 0;  // pairs of layer 1 already filtered
      while (pr0 < npair1) {
        // ---- C (a6): keep the middle hits whose fine cell is in J, up to KCAP per round
        uint32_t nk = 0;
        while (pr0 < npair1) {
          const uint32_t pi = pr0 + lane;
          int2 xn = make_int2(0, 0), yn = xn;
          if (pi + 32 < npair1) { xn = __ldg(x1p + pi + 32); yn = __ldg(y1p + pi + 32); }
          const int32_t xs[2] = {xc.x, xc.y}, ys[2] = {yc.x, yc.y};
          uint32_t km[2], P1[2];
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const int kx = __mulhi(xs[k], M1), ky = __mulhi(ys[k], M1);
            const uint32_t fx = (uint32_t)(kx >> fsh);
            const uint32_t wi = ((uint32_t)(ky >> (fsh - 1)) & 0x7Eu) | ((fx >> 5) & 1u);
            const uint32_t jw = lds_addr(a_J + 4u * wi);
            const bool keep = (2 * pi + k - sp1 < n1) & ((jw >> (fx & 31u)) & 1u);  // pi >= npair1: index >= n1
            km[k] = __ballot_sync(FULL, keep);
            P1[k] = __byte_perm((uint32_t)kx, (uint32_t)ky, 0x5410);
          }
          const uint32_t c0 = __popc(km[0]);
          if (nk + c0 + __popc(km[1]) > (uint32_t)KCAP) break;  // the round is full: this trip opens the next one
          if ((km[0] >> lane) & 1u) {
            const uint32_t w = nk + __popc(km[0] & lt);
            sm.kP[w] = P1[0];
            sm.kI[w] = (uint16_t)(2 * pi - sp1);
          }
          if ((km[1] >> lane) & 1u) {
            const uint32_t w = nk + c0 + __popc(km[1] & lt);
            sm.kP[w] = P1[1];
            sm.kI[w] = (uint16_t)(2 * pi + 1u - sp1);
          }
          nk += c0 + __popc(km[1]);
          pr0 += 32;
          xc = xn; yc = yn;
        }
        ST_DBG(0, 1); ST_DBG(1, nk);
        __syncwarp();
        // ---- D1 / D2: heads, then the chains' further elements as items, drained in full warp passes
        uint32_t ni = 0;
        auto drain_items = [&](bool all) {
          while (ni >= 32u || (all && ni)) {
            const uint32_t take = min(ni, 32u);
            ni -= take;
            ST_DBG(2, 1); ST_DBG(3, take);
            __syncwarp();
            uint32_t k = 0, link = 0;
            if (lane < take) {
              const uint32_t it = sm.items[ni + lane];
              k = it & 0xFFu;
              const uint32_t el1 = it >> 8;  // element + 1
              const uint32_t w = lds_addr(a_node + 4u * el1 - 4u);
              link = w & 0x3FFu;
              if (((sm.kP[k] - w) & nmask) == 0) {
                const bool side = el1 > (uint32_t)LCAP;
                const uint32_t a_sl = a_slot + 8u * k + (side ? 4u : 0u);
                if ((lds_addr(a_sl) >> 27) <= kSlotCap) {  // at most 4 items of a middle hit per pass: no wrap
                  const uint32_t c = atoms_add_addr(a_sl, 1u << 27) >> 27;
                  if (c < kSlotCap) atoms_add_addr(a_sl, (el1 - (side ? (uint32_t)LCAP : 0u)) << (9u * c));
                }
              }
            }
            const uint32_t cm = __ballot_sync(FULL, link != 0);
            __syncwarp();
            if (link) sm.items[ni + __popc(cm & lt)] = k | (link << 8);
            ni += __popc(cm);
          }
        };
        for (uint32_t kb = 0; kb < nk; kb += 32) {
          const uint32_t k = kb + lane;
          uint32_t hv[4] = {0, 0, 0, 0};
          uint32_t A = 0;
          if (k < nk) {
            const uint32_t P1 = sm.kP[k];
            const uint32_t kx = P1 & 0xFFFFu, ky = P1 >> 16;
            A = ((((kx & 0x7FFu) << 10) | (ky << 21)) + nadd) | 0x3FFu;
            // key_R <= 2^cell_sh and a coarse cell is >= 2^(cell_sh+1) wide: at most two columns and two rows (cyclic)
            const uint32_t lox = ((kx - R) >> (fsh + XS)) & MX, hix = ((kx + R) >> (fsh + XS)) & MX;
            const uint32_t loy = ((ky - R) >> (fsh + YS)) & MY, hiy = ((ky + R) >> (fsh + YS)) & MY;
            hv[0] = sm.head[(lox << SM::TYB) | loy];
            if (hiy != loy) hv[1] = sm.head[(lox << SM::TYB) | hiy];
            if (hix != lox) {
              hv[2] = sm.head[(hix << SM::TYB) | loy];
              if (hiy != loy) hv[3] = sm.head[(hix << SM::TYB) | hiy];
            }
          }
          uint32_t sl[2] = {0, 0};  // this middle hit's slots (layer 0, layer 2), in registers for the heads
          uint32_t lk[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            lk[c] = 0;
            if (hv[c]) {
              const uint32_t w = lds_addr(a_node + 4u * hv[c] - 4u);
              lk[c] = w & 0x3FFu;
              if (((A - w) & nmask) == 0) {
                const bool side = hv[c] > (uint32_t)LCAP;
                const uint32_t j1 = hv[c] - (side ? (uint32_t)LCAP : 0u);  // element in its layer + 1
                uint32_t& r = side ? sl[1] : sl[0];
                if ((r >> 27) < kSlotCap) r += j1 << (9u * (r >> 27));  // a fourth one is counted, not recorded
                r += 1u << 27;
              }
            }
          }
          if (k < nk) {
            sm.kP[k] = A;
            *reinterpret_cast<uint2*>(&sm.occ[0][0] + 2 * k) = make_uint2(sl[0], sl[1]);
          }
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const uint32_t m = __ballot_sync(FULL, lk[c] != 0);
            if (lk[c]) sm.items[ni + __popc(m & lt)] = k | (lk[c] << 8);
            ni += __popc(m);
          }
          drain_items(false);
        }
        drain_items(true);
        __syncwarp();
        // ---- D4: middle hits with candidates in both layers -> exact tests
        uint32_t nj = 0;  // their numbers, compacted into sm.items
        for (uint32_t kb = 0; kb < nk; kb += 32) {
          const uint32_t k = kb + lane;
          bool both = false;
          if (k < nk) {
            const uint2 s02 = *reinterpret_cast<const uint2*>(&sm.occ[0][0] + 2 * k);
            both = (s02.x >> 27) != 0 && (s02.y >> 27) != 0;
          }
#ifdef ST_DEBUG
          {
            uint32_t cc_ = 0, c4_ = 0;
            if (k < nk) { const uint2 s02 = *reinterpret_cast<const uint2*>(&sm.occ[0][0] + 2 * k); cc_ = (s02.x >> 27) + (s02.y >> 27); c4_ = ((s02.x >> 27) > 3) + ((s02.y >> 27) > 3); }
            ST_DBG(9, __reduce_add_sync(FULL, cc_)); ST_DBG(10, __reduce_add_sync(FULL, c4_));
          }
#endif
          const uint32_t m = __ballot_sync(FULL, both);
          if (both) sm.items[nj + __popc(m & lt)] = k;
          nj += __popc(m);
        }
        __syncwarp();
        const int64_t T01 = p.thr_in[s][0], T02 = p.thr_in[s][1], T12 = p.thr_in[s][2];
        const uint64_t T01x2 = p.thr2_in[s][0], T02x2 = p.thr2_in[s][1], T12x2 = p.thr2_in[s][2];
        ST_DBG(4, nj);
        for (uint32_t jb = 0; jb < nj; jb += 32) {
          uint32_t t = 0, i1 = 0, c0 = 0, c2 = 0, s0 = 0, s2w = 0;
          bool slow = false;
          int32_t x1 = 0, y1 = 0;
          if (jb + lane < nj) {
            const uint32_t k = sm.items[jb + lane];
            const uint2 s02 = *reinterpret_cast<const uint2*>(&sm.occ[0][0] + 2 * k);
            s0 = s02.x; s2w = s02.y;
            c0 = s0 >> 27; c2 = s2w >> 27;
            i1 = sm.kI[k];
            slow = c0 > kSlotCap || c2 > kSlotCap;
            if (slow) c0 = c2 = 0;
            x1 = __ldg(x + b1 + i1); y1 = __ldg(y + b1 + i1);
          }
          const uint32_t mc0 = __reduce_max_sync(FULL, c0), mc2 = __reduce_max_sync(FULL, c2);
          ST_DBG(5, mc0); ST_DBG(6, mc2); ST_DBG(7, __popc(__ballot_sync(FULL, slow))); ST_DBG(8, __reduce_add_sync(FULL, c0 + c2));
          // h2 compatible with h1:  |x2*z1 - x1*z2| <= T12
          int32_t x2[kSlotCap], y2[kSlotCap];
          bool ok2[kSlotCap];
          {
            const int64_t Qx = anchor_q(x1, -z2, T12), Qy = anchor_q(y1, -z2, T12);
#pragma unroll
            for (uint32_t b = 0; b < kSlotCap; ++b) {
              x2[b] = 0; y2[b] = 0; ok2[b] = false;
              if (b < mc2) {
                if (b < c2) {
                  const uint32_t j2 = ((s2w >> (9 * b)) & 0x1FFu) - 1u;
                  x2[b] = __ldg(x + g2 + j2); y2[b] = __ldg(y + g2 + j2);
                  ok2[b] = win_q(x2[b], z1, Qx, T12x2) & win_q(y2[b], z1, Qy, T12x2);
                }
              }
            }
          }
          {
            const int64_t Qx = anchor_q(x1, -z0, T01), Qy = anchor_q(y1, -z0, T01);
            for (uint32_t a = 0; a < mc0; ++a) {
              if (a < c0) {
                const uint32_t j0 = ((s0 >> (9 * a)) & 0x1FFu) - 1u;
                const int32_t x0 = __ldg(x + g0 + j0), y0 = __ldg(y + g0 + j0);
                // h0 with h1: |x0*z1 - x1*z0| <= T01;  h2 with h0: |x2*z0 - x0*z2| <= T02
                if (win_q(x0, z1, Qx, T01x2) & win_q(y0, z1, Qy, T01x2)) {
                  const int64_t Px = anchor_q(x0, -z2, T02), Py = anchor_q(y0, -z2, T02);
#pragma unroll
                  for (uint32_t b = 0; b < kSlotCap; ++b)
                    if (ok2[b]) t += (win_q(x2[b], z0, Px, T02x2) & win_q(y2[b], z0, Py, T02x2)) ? 1u : 0u;
                }
              }
            }
          }
          uint32_t sm_ = __ballot_sync(FULL, slow);
          while (sm_) {  // rare: more than kSlotCap candidates in a layer
            const int src = __ffs((int)sm_) - 1;
            sm_ &= sm_ - 1;
            const int32_t xs1 = __shfl_sync(FULL, x1, src), ys1 = __shfl_sync(FULL, y1, src);
            const uint32_t ts = station_triplets_slow(StationGeo{x, y, b0, b1, b2, n0, n1, n2, z0, z1, z2, T01, T02, T12}, xs1, ys1);
            if ((int)lane == src) t = ts;
          }
          trip += t;
          // a6: (index, triplets) of the middle hits with triplets -> the station's list
          const uint32_t am = __ballot_sync(FULL, t != 0);
          if (t) {
            const uint32_t pos = ne + __popc(am & lt);
            if (pos < (uint32_t)kStEnt) st_ent[(size_t)w0 * kStEnt + pos] = i1 | (t << 9);
          }
          ne += __popc(am);
        }
        __syncwarp();
      }
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) trip += __shfl_xor_sync(FULL, trip, d);
    }
    // ---- F: the station's results; the event's last station links
    if (lane == 0) {
      n_triplets[(size_t)e * S + s] = trip;
      st_cnt[w0] = ne;
    }
    __threadfence();
    __syncwarp();
    {
      const uint32_t li = w0 / S;
      uint32_t old = 0;
      if (lane == 0) old = atomicAdd(&done[li], 1u);
      old = __shfl_sync(FULL, old, 0);
      if (old == S - 1u) {
        __threadfence();
        const bool ok = station_link(p, x, y, off, e, li, st_cnt, st_ent, n_candidates, accept);
        if (lane == 0) {
          done[li] = 0;  // ready for the next run
          if (!ok) list_x[atomicAdd(&ctrl->count[kClsX], 1u)] = e;
        }
      }
    }
    // the item after the next one: offsets, hits -> L2 (they are read one item from now)
    if (v2 && !search && lane < 4) o2 = __ldg(off + (size_t)e2 * L + 3 * s2 + lane);
    const uint32_t pb0 = __shfl_sync(FULL, o2, 0), pb1 = __shfl_sync(FULL, o2, 1), pb2 = __shfl_sync(FULL, o2, 2),
                   pb3 = __shfl_sync(FULL, o2, 3);
    if (v2) {
      const uint32_t la = pb0 >> 5, lb = (pb3 + 31u) >> 5;  // 128-byte lines of x[] and of y[]
      for (uint32_t l = la + lane; l < lb; l += 32) {
        prefetch_l2(x + (size_t)l * 32);
        prefetch_l2(y + (size_t)l * 32);
      }
    }
    w0 = w1; w1 = w2; w2 = __shfl_sync(FULL, wp, 0);
    e = e_n; s = s_n; b0 = nb0; b1 = nb1; b2 = nb2; b3 = nb3;
    e_n = e2; s_n = s2; nb0 = pb0; nb1 = pb1; nb2 = pb2; nb3 = pb3;
  }
}

}  // namespace cbm

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
#include <stddef.h>
#include "ptx.cuh"
#include "team.cuh"

namespace cbm {

constexpr int kStEnt = 32;
constexpr uint32_t kPriv = 8;  // candidates of one middle hit the fast path of phase D holds  // middle hits with triplets a station list holds; an event with more goes to list X

template <int CAP_, int TXB_, int TYB_>
struct StationSmem {
  static constexpr int CAP = CAP_, TXB = TXB_, TYB = TYB_;
  static constexpr int LCAP = CAP + 8;            // a layer as it lies in x[], from the 16-byte boundary below it
  static constexpr int NHEAD = 1 << (TXB + TYB);
  static constexpr int KCAP = 96;                 // kept middle hits per round of phases C and D
  static_assert(2 * LCAP + 1 < 1024 && LCAP < 512 && KCAP <= 128 && KCAP % 32 == 0, "field widths");
  static_assert((long long)CAP * CAP < (1 << 18), "entry = index | triplets << 9");
  alignas(16) uint32_t node[2 * LCAP];            // layers 0 and 2: link | (kx mod 2^11) << 10 | (ky mod 2^11) << 21
  alignas(16) uint32_t head[NHEAD];               // chains of both layers: element + 1; 0 = empty
  alignas(16) uint32_t occ[2][128];               // occupancy bitmaps, row fy = 64 bits, bit fx; after B: the pair list
                                                  // (middle hit | (element + 1) << 8), then the joiners of phase D4
  alignas(16) uint32_t J[128];
  alignas(8) uint32_t slot[2 * KCAP];             // [kept middle hit][layer 0, layer 2]: count << 27 | e2 << 18 | e1 << 9 | e0
  uint32_t kP[KCAP];                              // kept middle hits: packed key (kx mod 2^16 | ky mod 2^16 << 16)
  uint16_t kI[KCAP];                              // kept middle hits: hit index in layer 1; bit 15: slow path
  uint16_t priv[32 * kPriv];                      // per lane: elements that passed the packed test (phase D1)
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
__device__ __forceinline__ void sts_addr(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void sts_u16_addr(uint32_t addr, uint32_t v) {
  asm volatile("{ .reg .u16 t; cvt.u16.u32 t, %1; st.shared.u16 [%0], t; }" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lds_u16_addr(uint32_t addr) {
  uint32_t v;
  asm volatile("{ .reg .u16 t; ld.shared.u16 t, [%1]; cvt.u32.u16 %0, t; }" : "=r"(v) : "r"(addr));
  return v;
}

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
  static_assert(32 * kPriv <= 256 && KCAP <= 256, "the pair list lives in the bitmaps");
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  SM& sm = reinterpret_cast<SM*>(smem_dyn)[warp];
  const uint32_t a_node = smem_u32(sm.node), a_head = smem_u32(sm.head), a_occ = smem_u32(sm.occ), a_J = smem_u32(sm.J);
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
      // layer 1, one hit per lane and trip: the first trip's loads fly during phase B
      const int32_t M1 = p.key_mul[3 * s + 1];
      const int32_t* const x1p = x + b1;
      const int32_t* const y1p = y + b1;
      int32_t xc = 0, yc = 0;
      if (lane < n1) { xc = __ldg(x1p + lane); yc = __ldg(y1p + lane); }
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
      __syncwarp();  // from here on the bitmaps are the pair list of phase D

      const int32_t z0 = p.z[3 * s], z1 = p.z[3 * s + 1], z2 = p.z[3 * s + 2];
      const uint32_t a_priv = smem_u32(sm.priv) + 2u * kPriv * lane, a_pairs = a_occ, a_kP = smem_u32(sm.kP);
      uint32_t i1b = 0;  // hits of layer 1 already filtered
      const int32_t* xq = x1p + lane + 32;  // this lane's hit of the next trip
      const int32_t* yq = y1p + lane + 32;
      while (i1b < n1) {
        // ---- C (a6): keep the middle hits whose fine cell is in J, up to KCAP per round
        uint32_t nk = 0;
        while (i1b < n1) {
          const uint32_t i1 = i1b + lane;
          int32_t xn = 0, yn = 0;
          if (i1 + 32 < n1) { xn = __ldg(xq); yn = __ldg(yq); }
          const int kx = __mulhi(xc, M1), ky = __mulhi(yc, M1);
          const uint32_t fx = (uint32_t)(kx >> fsh), ty = (uint32_t)(ky >> (fsh - 1));
          const uint32_t jw = lds_addr(a_J + (((ty << 2) & 0x1F8u) | ((fx >> 3) & 4u)));
          const bool keep = (i1 < n1) & ((jw >> (fx & 31u)) & 1u);
          const uint32_t km = __ballot_sync(FULL, keep);
          const uint32_t c = __popc(km);
          if (nk + c > (uint32_t)KCAP) break;  // the round is full: this trip opens the next one
          if (keep) {
            const uint32_t w = nk + __popc(km & lt);
            sm.kP[w] = __byte_perm((uint32_t)kx, (uint32_t)ky, 0x5410);
            sm.kI[w] = (uint16_t)i1;
          }
          nk += c;
          i1b += 32;
          xq += 32; yq += 32;
          xc = xn; yc = yn;
        }
        // the slots of this round: [survivor][layer] = count << 27 | e2 << 18 | e1 << 9 | e0  (hits COMPATIBLE with
        // the middle hit, element + 1)
        for (uint32_t i = lane; i < 2u * nk; i += 32) sm.slot[i] = 0;
        ST_DBG(0, 1); ST_DBG(1, nk);
        __syncwarp();
        const int64_t T01 = p.thr_in[s][0], T02 = p.thr_in[s][1], T12 = p.thr_in[s][2];
        const uint64_t T01x2 = p.thr2_in[s][0], T02x2 = p.thr2_in[s][1], T12x2 = p.thr2_in[s][2];
        // ---- D3: lane <-> pair (middle hit, element that passed the packed test): exact test, slot of the middle hit
        uint32_t np = 0;
        auto drain_pairs = [&](bool all) {
          while (np >= 32u || (all && np)) {
            const uint32_t take = min(np, 32u);
            np -= take;
            ST_DBG(2, 1); ST_DBG(3, take);
            __syncwarp();
            if (lane < take) {
              const uint32_t pr = lds_addr(a_pairs + 4u * (np + lane));
              const uint32_t k = pr & 0xFFu, el1 = pr >> 8;
              const bool side = el1 > (uint32_t)LCAP;                 // element of layer 2
              const uint32_t j1 = el1 - (side ? (uint32_t)LCAP : 0u);  // element in its layer (from the quad base) + 1
              const uint32_t gi = (side ? g2 : g0) + j1 - 1u;
              const uint32_t i1 = sm.kI[k] & 0x7FFFu;
              const int32_t x1 = __ldg(x1p + i1), y1 = __ldg(y1p + i1);
              const int32_t xe = __ldg(x + gi), ye = __ldg(y + gi);
              // |x_e*z1 - x1*z_e| <= T_e1
              const int32_t ze = side ? z2 : z0;
              const int64_t Te = side ? T12 : T01;
              const uint64_t Te2 = side ? T12x2 : T01x2;
              if (win_q(xe, z1, anchor_q(x1, -ze, Te), Te2) & win_q(ye, z1, anchor_q(y1, -ze, Te), Te2)) {
                // a pass holds at most kPriv pairs of one middle hit: with the check the count stays below 2^5
                const uint32_t a_sl = smem_u32(sm.slot) + 8u * k + (side ? 4u : 0u);
                if ((lds_addr(a_sl) >> 27) <= 3u) {
                  const uint32_t c = atoms_add_addr(a_sl, 1u << 27) >> 27;
                  if (c < 3u) atoms_add_addr(a_sl, j1 << (9u * c));
                }
              }
            }
          }
        };
        // ---- D1: lane <-> kept middle hit: the chains of the <= 2 x 2 coarse cells its window touches; elements that
        // pass the packed test go to the lane's private list, then all lists are packed into the pair list
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
            const uint32_t a_lo = a_head + (lox << (SM::TYB + 2)), a_hi = a_head + (hix << (SM::TYB + 2));
            hv[0] = lds_addr(a_lo + 4u * loy);
            if (hiy != loy) hv[1] = lds_addr(a_lo + 4u * hiy);
            if (hix != lox) {
              hv[2] = lds_addr(a_hi + 4u * loy);
              if (hiy != loy) hv[3] = lds_addr(a_hi + 4u * hiy);
            }
          }
          uint32_t c = 0;        // entries of the private list (kPriv hold; more: the middle hit takes the slow path)
          uint32_t a_pw = a_priv;
          auto test = [&](uint32_t el1) {  // element el1 - 1: packed test, private list; returns its chain link
            const uint32_t w = lds_addr(a_node + 4u * el1 - 4u);
            if (((A - w) & nmask) == 0) {
              if (c < kPriv) sts_u16_addr(a_pw, el1);
              a_pw += 2u;
              ++c;
            }
            return w & 0x3FFu;
          };
          uint32_t rem[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {  // the first two elements of every chain, straight-line
            rem[q] = 0;
            if (hv[q]) {
              const uint32_t l1 = test(hv[q]);
              if (l1) rem[q] = test(l1);
            }
          }
          while (__any_sync(FULL, (rem[0] | rem[1] | rem[2] | rem[3]) != 0)) {  // chains of three and more: rare
#pragma unroll
            for (int q = 0; q < 4; ++q)
              if (rem[q]) rem[q] = test(rem[q]);
          }
          if (c > kPriv) { sm.kI[k] |= 0x8000u; c = 0; }  // too many candidates: slow path in D4
          // pack the private lists: exclusive prefix of the counts
          uint32_t pre = c;
#pragma unroll
          for (int d = 1; d < 32; d <<= 1) {
            const uint32_t v = __shfl_up_sync(FULL, pre, d);
            if (lane >= (uint32_t)d) pre += v;
          }
          const uint32_t tot = __shfl_sync(FULL, pre, 31);
          pre -= c;
          const uint32_t mc = __reduce_max_sync(FULL, c);
          if (np + tot > 256u) drain_pairs(true);  // the pair list holds 256
          __syncwarp();
          for (uint32_t i = 0; i < mc; ++i)
            if (i < c) sts_addr(a_pairs + 4u * (np + pre + i), k | (lds_u16_addr(a_priv + 2u * i) << 8));
          np += tot;
          drain_pairs(false);
        }
        drain_pairs(true);
        __syncwarp();
        // ---- D4: middle hits with compatible hits in both layers -> exact (h0, h2) tests
        uint32_t nj = 0;  // their numbers, compacted into the pair list's memory
        for (uint32_t kb = 0; kb < nk; kb += 32) {
          const uint32_t k = kb + lane;
          bool both = false;
          if (k < nk) {
            const uint2 s02 = *reinterpret_cast<const uint2*>(&sm.slot[2 * k]);
            both = ((s02.x >> 27) != 0 && (s02.y >> 27) != 0) || (sm.kI[k] & 0x8000u);
          }
          const uint32_t m = __ballot_sync(FULL, both);
          if (both) sts_addr(a_pairs + 4u * (nj + __popc(m & lt)), k);
          nj += __popc(m);
        }
        ST_DBG(4, nj);
        __syncwarp();
        for (uint32_t jb = 0; jb < nj; jb += 32) {
          uint32_t t = 0, i1 = 0;
          bool slow = false;
          if (jb + lane < nj) {
            const uint32_t k = lds_addr(a_pairs + 4u * (jb + lane));
            const uint2 s02 = *reinterpret_cast<const uint2*>(&sm.slot[2 * k]);
            const uint32_t c0 = s02.x >> 27, c2 = s02.y >> 27;
            i1 = sm.kI[k];
            slow = c0 > 3u || c2 > 3u || (i1 & 0x8000u);
            i1 &= 0x7FFFu;
            if (!slow) {
              // |x2*z0 - x0*z2| <= T02 for the <= 3 x 3 pairs (h0, h2), both already compatible with h1
              int32_t x2[3] = {0, 0, 0}, y2[3] = {0, 0, 0};
#pragma unroll
              for (int b = 0; b < 3; ++b)
                if ((uint32_t)b < c2) {
                  const uint32_t j2 = ((s02.y >> (9 * b)) & 0x1FFu) - 1u;
                  x2[b] = __ldg(x + g2 + j2); y2[b] = __ldg(y + g2 + j2);
                }
              int32_t x0[3] = {0, 0, 0}, y0[3] = {0, 0, 0};
#pragma unroll
              for (int a = 0; a < 3; ++a)
                if ((uint32_t)a < c0) {
                  const uint32_t j0 = ((s02.x >> (9 * a)) & 0x1FFu) - 1u;
                  x0[a] = __ldg(x + g0 + j0); y0[a] = __ldg(y + g0 + j0);
                }
#pragma unroll
              for (int a = 0; a < 3; ++a)
                if ((uint32_t)a < c0) {
                  const int64_t Px = anchor_q(x0[a], -z2, T02), Py = anchor_q(y0[a], -z2, T02);
#pragma unroll
                  for (int b = 0; b < 3; ++b)
                    if ((uint32_t)b < c2) t += (win_q(x2[b], z0, Px, T02x2) & win_q(y2[b], z0, Py, T02x2)) ? 1u : 0u;
                }
            }
          }
          uint32_t sm_ = __ballot_sync(FULL, slow);
          ST_DBG(7, __popc(sm_));
          while (sm_) {  // rare: more than two compatible hits in a layer, or more than kPriv candidates
            const int src = __ffs((int)sm_) - 1;
            sm_ &= sm_ - 1;
            const uint32_t is = __shfl_sync(FULL, i1, src);
            const uint32_t ts = station_triplets_slow(StationGeo{x, y, b0, b1, b2, n0, n1, n2, z0, z1, z2, T01, T02, T12},
                                                      __ldg(x1p + is), __ldg(y1p + is));
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

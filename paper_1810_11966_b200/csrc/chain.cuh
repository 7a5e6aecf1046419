// chain.cuh -- chain_kernel: steps a4..a8 for the events of class H (the round-1 design, kept for the class it is
// still the fastest on; team.cuh holds the design used for classes M, G and list X).
//
// One team = one CTA of W warps works on one event at a time (persistent: events are fetched from the class list
// with an atomic cursor, two fetches ahead).  An L2 prefetch of the next event was measured and dropped: it re-read 17 %
// of the bytes from DRAM and did not shorten the kernel.
// CAP = fullest layer the class admits; NC = coarse cells per axis the shared-memory tables are sized for;
// LISTCAP = middle hits with triplets kept in shared memory per station (more spill to a global scratch).
//
// Per station:
//   stage   one 1-D TMA bulk copy per coordinate brings the station's three layers (contiguous in x[], y[])
//           into shared memory; it is issued as soon as the previous station's search is over.
//   A       every hit of layers 0 and 2 is pushed on the chain of its coarse slope cell (atomicExch on the
//           cell's head, `next` link per hit) and sets its bit in the layer's fine occupancy bitmap
//           (fine cell = half a coarse cell >= key_R).
//   B       J = dilate3x3(occ0) & dilate3x3(occ2), by row-wise shifts and ORs of 64-bit rows.
//   C       a middle hit h1 whose fine cell is not in J cannot have both a compatible h0 and a compatible h2
//           (DESIGN.md section 6.4); the others are compacted (ballot/popc) into a list.
//   D       one lane per surviving h1: walks the chains of the <= 2x2 coarse cells around it in layer 0
//           (exact test), then in layer 2 (exact tests against h1 and against the recorded h0), and appends
//           (x1, y1, number of triplets with this middle hit) to the station's list  (R8).
//   F       chain counts against the previous station's list (a7), result write (a8).
#pragma once
#include <stddef.h>

#include "team.cuh"

namespace cbm {

template <int OFS = 0>
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
  uint32_t v;
  asm volatile("{ .reg .u16 t; ld.shared.u16 t, [%1+%2]; cvt.u32.u16 %0, t; }" : "=r"(v) : "r"(addr), "n"(OFS));
  return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v) {
  asm volatile("{ .reg .u16 t; cvt.u16.u32 t, %1; st.shared.u16 [%0], t; }" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t atoms_exch(uint32_t addr, uint32_t v) {
  uint32_t old;
  asm volatile("atom.shared.exch.b32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(v) : "memory");
  return old;
}
__device__ __forceinline__ void reds_or_a(uint32_t addr, uint32_t v) {
  asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// per-station constants: filled into shared memory once per CTA, read back with 128-bit loads once per station and warp
struct alignas(16) ChainStationConst {
  int32_t z0, z1, z2, nz0, nz2;  // nz = -z
  int32_t M0, M1, M2;
  int64_t T01, T02, T12;
  uint64_t T01x2, T02x2, T12x2;
};

template <int W, int CAP, int NC, int LISTCAP>
struct ChainSmem {
  alignas(16) int32_t sx[3 * CAP + 8];        // the station as it lies in x[] (from the 16-byte boundary below its
  alignas(16) int32_t sy[3 * CAP + 8];        // first hit): layer 0, layer 1, layer 2
  alignas(16) uint32_t head[2 * NC * NC];     // chain heads (hit index in its layer + 1; 0 = empty) of layers 0 and 2
  uint32_t occ[2][128];                       // fine occupancy bitmaps of layers 0 and 2: row fx = 2 words, bit fy
  uint32_t J[128];                            // dilate(occ[0]) & dilate(occ[1])
  uint16_t next[2][CAP];                      // chain links (index + 1; 0 = end)
  uint16_t surv[CAP + 32 * W];                // middle hits that passed the bitmap filter, one part per warp
  uint32_t wcnt[W];                           // survivors in each part
  int32_t ux[2][LISTCAP], uy[2][LISTCAP];     // middle hits with triplets of the previous / current station
  uint32_t uc[2][LISTCAP];                    // their multiplicities, then saturated chain counts c_s[u]
  alignas(16) ChainStationConst sc[kMaxStations];
  uint32_t off[kMaxLayers + 1];
  unsigned long long acc[2];                  // triplets of the station (parity-buffered with the two below)
  uint32_t ucount[2];
  uint32_t alive[2];                          // some chain count of the station is not zero (parity-buffered)
  uint32_t li[3];                             // ring of fetched work indices
  alignas(8) uint64_t bar;                    // completion of the station's bulk copies
};

// fine cell of a slope key on the cyclic grid: floor(key / 2^sh) mod nf (nf a power of two, mask = nf - 1).
// Keys outside the covered range alias onto other cells; that only adds candidates, never loses one.
__device__ __forceinline__ uint32_t chain_cell_of(int key, int sh, uint32_t mask) { return (uint32_t)(key >> sh) & mask; }





// Chain heads (index + 1 <= 4096, 16 bits each) of the <= 2x2 coarse cells that can hold a hit compatible with
// a hit whose window covers rows lox..hix and columns loy..hiy (cyclic); non-empty heads only, packed from bit 0.
__device__ __forceinline__ unsigned long long chain_load_heads(const uint32_t* head, uint32_t lox, uint32_t hix, uint32_t loy,
                                                         uint32_t hiy, uint32_t nc) {
  unsigned long long hq = 0;
  const bool dx = hix != lox, dy = hiy != loy;
  uint32_t v = head[lox * nc + loy];
  if (v) hq = v;
  if (dy) { v = head[lox * nc + hiy]; if (v) hq = (hq << 16) | v; }
  if (dx) { v = head[hix * nc + loy]; if (v) hq = (hq << 16) | v; }
  if (dx && dy) { v = head[hix * nc + hiy]; if (v) hq = (hq << 16) | v; }
  return hq;
}

// Rare path of phase D (a middle hit with more than three compatible h0): number of h0 in the <= 2x2 cells
// compatible with both h1 (anchors Qx, Qy) and h2 (x2, y2).  No warp-level operation inside.
template <class SM>
__device__ __noinline__ uint32_t chain_count_h0_slow(const SM& sm, const uint32_t* head, uint32_t o0, uint32_t lox, uint32_t hix,
                                               uint32_t loy, uint32_t hiy, uint32_t nc, const ChainStationConst& c, int64_t Qx,
                                               int64_t Qy, int32_t x2, int32_t y2) {
  uint32_t n = 0;
  for (int q = 0; q < 4; ++q) {
    if ((q & 1) && hiy == loy) continue;
    if ((q & 2) && hix == lox) continue;
    for (uint32_t cur = head[((q & 2) ? hix : lox) * nc + ((q & 1) ? hiy : loy)]; cur; cur = sm.next[0][cur - 1]) {
      const int32_t x0 = sm.sx[o0 + cur - 1], y0 = sm.sy[o0 + cur - 1];
      const bool ok = win_q(x0, c.z1, Qx, c.T01x2) & win_q(y0, c.z1, Qy, c.T01x2) &
                      win_q(x2, c.z0, anchor_q(x0, c.nz2, c.T02), c.T02x2) &
                      win_q(y2, c.z0, anchor_q(y0, c.nz2, c.T02), c.T02x2);
      n += ok ? 1u : 0u;
    }
  }
  return n;
}

template <int W, int CAP, int NC, int LISTCAP, int CLS, int MINB, bool STATIC_SMEM, int FSH_ADD = 0>
__global__ void __launch_bounds__(32 * W, MINB)
    chain_kernel(const __grid_constant__ Params p, const int32_t* __restrict__ x, const int32_t* __restrict__ y,
                const uint32_t* __restrict__ off, uint32_t* __restrict__ n_triplets, uint32_t* __restrict__ n_candidates,
                uint8_t* __restrict__ accept, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ list,
                uint32_t* __restrict__ spill) {
  using SM = ChainSmem<W, CAP, NC, LISTCAP>;
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  __shared__ __align__(16) unsigned char smem_static[STATIC_SMEM ? sizeof(SM) : 16];
  SM& sm = *reinterpret_cast<SM*>(STATIC_SMEM ? smem_static : smem_dyn);
  constexpr uint32_t T = 32 * W;
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  constexpr uint32_t kZeroVec = (2 * NC * NC + 256) / 4;  // head[] and occ[][] are contiguous
  static_assert((2 * NC * NC) % 4 == 0 && offsetof(SM, occ) == offsetof(SM, head) + 2 * NC * NC * 4, "layout");
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t S = p.S, L = p.L;
  const uint32_t n_list = ctrl->count[CLS];
  const int R = p.key_R, fsh = p.cell_sh + FSH_ADD, csh = fsh + 1;  // FSH_ADD: wider cells for sparse classes
  const uint32_t nf = 2 * NC, nf1 = nf - 1u;  // fine cells per axis
  const uint32_t nc = max(nf >> 1, 1u), nc1 = nc - 1u;
  uint32_t* const head0 = sm.head;
  uint32_t* const head2 = sm.head + nc * nc;
  const uint32_t lnc = 31u - (uint32_t)__clz(nc);  // nc = 2^lnc: coarse cell (cx, cy) is head[(cx << lnc) | cy]
  constexpr int kDY = (int)(offsetof(SM, sy) - offsetof(SM, sx));
  const uint32_t a_sx = smem_u32(sm.sx);
  // spill area of this CTA: list entries beyond LISTCAP, [2 lists][x, y, c][CAP] words
  uint32_t* const spill_cta = spill + (size_t)blockIdx.x * 6 * CAP;
  int32_t* const spill_i = reinterpret_cast<int32_t*>(spill_cta);

  {
    uint4* const v = reinterpret_cast<uint4*>(sm.head);
    for (uint32_t i = tid; i < kZeroVec; i += T) v[i] = make_uint4(0, 0, 0, 0);
  }
  if (tid < S) {
    const uint32_t t = tid;
    ChainStationConst c;
    c.z0 = p.z[3 * t]; c.z1 = p.z[3 * t + 1]; c.z2 = p.z[3 * t + 2];
    c.nz0 = -c.z0; c.nz2 = -c.z2;
    c.M0 = p.key_mul[3 * t]; c.M1 = p.key_mul[3 * t + 1]; c.M2 = p.key_mul[3 * t + 2];
    c.T01 = p.thr_in[t][0]; c.T02 = p.thr_in[t][1]; c.T12 = p.thr_in[t][2];
    c.T01x2 = p.thr2_in[t][0]; c.T02x2 = p.thr2_in[t][1]; c.T12x2 = p.thr2_in[t][2];
    sm.sc[t] = c;
  }
  if (tid == 0) {
    sm.li[0] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.li[1] = atomicAdd(&ctrl->work[CLS], 1u);
    sm.acc[0] = sm.acc[1] = 0;
    sm.ucount[0] = sm.ucount[1] = 0;
    sm.alive[0] = sm.alive[1] = 0;
    mbar_init(&sm.bar, 1);
    fence_mbar_init();
  }
  team_sync<W>();
  uint32_t par = 0;  // phase parity of the staging barrier
  uint32_t sp = 0;   // parity of the per-station counters
  // Warp w of every resident CTA sits on scheduler w % 4, and phases B..D give the low warps more work
  // (row 0..63, the first 32-chunks): the roles rotate from station to station so that the schedulers even out.
  uint32_t rot = 0;

  // a4: thread 0 starts the bulk copies of station s of the event whose offsets are in sm.off
  auto searchable = [&](uint32_t s) {
    return (sm.off[3 * s] != sm.off[3 * s + 1]) & (sm.off[3 * s + 1] != sm.off[3 * s + 2]) & (sm.off[3 * s + 2] != sm.off[3 * s + 3]);
  };
  auto issue_stage = [&](uint32_t s) {
    const uint32_t a = sm.off[3 * s] & ~3u;
    const uint32_t bytes = (((sm.off[3 * s + 3] + 3u) & ~3u) - a) * 4u;  // <= (3*CAP + 6) * 4
    mbar_arrive_expect_tx(&sm.bar, 2u * bytes);
    bulk_g2s(sm.sx, x + a, bytes, &sm.bar);
    bulk_g2s(sm.sy, y + a, bytes, &sm.bar);
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
    bool dead = false;  // some station so far has no triplet => no chain; triplet counts are still needed
    int cur = 0;
    for (uint32_t s = 0; s < S; ++s) {
      const uint32_t b0 = sm.off[3 * s], b1 = sm.off[3 * s + 1], b2 = sm.off[3 * s + 2], b3 = sm.off[3 * s + 3];
      const uint32_t n0 = b1 - b0, n1 = b2 - b1, n2 = b3 - b2;
      const uint32_t o0 = b0 & 3u, o1 = o0 + n0, o2 = o1 + n1;  // layer starts in sm.sx / sm.sy
      const ChainStationConst c = sm.sc[s];
      const bool search = (n0 != 0) & (n1 != 0) & (n2 != 0);
      const uint32_t vwarp = (warp + rot) & (W - 1), vtid = vwarp * 32 + lane;
      rot = (rot + 1u) & (W - 1);
      if (search) {
        while (!mbar_try_wait(&sm.bar, par)) {
        }
        par ^= 1u;
        // ---- A: chains of layers 0 and 2 on the coarse grid, fine occupancy bitmaps.  The first half of the
        // team's warps takes layer 0, the second half layer 2 (one warp: both in turn).
        {
          constexpr uint32_t TH = W > 1 ? T / 2 : T;
#pragma unroll 1
          for (int pass = 0; pass < (W > 1 ? 1 : 2); ++pass) {
            const int l = W > 1 ? (int)(tid >= TH) : pass;  // 0: layer 0, 1: layer 2  (warp-uniform)
            const int32_t M = l ? c.M2 : c.M0;
            const uint32_t j0 = W > 1 ? tid - (l ? TH : 0u) : tid, n = l ? n2 : n0;
            uint32_t a_hit = a_sx + 4u * ((l ? o2 : o0) + j0);               // x of hit j; y at + kDY
            uint32_t a_nx = smem_u32(sm.next[l]) + 2u * j0;
            const uint32_t a_hd = smem_u32(l ? head2 : head0), a_oc = smem_u32(sm.occ[l]);
            for (uint32_t j = j0; j < n; j += TH, a_hit += 4u * TH, a_nx += 2u * TH) {
              const uint32_t fx = chain_cell_of(__mulhi(lds_s32(a_hit), M), fsh, nf1);
              const uint32_t fy = chain_cell_of(__mulhi(lds_s32<kDY>(a_hit), M), fsh, nf1);
              const uint32_t old = atoms_exch(a_hd + 4u * (((fx >> 1) << lnc) | (fy >> 1)), j + 1u);
              sts_u16(a_nx, old);
              reds_or_a(a_oc + 4u * ((fx << 1) | (fy >> 5)), 1u << (fy & 31));
            }
          }
        }
        team_sync<W>();
        // ---- B: J = dilate(occ0) & dilate(occ2) on the cyclic grid; a compatible pair lies in fine cells at
        // most one apart in x and in y
        for (uint32_t r = vtid; r < nf; r += T) {
          const unsigned long long full = nf == 64 ? ~0ull : ((1ull << nf) - 1ull);
          unsigned long long d[2];
#pragma unroll
          for (int l = 0; l < 2; ++l) {
            const unsigned long long* rows = reinterpret_cast<const unsigned long long*>(sm.occ[l]);
            const unsigned long long v = rows[r] | rows[(r - 1u) & nf1] | rows[(r + 1u) & nf1];
            d[l] = (v | (v << 1) | (v >> nf1) | (v >> 1) | (v << nf1)) & full;
          }
          const unsigned long long j = d[0] & d[1];
          sm.J[2 * r] = (uint32_t)j;
          sm.J[2 * r + 1] = (uint32_t)(j >> 32);
        }
        team_sync<W>();
        // ---- C (a6): middle hits whose fine cell is in J, compacted with ballot/popc
        const uint32_t a_J = smem_u32(sm.J);
        constexpr uint32_t kWReg = CAP / W + 32;                  // survivors a warp can meet
        const uint32_t a_ws = smem_u32(sm.surv) + 2u * warp * kWReg;  // this warp's part of the list (no atomics)
        uint32_t nws = 0;
        for (uint32_t base = vwarp * 32; base < n1; base += T) {
          const uint32_t i1 = base + lane;
          bool keep = false;
          if (i1 < n1) {
            const uint32_t a1 = a_sx + 4u * (o1 + i1);
            const uint32_t fx = chain_cell_of(__mulhi(lds_s32(a1), c.M1), fsh, nf1);
            const uint32_t fy = chain_cell_of(__mulhi(lds_s32<kDY>(a1), c.M1), fsh, nf1);
            keep = (lds_u32(a_J + 4u * ((fx << 1) | (fy >> 5))) >> (fy & 31)) & 1u;
          }
          const uint32_t km = __ballot_sync(FULL, keep);
          if (keep) sts_u16(a_ws + 2u * (nws + __popc(km & lanemask_lt())), i1);
          nws += __popc(km);
        }
        if (lane == 0) sm.wcnt[warp] = nws;
        team_sync<W>();
        // ---- D (a5): one lane per surviving middle hit
        // the team's survivors, numbered through the warps' parts: number k lies in part w at k - first[w]
        uint32_t nsv = 0, wfirst[W];
#pragma unroll
        for (int w = 0; w < W; ++w) { wfirst[w] = nsv; nsv += sm.wcnt[w]; }
        unsigned long long trip = 0;
        // hit with chain link cu (= index + 1) of layer 0 / 2: x at a_l + 4*cu, y kDY further; its link at a_n + 2*cu
        const uint32_t a_l0 = a_sx + 4u * o0 - 4u, a_l2 = a_sx + 4u * o2 - 4u;
        const uint32_t a_n0 = smem_u32(sm.next[0]) - 2u, a_n2 = smem_u32(sm.next[1]) - 2u;
        for (uint32_t cb = vwarp * 32; cb < nsv; cb += T) {
          const bool act = cb + lane < nsv;
          int32_t x1 = 0, y1 = 0;
          uint32_t lox = 0, hix = 0, loy = 0, hiy = 0;
          unsigned long long hq = 0;  // chain heads still to walk (16 bits each)
          if (act) {
            const uint32_t k = cb + lane;
            uint32_t ks = k;  // index in sm.surv
#pragma unroll
            for (int w = 1; w < W; ++w) if (k >= wfirst[w]) ks = k - wfirst[w] + w * kWReg;
            const uint32_t a1 = a_sx + 4u * (o1 + sm.surv[ks]);
            x1 = lds_s32(a1);
            y1 = lds_s32<kDY>(a1);
            const int kx = __mulhi(x1, c.M1), ky = __mulhi(y1, c.M1);
            lox = chain_cell_of(kx - R, csh, nc1); hix = chain_cell_of(kx + R, csh, nc1);
            loy = chain_cell_of(ky - R, csh, nc1); hiy = chain_cell_of(ky + R, csh, nc1);
            hq = chain_load_heads(head0, lox, hix, loy, hiy, nc);
          }
          // h0 compatible with h1:  |x0*z1 - x1*z0| <= T01  <=>  (uint64)(x0*z1 + (T01 - x1*z0)) <= 2*T01
          const int64_t Qx = anchor_q(x1, c.nz0, c.T01), Qy = anchor_q(y1, c.nz0, c.T01);
          uint32_t np = 0, pk = 0;  // number of compatible h0; the first two (index + 1, 16 bits each)
          uint32_t cu = (uint32_t)hq & 0xFFFFu;
          hq >>= 16;
          while (__any_sync(FULL, cu != 0)) {
            if (cu) {
              const int32_t x0 = lds_s32(a_l0 + 4u * cu), y0 = lds_s32<kDY>(a_l0 + 4u * cu);
              const uint32_t nx = lds_u16(a_n0 + 2u * cu);
              if (win_q(x0, c.z1, Qx, c.T01x2) & win_q(y0, c.z1, Qy, c.T01x2)) {
                if (np < 2) pk |= cu << (np << 4);
                ++np;
              }
              cu = nx;
              if (!cu) { cu = (uint32_t)hq & 0xFFFFu; hq >>= 16; }
            }
          }
          uint32_t t = 0;  // triplets with this middle hit
          if (__any_sync(FULL, np != 0)) {
            hq = np ? chain_load_heads(head2, lox, hix, loy, hiy, nc) : 0ull;
            // h2 compatible with h1:  |x2*z1 - x1*z2| <= T12;  with h0:  |x2*z0 - x0*z2| <= T02
            const int64_t Rx = anchor_q(x1, c.nz2, c.T12), Ry = anchor_q(y1, c.nz2, c.T12);
            cu = (uint32_t)hq & 0xFFFFu;
            hq >>= 16;
            while (__any_sync(FULL, cu != 0)) {
              if (cu) {
                const int32_t x2 = lds_s32(a_l2 + 4u * cu), y2 = lds_s32<kDY>(a_l2 + 4u * cu);
                const uint32_t nx = lds_u16(a_n2 + 2u * cu);
                if (win_q(x2, c.z1, Rx, c.T12x2) & win_q(y2, c.z1, Ry, c.T12x2)) {
                  if (np <= 2) {
                    uint32_t q = pk;
                    do {
                      const int32_t x0 = lds_s32(a_l0 + 4u * (q & 0xFFFFu)), y0 = lds_s32<kDY>(a_l0 + 4u * (q & 0xFFFFu));
                      const bool ok = win_q(x2, c.z0, anchor_q(x0, c.nz2, c.T02), c.T02x2) &
                                      win_q(y2, c.z0, anchor_q(y0, c.nz2, c.T02), c.T02x2);
                      t += ok ? 1u : 0u;
                      q >>= 16;
                    } while (q);
                  } else {
                    t += chain_count_h0_slow(sm, head0, o0, lox, hix, loy, hiy, nc, sm.sc[s], Qx, Qy, x2, y2);
                  }
                }
                cu = nx;
                if (!cu) { cu = (uint32_t)hq & 0xFFFFu; hq >>= 16; }
              }
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
              } else {
                const uint32_t o = pos - LISTCAP;
                spill_i[(cur * 3 + 0) * CAP + o] = x1; spill_i[(cur * 3 + 1) * CAP + o] = y1;
                spill_cta[(cur * 3 + 2) * CAP + o] = t;
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
      team_sync<W>();

      // ---- F: the search is over: the staging buffer, the chains and the bitmaps are free
      const uint32_t ncur = dead ? 0u : sm.ucount[sp];
      if (tid == 0) {
        n_triplets[(size_t)e * S + s] = sat32(sm.acc[sp]);
        sm.acc[sp ^ 1u] = 0;
        sm.ucount[sp ^ 1u] = 0;
        sm.alive[sp ^ 1u] = 0;
        if (s + 1 < S && searchable(s + 1)) issue_stage(s + 1);
      }
      if (search) {
        uint4* const v = reinterpret_cast<uint4*>(sm.head);
#pragma unroll
        for (uint32_t k = 0; k < (kZeroVec + T - 1) / T; ++k)  // straight-line: kZeroVec / T stores per thread
          if ((k + 1) * T <= kZeroVec || tid + k * T < kZeroVec) v[tid + k * T] = make_uint4(0, 0, 0, 0);
      }
      // ---- a7: chain counts c_s[u] = m_u * sum over linked t of c_{s-1}[t], saturating (R9)
      if (s > 0 && ncur) {
        const int32_t nzA = -p.z[3 * (s - 1) + 1], zB = c.z1;
        const int64_t TL = p.thr_link[s];
        const uint64_t TLx2 = p.thr2_link[s];
        if (ncur <= (uint32_t)LISTCAP && nprev <= (uint32_t)LISTCAP) {  // everything in shared memory
          // kLinkG lanes share one u: lane g tests the previous station's entries g, g + kLinkG, ...
          constexpr uint32_t kLinkG = 8;
          const uint32_t g = tid % kLinkG;
          for (uint32_t ub = 0; ub < ncur; ub += T / kLinkG) {
            const uint32_t u = ub + tid / kLinkG;
            unsigned long long a = 0;
            if (u < ncur) {
              // |x_t*zB - x_u*zA| <= TL
              const int64_t Qx = anchor_q(sm.ux[cur][u], nzA, TL), Qy = anchor_q(sm.uy[cur][u], nzA, TL);
              for (uint32_t t = g; t < nprev; t += kLinkG) {
                const bool ok = win_q(sm.ux[cur ^ 1][t], zB, Qx, TLx2) & win_q(sm.uy[cur ^ 1][t], zB, Qy, TLx2);
                if (ok) a += sm.uc[cur ^ 1][t];  // < 4096 * 2^32
              }
            }
#pragma unroll
            for (int d = kLinkG / 2; d >= 1; d >>= 1) a += __shfl_xor_sync(FULL, a, d);
            if (u < ncur && g == 0) {
              const uint32_t v = sat32((unsigned long long)sat32(a) * sm.uc[cur][u]);  // m_u <= 2^24
              sm.uc[cur][u] = v;
              if (v) sm.alive[sp] = 1;
            }
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
            if (v) sm.alive[sp] = 1;
          }
        }
      }
      if (ncur == 0) dead = true;
      nprev = ncur;
      cur ^= 1;
      sp ^= 1u;
      team_sync<W>();
      // every chain ends here (all c_s[u] are zero): no candidate, whatever the later stations hold; they are still
      // searched for their triplet counts, but build no lists and link nothing
      if (s > 0 && !dead && sm.alive[sp ^ 1u] == 0) dead = true;
    }

    // ---- candidates = sum over the last station's middle hits; a8: one writer per event
    if (warp == 0) {
      unsigned long long part = 0;
      if (!dead)
        for (uint32_t u = lane; u < nprev; u += 32)
          part += u < (uint32_t)LISTCAP ? sm.uc[cur ^ 1][u] : spill_cta[((cur ^ 1) * 3 + 2) * CAP + u - LISTCAP];
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(FULL, part, d);
      if (lane == 0) {
        const uint32_t cand = sat32(part);
        n_candidates[e] = cand;
        accept[e] = cand >= p.min_candidates ? 1 : 0;
      }
    }
  }
}

}  // namespace cbm

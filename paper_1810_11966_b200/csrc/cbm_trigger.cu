// cbm_trigger.cu -- host side of libcbmtrigger.so: the C ABI of include/cbm_trigger.h.
//
// Owns the slots (pinned host staging, device arrays, result buffers), the three streams of the
// H2D | kernels | D2H software pipeline ("it can be hidden by performing computation and
// transfer in parallel") and the launch sequence of the kernels (classify, tile, team, chain .cuh).  No CPU fallback exists:
// without a CUDA device cbm_trigger_create fails with CBM_ERR_CUDA.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <thread>
#include <vector>

#include "../../include/cbm_trigger.h"
#include "classify.cuh"
#include "tile.cuh"
#include "team.cuh"
#include "chain.cuh"
#include "select.cuh"
#include "wire.cuh"
#include "msd.cuh"
#include "ubench.cuh"
#include "filter.cuh"
#include "timeslice.cuh"

namespace {

using namespace cbm;

// team classes (team.cuh): warps per team, fullest layer admitted, kept middle hits, coarse table (log2
// columns, log2 rows), middle hits with triplets per station
using SmemM = TeamSmem<1, 128, 64, 4, 4, 32>;
using SmemG = TeamSmem<16, 4096, 4104, 5, 5, 256>;
constexpr int kCapM = SmemM::CAP, kCapG = SmemG::CAP;
constexpr int kMinBM = 24, kMinBG = 2;
#define TEAM_KERNEL_M team_kernel<SmemM, kClsM, kMinBM, false, true>
// class H, round-1 design (chain.cuh): 4 warps, 448 hits per layer, 32 x 32 coarse cells, 64 list entries, 8 CTAs/SM
constexpr int kWarpsH = 4, kCapH = 448;
using SmemHC = ChainSmem<kWarpsH, kCapH, 32, 64>;
#define CHAIN_KERNEL_H chain_kernel<kWarpsH, kCapH, 32, 64, kClsH, 8, true>
#define TEAM_KERNEL_G team_kernel<SmemG, kClsG, kMinBG, true, false>
#define TEAM_KERNEL_X team_kernel<SmemG, kClsX, kMinBG, true, false>
// kernels of one run, in the order of cbm_trigger_stats_t::kernel_ms
enum { kKClassify = 0, kKTile = 1, kKTeamM = 2, kKTeamH = 3, kKTeamG = 4, kKTeamX = 5 };
static_assert(CBM_TRIGGER_N_KERNELS == 6, "kernel_ms layout");

enum SlotState { kEmpty = 0, kUploaded = 1, kRunning = 2 };

struct Scratch {
  Ctrl* d_ctrl = nullptr;
  uint32_t* d_list[kNumLists] = {nullptr, nullptr, nullptr, nullptr};  // M, H, G, X
  uint32_t* d_spill[3] = {nullptr, nullptr, nullptr};  // class G, list X, class H (chain kernel); per CTA: middle-hit
                                                       // lists beyond shared memory
  uint32_t* d_selcnt = nullptr;  // accepted events per block of kSelEvents events (select.cuh)
  unsigned long long* d_gsum = nullptr;  // hits per block of kGatherEvents list entries of the gather (select.cuh)
  uint32_t* d_hitbase = nullptr; // first hit of every selected event in the gathered batch (select.cuh)
  uint32_t* d_fcnt = nullptr;    // hits per (event, layer) of the input filter (filter.cuh), then per-block sums behind
};

struct ProfEvents {
  cudaEvent_t k[2 * CBM_TRIGGER_N_KERNELS] = {};  // start, end of every kernel
  cudaEvent_t h2d[2] = {}, d2h[2] = {};
  bool valid = false;
};

struct Slot {
  int32_t *h_x = nullptr, *h_y = nullptr;
  uint8_t* h_p = nullptr;   // CBM_FLAG_PACKED_INPUT: pinned staging of the XY20 stream (instead of h_x, h_y)
  uint32_t* d_p = nullptr;  // ... and its device copy, expanded into d_x, d_y by `run`
  bool packed_pending = false;
  uint32_t* h_off = nullptr;
  int32_t *d_x = nullptr, *d_y = nullptr;
  uint32_t* d_off = nullptr;
  uint32_t *d_nt = nullptr, *d_nc = nullptr;
  uint8_t* d_ac = nullptr;
  uint32_t *d_sel = nullptr, *d_nsel = nullptr;  // ascending ids of the accepted events, their number
  uint32_t* h_nsel = nullptr;
  bool sel_valid = false;
  uint32_t *h_nt = nullptr, *h_nc = nullptr;
  uint8_t* h_ac = nullptr;
  Ctrl* h_ctrl = nullptr;
  Scratch scr;
  ProfEvents prof;
  cudaEvent_t ev_h2d = nullptr, ev_run = nullptr, ev_d2h = nullptr;
  int state = kEmpty;
  uint32_t n_events = 0;
  uint64_t n_hits = 0;
  cbm_trigger_stats_t stats = {};
};

}  // namespace

struct cbm_trigger {
  cbm_trigger_config_t cfg;
  Params p;
  int n_sm = 0;
  int grid[kNumLists] = {0, 0, 0, 0};
  int grid_hc = 0;          // chain_kernel (class H)
  Slot slot[CBM_TRIGGER_MAX_SLOTS];
  Scratch dev_scr;          // scratch of cbm_trigger_run_device
  Ctrl* h_dev_ctrl = nullptr;
  ProfEvents dev_prof[CBM_TRIGGER_PROFILE_RING];  // CBM_FLAG_PROFILE: event sets of the last run_device calls
  uint32_t dev_prof_head = 0;                       // number of run_device calls so far
  uint32_t dev_n_events = 0;
  uint64_t dev_n_hits = 0;
  cudaStream_t st_h2d = nullptr, st_run = nullptr, st_d2h = nullptr;
  cudaStream_t st_side[3] = {nullptr, nullptr, nullptr};  // tile, M and G run beside class H (after classify)
  cudaEvent_t ev_fork = nullptr, ev_join[3] = {nullptr, nullptr, nullptr};
  std::string err;
};

namespace {

thread_local std::string g_create_err;

// Staging copy of caller memory into a slot's pinned buffer: large copies are split over a few host threads (one
// thread moves about 13 GB/s, well below the H2D link it feeds).
void staging_copy(void* dst, const void* src, size_t bytes) {
  constexpr size_t kMinPerThread = 32u << 20;
  size_t n_thr = std::min<size_t>(8, bytes / kMinPerThread);
  const unsigned hw = std::thread::hardware_concurrency();
  if (hw) n_thr = std::min<size_t>(n_thr, hw);
  if (n_thr < 2) { memcpy(dst, src, bytes); return; }
  std::vector<std::thread> th;
  const size_t per = ((bytes / n_thr) + 4095) & ~(size_t)4095;
  for (size_t i = 0; i < n_thr; ++i) {
    const size_t a = i * per, b = std::min(bytes, a + per);
    if (a >= b) break;
    th.emplace_back([=] { memcpy((char*)dst + a, (const char*)src + a, b - a); });
  }
  for (auto& x : th) x.join();
}

int fail(cbm_trigger* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  if (h) h->err = buf; else g_create_err = buf;
  return code;
}

#define CBM_CUDA(h, expr)                                                                       \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess) return fail(h, CBM_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

// ---------------------------------------------------------------------------------------------- parameters
int build_params(const cbm_trigger_config_t& c, Params& p, std::string& why) {
  memset(&p, 0, sizeof(p));
  if (c.n_stations < 1 || c.n_stations > CBM_TRIGGER_MAX_STATIONS) { why = "n_stations must be 1..8"; return CBM_ERR_INVALID_ARG; }
  p.S = c.n_stations;
  p.L = 3 * c.n_stations;
  for (uint32_t l = 0; l < p.L; ++l) {
    const int32_t z = c.layer_z[l];
    if (z <= 0 || z > (1 << 23)) { why = "layer_z must be in (0, 2^23]"; return CBM_ERR_INVALID_ARG; }
    if (l && z <= c.layer_z[l - 1]) { why = "layer_z must be strictly increasing"; return CBM_ERR_INVALID_ARG; }
    p.z[l] = z;
  }
  if (c.win_in_den == 0 || c.win_in_den > 4096 || c.win_in_num > c.win_in_den ||
      c.win_link_den == 0 || c.win_link_den > 4096 || c.win_link_num > c.win_link_den) {
    why = "windows need 0 < den <= 4096 and num <= den";
    return CBM_ERR_INVALID_ARG;
  }
  if (c.max_hits_per_layer < 1 || c.max_hits_per_layer > CBM_TRIGGER_MAX_HITS_PER_LAYER) {
    why = "max_hits_per_layer must be 1..4096";
    return CBM_ERR_INVALID_ARG;
  }
  if (c.n_slots > CBM_TRIGGER_MAX_SLOTS) { why = "n_slots must be 0..4"; return CBM_ERR_INVALID_ARG; }
  if (c.max_events == 0) { why = "max_events must be > 0"; return CBM_ERR_INVALID_ARG; }
  if (c.max_hits >= (1ull << 32)) { why = "max_hits must be < 2^32"; return CBM_ERR_INVALID_ARG; }
  // the block-wise scans index in uint32 with blocks of 4096 elements: element counts stay 8192 below 2^32 so that
  // neither a block count nor the last block's element indices wrap (CBM_TRIGGER_MAX_INDEX)
  if ((uint64_t)c.max_events * p.L + 1 > CBM_TRIGGER_MAX_INDEX) { why = "max_events * layers must be < 2^32 - 8192"; return CBM_ERR_INVALID_ARG; }
  if (c.tiny_max_layer_hits > kTinyMaxLayerLimit) { why = "tiny_max_layer_hits must be <= 32"; return CBM_ERR_INVALID_ARG; }
  if (c.device < 0) { why = "device must be >= 0"; return CBM_ERR_INVALID_ARG; }

  // R4: per-layer-pair integer thresholds T_AB = floor(a*z_A*z_B / b); a*z_A*z_B <= 2^12 * 2^46
  for (uint32_t s = 0; s < p.S; ++s) {
    const int64_t z0 = p.z[3 * s], z1 = p.z[3 * s + 1], z2 = p.z[3 * s + 2];
    const int64_t a = c.win_in_num, b = c.win_in_den;
    p.thr_in[s][0] = a * z0 * z1 / b;
    p.thr_in[s][1] = a * z0 * z2 / b;
    p.thr_in[s][2] = a * z1 * z2 / b;
    if (s) {
      const int64_t zA = p.z[3 * (s - 1) + 1];
      p.thr_link[s] = (int64_t)c.win_link_num * zA * z1 / (int64_t)c.win_link_den;
      p.thr2_link[s] = 2 * (uint64_t)p.thr_link[s];
    }
    for (int k = 0; k < 3; ++k) p.thr2_in[s][k] = 2 * (uint64_t)p.thr_in[s][k];
  }
  p.min_candidates = c.min_candidates;
  p.max_hits_per_layer = c.max_hits_per_layer;
  const bool tiny_on = !(c.flags & CBM_FLAG_NO_TINY_PATH);
  p.tiny_max_layer = c.tiny_max_layer_hits ? c.tiny_max_layer_hits : 24;
  p.tiny_max_total = tiny_on ? kTinyMaxTotal : 0;
  p.cls_max[kClsM] = kCapM; p.cls_max[kClsH] = kCapH; p.cls_max[kClsG] = kCapG;

  // Slope keys: key = floor(x*M_l/2^32), M_l = round(2^32*K/z_l) < 2^31.
  // For any int32 x: |x*M_l/2^32 - K*x/z_l| <= 2^31 * 0.5/2^32 = 0.25, floor loses < 1  =>  |key - K*x/z_l| < 1.25.
  // Two hits with |x_h/z_A - x_g/z_B| <= w therefore have |key_h - key_g| < w*K + 2.5 <= R := ceil(w*K) + 3.
  // K is the largest scale with R <= 254 (and K < z_min/2): then the packed 16-bit test below is as sharp as the
  // window itself.  Filter cell = floor(key / 2^cell_sh) mod 64 with 2^cell_sh >= R: hits that are pairwise
  // compatible span at most two adjacent cells per axis (cyclic grid: no slope range has to be covered).
  const double w = (double)c.win_in_num / (double)c.win_in_den;
  const double Kmax = 0.499 * (double)p.z[0];
  const double K = w > 0 ? std::min(Kmax, (254.0 - 3.0) / w * (1.0 - 1e-9)) : Kmax;
  if (!(K > 0)) { why = "internal: no slope key scale"; return CBM_ERR_INVALID_ARG; }
  const int R = (int)std::ceil(w * K) + 3;
  if (R < 3 || R > 254) { why = "internal: slope key window out of range"; return CBM_ERR_INVALID_ARG; }
  p.key_R = R;
  int sh = 2;
  while ((1 << sh) < R) ++sh;
  p.cell_sh = sh;
  // Packed test: P = (kx mod 2^16) | (ky mod 2^16) << 16.  With key_add = R | (R+1) << 16 the low half of
  // P_a + key_add - P_b is (dkx + R) mod 2^16 in [0, 2R] and the high half is (dky + R + 1 + carry) mod 2^16,
  // carry in {-1, 0, 1}, in [0, 2R+2], whenever |dkx|, |dky| <= R: both halves are below 2^m >= 2R + 3.
  int m = 3;
  while ((1 << m) < 2 * R + 3) ++m;
  const uint32_t half = 0xFFFFu & ~((1u << m) - 1u);
  p.key_mask = half | (half << 16);
  p.key_add = (uint32_t)R | ((uint32_t)(R + 1) << 16);
  for (uint32_t l = 0; l < p.L; ++l) {
    const double m = std::ldexp(K, 32) / (double)p.z[l];
    const long long mi = llround(m);
    if (mi < 0 || mi > 0x7FFFFFFFll) { why = "internal: key multiplier out of range"; return CBM_ERR_INVALID_ARG; }
    p.key_mul[l] = (int32_t)mi;
  }
  return CBM_OK;
}

// ---------------------------------------------------------------------------------------------- allocation
int alloc_scratch(cbm_trigger* h, Scratch& s) {
  CBM_CUDA(h, cudaMalloc(&s.d_ctrl, sizeof(Ctrl)));
  CBM_CUDA(h, cudaMalloc(&s.d_selcnt, ((size_t)h->cfg.max_events / kSelEvents + 1) * sizeof(uint32_t)));
  CBM_CUDA(h, cudaMalloc(&s.d_gsum, ((size_t)h->cfg.max_events / kGatherEvents + 1) * sizeof(unsigned long long)));
  CBM_CUDA(h, cudaMalloc(&s.d_hitbase, ((size_t)h->cfg.max_events + 1) * sizeof(uint32_t)));
  {
    const size_t n = (size_t)h->cfg.max_events * h->p.L;
    CBM_CUDA(h, cudaMalloc(&s.d_fcnt, (n + n / kSelEvents + 2) * sizeof(uint32_t)));
  }
  for (int c = 0; c < kNumLists; ++c) CBM_CUDA(h, cudaMalloc(&s.d_list[c], (size_t)h->cfg.max_events * sizeof(uint32_t)));
  CBM_CUDA(h, cudaMalloc(&s.d_spill[0], (size_t)h->grid[kClsG] * 6 * kCapG * sizeof(uint32_t)));
  CBM_CUDA(h, cudaMalloc(&s.d_spill[1], (size_t)h->grid[kClsX] * 6 * kCapG * sizeof(uint32_t)));
  CBM_CUDA(h, cudaMalloc(&s.d_spill[2], (size_t)h->grid_hc * 6 * kCapH * sizeof(uint32_t)));
  return CBM_OK;
}
void free_scratch(Scratch& s) {
  cudaFree(s.d_ctrl);
  cudaFree(s.d_selcnt);
  cudaFree(s.d_gsum);
  cudaFree(s.d_hitbase);
  cudaFree(s.d_fcnt);
  for (int c = 0; c < kNumLists; ++c) cudaFree(s.d_list[c]);
  for (auto& sp : s.d_spill) cudaFree(sp);
  s = Scratch();
}
int make_prof(cbm_trigger* h, ProfEvents& pe) {
  for (auto& e : pe.k) CBM_CUDA(h, cudaEventCreate(&e));
  for (auto& e : pe.h2d) CBM_CUDA(h, cudaEventCreate(&e));
  for (auto& e : pe.d2h) CBM_CUDA(h, cudaEventCreate(&e));
  return CBM_OK;
}
void free_prof(ProfEvents& pe) {
  for (auto& e : pe.k) if (e) cudaEventDestroy(e);
  for (auto& e : pe.h2d) if (e) cudaEventDestroy(e);
  for (auto& e : pe.d2h) if (e) cudaEventDestroy(e);
  pe = ProfEvents();
}

int alloc_slot(cbm_trigger* h, Slot& s) {
  const cbm_trigger_config_t& c = h->cfg;
  const size_t nh = (size_t)((c.max_hits + 3) & ~3ull) + 4;  // 16-byte tail padding for the bulk copies
  const size_t noff = (size_t)c.max_events * h->p.L + 1;
  const size_t ne = c.max_events, S = h->p.S;
  if (c.flags & CBM_FLAG_PACKED_INPUT) {
    CBM_CUDA(h, cudaHostAlloc(&s.h_p, nh * 5, cudaHostAllocDefault));  // nh is a multiple of 4: whole 20-byte groups
    CBM_CUDA(h, cudaMalloc(&s.d_p, nh * 5));
  } else {
    CBM_CUDA(h, cudaHostAlloc(&s.h_x, nh * 4, cudaHostAllocDefault));
    CBM_CUDA(h, cudaHostAlloc(&s.h_y, nh * 4, cudaHostAllocDefault));
  }
  CBM_CUDA(h, cudaHostAlloc(&s.h_off, noff * 4, cudaHostAllocDefault));
  CBM_CUDA(h, cudaMalloc(&s.d_x, nh * 4));
  CBM_CUDA(h, cudaMalloc(&s.d_y, nh * 4));
  CBM_CUDA(h, cudaMalloc(&s.d_off, noff * 4));
  CBM_CUDA(h, cudaMalloc(&s.d_nt, ne * S * 4));
  CBM_CUDA(h, cudaMalloc(&s.d_nc, ne * 4));
  CBM_CUDA(h, cudaMalloc(&s.d_ac, ne));
  CBM_CUDA(h, cudaMalloc(&s.d_sel, ne * 4));
  CBM_CUDA(h, cudaMalloc(&s.d_nsel, 4));
  CBM_CUDA(h, cudaHostAlloc(&s.h_nsel, 4, cudaHostAllocDefault));
  CBM_CUDA(h, cudaHostAlloc(&s.h_nt, ne * S * 4, cudaHostAllocDefault));
  CBM_CUDA(h, cudaHostAlloc(&s.h_nc, ne * 4, cudaHostAllocDefault));
  CBM_CUDA(h, cudaHostAlloc(&s.h_ac, ne, cudaHostAllocDefault));
  CBM_CUDA(h, cudaHostAlloc(&s.h_ctrl, sizeof(Ctrl), cudaHostAllocDefault));
  CBM_CUDA(h, cudaMemset(s.d_x + (nh - 8), 0, 32));
  CBM_CUDA(h, cudaMemset(s.d_y + (nh - 8), 0, 32));
  int rc = alloc_scratch(h, s.scr);
  if (rc) return rc;
  CBM_CUDA(h, cudaEventCreateWithFlags(&s.ev_h2d, cudaEventDisableTiming));
  CBM_CUDA(h, cudaEventCreateWithFlags(&s.ev_run, cudaEventDisableTiming));
  CBM_CUDA(h, cudaEventCreateWithFlags(&s.ev_d2h, cudaEventDisableTiming));
  if (c.flags & CBM_FLAG_PROFILE) { rc = make_prof(h, s.prof); if (rc) return rc; }
  return CBM_OK;
}
void free_slot(Slot& s) {
  cudaFreeHost(s.h_x); cudaFreeHost(s.h_y); cudaFreeHost(s.h_off);
  cudaFreeHost(s.h_p); cudaFree(s.d_p);
  cudaFree(s.d_x); cudaFree(s.d_y); cudaFree(s.d_off);
  cudaFree(s.d_nt); cudaFree(s.d_nc); cudaFree(s.d_ac);
  cudaFree(s.d_sel); cudaFree(s.d_nsel); cudaFreeHost(s.h_nsel);
  cudaFreeHost(s.h_nt); cudaFreeHost(s.h_nc); cudaFreeHost(s.h_ac); cudaFreeHost(s.h_ctrl);
  free_scratch(s.scr);
  free_prof(s.prof);
  if (s.ev_h2d) cudaEventDestroy(s.ev_h2d);
  if (s.ev_run) cudaEventDestroy(s.ev_run);
  if (s.ev_d2h) cudaEventDestroy(s.ev_d2h);
  s = Slot();
}

// ---------------------------------------------------------------------------------------------- launches
// a3..a8.  classify_kernel on the caller's stream; then the tile kernel and the class kernels M, G on side
// streams beside class H on the caller's stream (disjoint events), joined before the list-X kernel, which
// redoes the few events another kernel handed on.  CBM_FLAG_SERIAL: everything on the caller's stream, one
// kernel after the other (per-kernel times that are kernel times).
// Returns the number of kernels launched (0 on an empty batch), < 0 on error.
int launch_selection(cbm_trigger* h, const Scratch& scr, const int32_t* d_x, const int32_t* d_y, const uint32_t* d_off,
                     uint32_t n_events, uint64_t n_hits, uint32_t* d_nt, uint32_t* d_nc, uint8_t* d_ac,
                     cudaStream_t st, ProfEvents* prof) {
  const Params& p = h->p;
  CBM_CUDA(h, cudaMemsetAsync(scr.d_ctrl, 0, sizeof(Ctrl), st));
  if (prof) prof->valid = false;
  if (n_events == 0) return 0;
  const bool serial = h->cfg.flags & CBM_FLAG_SERIAL;
  cudaStream_t s_tile = serial ? st : h->st_side[2], s_m = serial ? st : h->st_side[0], s_g = serial ? st : h->st_side[1];
  auto rec = [&](int k, int end, cudaStream_t s) { return prof ? cudaEventRecord(prof->k[2 * k + end], s) : cudaSuccess; };
  CBM_CUDA(h, rec(kKClassify, 0, st));
  const uint32_t n_cta = (n_events + kClassifyWarps * kTileEvents - 1) / (kClassifyWarps * kTileEvents);
  classify_kernel<<<n_cta, 32 * kClassifyWarps, 0, st>>>(p, d_off, n_events, (uint32_t)n_hits, d_nt, d_nc, d_ac, scr.d_ctrl,
                                                         scr.d_list[kClsM], scr.d_list[kClsH], scr.d_list[kClsG]);
  CBM_CUDA(h, rec(kKClassify, 1, st));
  if (!serial) {
    CBM_CUDA(h, cudaEventRecord(h->ev_fork, st));
    for (auto& sd : h->st_side) CBM_CUDA(h, cudaStreamWaitEvent(sd, h->ev_fork, 0));
  }
  // From here on the side streams hang off the caller's stream.  A CUDA error must not leave them un-joined (their
  // kernels would run unordered against whatever the caller enqueues next, and against ev_run): the first error is
  // kept, nothing more is launched, and the join below is still recorded and waited on before the error is returned.
  cudaError_t err = cudaSuccess;
  const char* err_at = "";
#define FORKED(expr) do { if (err == cudaSuccess && (err = (expr)) != cudaSuccess) err_at = #expr; } while (0)
  // G and M first: on most workloads their persistent CTAs find a short list and leave at once
  FORKED(rec(kKTeamG, 0, s_g));
  if (err == cudaSuccess)
    TEAM_KERNEL_G<<<h->grid[kClsG], 32 * SmemG::W, sizeof(SmemG), s_g>>>(
        p, d_x, d_y, d_off, d_nt, d_nc, d_ac, scr.d_ctrl, scr.d_list[kClsG], scr.d_list[kClsX], scr.d_spill[0]);
  FORKED(cudaGetLastError());
  FORKED(rec(kKTeamG, 1, s_g));
  FORKED(rec(kKTeamM, 0, s_m));
  if (err == cudaSuccess)
    TEAM_KERNEL_M<<<h->grid[kClsM], 32 * SmemM::W, 0, s_m>>>(
        p, d_x, d_y, d_off, d_nt, d_nc, d_ac, scr.d_ctrl, scr.d_list[kClsM], scr.d_list[kClsX], nullptr);
  FORKED(cudaGetLastError());
  FORKED(rec(kKTeamM, 1, s_m));
  FORKED(rec(kKTeamH, 0, st));
  if (err == cudaSuccess)
    CHAIN_KERNEL_H<<<h->grid_hc, 32 * kWarpsH, 0, st>>>(p, d_x, d_y, d_off, d_nt, d_nc, d_ac, scr.d_ctrl, scr.d_list[kClsH],
                                                        scr.d_spill[2]);
  FORKED(cudaGetLastError());
  FORKED(rec(kKTeamH, 1, st));
  if (p.tiny_max_total) {
    FORKED(rec(kKTile, 0, s_tile));
    const uint32_t n_tiles = (n_events + kTileEvents - 1) / kTileEvents;
    if (err != cudaSuccess) {
    } else if (p.S <= 4)  // tables sized for 4 stations: more resident CTAs
      tile_kernel<4><<<n_tiles, kTileEvents * p.S, 0, s_tile>>>(p, d_x, d_y, d_off, n_events, (uint32_t)n_hits, d_nt, d_nc,
                                                                d_ac, scr.d_ctrl, scr.d_list[kClsX]);
    else
      tile_kernel<kMaxStations><<<n_tiles, kTileEvents * p.S, 0, s_tile>>>(p, d_x, d_y, d_off, n_events, (uint32_t)n_hits, d_nt,
                                                                           d_nc, d_ac, scr.d_ctrl, scr.d_list[kClsX]);
    FORKED(cudaGetLastError());
    FORKED(rec(kKTile, 1, s_tile));
  } else if (prof) {
    FORKED(rec(kKTile, 0, s_tile));
    FORKED(rec(kKTile, 1, s_tile));
  }
  if (!serial)
    for (int i = 0; i < 3; ++i) {  // always, also after an error above
      cudaError_t e1 = cudaEventRecord(h->ev_join[i], h->st_side[i]);
      if (e1 == cudaSuccess) e1 = cudaStreamWaitEvent(st, h->ev_join[i], 0);
      if (err == cudaSuccess && e1 != cudaSuccess) { err = e1; err_at = "join of the side streams"; }
    }
#undef FORKED
  if (err != cudaSuccess) return fail(h, CBM_ERR_CUDA, "%s: %s", err_at, cudaGetErrorString(err));
  CBM_CUDA(h, rec(kKTeamX, 0, st));
  TEAM_KERNEL_X<<<h->grid[kClsX], 32 * SmemG::W, sizeof(SmemG), st>>>(
      p, d_x, d_y, d_off, d_nt, d_nc, d_ac, scr.d_ctrl, scr.d_list[kClsX], scr.d_list[kClsX], scr.d_spill[1]);
  CBM_CUDA(h, rec(kKTeamX, 1, st));
  if (prof) prof->valid = true;
  CBM_CUDA(h, cudaGetLastError());
  return CBM_TRIGGER_N_KERNELS;
}

// The list of selected events: ascending ids of the events with accept != 0, and their number.
int launch_compaction(cbm_trigger* h, const Scratch& scr, const uint8_t* d_ac, uint32_t n_events, uint32_t* d_sel,
                      uint32_t* d_nsel, cudaStream_t st) {
  if (n_events == 0) {
    CBM_CUDA(h, cudaMemsetAsync(d_nsel, 0, sizeof(uint32_t), st));
    return 0;
  }
  const uint32_t nb = (n_events + kSelEvents - 1) / kSelEvents;
  select_count_kernel<<<nb, kSelThreads, 0, st>>>(d_ac, n_events, scr.d_selcnt);
  select_write_kernel<<<nb, kSelThreads, 0, st>>>(d_ac, n_events, scr.d_selcnt, d_sel, d_nsel);
  CBM_CUDA(h, cudaGetLastError());
  return 2;
}

void fill_stats(cbm_trigger_stats_t& st, const Ctrl& c, uint32_t n_events, uint64_t n_hits, uint32_t n_launches) {
  memset(&st, 0, sizeof(st));
  st.struct_size = sizeof(st);
  st.n_events = n_events;
  st.n_hits = n_hits;
  st.n_class[0] = c.n_tiny;
  st.n_class[1] = c.count[kClsM]; st.n_class[2] = c.count[kClsH]; st.n_class[3] = c.count[kClsG];
  st.n_redone = c.count[kClsX];
  st.n_invalid = c.n_invalid;
  st.first_invalid = c.first_invalid_inv ? ~c.first_invalid_inv : 0xFFFFFFFFu;
  st.n_launches = n_launches;
}

void fill_prof(cbm_trigger_stats_t& st, ProfEvents& pe, bool copies) {
  if (!pe.valid) return;
  for (int k = 0; k < CBM_TRIGGER_N_KERNELS; ++k) {
    float ms = 0;
    if (cudaEventElapsedTime(&ms, pe.k[2 * k], pe.k[2 * k + 1]) == cudaSuccess) st.kernel_ms[k] = ms;
  }
  if (copies) {
    float ms = 0;
    if (cudaEventElapsedTime(&ms, pe.h2d[0], pe.h2d[1]) == cudaSuccess) st.h2d_ms = ms;
    if (cudaEventElapsedTime(&ms, pe.d2h[0], pe.d2h[1]) == cudaSuccess) st.d2h_ms = ms;
  }
}

template <class K>
int occupancy_grid(cbm_trigger* h, K kernel, int threads, size_t smem, int* grid) {
  if (smem) CBM_CUDA(h, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  CBM_CUDA(h, cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
  int per_sm = 0;
  CBM_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem));
  if (per_sm < 1) return fail(h, CBM_ERR_CUDA, "a team kernel does not fit on this device");
  *grid = per_sm * h->n_sm;
  return CBM_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------- no allocation
// cbm_trigger_select_noalloc: the selection list for callers that may not allocate (a readout loop whose device
// memory was handed out at start of run; code that only gets pointers and a stream from its host framework).
// The per-block counts that select_count_kernel writes and select_write_kernel reads normally sit in a cudaMalloc'ed
// buffer of the handle (Scratch::d_selcnt).  Here they sit in this array, which is part of the library's device image:
// the driver places one copy on every device that loads the library and keeps it until the process ends (16 KB each).
// On the host, the name g_noalloc_block_count is only a stand-in that identifies the symbol; it is NOT the device
// address and must never be handed to a kernel.  noalloc_block_count() asks the runtime for the real address, once
// per device, with that device current, and hands that to the kernels.
constexpr uint32_t kNoAllocMaxBlocks = CBM_TRIGGER_NOALLOC_MAX_EVENTS / cbm::kSelEvents;
static_assert(CBM_TRIGGER_NOALLOC_MAX_EVENTS % cbm::kSelEvents == 0, "whole blocks");
static __device__ __align__(256) uint32_t g_noalloc_block_count[kNoAllocMaxBlocks];

namespace {

constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
uint32_t* g_noalloc_addr[kNoAllocMaxDevices];  // device address of the array on device i; nullptr = not looked up yet

// Device address of g_noalloc_block_count on the current device (looked up on the first call per device).
int noalloc_block_count(uint32_t** out) {
  int dev = -1;
  CBM_CUDA(nullptr, cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(nullptr, CBM_ERR_CUDA, "select_noalloc: device %d is beyond the %d this call supports", dev, kNoAllocMaxDevices);
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[dev]) {
    void* p = nullptr;
    CBM_CUDA(nullptr, cudaGetSymbolAddress(&p, g_noalloc_block_count));
    if (!p) return fail(nullptr, CBM_ERR_CUDA, "select_noalloc: cudaGetSymbolAddress returned no address");
    g_noalloc_addr[dev] = static_cast<uint32_t*>(p);
  }
  *out = g_noalloc_addr[dev];
  return CBM_OK;
}

}  // namespace

// ================================================================================================ C ABI
extern "C" {

int cbm_trigger_select_noalloc(uint32_t n_events, const uint8_t* d_accept, uint32_t* d_event_ids, uint32_t* d_n_selected,
                               void* stream) {
  if (n_events > CBM_TRIGGER_NOALLOC_MAX_EVENTS)
    return fail(nullptr, CBM_ERR_CAPACITY, "select_noalloc: n_events %u is above the fixed limit of %u events (the scratch of this call "
                "is a fixed array in the library image); split the batch or use cbm_trigger_select_device", n_events,
                CBM_TRIGGER_NOALLOC_MAX_EVENTS);
  if (!d_n_selected || (n_events && (!d_accept || !d_event_ids)))
    return fail(nullptr, CBM_ERR_INVALID_ARG, "select_noalloc: device pointers must not be NULL");
  cudaStream_t st = (cudaStream_t)stream;
  if (n_events == 0) {
    CBM_CUDA(nullptr, cudaMemsetAsync(d_n_selected, 0, sizeof(uint32_t), st));
    return CBM_OK;
  }
  uint32_t* d_block_count = nullptr;
  const int rc = noalloc_block_count(&d_block_count);
  if (rc) return rc;
  // select_count_kernel writes entries 0..nb-1, select_write_kernel reads entries below its block index: every entry
  // read was written by this call, so what an earlier call left in the array does not matter.
  const uint32_t nb = (n_events + kSelEvents - 1) / kSelEvents;  // <= kNoAllocMaxBlocks
  select_count_kernel<<<nb, kSelThreads, 0, st>>>(d_accept, n_events, d_block_count);
  select_write_kernel<<<nb, kSelThreads, 0, st>>>(d_accept, n_events, d_block_count, d_event_ids, d_n_selected);
  CBM_CUDA(nullptr, cudaGetLastError());
  return CBM_OK;
}

const char* cbm_trigger_version(void) { return "cbm-trigger 0.2 sm_100a"; }

const char* cbm_trigger_last_error(const cbm_trigger_t* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

int cbm_trigger_create(const cbm_trigger_config_t* cfg, cbm_trigger_t** out) {
  if (!cfg || !out) return fail(nullptr, CBM_ERR_INVALID_ARG, "cfg and out must not be NULL");
  if (cfg->struct_size != sizeof(cbm_trigger_config_t))
    return fail(nullptr, CBM_ERR_INVALID_ARG, "struct_size %u != %zu", cfg->struct_size, sizeof(cbm_trigger_config_t));
  Params p;
  std::string why;
  int rc = build_params(*cfg, p, why);
  if (rc) return fail(nullptr, rc, "%s", why.c_str());

  cbm_trigger* h = new (std::nothrow) cbm_trigger();
  if (!h) return fail(nullptr, CBM_ERR_CUDA, "out of host memory");
  h->cfg = *cfg;
  h->p = p;
  auto bail = [&](int code) {
    g_create_err = h->err;
    cbm_trigger_destroy(h);
    return code;
  };
  int n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess || n_dev == 0) {
    fail(h, CBM_ERR_CUDA, "no CUDA device: %s (there is no CPU fallback)", e != cudaSuccess ? cudaGetErrorString(e) : "count is 0");
    return bail(CBM_ERR_CUDA);
  }
  if (cfg->device >= n_dev) { fail(h, CBM_ERR_INVALID_ARG, "device %d of %d", cfg->device, n_dev); return bail(CBM_ERR_INVALID_ARG); }
#define CREATE_TRY(call) do { int rc_ = (call); if (rc_) return bail(rc_); } while (0)
#define CREATE_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { fail(h, CBM_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); return bail(CBM_ERR_CUDA); } } while (0)
  CREATE_CUDA(cudaSetDevice(cfg->device));
  cudaDeviceProp prop;
  CREATE_CUDA(cudaGetDeviceProperties(&prop, cfg->device));
  if (prop.major < 10) { fail(h, CBM_ERR_CUDA, "device is sm_%d%d; this library holds sm_100a code only", prop.major, prop.minor); return bail(CBM_ERR_CUDA); }
  h->n_sm = prop.multiProcessorCount;
  static_assert(sizeof(SmemM) <= 48 * 1024 && sizeof(SmemHC) <= 48 * 1024, "static shared memory limit");
  CREATE_CUDA(cudaFuncSetAttribute(tile_kernel<4>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
  CREATE_CUDA(cudaFuncSetAttribute(tile_kernel<kMaxStations>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
  CREATE_TRY(occupancy_grid(h, TEAM_KERNEL_M, 32 * SmemM::W, 0, &h->grid[kClsM]));
  CREATE_TRY(occupancy_grid(h, CHAIN_KERNEL_H, 32 * kWarpsH, 0, &h->grid_hc));
  CREATE_TRY(occupancy_grid(h, TEAM_KERNEL_G, 32 * SmemG::W, sizeof(SmemG), &h->grid[kClsG]));
  CREATE_TRY(occupancy_grid(h, TEAM_KERNEL_X, 32 * SmemG::W, sizeof(SmemG), &h->grid[kClsX]));
  CREATE_CUDA(cudaStreamCreateWithFlags(&h->st_h2d, cudaStreamNonBlocking));
  CREATE_CUDA(cudaStreamCreateWithFlags(&h->st_run, cudaStreamNonBlocking));
  CREATE_CUDA(cudaStreamCreateWithFlags(&h->st_d2h, cudaStreamNonBlocking));
  for (auto& sd : h->st_side) CREATE_CUDA(cudaStreamCreateWithFlags(&sd, cudaStreamNonBlocking));
  CREATE_CUDA(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
  for (auto& ej : h->ev_join) CREATE_CUDA(cudaEventCreateWithFlags(&ej, cudaEventDisableTiming));
  CREATE_TRY(alloc_scratch(h, h->dev_scr));
  CREATE_CUDA(cudaHostAlloc(&h->h_dev_ctrl, sizeof(Ctrl), cudaHostAllocDefault));
  if (cfg->flags & CBM_FLAG_PROFILE)
    for (auto& pe : h->dev_prof) CREATE_TRY(make_prof(h, pe));
  for (uint32_t i = 0; i < cfg->n_slots; ++i) CREATE_TRY(alloc_slot(h, h->slot[i]));
#undef CREATE_TRY
#undef CREATE_CUDA
  *out = h;
  return CBM_OK;
}

void cbm_trigger_destroy(cbm_trigger_t* h) {
  if (!h) return;
  if (h->st_h2d || h->st_run || h->st_d2h) {
    cudaSetDevice(h->cfg.device);
    if (h->st_h2d) cudaStreamSynchronize(h->st_h2d);
    if (h->st_run) cudaStreamSynchronize(h->st_run);
    if (h->st_d2h) cudaStreamSynchronize(h->st_d2h);
  }
  for (auto& s : h->slot) free_slot(s);
  free_scratch(h->dev_scr);
  for (auto& pe : h->dev_prof) free_prof(pe);
  if (h->h_dev_ctrl) cudaFreeHost(h->h_dev_ctrl);
  if (h->st_h2d) cudaStreamDestroy(h->st_h2d);
  if (h->st_run) cudaStreamDestroy(h->st_run);
  if (h->st_d2h) cudaStreamDestroy(h->st_d2h);
  for (auto& sd : h->st_side) if (sd) cudaStreamDestroy(sd);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  for (auto& ej : h->ev_join) if (ej) cudaEventDestroy(ej);
  delete h;
}

static int check_slot(cbm_trigger_t* h, uint32_t slot) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (slot >= h->cfg.n_slots) return fail(h, CBM_ERR_STATE, "slot %u of %u", slot, h->cfg.n_slots);
  return CBM_OK;
}

int cbm_trigger_host_buffers(cbm_trigger_t* h, uint32_t slot, int32_t** x, int32_t** y, uint32_t** off) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  if (!x || !y || !off) return fail(h, CBM_ERR_INVALID_ARG, "x, y, off must not be NULL");
  if (h->cfg.flags & CBM_FLAG_PACKED_INPUT) return fail(h, CBM_ERR_STATE, "the handle takes packed input (CBM_FLAG_PACKED_INPUT)");
  *x = h->slot[slot].h_x; *y = h->slot[slot].h_y; *off = h->slot[slot].h_off;
  return CBM_OK;
}

int cbm_trigger_upload_events(cbm_trigger_t* h, uint32_t slot, uint32_t n_events, uint64_t n_hits, const int32_t* x,
                              const int32_t* y, const uint32_t* off) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  Slot& s = h->slot[slot];
  if (h->cfg.flags & CBM_FLAG_PACKED_INPUT) return fail(h, CBM_ERR_STATE, "the handle takes packed input (CBM_FLAG_PACKED_INPUT)");
  if (!off || (n_hits && (!x || !y))) return fail(h, CBM_ERR_INVALID_ARG, "x, y, off must not be NULL");
  if (n_events > h->cfg.max_events) return fail(h, CBM_ERR_CAPACITY, "n_events %u > max_events %u", n_events, h->cfg.max_events);
  if (n_hits > h->cfg.max_hits) return fail(h, CBM_ERR_CAPACITY, "n_hits %llu > max_hits %llu", (unsigned long long)n_hits, (unsigned long long)h->cfg.max_hits);
  if (s.state == kRunning) return fail(h, CBM_ERR_STATE, "slot %u holds unfetched results", slot);
  const size_t n_off = (size_t)n_events * h->p.L + 1;
  if (off[0] != 0 || off[n_off - 1] != n_hits)
    return fail(h, CBM_ERR_RANGE, "off[0] must be 0 and off[n_events*L] must equal n_hits");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  // the staging buffers may still be the source of the slot's previous H2D
  CBM_CUDA(h, cudaEventSynchronize(s.ev_h2d));
  if (x != s.h_x && n_hits) staging_copy(s.h_x, x, n_hits * 4);
  if (y != s.h_y && n_hits) staging_copy(s.h_y, y, n_hits * 4);
  if (off != s.h_off) staging_copy(s.h_off, off, n_off * 4);
  // the device arrays may still be read by the slot's previous kernels
  CBM_CUDA(h, cudaStreamWaitEvent(h->st_h2d, s.ev_run, 0));
  const bool prof = h->cfg.flags & CBM_FLAG_PROFILE;
  if (prof) CBM_CUDA(h, cudaEventRecord(s.prof.h2d[0], h->st_h2d));
  if (n_hits) {
    CBM_CUDA(h, cudaMemcpyAsync(s.d_x, s.h_x, n_hits * 4, cudaMemcpyHostToDevice, h->st_h2d));
    CBM_CUDA(h, cudaMemcpyAsync(s.d_y, s.h_y, n_hits * 4, cudaMemcpyHostToDevice, h->st_h2d));
  }
  CBM_CUDA(h, cudaMemcpyAsync(s.d_off, s.h_off, n_off * 4, cudaMemcpyHostToDevice, h->st_h2d));
  if (prof) CBM_CUDA(h, cudaEventRecord(s.prof.h2d[1], h->st_h2d));
  CBM_CUDA(h, cudaEventRecord(s.ev_h2d, h->st_h2d));
  s.n_events = n_events;
  s.n_hits = n_hits;
  s.sel_valid = false;
  s.state = kUploaded;
  return CBM_OK;
}

int cbm_trigger_host_buffers_packed(cbm_trigger_t* h, uint32_t slot, uint8_t** xy20, uint32_t** off) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  if (!xy20 || !off) return fail(h, CBM_ERR_INVALID_ARG, "xy20, off must not be NULL");
  if (!(h->cfg.flags & CBM_FLAG_PACKED_INPUT)) return fail(h, CBM_ERR_STATE, "the handle was created without CBM_FLAG_PACKED_INPUT");
  *xy20 = h->slot[slot].h_p; *off = h->slot[slot].h_off;
  return CBM_OK;
}

int cbm_trigger_upload_events_packed(cbm_trigger_t* h, uint32_t slot, uint32_t n_events, uint64_t n_hits,
                                     const uint8_t* xy20, const uint32_t* off) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  Slot& s = h->slot[slot];
  if (!(h->cfg.flags & CBM_FLAG_PACKED_INPUT)) return fail(h, CBM_ERR_STATE, "the handle was created without CBM_FLAG_PACKED_INPUT");
  if (!off || (n_hits && !xy20)) return fail(h, CBM_ERR_INVALID_ARG, "xy20, off must not be NULL");
  if (n_events > h->cfg.max_events) return fail(h, CBM_ERR_CAPACITY, "n_events %u > max_events %u", n_events, h->cfg.max_events);
  if (n_hits > h->cfg.max_hits) return fail(h, CBM_ERR_CAPACITY, "n_hits %llu > max_hits %llu", (unsigned long long)n_hits, (unsigned long long)h->cfg.max_hits);
  if (s.state == kRunning) return fail(h, CBM_ERR_STATE, "slot %u holds unfetched results", slot);
  const size_t n_off = (size_t)n_events * h->p.L + 1;
  if (off[0] != 0 || off[n_off - 1] != n_hits)
    return fail(h, CBM_ERR_RANGE, "off[0] must be 0 and off[n_events*L] must equal n_hits");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  CBM_CUDA(h, cudaEventSynchronize(s.ev_h2d));  // the staging buffers may still be the source of the previous H2D
  const size_t n_bytes = (size_t)n_hits * 5, n_copy = (size_t)((n_hits + 3) / 4) * 20;  // whole 20-byte groups
  if (xy20 != s.h_p && n_hits) staging_copy(s.h_p, xy20, n_bytes);
  if (off != s.h_off) staging_copy(s.h_off, off, n_off * 4);
  CBM_CUDA(h, cudaStreamWaitEvent(h->st_h2d, s.ev_run, 0));  // the device arrays may still be read by the previous kernels
  const bool prof = h->cfg.flags & CBM_FLAG_PROFILE;
  if (prof) CBM_CUDA(h, cudaEventRecord(s.prof.h2d[0], h->st_h2d));
  if (n_hits) CBM_CUDA(h, cudaMemcpyAsync(s.d_p, s.h_p, n_copy, cudaMemcpyHostToDevice, h->st_h2d));
  CBM_CUDA(h, cudaMemcpyAsync(s.d_off, s.h_off, n_off * 4, cudaMemcpyHostToDevice, h->st_h2d));
  if (prof) CBM_CUDA(h, cudaEventRecord(s.prof.h2d[1], h->st_h2d));
  CBM_CUDA(h, cudaEventRecord(s.ev_h2d, h->st_h2d));
  s.n_events = n_events;
  s.n_hits = n_hits;
  s.sel_valid = false;
  s.packed_pending = true;
  s.state = kUploaded;
  return CBM_OK;
}

int cbm_trigger_pack_xy20(const int32_t* x, const int32_t* y, uint64_t n_hits, uint8_t* out, uint64_t* first_bad) {
  if (first_bad) *first_bad = n_hits;
  if (n_hits && (!x || !y || !out)) return fail(nullptr, CBM_ERR_INVALID_ARG, "pack_xy20: x, y, out must not be NULL");
  constexpr int32_t kMin = -(1 << 19), kMax = (1 << 19) - 1;
  for (uint64_t i = 0; i < n_hits; ++i) {
    const int32_t xv = x[i], yv = y[i];
    if (xv < kMin || xv > kMax || yv < kMin || yv > kMax) {
      if (first_bad) *first_bad = i;
      return fail(nullptr, CBM_ERR_RANGE, "pack_xy20: hit %llu (%d, %d) is outside the 20-bit range of XY20", (unsigned long long)i, xv, yv);
    }
    // bits 0..19 = x, bits 20..39 = y (two's complement), little endian
    const uint64_t v = ((uint64_t)(uint32_t)xv & 0xFFFFFu) | (((uint64_t)(uint32_t)yv & 0xFFFFFu) << 20);
    uint8_t* o = out + 5 * i;
    o[0] = (uint8_t)v; o[1] = (uint8_t)(v >> 8); o[2] = (uint8_t)(v >> 16); o[3] = (uint8_t)(v >> 24); o[4] = (uint8_t)(v >> 32);
  }
  return CBM_OK;
}

int cbm_trigger_run(cbm_trigger_t* h, uint32_t slot) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  Slot& s = h->slot[slot];
  if (s.state != kUploaded) return fail(h, CBM_ERR_STATE, "slot %u: run needs a preceding upload_events", slot);
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  const bool prof = h->cfg.flags & CBM_FLAG_PROFILE;
  CBM_CUDA(h, cudaStreamWaitEvent(h->st_run, s.ev_h2d, 0));
  CBM_CUDA(h, cudaStreamWaitEvent(h->st_run, s.ev_d2h, 0));  // previous results of this slot must have left
  if (s.packed_pending) {  // a2': expand the XY20 stream into the int32 arrays the kernels read
    if (s.n_hits) {
      const uint64_t groups = (s.n_hits + 3) / 4;
      unpack_xy20_kernel<<<(unsigned)((groups + kWireThreads - 1) / kWireThreads), kWireThreads, 0, h->st_run>>>(
          s.d_p, s.n_hits, s.d_x, s.d_y);
      CBM_CUDA(h, cudaGetLastError());
    }
    s.packed_pending = false;
  }
  const int nl = launch_selection(h, s.scr, s.d_x, s.d_y, s.d_off, s.n_events, s.n_hits, s.d_nt, s.d_nc, s.d_ac,
                                  h->st_run, prof ? &s.prof : nullptr);
  if (nl < 0) return nl;
  const int nl2 = launch_compaction(h, s.scr, s.d_ac, s.n_events, s.d_sel, s.d_nsel, h->st_run);
  if (nl2 < 0) return nl2;
  CBM_CUDA(h, cudaEventRecord(s.ev_run, h->st_run));
  CBM_CUDA(h, cudaStreamWaitEvent(h->st_d2h, s.ev_run, 0));
  if (prof) CBM_CUDA(h, cudaEventRecord(s.prof.d2h[0], h->st_d2h));
  const size_t ne = s.n_events, S = h->p.S;
  if (ne) {
    CBM_CUDA(h, cudaMemcpyAsync(s.h_nt, s.d_nt, ne * S * 4, cudaMemcpyDeviceToHost, h->st_d2h));
    CBM_CUDA(h, cudaMemcpyAsync(s.h_nc, s.d_nc, ne * 4, cudaMemcpyDeviceToHost, h->st_d2h));
    CBM_CUDA(h, cudaMemcpyAsync(s.h_ac, s.d_ac, ne, cudaMemcpyDeviceToHost, h->st_d2h));
  }
  CBM_CUDA(h, cudaMemcpyAsync(s.h_ctrl, s.scr.d_ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, h->st_d2h));
  CBM_CUDA(h, cudaMemcpyAsync(s.h_nsel, s.d_nsel, sizeof(uint32_t), cudaMemcpyDeviceToHost, h->st_d2h));
  if (prof) CBM_CUDA(h, cudaEventRecord(s.prof.d2h[1], h->st_d2h));
  CBM_CUDA(h, cudaEventRecord(s.ev_d2h, h->st_d2h));
  s.stats.n_launches = (uint32_t)(nl + nl2);
  s.sel_valid = true;
  s.state = kRunning;
  return CBM_OK;
}

int cbm_trigger_fetch_results(cbm_trigger_t* h, uint32_t slot, uint32_t* n_triplets, uint32_t* n_candidates,
                              uint8_t* accept) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  Slot& s = h->slot[slot];
  if (s.state != kRunning) return fail(h, CBM_ERR_STATE, "slot %u: fetch_results needs a preceding run", slot);
  if (!n_candidates && s.n_events) return fail(h, CBM_ERR_INVALID_ARG, "n_candidates must not be NULL");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  CBM_CUDA(h, cudaEventSynchronize(s.ev_d2h));
  const size_t ne = s.n_events, S = h->p.S;
  if (ne) {
    if (n_triplets) memcpy(n_triplets, s.h_nt, ne * S * 4);
    memcpy(n_candidates, s.h_nc, ne * 4);
    if (accept) memcpy(accept, s.h_ac, ne);
  }
  const uint32_t nl = s.stats.n_launches;
  fill_stats(s.stats, *s.h_ctrl, s.n_events, s.n_hits, nl);
  if (h->cfg.flags & CBM_FLAG_PROFILE) fill_prof(s.stats, s.prof, true);
  s.state = kEmpty;
  if (s.stats.n_invalid)
    return fail(h, CBM_ERR_RANGE, "%u event(s) rejected on the device (offsets not monotone, beyond n_hits, or a layer above max_hits_per_layer); first: event %u",
                s.stats.n_invalid, s.stats.first_invalid);
  return CBM_OK;
}

int cbm_trigger_fetch_selected(cbm_trigger_t* h, uint32_t slot, uint32_t* event_ids, uint32_t capacity,
                               uint32_t* n_selected) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  Slot& s = h->slot[slot];
  if (!s.sel_valid) return fail(h, CBM_ERR_STATE, "slot %u: fetch_selected needs a preceding run", slot);
  if (!n_selected) return fail(h, CBM_ERR_INVALID_ARG, "n_selected must not be NULL");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  CBM_CUDA(h, cudaEventSynchronize(s.ev_d2h));  // the count came back with the results
  const uint32_t n = *s.h_nsel;
  *n_selected = n;
  if (n > capacity) return fail(h, CBM_ERR_CAPACITY, "%u events selected, room for %u", n, capacity);
  if (n) {
    if (!event_ids) return fail(h, CBM_ERR_INVALID_ARG, "event_ids must not be NULL");
    CBM_CUDA(h, cudaMemcpyAsync(event_ids, s.d_sel, (size_t)n * 4, cudaMemcpyDeviceToHost, h->st_d2h));
    CBM_CUDA(h, cudaStreamSynchronize(h->st_d2h));
  }
  return CBM_OK;
}

int cbm_trigger_select_device(cbm_trigger_t* h, uint32_t n_events, const uint8_t* d_accept, uint32_t* d_event_ids,
                              uint32_t* d_n_selected, void* stream) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (n_events > h->cfg.max_events) return fail(h, CBM_ERR_CAPACITY, "n_events %u > max_events %u", n_events, h->cfg.max_events);
  if (!d_n_selected || (n_events && (!d_accept || !d_event_ids))) return fail(h, CBM_ERR_INVALID_ARG, "device pointers must not be NULL");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  const int nl = launch_compaction(h, h->dev_scr, d_accept, n_events, d_event_ids, d_n_selected, (cudaStream_t)stream);
  return nl < 0 ? nl : CBM_OK;
}

int cbm_trigger_gather_device(cbm_trigger_t* h, uint32_t n_events, uint64_t n_hits, const int32_t* d_x, const int32_t* d_y,
                              const uint32_t* d_off, const uint32_t* d_event_ids, const uint32_t* d_n_selected,
                              int32_t* d_out_x, int32_t* d_out_y, uint32_t* d_out_off, unsigned long long* d_out_n_hits,
                              void* stream) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (n_events > h->cfg.max_events) return fail(h, CBM_ERR_CAPACITY, "n_events %u > max_events %u", n_events, h->cfg.max_events);
  if (n_hits >= (1ull << 32)) return fail(h, CBM_ERR_CAPACITY, "n_hits must be < 2^32");
  if (!d_n_selected || !d_out_off || !d_out_n_hits || (n_events && (!d_off || !d_event_ids || !d_x || !d_y || !d_out_x || !d_out_y)))
    return fail(h, CBM_ERR_INVALID_ARG, "device pointers must not be NULL");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  cudaStream_t st = (cudaStream_t)stream;
  const uint32_t nb = n_events / kGatherEvents + 1;
  const Scratch& scr = h->dev_scr;
  gather_size_kernel<<<nb, kSelThreads, 0, st>>>(d_off, h->p.L, n_events, (uint32_t)n_hits, d_event_ids, d_n_selected, scr.d_gsum);
  gather_base_kernel<<<nb, kSelThreads, 0, st>>>(d_off, h->p.L, n_events, (uint32_t)n_hits, d_event_ids, d_n_selected, scr.d_gsum, scr.d_hitbase,
                                                 d_out_off, d_out_n_hits);
  if (n_events)
    gather_copy_kernel<<<h->n_sm * 8, kSelThreads, 0, st>>>(d_x, d_y, d_off, h->p.L, n_events, (uint32_t)n_hits, d_event_ids, d_n_selected,
                                                            scr.d_hitbase, d_out_x, d_out_y, d_out_off, d_out_n_hits);
  CBM_CUDA(h, cudaGetLastError());
  return CBM_OK;
}

int cbm_trigger_filter_device(cbm_trigger_t* h, uint32_t n_events, uint64_t n_records, const int32_t* d_xyz,
                              const uint32_t* d_ev_off, int32_t* d_out_x, int32_t* d_out_y, uint32_t* d_out_off, void* stream) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (n_events > h->cfg.max_events) return fail(h, CBM_ERR_CAPACITY, "n_events %u > max_events %u", n_events, h->cfg.max_events);
  if (n_records > CBM_TRIGGER_MAX_INDEX) return fail(h, CBM_ERR_CAPACITY, "n_records must be <= 2^32 - 8192");
  if (!d_out_off || (n_events && (!d_ev_off || (n_records && (!d_xyz || !d_out_x || !d_out_y)))))
    return fail(h, CBM_ERR_INVALID_ARG, "device pointers must not be NULL");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  cudaStream_t st = (cudaStream_t)stream;
  const uint32_t L = h->p.L;
  if (n_events == 0) {
    CBM_CUDA(h, cudaMemsetAsync(d_out_off, 0, sizeof(uint32_t), st));
    return CBM_OK;
  }
  FilterDev fp;
  fp.L = L;
  for (uint32_t l = 0; l < (uint32_t)kMaxLayers; ++l) fp.z[l] = l < L ? h->p.z[l] : 0x7FFFFFFF;
  const Scratch& scr = h->dev_scr;
  const uint32_t n = n_events * L;  // < 2^32 (checked at create)
  const uint32_t nb = (n + kSelEvents - 1) / kSelEvents;
  uint32_t* const d_bsum = scr.d_fcnt + n;
  filter_count_kernel<<<n_events, kFilterThreads, 0, st>>>(fp, d_xyz, d_ev_off, n_events, (uint32_t)n_records, scr.d_fcnt);
  scan_sums_kernel<<<nb, kSelThreads, 0, st>>>(scr.d_fcnt, n, d_bsum);
  scan_write_kernel<<<nb, kSelThreads, 0, st>>>(scr.d_fcnt, n, d_bsum, d_out_off);
  filter_scatter_kernel<<<n_events, kFilterThreads, 0, st>>>(fp, d_xyz, d_ev_off, n_events, (uint32_t)n_records, d_out_off, d_out_x, d_out_y);
  CBM_CUDA(h, cudaGetLastError());
  return CBM_OK;
}

int cbm_trigger_build_events_device(cbm_trigger_t* h, uint64_t n_records, const int32_t* d_t, uint32_t t_gap, uint32_t* d_ev_off,
                                    uint32_t* n_events, void* stream) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (!n_events || !d_ev_off || (n_records && !d_t)) return fail(h, CBM_ERR_INVALID_ARG, "pointers must not be NULL");
  if (n_records > CBM_TRIGGER_MAX_INDEX) return fail(h, CBM_ERR_CAPACITY, "n_records must be <= 2^32 - 8192");
  cudaStream_t st = (cudaStream_t)stream;
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  *n_events = 0;
  if (n_records == 0) {
    CBM_CUDA(h, cudaMemsetAsync(d_ev_off, 0, sizeof(uint32_t), st));
    CBM_CUDA(h, cudaStreamSynchronize(st));
    return CBM_OK;
  }
  static_assert(kSelEvents <= 4096 && kFlagThreads <= 4096, "CBM_TRIGGER_MAX_INDEX leaves room for one block of 4096 and one of 4096");
  const uint32_t n = (uint32_t)n_records;                   // <= 2^32 - 8192: the sums below do not wrap
  const uint32_t nb = (n + kSelEvents - 1) / kSelEvents;
  // scratch of this call (stream-ordered allocation): the flags, the per-block counts of the compaction, the count
  uint8_t* d_flag = nullptr;
  uint32_t* d_cnt = nullptr;
  CBM_CUDA(h, cudaMallocAsync((void**)&d_flag, ((size_t)n + 15) & ~(size_t)15, st));
  cudaError_t e = cudaMallocAsync((void**)&d_cnt, ((size_t)nb + 2) * sizeof(uint32_t), st);
  if (e != cudaSuccess) { cudaFreeAsync(d_flag, st); return fail(h, CBM_ERR_CUDA, "cudaMallocAsync: %s", cudaGetErrorString(e)); }
  uint32_t* const d_n = d_cnt + nb + 1;
  event_flag_kernel<<<(n + kFlagThreads - 1) / kFlagThreads, kFlagThreads, 0, st>>>(d_t, n, t_gap, d_flag);
  select_count_kernel<<<nb, kSelThreads, 0, st>>>(d_flag, n, d_cnt);
  select_write_kernel<<<nb, kSelThreads, 0, st>>>(d_flag, n, d_cnt, d_ev_off, d_n);
  event_close_kernel<<<1, 1, 0, st>>>(d_ev_off, d_n, n);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(n_events, d_n, sizeof(uint32_t), cudaMemcpyDeviceToHost, st);
  cudaFreeAsync(d_flag, st);
  cudaFreeAsync(d_cnt, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail(h, CBM_ERR_CUDA, "event building: %s", cudaGetErrorString(e));
  return CBM_OK;
}

int cbm_trigger_msd_device(cbm_trigger_t* h, const cbm_trigger_msd_params_t* mp, uint32_t n_events, uint64_t n_hits,
                           const int32_t* d_x, const int32_t* d_y, const uint32_t* d_off, uint32_t* d_n_passing,
                           uint8_t* d_accept, void* stream) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (!mp || mp->struct_size != sizeof(cbm_trigger_msd_params_t)) return fail(h, CBM_ERR_INVALID_ARG, "msd params: NULL or bad struct_size");
  const uint32_t st = mp->station == 0xFFFFFFFFu ? h->p.S - 1 : mp->station;
  if (st >= h->p.S) return fail(h, CBM_ERR_INVALID_ARG, "msd params: station %u of %u", mp->station, h->p.S);
  if (mp->thr_x_den == 0 || mp->thr_x_den > 4096 || mp->thr_y_den == 0 || mp->thr_y_den > 4096 ||
      mp->thr_x_num > (1u << 20) || mp->thr_y_num > (1u << 20) || mp->ndf == 0 || mp->ndf > 16)
    return fail(h, CBM_ERR_INVALID_ARG, "msd params: need 0 < den <= 4096, num <= 2^20, 1 <= ndf <= 16");
  if (n_hits >= (1ull << 32)) return fail(h, CBM_ERR_CAPACITY, "n_hits must be < 2^32");
  if (n_events && (!d_off || !d_n_passing || !d_accept || (n_hits && (!d_x || !d_y))))
    return fail(h, CBM_ERR_INVALID_ARG, "device pointers must not be NULL");
  if (n_events == 0) return CBM_OK;
  MsdDev d;
  d.L = h->p.L; d.first_layer = 3 * st;
  d.z0 = h->p.z[3 * st]; d.z1 = h->p.z[3 * st + 1]; d.z2 = h->p.z[3 * st + 2];
  d.num_x = mp->thr_x_num; d.den_x = mp->thr_x_den; d.num_y = mp->thr_y_num; d.den_y = mp->thr_y_den;
  d.ndf = mp->ndf; d.min_triplets = mp->min_triplets;
  // delta = floor(sqrt(thr * ndf)) + 1 in 10-um units: every residual of a passing triplet is smaller
  auto delta = [&](uint32_t num, uint32_t den) {
    const long double v = (long double)num * 1000000.0L * (long double)mp->ndf / (long double)den;
    return (int64_t)std::floor(std::sqrt(v)) + 2;  // + 1 for the bound, + 1 against the rounding of sqrt
  };
  d.pre_x = delta(d.num_x, d.den_x) * ((int64_t)d.z0 + d.z1);
  d.pre_y = delta(d.num_y, d.den_y) * ((int64_t)d.z0 + d.z1);
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  constexpr uint32_t kMsdEventsPerCta = kMsdWarps * 32 / kMsdLanes;
  msd_kernel<<<(n_events + kMsdEventsPerCta - 1) / kMsdEventsPerCta, 32 * kMsdWarps, 0, (cudaStream_t)stream>>>(
      d, d_x, d_y, d_off, n_events, (uint32_t)n_hits, d_n_passing, d_accept);
  CBM_CUDA(h, cudaGetLastError());
  return CBM_OK;
}

int cbm_trigger_get_stats(cbm_trigger_t* h, uint32_t slot, cbm_trigger_stats_t* stats) {
  int rc = check_slot(h, slot);
  if (rc) return rc;
  if (!stats) return fail(h, CBM_ERR_INVALID_ARG, "stats must not be NULL");
  *stats = h->slot[slot].stats;
  stats->struct_size = sizeof(*stats);
  return CBM_OK;
}

int cbm_trigger_run_device(cbm_trigger_t* h, uint32_t n_events, uint64_t n_hits, const int32_t* d_x, const int32_t* d_y,
                           const uint32_t* d_off, uint32_t* d_n_triplets, uint32_t* d_n_candidates, uint8_t* d_accept,
                           void* stream) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (n_events > h->cfg.max_events) return fail(h, CBM_ERR_CAPACITY, "n_events %u > max_events %u", n_events, h->cfg.max_events);
  if (n_hits >= (1ull << 32)) return fail(h, CBM_ERR_CAPACITY, "n_hits must be < 2^32");
  if (n_events && (!d_off || !d_n_triplets || !d_n_candidates || !d_accept || (n_hits && (!d_x || !d_y))))
    return fail(h, CBM_ERR_INVALID_ARG, "device pointers must not be NULL");
  if (((uintptr_t)d_x | (uintptr_t)d_y) & 15) return fail(h, CBM_ERR_INVALID_ARG, "d_x and d_y must be 16-byte aligned");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  ProfEvents* pe = (h->cfg.flags & CBM_FLAG_PROFILE) ? &h->dev_prof[h->dev_prof_head % CBM_TRIGGER_PROFILE_RING] : nullptr;
  const int nl = launch_selection(h, h->dev_scr, d_x, d_y, d_off, n_events, n_hits, d_n_triplets, d_n_candidates,
                                  d_accept, (cudaStream_t)stream, pe);
  if (nl < 0) return nl;
  ++h->dev_prof_head;
  h->dev_n_events = n_events;
  h->dev_n_hits = n_hits;
  return CBM_OK;
}

int cbm_trigger_ubench(cbm_trigger_t* h, cbm_trigger_ubench_t* out) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (!out || out->struct_size != sizeof(cbm_trigger_ubench_t)) return fail(h, CBM_ERR_INVALID_ARG, "ubench: NULL or bad struct_size");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  const int grid = h->n_sm * kUbCtasPerSm;
  uint32_t* d_out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  // every exit, also a failing one, releases the buffer and the two events
  auto done = [&](cudaError_t e, const char* what) {
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(d_out);
    return e == cudaSuccess ? CBM_OK : fail(h, CBM_ERR_CUDA, "ubench: %s: %s", what, cudaGetErrorString(e));
  };
  cudaError_t err = cudaMalloc(&d_out, (size_t)grid * kUbThreads * sizeof(uint32_t));
  if (err != cudaSuccess) return done(err, "cudaMalloc");
  if ((err = cudaEventCreate(&e0)) != cudaSuccess || (err = cudaEventCreate(&e1)) != cudaSuccess) return done(err, "cudaEventCreate");
  const double lanes = (double)grid * kUbThreads * (double)kUbIter * 8.0;  // chain steps of one launch
  auto timed = [&](int which, double* per_s, double per_step) -> cudaError_t {
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {  // first repetition warms up
      cudaEventRecord(e0, h->st_run);
      switch (which) {
        case 0: ub_alu_kernel<<<grid, kUbThreads, 0, h->st_run>>>(d_out, 0x9E3779B9u, 0x7F4A7C15u); break;
        case 1: ub_imad_kernel<<<grid, kUbThreads, 0, h->st_run>>>(d_out, 1664525u, 1013904223u); break;
        case 2: ub_window_kernel<<<grid, kUbThreads, 0, h->st_run>>>(d_out, 70000, 123456789012ll, 84000000ull); break;
        default: ub_packed_kernel<<<grid, kUbThreads, 0, h->st_run>>>(d_out, 0x01230456u, 0xFE00FE00u); break;
      }
      cudaEventRecord(e1, h->st_run);
      cudaError_t e = cudaEventSynchronize(e1);
      if (e != cudaSuccess) return e;
      float ms = 0;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep && ms < best) best = ms;
    }
    *per_s = lanes * per_step / (best * 1e-3);
    return cudaGetLastError();
  };
  if ((err = timed(0, &out->alu_lane_ops_per_s, 2.0)) != cudaSuccess) return done(err, "alu kernel");        // IADD3 + LOP3
  if ((err = timed(1, &out->imad_lane_ops_per_s, 1.0)) != cudaSuccess) return done(err, "imad kernel");      // IMAD
  if ((err = timed(2, &out->window_evals_per_s, 1.0)) != cudaSuccess) return done(err, "window kernel");     // one evaluation = x and y
  if ((err = timed(3, &out->packed_tests_per_s, 1.0)) != cudaSuccess) return done(err, "packed kernel");
  out->n_sm = (uint32_t)h->n_sm;
  return done(cudaSuccess, "");
}

int cbm_trigger_device_status(cbm_trigger_t* h, void* stream, cbm_trigger_stats_t* stats) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (!stats) return fail(h, CBM_ERR_INVALID_ARG, "stats must not be NULL");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  CBM_CUDA(h, cudaMemcpyAsync(h->h_dev_ctrl, h->dev_scr.d_ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CBM_CUDA(h, cudaStreamSynchronize((cudaStream_t)stream));
  fill_stats(*stats, *h->h_dev_ctrl, h->dev_n_events, h->dev_n_hits, h->dev_n_events ? CBM_TRIGGER_N_KERNELS : 0);
  if ((h->cfg.flags & CBM_FLAG_PROFILE) && h->dev_prof_head)
    fill_prof(*stats, h->dev_prof[(h->dev_prof_head - 1) % CBM_TRIGGER_PROFILE_RING], false);
  if (stats->n_invalid)
    return fail(h, CBM_ERR_RANGE, "%u event(s) rejected on the device; first: event %u", stats->n_invalid, stats->first_invalid);
  return CBM_OK;
}

int cbm_trigger_device_kernel_times(cbm_trigger_t* h, void* stream, uint32_t n_last, float* kernel_ms) {
  if (!h) return CBM_ERR_INVALID_ARG;
  if (!kernel_ms) return fail(h, CBM_ERR_INVALID_ARG, "kernel_ms must not be NULL");
  if (!(h->cfg.flags & CBM_FLAG_PROFILE)) return fail(h, CBM_ERR_STATE, "the handle was created without CBM_FLAG_PROFILE");
  CBM_CUDA(h, cudaSetDevice(h->cfg.device));
  CBM_CUDA(h, cudaStreamSynchronize((cudaStream_t)stream));
  uint32_t n = n_last;
  if (n > CBM_TRIGGER_PROFILE_RING) n = CBM_TRIGGER_PROFILE_RING;
  if (n > h->dev_prof_head) n = h->dev_prof_head;
  for (uint32_t i = 0; i < n; ++i) {
    ProfEvents& pe = h->dev_prof[(h->dev_prof_head - n + i) % CBM_TRIGGER_PROFILE_RING];
    for (int k = 0; k < CBM_TRIGGER_N_KERNELS; ++k) {
      float ms = 0;
      if (pe.valid) CBM_CUDA(h, cudaEventElapsedTime(&ms, pe.k[2 * k], pe.k[2 * k + 1]));
      kernel_ms[i * CBM_TRIGGER_N_KERNELS + k] = ms;
    }
  }
  return (int)n;
}

}  // extern "C"

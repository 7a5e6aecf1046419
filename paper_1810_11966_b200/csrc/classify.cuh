// classify.cuh -- a3: one pass over off[] decides every event's class and fills the
// class lists, so that the tile kernel (tiny events) and the team kernels (M, H, G) can start together.
//
// One warp = one tile of 32 consecutive events (lane <-> event), the same tile the tile kernel works on: the
// admission of tiny events to a tile's staging buffer depends on the tile's other events, and both kernels
// take that decision with the same function (tile_admit).
#pragma once
#include "ptx.cuh"

namespace cbm {

constexpr int kClassifyWarps = 8;  // tiles per CTA

// Per-lane facts of event `lane` of a tile -> is it finished by the tile kernel?  (all 32 lanes must call)
// Tiny events are admitted to the tile's staging buffer in order while their sizes (+ alignment slack) fit.
__device__ __forceinline__ bool tile_admit(const Params& p, uint32_t lane, bool in, bool invalid, uint32_t mx, uint32_t tot) {
  bool tiny = in && !invalid && p.tiny_max_total != 0 && mx <= p.tiny_max_layer && tot <= p.tiny_max_total;
  uint32_t need = tiny ? tot + kTinySlack : 0u;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, need, d);
    if (lane >= (uint32_t)d) need += v;
  }
  return tiny && need <= kTileHitCap;
}

// Structural check of one event (B1): offsets monotone and within n_hits, no layer above max_hits_per_layer.
// Returns the fullest layer, 0xFFFFFFFF for an invalid event.  o points at the event's L + 1 offsets.
template <class Ld>
__device__ __forceinline__ uint32_t event_max_layer(Ld&& ld, uint32_t L, uint32_t n_hits, uint32_t cap) {
  uint32_t prev = ld(0), mx = 0;
  bool valid = true;
  for (uint32_t l = 1; l <= L; ++l) {
    const uint32_t o = ld(l);
    valid &= prev <= o;
    mx = max(mx, o - prev);
    prev = o;
  }
  valid &= prev <= n_hits;
  return (valid && mx <= cap) ? mx : 0xFFFFFFFFu;
}

__global__ void __launch_bounds__(32 * kClassifyWarps)
    classify_kernel(const __grid_constant__ Params p, const uint32_t* __restrict__ off, uint32_t n_events, uint32_t n_hits,
                    uint32_t* __restrict__ n_triplets, uint32_t* __restrict__ n_candidates, uint8_t* __restrict__ accept,
                    Ctrl* __restrict__ ctrl, uint32_t* __restrict__ list_M, uint32_t* __restrict__ list_H,
                    uint32_t* __restrict__ list_G) {
  __shared__ uint32_t so[kClassifyWarps * kTileEvents * kMaxLayers + 1];
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t L = p.L, S = p.S;
  const uint32_t e_cta = blockIdx.x * (kClassifyWarps * kTileEvents);
  const uint32_t ne_cta = min((uint32_t)(kClassifyWarps * kTileEvents), n_events - e_cta);
  {  // the CTA's offsets, read once, coalesced
    const uint32_t n_off = ne_cta * L + 1;
    const uint32_t* src = off + (size_t)e_cta * L;
    for (uint32_t i = tid; i < n_off; i += blockDim.x) so[i] = __ldg(src + i);
  }
  __syncthreads();
  const uint32_t el = warp * kTileEvents + lane;  // event within the CTA
  const bool in = el < ne_cta;
  const uint32_t e = e_cta + el;
  uint32_t mx = 0, tot = 0;
  if (in) {
    const uint32_t* o = &so[el * L];
    mx = event_max_layer([&](uint32_t l) { return o[l]; }, L, n_hits, p.max_hits_per_layer);
    tot = o[L] - o[0];
  }
  const bool invalid = in && mx == 0xFFFFFFFFu;
  const bool tiny = tile_admit(p, lane, in, invalid, mx, tot);
  int cls = -1;
  if (in && !invalid && !tiny) cls = mx <= p.cls_max[kClsM] ? kClsM : (mx <= p.cls_max[kClsH] ? kClsH : kClsG);
  // List positions: counts per warp and class -> one atomicAdd per class and CTA -> every lane's slot.  The order
  // inside a list is irrelevant: results are indexed by event, one writer per address.
  __shared__ uint32_t wcnt[kClassifyWarps][kNumTeamClasses + 1];  // [warp][class], [3] = tiny
  __shared__ uint32_t cbase[kNumTeamClasses];
  uint32_t bal[kNumTeamClasses];
#pragma unroll
  for (int c = 0; c < kNumTeamClasses; ++c) bal[c] = __ballot_sync(FULL, cls == c);
  const uint32_t tm = __ballot_sync(FULL, tiny);
  if (lane == 0) {
#pragma unroll
    for (int c = 0; c < kNumTeamClasses; ++c) wcnt[warp][c] = __popc(bal[c]);
    wcnt[warp][kNumTeamClasses] = __popc(tm);
  }
  __syncthreads();
  if (tid <= kNumTeamClasses) {
    uint32_t tot = 0;
    for (int w = 0; w < kClassifyWarps; ++w) tot += wcnt[w][tid];
    if (tid < kNumTeamClasses) cbase[tid] = tot ? atomicAdd(&ctrl->count[tid], tot) : 0u;
    else if (tot) atomicAdd(&ctrl->n_tiny, tot);
  }
  __syncthreads();
  if (cls >= 0) {
    const uint32_t mine = cls == kClsM ? bal[kClsM] : (cls == kClsH ? bal[kClsH] : bal[kClsG]);
    uint32_t pos = cbase[cls] + __popc(mine & lanemask_lt());
    for (uint32_t w = 0; w < warp; ++w) pos += wcnt[w][cls];
    (cls == kClsM ? list_M : (cls == kClsH ? list_H : list_G))[pos] = e;
  }
  if (invalid) {  // rejected on the device: outputs 0, reported by fetch_results / device_status
    for (uint32_t k = 0; k < S; ++k) n_triplets[(size_t)e * S + k] = 0;
    n_candidates[e] = 0;
    accept[e] = 0;
    atomicAdd(&ctrl->n_invalid, 1u);
    atomicMax(&ctrl->first_invalid_inv, ~e);
  }
}

}  // namespace cbm

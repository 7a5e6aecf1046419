// filter.cuh -- the input filter of the paper's implementation "i3": out of the full-setup hit
// data of every event (about 5000 records x, y, z per event) only the hits of the layers the
// selection works on are kept, "such that only hit data in the trigger station are transferred".  Here: on the
// device, for a stream that already lies there; the output is the CSR-SoA batch of include/cbm_trigger.h.
//
// A record belongs to layer l iff its z equals layer_z[l] (z is a per-layer constant, reading R6).  The
// kept hits of an event are grouped by layer in stream order (stable), so the output is unique:
//   filter_count_kernel    one CTA per event: hits per layer -> cnt[e*L + l]
//   scan (two kernels)     exclusive prefix of cnt -> off[E*L + 1]   (per-block sums, then every block adds the
//                          sums of the blocks before it: no atomics, no spin between CTAs)
//   filter_scatter_kernel  one CTA per event, chunk by chunk in stream order: rank of a hit among the earlier hits
//                          of its layer (match.any + popc inside a warp, per-warp counts across the CTA, running
//                          count across chunks) -> x, y at off[e*L + l] + rank
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "select.cuh"

namespace cbm {

constexpr int kFilterThreads = 256;
constexpr int kFilterWarps = kFilterThreads / 32;

struct FilterDev {
  uint32_t L;
  int32_t z[kMaxLayers];  // strictly increasing
};

// layer of a record's z, or -1 (binary search over the increasing layer z)
__device__ __forceinline__ int filter_layer_of(const int32_t* sz, uint32_t L, int32_t z) {
  uint32_t lo = 0, hi = L;
  while (lo < hi) {
    const uint32_t mid = (lo + hi) >> 1;
    if (sz[mid] < z) lo = mid + 1; else hi = mid;
  }
  return (lo < L && sz[lo] == z) ? (int)lo : -1;
}

__global__ void __launch_bounds__(kFilterThreads)
    filter_count_kernel(const FilterDev p, const int32_t* __restrict__ xyz, const uint32_t* __restrict__ ev_off, uint32_t n_events,
                        uint32_t n_records, uint32_t* __restrict__ cnt) {
  __shared__ int32_t sz[kMaxLayers];
  __shared__ uint32_t c[kMaxLayers];
  if (threadIdx.x < kMaxLayers) { sz[threadIdx.x] = threadIdx.x < p.L ? p.z[threadIdx.x] : 0x7FFFFFFF; c[threadIdx.x] = 0; }
  __syncthreads();
  const uint32_t e = blockIdx.x;
  uint32_t a = __ldg(ev_off + e), b = __ldg(ev_off + e + 1);
  if (a > b || b > n_records) a = b = 0;  // a malformed event keeps nothing
  for (uint32_t i = a + threadIdx.x; i < b; i += kFilterThreads) {
    const int l = filter_layer_of(sz, p.L, __ldg(xyz + 3 * (size_t)i + 2));
    if (l >= 0) atomicAdd(&c[l], 1u);
  }
  __syncthreads();
  if (threadIdx.x < p.L) cnt[(size_t)e * p.L + threadIdx.x] = c[threadIdx.x];
}

// exclusive scan of v[n] into out[n + 1] (out[n] = total): per-block sums, then the bases
__global__ void __launch_bounds__(kSelThreads)
    scan_sums_kernel(const uint32_t* __restrict__ v, uint32_t n, uint32_t* __restrict__ block_sum) {
  __shared__ uint32_t warp_sums[kSelThreads / 32];
  const uint32_t first = (blockIdx.x * kSelThreads + threadIdx.x) * kSelPerThread;
  uint32_t s = 0;
  for (uint32_t i = first; i < min(first + kSelPerThread, n); ++i) s += __ldg(v + i);
  uint32_t total;
  sel_block_exclusive_scan(s, warp_sums, &total);
  if (threadIdx.x == 0) block_sum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kSelThreads)
    scan_write_kernel(const uint32_t* __restrict__ v, uint32_t n, const uint32_t* __restrict__ block_sum, uint32_t* __restrict__ out) {
  __shared__ uint32_t warp_sums[kSelThreads / 32];
  __shared__ uint32_t base_sh;
  uint32_t part = 0;
  for (uint32_t b = threadIdx.x; b < blockIdx.x; b += kSelThreads) part += block_sum[b];
  uint32_t before;
  sel_block_exclusive_scan(part, warp_sums, &before);
  if (threadIdx.x == 0) base_sh = before;
  __syncthreads();
  const uint32_t first = (blockIdx.x * kSelThreads + threadIdx.x) * kSelPerThread;
  uint32_t val[kSelPerThread], s = 0;
#pragma unroll
  for (int k = 0; k < kSelPerThread; ++k) {
    val[k] = first + k < n ? __ldg(v + first + k) : 0u;
    s += val[k];
  }
  uint32_t total;
  uint32_t pos = base_sh + sel_block_exclusive_scan(s, warp_sums, &total);
#pragma unroll
  for (int k = 0; k < kSelPerThread; ++k) {
    if (first + k < n) out[first + k] = pos;
    pos += val[k];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) out[n] = base_sh + total;
}

__global__ void __launch_bounds__(kFilterThreads)
    filter_scatter_kernel(const FilterDev p, const int32_t* __restrict__ xyz, const uint32_t* __restrict__ ev_off, uint32_t n_events,
                          uint32_t n_records, const uint32_t* __restrict__ off, int32_t* __restrict__ out_x, int32_t* __restrict__ out_y) {
  __shared__ int32_t sz[kMaxLayers];
  __shared__ uint32_t run[kMaxLayers];                 // hits of every layer in the chunks before this one
  __shared__ uint32_t wc[kFilterWarps][kMaxLayers];    // hits of every layer in this chunk, per warp
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t e = blockIdx.x;
  if (threadIdx.x < kMaxLayers) {
    sz[threadIdx.x] = threadIdx.x < p.L ? p.z[threadIdx.x] : 0x7FFFFFFF;
    run[threadIdx.x] = threadIdx.x < p.L ? __ldg(off + (size_t)e * p.L + threadIdx.x) : 0u;
  }
  uint32_t a = __ldg(ev_off + e), b = __ldg(ev_off + e + 1);
  if (a > b || b > n_records) a = b = 0;
  for (uint32_t c0 = a; c0 < b; c0 += kFilterThreads) {  // chunks in stream order
    for (uint32_t i = threadIdx.x; i < kFilterWarps * kMaxLayers; i += kFilterThreads) (&wc[0][0])[i] = 0;
    __syncthreads();
    const uint32_t i = c0 + threadIdx.x;
    int l = -1;
    int32_t hx = 0, hy = 0;
    if (i < b) {
      const int32_t* r = xyz + 3 * (size_t)i;
      hx = __ldg(r); hy = __ldg(r + 1);
      l = filter_layer_of(sz, p.L, __ldg(r + 2));
    }
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, l);  // lanes of this warp with the same layer (or all dropped ones)
    const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
    if (l >= 0 && rank == 0) wc[warp][l] = __popc(peers);
    __syncthreads();
    if (l >= 0) {
      uint32_t pos = run[l] + rank;
      for (uint32_t w = 0; w < warp; ++w) pos += wc[w][l];
      out_x[pos] = hx;
      out_y[pos] = hy;
    }
    __syncthreads();
    if (threadIdx.x < p.L) {
      uint32_t t = 0;
      for (uint32_t w = 0; w < kFilterWarps; ++w) t += wc[w][threadIdx.x];
      run[threadIdx.x] += t;
    }
    // the next chunk's zeroing of wc comes after the barrier at the loop top... it is separated from these reads by
    // the barrier below
    __syncthreads();
  }
}

}  // namespace cbm

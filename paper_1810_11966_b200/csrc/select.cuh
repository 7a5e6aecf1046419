// select.cuh -- the list of selected events ("the list of selected events is transferred back").
//
// Order-preserving stream compaction of accept[] into ascending event ids, without atomics, so the list is
// the same on every run: select_count_kernel counts the accepted events of every block of kSelEvents events,
// select_write_kernel sums the counts of the blocks before its own and writes its ids at that base.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cbm {

constexpr int kSelThreads = 256;
constexpr int kSelPerThread = 16;                          // one 128-bit load of accept bytes per thread
constexpr int kSelEvents = kSelThreads * kSelPerThread;    // events per block

// number of non-zero bytes among the (up to) 16 accept bytes of this thread; also returns them as a bit mask
__device__ __forceinline__ uint32_t sel_load_mask(const uint8_t* __restrict__ accept, uint32_t n, uint32_t first) {
  uint32_t mask = 0;
  if (first + kSelPerThread <= n && ((reinterpret_cast<uintptr_t>(accept) + first) & 15) == 0) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(accept + first));
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int b = 0; b < 4; ++b) mask |= ((w[i] >> (8 * b)) & 0xFFu) ? (1u << (4 * i + b)) : 0u;
  } else {
    for (uint32_t i = 0; i < (uint32_t)kSelPerThread && first + i < n; ++i) mask |= accept[first + i] ? (1u << i) : 0u;
  }
  return mask;
}

__device__ __forceinline__ uint32_t sel_block_exclusive_scan(uint32_t v, uint32_t* warp_sums, uint32_t* total) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= (uint32_t)d) incl += u;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < kSelThreads / 32; ++w) {
    const uint32_t s = warp_sums[w];
    base += (uint32_t)w < warp ? s : 0u;
    tot += s;
  }
  *total = tot;
  return base + incl - v;
}

// the same for 64-bit values (hit totals of the gather: a list may name large events many times)
__device__ __forceinline__ unsigned long long sel_block_exclusive_scan64(unsigned long long v, unsigned long long* warp_sums,
                                                                         unsigned long long* total) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned long long incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const unsigned long long u = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= (uint32_t)d) incl += u;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  unsigned long long base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < kSelThreads / 32; ++w) {
    const unsigned long long s = warp_sums[w];
    base += (uint32_t)w < warp ? s : 0ull;
    tot += s;
  }
  *total = tot;
  return base + incl - v;
}

__global__ void __launch_bounds__(kSelThreads)
    select_count_kernel(const uint8_t* __restrict__ accept, uint32_t n_events, uint32_t* __restrict__ block_count) {
  __shared__ uint32_t warp_sums[kSelThreads / 32];
  const uint32_t first = (blockIdx.x * kSelThreads + threadIdx.x) * kSelPerThread;
  const uint32_t c = first < n_events ? (uint32_t)__popc(sel_load_mask(accept, n_events, first)) : 0u;
  uint32_t total;
  sel_block_exclusive_scan(c, warp_sums, &total);
  if (threadIdx.x == 0) block_count[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kSelThreads)
    select_write_kernel(const uint8_t* __restrict__ accept, uint32_t n_events, const uint32_t* __restrict__ block_count,
                        uint32_t* __restrict__ selected, uint32_t* __restrict__ n_selected) {
  __shared__ uint32_t warp_sums[kSelThreads / 32];
  __shared__ uint32_t base_sh;
  // accepted events in the blocks before this one
  uint32_t part = 0;
  for (uint32_t b = threadIdx.x; b < blockIdx.x; b += kSelThreads) part += block_count[b];
  uint32_t before;
  sel_block_exclusive_scan(part, warp_sums, &before);
  if (threadIdx.x == 0) base_sh = before;
  __syncthreads();  // warp_sums is reused below
  const uint32_t first = (blockIdx.x * kSelThreads + threadIdx.x) * kSelPerThread;
  uint32_t mask = first < n_events ? sel_load_mask(accept, n_events, first) : 0u;
  uint32_t total;
  uint32_t pos = base_sh + sel_block_exclusive_scan((uint32_t)__popc(mask), warp_sums, &total);
  while (mask) {
    const uint32_t i = (uint32_t)__ffs(mask) - 1u;
    selected[pos++] = first + i;
    mask &= mask - 1u;
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) *n_selected = base_sh + total;
}

// ---------------------------------------------------------------------------------------------- gather
// The hits of the selected events as a compact batch of the same layout (what the
// next trigger level, full track reconstruction, reads).  Three steps, no atomics, so the
// output is unique: sizes of the selected events and their per-block sums; exclusive prefix of the sizes (every
// block adds the sums of the blocks before it); one CTA per selected event copies its hits and writes its
// offsets rebased to the new batch.
constexpr int kGatherPerThread = 16;
constexpr int kGatherEvents = kSelThreads * kGatherPerThread;

// Hits of selected event e; 0 for an id beyond the batch or an event whose offsets are not non-decreasing inside
// [0, n_hits] (caller-supplied ids and offsets are not trusted: such an event is gathered as empty).
__device__ __forceinline__ uint32_t gather_event_size(const uint32_t* __restrict__ off, uint32_t L, uint32_t e, uint32_t n_events,
                                                      uint32_t n_hits) {
  if (e >= n_events) return 0u;
  const uint32_t* o = off + (size_t)e * L;
  const uint32_t src = __ldg(o);
  uint32_t prev = src;
  bool ok = true;
  for (uint32_t l = 1; l <= L; ++l) {
    const uint32_t v = __ldg(o + l);
    ok &= prev <= v;
    prev = v;
  }
  return (ok && prev <= n_hits) ? prev - src : 0u;
}

// Sizes are summed in 64 bits: one event holds < 2^32 hits, a list of up to n_events < 2^32 entries that repeats large
// events can name 2^32 hits and more, and a wrapped total would pass the "fits the output" test of gather_copy_kernel.
__global__ void __launch_bounds__(kSelThreads)
    gather_size_kernel(const uint32_t* __restrict__ off, uint32_t L, uint32_t n_events, uint32_t n_hits,
                       const uint32_t* __restrict__ ids, const uint32_t* __restrict__ n_selected,
                       unsigned long long* __restrict__ block_sum) {
  __shared__ unsigned long long warp_sums[kSelThreads / 32];
  const uint32_t n = min(*n_selected, n_events);
  const uint64_t first = ((uint64_t)blockIdx.x * kSelThreads + threadIdx.x) * kGatherPerThread;
  unsigned long long sum = 0;
  for (uint64_t i = first; i < min(first + kGatherPerThread, (uint64_t)n); ++i) sum += gather_event_size(off, L, __ldg(ids + i), n_events, n_hits);
  unsigned long long total;
  sel_block_exclusive_scan64(sum, warp_sums, &total);
  if (threadIdx.x == 0) block_sum[blockIdx.x] = total;
}

// hit_base[i] = first hit of list entry i in the gathered batch; only meaningful (and only used) when the total fits
// n_hits < 2^32, so the low 32 bits are kept.  The offset table is closed only in that case; the 64-bit total is
// always reported.
__global__ void __launch_bounds__(kSelThreads)
    gather_base_kernel(const uint32_t* __restrict__ off, uint32_t L, uint32_t n_events, uint32_t n_hits,
                       const uint32_t* __restrict__ ids, const uint32_t* __restrict__ n_selected,
                       const unsigned long long* __restrict__ block_sum, uint32_t* __restrict__ hit_base, uint32_t* __restrict__ out_off,
                       unsigned long long* __restrict__ out_n_hits) {
  __shared__ unsigned long long warp_sums[kSelThreads / 32];
  __shared__ unsigned long long base_sh;
  const uint32_t n = min(*n_selected, n_events);
  unsigned long long part = 0;
  for (uint32_t b = threadIdx.x; b < blockIdx.x; b += kSelThreads) part += block_sum[b];
  unsigned long long before;
  sel_block_exclusive_scan64(part, warp_sums, &before);
  if (threadIdx.x == 0) base_sh = before;
  __syncthreads();
  const uint64_t first = ((uint64_t)blockIdx.x * kSelThreads + threadIdx.x) * kGatherPerThread;
  uint32_t sz[kGatherPerThread];
  unsigned long long sum = 0;
#pragma unroll
  for (int k = 0; k < kGatherPerThread; ++k) {
    sz[k] = first + k < n ? gather_event_size(off, L, __ldg(ids + first + k), n_events, n_hits) : 0u;
    sum += sz[k];
  }
  unsigned long long total;
  unsigned long long pos = base_sh + sel_block_exclusive_scan64(sum, warp_sums, &total);
#pragma unroll
  for (int k = 0; k < kGatherPerThread; ++k) {
    if (first + k < n) hit_base[first + k] = (uint32_t)pos;
    pos += sz[k];
  }
  // the block holding the end of the list reports the number of hits and, if they fit, closes the offset table
  const uint32_t last_block = n ? (n - 1) / kGatherEvents : 0u;
  if (blockIdx.x == last_block && threadIdx.x == 0) {
    const unsigned long long all = base_sh + total;
    if (all <= n_hits) out_off[(size_t)n * L] = (uint32_t)all;
    *out_n_hits = all;
  }
}

// one CTA per selected event (grid-stride)
__global__ void __launch_bounds__(kSelThreads)
    gather_copy_kernel(const int32_t* __restrict__ x, const int32_t* __restrict__ y, const uint32_t* __restrict__ off,
                       uint32_t L, uint32_t n_events, uint32_t n_hits, const uint32_t* __restrict__ ids,
                       const uint32_t* __restrict__ n_selected, const uint32_t* __restrict__ hit_base, int32_t* __restrict__ out_x,
                       int32_t* __restrict__ out_y, uint32_t* __restrict__ out_off, const unsigned long long* __restrict__ out_n_hits) {
  const uint32_t n = min(*n_selected, n_events);
  // a list that names an event more than once can gather more than the n_hits the output arrays hold: then nothing
  // is copied (gather_base_kernel has reported the 64-bit total, which tells the caller)
  if (*out_n_hits > n_hits) return;
  for (uint32_t i = blockIdx.x; i < n; i += gridDim.x) {
    const uint32_t e = __ldg(ids + i), dst = hit_base[i];
    const uint32_t size = gather_event_size(off, L, e, n_events, n_hits);  // 0: empty, or not a well-formed event
    const uint32_t src = size ? __ldg(off + (size_t)e * L) : 0u;
    for (uint32_t l = threadIdx.x; l < L; l += kSelThreads)
      out_off[(size_t)i * L + l] = dst + (size ? __ldg(off + (size_t)e * L + l) - src : 0u);
    for (uint32_t k = threadIdx.x; k < size; k += kSelThreads) {
      out_x[dst + k] = __ldg(x + src + k);
      out_y[dst + k] = __ldg(y + src + k);
    }
  }
}

}  // namespace cbm

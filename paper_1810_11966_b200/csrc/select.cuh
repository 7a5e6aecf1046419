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

}  // namespace cbm

// timeslice.cuh -- event building from a free-streaming, time-stamped hit stream (section 8: the data
// acquisition "will deliver free-streaming data not associated to single event by a hardware trigger ... the time
// measurement of each hit must be considered"; the rule is DESIGN.md reading B9).
//
// The records of a timeslice come in stream order, record i with the integer time stamp t[i].  Record i opens a new
// event iff i == 0 or t[i] - t[i-1] > t_gap (64-bit difference: exact for any int32 stamps); an event is a maximal run
// of records without such a gap.  event_flag_kernel writes the flags, the order-preserving compaction of select.cuh
// turns them into the ascending record indices of the event starts (= ev_off[0 .. n_events)), and event_close_kernel
// appends ev_off[n_events] = n_records.  No atomics: the output is unique.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cbm {

constexpr int kFlagThreads = 256;

__global__ void __launch_bounds__(kFlagThreads)
    event_flag_kernel(const int32_t* __restrict__ t, uint32_t n_records, uint32_t t_gap, uint8_t* __restrict__ flag) {
  const uint32_t i = blockIdx.x * kFlagThreads + threadIdx.x;
  if (i >= n_records) return;
  flag[i] = (i == 0 || (long long)__ldg(t + i) - (long long)__ldg(t + i - 1) > (long long)t_gap) ? 1 : 0;
}

__global__ void event_close_kernel(uint32_t* __restrict__ ev_off, const uint32_t* __restrict__ n_events, uint32_t n_records) {
  ev_off[*n_events] = n_records;
}

}  // namespace cbm

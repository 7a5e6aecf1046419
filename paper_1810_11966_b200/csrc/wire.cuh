// wire.cuh -- the packed wire format XY20 (the paper's biggest
// single win was shrinking the host-to-device transfer).
//
// 5 bytes per hit instead of 8: bits 0..19 = x, bits 20..39 = y, both 20-bit two's complement (10-um units:
// +-5.24 m), little endian, hits in the order of x[] / y[].  The batch crosses PCIe packed and is expanded to
// the int32 arrays the selection kernels read by unpack_xy20_kernel: 13 bytes of HBM traffic per hit instead
// of 3 more bytes over the link.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cbm {

constexpr int kWireThreads = 256;

__device__ __forceinline__ int32_t sext20(uint32_t v) { return (int32_t)(v << 12) >> 12; }

// Thread t expands hits 4t .. 4t+3 = bytes 20t .. 20t+19 = words 5t .. 5t+4 of the packed stream.
// `packed` is 4-byte aligned and readable up to the next multiple of 20 bytes; x, y are 16-byte aligned and
// writable up to the next multiple of 4 hits (the slot buffers are padded).
__global__ void __launch_bounds__(kWireThreads)
    unpack_xy20_kernel(const uint32_t* __restrict__ packed, uint64_t n_hits, int32_t* __restrict__ x, int32_t* __restrict__ y) {
  const uint64_t t = (uint64_t)blockIdx.x * kWireThreads + threadIdx.x;
  if (4 * t >= n_hits) return;
  const uint32_t* w = packed + 5 * t;
  const uint32_t w0 = __ldg(w), w1 = __ldg(w + 1), w2 = __ldg(w + 2), w3 = __ldg(w + 3), w4 = __ldg(w + 4);
  // hit k occupies bits 40k .. 40k+39 of the 160-bit group
  int4 vx, vy;
  vx.x = sext20(w0 & 0xFFFFFu);
  vy.x = sext20((w0 >> 20) | ((w1 & 0xFFu) << 12));
  vx.y = sext20((w1 >> 8) & 0xFFFFFu);
  vy.y = sext20((w1 >> 28) | ((w2 & 0xFFFFu) << 4));
  vx.z = sext20((w2 >> 16) | ((w3 & 0xFu) << 16));
  vy.z = sext20((w3 >> 4) & 0xFFFFFu);
  vx.w = sext20((w3 >> 24) | ((w4 & 0xFFFu) << 8));
  vy.w = sext20(w4 >> 12);
  *reinterpret_cast<int4*>(x + 4 * t) = vx;
  *reinterpret_cast<int4*>(y + 4 * t) = vy;
}

}  // namespace cbm

// ubench.cuh -- micro-benchmarks behind cbm_trigger_ubench(): the integer-pipe denominators of the roofline
// ("R_int = INT32 lane-ops/s measured on the box").  Every kernel keeps 8 independent
// dependency chains per thread, so that with 8 warps per scheduler the pipe, not latency, is what is measured.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cbm {

constexpr int kUbThreads = 256, kUbCtasPerSm = 8, kUbIter = 4096;

// ALU pipe: IADD3 + LOP3 per chain and iteration (the compiler must not fold them: operands come from memory)
__global__ void __launch_bounds__(kUbThreads) ub_alu_kernel(uint32_t* out, uint32_t c, uint32_t d) {
  uint32_t a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = threadIdx.x * 8u + i;
#pragma unroll 1
  for (int it = 0; it < kUbIter; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = (a[i] + c) ^ (d + it);
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// FMA pipe: IMAD (32-bit multiply-add) per chain and iteration
__global__ void __launch_bounds__(kUbThreads) ub_imad_kernel(uint32_t* out, uint32_t m, uint32_t c) {
  uint32_t a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = threadIdx.x * 8u + i;
#pragma unroll 1
  for (int it = 0; it < kUbIter; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = a[i] * m + c;
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// The window evaluation itself, as the kernels compile it: (uint64)(a*z + Q) <= 2T in x and in y
// (IMAD.WIDE + 64-bit unsigned compare, twice), 8 independent evaluations per iteration.
__global__ void __launch_bounds__(kUbThreads) ub_window_kernel(uint32_t* out, int32_t z, long long q, unsigned long long t2) {
  int32_t xs[8], ys[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { xs[i] = (int32_t)(threadIdx.x * 8u + i); ys[i] = xs[i] ^ 0x5555; }
  uint32_t cnt = 0;
#pragma unroll 1
  for (int it = 0; it < kUbIter; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool ok = ((unsigned long long)((long long)xs[i] * z + q) <= t2) & ((unsigned long long)((long long)ys[i] * z + q) <= t2);
      cnt += ok ? 1u : 0u;
      xs[i] += it;          // new operands every iteration (not counted: 2 IADD per evaluation)
      ys[i] -= it;
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = cnt;
}

// The packed key test: ((A - P) & mask) == 0 for both projections at once (IADD + LOP3), 8 per iteration
__global__ void __launch_bounds__(kUbThreads) ub_packed_kernel(uint32_t* out, uint32_t a1, uint32_t mask) {
  uint32_t ps[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) ps[i] = threadIdx.x * 8u + i;
  uint32_t cnt = 0;
#pragma unroll 1
  for (int it = 0; it < kUbIter; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      cnt += (((a1 - ps[i]) & mask) == 0) ? 1u : 0u;
      ps[i] += 0x10001u * it;  // new operand (not counted)
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = cnt;
}

}  // namespace cbm

// ptx.cuh -- small PTX helpers shared by the kernels: mbarrier, 1-D TMA bulk copy, explicit shared-memory
// accesses, the exact window test.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "params.h"

namespace cbm {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// Shared-memory loads by 32-bit shared address (+ compile-time byte offset): the hot loops keep one address
// register and step it, instead of re-deriving generic addresses.
template <int OFS = 0>
__device__ __forceinline__ int32_t lds_s32(uint32_t addr) {
  int32_t v;
  asm volatile("ld.shared.s32 %0, [%1+%2];" : "=r"(v) : "r"(addr), "n"(OFS));
  return v;
}
// shared-memory atomics issued as plain ATOMS / RED (the compiler must not wrap them in its own warp aggregation)
__device__ __forceinline__ uint32_t atoms_add(uint32_t* addr, uint32_t v) {
  uint32_t old;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(smem_u32(addr)), "r"(v) : "memory");
  return old;
}
__device__ __forceinline__ void reds_or(uint32_t* addr, uint32_t v) {
  asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(smem_u32(addr)), "r"(v) : "memory");
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
// dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---------------------------------------------------------------------------------------------- window test
// The exact int64 inequality (PAPER.md:75-76 with the north_star's window, R4):
//   |a*z_o - b*z_a| <= T   <=>   (uint64)(a*z_o + (T - b*z_a)) <= 2*T
// P = a*z_other + T (hoisted per anchor hit);  pass  <=>  |a*z_other - b*z_a| <= T
__device__ __forceinline__ bool win(int64_t P, int32_t b, int32_t za, uint64_t T2) {
  return (uint64_t)(P - (int64_t)b * (int64_t)za) <= T2;
}
// anchor side hoisted: Q = T - b*z_a (int64), pass <=> (uint64)(a*z_o + Q) <= 2T
__device__ __forceinline__ int64_t anchor_q(int32_t b, int32_t neg_za, int64_t T) { return (int64_t)b * neg_za + T; }
__device__ __forceinline__ bool win_q(int32_t a, int32_t zo, int64_t Q, uint64_t T2) {
  return (uint64_t)((int64_t)a * zo + Q) <= T2;
}
__device__ __forceinline__ uint32_t sat32(unsigned long long v) { return v > (unsigned long long)kSat ? kSat : (uint32_t)v; }

__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// packed slope key of a hit: (key_x mod 2^16) | (key_y mod 2^16) << 16   (SASS: 2 IMAD.HI + PRMT)
__device__ __forceinline__ uint32_t packed_key(int32_t x, int32_t y, int32_t M) {
  return __byte_perm((uint32_t)__mulhi(x, M), (uint32_t)__mulhi(y, M), 0x5410);
}

}  // namespace cbm

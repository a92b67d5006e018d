// tma.cuh -- the PTX this library uses for TMA (cp.async.bulk.tensor) and mbarriers on sm_100a:
// thin wrappers, the ISA's own spellings.
#pragma once
#include <cuda.h>

namespace gk {

__device__ __forceinline__ unsigned ft_saddr(const void* p) {
  return (unsigned)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void ft_mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ft_saddr(bar)), "r"(count));
}
__device__ __forceinline__ void ft_mbar_expect(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(ft_saddr(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void ft_mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "FT_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra FT_DONE_%=;\n"
      "bra FT_WAIT_%=;\n"
      "FT_DONE_%=:\n"
      "}\n" ::"r"(ft_saddr(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void ft_tma_4d(void* dst, const CUtensorMap* tm,
                                          unsigned long long* bar, int c0, int c1, int c2,
                                          int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(ft_saddr(dst)),
      "l"(tm), "r"(ft_saddr(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

}  // namespace gk

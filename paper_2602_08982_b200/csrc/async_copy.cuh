// async_copy.cuh -- mbarrier + bulk asynchronous copy (cp.async.bulk, the 1-D form of TMA) wrappers, sm_90+/sm_100a.
// A bulk copy moves a contiguous run of bytes global -> shared without passing through registers and signals an
// mbarrier by transaction bytes when it lands; SASS: UBLKCP / SYNCS.  All sizes and addresses are multiples of 16.
#pragma once
#include <stdint.h>

__device__ __forceinline__ uint32_t ac_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void ac_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void ac_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival + the number of bytes the copies of this phase will deliver
__device__ __forceinline__ void ac_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void ac_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
// blocks until the phase with the given parity has completed (try_wait suspends the thread in hardware)
__device__ __forceinline__ void ac_mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "AC_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra AC_DONE_%=;\n"
      "bra AC_WAIT_%=;\n"
      "AC_DONE_%=:\n"
      "}\n" :: "r"(bar), "r"(parity) : "memory");
}
// global -> shared, `bytes` contiguous bytes, completion counted on `bar`; L2 eviction policy `pol` (createpolicy word)
__device__ __forceinline__ void ac_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
// orders earlier generic-proxy accesses to global memory (made visible to this thread) before later async-proxy ones
__device__ __forceinline__ void ac_fence_proxy_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ void ac_fence_proxy_shared() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// register budget of a warpgroup (4 consecutive warps); N a multiple of 8
template <int N> __device__ __forceinline__ void ac_reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(N)); }
template <int N> __device__ __forceinline__ void ac_reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(N)); }

// named barrier over `count` threads (a multiple of 32), id in [1, 15]
__device__ __forceinline__ void ac_bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void ac_bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" :: "r"(id), "r"(count) : "memory"); }

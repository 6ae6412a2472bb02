// vd_tma.cuh -- bulk copies of parked polytopes between HBM and shared memory through the TMA unit (cp.async.bulk, sm_90+;
// UBLKCP in SASS) instead of per-lane load / store loops: one instruction of one lane moves the 2-4 KB of a CellState prefix,
// completion arrives on an mbarrier in shared memory (loads) or through the bulk async-group (stores).
// Addresses and sizes are multiples of 16 bytes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace vd {

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// one lane of the warp; the others wait at the __syncwarp that follows in the caller
__device__ __forceinline__ void tma_bar_init(unsigned long long* bar) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_addr(bar)));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// global -> shared, `bytes` > 0; completion: `bytes` transaction bytes on bar.  One lane.  The destination may have been
// read or written through ordinary loads / stores before: the proxy fence orders those against the copy.
__device__ __forceinline__ void tma_load(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}

// every lane: wait until the phase `parity` of bar has completed
__device__ __forceinline__ void tma_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}

// shared -> global.  One lane, after the warp's ordinary stores to `src` (the caller synchronises the warp first).
__device__ __forceinline__ void tma_store(void* dst, const void* src, unsigned bytes) {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_addr(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// the lane that issued the stores: until their shared-memory source has been read (it may be overwritten afterwards)
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

}  // namespace vd

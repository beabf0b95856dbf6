// tma.cuh -- sm_100a plumbing of the TMA-fed sweeps: mbarrier, cp.async.bulk.tensor (4-D tiles).
// Inline PTX only; no arithmetic of the method lives here.
//
// All field and material arrays of a handle are equally spaced in the caller's workspace
// (kernels.cuh "DEVICE LAYOUT"), so ONE 4-D tensor (x = row pitch sy, y = ny+2, z = nz+2,
// a = array index) describes them all; a tensor map per box shape selects (x, y, z, a) tiles of it.
// Out-of-range coordinates are zero-filled by the hardware, so a tile may hang over the ghost layer.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace fl {

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t *b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
// make the barrier initialisation visible to the async proxy (TMA completes on these barriers)
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *b, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(b)), "r"(parity)
      : "memory");
  return ok != 0;
}
// try_wait that may sleep in hardware for up to `ns` nanoseconds before it reports "not yet"
__device__ __forceinline__ bool mbar_try_wait_sleep(uint64_t *b, uint32_t parity, uint32_t ns) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(b)), "r"(parity), "r"(ns)
      : "memory");
  return ok != 0;
}
// Wait for the phase with the given parity.  The waiting warp sleeps in the barrier unit (a
// polling loop of its own costs issue slots and power: it was 8 % of the sweep's instructions).
// A pipeline bug must not hang the GPU: about once a millisecond the wait looks at the wall clock
// (%globaltimer: independent of the SM clock, of time slicing and of profiler replays) and at
// *err; after 4 s, or when another wait has given up, it records `tag` in *err (first writer
// wins) and returns false; the caller then leaves its loop and the kernel ends.  The host reports
// the error from every call that synchronises (fdtd_llg_read_fields, _get_stats, _step_timed).
__device__ __forceinline__ bool mbar_wait(uint64_t *b, uint32_t parity, int *err, int tag) {
  if (mbar_try_wait(b, parity)) return true;
  long long t0 = 0;
  for (unsigned spins = 1;; ++spins) {
    if (mbar_try_wait_sleep(b, parity, 20000u)) return true;
    if ((spins & 63u) == 0) {
      unsigned long long now;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
      if (t0 == 0) t0 = (long long)now;
      if ((long long)now - t0 > 4000000000LL || *(volatile int *)err != 0) {
        atomicCAS(err, 0, tag);
        return false;
      }
    }
  }
}

// global -> shared tile; completion is signalled on `bar` (complete_tx::bytes)
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0,
                                            int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

}  // namespace fl

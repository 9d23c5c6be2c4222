// mhd_async.cuh -- sm_90+/sm_100a asynchronous-copy primitives used by the marching kernels:
// mbarrier + cp.async.bulk (the 1-D form of the Tensor Memory Accelerator, SASS UBLKCP).
// A march along y or z is limited by bytes in flight, not by bandwidth: one 128-byte line per field
// per warp per step with register prefetch keeps ~20 KB per SM outstanding.  Bulk copies into a
// shared-memory ring are issued several march steps ahead by one producer thread and cost the
// consumers neither registers nor address arithmetic.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mhd {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// MHD_JITTER (the second library build.py makes, libmhd_jitter.so; tests/test_gpu_jitter.py): every mbarrier wait, arrive and
// expect_tx is preceded, about one time in sixteen, by a sleep of 0.2-2.2 us chosen from the clock and the warp's
// position.  The march kernels have no block barrier; their warps drift and hand ring stages over through full/empty
// mbarriers (the neighbour hazard of PAPER.md:319).  compute-sanitizer is closed on this pool, so the guard is this:
// a protocol that only works for the interleavings the hardware happens to produce gives different bits (or hangs)
// once the interleavings are scrambled, and the test demands identical bits.
#ifdef MHD_JITTER
__device__ __forceinline__ void jitter() {
  unsigned t;
  asm volatile("mov.u32 %0, %%clock;" : "=r"(t));
  const unsigned w = (threadIdx.x >> 5) * 9u + blockIdx.x * 7u + blockIdx.y * 13u + blockIdx.z * 5u;
  const unsigned h = (t * 2654435761u) ^ (w * 40503u);
  if ((h >> 28) == 0u) __nanosleep(200u + ((h >> 8) & 2047u));
}
#else
__device__ __forceinline__ void jitter() {}
#endif

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  jitter();
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  jitter();
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  jitter();
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// global -> shared bulk copy; bytes a multiple of 16, both addresses 16-byte aligned; completes on bar
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// One lane of a fully converged warp.  ptxas recognises the elect.sync predicate: a cp.async.bulk guarded by it
// becomes one UBLKCP with operands in uniform registers.  Guarded by a lane-index test instead, every copy is
// wrapped in an ELECT / 5 x R2UR.BROADCAST / BRA.U.ANY loop over the active lanes (10 instructions per copy,
// measured: 12 % of the B-pair ring kernel's issued instructions, a round-1 ncu capture; today's opcode mix is in profiles/r02_c4_step_ncu_full.md).
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "elect.sync _|p, 0xffffffff;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(pred));
  return pred != 0;
}

}  // namespace mhd

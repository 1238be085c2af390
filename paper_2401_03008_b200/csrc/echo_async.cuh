// echo_async.cuh — sm_100a asynchronous-copy primitives used by the tile-marching kernels: TMA box copies
// global -> shared issued by ONE thread (cp.async.bulk.tensor, SASS UTMALDG) that complete on a shared-memory mbarrier
// by transaction bytes (SASS SYNCS), and the classic per-thread 8-byte cp.async (LDGSTS), which can arrive on the same
// mbarrier, for tiles that wrap around a periodic seam.  Plain wrappers around the PTX; no arithmetic of the method.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace echo {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// ---- per-thread 8-byte asynchronous copies (LDGSTS)
__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const double *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- mbarrier (one 8-byte word in shared memory)
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned arrivals) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(arrivals) : "memory");
}
// makes the initialised barriers visible to the asynchronous proxy (the bulk copies) before the first use
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival that also announces `bytes` of asynchronous-copy transactions still to land on this phase
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// blocks until the phase of the given parity has completed (try_wait suspends the thread in hardware between polls)
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MBAR_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MBAR_DONE_%=;\n"
        "bra MBAR_WAIT_%=;\n"
        "MBAR_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// ---- TMA: one thread copies a whole 3-D box {bx, by, 1} of a field (tensor map = CUtensorMap in kernel-parameter
// space, built by cuTensorMapEncodeTiled on the host) to shared memory, rows dense (pitch = bx); completion on `bar`
// as bx*by*8 transaction bytes.  SASS: UTMALDG.
__device__ __forceinline__ void tma_load_3d(void *smem_dst, const void *tensor_map, int cx, int cy, int cz, uint64_t *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(tensor_map), "r"(cx), "r"(cy), "r"(cz), "r"(smem_u32(bar))
                 : "memory");
}
// per-thread cp.async copies issued so far by this thread arrive on `bar` when they have landed (the barrier's
// expected-arrival count includes one such arrival per issuing thread: .noinc)
__device__ __forceinline__ void cp_async_arrive_on(uint64_t *bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

}  // namespace echo

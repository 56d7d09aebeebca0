// Minimal inline-PTX wrappers for the sm_100a asynchronous-copy machinery the pruned search uses:
// mbarrier (init / expect_tx / try_wait.parity), the 3-D TMA tile load (cp.async.bulk.tensor ->
// SASS UTMALDG) and the generic->async proxy fence.  Host side: cuTensorMapEncodeTiled resolved at
// run time through cudaGetDriverEntryPoint (no link-time dependency on libcuda).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

__device__ __forceinline__ uint32_t kb_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void kb_mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(kb_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void kb_fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void kb_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(kb_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void kb_mbar_wait(uint64_t* bar, uint32_t parity) {
    // try_wait suspends the thread in hardware until the phase completes or the time hint (ns) runs out, so a
    // waiting warp costs a few issue slots per microsecond instead of spinning against the warps that have work
#ifdef KB_WAIT_PLAIN
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "KB_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra KB_DONE_%=;\n\t"
        "bra KB_WAIT_%=;\n\t"
        "KB_DONE_%=:\n\t"
        "}" ::"r"(kb_smem_u32(bar)), "r"(parity) : "memory");
#else
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "KB_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
        "@p bra KB_DONE_%=;\n\t"
        "bra KB_WAIT_%=;\n\t"
        "KB_DONE_%=:\n\t"
        "}" ::"r"(kb_smem_u32(bar)), "r"(parity), "r"(2000u) : "memory");
#endif
}
// non-blocking test of a phase (acquire): true once the phase with this parity has completed
__device__ __forceinline__ bool kb_mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(ok) : "r"(kb_smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// generic-proxy writes to shared memory (st.shared) must be ordered before async-proxy (TMA) writes
__device__ __forceinline__ void kb_fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// 3-D tile load: box (boxDim of the map) at element coordinates (x, y, z) -> dense smem block; signed
// coordinates; out-of-bounds elements are zero-filled (this IS the off-image rule of the search).
__device__ __forceinline__ void kb_tma_load_3d(void* smem_dst, const CUtensorMap* map, int x, int y, int z,
                                               uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(kb_smem_u32(smem_dst)), "l"(map), "r"(x), "r"(y), "r"(z), "r"(kb_smem_u32(bar))
        : "memory");
}
// 1-D bulk copy global -> shared (SASS UBLKCP); src, dst 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void kb_bulk_load_1d(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(kb_smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(kb_smem_u32(bar))
                 : "memory");
}
// plain arrive (release.cta): a consumer warp hands a ring slot back to the producer
__device__ __forceinline__ void kb_mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(kb_smem_u32(bar)) : "memory");
}
// warp-group register reallocation (setmaxnreg): the producer warp gives registers back, the consumer
// warps take them; every warp of a warp group (4 consecutive warps) must execute the same instruction
template <int R> __device__ __forceinline__ void kb_reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R> __device__ __forceinline__ void kb_reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }
__device__ __forceinline__ void kb_prefetch_tensormap(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// host: driver entry point for cuTensorMapEncodeTiled
typedef CUresult (*kb_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                       const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                       CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
kb_encode_tiled_fn kb_get_encode_tiled();

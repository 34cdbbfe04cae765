// TMA (cp.async.bulk.tensor) and mbarrier plumbing for sm_100a, as inline PTX, plus the host-side tensor-map encoder.
// The driver entry point cuTensorMapEncodeTiled is looked up at run time (cudaGetDriverEntryPoint), so libcbct.so keeps
// loading on a box without libcuda (the CPU-only ABI tests).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>

#include "cbct_internal.h"

// ---- host ---------------------------------------------------------------------------------------------------------
// 3-D fp32 tensor [d2][d1][d0] (d0 fastest, contiguous; pitches in BYTES, multiples of 16; base 16-byte aligned) with a
// box of b0 x b1 x b2 elements (each <= 256, b0 * 4 a multiple of 16).  Out-of-bounds elements of a box read as 0.
cbct_status cbct_tensor_map_3d(CUtensorMap *out, const float *base, unsigned long long d0, unsigned long long d1,
                               unsigned long long d2, unsigned long long pitch1_bytes, unsigned long long pitch2_bytes,
                               unsigned b0, unsigned b1, unsigned b2);

// ---- device -------------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// makes the initialised barriers visible to the async proxy (the TMA unit)
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// box -> shared memory; completes `bytes of the box` on the mbarrier
__device__ __forceinline__ void tma_load_3d(void *smem_dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
#endif

// dslash_async.cuh -- sm_100a asynchronous-copy plumbing shared by the shared-memory-staged kernels (dslash_tma.cu,
// dslash_ring.cu): mbarrier + cp.async.bulk (the TMA unit, SASS UBLKCP) PTX wrappers and spinor reads from a shared-memory
// copy of a 32-site vector in the global blocked-SoA format.
#pragma once
#include <stdint.h>

#include "dslash_site.cuh"

namespace dslash {

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// the same wait without PTX labels (can be inlined any number of times into one kernel)
__device__ __forceinline__ void mbar_wait_spin(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// Orders this thread's earlier generic-proxy accesses to shared memory (and, through a preceding barrier, those of the threads
// it synchronised with) before its later async-proxy operations: needed before a bulk copy REFILLS a buffer that was just read.
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// global -> shared bulk copy, completion (bytes) signalled on the mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------ shared-memory field access
// Same vector format as global memory, indexed by the tile-local site number (plain ld.shared).
template <typename Real>
struct unit16;
template <>
struct unit16<double> {
    using type = double2;
};
template <>
struct unit16<float> {
    using type = float4;
};

__device__ __forceinline__ void load_spinor_smem(cplx<double> (&psi)[12], const void* base, unsigned ls) {
    const double2* p = reinterpret_cast<const double2*>(base) + (size_t)(ls >> VL_LOG2) * (12u * VL) + (ls & (VL - 1u));
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        double2 v = p[k * VL];
        psi[k] = {v.x, v.y};
    }
}
__device__ __forceinline__ void load_spinor_smem(cplx<float> (&psi)[12], const void* base, unsigned ls) {
    const float4* p = reinterpret_cast<const float4*>(base) + (size_t)(ls >> VL_LOG2) * (6u * VL) + (ls & (VL - 1u));
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        float4 v = p[q * VL];
        psi[2 * q] = {v.x, v.y};
        psi[2 * q + 1] = {v.z, v.w};
    }
}
}  // namespace dslash

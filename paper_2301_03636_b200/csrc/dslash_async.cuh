// dslash_async.cuh -- sm_100a asynchronous-copy plumbing shared by the shared-memory-staged kernels (dslash_march.cu,
// dslash_wpipe.cu): mbarrier + cp.async.bulk (the TMA unit's flat bulk copy, SASS UBLKCP) PTX wrappers, reads of spinors and
// links from a shared-memory copy of a 32-site vector in the global blocked-SoA format, and hops on operands in registers.
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
// non-blocking test of a phase (the producer warp polls many barriers in turn)
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return done != 0u;
}
// plain arrival (release semantics at CTA scope): "this warp has finished reading / writing the buffer"
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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

// the same copy with an L2 eviction policy (createpolicy, see make_policy) for the global read
__device__ __forceinline__ void bulk_g2s_hint(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
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
// ------------------------------------------------------------------ one 32-site vector in shared memory, lane = site
// spinor of lane `lane` from a shared-memory copy of one spinor vector (global blocked-SoA format)
template <typename Real>
__device__ __forceinline__ void load_psi_slot(cplx<Real> (&psi)[12], const unsigned char* p, unsigned lane);
template <>
__device__ __forceinline__ void load_psi_slot<double>(cplx<double> (&psi)[12], const unsigned char* p, unsigned lane) {
    const double2* q = reinterpret_cast<const double2*>(p) + lane;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const double2 v = q[k * VL];
        psi[k] = {v.x, v.y};
    }
}
template <>
__device__ __forceinline__ void load_psi_slot<float>(cplx<float> (&psi)[12], const unsigned char* p, unsigned lane) {
    const float4* q = reinterpret_cast<const float4*>(p) + lane;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float4 v = q[k * VL];
        psi[2 * k] = {v.x, v.y};
        psi[2 * k + 1] = {v.z, v.w};
    }
}

// link of lane `lane` from a shared-memory copy of one (vector, mu) block of the gauge field; RECON == 12 rebuilds row 2
// exactly as load_link() does.
template <typename Real, int RECON>
__device__ __forceinline__ void load_link_slot(cplx<Real> (&u)[9], const unsigned char* p, unsigned lane) {
    using V2 = typename vec2<Real>::type;
    constexpr int R = (RECON == 12) ? 6 : 9;
    const V2* q = reinterpret_cast<const V2*>(p) + lane;
#pragma unroll
    for (int e = 0; e < R; ++e) {
        const V2 v = q[e * VL];
        u[e] = {v.x, v.y};
    }
    if (RECON == 12) reconstruct_row2(u);
}

// a 32-site vector of half-spinors (6 complex per site, component-major like the fields): the exchange buffers of the
// marching kernels
template <typename Real>
__device__ __forceinline__ void store_half(unsigned char* p, unsigned lane, const cplx<Real> (&h)[6]) {
    using V2 = typename vec2<Real>::type;
    V2* q = reinterpret_cast<V2*>(p) + lane;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        V2 v;
        v.x = h[k].re;
        v.y = h[k].im;
        q[k * VL] = v;
    }
}
template <typename Real>
__device__ __forceinline__ void load_half(cplx<Real> (&h)[6], const unsigned char* p, unsigned lane) {
    using V2 = typename vec2<Real>::type;
    const V2* q = reinterpret_cast<const V2*>(p) + lane;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const V2 v = q[k * VL];
        h[k] = {v.x, v.y};
    }
}

// the two x hops from the row's own spinors and links (the arithmetic of x_hops_shuffle with the operands in registers)
template <typename Real>
__device__ __forceinline__ void x_hops_regs(cplx<Real> (&acc)[12], const cplx<Real> (&psi)[12], const cplx<Real> (&u)[9],
                                            int lane_fwd, int lane_bwd) {
    cplx<Real> hm[6], hq[6], w[6], hp[6];
    project<0, -1>(hm, psi);
    project<0, +1>(hq, psi);
    su3_mul<true>(w, u, hq);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        hm[k].re = shfl_(hm[k].re, lane_fwd);
        hm[k].im = shfl_(hm[k].im, lane_fwd);
        w[k].re = shfl_(w[k].re, lane_bwd);
        w[k].im = shfl_(w[k].im, lane_bwd);
    }
    su3_mul<false>(hp, u, hm);
    reconstruct_accumulate<0, -1, true>(acc, hp);
    reconstruct_accumulate<0, +1, false>(acc, w);
}

// one hop with both operands in registers
template <int MU, int SIGN, typename Real>
__device__ __forceinline__ void hop_regs(cplx<Real> (&acc)[12], const cplx<Real> (&psi)[12], const cplx<Real> (&u)[9]) {
    cplx<Real> h[6], hp[6];
    project<MU, SIGN>(h, psi);
    su3_mul<(SIGN > 0)>(hp, u, h);
    reconstruct_accumulate<MU, SIGN, false>(acc, hp);
}
}  // namespace dslash

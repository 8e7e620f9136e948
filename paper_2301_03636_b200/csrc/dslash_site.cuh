// dslash_site.cuh -- per-site body of the Wilson Dslash for sm_100a (device code only).
//
// Operator: PAPER.md:47-50 (section 1.1, Eq. 1) with the backward link at x-mu^ (DESIGN.md Reading R1):
//   out(x) = sum_mu [ (1 - gamma_mu) U_mu(x) psi(x+mu^) + (1 + gamma_mu) U_mu(x-mu^)^dagger psi(x-mu^) ]
//
// Unlike the oracle (which multiplies by the full 4x4 gamma matrices) this path uses the rank-2
// structure of (1 -+ gamma_mu) in the DeGrand-Rossi basis: project the neighbour spinor to a
// half-spinor h (2 spin rows x 3 colours), multiply both rows by the 3x3 link in registers, and
// rebuild spin rows 2,3 from rows 0,1.  1320 flop per site.
//
// This file shares nothing with oracle/: the projection table below was derived by hand from the
// gamma matrices of DESIGN.md Reading R4 and is checked only through GPU-vs-oracle parity.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dslash {

enum : int { LAYOUT_AOS = 0, LAYOUT_SOA = 1 };

// The SoA layout is blocked ("array of structures of arrays"): sites are grouped in vectors of VL = 32
// consecutive site indices; within a vector every component is a contiguous run of 32 elements.
//   spinor  unit16[ (s / 32) * (NU * 32) + k * 32 + (s % 32) ]          NU = 12 (fp64, double2) or 6 (fp32, float4)
//   gauge   vec2  [ ((s / 32) * 4 + mu) * (R * 32) + e * 32 + (s % 32) ]  R = 9 or 6
// A warp that handles 32 consecutive sites still reads one contiguous 512-byte (fp32 links: 256-byte) run
// per component, but the component stride is the compile-time constant 32 elements, so the 12 (9) loads of
// a spinor (link) share ONE 64-bit base address and differ only in the instruction's immediate offset
// (SASS: LDG.E.128 [R.64 + imm]) -- the planar [k][V] form spent ~4.5 integer instructions per load on
// addresses.  V is padded up to a multiple of 32; the padding is never read by the operator.
constexpr unsigned VL = 32u;
constexpr unsigned VL_LOG2 = 5u;

struct Geom {
    int L[4];    // L_X, L_Y, L_Z, L_T
    unsigned V;  // number of sites
};

template <typename Real>
struct cplx {
    Real re, im;
};

// ------------------------------------------------------------------ complex helpers
template <typename Real>
__device__ __forceinline__ cplx<Real> c_add(cplx<Real> a, cplx<Real> b) { return {a.re + b.re, a.im + b.im}; }
template <typename Real>
__device__ __forceinline__ cplx<Real> c_sub(cplx<Real> a, cplx<Real> b) { return {a.re - b.re, a.im - b.im}; }
// a + i*b
template <typename Real>
__device__ __forceinline__ cplx<Real> c_add_i(cplx<Real> a, cplx<Real> b) { return {a.re - b.im, a.im + b.re}; }
// a - i*b
template <typename Real>
__device__ __forceinline__ cplx<Real> c_sub_i(cplx<Real> a, cplx<Real> b) { return {a.re + b.im, a.im - b.re}; }

__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

// ------------------------------------------------------------------ global loads/stores with an optional L2 eviction policy
// HINT = false: plain read-only loads (__ldg) and plain stores.  HINT = true: the same accesses carry a 64-bit L2
// cache policy made by `createpolicy` (evict_last for data that is re-read one or two time-slices later,
// evict_first for data that is dead after this access) -- SASS LDG/STG with a desc[UR] operand.
struct Policies {
    uint64_t psi, u_t, u_s, out;  // spinor loads, U_t loads, U_x/U_y/U_z loads, stores of `out`
};
enum : int { POLICY_NORMAL = 0, POLICY_EVICT_LAST = 1, POLICY_EVICT_FIRST = 2 };
__device__ __forceinline__ uint64_t make_policy(int kind) {
    uint64_t p;
    if (kind == POLICY_EVICT_LAST)
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else if (kind == POLICY_EVICT_FIRST)
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else
        asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// HINT: 0 plain __ldg, 1 with the L2 policy, 2 with the L2 policy and L1::no_allocate (data with no reuse inside the block)
template <int HINT>
__device__ __forceinline__ double2 ld_ro(const double2* p, uint64_t pol) {
    if (HINT == 0) return __ldg(p);
    double2 v;
    if (HINT == 2)
        asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    else
        asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
template <int HINT>
__device__ __forceinline__ float4 ld_ro(const float4* p, uint64_t pol) {
    if (HINT == 0) return __ldg(p);
    float4 v;
    if (HINT == 2)
        asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                     : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                     : "l"(p), "l"(pol));
    else
        asm volatile("ld.global.nc.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                     : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                     : "l"(p), "l"(pol));
    return v;
}
template <int HINT>
__device__ __forceinline__ float2 ld_ro(const float2* p, uint64_t pol) {
    if (HINT == 0) return __ldg(p);
    float2 v;
    if (HINT == 2)
        asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    else
        asm volatile("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}
template <int HINT>
__device__ __forceinline__ void st_g(double2* p, double2 v, uint64_t pol) {
    if (!HINT) {
        *p = v;
        return;
    }
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
template <int HINT>
__device__ __forceinline__ void st_g(float4* p, float4 v, uint64_t pol) {
    if (!HINT) {
        *p = v;
        return;
    }
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w),
                 "l"(pol)
                 : "memory");
}

// acc += a * b
template <typename Real>
__device__ __forceinline__ void c_madd(cplx<Real>& acc, cplx<Real> a, cplx<Real> b) {
    acc.re = fma_(a.re, b.re, acc.re);
    acc.re = fma_(-a.im, b.im, acc.re);
    acc.im = fma_(a.re, b.im, acc.im);
    acc.im = fma_(a.im, b.re, acc.im);
}
// acc += conj(a) * b
template <typename Real>
__device__ __forceinline__ void c_madd_conj(cplx<Real>& acc, cplx<Real> a, cplx<Real> b) {
    acc.re = fma_(a.re, b.re, acc.re);
    acc.re = fma_(a.im, b.im, acc.re);
    acc.im = fma_(a.re, b.im, acc.im);
    acc.im = fma_(-a.im, b.re, acc.im);
}
// a * b
template <typename Real>
__device__ __forceinline__ cplx<Real> c_mul(cplx<Real> a, cplx<Real> b) {
    cplx<Real> r;
    r.re = a.re * b.re;
    r.re = fma_(-a.im, b.im, r.re);
    r.im = a.re * b.im;
    r.im = fma_(a.im, b.re, r.im);
    return r;
}
// conj(a) * b
template <typename Real>
__device__ __forceinline__ cplx<Real> c_mul_conj(cplx<Real> a, cplx<Real> b) {
    cplx<Real> r;
    r.re = a.re * b.re;
    r.re = fma_(a.im, b.im, r.re);
    r.im = a.re * b.im;
    r.im = fma_(-a.im, b.re, r.im);
    return r;
}

// ------------------------------------------------------------------ FP32: two lanes per instruction (sm_100a f32x2)
// Blackwell's FP32 pipe executes add / mul / fma on PAIRS of floats held in a 64-bit register (PTX add/mul/fma.rn.f32x2,
// SASS FADD2 / FMUL2 / FFMA2), and ptxas folds a scalar broadcast (R.F32), a lane swap (.LO_HI) and a one-lane negation (.NP)
// into the operand, so a complex number IS a pair: c_madd is two FFMA2 instead of four FFMA, c_add_i one FADD2 instead of two
// FADD, with no packing instructions (the mov.b64 below disappear when (re, im) sit in an aligned register pair, which is how
// the float4 / float2 loads deliver them).  Every component sees the same operations in the same order as in the scalar
// templates above (one IEEE fma / add / mul per lane), so results are bit-identical to them -- and to one another across
// kernels, whichever form a translation unit uses.  A translation unit opts in with #define DSLASH_F32X2 before including
// this header.  Measured in one call, scalar vs packed (profiles/r02b_f32x2.md): the marching kernels gain 10-12 % in FP32
// (fewer instructions in the compute warps' serial timeline: 32^3x64 0.244 -> 0.221 ms, 48^3x96 (generalised march, since removed) gmarch 2.36 -> 2.09 ms); the
// direct kernel gains nothing at 48^3x96 (0.915 vs 0.916 ms) and LOSES 4.5 % at 32^3x64 (0.184 vs 0.1765 ms: with 128
// registers and aligned pairs the compiler keeps fewer loads in flight), so dslash_tuned.cu and the other one-thread-per-site
// units stay scalar.  For A/B measurements the whole library can be built one way or the other:
//   DSLASH_NVCC_EXTRA=-DDSLASH_F32X2 (packed everywhere) / -DDSLASH_SCALAR_F32 (scalar everywhere), see build.py.
#if defined(DSLASH_F32X2) && !defined(DSLASH_SCALAR_F32)
__device__ __forceinline__ uint64_t f2_pack(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ cplx<float> f2_unpack(uint64_t v) {
    cplx<float> c;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(c.re), "=f"(c.im) : "l"(v));
    return c;
}
__device__ __forceinline__ uint64_t f2_add(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t f2_sub(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t f2_mul(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// non-template overloads: preferred over the templates above for cplx<float>
__device__ __forceinline__ cplx<float> c_add(cplx<float> a, cplx<float> b) { return f2_unpack(f2_add(f2_pack(a.re, a.im), f2_pack(b.re, b.im))); }
__device__ __forceinline__ cplx<float> c_sub(cplx<float> a, cplx<float> b) { return f2_unpack(f2_sub(f2_pack(a.re, a.im), f2_pack(b.re, b.im))); }
// a + i*b = (a.re - b.im, a.im + b.re);  a - i*b = (a.re + b.im, a.im - b.re)
__device__ __forceinline__ cplx<float> c_add_i(cplx<float> a, cplx<float> b) { return f2_unpack(f2_add(f2_pack(a.re, a.im), f2_pack(-b.im, b.re))); }
__device__ __forceinline__ cplx<float> c_sub_i(cplx<float> a, cplx<float> b) { return f2_unpack(f2_add(f2_pack(a.re, a.im), f2_pack(b.im, -b.re))); }
// acc += a * b:        re: fma(a.re, b.re, .) then fma(-a.im, b.im, .);   im: fma(a.re, b.im, .) then fma(a.im, b.re, .)
__device__ __forceinline__ void c_madd(cplx<float>& acc, cplx<float> a, cplx<float> b) {
    uint64_t r = f2_fma(f2_pack(a.re, a.re), f2_pack(b.re, b.im), f2_pack(acc.re, acc.im));
    acc = f2_unpack(f2_fma(f2_pack(-a.im, a.im), f2_pack(b.im, b.re), r));
}
// acc += conj(a) * b:  re: fma(a.re, b.re, .) then fma(a.im, b.im, .);    im: fma(a.re, b.im, .) then fma(-a.im, b.re, .)
__device__ __forceinline__ void c_madd_conj(cplx<float>& acc, cplx<float> a, cplx<float> b) {
    uint64_t r = f2_fma(f2_pack(a.re, a.re), f2_pack(b.re, b.im), f2_pack(acc.re, acc.im));
    acc = f2_unpack(f2_fma(f2_pack(a.im, -a.im), f2_pack(b.im, b.re), r));
}
__device__ __forceinline__ cplx<float> c_mul(cplx<float> a, cplx<float> b) {
    uint64_t r = f2_mul(f2_pack(a.re, a.re), f2_pack(b.re, b.im));
    return f2_unpack(f2_fma(f2_pack(-a.im, a.im), f2_pack(b.im, b.re), r));
}
__device__ __forceinline__ cplx<float> c_mul_conj(cplx<float> a, cplx<float> b) {
    uint64_t r = f2_mul(f2_pack(a.re, a.re), f2_pack(b.re, b.im));
    return f2_unpack(f2_fma(f2_pack(a.im, -a.im), f2_pack(b.im, b.re), r));
}
#endif

// ------------------------------------------------------------------ field access (read-only path, 128-bit where the layout allows)
// Spinor, 12 complex components of site s.
template <typename Real, int LAYOUT>
struct SpinorIO;

template <int LAYOUT>
struct SpinorIO<double, LAYOUT> {
    __device__ __forceinline__ static size_t idx(unsigned V, unsigned s, int k) {
        return LAYOUT == LAYOUT_AOS ? (size_t)s * 12 + k : (size_t)(s >> VL_LOG2) * (12u * VL) + (s & (VL - 1u)) + (unsigned)k * VL;
    }
    template <int HINT = 0>
    __device__ __forceinline__ static void load(cplx<double> (&psi)[12], const void* base, unsigned V, unsigned s, uint64_t pol = 0) {
        const double2* p = reinterpret_cast<const double2*>(base);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            double2 v = ld_ro<HINT>(p + idx(V, s, k), pol);
            psi[k] = {v.x, v.y};
        }
    }
    template <int HINT = 0>
    __device__ __forceinline__ static void store(void* base, unsigned V, unsigned s, const cplx<double> (&psi)[12], uint64_t pol = 0) {
        double2* p = reinterpret_cast<double2*>(base);
#pragma unroll
        for (int k = 0; k < 12; ++k) st_g<HINT>(p + idx(V, s, k), make_double2(psi[k].re, psi[k].im), pol);
    }
};
template <int LAYOUT>
struct SpinorIO<float, LAYOUT> {
    __device__ __forceinline__ static size_t idx(unsigned V, unsigned s, int q) {
        return LAYOUT == LAYOUT_AOS ? (size_t)s * 6 + q : (size_t)(s >> VL_LOG2) * (6u * VL) + (s & (VL - 1u)) + (unsigned)q * VL;
    }
    template <int HINT = 0>
    __device__ __forceinline__ static void load(cplx<float> (&psi)[12], const void* base, unsigned V, unsigned s, uint64_t pol = 0) {
        const float4* p = reinterpret_cast<const float4*>(base);
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            float4 v = ld_ro<HINT>(p + idx(V, s, q), pol);
            psi[2 * q] = {v.x, v.y};
            psi[2 * q + 1] = {v.z, v.w};
        }
    }
    template <int HINT = 0>
    __device__ __forceinline__ static void store(void* base, unsigned V, unsigned s, const cplx<float> (&psi)[12], uint64_t pol = 0) {
        float4* p = reinterpret_cast<float4*>(base);
#pragma unroll
        for (int q = 0; q < 6; ++q)
            st_g<HINT>(p + idx(V, s, q), make_float4(psi[2 * q].re, psi[2 * q].im, psi[2 * q + 1].re, psi[2 * q + 1].im), pol);
    }
};

template <typename Real>
struct vec2;
template <>
struct vec2<double> {
    using type = double2;
};
template <>
struct vec2<float> {
    using type = float2;
};

// Row 2 of an SU(3) link from rows 0 and 1: row2 = conj(row0 x row1) (exact for SU(3), DESIGN.md Reading R14).
// u[0..5] = rows 0,1 on entry; u[6..8] written.  The ONE place this is computed: every kernel with RECON == 12 calls it.
template <typename Real>
__device__ __forceinline__ void reconstruct_row2(cplx<Real> (&u)[9]) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int j1 = (j + 1) % 3, j2 = (j + 2) % 3;
        // row2[j] = conj(row0[j1]*row1[j2] - row0[j2]*row1[j1])
        cplx<Real> a = c_mul(u[j1], u[3 + j2]);
        Real re = fma_(-u[j2].re, u[3 + j1].re, a.re);
        re = fma_(u[j2].im, u[3 + j1].im, re);
        Real im = fma_(-u[j2].re, u[3 + j1].im, a.im);
        im = fma_(-u[j2].im, u[3 + j1].re, im);
        u[6 + j] = {re, -im};
    }
}

// Link U_mu(s): 9 complex entries u[row*3+col]; with RECON == 12 only rows 0,1 are stored and row 2
// is rebuilt by reconstruct_row2().
template <typename Real, int LAYOUT, int RECON, int HINT = 0>
__device__ __forceinline__ void load_link(cplx<Real> (&u)[9], const void* base, unsigned V, unsigned s, int mu, uint64_t pol = 0) {
    using V2 = typename vec2<Real>::type;
    constexpr int R = (RECON == 12) ? 6 : 9;
    const V2* p = reinterpret_cast<const V2*>(base);
    if (LAYOUT == LAYOUT_AOS) {
        p += (size_t)(s * 4u + (unsigned)mu) * R;
#pragma unroll
        for (int e = 0; e < R; ++e) {
            V2 v = ld_ro<HINT>(p + e, pol);
            u[e] = {v.x, v.y};
        }
    } else {
        p += (size_t)((s >> VL_LOG2) * 4u + (unsigned)mu) * (R * VL) + (s & (VL - 1u));
#pragma unroll
        for (int e = 0; e < R; ++e) {
            V2 v = ld_ro<HINT>(p + e * VL, pol);
            u[e] = {v.x, v.y};
        }
    }
    if (RECON == 12) reconstruct_row2(u);
}

// ------------------------------------------------------------------ measurement aid: the data-movement skeleton
// Compiled with -DDSLASH_NO_MATH (python -m paper_2301_03636_b200.build --skeleton -> libdslash_b200_skeleton.so) the three
// arithmetic building blocks below are replaced by a handful of additions that keep the data dependence on every loaded
// value, so every kernel moves exactly the bytes it moves in the product, through the same loads, copies, hand-offs and
// stores, and computes (almost) nothing.  The result is NOT the operator; bench.py --skeleton times it to show how close a
// kernel is to its own data movement (profiles/r02b_skeleton.md).  The product library never defines the macro.
// ------------------------------------------------------------------ spin projection / reconstruction
// SIGN = -1: (1 - gamma_MU)  (forward hop);  SIGN = +1: (1 + gamma_MU)  (backward hop).
// h[0..2] = kept row 0, h[3..5] = kept row 1 (colour index fastest).
template <int MU, int SIGN, typename Real>
__device__ __forceinline__ void project(cplx<Real> (&h)[6], const cplx<Real> (&psi)[12]) {
#ifdef DSLASH_NO_MATH
#pragma unroll
    for (int k = 0; k < 6; ++k) h[k] = {psi[k].re + psi[k + 6].re, psi[k].im + psi[k + 6].im};
    if (MU >= 0) return;
#endif
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cplx<Real> p0 = psi[c], p1 = psi[3 + c], p2 = psi[6 + c], p3 = psi[9 + c];
        if (MU == 0) {          // h0 = p0 -+ i p3, h1 = p1 -+ i p2
            h[c] = (SIGN < 0) ? c_sub_i(p0, p3) : c_add_i(p0, p3);
            h[3 + c] = (SIGN < 0) ? c_sub_i(p1, p2) : c_add_i(p1, p2);
        } else if (MU == 1) {   // h0 = p0 +- p3, h1 = p1 -+ p2
            h[c] = (SIGN < 0) ? c_add(p0, p3) : c_sub(p0, p3);
            h[3 + c] = (SIGN < 0) ? c_sub(p1, p2) : c_add(p1, p2);
        } else if (MU == 2) {   // h0 = p0 -+ i p2, h1 = p1 +- i p3
            h[c] = (SIGN < 0) ? c_sub_i(p0, p2) : c_add_i(p0, p2);
            h[3 + c] = (SIGN < 0) ? c_add_i(p1, p3) : c_sub_i(p1, p3);
        } else {                // h0 = p0 -+ p2, h1 = p1 -+ p3
            h[c] = (SIGN < 0) ? c_sub(p0, p2) : c_add(p0, p2);
            h[3 + c] = (SIGN < 0) ? c_sub(p1, p3) : c_add(p1, p3);
        }
    }
}

// acc += R(h) where rows 0,1 = h0,h1 and rows 2,3 follow from the projector:
//   MU 0: r2 = +-i h1, r3 = +-i h0    MU 1: r2 = -+ h1, r3 = +- h0
//   MU 2: r2 = +-i h0, r3 = -+i h1    MU 3: r2 = -+ h0, r3 = -+ h1       (upper sign: SIGN = -1)
template <int MU, int SIGN, bool FIRST, typename Real>
__device__ __forceinline__ void reconstruct_accumulate(cplx<Real> (&acc)[12], const cplx<Real> (&h)[6]) {
#ifdef DSLASH_NO_MATH
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        if (FIRST) {
            acc[k] = h[k];
            acc[k + 6] = h[k];
        } else {
            acc[k].re += h[k].re;
            acc[k + 6].im += h[k].im;
        }
    }
    if (MU >= 0) return;
#endif
    constexpr bool M = SIGN < 0;  // the (1 - gamma) projector
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cplx<Real> h0 = h[c], h1 = h[3 + c];
        // rows 2,3 are updated in place (acc +- h, acc +- i h) so that no separate negation is executed
        cplx<Real> a2 = acc[6 + c], a3 = acc[9 + c];
        if (FIRST) {
            a2 = {Real(0), Real(0)};
            a3 = {Real(0), Real(0)};
        }
        if (MU == 0) {          // r2 = +-i h1, r3 = +-i h0
            a2 = M ? c_add_i(a2, h1) : c_sub_i(a2, h1);
            a3 = M ? c_add_i(a3, h0) : c_sub_i(a3, h0);
        } else if (MU == 1) {   // r2 = -+ h1, r3 = +- h0
            a2 = M ? c_sub(a2, h1) : c_add(a2, h1);
            a3 = M ? c_add(a3, h0) : c_sub(a3, h0);
        } else if (MU == 2) {   // r2 = +-i h0, r3 = -+i h1
            a2 = M ? c_add_i(a2, h0) : c_sub_i(a2, h0);
            a3 = M ? c_sub_i(a3, h1) : c_add_i(a3, h1);
        } else {                // r2 = -+ h0, r3 = -+ h1
            a2 = M ? c_sub(a2, h0) : c_add(a2, h0);
            a3 = M ? c_sub(a3, h1) : c_add(a3, h1);
        }
        acc[6 + c] = a2;
        acc[9 + c] = a3;
        if (FIRST) {
            acc[c] = h0;
            acc[3 + c] = h1;
        } else {
            acc[c] = c_add(acc[c], h0);
            acc[3 + c] = c_add(acc[3 + c], h1);
        }
    }
}

// hp = U h (DAGGER = false) or U^dagger h (DAGGER = true), both spin rows.
template <bool DAGGER, typename Real>
__device__ __forceinline__ void su3_mul(cplx<Real> (&hp)[6], const cplx<Real> (&u)[9], const cplx<Real> (&h)[6]) {
#ifdef DSLASH_NO_MATH
#pragma unroll
    for (int k = 0; k < 6; ++k) hp[k] = {h[k].re + u[k].re, h[k].im + u[(k + 3) % 9].im + u[8].re};
    if (sizeof(Real) > 0) return;
#endif
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            cplx<Real> a;
            if (!DAGGER) {
                a = c_mul(u[i * 3 + 0], h[r * 3 + 0]);
                c_madd(a, u[i * 3 + 1], h[r * 3 + 1]);
                c_madd(a, u[i * 3 + 2], h[r * 3 + 2]);
            } else {
                a = c_mul_conj(u[0 * 3 + i], h[r * 3 + 0]);
                c_madd_conj(a, u[1 * 3 + i], h[r * 3 + 1]);
                c_madd_conj(a, u[2 * 3 + i], h[r * 3 + 2]);
            }
            hp[r * 3 + i] = a;
        }
}

// One hop: acc (+)= R_{MU,SIGN}( U^(dagger) P_{MU,SIGN} psi(sn) ), link taken at site sl.
template <int MU, int SIGN, bool FIRST, typename Real, int LAYOUT, int RECON, int HINT = 0>
__device__ __forceinline__ void hop(cplx<Real> (&acc)[12], const void* in, const void* gauge, unsigned V, unsigned sn,
                                    unsigned sl, uint64_t pol_psi = 0, uint64_t pol_u = 0) {
    cplx<Real> psi[12], h[6], hp[6], u[9];
    SpinorIO<Real, LAYOUT>::template load<HINT>(psi, in, V, sn, pol_psi);
    load_link<Real, LAYOUT, RECON, HINT>(u, gauge, V, sl, MU, pol_u);
    project<MU, SIGN>(h, psi);
    su3_mul<(SIGN > 0)>(hp, u, h);
    reconstruct_accumulate<MU, SIGN, FIRST>(acc, hp);
}

// ------------------------------------------------------------------ x hops exchanged inside the warp
// When a whole x row lives in one warp (tile x-extent == L_X, a power of two <= 32, so lane bits [0, log2 L_X) are the
// x coordinate and x+-1 wraps inside the row), the two x hops need no neighbour loads at all.  Each thread loads its OWN
// psi(s) and U_x(s) once (aligned, 21 loads instead of 42 shifted ones) and computes the two half-spinors its neighbours
// want from it:   hm = P^-_x psi(s)                (the site at x-1 multiplies it by its own U_x: forward hop there)
//                 w  = U_x(s)^dagger P^+_x psi(s)  (the complete backward-hop contribution of the site at x+1)
// and the warp rotates them by one lane with shuffles.  The arithmetic per site is the same as two hop<> calls (two
// projections, two SU(3) products), and so is the result, bit for bit; with RECON == 12 row 2 of U_x(s) is rebuilt once
// instead of twice.  Measured on 32^3x64 fp64: 0.351 -> 0.331 ms (profiles/).
__device__ __forceinline__ double shfl_(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ float shfl_(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// lanes holding the x+1 / x-1 neighbours of this thread's site (wrap inside the row segment of the warp)
__device__ __forceinline__ void x_shuffle_lanes(int LX, int& lane_fwd, int& lane_bwd) {
    const int lane = (int)(threadIdx.x & 31u), m = LX - 1;
    lane_fwd = (lane & ~m) | ((lane + 1) & m);
    lane_bwd = (lane & ~m) | ((lane - 1) & m);
}

template <typename Real, int LAYOUT, int RECON, int HINT = 0>
__device__ __forceinline__ void x_hops_shuffle(cplx<Real> (&acc)[12], const void* in, const void* gauge, unsigned V, unsigned s,
                                               int lane_fwd, int lane_bwd, uint64_t pol_psi = 0, uint64_t pol_u = 0) {
    cplx<Real> psi[12], u[9], hm[6], hq[6], w[6], hp[6];
    SpinorIO<Real, LAYOUT>::template load<HINT>(psi, in, V, s, pol_psi);
    load_link<Real, LAYOUT, RECON, HINT>(u, gauge, V, s, 0, pol_u);
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

// out(s) for the site with coordinates (x, y, z, t), s = x + L_X*(y + L_Y*(z + L_Z*t)).
// Neighbour coordinates wrap modulo L_mu (the Kronecker deltas of Eq. 1 on a periodic lattice).
// XSHFL: the x hops come from x_hops_shuffle (every lane of the warp must make the call; `active` = false lanes
// compute on a clamped site and skip the store).
template <typename Real, int LAYOUT, int RECON, int HINT = 0, bool XSHFL = false>
__device__ __forceinline__ void dslash_site(void* out, const void* in, const void* gauge, const Geom& g, int x, int y,
                                            int z, int t, unsigned s, const Policies& pol = Policies{0, 0, 0, 0},
                                            bool active = true) {
    const unsigned V = g.V;
    const unsigned sx = 1u, sy = (unsigned)g.L[0], sz = sy * (unsigned)g.L[1], st = sz * (unsigned)g.L[2];
    const unsigned xf = (x + 1 == g.L[0]) ? s - (unsigned)(g.L[0] - 1) * sx : s + sx;
    const unsigned xb = (x == 0) ? s + (unsigned)(g.L[0] - 1) * sx : s - sx;
    const unsigned yf = (y + 1 == g.L[1]) ? s - (unsigned)(g.L[1] - 1) * sy : s + sy;
    const unsigned yb = (y == 0) ? s + (unsigned)(g.L[1] - 1) * sy : s - sy;
    const unsigned zf = (z + 1 == g.L[2]) ? s - (unsigned)(g.L[2] - 1) * sz : s + sz;
    const unsigned zb = (z == 0) ? s + (unsigned)(g.L[2] - 1) * sz : s - sz;
    const unsigned tf = (t + 1 == g.L[3]) ? s - (unsigned)(g.L[3] - 1) * st : s + st;
    const unsigned tb = (t == 0) ? s + (unsigned)(g.L[3] - 1) * st : s - st;

    cplx<Real> acc[12];
    if (XSHFL) {
        int lane_fwd, lane_bwd;
        x_shuffle_lanes(g.L[0], lane_fwd, lane_bwd);
        x_hops_shuffle<Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, s, lane_fwd, lane_bwd, pol.psi, pol.u_s);
    } else {
        hop<0, -1, true, Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, xf, s, pol.psi, pol.u_s);
        hop<0, +1, false, Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, xb, xb, pol.psi, pol.u_s);
    }
    // ORDER of the sum (every tuned kernel of the library uses it, so their results are bit-identical):
    // x forward, x backward, y forward, z forward, t forward, t backward, y backward, z backward
    hop<1, -1, false, Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, yf, s, pol.psi, pol.u_s);
    hop<2, -1, false, Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, zf, s, pol.psi, pol.u_s);
    // HINT == 2: the t-direction loads bypass L1 allocation (a block's tile is one slice thick in t: no reuse inside the block)
    hop<3, -1, false, Real, LAYOUT, RECON, HINT>(acc, in, gauge, V, tf, s, pol.psi, pol.u_t);
    hop<3, +1, false, Real, LAYOUT, RECON, HINT>(acc, in, gauge, V, tb, tb, pol.psi, pol.u_t);
    hop<1, +1, false, Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, yb, yb, pol.psi, pol.u_s);
    hop<2, +1, false, Real, LAYOUT, RECON, (HINT ? 1 : 0)>(acc, in, gauge, V, zb, zb, pol.psi, pol.u_s);
    if (active) SpinorIO<Real, LAYOUT>::template store<(HINT ? 1 : 0)>(out, V, s, acc, pol.out);
}

}  // namespace dslash

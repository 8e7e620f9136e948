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

// ------------------------------------------------------------------ field access (read-only path, 128-bit where the layout allows)
// Spinor, 12 complex components of site s.
template <typename Real, int LAYOUT>
struct SpinorIO;

template <>
struct SpinorIO<double, LAYOUT_AOS> {
    __device__ __forceinline__ static void load(cplx<double> (&psi)[12], const void* base, unsigned V, unsigned s) {
        const double2* p = reinterpret_cast<const double2*>(base) + (size_t)s * 12;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            double2 v = __ldg(p + k);
            psi[k] = {v.x, v.y};
        }
    }
    __device__ __forceinline__ static void store(void* base, unsigned V, unsigned s, const cplx<double> (&psi)[12]) {
        double2* p = reinterpret_cast<double2*>(base) + (size_t)s * 12;
#pragma unroll
        for (int k = 0; k < 12; ++k) p[k] = make_double2(psi[k].re, psi[k].im);
    }
};
template <>
struct SpinorIO<double, LAYOUT_SOA> {
    __device__ __forceinline__ static void load(cplx<double> (&psi)[12], const void* base, unsigned V, unsigned s) {
        const double2* p = reinterpret_cast<const double2*>(base) + s;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            double2 v = __ldg(p + (size_t)k * V);
            psi[k] = {v.x, v.y};
        }
    }
    __device__ __forceinline__ static void store(void* base, unsigned V, unsigned s, const cplx<double> (&psi)[12]) {
        double2* p = reinterpret_cast<double2*>(base) + s;
#pragma unroll
        for (int k = 0; k < 12; ++k) p[(size_t)k * V] = make_double2(psi[k].re, psi[k].im);
    }
};
template <>
struct SpinorIO<float, LAYOUT_AOS> {
    __device__ __forceinline__ static void load(cplx<float> (&psi)[12], const void* base, unsigned V, unsigned s) {
        const float4* p = reinterpret_cast<const float4*>(base) + (size_t)s * 6;
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            float4 v = __ldg(p + q);
            psi[2 * q] = {v.x, v.y};
            psi[2 * q + 1] = {v.z, v.w};
        }
    }
    __device__ __forceinline__ static void store(void* base, unsigned V, unsigned s, const cplx<float> (&psi)[12]) {
        float4* p = reinterpret_cast<float4*>(base) + (size_t)s * 6;
#pragma unroll
        for (int q = 0; q < 6; ++q) p[q] = make_float4(psi[2 * q].re, psi[2 * q].im, psi[2 * q + 1].re, psi[2 * q + 1].im);
    }
};
template <>
struct SpinorIO<float, LAYOUT_SOA> {
    __device__ __forceinline__ static void load(cplx<float> (&psi)[12], const void* base, unsigned V, unsigned s) {
        const float4* p = reinterpret_cast<const float4*>(base) + s;
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            float4 v = __ldg(p + (size_t)q * V);
            psi[2 * q] = {v.x, v.y};
            psi[2 * q + 1] = {v.z, v.w};
        }
    }
    __device__ __forceinline__ static void store(void* base, unsigned V, unsigned s, const cplx<float> (&psi)[12]) {
        float4* p = reinterpret_cast<float4*>(base) + s;
#pragma unroll
        for (int q = 0; q < 6; ++q)
            p[(size_t)q * V] = make_float4(psi[2 * q].re, psi[2 * q].im, psi[2 * q + 1].re, psi[2 * q + 1].im);
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

// Link U_mu(s): 9 complex entries u[row*3+col]; with RECON == 12 only rows 0,1 are stored and row 2
// is rebuilt as conj(row0 x row1) (exact for SU(3), DESIGN.md Reading R14).
template <typename Real, int LAYOUT, int RECON>
__device__ __forceinline__ void load_link(cplx<Real> (&u)[9], const void* base, unsigned V, unsigned s, int mu) {
    using V2 = typename vec2<Real>::type;
    constexpr int R = (RECON == 12) ? 6 : 9;
    const V2* p = reinterpret_cast<const V2*>(base);
    if (LAYOUT == LAYOUT_AOS) {
        p += (size_t)(s * 4u + (unsigned)mu) * R;
#pragma unroll
        for (int e = 0; e < R; ++e) {
            V2 v = __ldg(p + e);
            u[e] = {v.x, v.y};
        }
    } else {
        p += (size_t)(mu * R) * V + s;
#pragma unroll
        for (int e = 0; e < R; ++e) {
            V2 v = __ldg(p + (size_t)e * V);
            u[e] = {v.x, v.y};
        }
    }
    if (RECON == 12) {
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
}

// ------------------------------------------------------------------ spin projection / reconstruction
// SIGN = -1: (1 - gamma_MU)  (forward hop);  SIGN = +1: (1 + gamma_MU)  (backward hop).
// h[0..2] = kept row 0, h[3..5] = kept row 1 (colour index fastest).
template <int MU, int SIGN, typename Real>
__device__ __forceinline__ void project(cplx<Real> (&h)[6], const cplx<Real> (&psi)[12]) {
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
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cplx<Real> h0 = h[c], h1 = h[3 + c];
        cplx<Real> r2, r3;
        const cplx<Real> zero = {Real(0), Real(0)};
        if (MU == 0) {
            r2 = (SIGN < 0) ? c_add_i(zero, h1) : c_sub_i(zero, h1);
            r3 = (SIGN < 0) ? c_add_i(zero, h0) : c_sub_i(zero, h0);
        } else if (MU == 1) {
            r2 = (SIGN < 0) ? c_sub(zero, h1) : h1;
            r3 = (SIGN < 0) ? h0 : c_sub(zero, h0);
        } else if (MU == 2) {
            r2 = (SIGN < 0) ? c_add_i(zero, h0) : c_sub_i(zero, h0);
            r3 = (SIGN < 0) ? c_sub_i(zero, h1) : c_add_i(zero, h1);
        } else {
            r2 = (SIGN < 0) ? c_sub(zero, h0) : h0;
            r3 = (SIGN < 0) ? c_sub(zero, h1) : h1;
        }
        if (FIRST) {
            acc[c] = h0;
            acc[3 + c] = h1;
            acc[6 + c] = r2;
            acc[9 + c] = r3;
        } else {
            acc[c] = c_add(acc[c], h0);
            acc[3 + c] = c_add(acc[3 + c], h1);
            acc[6 + c] = c_add(acc[6 + c], r2);
            acc[9 + c] = c_add(acc[9 + c], r3);
        }
    }
}

// hp = U h (DAGGER = false) or U^dagger h (DAGGER = true), both spin rows.
template <bool DAGGER, typename Real>
__device__ __forceinline__ void su3_mul(cplx<Real> (&hp)[6], const cplx<Real> (&u)[9], const cplx<Real> (&h)[6]) {
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
template <int MU, int SIGN, bool FIRST, typename Real, int LAYOUT, int RECON>
__device__ __forceinline__ void hop(cplx<Real> (&acc)[12], const void* in, const void* gauge, unsigned V, unsigned sn,
                                    unsigned sl) {
    cplx<Real> psi[12], h[6], hp[6], u[9];
    SpinorIO<Real, LAYOUT>::load(psi, in, V, sn);
    load_link<Real, LAYOUT, RECON>(u, gauge, V, sl, MU);
    project<MU, SIGN>(h, psi);
    su3_mul<(SIGN > 0)>(hp, u, h);
    reconstruct_accumulate<MU, SIGN, FIRST>(acc, hp);
}

// out(s) for the site with coordinates (x, y, z, t), s = x + L_X*(y + L_Y*(z + L_Z*t)).
// Neighbour coordinates wrap modulo L_mu (the Kronecker deltas of Eq. 1 on a periodic lattice).
template <typename Real, int LAYOUT, int RECON>
__device__ __forceinline__ void dslash_site(void* out, const void* in, const void* gauge, const Geom& g, int x, int y,
                                            int z, int t, unsigned s) {
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
    hop<0, -1, true, Real, LAYOUT, RECON>(acc, in, gauge, V, xf, s);
    hop<0, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, xb, xb);
    hop<1, -1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, yf, s);
    hop<1, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, yb, yb);
    hop<2, -1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, zf, s);
    hop<2, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, zb, zb);
    hop<3, -1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, tf, s);
    hop<3, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, tb, tb);
    SpinorIO<Real, LAYOUT>::store(out, V, s, acc);
}

}  // namespace dslash

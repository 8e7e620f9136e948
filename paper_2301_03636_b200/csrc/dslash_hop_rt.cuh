// dslash_hop_rt.cuh -- one hop of Eq. 1 with a RUN-TIME projector sign, shared by the operator kernels
// around Dslash (dslash_ops.cu: D, D^dagger, M, M^dagger; dslash_eo.cu: the checkerboarded D_eo / D_oe).
// The sign enters the projection and the reconstruction as the multiplier of an FMA: a + s*b costs what a + b costs and
// is bit-identical for s = +-1.
#pragma once
#include "dslash_site.cuh"

namespace dslash {

// h = P psi for the projector (1 + s*gamma_MU), s = +-1
template <int MU, typename Real>
__device__ __forceinline__ void project_rt(cplx<Real> (&h)[6], const cplx<Real> (&psi)[12], Real s) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cplx<Real> p0 = psi[c], p1 = psi[3 + c], p2 = psi[6 + c], p3 = psi[9 + c];
        if (MU == 0) {          // h0 = p0 + s i p3, h1 = p1 + s i p2
            h[c] = {fma_(-s, p3.im, p0.re), fma_(s, p3.re, p0.im)};
            h[3 + c] = {fma_(-s, p2.im, p1.re), fma_(s, p2.re, p1.im)};
        } else if (MU == 1) {   // h0 = p0 - s p3, h1 = p1 + s p2
            h[c] = {fma_(-s, p3.re, p0.re), fma_(-s, p3.im, p0.im)};
            h[3 + c] = {fma_(s, p2.re, p1.re), fma_(s, p2.im, p1.im)};
        } else if (MU == 2) {   // h0 = p0 + s i p2, h1 = p1 - s i p3
            h[c] = {fma_(-s, p2.im, p0.re), fma_(s, p2.re, p0.im)};
            h[3 + c] = {fma_(s, p3.im, p1.re), fma_(-s, p3.re, p1.im)};
        } else {                // h0 = p0 + s p2, h1 = p1 + s p3
            h[c] = {fma_(s, p2.re, p0.re), fma_(s, p2.im, p0.im)};
            h[3 + c] = {fma_(s, p3.re, p1.re), fma_(s, p3.im, p1.im)};
        }
    }
}

// acc += R(h): rows 0,1 += h0,h1; rows 2,3 from the projector (1 + s*gamma_MU):
//   MU 0: r2 = -s i h1, r3 = -s i h0    MU 1: r2 = s h1, r3 = -s h0    MU 2: r2 = -s i h0, r3 = s i h1    MU 3: r2 = s h0, r3 = s h1
template <int MU, typename Real>
__device__ __forceinline__ void reconstruct_accumulate_rt(cplx<Real> (&acc)[12], const cplx<Real> (&h)[6], Real s) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cplx<Real> h0 = h[c], h1 = h[3 + c];
        cplx<Real> a2 = acc[6 + c], a3 = acc[9 + c];
        if (MU == 0) {
            a2 = {fma_(s, h1.im, a2.re), fma_(-s, h1.re, a2.im)};
            a3 = {fma_(s, h0.im, a3.re), fma_(-s, h0.re, a3.im)};
        } else if (MU == 1) {
            a2 = {fma_(s, h1.re, a2.re), fma_(s, h1.im, a2.im)};
            a3 = {fma_(-s, h0.re, a3.re), fma_(-s, h0.im, a3.im)};
        } else if (MU == 2) {
            a2 = {fma_(s, h0.im, a2.re), fma_(-s, h0.re, a2.im)};
            a3 = {fma_(-s, h1.im, a3.re), fma_(s, h1.re, a3.im)};
        } else {
            a2 = {fma_(s, h0.re, a2.re), fma_(s, h0.im, a2.im)};
            a3 = {fma_(s, h1.re, a3.re), fma_(s, h1.im, a3.im)};
        }
        acc[6 + c] = a2;
        acc[9 + c] = a3;
        acc[c] = c_add(acc[c], h0);
        acc[3 + c] = c_add(acc[3 + c], h1);
    }
}

template <int MU, bool UDAG, typename Real, int LAYOUT, int RECON>
__device__ __forceinline__ void hop_rt(cplx<Real> (&acc)[12], const void* in, const void* gauge, unsigned V, unsigned sn, unsigned sl,
                                       Real s) {
    cplx<Real> psi[12], h[6], hp[6], u[9];
    SpinorIO<Real, LAYOUT>::load(psi, in, V, sn);
    load_link<Real, LAYOUT, RECON>(u, gauge, V, sl, MU);
    project_rt<MU>(h, psi, s);
    su3_mul<UDAG>(hp, u, h);
    reconstruct_accumulate_rt<MU>(acc, hp, s);
}

}  // namespace dslash

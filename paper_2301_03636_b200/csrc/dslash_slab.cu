// dslash_slab.cu -- the kernels of the multi-GPU T-slab form of Eq. 1 (the paper's future work,
// PAPER.md:253, :346): spin-projected half-spinor faces and the boundary slices that consume them.
//
// A rank owns lt consecutive time slices of the global lattice (its ctx is created with dims {L_X, L_Y, L_Z, lt}); fields
// carry NO ghost slices.  Of the eight hops of Eq. 1 only two leave the slab:
//   the forward t hop of the last slice   (1 - g_t) U_t(x, lt-1) psi(x, lt)      needs psi of the rank ABOVE,
//   the backward t hop of the first slice (1 + g_t) U_t(x, -1)^dagger psi(x, -1) needs psi AND U_t of the rank BELOW.
// Both projectors have rank 2, so what travels is a half-spinor (6 complex numbers per site instead of 12):
//   face DOWN (to the rank below)  h(x) = P^-_t psi(x, 0)                         -- the receiver multiplies by its own U_t
//   face UP   (to the rank above)  w(x) = U_t(x, lt-1)^dagger P^+_t psi(x, lt-1)  -- already multiplied: links never travel
// (3.1 MB per face at 32^3 fp64).  dslash_slab_pack_faces writes both; the interior slices 1 .. lt-2 are computed by the
// direct kernel while the faces are in flight; dslash_slab_boundary computes slices 0 and lt-1 with the received faces.
// The arithmetic per hop and the order of the sum are those of dslash_site.cuh, merely split between two ranks: the result
// is bit-identical to the single-GPU kernels.
//
// Face layout (opaque to the caller, the same on sender and receiver): the native layout of the ctx restricted to one time
// slice and six components -- blocked SoA: vec2[(v * 6 + k) * 32 + l] with v, l of the site's index inside the slice
// (a slice is padded up to whole vectors); AoS: vec2[site * 6 + k].
#include "dslash_kernels.cuh"

namespace dslash {

namespace {

template <typename Real, int LAYOUT>
__device__ __forceinline__ size_t face_index(unsigned ss, int k) {
    return LAYOUT == LAYOUT_AOS ? (size_t)ss * 6u + (unsigned)k : (size_t)(ss >> VL_LOG2) * (6u * VL) + (unsigned)k * VL + (ss & (VL - 1u));
}
template <typename Real, int LAYOUT>
__device__ __forceinline__ void store_face(void* face, unsigned ss, const cplx<Real> (&h)[6]) {
    using V2 = typename vec2<Real>::type;
    V2* p = reinterpret_cast<V2*>(face);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        V2 v;
        v.x = h[k].re;
        v.y = h[k].im;
        p[face_index<Real, LAYOUT>(ss, k)] = v;
    }
}
template <typename Real, int LAYOUT>
__device__ __forceinline__ void load_face(cplx<Real> (&h)[6], const void* face, unsigned ss) {
    using V2 = typename vec2<Real>::type;
    const V2* p = reinterpret_cast<const V2*>(face);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const V2 v = p[face_index<Real, LAYOUT>(ss, k)];
        h[k] = {v.x, v.y};
    }
}

// blockIdx.y = 0: face DOWN from slice 0; 1: face UP from slice lt-1.  One thread per site of the slice.
template <typename Real, int LAYOUT, int RECON>
__global__ void __launch_bounds__(128) slab_pack_faces_kernel(void* __restrict__ face_down, void* __restrict__ face_up,
                                                              const void* __restrict__ in, const void* __restrict__ gauge, Geom g) {
    const unsigned slice = (unsigned)g.L[0] * (unsigned)g.L[1] * (unsigned)g.L[2];
    const unsigned ss = blockIdx.x * blockDim.x + threadIdx.x;
    if (ss >= slice) return;
    cplx<Real> psi[12], h[6];
    if (blockIdx.y == 0) {
        SpinorIO<Real, LAYOUT>::load(psi, in, g.V, ss);
        project<3, -1>(h, psi);
        store_face<Real, LAYOUT>(face_down, ss, h);
    } else {
        const unsigned s = ss + slice * (unsigned)(g.L[3] - 1);
        cplx<Real> u[9], w[6];
        SpinorIO<Real, LAYOUT>::load(psi, in, g.V, s);
        load_link<Real, LAYOUT, RECON>(u, gauge, g.V, s, 3);
        project<3, +1>(h, psi);
        su3_mul<true>(w, u, h);
        store_face<Real, LAYOUT>(face_up, ss, w);
    }
}

// Slices 0 and lt-1 (blockIdx.y; one slice if lt == 1).  The hops that stay inside the slab are those of dslash_site(); the
// two that leave it take their half-spinor from the received faces.  Same order of the sum as dslash_site().
template <typename Real, int LAYOUT, int RECON>
__global__ void __launch_bounds__(128, 2)
    slab_boundary_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge,
                         const void* __restrict__ face_from_below, const void* __restrict__ face_from_above, Geom g) {
    const unsigned slice = (unsigned)g.L[0] * (unsigned)g.L[1] * (unsigned)g.L[2];
    const unsigned ss = blockIdx.x * blockDim.x + threadIdx.x;
    if (ss >= slice) return;
    const int t = blockIdx.y == 0 ? 0 : g.L[3] - 1;
    const int x = (int)(ss % (unsigned)g.L[0]);
    const int y = (int)((ss / (unsigned)g.L[0]) % (unsigned)g.L[1]);
    const int z = (int)(ss / ((unsigned)g.L[0] * (unsigned)g.L[1]));
    const unsigned V = g.V, s = ss + slice * (unsigned)t;
    const unsigned sy = (unsigned)g.L[0], sz = sy * (unsigned)g.L[1];
    const unsigned xf = (x + 1 == g.L[0]) ? s - (unsigned)(g.L[0] - 1) : s + 1u;
    const unsigned xb = (x == 0) ? s + (unsigned)(g.L[0] - 1) : s - 1u;
    const unsigned yf = (y + 1 == g.L[1]) ? s - (unsigned)(g.L[1] - 1) * sy : s + sy;
    const unsigned yb = (y == 0) ? s + (unsigned)(g.L[1] - 1) * sy : s - sy;
    const unsigned zf = (z + 1 == g.L[2]) ? s - (unsigned)(g.L[2] - 1) * sz : s + sz;
    const unsigned zb = (z == 0) ? s + (unsigned)(g.L[2] - 1) * sz : s - sz;
    cplx<Real> acc[12];
    hop<0, -1, true, Real, LAYOUT, RECON>(acc, in, gauge, V, xf, s);
    hop<0, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, xb, xb);
    hop<1, -1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, yf, s);
    hop<2, -1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, zf, s);
    if (t == g.L[3] - 1) {  // forward t hop across the upper slab boundary: P^-_t psi(x, lt) arrived as the face from above
        cplx<Real> h[6], hp[6], u[9];
        load_face<Real, LAYOUT>(h, face_from_above, ss);
        load_link<Real, LAYOUT, RECON>(u, gauge, V, s, 3);
        su3_mul<false>(hp, u, h);
        reconstruct_accumulate<3, -1, false>(acc, hp);
    } else {
        hop<3, -1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, s + slice, s);
    }
    if (t == 0) {  // backward t hop across the lower boundary: U_t^dagger P^+_t psi(x, -1) arrived complete as the face from below
        cplx<Real> w[6];
        load_face<Real, LAYOUT>(w, face_from_below, ss);
        reconstruct_accumulate<3, +1, false>(acc, w);
    } else {
        hop<3, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, s - slice, s - slice);
    }
    hop<1, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, yb, yb);
    hop<2, +1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, zb, zb);
    SpinorIO<Real, LAYOUT>::store(out, V, s, acc);
}

template <typename Real, int LAYOUT, int RECON>
cudaError_t launch_slab_t(int which, void* a0, void* a1, const void* in, const void* gauge, const void* f0, const void* f1, const Geom& g,
                          cudaStream_t st) {
    const unsigned slice = (unsigned)g.L[0] * (unsigned)g.L[1] * (unsigned)g.L[2];
    const dim3 grid((slice + 127u) / 128u, (which == 0 || g.L[3] > 1) ? 2u : 1u);
    if (which == 0)
        slab_pack_faces_kernel<Real, LAYOUT, RECON><<<grid, 128, 0, st>>>(a0, a1, in, gauge, g);
    else
        slab_boundary_kernel<Real, LAYOUT, RECON><<<grid, 128, 0, st>>>(a0, in, gauge, f0, f1, g);
    return cudaGetLastError();
}

template <typename Real>
cudaError_t launch_slab_p(int layout_base, int recon, int which, void* a0, void* a1, const void* in, const void* gauge, const void* f0,
                          const void* f1, const Geom& g, cudaStream_t st) {
    if (layout_base == LAYOUT_AOS)
        return recon == 12 ? launch_slab_t<Real, LAYOUT_AOS, 12>(which, a0, a1, in, gauge, f0, f1, g, st)
                           : launch_slab_t<Real, LAYOUT_AOS, 18>(which, a0, a1, in, gauge, f0, f1, g, st);
    return recon == 12 ? launch_slab_t<Real, LAYOUT_SOA, 12>(which, a0, a1, in, gauge, f0, f1, g, st)
                       : launch_slab_t<Real, LAYOUT_SOA, 18>(which, a0, a1, in, gauge, f0, f1, g, st);
}

}  // namespace

cudaError_t launch_slab_pack_faces(int precision, int layout_base, int recon, void* face_down, void* face_up, const void* in,
                                   const void* gauge, const Geom& g, cudaStream_t st) {
    return precision == 0 ? launch_slab_p<double>(layout_base, recon, 0, face_down, face_up, in, gauge, nullptr, nullptr, g, st)
                          : launch_slab_p<float>(layout_base, recon, 0, face_down, face_up, in, gauge, nullptr, nullptr, g, st);
}

cudaError_t launch_slab_boundary(int precision, int layout_base, int recon, void* out, const void* in, const void* gauge,
                                 const void* face_from_below, const void* face_from_above, const Geom& g, cudaStream_t st) {
    return precision == 0 ? launch_slab_p<double>(layout_base, recon, 1, out, nullptr, in, gauge, face_from_below, face_from_above, g, st)
                          : launch_slab_p<float>(layout_base, recon, 1, out, nullptr, in, gauge, face_from_below, face_from_above, g, st);
}

}  // namespace dslash

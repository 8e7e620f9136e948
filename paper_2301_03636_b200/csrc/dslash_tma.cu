// dslash_tma.cu -- TMA-staged Dslash kernel for sm_100a (blocked SoA layout).
//
// The thread block covers a 4-D tile of T sites whose x-extent is a multiple of 32, so the tile is a whole
// number of the layout's 32-site vectors (one vector per warp).  Lane 0 of every warp issues two bulk
// asynchronous copies (cp.async.bulk.shared::cluster.global, SASS UBLKCP -- the TMA unit) that bring its
// vector's own spinors (12 complex per site, 6 KB in fp64) and own links (4 x 9 or 4 x 6 complex per site,
// 18 or 12 KB) into shared memory in exactly the global vector format; completion is counted on one
// mbarrier.  While those bytes are in flight every thread works off the hops whose neighbour lies outside
// the tile ("halo hops": spinor and link read from global memory through L2), then waits on the mbarrier
// and does the in-tile hops entirely from shared memory: psi(x+-mu) and the backward link U_mu(x-mu) are the
// tile's own data at the neighbouring thread's slot.  Per site the SM pulls
//     (24 + 4*2R) reals once  +  halo ~ sum_mu 1/b_mu * (2*24 + 2R + 2R) reals
// through L2 instead of 8 spinors + 8 links, and none of the own-tile bytes is staged through registers.
// See DESIGN.md section 6 for why this is NOT the default on 32^3x64 (shared memory caps the block at one
// thread per 768 bytes, i.e. <= 9 warps per SM, and the kernel becomes issue-latency bound).
//
// Operator and conventions: PAPER.md:47-54 (Eq. 1) as read in DESIGN.md section 2; same per-hop arithmetic as
// dslash_site.cuh (project -> SU(3) multiply -> reconstruct/accumulate), only the order of the 8 hops
// differs from thread to thread (halo hops first).
#include "dslash_async.cuh"
#include "dslash_kernels.cuh"

namespace dslash {

template <typename Real, int RECON>
__device__ __forceinline__ void load_link_smem(cplx<Real> (&u)[9], const void* base, unsigned ls, int mu) {
    using V2 = typename vec2<Real>::type;
    constexpr unsigned R = (RECON == 12) ? 6u : 9u;
    const V2* p = reinterpret_cast<const V2*>(base) + (size_t)((ls >> VL_LOG2) * 4u + (unsigned)mu) * (R * VL) + (ls & (VL - 1u));
#pragma unroll
    for (int e = 0; e < (int)R; ++e) {
        V2 v = p[e * VL];
        u[e] = {v.x, v.y};
    }
    if (RECON == 12) {
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int j1 = (j + 1) % 3, j2 = (j + 2) % 3;
            cplx<Real> a = c_mul(u[j1], u[3 + j2]);
            Real re = fma_(-u[j2].re, u[3 + j1].re, a.re);
            re = fma_(u[j2].im, u[3 + j1].im, re);
            Real im = fma_(-u[j2].re, u[3 + j1].im, a.im);
            im = fma_(-u[j2].im, u[3 + j1].re, im);
            u[6 + j] = {re, -im};
        }
    }
}

// in-tile hop: neighbour spinor at local slot ln, link at local slot ll (both in shared memory)
template <int MU, int SIGN, typename Real, int RECON>
__device__ __forceinline__ void hop_smem(cplx<Real> (&acc)[12], const void* psi_s, const void* u_s, unsigned ln, unsigned ll) {
    cplx<Real> psi[12], h[6], hp[6], u[9];
    load_spinor_smem(psi, psi_s, ln);
    load_link_smem<Real, RECON>(u, u_s, ll, MU);
    project<MU, SIGN>(h, psi);
    su3_mul<(SIGN > 0)>(hp, u, h);
    reconstruct_accumulate<MU, SIGN, false>(acc, hp);
}

template <typename Real, int RECON>
__global__ void __launch_bounds__(128, 2)
    dslash_tma_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, const Geom g,
                      const TileGeom tg) {
    constexpr unsigned PSI_VEC_BYTES = 24u * VL * sizeof(Real);                          // one vector of spinors
    constexpr unsigned U_VEC_BYTES = 4u * (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);  // one vector of links
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned T = blockDim.x;
    const unsigned nvec = T >> VL_LOG2;
    unsigned char* psi_s = smem;
    unsigned char* u_s = smem + nvec * PSI_VEC_BYTES;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + nvec * (PSI_VEC_BYTES + U_VEC_BYTES));

    // tile origin
    unsigned b = blockIdx.x;
    const unsigned tbx = b % (unsigned)tg.nt[0];
    b /= (unsigned)tg.nt[0];
    const unsigned tby = b % (unsigned)tg.nt[1];
    b /= (unsigned)tg.nt[1];
    const unsigned tbz = b % (unsigned)tg.nt[2];
    const unsigned tbt = b / (unsigned)tg.nt[2];
    const int x0 = (int)(tbx << tg.lb[0]), y0 = (int)(tby << tg.lb[1]), z0 = (int)(tbz << tg.lb[2]), t0 = (int)(tbt << tg.lb[3]);

    // this thread's site
    const unsigned tid = threadIdx.x;
    unsigned r = tid;
    const int lx = (int)(r & ((1u << tg.lb[0]) - 1u));
    r >>= tg.lb[0];
    const int ly = (int)(r & ((1u << tg.lb[1]) - 1u));
    r >>= tg.lb[1];
    const int lz = (int)(r & ((1u << tg.lb[2]) - 1u));
    r >>= tg.lb[2];
    const int lt = (int)r;
    const int x = x0 + lx, y = y0 + ly, z = z0 + lz, t = t0 + lt;
    // x always fits (L_X is a multiple of the tile's x-extent); a whole warp is active or inactive together
    const bool active = (y < g.L[1]) && (z < g.L[2]) && (t < g.L[3]);
    const unsigned V = g.V;
    const unsigned sy = (unsigned)g.L[0], sz = sy * (unsigned)g.L[1], st = sz * (unsigned)g.L[2];
    const unsigned s = (unsigned)x + sy * (unsigned)y + sz * (unsigned)z + st * (unsigned)t;

    // number of active warps = vectors to copy (uniform across the block)
    const unsigned rows_y = min((unsigned)(g.L[1] - y0), 1u << tg.lb[1]);
    const unsigned rows_z = min((unsigned)(g.L[2] - z0), 1u << tg.lb[2]);
    const unsigned rows_t = min((unsigned)(g.L[3] - t0), 1u << tg.lb[3]);
    const unsigned nactive_vec = (rows_y * rows_z * rows_t) << (tg.lb[0] - (int)VL_LOG2);

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) mbar_arrive_expect_tx(bar, nactive_vec * (PSI_VEC_BYTES + U_VEC_BYTES));
    __syncthreads();  // the expected byte count is armed before any copy can complete
    if (active && (tid & (VL - 1u)) == 0) {
        const unsigned lvec = tid >> VL_LOG2, gvec = s >> VL_LOG2;  // s is the first site of this warp's vector
        bulk_g2s(psi_s + lvec * PSI_VEC_BYTES, reinterpret_cast<const unsigned char*>(in) + (size_t)gvec * PSI_VEC_BYTES,
                 PSI_VEC_BYTES, bar);
        bulk_g2s(u_s + lvec * U_VEC_BYTES, reinterpret_cast<const unsigned char*>(gauge) + (size_t)gvec * U_VEC_BYTES,
                 U_VEC_BYTES, bar);
    }

    const unsigned tsy = 1u << tg.lb[0], tsz = 1u << (tg.lb[0] + tg.lb[1]), tst = 1u << (tg.lb[0] + tg.lb[1] + tg.lb[2]);
    const int bxm = (1 << tg.lb[0]) - 1, bym = (1 << tg.lb[1]) - 1, bzm = (1 << tg.lb[2]) - 1, btm = (1 << tg.lb[3]) - 1;
    // in-tile predicates: forward neighbour inside iff local+1 stays in the box and the coordinate does not wrap;
    // backward neighbour inside iff local > 0.  (A tile that spans the whole extent takes the global path at
    // the wrap, which is correct for any extent.)
    const bool in_xf = (lx < bxm) && (x + 1 < g.L[0]), in_xb = lx > 0;
    const bool in_yf = (ly < bym) && (y + 1 < g.L[1]), in_yb = ly > 0;
    const bool in_zf = (lz < bzm) && (z + 1 < g.L[2]), in_zb = lz > 0;
    const bool in_tf = (lt < btm) && (t + 1 < g.L[3]), in_tb = lt > 0;

    cplx<Real> acc[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) acc[k] = {Real(0), Real(0)};

    if (active) {
        // ---- pass 1: halo hops from global memory (overlaps the bulk copies)
        const unsigned xf = (x + 1 == g.L[0]) ? s - (unsigned)(g.L[0] - 1) : s + 1u;
        const unsigned xb = (x == 0) ? s + (unsigned)(g.L[0] - 1) : s - 1u;
        const unsigned yf = (y + 1 == g.L[1]) ? s - (unsigned)(g.L[1] - 1) * sy : s + sy;
        const unsigned yb = (y == 0) ? s + (unsigned)(g.L[1] - 1) * sy : s - sy;
        const unsigned zf = (z + 1 == g.L[2]) ? s - (unsigned)(g.L[2] - 1) * sz : s + sz;
        const unsigned zb = (z == 0) ? s + (unsigned)(g.L[2] - 1) * sz : s - sz;
        const unsigned tf = (t + 1 == g.L[3]) ? s - (unsigned)(g.L[3] - 1) * st : s + st;
        const unsigned tb = (t == 0) ? s + (unsigned)(g.L[3] - 1) * st : s - st;
        if (!in_tf) hop<3, -1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, tf, s);
        if (!in_tb) hop<3, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, tb, tb);
        if (!in_zf) hop<2, -1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, zf, s);
        if (!in_zb) hop<2, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, zb, zb);
        if (!in_yf) hop<1, -1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, yf, s);
        if (!in_yb) hop<1, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, yb, yb);
        if (!in_xf) hop<0, -1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, xf, s);
        if (!in_xb) hop<0, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, xb, xb);
    }

    // ---- the tile's own spinors and links have landed
    mbar_wait(bar, 0);

    if (active) {
        // ---- pass 2: in-tile hops from shared memory
        if (in_xf) hop_smem<0, -1, Real, RECON>(acc, psi_s, u_s, tid + 1u, tid);
        if (in_xb) hop_smem<0, +1, Real, RECON>(acc, psi_s, u_s, tid - 1u, tid - 1u);
        if (in_yf) hop_smem<1, -1, Real, RECON>(acc, psi_s, u_s, tid + tsy, tid);
        if (in_yb) hop_smem<1, +1, Real, RECON>(acc, psi_s, u_s, tid - tsy, tid - tsy);
        if (in_zf) hop_smem<2, -1, Real, RECON>(acc, psi_s, u_s, tid + tsz, tid);
        if (in_zb) hop_smem<2, +1, Real, RECON>(acc, psi_s, u_s, tid - tsz, tid - tsz);
        if (in_tf) hop_smem<3, -1, Real, RECON>(acc, psi_s, u_s, tid + tst, tid);
        if (in_tb) hop_smem<3, +1, Real, RECON>(acc, psi_s, u_s, tid - tst, tid - tst);
        SpinorIO<Real, LAYOUT_SOA>::store(out, V, s, acc);
    }
}

// ------------------------------------------------------------------ links-only staging ("TMA-lite")
// Only the tile's own links U_mu(x) (60 % of the compulsory bytes, used by the four forward hops) are bulk-copied to
// shared memory.  All spinors and the backward links are gathered from global memory in straight-line code exactly as in
// the direct kernel (so the compiler keeps overlapping the loads of the next hop with the arithmetic of the current one),
// but the four backward hops run first and the four forward hops -- which need no register-staged link loads any more --
// run after the mbarrier wait.  36 of the 168 register-staged 16-byte loads per site disappear and their DRAM latency is
// taken by the TMA unit instead of by a warp.
template <int MU, typename Real, int RECON>
__device__ __forceinline__ void hop_fwd_smemlink(cplx<Real> (&acc)[12], const void* in, const void* u_s, unsigned V, unsigned sn,
                                                 unsigned ltid) {
    cplx<Real> psi[12], h[6], hp[6], u[9];
    SpinorIO<Real, LAYOUT_SOA>::load(psi, in, V, sn);
    load_link_smem<Real, RECON>(u, u_s, ltid, MU);
    project<MU, -1>(h, psi);
    su3_mul<false>(hp, u, h);
    reconstruct_accumulate<MU, -1, false>(acc, hp);
}

template <typename Real, int RECON>
__global__ void __launch_bounds__(128, 2)
    dslash_tma_links_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, const Geom g,
                            const TileGeom tg) {
    constexpr unsigned U_VEC_BYTES = 4u * (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned T = blockDim.x;
    const unsigned nvec = T >> VL_LOG2;
    unsigned char* u_s = smem;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + nvec * U_VEC_BYTES);

    unsigned b = blockIdx.x;
    const unsigned tbx = b % (unsigned)tg.nt[0];
    b /= (unsigned)tg.nt[0];
    const unsigned tby = b % (unsigned)tg.nt[1];
    b /= (unsigned)tg.nt[1];
    const unsigned tbz = b % (unsigned)tg.nt[2];
    const unsigned tbt = b / (unsigned)tg.nt[2];
    const int x0 = (int)(tbx << tg.lb[0]), y0 = (int)(tby << tg.lb[1]), z0 = (int)(tbz << tg.lb[2]), t0 = (int)(tbt << tg.lb[3]);
    const unsigned tid = threadIdx.x;
    unsigned r = tid;
    const int x = x0 + (int)(r & ((1u << tg.lb[0]) - 1u));
    r >>= tg.lb[0];
    const int y = y0 + (int)(r & ((1u << tg.lb[1]) - 1u));
    r >>= tg.lb[1];
    const int z = z0 + (int)(r & ((1u << tg.lb[2]) - 1u));
    r >>= tg.lb[2];
    const int t = t0 + (int)r;
    const bool active = (y < g.L[1]) && (z < g.L[2]) && (t < g.L[3]);
    const unsigned V = g.V;
    const unsigned sy = (unsigned)g.L[0], sz = sy * (unsigned)g.L[1], st = sz * (unsigned)g.L[2];
    const unsigned s = (unsigned)x + sy * (unsigned)y + sz * (unsigned)z + st * (unsigned)t;

    const unsigned rows_y = min((unsigned)(g.L[1] - y0), 1u << tg.lb[1]);
    const unsigned rows_z = min((unsigned)(g.L[2] - z0), 1u << tg.lb[2]);
    const unsigned rows_t = min((unsigned)(g.L[3] - t0), 1u << tg.lb[3]);
    const unsigned nactive_vec = (rows_y * rows_z * rows_t) << (tg.lb[0] - (int)VL_LOG2);

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) mbar_arrive_expect_tx(bar, nactive_vec * U_VEC_BYTES);
    __syncthreads();
    if (active && (tid & (VL - 1u)) == 0)
        bulk_g2s(u_s + (tid >> VL_LOG2) * U_VEC_BYTES,
                 reinterpret_cast<const unsigned char*>(gauge) + (size_t)(s >> VL_LOG2) * U_VEC_BYTES, U_VEC_BYTES, bar);

    cplx<Real> acc[12];
    if (active) {
        const unsigned xf = (x + 1 == g.L[0]) ? s - (unsigned)(g.L[0] - 1) : s + 1u;
        const unsigned xb = (x == 0) ? s + (unsigned)(g.L[0] - 1) : s - 1u;
        const unsigned yf = (y + 1 == g.L[1]) ? s - (unsigned)(g.L[1] - 1) * sy : s + sy;
        const unsigned yb = (y == 0) ? s + (unsigned)(g.L[1] - 1) * sy : s - sy;
        const unsigned zf = (z + 1 == g.L[2]) ? s - (unsigned)(g.L[2] - 1) * sz : s + sz;
        const unsigned zb = (z == 0) ? s + (unsigned)(g.L[2] - 1) * sz : s - sz;
        const unsigned tf = (t + 1 == g.L[3]) ? s - (unsigned)(g.L[3] - 1) * st : s + st;
        const unsigned tb = (t == 0) ? s + (unsigned)(g.L[3] - 1) * st : s - st;
        // backward hops: everything from global memory
        hop<3, +1, true, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, tb, tb);
        hop<2, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, zb, zb);
        hop<1, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, yb, yb);
        hop<0, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, xb, xb);
        mbar_wait(bar, 0);
        // forward hops: spinor from global memory, own link from shared memory
        hop_fwd_smemlink<0, Real, RECON>(acc, in, u_s, V, xf, tid);
        hop_fwd_smemlink<1, Real, RECON>(acc, in, u_s, V, yf, tid);
        hop_fwd_smemlink<2, Real, RECON>(acc, in, u_s, V, zf, tid);
        hop_fwd_smemlink<3, Real, RECON>(acc, in, u_s, V, tf, tid);
        SpinorIO<Real, LAYOUT_SOA>::store(out, V, s, acc);
    }
}

// ------------------------------------------------------------------ host side
static size_t tma_smem_bytes(int precision, int recon, int T) {
    const size_t rb = precision == 0 ? 8u : 4u;
    return (size_t)T * 24u * rb + (size_t)T * 4u * (recon == 12 ? 12u : 18u) * rb + 16u;
}

// Can the TMA kernel run this (precision, recon, lattice, tile)?  The tile's x-extent must be a multiple of
// the 32-site vector and divide L_X (so every tile row is whole vectors), the other extents must not
// exceed the lattice, the block has 32..128 threads, and two resident blocks must fit in shared memory.
bool tma_eligible(int precision, int recon, const Geom& g, const TileGeom& tg) {
    const int T = 1 << (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]);
    if (T < 32 || T > 128) return false;
    const int bx = 1 << tg.lb[0];
    if (bx < (int)VL || g.L[0] % bx) return false;
    for (int d = 1; d < 4; ++d)
        if ((1 << tg.lb[d]) > g.L[d]) return false;
    return tma_smem_bytes(precision, recon, T) <= 113u * 1024u;
}

template <typename Real, int RECON, bool LINKS_ONLY>
static cudaError_t launch_tma_t(const LaunchArgs& a, const TileGeom& tg) {
    const int T = 1 << (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]);
    const int prec = sizeof(Real) == 8 ? 0 : 1;
    const size_t smem = LINKS_ONLY ? tma_smem_bytes(prec, RECON, T) - (size_t)T * 24u * sizeof(Real) : tma_smem_bytes(prec, RECON, T);
    auto kernel = LINKS_ONLY ? dslash_tma_links_kernel<Real, RECON> : dslash_tma_kernel<Real, RECON>;
    static bool attr_set = false;  // per template instantiation
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, LINKS_ONLY ? 75 : 100);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const unsigned grid = (unsigned)tg.nt[0] * (unsigned)tg.nt[1] * (unsigned)tg.nt[2] * (unsigned)tg.nt[3];
    kernel<<<grid, T, smem, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg);
    return cudaGetLastError();
}

cudaError_t launch_tma(int precision, int recon, const LaunchArgs& a, const TileGeom& tg, bool links_only) {
    if (links_only) {
        if (precision == 0) return recon == 12 ? launch_tma_t<double, 12, true>(a, tg) : launch_tma_t<double, 18, true>(a, tg);
        return recon == 12 ? launch_tma_t<float, 12, true>(a, tg) : launch_tma_t<float, 18, true>(a, tg);
    }
    if (precision == 0) return recon == 12 ? launch_tma_t<double, 12, false>(a, tg) : launch_tma_t<double, 18, false>(a, tg);
    return recon == 12 ? launch_tma_t<float, 12, false>(a, tg) : launch_tma_t<float, 18, false>(a, tg);
}

}  // namespace dslash

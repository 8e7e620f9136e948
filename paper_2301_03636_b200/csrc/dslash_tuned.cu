// dslash_tuned.cu -- the tuned Dslash kernel for sm_100a.
//
// One thread per site; the thread block covers a 4-D tile of sites (x fastest inside the tile) so that
// the +-mu neighbours of most sites of a block belong to the same block and their spinors / backward
// links are served from the SM's L1 instead of L2 (hard part 1).  Tiles are numbered
// x fastest, so blocks that run at the same time touch adjacent memory and the halos they share stay
// in the 126 MB L2; HBM sees each field once per application.  See DESIGN.md "Kernels".
#include "dslash_kernels.cuh"

namespace dslash {

template <typename Real, int LAYOUT, int RECON, int MAXTPB, int MINBLK>
__global__ void __launch_bounds__(MAXTPB, MINBLK)
    dslash_tuned_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, Geom g,
                        TileGeom tg) {
    // tile coordinates of this block
    unsigned b = blockIdx.x;
    const unsigned bx = b % (unsigned)tg.nt[0];
    b /= (unsigned)tg.nt[0];
    const unsigned by = b % (unsigned)tg.nt[1];
    b /= (unsigned)tg.nt[1];
    const unsigned bz = b % (unsigned)tg.nt[2];
    const unsigned bt = b / (unsigned)tg.nt[2];
    // in-tile coordinates of this thread (power-of-two tile extents)
    unsigned r = threadIdx.x;
    const int x = (int)((bx << tg.lb[0]) + (r & ((1u << tg.lb[0]) - 1u)));
    r >>= tg.lb[0];
    const int y = (int)((by << tg.lb[1]) + (r & ((1u << tg.lb[1]) - 1u)));
    r >>= tg.lb[1];
    const int z = (int)((bz << tg.lb[2]) + (r & ((1u << tg.lb[2]) - 1u)));
    r >>= tg.lb[2];
    const int t = (int)((bt << tg.lb[3]) + r);
    if (x >= g.L[0] || y >= g.L[1] || z >= g.L[2] || t >= g.L[3]) return;
    const unsigned s = (unsigned)x + (unsigned)g.L[0] * ((unsigned)y + (unsigned)g.L[1] * ((unsigned)z + (unsigned)g.L[2] * (unsigned)t));
    dslash_site<Real, LAYOUT, RECON>(out, in, gauge, g, x, y, z, t, s);
}

template <typename Real, int LAYOUT, int RECON>
static cudaError_t launch_tuned_t(const LaunchArgs& a, const TileGeom& tg) {
    const int tpb = 1 << (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]);
    const unsigned grid = (unsigned)tg.nt[0] * (unsigned)tg.nt[1] * (unsigned)tg.nt[2] * (unsigned)tg.nt[3];
    if (tpb <= 128)
        dslash_tuned_kernel<Real, LAYOUT, RECON, 128, 3><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg);
    else if (tpb <= 256)
        dslash_tuned_kernel<Real, LAYOUT, RECON, 256, 1><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg);
    else if (tpb <= 512)
        dslash_tuned_kernel<Real, LAYOUT, RECON, 512, 1><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg);
    else
        dslash_tuned_kernel<Real, LAYOUT, RECON, 1024, 1><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg);
    return cudaGetLastError();
}

template <typename Real>
static cudaError_t launch_tuned_p(int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg) {
    if (layout_base == LAYOUT_AOS)
        return recon == 12 ? launch_tuned_t<Real, LAYOUT_AOS, 12>(a, tg) : launch_tuned_t<Real, LAYOUT_AOS, 18>(a, tg);
    return recon == 12 ? launch_tuned_t<Real, LAYOUT_SOA, 12>(a, tg) : launch_tuned_t<Real, LAYOUT_SOA, 18>(a, tg);
}

cudaError_t launch_tuned(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg) {
    return precision == 0 ? launch_tuned_p<double>(layout_base, recon, a, tg) : launch_tuned_p<float>(layout_base, recon, a, tg);
}

}  // namespace dslash

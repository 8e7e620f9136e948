// dslash_tuned.cu -- the direct (register-staged) tuned Dslash kernel for sm_100a.
//
// One thread per site; the thread block covers a 4-D tile of sites (x fastest inside the tile).  Tiles are
// numbered x fastest, so blocks that run at the same time touch adjacent memory and the halos they share
// stay in the 126 MB L2; HBM sees each field about once per application (profiles/r01_ncu_tuned_kernel.txt: 1.01x).
// With the blocked SoA layout the 12 (9) loads of a spinor (link) share one base address, which took the
// kernel from ~2100 to ~1500 SASS instructions per site -- that matters because under sustained load the
// B200 runs this kernel against its 1 kW power cap (SM clock ~1.4 GHz), not against a fixed clock.
//
// Options (dslash_set_option; both measured as no gain on 32^3x64 and left off by default):
//   OCCUPANCY 1 / 2   compile-time variants for blocks of <= 128 threads: 1 = 128 registers (16 warps per SM),
//                     2 = 255 registers (8 warps per SM, deeper load hoisting); 0 = 168 registers (12 warps).
//   L2_POLICY bits    per-access L2 eviction policies (createpolicy + ld/st .L2::cache_hint): 1 spinor loads evict_last,
//                     2 U_t loads evict_last, 4 U_x/U_y/U_z loads evict_first, 8 stores of `out` evict_first,
//                     16 t-direction loads with L1::no_allocate.
//   L1_CARVEOUT       preferred shared-memory carve-out in percent (the kernel uses no shared memory: 0 = all L1).
// See DESIGN.md section 6.
#include "dslash_kernels.cuh"

namespace dslash {

struct TunedOpts {
    int l2_policy;  // DSLASH_OPT_L2_POLICY bits
};

// A whole x row inside one warp: tile x-extent == L_X, L_X a power of two <= 32 (the tile has >= 32 threads and
// x is its fastest thread index, so lane bits [0, log2 L_X) are the x coordinate).
bool x_shuffle_eligible(const Geom& g, const TileGeom& tg) {
    const int lx = g.L[0];
    return lx <= 32 && (lx & (lx - 1)) == 0 && (1 << tg.lb[0]) == lx &&
           (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]) >= 5;
}

template <typename Real, int LAYOUT, int RECON, int MAXTPB, int MINBLK, int HINT, bool XSHFL>
__global__ void __launch_bounds__(MAXTPB, MINBLK)
    dslash_tuned_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, Geom g,
                        TileGeom tg, TunedOpts opt) {
    // tile coordinates of this block
    unsigned bx, by, bz, bt;
    decode_tile(blockIdx.x, tg, bx, by, bz, bt);
    // in-tile coordinates of this thread (power-of-two tile extents)
    unsigned r = threadIdx.x;
    const int x = (int)((bx << tg.lb[0]) + (r & ((1u << tg.lb[0]) - 1u)));
    r >>= tg.lb[0];
    int y = (int)((by << tg.lb[1]) + (r & ((1u << tg.lb[1]) - 1u)));
    r >>= tg.lb[1];
    int z = (int)((bz << tg.lb[2]) + (r & ((1u << tg.lb[2]) - 1u)));
    r >>= tg.lb[2];
    int t = tg.t_begin + (int)((bt << tg.lb[3]) + r);
    const bool active = !(x >= g.L[0] || y >= g.L[1] || z >= g.L[2] || t >= tg.t_end);
    if (!XSHFL) {
        if (!active) return;
    } else {
        // the warp shuffles of the x hops need every lane: rows beyond a ragged tile edge compute a clamped site and do
        // not store (x is always in range: the tile's x-extent is L_X)
        if (__all_sync(0xffffffffu, !active)) return;
        y = min(y, g.L[1] - 1);
        z = min(z, g.L[2] - 1);
        t = min(t, tg.t_end - 1);
    }
    const unsigned s = (unsigned)x + (unsigned)g.L[0] * ((unsigned)y + (unsigned)g.L[1] * ((unsigned)z + (unsigned)g.L[2] * (unsigned)t));
    Policies pol{0, 0, 0, 0};
    if (HINT) {
        pol.psi = make_policy((opt.l2_policy & 1) ? POLICY_EVICT_LAST : POLICY_NORMAL);
        pol.u_t = make_policy((opt.l2_policy & 2) ? POLICY_EVICT_LAST : POLICY_NORMAL);
        pol.u_s = make_policy((opt.l2_policy & 4) ? POLICY_EVICT_FIRST : POLICY_NORMAL);
        pol.out = make_policy((opt.l2_policy & 8) ? POLICY_EVICT_FIRST : POLICY_NORMAL);
    }
    dslash_site<Real, LAYOUT, RECON, HINT, XSHFL>(out, in, gauge, g, x, y, z, t, s, pol, active);
}

template <typename Real, int LAYOUT, int RECON, int HINT, bool XSHFL>
static cudaError_t launch_tuned_s(const LaunchArgs& a, const TileGeom& tg, const TunedConfig& cfg) {
    const int tpb = 1 << (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]);
    const unsigned grid = (unsigned)tg.nt[0] * (unsigned)tg.nt[1] * (unsigned)tg.nt[2] * (unsigned)tg.nt[3];
    TunedOpts o{cfg.l2_policy > 0 ? cfg.l2_policy : 0};
#define DSLASH_LAUNCH(MAXTPB, MINBLK)                                                                                        \
    do {                                                                                                                     \
        static int carve_set[64]; /* per device; value + 2 so that 0 means "never set" */                                    \
        int dev_ = 0;                                                                                                        \
        cudaGetDevice(&dev_);                                                                                                \
        if (carve_set[dev_ & 63] != cfg.l1_carveout + 2) {                                                                   \
            cudaFuncSetAttribute(dslash_tuned_kernel<Real, LAYOUT, RECON, MAXTPB, MINBLK, HINT, XSHFL>,                           \
                                 cudaFuncAttributePreferredSharedMemoryCarveout, cfg.l1_carveout);                          \
            carve_set[dev_ & 63] = cfg.l1_carveout + 2;                                                                      \
        }                                                                                                                    \
        dslash_tuned_kernel<Real, LAYOUT, RECON, MAXTPB, MINBLK, HINT, XSHFL><<<grid, tpb, 0, a.stream>>>(a.out, a.in,        \
                                                                                                          a.gauge, a.geom, \
                                                                                                          tg, o);          \
    } while (0)
    if (tpb <= 128) {
        if (cfg.occupancy == 1)
            DSLASH_LAUNCH(128, 4);
        else if (cfg.occupancy == 2)
            DSLASH_LAUNCH(128, 2);
        else
            DSLASH_LAUNCH(128, 3);
    } else if (tpb <= 256) {
        // fp32 fits 128 registers: two 256-thread blocks per SM (a bigger tile has less halo per site); fp64 needs the registers
        if (sizeof(Real) == 4 && cfg.occupancy == 1)
            DSLASH_LAUNCH(256, 2);
        else
            DSLASH_LAUNCH(256, 1);
    }
    else if (tpb <= 512)
        DSLASH_LAUNCH(512, 1);
    else
        DSLASH_LAUNCH(1024, 1);
#undef DSLASH_LAUNCH
    return cudaGetLastError();
}

template <typename Real, int LAYOUT, int RECON>
static cudaError_t launch_tuned_t(const LaunchArgs& a, const TileGeom& tg, const TunedConfig& cfg) {
    if (cfg.l2_policy > 0 && (cfg.l2_policy & 16)) return launch_tuned_s<Real, LAYOUT, RECON, 2, false>(a, tg, cfg);
    if (cfg.l2_policy > 0) return launch_tuned_s<Real, LAYOUT, RECON, 1, false>(a, tg, cfg);
    // x hops by warp shuffle when a whole x row sits inside one warp (see x_hops_shuffle in dslash_site.cuh)
    if (cfg.x_shuffle && x_shuffle_eligible(a.geom, tg)) return launch_tuned_s<Real, LAYOUT, RECON, 0, true>(a, tg, cfg);
    return launch_tuned_s<Real, LAYOUT, RECON, 0, false>(a, tg, cfg);
}

template <typename Real>
static cudaError_t launch_tuned_p(int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg, const TunedConfig& cfg) {
    if (layout_base == LAYOUT_AOS)
        return recon == 12 ? launch_tuned_t<Real, LAYOUT_AOS, 12>(a, tg, cfg) : launch_tuned_t<Real, LAYOUT_AOS, 18>(a, tg, cfg);
    return recon == 12 ? launch_tuned_t<Real, LAYOUT_SOA, 12>(a, tg, cfg) : launch_tuned_t<Real, LAYOUT_SOA, 18>(a, tg, cfg);
}

cudaError_t launch_tuned(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg,
                         const TunedConfig& cfg) {
    return precision == 0 ? launch_tuned_p<double>(layout_base, recon, a, tg, cfg)
                          : launch_tuned_p<float>(layout_base, recon, a, tg, cfg);
}

}  // namespace dslash

// dslash_eo.cu -- the even-odd (checkerboarded) form of Eq. 1.
//
// Eq. 1 only couples a site to its eight nearest neighbours, so on a lattice with even extents it maps
// fields on the sites of one parity, (x+y+z+t) mod 2, to fields on the other parity (oracle pin P9).  PAPER.md:52 calls
// Eq. 1 the "unpreconditioned" operator: the preconditioned one its callers solve with is the Schur complement of the
// Wilson matrix M = (4+m) - D/2 on the even sites,
//     Mhat = (4+m) - D_eo D_oe / (4 (4+m)),        D_{p,1-p} = P_p D P_{1-p}.
//
// Checkerboard layout.  With L_X even, the site s = x + L_X*(y + L_Y*(z + L_Z*t)) of parity p has the half-index
//     h = s >> 1 = (x >> 1) + (L_X/2)*(y + L_Y*(z + L_Z*t)),        x = 2*(x >> 1) + o,  o = (p + y + z + t) & 1,
// i.e. s = 2h + o.  A half-lattice spinor of one parity is an ordinary native spinor field over Vh = V/2 "sites" h (same
// AoS / blocked-SoA formulas as the full field); the checkerboarded gauge field is two such native gauge fields, the links
// U_mu(s) of the even sites first, then those of the odd sites.  Neighbours in y, z, t keep (x >> 1) and o, so their
// half-index is h -+ a row stride exactly as on the full lattice; the x neighbours are h itself or h -+ 1:
//     x+1: o == 0 -> h         o == 1 -> h + 1 (wrap to the start of the row)
//     x-1: o == 1 -> h         o == 0 -> h - 1 (wrap to the end of the row)
// so all eight gathers of a warp stay contiguous.  The forward link U_mu(x) comes from the output parity's half of the
// gauge field at h, the backward link U_mu(x - mu^) from the other half at the neighbour's half-index.
#include <mutex>

#include "../../include/dslash_b200.h"
#include "dslash_hop_rt.cuh"
#include "dslash_kernels.cuh"

// Scratch field of dslash_eo_apply_schur_static() (see "Schur operator with the library's own scratch field" below).
// g_schur_scratch is a DEVICE symbol.  In host code its name only stands for it -- taking its address on the host gives
// a host address that a kernel cannot use -- so the device address is asked for with cudaGetSymbolAddress(), once per
// device, while that device is current, and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char g_schur_scratch[DSLASH_STATIC_SCRATCH_BYTES];

namespace dslash {

struct EoParams {
    int parity;     // parity of the OUTPUT sites (input lives on 1 - parity)
    double sigma;   // +1: D, -1: D^dagger
    int xpay;       // out = a * c(h) + b * (D in)(h) instead of out = (D in)(h)
    double a, b;
    const void* c;  // half-lattice field of the output parity (xpay only); may alias nothing else
};

template <typename Real, int LAYOUT, int RECON, int MINBLK>
__global__ void __launch_bounds__(128, MINBLK)
    dslash_eo_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge_out_parity,
                     const void* __restrict__ gauge_in_parity, Geom gh, TileGeom tg, EoParams op) {
    // gh = the half geometry {L_X/2, L_Y, L_Z, L_T}, gh.V = V/2; tiles and threads are laid over (xh, y, z, t)
    unsigned bx, by, bz, bt;
    decode_tile(blockIdx.x, tg, bx, by, bz, bt);
    unsigned r = threadIdx.x;
    const int xh = (int)((bx << tg.lb[0]) + (r & ((1u << tg.lb[0]) - 1u)));
    r >>= tg.lb[0];
    const int y = (int)((by << tg.lb[1]) + (r & ((1u << tg.lb[1]) - 1u)));
    r >>= tg.lb[1];
    const int z = (int)((bz << tg.lb[2]) + (r & ((1u << tg.lb[2]) - 1u)));
    r >>= tg.lb[2];
    const int t = (int)((bt << tg.lb[3]) + r);
    if (xh >= gh.L[0] || y >= gh.L[1] || z >= gh.L[2] || t >= gh.L[3]) return;
    const unsigned Vh = gh.V;
    const unsigned sy = (unsigned)gh.L[0], sz = sy * (unsigned)gh.L[1], st = sz * (unsigned)gh.L[2];
    const unsigned h = (unsigned)xh + sy * (unsigned)y + sz * (unsigned)z + st * (unsigned)t;
    const int o = (op.parity + y + z + t) & 1;  // x = 2*xh + o
    const unsigned xf = o ? ((xh + 1 == gh.L[0]) ? h - (unsigned)(gh.L[0] - 1) : h + 1u) : h;
    const unsigned xb = o ? h : ((xh == 0) ? h + (unsigned)(gh.L[0] - 1) : h - 1u);
    const unsigned yf = (y + 1 == gh.L[1]) ? h - (unsigned)(gh.L[1] - 1) * sy : h + sy;
    const unsigned yb = (y == 0) ? h + (unsigned)(gh.L[1] - 1) * sy : h - sy;
    const unsigned zf = (z + 1 == gh.L[2]) ? h - (unsigned)(gh.L[2] - 1) * sz : h + sz;
    const unsigned zb = (z == 0) ? h + (unsigned)(gh.L[2] - 1) * sz : h - sz;
    const unsigned tf = (t + 1 == gh.L[3]) ? h - (unsigned)(gh.L[3] - 1) * st : h + st;
    const unsigned tb = (t == 0) ? h + (unsigned)(gh.L[3] - 1) * st : h - st;

    const Real sf = (Real)(-op.sigma), sb = (Real)op.sigma;  // forward projector 1 - sigma*gamma, backward 1 + sigma*gamma
    const void* gf = gauge_out_parity;  // U_mu(x):       links of the output-parity sites
    const void* gb = gauge_in_parity;   // U_mu(x - mu^): links of the input-parity sites
    cplx<Real> acc[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) acc[k] = {Real(0), Real(0)};
    hop_rt<0, false, Real, LAYOUT, RECON>(acc, in, gf, Vh, xf, h, sf);
    hop_rt<0, true, Real, LAYOUT, RECON>(acc, in, gb, Vh, xb, xb, sb);
    hop_rt<1, false, Real, LAYOUT, RECON>(acc, in, gf, Vh, yf, h, sf);
    hop_rt<1, true, Real, LAYOUT, RECON>(acc, in, gb, Vh, yb, yb, sb);
    hop_rt<2, false, Real, LAYOUT, RECON>(acc, in, gf, Vh, zf, h, sf);
    hop_rt<2, true, Real, LAYOUT, RECON>(acc, in, gb, Vh, zb, zb, sb);
    hop_rt<3, false, Real, LAYOUT, RECON>(acc, in, gf, Vh, tf, h, sf);
    hop_rt<3, true, Real, LAYOUT, RECON>(acc, in, gb, Vh, tb, tb, sb);
    if (op.xpay) {
        cplx<Real> c[12];
        SpinorIO<Real, LAYOUT>::load(c, op.c, Vh, h);
        const Real a = (Real)op.a, bb = (Real)op.b;
#pragma unroll
        for (int k = 0; k < 12; ++k) acc[k] = {fma_(bb, acc[k].re, a * c[k].re), fma_(bb, acc[k].im, a * c[k].im)};
    }
    SpinorIO<Real, LAYOUT>::store(out, Vh, h, acc);
}

template <typename Real, int LAYOUT, int RECON>
static cudaError_t launch_eo_t(void* out, const void* in, const void* g_out, const void* g_in, const Geom& gh, const TileGeom& tg,
                               const EoParams& op, cudaStream_t st) {
    const int tpb = 1 << (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]);
    if (tpb > 128) return cudaErrorInvalidConfiguration;
    const unsigned grid = (unsigned)tg.nt[0] * (unsigned)tg.nt[1] * (unsigned)tg.nt[2] * (unsigned)tg.nt[3];
    constexpr int MINBLK = sizeof(Real) == 8 ? 2 : 4;  // same register budgets as the tuned Dslash kernel
    dslash_eo_kernel<Real, LAYOUT, RECON, MINBLK><<<grid, tpb, 0, st>>>(out, in, g_out, g_in, gh, tg, op);
    return cudaGetLastError();
}

// out (parity `parity`) = [a * c + b *] D_{parity,1-parity} in;  gauge_eo = even-site links then odd-site links
cudaError_t launch_eo(int precision, int layout_base, int recon, void* out, const void* in, const void* gauge_eo,
                      size_t gauge_half_bytes, const Geom& gh, const TileGeom& tg, int parity, int dagger, int xpay, double a,
                      double b, const void* c, cudaStream_t st) {
    EoParams p;
    p.parity = parity;
    p.sigma = dagger ? -1.0 : 1.0;
    p.xpay = xpay;
    p.a = a;
    p.b = b;
    p.c = c;
    const char* g = static_cast<const char*>(gauge_eo);
    const void* g_out = g + (parity ? gauge_half_bytes : 0);
    const void* g_in = g + (parity ? 0 : gauge_half_bytes);
#define DSLASH_EO(REAL)                                                                                              \
    (layout_base == LAYOUT_AOS ? (recon == 12 ? launch_eo_t<REAL, LAYOUT_AOS, 12>(out, in, g_out, g_in, gh, tg, p, st) \
                                              : launch_eo_t<REAL, LAYOUT_AOS, 18>(out, in, g_out, g_in, gh, tg, p, st)) \
                               : (recon == 12 ? launch_eo_t<REAL, LAYOUT_SOA, 12>(out, in, g_out, g_in, gh, tg, p, st) \
                                              : launch_eo_t<REAL, LAYOUT_SOA, 18>(out, in, g_out, g_in, gh, tg, p, st)))
    return precision == 0 ? DSLASH_EO(double) : DSLASH_EO(float);
#undef DSLASH_EO
}

// ------------------------------------------------------------------ Schur operator with the library's own scratch field
// dslash_eo_apply_schur_static() (include/dslash_b200.h) serves callers that cannot allocate device memory -- their
// application owns all of it, or an allocation's device-wide stall is not affordable where they run -- so the odd-parity
// intermediate of Mhat lives here, in the library image: one array per GPU the library is loaded on, there until exit.
//
// (the array itself, g_schur_scratch, is defined at file scope at the top of this file)
static constexpr int kMaxDevices = 64;
static std::mutex g_schur_scratch_mutex;
static void* g_schur_scratch_addr[kMaxDevices];  // per device, filled by the first call made with that device current

size_t eo_static_scratch_bytes() { return sizeof(g_schur_scratch); }

// Device address of the scratch array on the CURRENT device.  The first call per device does the look-up (set-up: do it
// before any stream capture); later calls read the cached pointer.  Never allocates.
static cudaError_t schur_scratch_address(void** ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_schur_scratch_mutex);
    if (!g_schur_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_schur_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_schur_scratch_addr[dev] = p;
    }
    *ptr = g_schur_scratch_addr[dev];
    return cudaSuccess;
}

// out_even = a * in_even - D_eo (D_oe in_even) / (4a), a = 4 + mass, with D_oe in_even in g_schur_scratch.  half_bytes =
// size of a half-lattice spinor; the caller has checked that it fits.  The array keeps the previous call's contents: the
// first launch overwrites every site the second one reads (padding lanes of a blocked-SoA field are never read), so
// nothing is cleared.  Calls that overlap on the GPU share the array and race.
cudaError_t launch_eo_schur_static(int precision, int layout_base, int recon, void* out_even, const void* in_even, const void* gauge_eo,
                                   size_t gauge_half_bytes, size_t half_bytes, const Geom& gh, const TileGeom& tg, int dagger, double a,
                                   cudaStream_t st) {
    if (half_bytes > sizeof(g_schur_scratch)) return cudaErrorInvalidValue;
    void* tmp_odd = nullptr;
    cudaError_t e = schur_scratch_address(&tmp_odd);
    if (e != cudaSuccess) return e;
    e = launch_eo(precision, layout_base, recon, tmp_odd, in_even, gauge_eo, gauge_half_bytes, gh, tg, 1, dagger, 0, 0.0, 1.0, nullptr, st);
    if (e != cudaSuccess) return e;
    return launch_eo(precision, layout_base, recon, out_even, tmp_odd, gauge_eo, gauge_half_bytes, gh, tg, 0, dagger, 1, a,
                     -1.0 / (4.0 * a), in_even, st);
}

// ------------------------------------------------------------------ layout: canonical full lattice <-> checkerboard halves
// half-index h -> full site index s = 2h + o(parity, row of h)
__device__ __forceinline__ unsigned eo_site(unsigned h, const Geom& gh, int parity) {
    unsigned row = h / (unsigned)gh.L[0];
    const unsigned y = row % (unsigned)gh.L[1];
    row /= (unsigned)gh.L[1];
    const unsigned z = row % (unsigned)gh.L[2];
    const unsigned t = row / (unsigned)gh.L[2];
    return 2u * h + (((unsigned)parity + y + z + t) & 1u);
}

// spinor: NU 16-byte units per site.  dir 0: native half <- canonical full;  dir 1: canonical full <- native half (only
// the sites of `parity` are written).
template <typename U>
__global__ void __launch_bounds__(256) eo_convert_spinor_kernel(U* __restrict__ dst, const U* __restrict__ src, Geom gh, unsigned NU,
                                                                int parity, int soa, int dir) {
    const unsigned Vh = gh.V;
    const size_t n = soa ? (size_t)((Vh + VL - 1u) / VL) * NU * VL : (size_t)Vh * NU;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        unsigned h, u;
        if (soa) {
            const size_t vu = i >> VL_LOG2;
            u = (unsigned)(vu % NU);
            h = (unsigned)(vu / NU) * VL + (unsigned)(i & (VL - 1u));
            if (h >= Vh) continue;
        } else {
            h = (unsigned)(i / NU);
            u = (unsigned)(i - (size_t)h * NU);
        }
        const size_t can = (size_t)eo_site(h, gh, parity) * NU + u;
        if (dir == 0)
            dst[i] = src[can];
        else
            dst[can] = src[i];
    }
}

// gauge: one parity half.  canonical src[(s*4 + mu)*9 + e] -> native half (R = 9 or 6 entries per link)
template <typename U>
__global__ void __launch_bounds__(256) eo_pack_gauge_kernel(U* __restrict__ dst, const U* __restrict__ src, Geom gh, unsigned R,
                                                            int parity, int soa) {
    const unsigned Vh = gh.V, NU = 4u * R;
    const size_t n = soa ? (size_t)((Vh + VL - 1u) / VL) * NU * VL : (size_t)Vh * NU;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        unsigned h, me;
        if (soa) {
            const size_t vu = i >> VL_LOG2;
            me = (unsigned)(vu % NU);
            h = (unsigned)(vu / NU) * VL + (unsigned)(i & (VL - 1u));
            if (h >= Vh) continue;
        } else {
            h = (unsigned)(i / NU);
            me = (unsigned)(i - (size_t)h * NU);
        }
        const unsigned mu = me / R, e = me - mu * R;
        dst[i] = src[((size_t)eo_site(h, gh, parity) * 4u + mu) * 9u + e];
    }
}

static unsigned eo_grid_for(size_t n) {
    size_t b = (n + 255) / 256;
    const size_t cap = 148u * 32u;
    return (unsigned)(b < cap ? (b ? b : 1) : cap);
}

cudaError_t launch_eo_convert_spinor(int precision, int layout_base, void* dst, const void* src, const Geom& gh, int parity, int dir,
                                     cudaStream_t st) {
    const unsigned NU = precision == 0 ? 12u : 6u;
    eo_convert_spinor_kernel<uint4><<<eo_grid_for((size_t)gh.V * NU), 256, 0, st>>>(
        reinterpret_cast<uint4*>(dst), reinterpret_cast<const uint4*>(src), gh, NU, parity, layout_base == LAYOUT_SOA, dir);
    return cudaGetLastError();
}

cudaError_t launch_eo_pack_gauge(int precision, int layout_base, int recon, void* dst_eo, const void* src, size_t gauge_half_bytes,
                                 const Geom& gh, cudaStream_t st) {
    const unsigned R = recon == 12 ? 6u : 9u;
    const size_t n = (size_t)gh.V * 4u * R;
    for (int parity = 0; parity < 2; ++parity) {
        void* dst = static_cast<char*>(dst_eo) + (parity ? gauge_half_bytes : 0);
        if (precision == 0)
            eo_pack_gauge_kernel<uint4><<<eo_grid_for(n), 256, 0, st>>>(reinterpret_cast<uint4*>(dst), reinterpret_cast<const uint4*>(src),
                                                                       gh, R, parity, layout_base == LAYOUT_SOA);
        else
            eo_pack_gauge_kernel<uint2><<<eo_grid_for(n), 256, 0, st>>>(reinterpret_cast<uint2*>(dst), reinterpret_cast<const uint2*>(src),
                                                                       gh, R, parity, layout_base == LAYOUT_SOA);
    }
    return cudaGetLastError();
}

}  // namespace dslash

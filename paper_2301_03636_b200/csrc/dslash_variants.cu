// dslash_variants.cu -- the Advisor-style offload variants of the Dslash loop nest.
//
// PAPER.md:150-164 (section 4.1.3) generates variants of the four nested loops of Code 1
// (i,j,k,l = t,z,y,x) that differ in how many loops are collapsed into
// the parallel iteration space, and the training mode executes every one on the device and records
// its runtime.  BASELINE.json configs[4] fixes the swept axes for this build:
// collapse depth 1-4 x threads/block {64..1024} x sites/thread {1,2,4} x layout {AoS, SoA}.
//
// CUDA meaning of a variant (collapse depth d, B threads/block, S iterations/thread):
//   parallel iteration space  P = product of the first d extents of (L_T, L_Z, L_Y, L_X)
//   iteration id              it = (blockIdx.x*S + k)*B + threadIdx.x,  k = 0..S-1  (block-cyclic)
//   each iteration            runs the remaining 4-d inner loops serially: sites it*inner .. it*inner+inner-1
//                             (inner = V / P; the site index s = x + L_X*(y + L_Y*(z + L_Z*t)) makes the
//                             inner loops a contiguous run of s)
//   grid                      ceil(P / (B*S)) blocks
// This is the analogue of `target teams distribute parallel for collapse(d)` on Loop 0.
#include "dslash_kernels.cuh"

namespace dslash {

template <typename Real, int LAYOUT, int RECON, int MAXTPB>
__global__ void __launch_bounds__(MAXTPB)
    dslash_variant_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, Geom g,
                          unsigned P, unsigned inner, int S) {
    for (int k = 0; k < S; ++k) {
        const unsigned it = (blockIdx.x * (unsigned)S + (unsigned)k) * blockDim.x + threadIdx.x;
        if (it >= P) return;
        const unsigned s0 = it * inner;
        // decode the first site of the run once, then step coordinates like the serial loops would
        unsigned r = s0;
        int x = (int)(r % (unsigned)g.L[0]);
        r /= (unsigned)g.L[0];
        int y = (int)(r % (unsigned)g.L[1]);
        r /= (unsigned)g.L[1];
        int z = (int)(r % (unsigned)g.L[2]);
        int t = (int)(r / (unsigned)g.L[2]);
        for (unsigned i = 0; i < inner; ++i) {
            dslash_site<Real, LAYOUT, RECON>(out, in, gauge, g, x, y, z, t, s0 + i);
            if (++x == g.L[0]) {
                x = 0;
                if (++y == g.L[1]) {
                    y = 0;
                    if (++z == g.L[2]) {
                        z = 0;
                        ++t;
                    }
                }
            }
        }
    }
}

template <typename Real, int LAYOUT, int RECON>
static cudaError_t launch_variant_t(const LaunchArgs& a, int depth, int tpb, int spt) {
    const Geom& g = a.geom;
    unsigned P = 1;
    for (int d = 0; d < depth; ++d) P *= (unsigned)g.L[3 - d];  // t, z, y, x
    const unsigned inner = g.V / P;
    const unsigned per_block = (unsigned)tpb * (unsigned)spt;
    const unsigned grid = (P + per_block - 1) / per_block;
    if (tpb <= 256)
        dslash_variant_kernel<Real, LAYOUT, RECON, 256><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, g, P, inner, spt);
    else if (tpb <= 512)
        dslash_variant_kernel<Real, LAYOUT, RECON, 512><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, g, P, inner, spt);
    else
        dslash_variant_kernel<Real, LAYOUT, RECON, 1024><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, g, P, inner, spt);
    return cudaGetLastError();
}

template <typename Real>
static cudaError_t launch_variant_p(int layout_base, int recon, const LaunchArgs& a, int depth, int tpb, int spt) {
    if (layout_base == LAYOUT_AOS)
        return recon == 12 ? launch_variant_t<Real, LAYOUT_AOS, 12>(a, depth, tpb, spt)
                           : launch_variant_t<Real, LAYOUT_AOS, 18>(a, depth, tpb, spt);
    return recon == 12 ? launch_variant_t<Real, LAYOUT_SOA, 12>(a, depth, tpb, spt)
                       : launch_variant_t<Real, LAYOUT_SOA, 18>(a, depth, tpb, spt);
}

cudaError_t launch_variant(int precision, int layout_base, int recon, const LaunchArgs& a, int depth, int tpb, int spt) {
    return precision == 0 ? launch_variant_p<double>(layout_base, recon, a, depth, tpb, spt)
                          : launch_variant_p<float>(layout_base, recon, a, depth, tpb, spt);
}

}  // namespace dslash

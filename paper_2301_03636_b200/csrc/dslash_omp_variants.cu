// dslash_omp_variants.cu -- CUDA analogues of the paper's exact offload-variant space for the Dslash loop nest.
//
// PAPER.md:150-173 (section 4.1.3, Table 1): for NUM nested loops (Loop 0 .. Loop NUM-1; for Dslash Loop 0..3 = t,z,y,x,
// PAPER.md:27-39, :54) a variant is fixed by
//   x  the position of the `parallel for` directive (0 <= x <= NUM-1),
//   a  the collapse value of `teams distribute` (Loop 0 is always distributed over the teams; if x = 0 the two
//      directives are combined into `teams distribute parallel for` and a does not exist; else 1 <= a <= x),
//   b  the collapse value of `parallel for` (1 <= b <= NUM-x),
//   the schedule of the parallel loop (static, dynamic, guided),
//   and one of two host<->device data-transfer modes (the latter is not a kernel property: dslash_apply_host's
//   DSLASH_MAP_TOFROM / DSLASH_MAP_MINIMAL, DESIGN.md Reading R18).
// That gives NUM + sum_{x>=1} x*(NUM-x) loop structures = 1, 3, 7, 14 for NUM = 1..4, times 3 x 2 = 6, 18, 42, 84
// variants -- Table 1 (tests/golden/table1_variant_counts.txt).
//
// CUDA meaning (a team = a thread block, the league = the grid):
//   distribute      the collapsed iteration space of loops 0..a-1 (x = 0: of loops 0..b-1) is cut into `gridDim.x`
//                   contiguous chunks, one per team (OpenMP's default dist_schedule(static));
//   loops a..x-1    run serially, uniformly by the whole team (in OpenMP: by the team's initial thread);
//   parallel for    the collapsed space of loops x..x+b-1 (x = 0: the team's chunk) is shared among the team's threads:
//                     static   contiguous blocks of ceil(n / team_size) iterations per thread (schedule(static) without
//                              a chunk size, as the OpenMP specification defines it),
//                     dynamic  threads take one iteration at a time from a shared-memory counter (atomicAdd),
//                     guided   threads take max(1, remaining / team_size) iterations at a time (atomicCAS);
//                   a barrier ends every parallel region (OpenMP's implicit barrier);
//   loops x+b..3    run serially inside one thread.
// Every variant computes exactly Eq. 1 (same per-site body as all other kernels); only the mapping of sites to threads
// and the order of sites differ, which is what the paper's tool times and ranks.
#include "dslash_kernels.cuh"

namespace dslash {

struct OmpShape {
    unsigned D;      // distribute space (number of iterations shared among teams)
    unsigned Mid;    // serial-in-team iterations between distribute and parallel for (x >= 1), else 1
    unsigned Q;      // parallel-for space per (d, m) (x >= 1); unused for x = 0
    unsigned inner;  // sites run serially by one thread per parallel iteration
    int combined;    // 1: x = 0 (teams distribute parallel for), the parallel loop is the team's chunk of D
    int sched;       // 0 static, 1 dynamic, 2 guided
};

template <typename Real, int LAYOUT, int RECON>
__device__ __forceinline__ void run_sites(void* out, const void* in, const void* gauge, const Geom& g, unsigned s0, unsigned n) {
    unsigned r = s0;
    int x = (int)(r % (unsigned)g.L[0]);
    r /= (unsigned)g.L[0];
    int y = (int)(r % (unsigned)g.L[1]);
    r /= (unsigned)g.L[1];
    int z = (int)(r % (unsigned)g.L[2]);
    int t = (int)(r / (unsigned)g.L[2]);
    for (unsigned i = 0; i < n; ++i) {
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

// one parallel region: iterations 0..n-1, iteration j covers sites base + j*inner .. + inner
template <typename Real, int LAYOUT, int RECON>
__device__ __forceinline__ void parallel_region(void* out, const void* in, const void* gauge, const Geom& g, unsigned base,
                                                unsigned n, unsigned inner, int sched, unsigned* counter) {
    const unsigned B = blockDim.x, tid = threadIdx.x;
    if (sched == 0) {
        const unsigned chunk = (n + B - 1) / B;
        const unsigned j0 = tid * chunk;
        const unsigned j1 = j0 + chunk < n ? j0 + chunk : n;
        for (unsigned j = j0; j < j1; ++j) run_sites<Real, LAYOUT, RECON>(out, in, gauge, g, base + j * inner, inner);
    } else if (sched == 1) {
        for (;;) {
            const unsigned j = atomicAdd(counter, 1u);
            if (j >= n) break;
            run_sites<Real, LAYOUT, RECON>(out, in, gauge, g, base + j * inner, inner);
        }
    } else {
        for (;;) {
            unsigned cur = *reinterpret_cast<volatile unsigned*>(counter), take;
            for (;;) {
                if (cur >= n) break;
                take = (n - cur) / B;
                if (take < 1u) take = 1u;
                const unsigned seen = atomicCAS(counter, cur, cur + take);
                if (seen == cur) break;
                cur = seen;
            }
            if (cur >= n) break;
            for (unsigned j = cur; j < cur + take; ++j) run_sites<Real, LAYOUT, RECON>(out, in, gauge, g, base + j * inner, inner);
        }
    }
    __syncthreads();  // implicit barrier at the end of the parallel region
    if (sched != 0) {
        if (tid == 0) *counter = 0u;
        __syncthreads();
    }
}

template <typename Real, int LAYOUT, int RECON>
__global__ void __launch_bounds__(256)
    dslash_omp_variant_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, Geom g,
                              OmpShape sh) {
    __shared__ unsigned counter;
    if (threadIdx.x == 0) counter = 0u;
    __syncthreads();
    // distribute: contiguous chunk of the D iterations for this team
    const unsigned G = gridDim.x;
    const unsigned per = (sh.D + G - 1) / G;
    const unsigned d0 = blockIdx.x * per;
    const unsigned d1 = d0 + per < sh.D ? d0 + per : sh.D;
    if (d0 >= d1) return;
    if (sh.combined) {
        parallel_region<Real, LAYOUT, RECON>(out, in, gauge, g, d0 * sh.inner, d1 - d0, sh.inner, sh.sched, &counter);
    } else {
        for (unsigned d = d0; d < d1; ++d)
            for (unsigned m = 0; m < sh.Mid; ++m)
                parallel_region<Real, LAYOUT, RECON>(out, in, gauge, g, (d * sh.Mid + m) * sh.Q * sh.inner, sh.Q, sh.inner,
                                                     sh.sched, &counter);
    }
}

template <typename Real, int LAYOUT, int RECON>
static cudaError_t launch_omp_t(const LaunchArgs& a, const OmpShape& sh, int teams, int team_size) {
    dslash_omp_variant_kernel<Real, LAYOUT, RECON><<<teams, team_size, 0, a.stream>>>(a.out, a.in, a.gauge, a.geom, sh);
    return cudaGetLastError();
}

// a = distribute collapse (0 when x == 0), x = parallel-for position, b = parallel-for collapse
cudaError_t launch_omp_variant(int precision, int layout_base, int recon, const LaunchArgs& a, int da, int x, int b, int sched,
                               int teams, int team_size) {
    const unsigned E[4] = {(unsigned)a.geom.L[3], (unsigned)a.geom.L[2], (unsigned)a.geom.L[1], (unsigned)a.geom.L[0]};  // t,z,y,x
    OmpShape sh;
    sh.sched = sched;
    sh.combined = (x == 0);
    sh.D = sh.Mid = sh.Q = sh.inner = 1u;
    if (x == 0) {
        for (int l = 0; l < b; ++l) sh.D *= E[l];
        for (int l = b; l < 4; ++l) sh.inner *= E[l];
    } else {
        for (int l = 0; l < da; ++l) sh.D *= E[l];
        for (int l = da; l < x; ++l) sh.Mid *= E[l];
        for (int l = x; l < x + b; ++l) sh.Q *= E[l];
        for (int l = x + b; l < 4; ++l) sh.inner *= E[l];
    }
    if ((unsigned)teams > sh.D) teams = (int)sh.D;
    if (teams < 1) teams = 1;
#define DSLASH_OMP(REAL)                                                                                              \
    (layout_base == LAYOUT_AOS ? (recon == 12 ? launch_omp_t<REAL, LAYOUT_AOS, 12>(a, sh, teams, team_size)          \
                                              : launch_omp_t<REAL, LAYOUT_AOS, 18>(a, sh, teams, team_size))         \
                               : (recon == 12 ? launch_omp_t<REAL, LAYOUT_SOA, 12>(a, sh, teams, team_size)          \
                                              : launch_omp_t<REAL, LAYOUT_SOA, 18>(a, sh, teams, team_size)))
    return precision == 0 ? DSLASH_OMP(double) : DSLASH_OMP(float);
#undef DSLASH_OMP
}

}  // namespace dslash

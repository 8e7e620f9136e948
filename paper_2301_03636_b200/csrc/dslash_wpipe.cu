// dslash_wpipe.cu -- warp-pipelined Dslash kernel (DSLASH_KERNEL_WARP_PIPE), sm_100a.
//
// Same operator, same per-hop arithmetic and the same order of the sum as dslash_tuned.cu (Eq. 1; results
// bit-identical).  What changes is how the operands travel.  The direct kernel is bound by the bytes its ~8 resident warps
// per SM can keep in flight in REGISTERS (profiles/r01d_ncu_direct_ring_eo.txt: at most one hop = 336 B per thread).  Here
// the in-flight operands sit in SHARED MEMORY, written by the TMA unit, and cost neither registers nor LSU instructions:
//
//   * L_X == 32, blocked SoA: a warp owns one x row = one 32-site vector.  Everything a hop needs is then CONTIGUOUS in
//     global memory: the 12 components of the 32 neighbour spinors are one 6 KB run, the 9 entries of their 32 links
//     U_mu one 4.5 KB run (fp64).  One hop stage = two cp.async.bulk copies (SASS UBLKCP) issued by one lane, completion
//     counted in bytes on an mbarrier -- instead of 21 LDG.128 per thread with their address arithmetic.
//   * A warp is a persistent stream of stages: 7 per row (x pair by warp shuffle from the row's own psi and U_x; y-, y+,
//     z-, z+, t-, t+).  Rows are handed out IN ORDER from a global counter, so the rows in flight at any time are one
//     contiguous window of the lattice and their y/z/t neighbours are L2 hits (with a static stride w, w + W, ... slow SMs
//     fall whole windows behind and the t reuse misses L2: measured 0.47 ms vs 0.34 ms with 10 warps per SM).  NSLOT
//     stages per warp are always in flight, across row boundaries (no ramp per row): with 8 warps x 2 slots x 10.5 KB
//     an SM keeps 172 KB on order.
//   * No block barrier anywhere: every warp has its own slots and mbarriers.  A stage is consumed by 21 conflict-free
//     LDS.128 per thread, __syncwarp(), and the slot is refilled at once with the stage NSLOT ahead.
//
// Eligibility: blocked SoA, L_X == 32 (x wrap inside the warp).  Otherwise dslash_apply() answers DSLASH_ERR_UNSUPPORTED
// when this kernel was asked for explicitly.
#include "dslash_async.cuh"
#include "dslash_kernels.cuh"

namespace dslash {

namespace {

struct PipeGeom {
    int LY, LZ, LT;      // rows are indexed v = y + LY * (z + LZ * t); one row = one 32-site vector
    int t_begin;         // first time slice computed
    int nt;              // time slices computed
    int zb;              // rows are visited y fastest, then z inside a block of zb planes, then t, then the z blocks: the slice
                         // spacing of the t-neighbour reuse shrinks from LY*LZ rows to LY*zb rows (L2 capacity)
    unsigned nrows;      // LY * LZ * nt
};

}  // namespace

namespace {

template <typename Real, int RECON>
struct PipeBytes {
    static constexpr unsigned PSI = 24u * VL * sizeof(Real);                        // one spinor vector (6144 B in fp64)
    static constexpr unsigned LINK = (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);  // one (vector, mu) link block (4608 B)
    static constexpr unsigned SLOT = PSI + LINK;
};

constexpr unsigned kPipeHeader = 128;  // the mbarriers of the block's warps

// Row coordinates of a warp (all lanes hold the same values).
struct Row {
    int y, z, t;
    unsigned v;
};

__device__ __forceinline__ Row decode_row(const PipeGeom& pg, unsigned r) {
    Row w;
    w.y = (int)(r % (unsigned)pg.LY);
    unsigned q = r / (unsigned)pg.LY;
    const unsigned zl = q % (unsigned)pg.zb;
    q /= (unsigned)pg.zb;
    w.t = pg.t_begin + (int)(q % (unsigned)pg.nt);
    w.z = (int)(zl + (q / (unsigned)pg.nt) * (unsigned)pg.zb);
    w.v = (unsigned)w.y + (unsigned)pg.LY * ((unsigned)w.z + (unsigned)pg.LZ * (unsigned)w.t);
    return w;
}

// Stage I of a row, in the order of the sum (dslash_site.cuh): 0 own psi + U_x(row) for the shuffled x pair; 1 y forward
// (psi(y+1), U_y(row)); 2 z forward; 3 t forward; 4 t backward (psi(t-1), U_t(t-1)); 5 y backward; 6 z backward.
// Two bulk copies into `slot`, completion on `bar`.  Called by one lane.
__host__ __device__ constexpr int stage_mu(int I) { return I == 0 ? 0 : (I == 1 || I == 5) ? 1 : (I == 2 || I == 6) ? 2 : 3; }
__host__ __device__ constexpr bool stage_forward(int I) { return I >= 1 && I <= 3; }

template <int I, typename Real, int RECON>
__device__ __forceinline__ void issue_stage(const PipeGeom& pg, const Row& w, const unsigned char* in, const unsigned char* gauge,
                                            unsigned char* slot, uint64_t* bar) {
    using PB = PipeBytes<Real, RECON>;
    constexpr int MU = stage_mu(I);
    constexpr bool FWD = stage_forward(I);
    unsigned vp = w.v;
    if (MU == 1 && FWD) vp = (w.y + 1 == pg.LY) ? w.v - (unsigned)(pg.LY - 1) : w.v + 1u;
    if (MU == 1 && !FWD) vp = (w.y == 0) ? w.v + (unsigned)(pg.LY - 1) : w.v - 1u;
    if (MU == 2 && FWD) vp = (w.z + 1 == pg.LZ) ? w.v - (unsigned)((pg.LZ - 1) * pg.LY) : w.v + (unsigned)pg.LY;
    if (MU == 2 && !FWD) vp = (w.z == 0) ? w.v + (unsigned)((pg.LZ - 1) * pg.LY) : w.v - (unsigned)pg.LY;
    if (MU == 3 && FWD) vp = (w.t + 1 == pg.LT) ? w.v - (unsigned)((pg.LT - 1) * pg.LZ * pg.LY) : w.v + (unsigned)(pg.LZ * pg.LY);
    if (MU == 3 && !FWD) vp = (w.t == 0) ? w.v + (unsigned)((pg.LT - 1) * pg.LZ * pg.LY) : w.v - (unsigned)(pg.LZ * pg.LY);
    const unsigned vl = (I == 0 || FWD) ? w.v : vp;  // forward hops use the row's own link, backward hops the neighbour's
    mbar_arrive_expect_tx(bar, PB::SLOT);
    bulk_g2s(slot, in + (size_t)vp * PB::PSI, PB::PSI, bar);
    bulk_g2s(slot + PB::PSI, gauge + ((size_t)vl * 4u + (unsigned)MU) * PB::LINK, PB::LINK, bar);
}

template <typename Real, int RECON, int NSLOT>
struct PipeState {
    const PipeGeom& pg;
    const unsigned char* in;
    const unsigned char* gauge;
    unsigned char* slots;  // this warp's NSLOT slots
    uint64_t* bars;        // this warp's NSLOT mbarriers
    unsigned lane;
    int slot;              // slot of the next stage to consume
    unsigned phase;        // bit s = parity of the next completion of slot s
    Row cur, nxt;
    bool nxt_valid;

    // wait for stage I of the current row, move it to registers, refill its slot with the stage NSLOT ahead
    template <int I>
    __device__ __forceinline__ void fetch(cplx<Real> (&psi)[12], cplx<Real> (&u)[9]) {
        using PB = PipeBytes<Real, RECON>;
        unsigned char* sp = slots + (unsigned)slot * PB::SLOT;
        uint64_t* bar = bars + slot;
        mbar_wait_spin(bar, (phase >> slot) & 1u);
        load_psi_slot<Real>(psi, sp, lane);
        load_link_slot<Real, RECON>(u, sp + PB::PSI, lane);
        __syncwarp();  // every lane has its copy: the slot may be overwritten ...
        phase ^= 1u << slot;
        if (lane == 0) {
            // ... by the ASYNC proxy, which is not ordered after the generic-proxy reads above without this fence.  Measured:
            // without it 9 % of the launches of a small L2-resident fp32 lattice (13 one-warp blocks per SM, bulk copies
            // landing within a few hundred cycles) returned one wrong row; with it 0 of 600.
            fence_proxy_async();
            constexpr int J = I + NSLOT;
            if (J < 7)
                issue_stage<(J < 7 ? J : 0), Real, RECON>(pg, cur, in, gauge, sp, bar);
            else if (nxt_valid)
                issue_stage<(J >= 7 ? J - 7 : 0), Real, RECON>(pg, nxt, in, gauge, sp, bar);
        }
        slot = (slot + 1 == NSLOT) ? 0 : slot + 1;
    }
};

template <typename Real, int RECON, int NSLOT, int NW, int MINBLK>
__global__ void __launch_bounds__(NW * 32, MINBLK)
    dslash_wpipe_kernel(void* __restrict__ out, const void* __restrict__ in_, const void* __restrict__ gauge_, Geom g, PipeGeom pg,
                        unsigned* __restrict__ ctr) {
    using PB = PipeBytes<Real, RECON>;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned lane = threadIdx.x & 31u, wib = threadIdx.x >> 5;
    const unsigned W = gridDim.x * (unsigned)NW;
    // Rows are handed out in order: the first W statically (row = global warp number), every further one from the counter
    // ctr[0], so that the rows in flight stay ONE contiguous window of the lattice however the SMs drift apart (a static
    // stride lets slow SMs fall behind by whole windows, and the t-neighbour reuse then misses L2).  ctr[1] counts finished
    // warps; the last one resets both for the next launch.
    unsigned r = blockIdx.x * (unsigned)NW + wib;
    if (r >= pg.nrows) {  // warp-uniform; no block barrier is ever used
        if (lane == 0) {
            __threadfence();
            if (atomicAdd(ctr + 1, 1u) == W - 1u) {
                ctr[0] = 0u;
                ctr[1] = 0u;
            }
        }
        return;
    }
    PipeState<Real, RECON, NSLOT> st{pg,
                                    static_cast<const unsigned char*>(in_),
                                    static_cast<const unsigned char*>(gauge_),
                                    smem + kPipeHeader + (size_t)wib * NSLOT * PB::SLOT,
                                    reinterpret_cast<uint64_t*>(smem) + wib * NSLOT,
                                    lane,
                                    0,
                                    0u,
                                    decode_row(pg, r),
                                    Row{0, 0, 0, 0u},
                                    false};
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) mbar_init(st.bars + s, 1u);
        mbar_fence_init();
        // prologue: the first NSLOT stages of the first row
        issue_stage<0, Real, RECON>(pg, st.cur, st.in, st.gauge, st.slots, st.bars);
        if (NSLOT > 1) issue_stage<1, Real, RECON>(pg, st.cur, st.in, st.gauge, st.slots + PB::SLOT, st.bars + 1);
        if (NSLOT > 2) issue_stage<2, Real, RECON>(pg, st.cur, st.in, st.gauge, st.slots + 2 * PB::SLOT, st.bars + 2);
        if (NSLOT > 3) issue_stage<3, Real, RECON>(pg, st.cur, st.in, st.gauge, st.slots + 3 * PB::SLOT, st.bars + 3);
    }
    __syncwarp();
    const int lane_fwd = (int)((lane + 1u) & 31u), lane_bwd = (int)((lane - 1u) & 31u);
    bool more = true;
    while (more) {
        unsigned rn = 0u;
        if (lane == 0) rn = W + atomicAdd(ctr, 1u);  // the next row of this warp; needed NSLOT stages before its first use
        cplx<Real> acc[12], psi[12], u[9];
        st.template fetch<0>(psi, u);  // refills with stage NSLOT of the SAME row: the atomic's latency hides behind this stage
        x_hops_regs(acc, psi, u, lane_fwd, lane_bwd);
        rn = __shfl_sync(0xffffffffu, rn, 0);
        st.nxt_valid = rn < pg.nrows;
        if (st.nxt_valid) st.nxt = decode_row(pg, rn);
        st.template fetch<1>(psi, u);
        hop_regs<1, -1>(acc, psi, u);
        st.template fetch<2>(psi, u);
        hop_regs<2, -1>(acc, psi, u);
        st.template fetch<3>(psi, u);
        hop_regs<3, -1>(acc, psi, u);
        st.template fetch<4>(psi, u);
        hop_regs<3, +1>(acc, psi, u);
        st.template fetch<5>(psi, u);
        hop_regs<1, +1>(acc, psi, u);
        st.template fetch<6>(psi, u);
        hop_regs<2, +1>(acc, psi, u);
        SpinorIO<Real, LAYOUT_SOA>::store(out, g.V, st.cur.v * VL + lane, acc);
        st.cur = st.nxt;
        more = st.nxt_valid;
    }
    if (lane == 0) {
        __threadfence();
        if (atomicAdd(ctr + 1, 1u) == W - 1u) {
            ctr[0] = 0u;
            ctr[1] = 0u;
        }
    }
}

}  // namespace

// blocked SoA, one x row = one 32-site vector = one warp (x wraps inside the warp)
bool wpipe_eligible(int layout_base, const Geom& g) { return layout_base == LAYOUT_SOA && g.L[0] == (int)VL; }

namespace {

template <typename Real, int RECON, int NSLOT, int NW>
cudaError_t launch_wpipe_k(const LaunchArgs& a, const TileGeom& tg, int zblock, unsigned* ctr) {
    using PB = PipeBytes<Real, RECON>;
    constexpr size_t smem = kPipeHeader + (size_t)NW * NSLOT * PB::SLOT;
    constexpr int fit = (int)(232448u / (smem + 1024u));  // blocks per SM by shared memory (1 KB reserved per block)
    constexpr int cap = 16 / NW > 0 ? 16 / NW : 1;        // no more than 16 warps per SM: keep >= 128 registers per thread
    constexpr int MINBLK = fit < 1 ? 1 : (fit < cap ? fit : cap);
    auto kernel = dslash_wpipe_kernel<Real, RECON, NSLOT, NW, MINBLK>;
    // occupancy and the dynamic shared-memory attribute are per DEVICE: cached per device id, not per process
    static int blocks_per_sm_of[64] = {0}, sms_of[64] = {0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const int di = dev & 63;
    if (blocks_per_sm_of[di] == 0) {
        if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        int bps = 0, nsm = 0;
        if ((e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, NW * 32, smem)) != cudaSuccess) return e;
        if (bps < 1) return cudaErrorInvalidConfiguration;
        sms_of[di] = nsm;
        blocks_per_sm_of[di] = bps;
    }
    const int blocks_per_sm = blocks_per_sm_of[di], sms = sms_of[di];
    PipeGeom pg{a.geom.L[1], a.geom.L[2], a.geom.L[3], tg.t_begin, tg.t_end - tg.t_begin, a.geom.L[2], 0u};
    if (zblock > 0 && zblock < a.geom.L[2] && a.geom.L[2] % zblock == 0) pg.zb = zblock;
    pg.nrows = (unsigned)a.geom.L[1] * (unsigned)a.geom.L[2] * (unsigned)pg.nt;
    if (pg.nrows == 0) return cudaSuccess;
    const unsigned need = (pg.nrows + NW - 1) / NW, resident = (unsigned)(blocks_per_sm * sms);
    kernel<<<need < resident ? need : resident, NW * 32, smem, a.stream>>>(a.out, a.in, a.gauge, a.geom, pg, ctr);
    return cudaGetLastError();
}

template <typename Real, int RECON>
cudaError_t launch_wpipe_r(const LaunchArgs& a, const TileGeom& tg, int slots, int warps, int zblock, unsigned* ctr) {
    if (warps == 1) {
        if (slots == 2) return launch_wpipe_k<Real, RECON, 2, 1>(a, tg, zblock, ctr);
        if (slots == 3) return launch_wpipe_k<Real, RECON, 3, 1>(a, tg, zblock, ctr);
        return launch_wpipe_k<Real, RECON, 4, 1>(a, tg, zblock, ctr);
    }
    if (warps == 2) {
        if (slots == 2) return launch_wpipe_k<Real, RECON, 2, 2>(a, tg, zblock, ctr);
        if (slots == 3) return launch_wpipe_k<Real, RECON, 3, 2>(a, tg, zblock, ctr);
        return launch_wpipe_k<Real, RECON, 4, 2>(a, tg, zblock, ctr);
    }
    if (slots == 2) return launch_wpipe_k<Real, RECON, 2, 4>(a, tg, zblock, ctr);
    if (slots == 3) return launch_wpipe_k<Real, RECON, 3, 4>(a, tg, zblock, ctr);
    return launch_wpipe_k<Real, RECON, 4, 4>(a, tg, zblock, ctr);
}

}  // namespace

cudaError_t launch_wpipe(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg, const TunedConfig& cfg) {
    if (!wpipe_eligible(layout_base, a.geom) || !cfg.pipe_counters) return cudaErrorInvalidConfiguration;
    const int slots = cfg.pipe_slots >= 2 && cfg.pipe_slots <= 4 ? cfg.pipe_slots : 2;
    const int warps = cfg.pipe_warps == 1 ? 1 : (cfg.pipe_warps == 2 ? 2 : 4);  // default 4: 2 blocks x 4 warps x 2 slots per SM
    const int zblock = cfg.pipe_zblock;
    if (precision == 0) return recon == 12 ? launch_wpipe_r<double, 12>(a, tg, slots, warps, zblock, cfg.pipe_counters) : launch_wpipe_r<double, 18>(a, tg, slots, warps, zblock, cfg.pipe_counters);
    return recon == 12 ? launch_wpipe_r<float, 12>(a, tg, slots, warps, zblock, cfg.pipe_counters) : launch_wpipe_r<float, 18>(a, tg, slots, warps, zblock, cfg.pipe_counters);
}

}  // namespace dslash

// dslash_gmarch.cu -- the block-cooperative t-marching Dslash kernel for ANY x extent (DSLASH_KERNEL_GMARCH), sm_100a.
//
// dslash_march.cu needs L_X == 32: there a storage vector (32 consecutive sites of the blocked SoA layout) is an x row, x hops
// are warp shuffles and a y / z neighbour is one whole vector.  For 48^3x96, 24^4, 16^4 (BASELINE.json configs[3], [4], [1]) a
// vector is 2/3 of a row, 4/3 of a row, two rows: neighbours in x and y are lane-shifted and spread over two or three vectors.
// This kernel keeps the design of dslash_march.cu --
//   * a thread block owns a patch of the (y,z) plane and marches through the time slices;
//   * every link is fetched once, by the warp that owns its site, and used for the site's forward hop and for the complete
//     backward contribution of the neighbour, w_mu(x) = U_mu(x)^dagger P^+_mu psi(x), which travels through a shared-memory
//     exchange buffer;
//   * every spinor vector of the patch is fetched once into a two-slot shared-memory ring (psi(t+1) of the t hop, a step later
//     the warp's own spinors and its neighbours' forward operands); only halo vectors are fetched twice;
//   * nothing is loaded by LDG inside the loop: links, halo spinors and ring rows arrive by cp.async.bulk issued by four
//     producer warps (setmaxnreg), completion on mbarriers, no block barrier in the loop --
// and generalises the addressing: a compute warp owns one VECTOR; a block owns whole UNITS (lcm(L_X, 32) sites = whole rows
// = whole vectors), so x neighbours never leave the block; every hop of a lane is resolved through the host-built plan
// (GmWarpPlan, dslash_kernels.cuh): per (warp, direction) up to three source vectors with the mask of the lanes they serve.
// The lane INSIDE the source follows from the geometry alone: x+1 is the next lane (or, at the end of a row, L_X - 1 lanes
// back), y+1 is L_X lanes on (mod 32, because L_X * L_Y is a multiple of 32), z+1 and t+1 the same lane.  x hops go through
// the ring and an exchange buffer like y and z hops (a shuffle cannot cross warps); for L_X == 32 the kernel degenerates to
// dslash_march.cu with x by shared memory.
//
// Same per-hop arithmetic and the same ORDER of the sum as every tuned kernel of the library (dslash_site.cuh):
//   x forward, x backward, y forward, z forward, t forward, t backward, y backward, z backward
// so the result is bit-identical to the direct kernel (Eq. 1).
#include <algorithm>
#include <vector>

#define DSLASH_F32X2  // packed FP32 arithmetic (FFMA2 / FADD2), see dslash_site.cuh
#include "../../include/dslash_b200.h"
#include "dslash_async.cuh"
#include "dslash_kernels.cuh"

namespace dslash {

namespace {

constexpr unsigned GM_TAB = 12u;  // stage-table entries per copy queue
#ifndef GM_IDLE_NS
#define GM_IDLE_NS 200
#endif

// Shared-memory map of a block (all run-time: NW, NLS, NHS, NWB depend on the lattice).  Barrier fields are indices into the
// uint64 array at offset 0, the others byte offsets.
struct GmLayout {
    int NW, NLS, NHS, NWB;
    unsigned b_ring_full, b_ring_empty;  // [2][NW]
    unsigned b_lfull, b_lempty;          // [NW][NLS]
    unsigned b_hfull, b_hempty;          // [NW][NHS]
    unsigned b_wfull, b_wempty;          // [NWB]
    unsigned b_count;
    unsigned table;  // uint32 [3 * NW][GM_TAB]: the producers' stage tables (units of 256 B)
    unsigned plan;   // GmBlockPlan of this block
    unsigned ring;   // [2][NW][PSI]
    unsigned lslot;  // [NW][NLS][LINK]
    unsigned hslot;  // [NW][NHS][PSI]
    unsigned wbuf;   // [NWB][HALF]
    unsigned total;
};

unsigned real_size(int precision) { return precision == 0 ? 8u : 4u; }

GmLayout gm_layout(int precision, int recon, int NW, int NLS, int NHS, int NWB) {
    const unsigned rs = real_size(precision), PSI = 24u * VL * rs, LINK = (recon == 12 ? 12u : 18u) * VL * rs, HALF = 12u * VL * rs;
    GmLayout L;
    L.NW = NW;
    L.NLS = NLS;
    L.NHS = NHS;
    L.NWB = NWB;
    const unsigned nw = (unsigned)NW;
    L.b_ring_full = 0u;
    L.b_ring_empty = 2u * nw;
    L.b_lfull = 4u * nw;
    L.b_lempty = L.b_lfull + nw * (unsigned)NLS;
    L.b_hfull = L.b_lempty + nw * (unsigned)NLS;
    L.b_hempty = L.b_hfull + nw * (unsigned)NHS;
    L.b_wfull = L.b_hempty + nw * (unsigned)NHS;
    L.b_wempty = L.b_wfull + (unsigned)NWB;
    L.b_count = L.b_wempty + (unsigned)NWB;
    auto up = [](unsigned v) { return (v + 127u) & ~127u; };
    L.table = up(L.b_count * 8u);
    L.plan = up(L.table + 3u * nw * GM_TAB * 4u);
    L.ring = up(L.plan + (unsigned)sizeof(GmBlockPlan));
    L.lslot = L.ring + 2u * nw * PSI;
    L.hslot = L.lslot + nw * (unsigned)NLS * LINK;
    L.wbuf = L.hslot + nw * (unsigned)NHS * PSI;
    L.total = L.wbuf + (unsigned)NWB * HALF;
    return L;
}

constexpr unsigned GM_SMEM_MAX = 232448u;  // 227 KB

// State of one compute warp.  Every member is warp-uniform except `lane`.
template <typename Real, int RECON>
struct GmWarp {
    static constexpr unsigned PSI = 24u * VL * sizeof(Real);
    static constexpr unsigned LINK = (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);
    static constexpr unsigned HALF = 12u * VL * sizeof(Real);
    unsigned char* smem;
    uint64_t* bars;
    const GmLayout* L;     // the kernel parameter (constant bank)
    const GmWarpPlan* wp;  // this warp's plan (shared memory)
    unsigned lane, w;
    bool late;             // late ring fill (DSLASH_OPT_L2_POLICY bit 16): see read_own()
    int step;              // current step i
    int lslot, hslot;      // slot of the next link / halo stage to consume
    unsigned lphase, hphase;  // parity of the next completion, bit s = slot s

    // "this warp is done with the buffer": all lanes have issued their reads/writes, lane 0 tells the other side
    __device__ __forceinline__ void hand_over(uint64_t* bar) const {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar);
    }
    // next link stage of this warp -> registers, every lane taking the link of lane `ln` of the staged vector
    __device__ __forceinline__ void fetch_link(cplx<Real> (&u)[9], unsigned ln) {
        const unsigned b = w * (unsigned)L->NLS + (unsigned)lslot;
        mbar_wait_spin(bars + L->b_lfull + b, (lphase >> lslot) & 1u);
        load_link_slot<Real, RECON>(u, smem + L->lslot + b * LINK, ln);
        hand_over(bars + L->b_lempty + b);
        lphase ^= 1u << lslot;
        lslot = (lslot + 1 == L->NLS) ? 0 : lslot + 1;
    }
    // next halo spinor stage of this warp; the lanes with `pred` take the spinor of lane `ln` of the staged vector
    __device__ __forceinline__ void fetch_halo(cplx<Real> (&psi)[12], unsigned ln, bool pred) {
        const unsigned b = w * (unsigned)L->NHS + (unsigned)hslot;
        mbar_wait_spin(bars + L->b_hfull + b, (hphase >> hslot) & 1u);
        if (pred) load_psi_slot<Real>(psi, smem + L->hslot + b * PSI, ln);
        hand_over(bars + L->b_hempty + b);
        hphase ^= 1u << hslot;
        hslot = (hslot + 1 == L->NHS) ? 0 : hslot + 1;
    }
    // ring row `r` of the slice of step `step` + ahead (0: current slice, 1: next slice); done = the warp's last read of this fill
    __device__ __forceinline__ void read_ring(cplx<Real> (&psi)[12], unsigned r, int ahead, bool done, unsigned ln, bool pred) const {
        const unsigned q = (unsigned)(step + ahead), b = (q & 1u) * (unsigned)L->NW + r;
        mbar_wait_spin(bars + L->b_ring_full + b, (q >> 1) & 1u);
        if (pred) load_psi_slot<Real>(psi, smem + L->ring + b * PSI, ln);
        if (done) hand_over(bars + L->b_ring_empty + b);
    }
    // forward operand psi(x + d^) of every lane: from the ring rows and halo stages the plan lists for direction D
    template <int D>
    __device__ __forceinline__ void gather_fwd(cplx<Real> (&psi)[12], unsigned ln) {
        const int n = wp->nf[D];
#pragma unroll 1
        for (int e = 0; e < n; ++e) {
            const int id = wp->f[D][e].id;
            const bool pred = (wp->f[D][e].mask >> lane) & 1u;
            if (id >= 0)
                read_ring(psi, (unsigned)(id & 0xff), 0, ((id >> 8) & 1) != 0 && (late || (unsigned)(id & 0xff) != w), ln, pred);
            else
                fetch_halo(psi, ln, pred);
        }
    }
    // backward contribution w_MU(x - mu^) of every lane: from the neighbours' exchange buffers, or formed here from a halo
    // spinor and its link (next stages of the halo and link streams)
    template <int MU>
    __device__ __forceinline__ void gather_bwd(cplx<Real> (&wv)[6], unsigned ln) {
        const int n = wp->nb[MU];
#pragma unroll 1
        for (int e = 0; e < n; ++e) {
            const int id = wp->b[MU][e].id;
            const bool pred = (wp->b[MU][e].mask >> lane) & 1u;
            if (id >= 0) {
                mbar_wait_spin(bars + L->b_wfull + (unsigned)id, (unsigned)step & 1u);
                if (pred) load_half<Real>(wv, smem + L->wbuf + (unsigned)id * HALF, ln);
                hand_over(bars + L->b_wempty + (unsigned)id);
            } else {
                cplx<Real> psi[12], u[9];
                fetch_halo(psi, ln, true);
                fetch_link(u, ln);
                if (pred) {  // the other lanes keep what their own source gave them
                    cplx<Real> h[6];
                    project<MU, +1>(h, psi);
                    su3_mul<true>(wv, u, h);
                }
            }
        }
    }
    // The warp's own spinors of the current slice.  They are NOT kept in registers across the step (48 registers in fp64) but
    // re-read from the ring row where needed, the last time in the t phase.  Two ways to hand the row back:
    //   late fill (bit 16 of DSLASH_OPT_L2_POLICY, default): at the warp's last FORWARD read, as in dslash_march.cu.  The slot
    //     is refilled with slice step + 2, and that fill is issued only after every reader of slice step + 1 -- this warp
    //     among them, during the NEXT step -- is done (gm_producer), so the row outlives the step although it was handed back;
    //   early fill: at the t-phase read, the warp's last read of the row; the refill may then start a whole step before it
    //     is needed (more time for the copy, but the owner's fetch and the neighbouring blocks' halo fetches of the same
    //     vector drift a step apart in L2).
    __device__ __forceinline__ void read_own(cplx<Real> (&own)[12], bool done) const { read_ring(own, w, 0, done, lane, true); }
    // w_MU of the warp's own sites for the neighbours that sit in this block
    template <int MU>
    __device__ __forceinline__ void publish(const cplx<Real> (&u)[9], bool done) {
        const int b = wp->wr[MU];
        if (b >= 0 || done) {
            cplx<Real> h[6], wv[6];
            {
                cplx<Real> own[12];
                read_own(own, done);
                project<MU, +1>(h, own);
            }
            if (b < 0) return;
            su3_mul<true>(wv, u, h);
            if (step > 0) mbar_wait_spin(bars + L->b_wempty + (unsigned)b, ((unsigned)step - 1u) & 1u);  // the readers took the previous one
            store_half<Real>(smem + L->wbuf + (unsigned)b * HALF, lane, wv);
            hand_over(bars + L->b_wfull + (unsigned)b);
        }
    }
    // y (MU = 1) or z (MU = 2): the link of the own site gives the neighbours' backward contribution and the own forward hop
    template <int MU>
    __device__ __forceinline__ void forward_phase(cplx<Real> (&acc)[12], unsigned ln) {
        cplx<Real> u[9];
        fetch_link(u, lane);
        publish<MU>(u, false);
        cplx<Real> psi[12];
        gather_fwd<MU>(psi, ln);
        hop_regs<MU, -1>(acc, psi, u);
    }
};

// A producer warp: each of its first lanes owns one of the block's 3 * NW copy queues -- queue / NW = 0: the link stream of
// compute warp queue % NW (NLS slots), 1: its halo spinor stream (NHS slots), 2: its ring row (two slots, slices t0 .. t0+n).
// A queue is a cyclic list of `nstage` sources per step; fill number q goes to slot q % nslots and may be issued once the
// slot's previous fill has been released (its "empty" barrier has completed round - 1 phases).
template <typename Real, int RECON>
__device__ __forceinline__ void gm_producer(unsigned char* smem, const unsigned char* in, const unsigned char* gauge, const GmBlockPlan& bp,
                                            const GmLayout& L, unsigned queue, int slice_vecs, int LT, int hints) {
    constexpr unsigned PSI = 24u * VL * sizeof(Real), LINK = (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);
    constexpr unsigned LU = LINK / 256u, PU = PSI / 256u;
    static_assert(PSI % 256u == 0 && LINK % 256u == 0, "stage tables hold offsets in units of 256 bytes");
    const unsigned NW = (unsigned)L.NW, nq = 3u * NW;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    uint32_t* tab = reinterpret_cast<uint32_t*>(smem + L.table) + (queue < nq ? queue : 0u) * GM_TAB;
    const unsigned qw = queue % NW, kind = queue / NW;
    const int n = bp.nt, t0 = bp.t0;
    int nstage = 0, total = 0, nslots = 1;
    unsigned bytes = 0, dst = 0, dst_stride = 0, bar_full = 0, bar_empty = 0, bar_stride = 1;
    unsigned shared_stage = ~0u;  // bit k: stage k of this queue is read by another block as well
    const unsigned char* src = in;
    size_t slice_stride = 0;
    if (queue < nq && bp.w[qw].vec >= 0) {
        const GmWarpPlan& pw = bp.w[qw];
        if (kind == 0u) {
            // links in the order the compute warp consumes them: U_x, U_y, U_z, U_t of its own vector, then U_y / U_z of the
            // vectors its backward halo hops reach
            for (int mu = 0; mu < 4; ++mu) tab[nstage++] = ((unsigned)pw.vec * 4u + (unsigned)mu) * LU;
            for (int d = 1; d <= 2; ++d)
                for (int e = 0; e < pw.nb[d]; ++e)
                    if (pw.b[d][e].id < 0 && nstage < (int)GM_TAB) tab[nstage++] = ((unsigned)(-pw.b[d][e].id - 1) * 4u + (unsigned)d) * LU;
            total = nstage * n;
            nslots = L.NLS;
            bytes = LINK;
            src = gauge;
            slice_stride = (size_t)slice_vecs * 4u * LINK;
            dst = L.lslot + qw * (unsigned)L.NLS * LINK;
            dst_stride = LINK;
            bar_full = L.b_lfull + qw * (unsigned)L.NLS;
            bar_empty = L.b_lempty + qw * (unsigned)L.NLS;
            shared_stage = ~0xFu | (pw.link_shared & 6u);
        } else if (kind == 1u) {
            // halo spinors: forward y, forward z, backward y, backward z
            for (int d = 1; d <= 2; ++d)
                for (int e = 0; e < pw.nf[d]; ++e)
                    if (pw.f[d][e].id < 0 && nstage < (int)GM_TAB) tab[nstage++] = (unsigned)(-pw.f[d][e].id - 1) * PU;
            for (int d = 1; d <= 2; ++d)
                for (int e = 0; e < pw.nb[d]; ++e)
                    if (pw.b[d][e].id < 0 && nstage < (int)GM_TAB) tab[nstage++] = (unsigned)(-pw.b[d][e].id - 1) * PU;
            total = nstage * n;
            nslots = L.NHS;
            bytes = PSI;
            slice_stride = (size_t)slice_vecs * PSI;
            dst = L.hslot + qw * (unsigned)L.NHS * PSI;
            dst_stride = PSI;
            bar_full = L.b_hfull + qw * (unsigned)L.NHS;
            bar_empty = L.b_hempty + qw * (unsigned)L.NHS;
        } else {
            tab[nstage++] = (unsigned)pw.vec * PU;
            total = n + 1;
            nslots = 2;
            bytes = PSI;
            slice_stride = (size_t)slice_vecs * PSI;
            dst = L.ring + qw * PSI;
            dst_stride = NW * PSI;
            bar_full = L.b_ring_full + qw;
            bar_empty = L.b_ring_empty + qw;
            bar_stride = NW;
        }
    }
    // L2 eviction policies (DSLASH_OPT_L2_POLICY bits) as in dslash_march.cu: 4 = what is read exactly once per application is
    // evict_first, 1 = what another block reads too is evict_last
    const uint64_t pol_shared = (hints & 1) ? make_policy(POLICY_EVICT_LAST) : 0ull;
    const uint64_t pol_stream = (hints & 4) ? make_policy(POLICY_EVICT_FIRST) : 0ull;
    int q = 0, k = 0, i = 0, slot = 0, round = 0;
    while (__any_sync(0xffffffffu, q < total)) {
        bool ready = false;
        if (q < total) ready = round == 0 || mbar_test(bars + bar_empty + (unsigned)slot * bar_stride, ((unsigned)round - 1u) & 1u);
        // late ring fill (bit 16, dslash_march.cu): hold the fill of slice q back until the readers of slice q - 1 are done, so
        // that the owner's fetch and the neighbouring blocks' halo fetches of the same vector are about one step apart -- and
        // so that the slot it overwrites (slice q - 2), handed back early in this mode, is no longer re-read by its owner
        // (GmWarp::read_own)
        if (ready && kind == 2u && (hints & 16) && q >= 2)
            ready = mbar_test(bars + bar_empty + (unsigned)(slot ^ 1) * bar_stride, (((unsigned)q - 1u) >> 1) & 1u);
        if (ready) {
            int ts = t0 + i;
            if (ts >= LT) ts -= LT;
            const unsigned char* from = src + (size_t)tab[k] * 256u + (size_t)ts * slice_stride;
            unsigned char* to = smem + dst + (unsigned)slot * dst_stride;
            uint64_t* full = bars + bar_full + (unsigned)slot * bar_stride;
            fence_proxy_async();  // the readers' generic-proxy accesses (ordered before us by the empty barrier) before the async write
            mbar_arrive_expect_tx(full, bytes);
            const uint64_t pol = ((shared_stage >> k) & 1u) ? pol_shared : pol_stream;
            if (pol)
                bulk_g2s_hint(to, from, bytes, full, pol);
            else
                bulk_g2s(to, from, bytes, full);
            ++q;
            if (++k == nstage) {
                k = 0;
                ++i;
            }
            if (++slot == nslots) {
                slot = 0;
                ++round;
            }
        }
        // nothing to issue: sleep.  ncu on 48^3x96 fp32: with 32 ns the four producer warps executed 40 % of the block's
        // instructions, and the compute warps (three per scheduler) are bound by instruction issue
        if (!__any_sync(0xffffffffu, ready)) __nanosleep(GM_IDLE_NS);
    }
}

// Register split between the roles (setmaxnreg works on warpgroups of four warps): warpgroup 0 = four producer warps at 40
// registers per thread; CWG compute warpgroups at 232 (CWG = 2: 128 x 40 + 256 x 232 = 64512) or 152 registers
// (CWG = 3: 128 x 40 + 384 x 152 = 63488 <= 65536).
constexpr int GM_PRODUCER_WARPS = 4, GM_REGS_PRODUCER = 40;

template <typename Real, int RECON, int CWG>
__global__ void __launch_bounds__(128 * (1 + CWG), 1)
    dslash_gmarch_kernel(void* __restrict__ out, const void* __restrict__ in_, const void* __restrict__ gauge_, unsigned V, int slice_vecs,
                         int LX, int LT, const GmBlockPlan* __restrict__ plan, const __grid_constant__ GmLayout L, int hints) {
    constexpr int REGS_COMPUTE = CWG == 2 ? 232 : 152;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    {
        const int* src = reinterpret_cast<const int*>(plan + blockIdx.x);
        int* dst = reinterpret_cast<int*>(smem + L.plan);
        for (unsigned i = threadIdx.x; i < sizeof(GmBlockPlan) / sizeof(int); i += blockDim.x) dst[i] = src[i];
    }
    __syncthreads();
    const GmBlockPlan& bp = *reinterpret_cast<const GmBlockPlan*>(smem + L.plan);
    // every barrier takes ONE arrival per phase (the producer's expect_tx, or lane 0 of the one warp that hands the buffer
    // over), except "ring row r is free" and "exchange buffer b is free": one arrival per reading warp
    for (unsigned b = threadIdx.x; b < L.b_count; b += blockDim.x) {
        int count = 1;
        if (b >= L.b_ring_empty && b < L.b_lfull) count = bp.ring_readers[(b - L.b_ring_empty) % (unsigned)L.NW];
        if (b >= L.b_wempty) count = bp.wbuf_readers[b - L.b_wempty];
        mbar_init(bars + b, (unsigned)(count < 1 ? 1 : count));
    }
    mbar_fence_init();
    __syncthreads();

    if (warp < (unsigned)GM_PRODUCER_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(GM_REGS_PRODUCER));
        // queue q is served by lane q / 4 of producer warp q % 4: the copies of one compute warp are spread over the producers
        const unsigned nq = 3u * (unsigned)L.NW;
        const unsigned queue = lane < (nq + 3u) / 4u ? warp + (unsigned)GM_PRODUCER_WARPS * lane : nq;
        gm_producer<Real, RECON>(smem, static_cast<const unsigned char*>(in_), static_cast<const unsigned char*>(gauge_), bp, L,
                                 queue < nq ? queue : nq, slice_vecs, LT, hints);
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(REGS_COMPUTE));
    const unsigned w = warp - (unsigned)GM_PRODUCER_WARPS;  // compute warp number
    if (w >= (unsigned)L.NW) return;
    GmWarp<Real, RECON> m;
    m.smem = smem;
    m.bars = bars;
    m.L = &L;
    m.wp = &bp.w[w];
    m.lane = lane;
    m.w = w;
    m.late = (hints & 16) != 0;
    m.lslot = 0;
    m.hslot = 0;
    m.lphase = 0u;
    m.hphase = 0u;
    const int vec = m.wp->vec;
    if (vec < 0) return;  // idle warp of a short patch
    const int n = bp.nt, t0 = bp.t0;

    // the lane that holds this lane's neighbour inside the source vector (which vector: the plan's masks)
    const unsigned x = ((unsigned)vec * VL + lane) % (unsigned)LX;
    const unsigned lane_xf = (x + 1u == (unsigned)LX) ? (lane - (unsigned)(LX - 1)) & 31u : (lane + 1u) & 31u;
    const unsigned lane_xb = (x == 0u) ? (lane + (unsigned)(LX - 1)) & 31u : (lane - 1u) & 31u;
    const unsigned lane_yf = (lane + (unsigned)LX) & 31u, lane_yb = (lane - (unsigned)LX) & 31u;

    // prologue: U_t(x,t0-1)^dagger P^+_t psi(x,t0-1), the backward t contribution of the first step, operands straight from
    // global memory (once per block; in the loop it is carried in registers from the previous step)
    cplx<Real> wt[6];
    {
        const int tb = (t0 == 0) ? LT - 1 : t0 - 1;
        const unsigned sb = (unsigned)(((size_t)vec + (size_t)slice_vecs * (size_t)tb) * VL) + lane;
        cplx<Real> psi[12], u[9], h[6];
        SpinorIO<Real, LAYOUT_SOA>::load(psi, in_, V, sb);
        load_link<Real, LAYOUT_SOA, RECON>(u, gauge_, V, sb, 3);
        project<3, +1>(h, psi);
        su3_mul<true>(wt, u, h);
    }

#pragma unroll 1
    for (int i = 0; i < n; ++i) {
        m.step = i;
        cplx<Real> acc[12];
        {
            cplx<Real> u[9], psi[12], h[6], hp[6];
            m.fetch_link(u, lane);
            m.template publish<0>(u, m.wp->own_done != 0 && m.late);
            m.template gather_fwd<0>(psi, lane_xf);
            project<0, -1>(h, psi);
            su3_mul<false>(hp, u, h);
            reconstruct_accumulate<0, -1, true>(acc, hp);
            m.template gather_bwd<0>(hp, lane_xb);
            reconstruct_accumulate<0, +1, false>(acc, hp);
        }
        m.template forward_phase<1>(acc, lane_yf);
        m.template forward_phase<2>(acc, lane);
        {
            cplx<Real> u[9], h[6], hp[6];
            m.fetch_link(u, lane);
            {
                cplx<Real> psi[12];
                m.read_ring(psi, w, 1, false, lane, true);
                project<3, -1>(h, psi);
            }
            su3_mul<false>(hp, u, h);
            reconstruct_accumulate<3, -1, false>(acc, hp);
            reconstruct_accumulate<3, +1, false>(acc, wt);
            {
                cplx<Real> own[12];
                m.read_own(own, !m.late);
                project<3, +1>(h, own);
            }
            su3_mul<true>(wt, u, h);
        }
        {
            cplx<Real> wv[6];
            m.template gather_bwd<1>(wv, lane_yb);
            reconstruct_accumulate<1, +1, false>(acc, wv);
            m.template gather_bwd<2>(wv, lane);
            reconstruct_accumulate<2, +1, false>(acc, wv);
        }
        int t = t0 + i;
        if (t >= LT) t -= LT;
        const unsigned s = (unsigned)(((size_t)vec + (size_t)slice_vecs * (size_t)t) * VL) + lane;
        if (hints & 8)  // `out` is not read again by this application
            SpinorIO<Real, LAYOUT_SOA>::template store<1>(out, V, s, acc, make_policy(POLICY_EVICT_FIRST));
        else
            SpinorIO<Real, LAYOUT_SOA>::store(out, V, s, acc);
    }
}

// ------------------------------------------------------------------ host: decomposition and plan
int gcd_int(int a, int b) { return b == 0 ? a : gcd_int(b, a % b); }

// Units of the (y,z) plane in an order whose every run of consecutive units is a compact patch: strips of two z planes, a
// snake in y inside a strip, the strips joined end to end (the order dslash_march.cu uses for rows).
void snake_units(int NY, int LZ, std::vector<int>& order) {
    bool up = true;
    for (int zs = 0; zs < LZ; zs += 2) {
        const int wz = std::min(2, LZ - zs);
        for (int iy = 0; iy < NY; ++iy) {
            const int y = up ? iy : NY - 1 - iy;
            for (int iz = 0; iz < wz; ++iz) {
                const int z = zs + (((iy & 1) == 0) ? iz : wz - 1 - iz);
                order.push_back(y + NY * z);
            }
        }
        up = !up;
    }
}

// S segments of the unit list x G chunks of the time range for blocks of at most `ub` units of `nvu` vectors; returns the
// estimated cost.  The model of march_plan_shape (dslash_march.cu) -- waves x steps x time of a step, a chunk costing about
// 1.5 steps of prologue -- with a step that takes a fixed latency chain (about what six warps' worth of work takes) plus
// time in proportion to the warps of the block: without the fixed part one-warp blocks in many waves look cheapest.
double gm_shape(int NU, int nvu, int NT, int ub, int wave, int* S_out, int* G_out) {
    const int s_min = (NU + ub - 1) / ub;
    double best = 0.0;
    for (int G = 1; G <= NT && G <= MARCH_MAX_CHUNKS; ++G) {
        const int chunk = (NT + G - 1) / G;
        long long waves = ((long long)s_min * G + wave - 1) / wave;
        int S = (int)std::min<long long>(NU, std::max<long long>(s_min, waves * wave / G));
        waves = ((long long)S * G + wave - 1) / wave;
        const int units_max = (NU + S - 1) / S;
        const double cost = (double)waves * (6.0 + units_max * nvu) * (chunk + 1.5);
        if (best == 0.0 || cost < best * 0.999) {
            best = cost;
            *S_out = S;
            *G_out = G;
        }
    }
    return best;
}

struct GmGeom {
    int LX, LY, LZ, nvu, nru, NY, NU, slice_vecs;
};
GmGeom gm_geom(const Geom& g) {
    GmGeom q;
    q.LX = g.L[0];
    q.LY = g.L[1];
    q.LZ = g.L[2];
    const int unit = q.LX / gcd_int(q.LX, (int)VL) * (int)VL;  // lcm(L_X, 32) sites
    q.nvu = unit / (int)VL;
    q.nru = unit / q.LX;
    q.NY = q.LY / q.nru;
    q.NU = q.NY * q.LZ;
    q.slice_vecs = q.LX * q.LY * q.LZ / (int)VL;
    return q;
}

// The blocks of a decomposition into S segments x G chunks with at most GM_NWB_MAX exchange buffers per block; returns the
// largest number of exchange buffers a block uses, or -1 if some hop has more than GM_SRC_MAX source vectors.
int gm_fill_plan(const GmGeom& q, int t_begin, int NT, int S, int G, std::vector<GmBlockPlan>& plan) {
    std::vector<int> order;
    order.reserve(q.NU);
    snake_units(q.NY, q.LZ, order);
    // block-local warp of every vector of the slice, per segment
    std::vector<int> seg_of(q.slice_vecs), loc_of(q.slice_vecs);
    for (int s = 0; s < S; ++s) {
        const int a = (int)((long long)s * q.NU / S), b = (int)((long long)(s + 1) * q.NU / S);
        for (int k = a; k < b; ++k) {
            const int uy = order[k] % q.NY, uz = order[k] / q.NY;
            const int v0 = (uz * q.LY * q.LX + uy * q.nru * q.LX) / (int)VL;  // first vector of the unit
            for (int j = 0; j < q.nvu; ++j) {
                seg_of[v0 + j] = s;
                loc_of[v0 + j] = (k - a) * q.nvu + j;
            }
        }
    }
    plan.assign((size_t)S * G, GmBlockPlan());
    int nwb_max = 0;
    const int plane = q.LX * q.LY;
    for (int s = 0; s < S; ++s) {
        const int a = (int)((long long)s * q.NU / S), b = (int)((long long)(s + 1) * q.NU / S);
        GmBlockPlan bp;
        bp.t0 = bp.nt = bp.chunk = 0;
        bp.nact = (b - a) * q.nvu;
        for (int r = 0; r < GM_NW_MAX; ++r) bp.ring_readers[r] = 0;
        for (int r = 0; r < GM_NWB_MAX; ++r) bp.wbuf_readers[r] = 0;
        std::vector<int> vec_of(bp.nact);
        for (int wi = 0; wi < GM_NW_MAX; ++wi) {
            GmWarpPlan& wp = bp.w[wi];
            wp.vec = -1;
            wp.own_done = 1;
            wp.link_shared = 0u;
            for (int d = 0; d < 3; ++d) {
                wp.wr[d] = -1;
                wp.nf[d] = wp.nb[d] = 0;
                for (int e = 0; e < GM_SRC_MAX; ++e) wp.f[d][e] = wp.b[d][e] = GmSrc{0, 0u};
            }
        }
        for (int k = a; k < b; ++k) {
            const int uy = order[k] % q.NY, uz = order[k] / q.NY;
            const int v0 = (uz * q.LY * q.LX + uy * q.nru * q.LX) / (int)VL;
            for (int j = 0; j < q.nvu; ++j) {
                bp.w[(k - a) * q.nvu + j].vec = v0 + j;
                vec_of[(k - a) * q.nvu + j] = v0 + j;
            }
        }
        // neighbour vectors of every lane, per warp and direction; sources in order of first appearance
        // tmp_b[wi][d][e] = source VECTOR of backward entry e (resolved to an exchange buffer or a halo below)
        std::vector<int> tmp_b((size_t)bp.nact * 3 * GM_SRC_MAX, -1);
        for (int wi = 0; wi < bp.nact; ++wi) {
            GmWarpPlan& wp = bp.w[wi];
            for (int l = 0; l < (int)VL; ++l) {
                const int sl = wp.vec * (int)VL + l;
                const int x = sl % q.LX, y = (sl / q.LX) % q.LY, z = sl / plane;
                const int nf[3] = {sl - x + (x + 1) % q.LX, sl + ((y + 1) % q.LY - y) * q.LX, sl + ((z + 1) % q.LZ - z) * plane};
                const int nb[3] = {sl - x + (x + q.LX - 1) % q.LX, sl + ((y + q.LY - 1) % q.LY - y) * q.LX,
                                   sl + ((z + q.LZ - 1) % q.LZ - z) * plane};
                for (int d = 0; d < 3; ++d) {
                    // forward: ring row of this block or halo vector
                    const int vf = nf[d] / (int)VL;
                    const int idf = seg_of[vf] == s ? loc_of[vf] : -vf - 1;
                    int e = 0;
                    while (e < wp.nf[d] && wp.f[d][e].id != idf) ++e;
                    if (e == wp.nf[d]) {
                        if (e == GM_SRC_MAX) return -1;
                        wp.f[d][wp.nf[d]++] = GmSrc{idf, 0u};
                    }
                    wp.f[d][e].mask |= 1u << l;
                    if (idf < 0) wp.link_shared |= 1u << d;  // the owner of that site comes back for U_d of this lane's site
                    // backward: remember the source vector
                    const int vb = nb[d] / (int)VL;
                    int* tb = &tmp_b[((size_t)wi * 3 + d) * GM_SRC_MAX];
                    e = 0;
                    while (e < wp.nb[d] && tb[e] != vb) ++e;
                    if (e == wp.nb[d]) {
                        if (e == GM_SRC_MAX) return -1;
                        tb[wp.nb[d]++] = vb;
                    }
                    wp.b[d][e].mask |= 1u << l;
                }
            }
            if (wp.link_shared & 1u) return -1;  // x neighbours never leave the block (whole units)
        }
        // exchange buffers: one per (writer warp, direction) that has a reader in this block, as long as buffers last;
        // x first (an x hop has no halo form), then y, then z
        int nslot = 0;
        for (int d = 0; d < 3; ++d)
            for (int wi = 0; wi < bp.nact; ++wi)
                for (int e = 0; e < bp.w[wi].nb[d]; ++e) {
                    const int vb = tmp_b[((size_t)wi * 3 + d) * GM_SRC_MAX + e];
                    if (seg_of[vb] != s) continue;
                    GmWarpPlan& src = bp.w[loc_of[vb]];
                    if (src.wr[d] < 0 && nslot < GM_NWB_MAX) src.wr[d] = nslot++;
                }
        for (int wi = 0; wi < bp.nact; ++wi)
            for (int d = 0; d < 3; ++d)
                for (int e = 0; e < bp.w[wi].nb[d]; ++e) {
                    const int vb = tmp_b[((size_t)wi * 3 + d) * GM_SRC_MAX + e];
                    int id = -vb - 1;
                    if (seg_of[vb] == s && bp.w[loc_of[vb]].wr[d] >= 0) {
                        id = bp.w[loc_of[vb]].wr[d];
                        bp.wbuf_readers[id] += 1;
                    } else if (d == 0) {
                        return -1;  // out of buffers for an x hop
                    }
                    bp.w[wi].b[d][e].id = id;
                }
        nwb_max = std::max(nwb_max, nslot);
        // ring rows: who reads them, and which read is a warp's last one in a step (program order: own spinors, then the
        // forward sources of x, y, z)
        for (int wi = 0; wi < bp.nact; ++wi) {
            GmWarpPlan& wp = bp.w[wi];
            int last_d[GM_NW_MAX], last_e[GM_NW_MAX];
            for (int r = 0; r < GM_NW_MAX; ++r) last_d[r] = last_e[r] = -1;
            for (int d = 0; d < 3; ++d)
                for (int e = 0; e < wp.nf[d]; ++e)
                    if (wp.f[d][e].id >= 0) {
                        last_d[wp.f[d][e].id] = d;
                        last_e[wp.f[d][e].id] = e;
                    }
            for (int r = 0; r < bp.nact; ++r) {
                if (last_d[r] >= 0) {
                    wp.f[last_d[r]][last_e[r]].id |= 0x100;
                    bp.ring_readers[r] += 1;
                    if (r == wi) wp.own_done = 0;
                } else if (r == wi) {
                    bp.ring_readers[r] += 1;  // the owner always reads its row
                }
            }
        }
        for (int c = 0; c < G; ++c) {
            const int ta = t_begin + (int)((long long)c * NT / G), tb = t_begin + (int)((long long)(c + 1) * NT / G);
            bp.t0 = ta;
            bp.nt = tb - ta;
            bp.chunk = c;
            plan[(size_t)c * S + s] = bp;
        }
    }
    return nwb_max;
}

unsigned gm_cwg(int precision) { return precision == 0 ? 2u : 3u; }

}  // namespace

bool gmarch_eligible(int precision, int layout_base, int recon, const Geom& g) {
    (void)recon;
    if (layout_base != LAYOUT_SOA) return false;
    if ((g.L[0] * g.L[1]) % (int)VL != 0) return false;
    const GmGeom q = gm_geom(g);
    // a unit must fit the compute warps of a block: 8 at 232 registers (fp64), 12 at 152 (fp32)
    return q.nvu <= (precision == 0 ? 8 : GM_NW_MAX);
}

int gmarch_plan_build(int precision, int recon, const Geom& g, int t_begin, int t_end, int wave, int max_units, GmShape* shape,
                      GmBlockPlan* plan_out, size_t capacity_blocks) {
    const int NT = t_end - t_begin;
    if (NT < 1 || wave < 1 || !gmarch_eligible(precision, LAYOUT_SOA, recon, g)) return 0;
    const GmGeom q = gm_geom(g);
    const int nw_cap = precision == 0 ? 8 : GM_NW_MAX;
    // candidates: blocks of ub units; the smallest estimated cost among those whose minimal configuration (2 link slots,
    // 1 halo slot per warp) fits in shared memory wins; what is left over goes to more slots
    double best = 0.0;
    GmShape bs{};
    std::vector<GmBlockPlan> best_plan, plan;
    int ub_max = nw_cap / q.nvu;
    if (max_units > 0) ub_max = std::min(ub_max, max_units);
    for (int ub = ub_max; ub >= 1; --ub) {
        int S = 0, G = 1;
        const double cost = gm_shape(q.NU, q.nvu, NT, ub, wave, &S, &G);
        if (best != 0.0 && cost >= best * 0.999) continue;
        const int nwb = gm_fill_plan(q, t_begin, NT, S, G, plan);
        if (nwb < 0) continue;
        const int NW = ((q.NU + S - 1) / S) * q.nvu;
        GmLayout L = gm_layout(precision, recon, NW, 2, 1, nwb);
        if (L.total > GM_SMEM_MAX) continue;
        int NLS = 2, NHS = 1;
        // more data in flight while shared memory lasts: third link slot, second halo slot, fourth link slot, third halo slot
        const int try_l[4] = {3, 3, 4, 4}, try_h[4] = {1, 2, 2, 3};
        for (int k = 0; k < 4; ++k) {
            L = gm_layout(precision, recon, NW, try_l[k], try_h[k], nwb);
            if (L.total > GM_SMEM_MAX) break;
            NLS = try_l[k];
            NHS = try_h[k];
        }
        L = gm_layout(precision, recon, NW, NLS, NHS, nwb);
        best = cost;
        bs.NW = NW;
        bs.NLS = NLS;
        bs.NHS = NHS;
        bs.NWB = nwb;
        bs.units_per_block = (q.NU + S - 1) / S;
        bs.vecs_per_unit = q.nvu;
        bs.S = S;
        bs.G = G;
        bs.smem_bytes = L.total;
        best_plan.swap(plan);
    }
    if (best == 0.0) return 0;
    if (shape) *shape = bs;
    if (plan_out) {
        if (capacity_blocks < best_plan.size()) return 0;
        std::copy(best_plan.begin(), best_plan.end(), plan_out);
    }
    return (int)best_plan.size();
}

cudaError_t gmarch_plan_create(int precision, int recon, const Geom& g, int t_begin, int t_end, int device, int max_units, void** d_plan,
                               int* nblocks, GmShape* shape) {
    int sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    if (*d_plan) {
        if ((e = cudaFree(*d_plan)) != cudaSuccess) return e;
        *d_plan = nullptr;
    }
    *nblocks = 0;
    const int nb = gmarch_plan_build(precision, recon, g, t_begin, t_end, sms, max_units, shape, nullptr, 0);
    if (nb < 1) return cudaErrorInvalidValue;
    std::vector<GmBlockPlan> plan((size_t)nb);
    if (gmarch_plan_build(precision, recon, g, t_begin, t_end, sms, max_units, shape, plan.data(), plan.size()) != nb) return cudaErrorInvalidValue;
    if ((e = cudaMalloc(d_plan, plan.size() * sizeof(GmBlockPlan))) != cudaSuccess) {
        *d_plan = nullptr;
        return e;
    }
    if ((e = cudaMemcpy(*d_plan, plan.data(), plan.size() * sizeof(GmBlockPlan), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    *nblocks = nb;
    return cudaSuccess;
}

namespace {

template <typename Real, int RECON, int CWG>
cudaError_t launch_gmarch_k(const LaunchArgs& a, const GmBlockPlan* d_plan, int nblocks, const GmLayout& L, int hints) {
    auto kernel = dslash_gmarch_kernel<Real, RECON, CWG>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total);
    if (e != cudaSuccess) return e;
    kernel<<<(unsigned)nblocks, 128 * (1 + CWG), L.total, a.stream>>>(a.out, a.in, a.gauge, a.geom.V,
                                                                      a.geom.L[0] * a.geom.L[1] * a.geom.L[2] / (int)VL, a.geom.L[0], a.geom.L[3],
                                                                      d_plan, L, hints);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_gmarch(int precision, int layout_base, int recon, const LaunchArgs& a, const void* d_plan, int nblocks,
                          const GmShape& shape, const TunedConfig& cfg) {
    if (!gmarch_eligible(precision, layout_base, recon, a.geom) || !d_plan || nblocks < 1) return cudaErrorInvalidConfiguration;
    const GmLayout L = gm_layout(precision, recon, shape.NW, shape.NLS, shape.NHS, shape.NWB);
    if (L.total > GM_SMEM_MAX || shape.NW > (int)(4u * gm_cwg(precision))) return cudaErrorInvalidConfiguration;
    const GmBlockPlan* p = static_cast<const GmBlockPlan*>(d_plan);
    const int h = cfg.march_policy >= 0 ? cfg.march_policy : (4 | 8 | 16);  // the defaults dslash_march.cu measured
    if (precision == 0)
        return recon == 12 ? launch_gmarch_k<double, 12, 2>(a, p, nblocks, L, h) : launch_gmarch_k<double, 18, 2>(a, p, nblocks, L, h);
    return recon == 12 ? launch_gmarch_k<float, 12, 3>(a, p, nblocks, L, h) : launch_gmarch_k<float, 18, 3>(a, p, nblocks, L, h);
}

}  // namespace dslash

// Host-only view of the plan (no device needed): what tests/test_gmarch_plan.py checks.
extern "C" int dslash_gmarch_plan(const int dims[4], int precision, int recon, int t_begin, int t_end, int wave, int shape[9], int* ints,
                                  size_t capacity_ints, int* nblocks) {
    if (!dims || !nblocks) return DSLASH_ERR_NULL;
    for (int d = 0; d < 4; ++d)
        if (dims[d] < 1) return DSLASH_ERR_DIMS;
    if (precision != DSLASH_FP64 && precision != DSLASH_FP32) return DSLASH_ERR_PRECISION;
    if (recon != 12 && recon != 18) return DSLASH_ERR_LAYOUT;
    dslash::Geom g;
    unsigned long long V = 1;
    for (int d = 0; d < 4; ++d) {
        g.L[d] = dims[d];
        V *= (unsigned long long)dims[d];
        if (V * 36ull >= (1ull << 31)) return DSLASH_ERR_DIMS;
    }
    g.V = (unsigned)V;
    if (t_begin < 0 || t_end > dims[3] || t_begin >= t_end || wave < 1) return DSLASH_ERR_UNSUPPORTED;
    if (!dslash::gmarch_eligible(precision, dslash::LAYOUT_SOA, recon, g)) return DSLASH_ERR_UNSUPPORTED;
    dslash::GmShape sh{};
    const int nb = dslash::gmarch_plan_build(precision, recon, g, t_begin, t_end, wave, 0, &sh, nullptr, 0);
    if (nb < 1) return DSLASH_ERR_UNSUPPORTED;
    *nblocks = nb;
    if (shape) {
        const int v[9] = {sh.NW, sh.NLS, sh.NHS, sh.NWB, sh.units_per_block, sh.vecs_per_unit, sh.S, sh.G, (int)sh.smem_bytes};
        for (int k = 0; k < 9; ++k) shape[k] = v[k];
    }
    if (ints) {
        const size_t per = sizeof(dslash::GmBlockPlan) / sizeof(int);
        if (capacity_ints < per * (size_t)nb) return DSLASH_ERR_UNSUPPORTED;
        std::vector<dslash::GmBlockPlan> plan((size_t)nb);
        if (dslash::gmarch_plan_build(precision, recon, g, t_begin, t_end, wave, 0, &sh, plan.data(), plan.size()) != nb) return DSLASH_ERR_UNSUPPORTED;
        std::copy(reinterpret_cast<const int*>(plan.data()), reinterpret_cast<const int*>(plan.data()) + per * (size_t)nb, ints);
    }
    return DSLASH_OK;
}

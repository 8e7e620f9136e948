// dslash_march.cu -- block-cooperative, t-marching, warp-specialised Dslash kernel (DSLASH_KERNEL_MARCH), sm_100a.
//
// Same operator and the same per-hop arithmetic as dslash_tuned.cu (Eq. 1), the eight hop contributions
// summed in the same order (ORDER below): results are bit-identical to the direct kernel.  What changes is how often an
// operand crosses the L2 -> SM crossbar.  The direct kernel pulls 1.94 KB per site through it for 0.96 KB of compulsory
// HBM traffic, the warp-pipelined kernel 2.35 KB; under sustained load (board at its power cap, ~1.45 GHz) that crossbar
// traffic and the instructions that move it are what bound them (profiles/r01d, r01f).  Here
//
//   * a thread block owns a PATCH of x rows (L_X == 32: one row = one 32-site vector = one consumer warp; up to 7 rows that
//     are neighbours in the (y,z) plane) and MARCHES through the time slices t0 .. t0+nt-1;
//   * every link is fetched ONCE, by the warp that owns its site, and used for both products it appears in:
//     the forward hop of its own site,  U_mu(x) P^-_mu psi(x+mu^),  and the complete backward-hop contribution of the
//     neighbour,  w_mu(x) = U_mu(x)^dagger P^+_mu psi(x)  (what the site x+mu^ adds).  w travels: in x by warp shuffle,
//     in y and z through a 3 KB shared-memory exchange buffer to the neighbouring warp of the block, in t in registers
//     to the next step of the same thread.  With 12-real links row 2 is therefore rebuilt once per link, not twice;
//   * every spinor row of the patch is fetched ONCE (one 6 KB bulk async copy) into a two-slot shared-memory ring, where
//     it serves as psi(t+1) of the forward t hop, then as the row's own spinor and as the y/z neighbour of other warps;
//   * only the rows around the patch (halo) are fetched a second time: a forward halo hop needs the neighbour's spinor,
//     a backward halo hop its spinor and its link;
//   * NOTHING is loaded by LDG inside the loop: links stream through NLS per-warp slots, halo spinors through one
//     per-warp slot, all by cp.async.bulk (SASS UBLKCP) with completion counted on mbarriers.
//
// Warp specialisation.  Seven warps compute (one row each).  Four PRODUCER warps feed them: the block has 21 copy queues
// (7 link streams, 7 halo-spinor streams, 7 ring rows), each owned by one lane of a producer warp, which polls the queue's
// "empty" mbarrier (test_wait, never blocking) and issues the next bulk copy of the stream once its slot has been released.
// setmaxnreg gives the producers 40 registers per thread and the compute warps 232.  The compute warps never issue a
// copy, a proxy fence or an expect_tx: a stage costs them one try_wait, the LDS.128s, and one mbarrier.arrive by lane 0.
// There is NO block barrier inside the loop: the exchange buffers and the ring rows are handed over warp to warp through
// full/empty mbarrier pairs, so a warp only ever waits for the one neighbour it needs (ncu of the barrier version:
// 18.6 % of the warp samples sat in the two __syncthreads() of a step, 6 % behind lane 0's fence + expect_tx).
//
// L2 -> SM traffic per site (fp64, 7-row patches of 32^3x64): 192 (psi) + 576 (links) + ~460 (halo) = 1.23 KB.
// The patches are cut from a snake through the (y,z) plane so that 148 blocks x 7 warps cover 32 x 32 rows in ONE wave,
// all blocks marching through t together: a halo row is in L2 because its owner fetched it two steps earlier.
//
// ORDER of the sum (fixed, independent of how the plane is cut into patches):
//   x forward, x backward, y forward, z forward, t forward, t backward, y backward, z backward.
// (The t hops sit between producing the exchange buffers and consuming them: moving them to the end of the step, where
// their late-fetched operand psi(t+1) would have more time, exposes the wait for the neighbour warp instead: 0.344 -> 0.389 ms.)
#include <algorithm>
#include <vector>

#define DSLASH_F32X2  // packed FP32 arithmetic (FFMA2 / FADD2), see dslash_site.cuh
#include "../../include/dslash_b200.h"
#include "dslash_async.cuh"
#include "dslash_kernels.cuh"

// A producer warp with nothing to issue sleeps this long.  Measured in one call (DSLASH_NVCC_EXTRA=-DMARCH_IDLE_NS=..., burst /
// sustained ms on 32^3x64 fp64): 32 ns 0.3397 / 0.3760, 128 ns 0.3421 / 0.3792, 512 ns 0.3774 / 0.3896, 2000 ns 0.4262 / 0.4345:
// a late refill costs more than the polling instructions do, also under the power cap.
#ifndef MARCH_IDLE_NS
#define MARCH_IDLE_NS 32
#endif

namespace dslash {

namespace {

template <typename Real, int RECON, int NLS>
struct MarchSmem {
    static constexpr unsigned NW = MARCH_NW;
    static constexpr unsigned NWS = MARCH_NWS;
    static constexpr unsigned PSI = 24u * VL * sizeof(Real);                          // one spinor vector (6144 B in fp64)
    static constexpr unsigned LINK = (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);   // one (vector, mu) link block (4608 B)
    static constexpr unsigned HALF = 12u * VL * sizeof(Real);                         // one half-spinor vector (3072 B)
    // mbarriers (indices into a uint64 array at offset 0)
    static constexpr unsigned B_RING_FULL = 0u;                     // [2][NW]   a ring row has landed
    static constexpr unsigned B_RING_EMPTY = B_RING_FULL + 2u * NW; // [2][NW]   every reader of the row is done with it
    static constexpr unsigned B_LFULL = B_RING_EMPTY + 2u * NW;     // [NW][NLS] link slots
    static constexpr unsigned B_LEMPTY = B_LFULL + NW * NLS;
    static constexpr unsigned B_HFULL = B_LEMPTY + NW * NLS;        // [NW]      halo spinor slot
    static constexpr unsigned B_HEMPTY = B_HFULL + NW;
    static constexpr unsigned B_WFULL = B_HEMPTY + NW;              // [NWS]     exchange buffers
    static constexpr unsigned B_WEMPTY = B_WFULL + NWS;
    static constexpr unsigned B_COUNT = B_WEMPTY + NWS;
    static constexpr unsigned TABLE = 1024u;                        // uint32 [3 * NW][8]: the producers' stage tables (units of 256 B)
    static constexpr unsigned HEADER = 2048u;
    static constexpr unsigned RING = HEADER;                        // [2][NW][PSI]
    static constexpr unsigned LSLOT = RING + 2u * NW * PSI;         // [NW][NLS][LINK]
    static constexpr unsigned HSLOT = LSLOT + NW * NLS * LINK;      // [NW][PSI]
    static constexpr unsigned WBUF = HSLOT + NW * PSI;              // [NWS][HALF]
    static constexpr unsigned TOTAL = WBUF + NWS * HALF;
    static_assert(TOTAL <= 232448u, "exceeds the 227 KB of shared memory a block may have");
    static_assert(B_COUNT * 8u <= TABLE && TABLE + 3u * NW * 8u * 4u <= HEADER, "header layout");
    static_assert(PSI % 256u == 0 && LINK % 256u == 0, "stage tables hold offsets in units of 256 bytes");
};

// State of one compute warp.  Every member is warp-uniform except `lane`.
template <typename Real, int RECON, int NLS>
struct MarchWarp {
    using S = MarchSmem<Real, RECON, NLS>;
    unsigned char* smem;
    uint64_t* bars;
    MarchWarpPlan wp;
    unsigned lane, w;
    int step;                 // current step i
    int lslot;                // link slot of the next stage to consume
    unsigned lphase, hphase;  // parity of the next completion: bit s = link slot s; halo slot

    // "this warp is done with the buffer": all lanes have issued their reads/writes, lane 0 tells the other side
    __device__ __forceinline__ void hand_over(uint64_t* bar) const {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar);
    }
    // next link stage of this warp -> registers
    __device__ __forceinline__ void fetch_link(cplx<Real> (&u)[9]) {
        const unsigned b = w * NLS + (unsigned)lslot;
        mbar_wait_spin(bars + S::B_LFULL + b, (lphase >> lslot) & 1u);
        load_link_slot<Real, RECON>(u, smem + S::LSLOT + b * S::LINK, lane);
        hand_over(bars + S::B_LEMPTY + b);
        lphase ^= 1u << lslot;
        lslot = (lslot + 1 == NLS) ? 0 : lslot + 1;
    }
    // next halo spinor stage of this warp -> registers
    __device__ __forceinline__ void fetch_halo(cplx<Real> (&psi)[12]) {
        mbar_wait_spin(bars + S::B_HFULL + w, hphase);
        load_psi_slot<Real>(psi, smem + S::HSLOT + w * S::PSI, lane);
        hand_over(bars + S::B_HEMPTY + w);
        hphase ^= 1u;
    }
    // ring row `r` of the slice of step `step` + ahead (ahead = 0: current slice, 1: next slice); done = this was the warp's last read
    __device__ __forceinline__ void read_ring(cplx<Real> (&psi)[12], unsigned r, int ahead, bool done) const {
        const unsigned q = (unsigned)(step + ahead), b = (q & 1u) * S::NW + r;
        mbar_wait_spin(bars + S::B_RING_FULL + b, (q >> 1) & 1u);
        load_psi_slot<Real>(psi, smem + S::RING + b * S::PSI, lane);
        if (done) hand_over(bars + S::B_RING_EMPTY + b);
    }

    // y (MU = 1) or z (MU = 2): the link of the own site gives the neighbour's backward contribution and the own forward hop
    template <int MU>
    __device__ __forceinline__ void forward_phase(cplx<Real> (&acc)[12], const cplx<Real> (&own)[12]) {
        constexpr int d = MU - 1;
        cplx<Real> u[9];
        fetch_link(u);
        if (wp.wr[d] >= 0) {
            cplx<Real> h[6], wv[6];
            project<MU, +1>(h, own);
            su3_mul<true>(wv, u, h);
            const unsigned b = (unsigned)wp.wr[d];
            if (step > 0) mbar_wait_spin(bars + S::B_WEMPTY + b, ((unsigned)step - 1u) & 1u);  // the reader took the previous one
            store_half<Real>(smem + S::WBUF + b * S::HALF, lane, wv);
            hand_over(bars + S::B_WFULL + b);
        }
        cplx<Real> psi[12];
        if (wp.fwd[d] >= 0)
            read_ring(psi, (unsigned)wp.fwd[d], 0, true);
        else
            fetch_halo(psi);
        hop_regs<MU, -1>(acc, psi, u);
    }
    // w = U_MU(row)^dagger P+_MU psi(row) of a halo row (next stages of the halo and link streams)
    template <int MU>
    __device__ __forceinline__ void halo_backward(cplx<Real> (&wv)[6]) {
        cplx<Real> psi[12], u[9], h[6];
        fetch_halo(psi);
        fetch_link(u);
        project<MU, +1>(h, psi);
        su3_mul<true>(wv, u, h);
    }
    // backward hop in y or z: from the exchange buffer when the neighbour row belongs to this block, else a halo hop
    template <int MU>
    __device__ __forceinline__ void backward_phase(cplx<Real> (&acc)[12]) {
        constexpr int d = MU - 1;
        cplx<Real> wv[6];
        if (wp.rd[d] >= 0) {
            const unsigned b = (unsigned)wp.rd[d];
            mbar_wait_spin(bars + S::B_WFULL + b, (unsigned)step & 1u);
            load_half<Real>(wv, smem + S::WBUF + b * S::HALF, lane);
            hand_over(bars + S::B_WEMPTY + b);
        } else {
            halo_backward<MU>(wv);
        }
        reconstruct_accumulate<MU, +1, false>(acc, wv);
    }
};

// A producer warp: each of its first lanes owns one of the block's 3 * NW copy queues -- queue / NW = 0: the link stream of
// compute warp queue % NW (NLS slots), 1: its halo spinor stream (one slot), 2: its ring row (two slots, slices t0 .. t0+n).  A queue is a cyclic list of
// `nstage` sources per step; fill number q goes to slot q % nslots and may be issued once the slot's previous fill has been
// released (its "empty" barrier has completed round - 1 phases).
template <typename Real, int RECON, int NLS>
__device__ __forceinline__ void march_producer(unsigned char* smem, const unsigned char* in, const unsigned char* gauge,
                                               const MarchBlockPlan& bp, unsigned queue, int slice_rows, int LT, int hints,
                                               const unsigned* progress, unsigned target, int lead) {
    using S = MarchSmem<Real, RECON, NLS>;
    constexpr unsigned NW = MARCH_NW;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    // stages of one step in the order the compute warp consumes them, as offsets (in 256-byte units) into the field at t = 0:
    //   links:  U_x, U_y, U_z, U_t of the own row; U_y(y-), U_z(z-) of the warp's halo hops
    //   halo spinors: psi(y+), psi(z+), psi(y-), psi(z-) as far as those rows are not in the block
    uint32_t* tab = reinterpret_cast<uint32_t*>(smem + S::TABLE) + (queue < 3u * NW ? queue : 0u) * 8u;
    const unsigned qw = queue % NW, kind = queue / NW;
    const int n = bp.nt, t0 = bp.t0;
    int nstage = 0, total = 0, nslots = 1;
    unsigned bytes = 0, dst = 0, dst_stride = 0, bar_full = 0, bar_empty = 0, bar_stride = 1;
    const unsigned char* src = in;
    size_t slice_stride = 0;
    if (kind < 3u) {
        const MarchWarpPlan pw = bp.w[qw];
        if (pw.row >= 0) {
            constexpr unsigned LU = S::LINK / 256u, PU = S::PSI / 256u;
            if (kind == 0u) {
                for (int mu = 0; mu < 4; ++mu) tab[nstage++] = ((unsigned)pw.row * 4u + (unsigned)mu) * LU;
                if (pw.rd[0] < 0) tab[nstage++] = ((unsigned)pw.bwd[0] * 4u + 1u) * LU;
                if (pw.rd[1] < 0) tab[nstage++] = ((unsigned)pw.bwd[1] * 4u + 2u) * LU;
                total = nstage * n;
                nslots = NLS;
                bytes = S::LINK;
                src = gauge;
                slice_stride = (size_t)slice_rows * 4u * S::LINK;
                dst = S::LSLOT + qw * NLS * S::LINK;
                dst_stride = S::LINK;
                bar_full = S::B_LFULL + qw * NLS;
                bar_empty = S::B_LEMPTY + qw * NLS;
            } else if (kind == 1u) {
                if (pw.fwd[0] < 0) tab[nstage++] = (unsigned)(-pw.fwd[0] - 1) * PU;
                if (pw.fwd[1] < 0) tab[nstage++] = (unsigned)(-pw.fwd[1] - 1) * PU;
                if (pw.rd[0] < 0) tab[nstage++] = (unsigned)pw.bwd[0] * PU;
                if (pw.rd[1] < 0) tab[nstage++] = (unsigned)pw.bwd[1] * PU;
                total = nstage * n;
                bytes = S::PSI;
                slice_stride = (size_t)slice_rows * S::PSI;
                dst = S::HSLOT + qw * S::PSI;
                bar_full = S::B_HFULL + qw;
                bar_empty = S::B_HEMPTY + qw;
            } else {
                tab[nstage++] = (unsigned)pw.row * PU;
                total = n + 1;
                nslots = 2;
                bytes = S::PSI;
                slice_stride = (size_t)slice_rows * S::PSI;
                dst = S::RING + qw * S::PSI;
                dst_stride = NW * S::PSI;
                bar_full = S::B_RING_FULL + qw;
                bar_empty = S::B_RING_EMPTY + qw;
                bar_stride = NW;
            }
        }
    }
    // L2 eviction policies (DSLASH_OPT_L2_POLICY bits).  4: what is read exactly once per application is evict_first -- U_x, U_t,
    // and U_y / U_z of rows whose forward neighbour is in the block (with bits 8 and 16: HBM reads 1.80 -> 1.63 GB on 32^3x64,
    // 1.011 x compulsory).  1: what ANOTHER block reads too is evict_last -- every spinor row and the links a halo hop of another
    // block needs (U_y / U_z of a row whose y+ / z+ neighbour is outside the block, the halo links themselves); measured
    // harmful (1.77 GB with 4, 8, 16 also set), so it is not part of the default.
    const uint64_t pol_shared = (hints & 1) ? make_policy(POLICY_EVICT_LAST) : 0ull;
    const uint64_t pol_stream = (hints & 4) ? make_policy(POLICY_EVICT_FIRST) : 0ull;
    unsigned shared_stage = ~0u;  // bit k: stage k of this queue is read by another block as well
    if (kind == 0u && queue < 3u * NW) shared_stage = ~0xFu | (bp.w[qw].fwd[0] < 0 ? 2u : 0u) | (bp.w[qw].fwd[1] < 0 ? 4u : 0u);
    // Throttle (lead > 0): the blocks of a chunk share the halo rows through L2, which only works while they are within a step
    // or two of each other (measured without it: 4 steps apart at mid-march, 8 % more HBM reads).  Every compute warp counts
    // the steps it starts in progress[step] (global memory, accumulating over launches: `target` = the count that means "all
    // rows of the chunk, this launch").  A ring row of slice q is fetched while the block is in step q - 2, so it is held back
    // until every row of the chunk has started step q - 2 - lead.  Purely a hint: after ~50 us without progress (blocks of the
    // chunk not resident: a multi-wave plan, a second stream) the block stops looking.
    int allowed = lead > 0 ? lead + 1 : 0x7fffffff;  // ring fills up to this slice need not ask
    int patience = 400;
    int q = 0, k = 0, i = 0, slot = 0, round = 0;
    while (__any_sync(0xffffffffu, q < total)) {
        bool ready = false;
        if (q < total) ready = round == 0 || mbar_test(bars + bar_empty + (unsigned)slot * bar_stride, ((unsigned)round - 1u) & 1u);
        // Late ring fill (DSLASH_OPT_L2_POLICY bit 16): slice q of a row is needed at the END of step q - 1, but its slot is free
        // from early in step q - 2.  Fetching it that early puts ~2 steps (60 MB of traffic) between the owner's fetch and the
        // neighbouring blocks' halo fetches of the same row, which is about what one L2 partition holds.  Hold the fill back until
        // the readers of slice q - 1 are done too (the block is well inside step q - 1): the two fetches are then ~1 step apart.
        // (Gating on "the row's own warp has started step q - 1" instead, half a step earlier, was measured slower.)
        if (ready && kind == 2u && (hints & 16) && q >= 2)
            ready = mbar_test(bars + bar_empty + (unsigned)(slot ^ 1) * bar_stride, (((unsigned)q - 1u) >> 1) & 1u);
        if (ready && kind == 2u && q > allowed) {
            // steps s <= q - 2 - lead must have been started by everyone; progress only ever grows, so look ahead as well
            int s = q - 2 - lead;
            const unsigned v = *reinterpret_cast<const volatile unsigned*>(progress + s);
            if ((int)(v - target) >= 0) {
                allowed = q;
                patience = 400;
            } else if (--patience < 0) {
                allowed = 0x7fffffff;
            } else {
                ready = false;
            }
        }
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
        if (!__any_sync(0xffffffffu, ready)) __nanosleep(MARCH_IDLE_NS);
    }
}

// Register split between the roles (setmaxnreg works on warpgroups of four warps): the block is launched with
// 384 threads x 168 registers; warpgroup 0 (four producer warps) shrinks to 40 registers per thread, warpgroups 1 and 2
// (the compute warps) grow to 232: 128 x 40 + 256 x 232 = 64512 <= 65536.
constexpr int MARCH_THREADS = 384, MARCH_PRODUCER_WARPS = 4, MARCH_REGS_PRODUCER = 40, MARCH_REGS_COMPUTE = 232;

template <typename Real, int RECON, int NLS>
__global__ void __launch_bounds__(MARCH_THREADS, 1)
    dslash_march_kernel(void* __restrict__ out, const void* __restrict__ in_, const void* __restrict__ gauge_, unsigned V, int slice_rows,
                        int LT, const MarchBlockPlan* __restrict__ plan, int hints, unsigned* __restrict__ stats,
                        unsigned* __restrict__ progress, unsigned target, int lead) {
    using S = MarchSmem<Real, RECON, NLS>;
    constexpr unsigned NW = MARCH_NW;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const long long clock_begin = clock64();
    const MarchBlockPlan& bp = plan[blockIdx.x];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);

    // one thread per mbarrier.  Every barrier takes ONE arrival per phase (the producer's expect_tx, or lane 0 of the one warp
    // that hands the buffer over), except "ring row r is free": the row's own warp and every warp that reads it as y+/z+ neighbour
    if (threadIdx.x < S::B_COUNT) {
        unsigned count = 1u;
        if (threadIdx.x >= S::B_RING_EMPTY && threadIdx.x < S::B_LFULL) {
            const int r = (int)((threadIdx.x - S::B_RING_EMPTY) % NW);
            for (int q = 0; q < bp.nact; ++q) count += (unsigned)(bp.w[q].fwd[0] == r) + (unsigned)(bp.w[q].fwd[1] == r);
        }
        mbar_init(bars + threadIdx.x, count);
        mbar_fence_init();
    }
    __syncthreads();

    if (warp < (unsigned)MARCH_PRODUCER_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(MARCH_REGS_PRODUCER));
        // queue q is served by lane q / 4 of producer warp q % 4: the copies of one compute warp are spread over the producers
        const unsigned queue = lane < 6u ? warp + (unsigned)MARCH_PRODUCER_WARPS * lane : 3u * NW;
        march_producer<Real, RECON, NLS>(smem, static_cast<const unsigned char*>(in_), static_cast<const unsigned char*>(gauge_), bp, queue,
                                         slice_rows, LT, hints, progress + (size_t)bp.chunk * (unsigned)LT, target, lead);
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(MARCH_REGS_COMPUTE));
    const unsigned w = warp - (unsigned)MARCH_PRODUCER_WARPS;  // compute warp number
    if (w >= NW) return;
    MarchWarp<Real, RECON, NLS> m;
    m.smem = smem;
    m.bars = bars;
    m.wp = bp.w[w];
    m.lane = lane;
    m.w = w;
    m.lslot = 0;
    m.lphase = 0u;
    m.hphase = 0u;
    if (m.wp.row < 0) return;  // idle warp of a short patch
    const int n = bp.nt, t0 = bp.t0;

    // prologue: U_t(x,t0-1)^dagger P^+_t psi(x,t0-1), the backward t contribution of the first step, operands straight from
    // global memory (once per block; in the loop it is carried in registers from the previous step)
    cplx<Real> wt[6];
    {
        const int tb = (t0 == 0) ? LT - 1 : t0 - 1;
        const unsigned sb = (unsigned)(((size_t)m.wp.row + (size_t)slice_rows * (size_t)tb) * VL) + lane;
        cplx<Real> psi[12], u[9], h[6];
        SpinorIO<Real, LAYOUT_SOA>::load(psi, in_, V, sb);
        load_link<Real, LAYOUT_SOA, RECON>(u, gauge_, V, sb, 3);
        project<3, +1>(h, psi);
        su3_mul<true>(wt, u, h);
    }
    const int lane_fwd = (int)((lane + 1u) & 31u), lane_bwd = (int)((lane - 1u) & 31u);

#pragma unroll 1
    for (int i = 0; i < n; ++i) {
        m.step = i;
        if (lead > 0 && lane == 0) atomicAdd(progress + (size_t)bp.chunk * (unsigned)LT + (unsigned)i, 1u);  // this row has started step i
        if (stats && i == (n >> 1) && w == 0 && lane == 0) {  // wall-clock time at mid-march: how far the blocks have drifted apart
            unsigned long long ns;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns));
            stats[3u * blockIdx.x + 2u] = (unsigned)ns;
        }
        cplx<Real> acc[12], own[12];
        m.read_ring(own, w, 0, true);  // the row's own spinors: the warp's last read of this fill (it was psi(t+1) a step ago)
        {
            cplx<Real> u[9];
            m.fetch_link(u);
            x_hops_regs(acc, own, u, lane_fwd, lane_bwd);
        }
        m.template forward_phase<1>(acc, own);
        m.template forward_phase<2>(acc, own);
        {
            cplx<Real> u[9], psi[12], h[6], hp[6];
            m.fetch_link(u);
            m.read_ring(psi, w, 1, false);
            project<3, -1>(h, psi);
            su3_mul<false>(hp, u, h);
            reconstruct_accumulate<3, -1, false>(acc, hp);
            reconstruct_accumulate<3, +1, false>(acc, wt);
            project<3, +1>(h, own);
            su3_mul<true>(wt, u, h);
        }
        m.template backward_phase<1>(acc);
        m.template backward_phase<2>(acc);
        int t = t0 + i;
        if (t >= LT) t -= LT;
        const unsigned s = (unsigned)(((size_t)m.wp.row + (size_t)slice_rows * (size_t)t) * VL) + lane;
        if (hints & 8)  // `out` is not read again by this application
            SpinorIO<Real, LAYOUT_SOA>::template store<1>(out, V, s, acc, make_policy(POLICY_EVICT_FIRST));
        else
            SpinorIO<Real, LAYOUT_SOA>::store(out, V, s, acc);
    }
    if (stats && w == 0 && lane == 0) {  // dslash_march_stats(): where this block ran and how long its first compute warp took
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        stats[3u * blockIdx.x] = smid;
        stats[3u * blockIdx.x + 1u] = (unsigned)(clock64() - clock_begin);
    }
}

// ------------------------------------------------------------------ host: the block plan
// Rows of the (y,z) plane in an order whose every run of consecutive rows is a compact patch: strips of two z planes,
// a snake in y inside a strip, the strips joined end to end.
void snake_rows(int LY, int LZ, std::vector<int>& order) {
    bool up = true;
    for (int zs = 0; zs < LZ; zs += 2) {
        const int wz = std::min(2, LZ - zs);
        for (int iy = 0; iy < LY; ++iy) {
            const int y = up ? iy : LY - 1 - iy;
            for (int iz = 0; iz < wz; ++iz) {
                const int z = zs + (((iy & 1) == 0) ? iz : wz - 1 - iz);
                order.push_back(y + LY * z);
            }
        }
        up = !up;
    }
}

}  // namespace

bool march_eligible(int layout_base, const Geom& g) { return layout_base == LAYOUT_SOA && g.L[0] == (int)VL; }

// S segments of the plane x G chunks of the time range; `wave` = blocks that are resident at the same time.
void march_plan_shape(const Geom& g, int t_begin, int t_end, int wave, int* S_out, int* G_out) {
    const int NR = g.L[1] * g.L[2], NT = t_end - t_begin;
    const int s_min = (NR + MARCH_NW - 1) / MARCH_NW;
    double best = 0.0;
    int bestS = s_min, bestG = 1;
    for (int G = 1; G <= NT && G <= MARCH_MAX_CHUNKS; ++G) {
        const int chunk = (NT + G - 1) / G;
        long long waves = ((long long)s_min * G + wave - 1) / wave;
        int S = (int)std::min<long long>(NR, std::max<long long>(s_min, waves * wave / G));
        waves = ((long long)S * G + wave - 1) / wave;
        const int rows_max = (NR + S - 1) / S;
        // a step costs time in proportion to the rows of the block; a chunk costs about 1.5 steps of prologue
        const double cost = (double)waves * rows_max * (chunk + 1.5);
        if (best == 0.0 || cost < best * 0.999) {
            best = cost;
            bestS = S;
            bestG = G;
        }
    }
    *S_out = bestS;
    *G_out = bestG;
}

int march_plan_build(const Geom& g, int t_begin, int t_end, int wave, std::vector<MarchBlockPlan>& plan) {
    const int LY = g.L[1], LZ = g.L[2], NR = LY * LZ, NT = t_end - t_begin;
    if (NT < 1 || wave < 1) return 0;
    int S, G;
    march_plan_shape(g, t_begin, t_end, wave, &S, &G);
    std::vector<int> order;
    order.reserve(NR);
    snake_rows(LY, LZ, order);
    std::vector<int> seg_of(NR), loc_of(NR);
    for (int s = 0; s < S; ++s) {
        const int a = (int)((long long)s * NR / S), b = (int)((long long)(s + 1) * NR / S);
        for (int k = a; k < b; ++k) {
            seg_of[order[k]] = s;
            loc_of[order[k]] = k - a;
        }
    }
    plan.assign((size_t)S * G, MarchBlockPlan());
    for (int c = 0; c < G; ++c) {
        const int ta = t_begin + (int)((long long)c * NT / G), tb = t_begin + (int)((long long)(c + 1) * NT / G);
        for (int s = 0; s < S; ++s) {
            MarchBlockPlan& bp = plan[(size_t)c * S + s];
            const int a = (int)((long long)s * NR / S), b = (int)((long long)(s + 1) * NR / S);
            bp.t0 = ta;
            bp.nt = tb - ta;
            bp.nact = b - a;
            bp.chunk = c;
            for (int wi = 0; wi < MARCH_NW; ++wi) {
                MarchWarpPlan& wp = bp.w[wi];
                wp.row = -1;
                wp.fwd[0] = wp.fwd[1] = -1;
                wp.wr[0] = wp.wr[1] = wp.rd[0] = wp.rd[1] = -1;
                wp.bwd[0] = wp.bwd[1] = 0;
            }
            int nslot = 0;
            for (int k = a; k < b; ++k) {
                const int row = order[k], y = row % LY, z = row / LY;
                MarchWarpPlan& wp = bp.w[k - a];
                wp.row = row;
                const int nb_f[2] = {(y + 1) % LY + LY * z, y + LY * ((z + 1) % LZ)};
                const int nb_b[2] = {(y + LY - 1) % LY + LY * z, y + LY * ((z + LZ - 1) % LZ)};
                for (int d = 0; d < 2; ++d) {
                    wp.fwd[d] = seg_of[nb_f[d]] == s ? loc_of[nb_f[d]] : -nb_f[d] - 1;
                    wp.bwd[d] = nb_b[d];
                }
            }
            // exchange buffers: one per (producer row, direction) whose forward neighbour is a row of this block
            for (int k = a; k < b; ++k) {
                MarchWarpPlan& wp = bp.w[k - a];
                for (int d = 0; d < 2; ++d)
                    if (wp.fwd[d] >= 0 && nslot < MARCH_NWS) {
                        wp.wr[d] = nslot;
                        bp.w[wp.fwd[d]].rd[d] = nslot;
                        ++nslot;
                    }
            }
        }
    }
    return S * G;
}

namespace {

template <typename Real, int RECON, int NLS>
cudaError_t launch_march_k(const LaunchArgs& a, const MarchBlockPlan* d_plan, int nblocks, int hints, unsigned* stats, unsigned* progress,
                           unsigned target, int lead) {
    using S = MarchSmem<Real, RECON, NLS>;
    dslash_march_kernel<Real, RECON, NLS><<<(unsigned)nblocks, MARCH_THREADS, S::TOTAL, a.stream>>>(
        a.out, a.in, a.gauge, a.geom.V, a.geom.L[1] * a.geom.L[2], a.geom.L[3], d_plan, hints, stats, progress, target, lead);
    return cudaGetLastError();
}

template <typename Real, int RECON, int NLS>
cudaError_t prepare_march_k() {
    return cudaFuncSetAttribute(dslash_march_kernel<Real, RECON, NLS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)MarchSmem<Real, RECON, NLS>::TOTAL);
}

}  // namespace

// What a launch needs from the runtime besides the plan, done once where the kernel is selected (the current device must be
// `device`): the dynamic shared-memory limit of this precision/recon's instantiation and the SM count.  launch_march() then
// makes no CUDA runtime query.
cudaError_t march_prepare(int precision, int recon, int device, int* sms) {
    cudaError_t e = cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    if (precision == 0) return recon == 12 ? prepare_march_k<double, 12, 3>() : prepare_march_k<double, 18, 2>();
    return recon == 12 ? prepare_march_k<float, 12, 4>() : prepare_march_k<float, 18, 4>();
}

// The plan is followed in device memory by 3 * nblocks unsigned: {SM id, cycles, globaltimer (ns, low word) at mid-march} of
// every block of the last launch, then by MARCH_MAX_CHUNKS * L_T progress counters (zero when the plan is made).
// sms: SM count from march_prepare().  *epoch counts the launches on this plan that ran WITH the throttle (lead > 0): only those
// add to the progress counters, so only those may move the target the counters are compared with.
cudaError_t launch_march(int precision, int layout_base, int recon, const LaunchArgs& a, const void* d_plan, int nblocks, const TunedConfig& cfg,
                         int sms, unsigned* epoch) {
    if (!march_eligible(layout_base, a.geom) || !d_plan || nblocks < 1 || !epoch) return cudaErrorInvalidConfiguration;
    const MarchBlockPlan* p = static_cast<const MarchBlockPlan*>(d_plan);
    unsigned* st = reinterpret_cast<unsigned*>(const_cast<MarchBlockPlan*>(p + nblocks));
    unsigned* pr = st + 3u * (unsigned)nblocks;
    // default policy of this kernel (measured, profiles/r02_march.md): 4 read-once links evict_first, 8 stores evict_first,
    // 16 late ring fill; 1 (shared data evict_last) is harmful
    const int h = cfg.march_policy >= 0 ? cfg.march_policy : (4 | 8 | 16);
    // the throttle needs every block of a chunk resident at the same time: single-wave plans only
    const int lead = nblocks <= sms ? cfg.march_lead : 0;
    if (lead > 0) ++*epoch;
    const unsigned target = *epoch * (unsigned)(a.geom.L[1] * a.geom.L[2]);  // rows of a chunk x throttled launches so far (mod 2^32)
    cudaError_t e;
    if (precision == 0)
        e = recon == 12 ? launch_march_k<double, 12, 3>(a, p, nblocks, h, st, pr, target, lead)
                        : launch_march_k<double, 18, 2>(a, p, nblocks, h, st, pr, target, lead);
    else
        e = recon == 12 ? launch_march_k<float, 12, 4>(a, p, nblocks, h, st, pr, target, lead)
                        : launch_march_k<float, 18, 4>(a, p, nblocks, h, st, pr, target, lead);
    if (e != cudaSuccess && lead > 0) --*epoch;  // nothing ran, nothing was counted
    return e;
}

// Builds the plan for the time range and uploads it (synchronous: cudaMalloc + cudaMemcpy).  *d_plan must be NULL or a plan
// made by this function (it is freed first).
cudaError_t march_plan_create(const Geom& g, int t_begin, int t_end, int device, void** d_plan, int* nblocks) {
    int sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    std::vector<MarchBlockPlan> plan;
    const int nb = march_plan_build(g, t_begin, t_end, sms, plan);
    if (*d_plan) {
        if ((e = cudaFree(*d_plan)) != cudaSuccess) return e;
        *d_plan = nullptr;
    }
    *nblocks = 0;
    if (nb < 1) return cudaErrorInvalidValue;
    const size_t extra = (plan.size() * 3 + (size_t)MARCH_MAX_CHUNKS * (size_t)g.L[3]) * sizeof(unsigned);  // stats + progress
    if ((e = cudaMalloc(d_plan, plan.size() * sizeof(MarchBlockPlan) + extra)) != cudaSuccess) {
        *d_plan = nullptr;
        return e;
    }
    if ((e = cudaMemset(static_cast<MarchBlockPlan*>(*d_plan) + plan.size(), 0, extra)) != cudaSuccess) return e;
    if ((e = cudaMemcpy(*d_plan, plan.data(), plan.size() * sizeof(MarchBlockPlan), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    *nblocks = nb;
    return cudaSuccess;
}

}  // namespace dslash

// Host-only view of the plan (no device needed): what tests/test_march_plan.py checks.
extern "C" int dslash_march_plan(const int dims[4], int t_begin, int t_end, int wave, int* ints, size_t capacity_ints, int* nblocks) {
    if (!dims || !nblocks) return DSLASH_ERR_NULL;
    for (int d = 0; d < 4; ++d)
        if (dims[d] < 1) return DSLASH_ERR_DIMS;
    if (dims[0] != (int)dslash::VL || t_begin < 0 || t_end > dims[3] || t_begin >= t_end || wave < 1) return DSLASH_ERR_UNSUPPORTED;
    dslash::Geom g;
    for (int d = 0; d < 4; ++d) g.L[d] = dims[d];
    g.V = (unsigned)dims[0] * (unsigned)dims[1] * (unsigned)dims[2] * (unsigned)dims[3];
    std::vector<dslash::MarchBlockPlan> plan;
    const int nb = dslash::march_plan_build(g, t_begin, t_end, wave, plan);
    *nblocks = nb;
    const size_t need = plan.size() * (sizeof(dslash::MarchBlockPlan) / sizeof(int));
    if (ints) {
        if (capacity_ints < need) return DSLASH_ERR_UNSUPPORTED;
        std::copy(reinterpret_cast<const int*>(plan.data()), reinterpret_cast<const int*>(plan.data()) + need, ints);
    }
    return DSLASH_OK;
}

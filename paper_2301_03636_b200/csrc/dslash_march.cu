// dslash_march.cu -- block-cooperative, t-marching, async-staged Dslash kernel (DSLASH_KERNEL_MARCH), sm_100a.
//
// Same operator and the same per-hop arithmetic as dslash_tuned.cu (Eq. 1), the eight hop contributions
// summed in the same order (x-, x+, y-, z-, t- forward projector first ... see ORDER below): results are bit-identical
// to the direct kernel.  What changes is how often an operand crosses the L2 -> SM crossbar.  The direct kernel pulls
// 1.94 KB per site through it for 0.96 KB of compulsory HBM traffic, the warp-pipelined kernel 2.35 KB; under sustained
// load (board at its power cap, ~1.45 GHz) that crossbar traffic is what bounds them (profiles/r01d, r01f).  Here
//
//   * a thread block owns a PATCH of x rows (L_X == 32: one row = one 32-site vector = one warp; up to 7 rows that are
//     neighbours in the (y,z) plane) and MARCHES through the time slices t0 .. t0+nt-1;
//   * every link is fetched ONCE, by the warp that owns its site, and used for both products it appears in:
//     the forward hop of its own site,  U_mu(x) P^-_mu psi(x+mu^),  and the complete backward-hop contribution of the
//     neighbour,  w_mu(x) = U_mu(x)^dagger P^+_mu psi(x)  (what the site x+mu^ adds).  w travels: in x by warp shuffle,
//     in y and z through a 3 KB shared-memory exchange buffer to the neighbouring warp of the block, in t in registers
//     to the next step of the same thread.  With 12-real links row 2 is therefore rebuilt once per link, not twice;
//   * every spinor row of the patch is fetched ONCE (one 6 KB bulk async copy, two steps before its slice is computed)
//     into a two-slot shared-memory ring, where it serves as psi(t+1) of the forward t hop, then as the row's own
//     spinor and as the y/z neighbour of up to four other warps;
//   * only the rows around the patch (halo) are fetched a second time: a forward halo hop needs the neighbour's spinor,
//     a backward halo hop its spinor and its link;
//   * NOTHING is loaded by LDG: links stream through NLS per-warp slots, halo spinors through one per-warp slot, all by
//     cp.async.bulk (SASS UBLKCP) with completion counted on mbarriers, refilled the moment they have been read.
//
// L2 -> SM traffic per site (fp64, 7-row patches of 32^3x64): 192 (psi) + 576 (links) + ~390 (halo) = ~1.16 KB.
// The patches are cut from a snake through the (y,z) plane so that 148 blocks x 7 warps cover 32 x 32 rows in ONE wave,
// all blocks marching through t together: a halo row is in L2 because its owner fetched it two steps earlier.
//
// ORDER of the sum (fixed, independent of how the plane is cut into patches):
//   x forward, x backward, y forward, z forward, t forward, t backward, y backward, z backward.
//
// Synchronisation per step: two block barriers.  B2 (before the first exchange-buffer write of the step) and B1 (after
// the last one).  After B1 the ring slot of the current slice is dead and each warp refills its own row with slice t+2.
#include <algorithm>
#include <vector>

#include "../../include/dslash_b200.h"
#include "dslash_async.cuh"
#include "dslash_kernels.cuh"

namespace dslash {

namespace {

template <typename Real, int RECON, int NLS>
struct MarchSmem {
    static constexpr unsigned NW = MARCH_NW;
    static constexpr unsigned PSI = 24u * VL * sizeof(Real);                          // one spinor vector (6144 B in fp64)
    static constexpr unsigned LINK = (RECON == 12 ? 12u : 18u) * VL * sizeof(Real);   // one (vector, mu) link block (4608 B)
    static constexpr unsigned HALF = 12u * VL * sizeof(Real);                         // one half-spinor vector (3072 B)
    static constexpr unsigned HEADER = 1024u;                                         // mbarriers, per-warp stage tables
    static constexpr unsigned RING = HEADER;                                          // [2][NW][PSI]
    static constexpr unsigned LSLOT = RING + 2u * NW * PSI;                           // [NW][NLS][LINK]
    static constexpr unsigned HSLOT = LSLOT + NW * NLS * LINK;                        // [NW][PSI]
    static constexpr unsigned WBUF = HSLOT + NW * PSI;                                // [MARCH_NWS][HALF]
    static constexpr unsigned TOTAL = WBUF + MARCH_NWS * HALF;
    static_assert(TOTAL <= 232448u, "exceeds the 227 KB of shared memory a block may have");
    static_assert(16u + 8u * NW * (NLS + 1u) <= 512u && 512u + 64u * NW <= HEADER, "header layout");
};

template <typename Real>
__device__ __forceinline__ void store_half(unsigned char* p, unsigned lane, const cplx<Real> (&h)[6]) {
    using V2 = typename vec2<Real>::type;
    V2* q = reinterpret_cast<V2*>(p) + lane;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        V2 v;
        v.x = h[k].re;
        v.y = h[k].im;
        q[k * VL] = v;
    }
}
template <typename Real>
__device__ __forceinline__ void load_half(cplx<Real> (&h)[6], const unsigned char* p, unsigned lane) {
    using V2 = typename vec2<Real>::type;
    const V2* q = reinterpret_cast<const V2*>(p) + lane;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const V2 v = q[k * VL];
        h[k] = {v.x, v.y};
    }
}

// State of one warp of the marching block.  Every member is warp-uniform except `lane`.
template <typename Real, int RECON, int NLS>
struct March {
    using S = MarchSmem<Real, RECON, NLS>;
    const unsigned char* in;
    const unsigned char* gauge;
    unsigned char* ring;       // the block's ring: [2][NW][PSI]
    unsigned char* lslots;     // this warp's NLS link slots
    unsigned char* hslot;      // this warp's halo spinor slot
    unsigned char* wbuf;       // the block's exchange buffers
    uint64_t* ring_full;       // [2]
    uint64_t* lbar;            // this warp's NLS link-slot mbarriers
    uint64_t* hbar;            // this warp's halo-slot mbarrier
    const int* ltab;           // link stages of one step in consumption order: (mu << 28) | row
    const int* htab;           // halo spinor stages of one step in consumption order: row
    MarchWarpPlan wp;
    unsigned lane, w;
    int slice_rows, LT, t0, n;
    int nL, nH;                // stages per step
    int lk, li, hk, hi;        // next stage to ISSUE: index within the step, step
    int lslot;                 // link slot of the next stage to consume
    unsigned lphase, hphase;   // parity of the next completion: bit s = link slot s; halo slot
    uint64_t pol_link;         // L2 policy of the link copies (0: none)

    __device__ __forceinline__ int tslice(int i) const {
        const int t = t0 + i;
        return t >= LT ? t - LT : t;
    }
    __device__ __forceinline__ size_t vec_of(int row, int i) const { return (size_t)row + (size_t)slice_rows * (size_t)tslice(i); }

    // called by lane 0
    __device__ __forceinline__ void issue_link(int k, int i, unsigned char* dst, uint64_t* bar) const {
        const unsigned e = (unsigned)ltab[k];
        const unsigned mu = e >> 28;
        const size_t vec = vec_of((int)(e & 0x0fffffffu), i);
        mbar_arrive_expect_tx(bar, S::LINK);
        const unsigned char* src = gauge + (vec * 4u + mu) * S::LINK;
        if (pol_link)
            bulk_g2s_hint(dst, src, S::LINK, bar, pol_link);
        else
            bulk_g2s(dst, src, S::LINK, bar);
    }
    __device__ __forceinline__ void issue_psi(int row, int i, unsigned char* dst, uint64_t* bar) const {
        mbar_arrive_expect_tx(bar, S::PSI);
        bulk_g2s(dst, in + vec_of(row, i) * S::PSI, S::PSI, bar);
    }

    // next link stage of this warp -> registers; its slot is refilled at once with the stage NLS ahead
    __device__ __forceinline__ void fetch_link(cplx<Real> (&u)[9]) {
        unsigned char* sp = lslots + (unsigned)lslot * S::LINK;
        uint64_t* bar = lbar + lslot;
        mbar_wait_spin(bar, (lphase >> lslot) & 1u);
        load_link_slot<Real, RECON>(u, sp, lane);
        __syncwarp();  // every lane has its copy
        lphase ^= 1u << lslot;
        if (lane == 0 && li < n) {
            fence_proxy_async();  // generic-proxy reads above before the async-proxy refill
            issue_link(lk, li, sp, bar);
        }
        if (++lk == nL) {
            lk = 0;
            ++li;
        }
        lslot = (lslot + 1 == NLS) ? 0 : lslot + 1;
    }
    // next halo spinor stage of this warp -> registers; the slot is refilled with the following one
    __device__ __forceinline__ void fetch_halo(cplx<Real> (&psi)[12]) {
        mbar_wait_spin(hbar, hphase);
        load_psi_slot<Real>(psi, hslot, lane);
        __syncwarp();
        hphase ^= 1u;
        if (lane == 0 && hi < n) {
            fence_proxy_async();
            issue_psi(htab[hk], hi, hslot, hbar);
        }
        if (++hk == nH) {
            hk = 0;
            ++hi;
        }
    }

    // y (MU = 1) or z (MU = 2): the link of the own site gives the neighbour's backward contribution and the own forward hop
    template <int MU>
    __device__ __forceinline__ void forward_phase(cplx<Real> (&acc)[12], const cplx<Real> (&own)[12], const unsigned char* ring_cur) {
        constexpr int d = MU - 1;
        cplx<Real> u[9];
        fetch_link(u);
        if (wp.wr[d] >= 0) {
            cplx<Real> h[6], wv[6];
            project<MU, +1>(h, own);
            su3_mul<true>(wv, u, h);
            store_half<Real>(wbuf + (unsigned)wp.wr[d] * S::HALF, lane, wv);
        }
        cplx<Real> psi[12];
        if (wp.fwd[d] >= 0)
            load_psi_slot<Real>(psi, ring_cur + (unsigned)wp.fwd[d] * S::PSI, lane);
        else
            fetch_halo(psi);
        hop_regs<MU, -1>(acc, psi, u);
    }
    // backward hop in y or z: from the exchange buffer when the neighbour row belongs to this block, else a halo hop
    template <int MU>
    __device__ __forceinline__ void backward_phase(cplx<Real> (&acc)[12]) {
        constexpr int d = MU - 1;
        cplx<Real> wv[6];
        if (wp.rd[d] >= 0) {
            load_half<Real>(wv, wbuf + (unsigned)wp.rd[d] * S::HALF, lane);
        } else {
            cplx<Real> psi[12], u[9], h[6];
            fetch_halo(psi);
            fetch_link(u);
            project<MU, +1>(h, psi);
            su3_mul<true>(wv, u, h);
        }
        reconstruct_accumulate<MU, +1, false>(acc, wv);
    }
};

template <typename Real, int RECON, int NLS>
__global__ void __launch_bounds__(MARCH_NW * 32, 1)
    dslash_march_kernel(void* __restrict__ out, const void* __restrict__ in_, const void* __restrict__ gauge_, unsigned V, int slice_rows,
                        int LT, const MarchBlockPlan* __restrict__ plan, int hints) {
    using S = MarchSmem<Real, RECON, NLS>;
    constexpr unsigned NW = MARCH_NW;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const MarchBlockPlan& bp = plan[blockIdx.x];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    int* tab = reinterpret_cast<int*>(smem + 512) + w * 16;  // [0..5] link stages, [8..11] halo stages

    March<Real, RECON, NLS> m;
    m.in = static_cast<const unsigned char*>(in_);
    m.gauge = static_cast<const unsigned char*>(gauge_);
    m.ring = smem + S::RING;
    m.lslots = smem + S::LSLOT + w * (NLS * S::LINK);
    m.hslot = smem + S::HSLOT + w * S::PSI;
    m.wbuf = smem + S::WBUF;
    m.ring_full = bars;
    m.lbar = bars + 2 + w * NLS;
    m.hbar = bars + 2 + NW * NLS + w;
    m.ltab = tab;
    m.htab = tab + 8;
    m.wp = bp.w[w];
    m.lane = lane;
    m.w = w;
    m.slice_rows = slice_rows;
    m.LT = LT;
    m.t0 = bp.t0;
    m.n = bp.nt;
    m.pol_link = (hints & 4) ? make_policy(POLICY_EVICT_FIRST) : 0ull;
    const bool active = m.wp.row >= 0;
    const int n = m.n;

    // stage tables of this warp (consumption order inside a step)
    int nL = 4, nH = 0;
    if (lane == 0 && active) {
        tab[0] = (0 << 28) | m.wp.row;
        tab[1] = (1 << 28) | m.wp.row;
        tab[2] = (2 << 28) | m.wp.row;
        tab[3] = (3 << 28) | m.wp.row;
    }
    if (active) {
        if (m.wp.fwd[0] < 0) {
            if (lane == 0) tab[8 + nH] = -m.wp.fwd[0] - 1;
            ++nH;
        }
        if (m.wp.fwd[1] < 0) {
            if (lane == 0) tab[8 + nH] = -m.wp.fwd[1] - 1;
            ++nH;
        }
        if (m.wp.rd[0] < 0) {
            if (lane == 0) {
                tab[8 + nH] = m.wp.bwd[0];
                tab[nL] = (1 << 28) | m.wp.bwd[0];
            }
            ++nH;
            ++nL;
        }
        if (m.wp.rd[1] < 0) {
            if (lane == 0) {
                tab[8 + nH] = m.wp.bwd[1];
                tab[nL] = (2 << 28) | m.wp.bwd[1];
            }
            ++nH;
            ++nL;
        }
    }
    m.nL = nL;
    m.nH = nH;
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], (unsigned)bp.nact);
        mbar_init(&bars[1], (unsigned)bp.nact);
    }
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NLS; ++s) mbar_init(m.lbar + s, 1u);
        mbar_init(m.hbar, 1u);
        mbar_fence_init();
    }
    __syncthreads();

    cplx<Real> wt[6];  // U_t(x,t-1)^dagger P^+_t psi(x,t-1): the backward t contribution carried from the previous step
    if (active) {
        if (lane == 0) {
            // ring: slices t0 and t0+1 (the forward t hop of the first step needs the second one)
            m.issue_psi(m.wp.row, 0, m.ring + (0u * NW + w) * S::PSI, &bars[0]);
            m.issue_psi(m.wp.row, 1, m.ring + (1u * NW + w) * S::PSI, &bars[1]);
#pragma unroll
            for (int s = 0; s < NLS; ++s) m.issue_link(s, 0, m.lslots + (unsigned)s * S::LINK, m.lbar + s);  // NLS <= 4 <= nL
            if (nH > 0) m.issue_psi(tab[8], 0, m.hslot, m.hbar);
        }
        m.lk = NLS;
        m.li = 0;
        if (m.lk >= nL) {
            m.lk -= nL;
            m.li = 1;
        }
        m.hk = nH > 1 ? 1 : 0;
        m.hi = nH > 1 ? 0 : 1;
        m.lslot = 0;
        m.lphase = 0u;
        m.hphase = 0u;
        // prologue: the backward t contribution of slice t0 - 1, operands straight from global memory (once per block)
        const int tb = (m.t0 == 0) ? LT - 1 : m.t0 - 1;
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
        const unsigned cur = (unsigned)i & 1u, nxt = cur ^ 1u;
        const unsigned char* ring_cur = m.ring + cur * NW * S::PSI;
        cplx<Real> acc[12], own[12];
        if (active) {
            mbar_wait_spin(&bars[cur], ((unsigned)i >> 1) & 1u);
            load_psi_slot<Real>(own, ring_cur + w * S::PSI, lane);
            cplx<Real> u[9];
            m.fetch_link(u);
            x_hops_regs(acc, own, u, lane_fwd, lane_bwd);
        }
        __syncthreads();  // B2: the exchange buffers of the previous step have been read
        if (active) {
            m.template forward_phase<1>(acc, own, ring_cur);
            m.template forward_phase<2>(acc, own, ring_cur);
        }
        __syncthreads();  // B1: every exchange buffer of this step is written; nobody reads ring[cur] any more
        if (active) {
            if (lane == 0 && i + 2 <= n) {
                fence_proxy_async();
                m.issue_psi(m.wp.row, i + 2, m.ring + (cur * NW + w) * S::PSI, &bars[cur]);
            }
            {
                cplx<Real> u[9], psi[12], h[6], hp[6];
                m.fetch_link(u);
                mbar_wait_spin(&bars[nxt], (((unsigned)i + 1u) >> 1) & 1u);
                load_psi_slot<Real>(psi, m.ring + (nxt * NW + w) * S::PSI, lane);
                project<3, -1>(h, psi);
                su3_mul<false>(hp, u, h);
                reconstruct_accumulate<3, -1, false>(acc, hp);
                reconstruct_accumulate<3, +1, false>(acc, wt);
                project<3, +1>(h, own);
                su3_mul<true>(wt, u, h);
            }
            m.template backward_phase<1>(acc);
            m.template backward_phase<2>(acc);
            const unsigned s = (unsigned)(m.vec_of(m.wp.row, i) * VL) + lane;
            SpinorIO<Real, LAYOUT_SOA>::store(out, V, s, acc);
        }
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
    for (int G = 1; G <= NT && G <= 64; ++G) {
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
            bp.pad = 0;
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
cudaError_t launch_march_k(const LaunchArgs& a, const MarchBlockPlan* d_plan, int nblocks, int hints) {
    using S = MarchSmem<Real, RECON, NLS>;
    auto kernel = dslash_march_kernel<Real, RECON, NLS>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::TOTAL);
    if (e != cudaSuccess) return e;
    kernel<<<(unsigned)nblocks, MARCH_NW * 32, S::TOTAL, a.stream>>>(a.out, a.in, a.gauge, a.geom.V, a.geom.L[1] * a.geom.L[2], a.geom.L[3],
                                                                      d_plan, hints);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_march(int precision, int layout_base, int recon, const LaunchArgs& a, const void* d_plan, int nblocks, const TunedConfig& cfg) {
    if (!march_eligible(layout_base, a.geom) || !d_plan || nblocks < 1) return cudaErrorInvalidConfiguration;
    const MarchBlockPlan* p = static_cast<const MarchBlockPlan*>(d_plan);
    if (precision == 0)
        return recon == 12 ? launch_march_k<double, 12, 3>(a, p, nblocks, cfg.l2_policy) : launch_march_k<double, 18, 2>(a, p, nblocks, cfg.l2_policy);
    return recon == 12 ? launch_march_k<float, 12, 4>(a, p, nblocks, cfg.l2_policy) : launch_march_k<float, 18, 4>(a, p, nblocks, cfg.l2_policy);
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
    if ((e = cudaMalloc(d_plan, plan.size() * sizeof(MarchBlockPlan))) != cudaSuccess) {
        *d_plan = nullptr;
        return e;
    }
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

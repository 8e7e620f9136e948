// dslash_ring.cu -- t-marching Dslash kernel with a shared-memory ring of spinor time slices (DSLASH_KERNEL_RING), sm_100a.
//
// Same operator, same per-hop arithmetic and the same hop order as dslash_tuned.cu (Eq. 1; results
// bit-identical).  What changes is where the spinors come from.  The direct kernel moves 1.95 KB per site from L2 into the
// SMs for 0.96 KB of compulsory HBM traffic.  Here a block owns a SPATIAL tile of 32 x by x bz sites (one warp per x row =
// one 32-site vector of the blocked SoA layout) and marches over a chunk of time slices.  The spinors of the tile's rows at
// t, t+1 (and t+2 in flight) live in a ring of three shared-memory slots, each row brought in ONCE by one cp.async.bulk (TMA
// unit, SASS UBLKCP; a row is 6 KB contiguous in fp64) a full step before it is needed, completion counted on one mbarrier
// per slot.  A step reads from shared memory: the site's own spinor (x hops by warp shuffle), the in-tile y and z
// neighbours, psi(x,t+1); the backward-t contribution w = U_t(x,t-1)^dagger P^+ psi(x,t-1) is carried in registers from the
// previous step, when both operands were at hand.  Only the y/z halo spinors and the links still come through L1/L2.
//
// MEASURED (profiles/r01d_ncu_direct_ring_eo.txt, 32^3x64 fp64): L2->SM traffic 4.07 -> 2.97 GB per launch and 45 % fewer
// LSU load sectors, as designed -- but 0.40 ms against 0.34 ms for the direct kernel: inside the marching loop the eight
// link-load wait points of a step are serialised and the kernel is bound by latency, not by L2->SM throughput.  It is
// therefore opt-in (dslash_set_kernel), kept because it is the correct pipeline skeleton for staging the LINKS the same way.
//
// Synchronisation per step: one __syncthreads() (all warps are done with the slot that is refilled next), lane 0 of every
// warp issues the bulk copy of its row for t+2 and arrives on that slot's mbarrier with the byte count, every thread waits
// on the mbarrier of a slot before its first read of that fill (parity = fill number & 1).
#include "dslash_async.cuh"
#include "dslash_kernels.cuh"

namespace dslash {

// spinor of lane `lane` in a shared-memory copy of one 32-site vector (global blocked-SoA format)
__device__ __forceinline__ void load_row_smem(cplx<double> (&psi)[12], const unsigned char* row, unsigned lane) {
    const double2* p = reinterpret_cast<const double2*>(row) + lane;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const double2 v = p[k * VL];
        psi[k] = {v.x, v.y};
    }
}
__device__ __forceinline__ void load_row_smem(cplx<float> (&psi)[12], const unsigned char* row, unsigned lane) {
    const float4* p = reinterpret_cast<const float4*>(row) + lane;
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        const float4 v = p[q * VL];
        psi[2 * q] = {v.x, v.y};
        psi[2 * q + 1] = {v.z, v.w};
    }
}

// one hop with the neighbour spinor already in registers
template <int MU, int SIGN, bool FIRST, typename Real, int RECON>
__device__ __forceinline__ void hop_psi(cplx<Real> (&acc)[12], const cplx<Real> (&psi)[12], const void* gauge, unsigned V, unsigned sl) {
    cplx<Real> h[6], hp[6], u[9];
    load_link<Real, LAYOUT_SOA, RECON>(u, gauge, V, sl, MU);
    project<MU, SIGN>(h, psi);
    su3_mul<(SIGN > 0)>(hp, u, h);
    reconstruct_accumulate<MU, SIGN, FIRST>(acc, hp);
}

// neighbour spinor: from the ring when the neighbouring row belongs to this block (warp-uniform), else from global memory
template <typename Real>
__device__ __forceinline__ void load_nbr(cplx<Real> (&psi)[12], bool in_tile, const unsigned char* row, unsigned lane, const void* in,
                                         unsigned V, unsigned sn) {
    if (in_tile)
        load_row_smem(psi, row, lane);
    else
        SpinorIO<Real, LAYOUT_SOA>::load(psi, in, V, sn);
}

template <typename Real, int RECON, int MAXTPB, int MINBLK, bool XSHFL>
__global__ void __launch_bounds__(MAXTPB, MINBLK)
    dslash_ring_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, Geom g, TileGeom tg,
                       int t_chunk) {
    constexpr unsigned ROW_BYTES = 24u * VL * sizeof(Real);  // one 32-site vector of spinors
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);  // three mbarriers, one per ring slot
    unsigned char* ring = smem + 128;                     // [3][nw][ROW_BYTES]
    const unsigned nw = blockDim.x >> 5, w = threadIdx.x >> 5, lane = threadIdx.x & 31u;

    // spatial tile and chunk of this block; warp w <-> row (ly, lz) of the tile
    unsigned b = blockIdx.x;
    const unsigned bx = b % (unsigned)tg.nt[0];
    b /= (unsigned)tg.nt[0];
    const unsigned by = b % (unsigned)tg.nt[1];
    b /= (unsigned)tg.nt[1];
    const unsigned bz = b % (unsigned)tg.nt[2];
    const unsigned bc = b / (unsigned)tg.nt[2];
    const unsigned ny = 1u << tg.lb[1], nz = 1u << tg.lb[2];
    const unsigned ly = w & (ny - 1u), lz = w >> tg.lb[1];
    const int x = (int)(bx * VL + lane), y = (int)((by << tg.lb[1]) + ly), z = (int)((bz << tg.lb[2]) + lz);
    const unsigned V = g.V;
    const unsigned sy = (unsigned)g.L[0], sz = sy * (unsigned)g.L[1], st = sz * (unsigned)g.L[2];
    const unsigned s3 = (unsigned)x + sy * (unsigned)y + sz * (unsigned)z;
    const unsigned dxf = (x + 1 == g.L[0]) ? 0u - (unsigned)(g.L[0] - 1) : 1u;
    const unsigned dxb = (x == 0) ? (unsigned)(g.L[0] - 1) : 0u - 1u;
    const unsigned dyf = (y + 1 == g.L[1]) ? 0u - (unsigned)(g.L[1] - 1) * sy : sy;
    const unsigned dyb = (y == 0) ? (unsigned)(g.L[1] - 1) * sy : 0u - sy;
    const unsigned dzf = (z + 1 == g.L[2]) ? 0u - (unsigned)(g.L[2] - 1) * sz : sz;
    const unsigned dzb = (z == 0) ? (unsigned)(g.L[2] - 1) * sz : 0u - sz;
    // in-tile neighbour rows (a tile spanning the whole extent takes the global path at the wrap: correct for any extent)
    const bool in_yf = ly + 1u < ny, in_yb = ly > 0u, in_zf = lz + 1u < nz, in_zb = lz > 0u;
    int lane_fwd = 0, lane_bwd = 0;
    if (XSHFL) x_shuffle_lanes(g.L[0], lane_fwd, lane_bwd);

    const int t0 = tg.t_begin + (int)bc * t_chunk;
    const int n = min(t_chunk, tg.t_end - t0);  // steps of this block

    if (threadIdx.x == 0) {
        mbar_init(&full[0], nw);
        mbar_init(&full[1], nw);
        mbar_init(&full[2], nw);
        mbar_fence_init();
    }
    __syncthreads();

    // lane 0 of each warp: bring this warp's row of time slice t0 + i (periodic) into ring slot `slot`
    const unsigned char* in_bytes = reinterpret_cast<const unsigned char*>(in);
    const unsigned row0 = s3 - lane;  // first site of the row: a multiple of 32 (L_X % 32 == 0)
    auto issue = [&](int i, unsigned slot) {
        if (lane == 0) {
            int t = t0 + i;
            if (t >= g.L[3]) t -= g.L[3];
            const unsigned vec = (row0 + st * (unsigned)t) >> VL_LOG2;
            fence_proxy_async();  // the slot was read through the generic proxy (before the block barrier): order those reads first
            mbar_arrive_expect_tx(&full[slot], ROW_BYTES);
            bulk_g2s(ring + (size_t)(slot * nw + w) * ROW_BYTES, in_bytes + (size_t)vec * ROW_BYTES, ROW_BYTES, &full[slot]);
        }
    };
    issue(0, 0);
    issue(1, 1);  // n >= 1: slice t0 + 1 is always needed (forward hop of the first step)

    // prologue: w = U_t(x, t0-1)^dagger P^+_t psi(x, t0-1) from global memory
    cplx<Real> wt[6];
    {
        const unsigned sb = s3 + st * (unsigned)((t0 == 0) ? g.L[3] - 1 : t0 - 1);
        cplx<Real> psi[12], u[9], h[6];
        SpinorIO<Real, LAYOUT_SOA>::load(psi, in, V, sb);
        load_link<Real, LAYOUT_SOA, RECON>(u, gauge, V, sb, 3);
        project<3, +1>(h, psi);
        su3_mul<true>(wt, u, h);
    }

    unsigned slot = 0;        // ring slot of time slice t0 + i
    unsigned phase_bits = 0;  // bit j: parity of the fill of slot j that holds the slice being read
#pragma unroll 1
    for (int i = 0; i < n; ++i) {
        const unsigned slot1 = slot == 2u ? 0u : slot + 1u, slot2 = slot1 == 2u ? 0u : slot1 + 1u;
        if (i > 0) __syncthreads();           // every warp has finished step i-1: slot2 (slice i-1) may be overwritten
        if (i + 2 <= n) issue(i + 2, slot2);  // lands during this step, first read in step i+1
        const unsigned s = s3 + st * (unsigned)(t0 + i);
        const unsigned char* cur = ring + (size_t)(slot * nw) * ROW_BYTES;
        mbar_wait_spin(&full[slot], (phase_bits >> slot) & 1u);

        cplx<Real> own[12], acc[12];
        load_row_smem(own, cur + (size_t)w * ROW_BYTES, lane);
        if (XSHFL) {
            cplx<Real> u[9], hm[6], hq[6], wx[6], hp[6];
            load_link<Real, LAYOUT_SOA, RECON>(u, gauge, V, s, 0);
            project<0, -1>(hm, own);
            project<0, +1>(hq, own);
            su3_mul<true>(wx, u, hq);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                hm[k].re = shfl_(hm[k].re, lane_fwd);
                hm[k].im = shfl_(hm[k].im, lane_fwd);
                wx[k].re = shfl_(wx[k].re, lane_bwd);
                wx[k].im = shfl_(wx[k].im, lane_bwd);
            }
            su3_mul<false>(hp, u, hm);
            reconstruct_accumulate<0, -1, true>(acc, hp);
            reconstruct_accumulate<0, +1, false>(acc, wx);
        } else {
            hop<0, -1, true, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, s + dxf, s);
            hop<0, +1, false, Real, LAYOUT_SOA, RECON>(acc, in, gauge, V, s + dxb, s + dxb);
        }
        {
            cplx<Real> psi[12];
            load_nbr<Real>(psi, in_yf, cur + (size_t)(w + 1u) * ROW_BYTES, lane, in, V, s + dyf);
            hop_psi<1, -1, false, Real, RECON>(acc, psi, gauge, V, s);
            load_nbr<Real>(psi, in_yb, cur + (size_t)(w - 1u) * ROW_BYTES, lane, in, V, s + dyb);
            hop_psi<1, +1, false, Real, RECON>(acc, psi, gauge, V, s + dyb);
            load_nbr<Real>(psi, in_zf, cur + (size_t)(w + ny) * ROW_BYTES, lane, in, V, s + dzf);
            hop_psi<2, -1, false, Real, RECON>(acc, psi, gauge, V, s);
            load_nbr<Real>(psi, in_zb, cur + (size_t)(w - ny) * ROW_BYTES, lane, in, V, s + dzb);
            hop_psi<2, +1, false, Real, RECON>(acc, psi, gauge, V, s + dzb);
        }
        {
            // forward t hop from the next slot; its link and the own spinor make the next step's backward contribution
            mbar_wait_spin(&full[slot1], (phase_bits >> slot1) & 1u);
            cplx<Real> nxt[12], u[9], h[6], hp[6];
            load_row_smem(nxt, ring + (size_t)(slot1 * nw + w) * ROW_BYTES, lane);
            load_link<Real, LAYOUT_SOA, RECON>(u, gauge, V, s, 3);
            project<3, -1>(h, nxt);
            su3_mul<false>(hp, u, h);
            reconstruct_accumulate<3, -1, false>(acc, hp);
            reconstruct_accumulate<3, +1, false>(acc, wt);
            project<3, +1>(h, own);
            su3_mul<true>(wt, u, h);
        }
        SpinorIO<Real, LAYOUT_SOA>::store(out, V, s, acc);
        phase_bits ^= 1u << slot;  // the next fill of this slot (slice i+3) has the other parity
        slot = slot1;
    }
}

// blocked SoA only; the tile is 32 x 2^lb[1] x 2^lb[2] x 1 and tiles the lattice exactly (rows = whole 32-site vectors)
bool ring_eligible(int layout_base, const Geom& g, const TileGeom& tg) {
    const int nw = 1 << (tg.lb[1] + tg.lb[2]);
    return layout_base == LAYOUT_SOA && tg.lb[0] == (int)VL_LOG2 && tg.lb[3] == 0 && g.L[0] % (int)VL == 0 &&
           g.L[1] % (1 << tg.lb[1]) == 0 && g.L[2] % (1 << tg.lb[2]) == 0 && nw >= 1 && nw <= 8;
}

template <typename Real, int RECON, int MAXTPB, int MINBLK, bool XSHFL>
static cudaError_t launch_ring_k(const LaunchArgs& a, const TileGeom& tg, int t_chunk) {
    const int nw = 1 << (tg.lb[1] + tg.lb[2]);
    const int nchunk = (tg.t_end - tg.t_begin + t_chunk - 1) / t_chunk;
    const unsigned grid = (unsigned)tg.nt[0] * (unsigned)tg.nt[1] * (unsigned)tg.nt[2] * (unsigned)nchunk;
    const size_t smem = 128u + 3u * (size_t)nw * (24u * VL * sizeof(Real));
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(dslash_ring_kernel<Real, RECON, MAXTPB, MINBLK, XSHFL>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, 128 + 3 * 8 * (int)(24u * VL * sizeof(Real)));
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    dslash_ring_kernel<Real, RECON, MAXTPB, MINBLK, XSHFL><<<grid, nw * 32, smem, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg, t_chunk);
    return cudaGetLastError();
}

template <typename Real, int RECON, bool XSHFL>
static cudaError_t launch_ring_s(const LaunchArgs& a, const TileGeom& tg, int t_chunk) {
    const int nw = 1 << (tg.lb[1] + tg.lb[2]);
    constexpr int MINBLK = sizeof(Real) == 8 ? 2 : 4;
    if (nw <= 4) return launch_ring_k<Real, RECON, 128, MINBLK, XSHFL>(a, tg, t_chunk);
    return launch_ring_k<Real, RECON, 256, MINBLK / 2, XSHFL>(a, tg, t_chunk);
}

cudaError_t launch_ring(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg, const TunedConfig& cfg) {
    if (!ring_eligible(layout_base, a.geom, tg)) return cudaErrorInvalidConfiguration;
    const int t_chunk = cfg.t_chunk > 0 ? cfg.t_chunk : 8;
    const bool xs = a.geom.L[0] == (int)VL;  // a whole x row in one warp: x hops by shuffle
#define DSLASH_RING(REAL, REC) (xs ? launch_ring_s<REAL, REC, true>(a, tg, t_chunk) : launch_ring_s<REAL, REC, false>(a, tg, t_chunk))
    if (precision == 0) return recon == 12 ? DSLASH_RING(double, 12) : DSLASH_RING(double, 18);
    return recon == 12 ? DSLASH_RING(float, 12) : DSLASH_RING(float, 18);
#undef DSLASH_RING
}

}  // namespace dslash

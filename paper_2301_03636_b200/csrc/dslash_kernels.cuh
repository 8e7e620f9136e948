// dslash_kernels.cuh -- kernel declarations shared by the translation units of libdslash_b200.so.
#pragma once
#include <cuda_runtime.h>

#include "dslash_site.cuh"

namespace dslash {

// Tile decomposition of the tuned kernel: a thread block covers 2^lb[0] x 2^lb[1] x 2^lb[2] x 2^lb[3]
// sites; nt[d] = ceil(L[d] / 2^lb[d]) tiles along d; tiles are numbered x fastest.
struct TileGeom {
    int lb[4];
    int nt[4];
    int t_begin, t_end;  // time slices [t_begin, t_end) are computed (dslash_set_time_range); nt[3] tiles cover that range
    int zb;              // tiles per z block of the block order (a divisor of nt[2]; nt[2] = plain x, y, z, t order)
};

// Block number -> tile coordinates.  Blocks run roughly in the order of their numbers, and what one block fetches the next
// ones find in L2, so the ORDER decides how far apart in time the two uses of a spinor by t-neighbours are.  Plain order
// (x, y, z, t) puts a whole time slice between them: 31 MB at 32^3 fp64, which L2 holds (HBM traffic 1.01 x compulsory), but
// 53 MB at 48^3 fp32, which it does not (ncu: 1.26 x).  So the z extent is cut into blocks of zb tiles and the order is
// x, y, z inside the z block, t, z block: the reuse distance shrinks to one slice of the z block, at the price of re-reading
// the z halo planes at the block boundaries (2 of 2 * zb * tile_z planes).
__device__ __forceinline__ void decode_tile(unsigned b, const TileGeom& tg, unsigned& bx, unsigned& by, unsigned& bz, unsigned& bt) {
    bx = b % (unsigned)tg.nt[0];
    b /= (unsigned)tg.nt[0];
    by = b % (unsigned)tg.nt[1];
    b /= (unsigned)tg.nt[1];
    const unsigned bzi = b % (unsigned)tg.zb;
    b /= (unsigned)tg.zb;
    bt = b % (unsigned)tg.nt[3];
    bz = (b / (unsigned)tg.nt[3]) * (unsigned)tg.zb + bzi;
}

struct LaunchArgs {
    void* out;
    const void* in;
    const void* gauge;
    Geom geom;
    cudaStream_t stream;
};

// Advisor-style variant (SURVEY.md section 8(d) "Sweep variant semantics"): collapse the first `depth`
// loops of (t,z,y,x); every parallel iteration runs the remaining loops serially.
cudaError_t launch_variant(int precision, int layout_base, int recon, const LaunchArgs& a, int depth, int tpb, int spt);

// The paper's exact variant space: distribute collapse da (0 if x == 0), parallel-for position x,
// parallel-for collapse b, schedule 0/1/2 = static/dynamic/guided, league and team size.
cudaError_t launch_omp_variant(int precision, int layout_base, int recon, const LaunchArgs& a, int da, int x, int b, int sched,
                               int teams, int team_size);

// Options of the tuned kernels (dslash_set_option).
struct TunedConfig {
    int occupancy;         // 0: default register budget, 1: 128-register variant
    int l2_policy;         // DSLASH_OPT_L2_POLICY bits (0: no cache hints); direct kernel only
    int march_policy;      // DSLASH_OPT_MARCH_POLICY bits (-1: the marching kernels' default 4|8|16)
    int l1_carveout;       // preferred shared-memory carve-out of the direct kernel in percent (-1: driver default)
    int pipe_slots;        // warp-pipelined kernel: stages in flight per warp (2..4; 0: default 2)
    int pipe_warps;        // warp-pipelined kernel: warps per block (1, 2 or 4; 0: default 4)
    unsigned* pipe_counters;  // warp-pipelined kernel: {next row, finished warps} of this launch (device memory, zero between launches)
    int pipe_zblock;       // warp-pipelined kernel: z planes per block of the row order (0: L_Z, i.e. plain lexicographic)
    int march_lead;        // marching kernel: steps a block may run ahead of the slowest block of its chunk (0: unbounded)
    int x_shuffle;         // 1: exchange the x hops inside the warp when the tile allows it (fp64 default), 0: always load them
};
bool x_shuffle_eligible(const Geom& g, const TileGeom& tg);

// Tuned kernel (direct, register-staged).
cudaError_t launch_tuned(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg,
                         const TunedConfig& cfg);

// warp-pipelined kernel: every hop stage of a 32-site row by two flat bulk async copies (cp.async.bulk, SASS UBLKCP) into
// per-warp shared-memory slots (dslash_wpipe.cu).
bool wpipe_eligible(int layout_base, const Geom& g);
cudaError_t launch_wpipe(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg, const TunedConfig& cfg);

// block-cooperative t-marching kernel (dslash_march.cu): a block owns up to MARCH_NW x rows that are neighbours in the (y,z)
// plane and marches through a chunk of time slices.  The decomposition is a host-built plan in device memory.
constexpr int MARCH_NW = 7;    // compute warps (= rows) per block: what 227 KB of shared memory hold in fp64; four more warps feed them
constexpr int MARCH_NWS = 9;   // exchange buffers per block (>= the 8 neighbour pairs 7 cells of a grid can form)
struct MarchWarpPlan {
    int row;     // the warp's row = vector index inside a time slice, y + L_Y * z (L_X == 32); -1: idle warp
    int fwd[2];  // spinor source of the forward y (0) / z (1) hop: >= 0 warp of this block whose ring row it is; < 0: -(row' + 1),
                 // row' = the neighbour row, fetched from global memory (halo)
    int wr[2];   // exchange buffer this warp fills with U^dagger P+ psi for its y+ / z+ neighbour (-1: none)
    int rd[2];   // exchange buffer holding the backward contribution of the y- / z- neighbour (-1: halo hop from row bwd[])
    int bwd[2];  // row of the y- / z- neighbour
};
struct MarchBlockPlan {
    int t0, nt;  // first time slice and number of steps
    int nact;    // active warps
    int chunk;   // which chunk of the time range (blocks of one chunk march together)
    MarchWarpPlan w[MARCH_NW];
};
constexpr int MARCH_MAX_CHUNKS = 64;
bool march_eligible(int layout_base, const Geom& g);
cudaError_t march_plan_create(const Geom& g, int t_begin, int t_end, int device, void** d_plan, int* nblocks);
// once per (ctx, device) where the kernel is selected: shared-memory attribute of the instantiation, SM count
cudaError_t march_prepare(int precision, int recon, int device, int* sms);
// sms from march_prepare(); *epoch = throttled launches on this plan so far (the progress counters behind the plan accumulate
// across exactly those launches); no CUDA runtime query on this path
cudaError_t launch_march(int precision, int layout_base, int recon, const LaunchArgs& a, const void* d_plan, int nblocks,
                         const TunedConfig& cfg, int sms, unsigned* epoch);

// Multi-GPU T-slab form (dslash_slab.cu): half-spinor faces and the boundary slices that consume them.
cudaError_t launch_slab_pack_faces(int precision, int layout_base, int recon, void* face_down, void* face_up, const void* in,
                                   const void* gauge, const Geom& g, cudaStream_t st);
cudaError_t launch_slab_boundary(int precision, int layout_base, int recon, void* out, const void* in, const void* gauge,
                                 const void* face_from_below, const void* face_from_above, const Geom& g, cudaStream_t st);

// Operators around Dslash (dslash_ops.cu): op 0 D, 1 D^dagger, 2 M = (4+m) - D/2, 3 M^dagger; solver vector kernels.
cudaError_t launch_op(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg, int op, double mass);
cudaError_t launch_axpby(int precision, int layout_base, unsigned V, void* y, const void* x, double a, double b, cudaStream_t st);
cudaError_t launch_dot(int precision, int layout_base, unsigned V, double* result, double* scratch, const void* x, const void* y,
                       cudaStream_t st);
cudaError_t launch_cg_update(int precision, int layout_base, unsigned V, void* x, void* r, const void* p, const void* q, double alpha,
                             double* result, double* scratch, cudaStream_t st);
int reduction_scratch_doubles();

// Even-odd (checkerboarded) operator and its layout kernels (dslash_eo.cu).  gh = half geometry {L_X/2, L_Y, L_Z, L_T}, V/2.
cudaError_t launch_eo(int precision, int layout_base, int recon, void* out, const void* in, const void* gauge_eo,
                      size_t gauge_half_bytes, const Geom& gh, const TileGeom& tg, int parity, int dagger, int xpay, double a,
                      double b, const void* c, cudaStream_t st);
// the same Schur operator as two launch_eo calls with the intermediate in the library's static device array (no allocation)
size_t eo_static_scratch_bytes();
cudaError_t launch_eo_schur_static(int precision, int layout_base, int recon, void* out_even, const void* in_even, const void* gauge_eo,
                                   size_t gauge_half_bytes, size_t half_bytes, const Geom& gh, const TileGeom& tg, int dagger, double a,
                                   cudaStream_t st);
cudaError_t launch_eo_convert_spinor(int precision, int layout_base, void* dst, const void* src, const Geom& gh, int parity, int dir,
                                     cudaStream_t st);
cudaError_t launch_eo_pack_gauge(int precision, int layout_base, int recon, void* dst_eo, const void* src, size_t gauge_half_bytes,
                                 const Geom& gh, cudaStream_t st);

// Layout module.  dir 0: canonical -> native (pack), 1: native -> canonical (unpack).
cudaError_t launch_convert_spinor(int precision, int layout_base, void* dst, const void* src, unsigned V, int dir,
                                  cudaStream_t stream);
cudaError_t launch_pack_gauge(int precision, int layout_base, int recon, void* dst, const void* src, unsigned V,
                              cudaStream_t stream);

}  // namespace dslash

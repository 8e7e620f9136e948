// dslash_ops.cu -- the operators around Dslash that its callers use:
//   D^dagger, the Wilson matrix M = (4 + m) - D/2 and M^dagger, and a conjugate-gradient solve of M^dagger M x = b.
//
// PAPER.md:52 calls Eq. 1 the "unpreconditioned Dirac operator" and PAPER.md:54 notes that it "is called several times
// throughout the LQCD application": the caller is a Krylov solver for the Wilson matrix, which is what is provided
// here.  D^dagger follows from Eq. 1 by taking the adjoint: gamma_mu is hermitian, so
//   (D^dagger psi)(x) = sum_mu [ (1 + gamma_mu) U_mu(x) psi(x+mu^) + (1 - gamma_mu) U_mu(x-mu^)^dagger psi(x-mu^) ],
// i.e. Eq. 1 with gamma_mu -> -gamma_mu (also = gamma_5 D gamma_5, oracle pin P5).
//
// One kernel serves all four operators: the projector sign is a run-time +-1 that enters the projection and the
// reconstruction as the multiplier of an FMA (a + s*b costs the same as a + b and is bit-identical for s = +-1), and
// the epilogue out = a*in(x) + b*acc is a uniform branch.
#include "dslash_kernels.cuh"
#include "dslash_hop_rt.cuh"

namespace dslash {

struct OpParams {
    double sigma;  // +1: D (forward projector 1 - gamma), -1: D^dagger (forward projector 1 + gamma)
    double a, b;   // out = a * in(x) + b * (D or D^dagger in)(x)
    int xpay;      // 0: out = b * acc only when b != 1 is not needed either (plain D / D^dagger)
};

template <typename Real, int LAYOUT, int RECON, int MINBLK>
__global__ void __launch_bounds__(128, MINBLK)
    dslash_op_kernel(void* __restrict__ out, const void* __restrict__ in, const void* __restrict__ gauge, Geom g, TileGeom tg,
                     OpParams op) {
    unsigned bx, by, bz, bt;
    decode_tile(blockIdx.x, tg, bx, by, bz, bt);
    unsigned r = threadIdx.x;
    const int x = (int)((bx << tg.lb[0]) + (r & ((1u << tg.lb[0]) - 1u)));
    r >>= tg.lb[0];
    const int y = (int)((by << tg.lb[1]) + (r & ((1u << tg.lb[1]) - 1u)));
    r >>= tg.lb[1];
    const int z = (int)((bz << tg.lb[2]) + (r & ((1u << tg.lb[2]) - 1u)));
    r >>= tg.lb[2];
    const int t = tg.t_begin + (int)((bt << tg.lb[3]) + r);
    if (x >= g.L[0] || y >= g.L[1] || z >= g.L[2] || t >= tg.t_end) return;
    const unsigned V = g.V;
    const unsigned sy = (unsigned)g.L[0], sz = sy * (unsigned)g.L[1], st = sz * (unsigned)g.L[2];
    const unsigned s = (unsigned)x + sy * (unsigned)y + sz * (unsigned)z + st * (unsigned)t;
    const unsigned xf = (x + 1 == g.L[0]) ? s - (unsigned)(g.L[0] - 1) : s + 1u;
    const unsigned xb = (x == 0) ? s + (unsigned)(g.L[0] - 1) : s - 1u;
    const unsigned yf = (y + 1 == g.L[1]) ? s - (unsigned)(g.L[1] - 1) * sy : s + sy;
    const unsigned yb = (y == 0) ? s + (unsigned)(g.L[1] - 1) * sy : s - sy;
    const unsigned zf = (z + 1 == g.L[2]) ? s - (unsigned)(g.L[2] - 1) * sz : s + sz;
    const unsigned zb = (z == 0) ? s + (unsigned)(g.L[2] - 1) * sz : s - sz;
    const unsigned tf = (t + 1 == g.L[3]) ? s - (unsigned)(g.L[3] - 1) * st : s + st;
    const unsigned tb = (t == 0) ? s + (unsigned)(g.L[3] - 1) * st : s - st;

    const Real sf = (Real)(-op.sigma), sb = (Real)op.sigma;  // forward projector 1 - sigma*gamma, backward 1 + sigma*gamma
    cplx<Real> acc[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) acc[k] = {Real(0), Real(0)};
    hop_rt<0, false, Real, LAYOUT, RECON>(acc, in, gauge, V, xf, s, sf);
    hop_rt<0, true, Real, LAYOUT, RECON>(acc, in, gauge, V, xb, xb, sb);
    hop_rt<1, false, Real, LAYOUT, RECON>(acc, in, gauge, V, yf, s, sf);
    hop_rt<1, true, Real, LAYOUT, RECON>(acc, in, gauge, V, yb, yb, sb);
    hop_rt<2, false, Real, LAYOUT, RECON>(acc, in, gauge, V, zf, s, sf);
    hop_rt<2, true, Real, LAYOUT, RECON>(acc, in, gauge, V, zb, zb, sb);
    hop_rt<3, false, Real, LAYOUT, RECON>(acc, in, gauge, V, tf, s, sf);
    hop_rt<3, true, Real, LAYOUT, RECON>(acc, in, gauge, V, tb, tb, sb);
    if (op.xpay) {
        cplx<Real> c[12];
        SpinorIO<Real, LAYOUT>::load(c, in, V, s);
        const Real a = (Real)op.a, bb = (Real)op.b;
#pragma unroll
        for (int k = 0; k < 12; ++k) acc[k] = {fma_(bb, acc[k].re, a * c[k].re), fma_(bb, acc[k].im, a * c[k].im)};
    }
    SpinorIO<Real, LAYOUT>::store(out, V, s, acc);
}

template <typename Real, int LAYOUT, int RECON>
static cudaError_t launch_op_t(const LaunchArgs& a, const TileGeom& tg, const OpParams& op) {
    const int tpb = 1 << (tg.lb[0] + tg.lb[1] + tg.lb[2] + tg.lb[3]);
    if (tpb > 128) return cudaErrorInvalidConfiguration;
    const unsigned grid = (unsigned)tg.nt[0] * (unsigned)tg.nt[1] * (unsigned)tg.nt[2] * (unsigned)tg.nt[3];
    constexpr int MINBLK = sizeof(Real) == 8 ? 2 : 4;  // same register budgets as the tuned Dslash kernel
    dslash_op_kernel<Real, LAYOUT, RECON, MINBLK><<<grid, tpb, 0, a.stream>>>(a.out, a.in, a.gauge, a.geom, tg, op);
    return cudaGetLastError();
}

// op: 0 D, 1 D^dagger, 2 M = (4+m) - D/2, 3 M^dagger
cudaError_t launch_op(int precision, int layout_base, int recon, const LaunchArgs& a, const TileGeom& tg, int op, double mass) {
    OpParams p;
    p.sigma = (op == 1 || op == 3) ? -1.0 : 1.0;
    p.xpay = (op >= 2);
    p.a = 4.0 + mass;
    p.b = -0.5;
#define DSLASH_OP(REAL)                                                                                   \
    (layout_base == LAYOUT_AOS ? (recon == 12 ? launch_op_t<REAL, LAYOUT_AOS, 12>(a, tg, p)              \
                                              : launch_op_t<REAL, LAYOUT_AOS, 18>(a, tg, p))             \
                               : (recon == 12 ? launch_op_t<REAL, LAYOUT_SOA, 12>(a, tg, p)              \
                                              : launch_op_t<REAL, LAYOUT_SOA, 18>(a, tg, p)))
    return precision == 0 ? DSLASH_OP(double) : DSLASH_OP(float);
#undef DSLASH_OP
}

// ------------------------------------------------------------------ vector kernels for the solver
// Fields are treated as arrays of 16-byte units in the native layout (fp64: one complex number, fp32: two).  With the
// blocked SoA layout the last vector may contain padding sites; `valid(u)` masks them out of the reductions and the
// updates leave them untouched (they are zero in the solver's own work spinors).
struct FieldShape {
    size_t nunits;  // 16-byte units in the buffer (including padding)
    unsigned V;     // real sites
    int soa;        // blocked SoA?
    unsigned upv;   // units per vector: 12 * 32 (fp64) or 6 * 32 (fp32)
};
__device__ __forceinline__ bool valid(const FieldShape& f, size_t u) {
    if (!f.soa) return true;
    const unsigned v = (unsigned)(u / f.upv);
    return v * VL + (unsigned)(u & (VL - 1u)) < f.V;
}

template <typename Real>
struct U16;
template <>
struct U16<double> {
    using type = double2;
    static constexpr int N = 2;
};
template <>
struct U16<float> {
    using type = float4;
    static constexpr int N = 4;
};
template <typename Real>
__device__ __forceinline__ void unpack(const typename U16<Real>::type& v, double (&a)[4]);
template <>
__device__ __forceinline__ void unpack<double>(const double2& v, double (&a)[4]) {
    a[0] = v.x;
    a[1] = v.y;
}
template <>
__device__ __forceinline__ void unpack<float>(const float4& v, double (&a)[4]) {
    a[0] = v.x;
    a[1] = v.y;
    a[2] = v.z;
    a[3] = v.w;
}
__device__ __forceinline__ void pack(double2& v, const double (&a)[4]) { v = make_double2(a[0], a[1]); }
__device__ __forceinline__ void pack(float4& v, const double (&a)[4]) {
    v = make_float4((float)a[0], (float)a[1], (float)a[2], (float)a[3]);
}

// block-level fp64 sum -> partial[blockIdx.x]
__device__ __forceinline__ void block_sum_to(double* partial, double s) {
    __shared__ double sh[256];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// y = a*x + b*y   (a, b real)
template <typename Real>
__global__ void __launch_bounds__(256) axpby_kernel(void* __restrict__ y_, const void* __restrict__ x_, double a, double b,
                                                    FieldShape f) {
    using U = typename U16<Real>::type;
    U* y = static_cast<U*>(y_);
    const U* x = static_cast<const U*>(x_);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < f.nunits; i += (size_t)gridDim.x * blockDim.x) {
        if (!valid(f, i)) continue;
        double xv[4], yv[4];
        unpack<Real>(x[i], xv);
        unpack<Real>(y[i], yv);
#pragma unroll
        for (int k = 0; k < U16<Real>::N; ++k) yv[k] = a * xv[k] + b * yv[k];
        U o;
        pack(o, yv);
        y[i] = o;
    }
}

// the fused CG update: x += alpha*p;  r -= alpha*q;  partial[block] = sum |r|^2  (fp64 accumulation)
template <typename Real>
__global__ void __launch_bounds__(256) cg_update_kernel(void* __restrict__ x_, void* __restrict__ r_, const void* __restrict__ p_,
                                                        const void* __restrict__ q_, double alpha, double* __restrict__ partial,
                                                        FieldShape f) {
    using U = typename U16<Real>::type;
    U* x = static_cast<U*>(x_);
    U* r = static_cast<U*>(r_);
    const U* p = static_cast<const U*>(p_);
    const U* q = static_cast<const U*>(q_);
    double s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < f.nunits; i += (size_t)gridDim.x * blockDim.x) {
        if (!valid(f, i)) continue;
        double xv[4], rv[4], pv[4], qv[4];
        unpack<Real>(x[i], xv);
        unpack<Real>(r[i], rv);
        unpack<Real>(p[i], pv);
        unpack<Real>(q[i], qv);
        U xo, ro;
#pragma unroll
        for (int k = 0; k < U16<Real>::N; ++k) {
            xv[k] += alpha * pv[k];
            rv[k] -= alpha * qv[k];
        }
        pack(xo, xv);
        pack(ro, rv);
        unpack<Real>(ro, rv);  // the norm is taken of r as it is stored (fp32 contexts round here)
#pragma unroll
        for (int k = 0; k < U16<Real>::N; ++k) s += rv[k] * rv[k];
        x[i] = xo;
        r[i] = ro;
    }
    block_sum_to(partial, s);
}

// partial[block] = sum_i x[i]*y[i] over the block's grid-stride range, accumulated in fp64 (deterministic two-pass sum)
template <typename Real>
__global__ void __launch_bounds__(256) dot_partial_kernel(double* __restrict__ partial, const void* __restrict__ x_,
                                                          const void* __restrict__ y_, FieldShape f) {
    using U = typename U16<Real>::type;
    const U* x = static_cast<const U*>(x_);
    const U* y = static_cast<const U*>(y_);
    double s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < f.nunits; i += (size_t)gridDim.x * blockDim.x) {
        if (!valid(f, i)) continue;
        double xv[4], yv[4];
        unpack<Real>(x[i], xv);
        unpack<Real>(y[i], yv);
#pragma unroll
        for (int k = 0; k < U16<Real>::N; ++k) s += xv[k] * yv[k];
    }
    block_sum_to(partial, s);
}
__global__ void __launch_bounds__(256) dot_final_kernel(double* __restrict__ result, const double* __restrict__ partial, int n) {
    __shared__ double sh[256];
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += 256) s += partial[i];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) *result = sh[0];
}

static FieldShape shape_of(int precision, int layout_base, unsigned V) {
    FieldShape f;
    f.V = V;
    f.soa = layout_base == LAYOUT_SOA;
    const size_t sites = f.soa ? (size_t)((V + VL - 1u) / VL) * VL : (size_t)V;
    const unsigned ups = precision == 0 ? 12u : 6u;  // 16-byte units per site
    f.nunits = sites * ups;
    f.upv = ups * VL;
    return f;
}

static const int kRedBlocks = 1184;  // 8 blocks of 256 threads per SM

cudaError_t launch_axpby(int precision, int layout_base, unsigned V, void* y, const void* x, double a, double b, cudaStream_t st) {
    const FieldShape f = shape_of(precision, layout_base, V);
    if (precision == 0)
        axpby_kernel<double><<<kRedBlocks, 256, 0, st>>>(y, x, a, b, f);
    else
        axpby_kernel<float><<<kRedBlocks, 256, 0, st>>>(y, x, a, b, f);
    return cudaGetLastError();
}

// result (device double) = <x, y> real inner product; scratch holds kRedBlocks doubles
cudaError_t launch_dot(int precision, int layout_base, unsigned V, double* result, double* scratch, const void* x, const void* y,
                       cudaStream_t st) {
    const FieldShape f = shape_of(precision, layout_base, V);
    if (precision == 0)
        dot_partial_kernel<double><<<kRedBlocks, 256, 0, st>>>(scratch, x, y, f);
    else
        dot_partial_kernel<float><<<kRedBlocks, 256, 0, st>>>(scratch, x, y, f);
    dot_final_kernel<<<1, 256, 0, st>>>(result, scratch, kRedBlocks);
    return cudaGetLastError();
}

// x += alpha p, r -= alpha q, result = |r|^2
cudaError_t launch_cg_update(int precision, int layout_base, unsigned V, void* x, void* r, const void* p, const void* q, double alpha,
                             double* result, double* scratch, cudaStream_t st) {
    const FieldShape f = shape_of(precision, layout_base, V);
    if (precision == 0)
        cg_update_kernel<double><<<kRedBlocks, 256, 0, st>>>(x, r, p, q, alpha, scratch, f);
    else
        cg_update_kernel<float><<<kRedBlocks, 256, 0, st>>>(x, r, p, q, alpha, scratch, f);
    dot_final_kernel<<<1, 256, 0, st>>>(result, scratch, kRedBlocks);
    return cudaGetLastError();
}

int reduction_scratch_doubles() { return kRedBlocks; }

}  // namespace dslash

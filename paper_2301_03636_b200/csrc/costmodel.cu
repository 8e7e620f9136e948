// costmodel.cu -- the Advisor's cost model as sm_100a kernels; C ABI in include/advisor_costmodel.h.
//
// Training is a chain of a few thousand tiny dependent steps (22 111 parameters for F = 33, mini-batches of 16), so the design
// goal is latency, not bandwidth: the WHOLE protocol (150 epochs x ceil(n/16) RMSprop steps) is one kernel launch, one
// thread-block cluster per model.  Block c of a cluster of C owns the output neurons [w*c/C, w*(c+1)/C) of every layer: their
// weight rows, biases and RMSprop accumulators stay in its shared memory from the Glorot initialisation to the final store.
//   forward  layer l: every block computes its neurons for the mini-batch and stores the activations into the activation
//            buffer of EVERY block of the cluster (distributed shared memory), then one cluster barrier;
//   backward layer l: every block forms, from its own rows, a partial of delta_{l-1} = delta_l W_l; barrier.cluster.arrive;
//            while the barrier is in flight it computes its rows' gradients (delta_l^T a_l) and applies the RMSprop update in
//            place (no gradient is ever stored); barrier.cluster.wait; then it sums, in block order, the C partials of the
//            neurons it owns in layer l-1 (distributed shared memory reads) and applies the ReLU mask.
// Global memory is touched for the mini-batch rows (L2 hits) and once at the end for the parameters.  Summation order is
// fixed, so a run is reproducible bit for bit.  Independent models (seeds, folds) are independent clusters of the same launch.
//
// Shares no code with oracle/costmodel.py (the NumPy restatement the tests compare against).
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <atomic>

#include "../../include/advisor_costmodel.h"

namespace cg = cooperative_groups;

namespace {

constexpr int kLayers = 5;
constexpr int kMaxBatch = 64;
constexpr int kMaxLrSteps = 32;
constexpr int kThreads = 256;       // block size of the small kernels
constexpr int kTrainMaxThreads = 1024;
constexpr size_t kMaxSmem = 232448;  // 227 KB opt-in limit of sm_100
constexpr double kAlpha = 0.99;      // RMSprop smoothing constant (Reading R22)
constexpr double kEps = 1e-8;        // added to sqrt(v) (Reading R22)

std::atomic<long long> g_launches{0};
std::atomic<int> g_train_threads{0};  // COSTMODEL_OPT_THREADS (0: default)
thread_local int g_last_cuda = 0;

inline int cuda_fail(cudaError_t e) {
    g_last_cuda = (int)e;
    return DSLASH_ERR_CUDA;
}

struct Shape {
    int w[kLayers + 1];   // F, 2F, 4F, 2F, F, 1
    int woff[kLayers];    // offset of W_l among the weights alone (= into the uniforms)
    int poff[kLayers];    // offset of W_l in the packed parameter vector (b_l follows W_l)
    int nparam, nweight;
};

__host__ __device__ inline Shape make_shape(int f) {
    Shape s;
    s.w[0] = f; s.w[1] = 2 * f; s.w[2] = 4 * f; s.w[3] = 2 * f; s.w[4] = f; s.w[5] = 1;
    int wo = 0, po = 0;
    for (int l = 0; l < kLayers; ++l) {
        s.woff[l] = wo;
        s.poff[l] = po;
        wo += s.w[l] * s.w[l + 1];
        po += s.w[l] * s.w[l + 1] + s.w[l + 1];
    }
    s.nweight = wo;
    s.nparam = po;
    return s;
}

__host__ __device__ inline int odd(int v) { return v | 1; }  // row strides in doubles: odd => no shared-memory bank conflicts
__host__ __device__ inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

// Shared-memory plan of one block (offsets in doubles); identical on every block of the cluster so that
// map_shared_rank() of a local address is the same object in the peer.
struct Plan {
    int wrow[kLayers];    // offset of the block's rows of W_l (row stride odd(w[l]))
    int brow[kLayers];    // offset of the block's biases of layer l
    int vshift;           // RMSprop accumulator of a parameter = its offset + vshift
    int act[kLayers];     // activations a_l [batch][odd(w[l])], l = 0..4 (a_0 = the mini-batch rows)
    int delta[2];         // delta of the block's own neurons [batch][drow], ping-pong over l
    int drow;
    int part[2];          // partial of delta_{l-1} from the block's rows [batch][odd(w[l])], ping-pong over l
    int pred, yb;         // [batch] each
    int idx;              // [batch] ints (stored in the space of doubles)
    int total;            // doubles
};

__host__ __device__ inline Plan make_plan(const Shape& s, int batch, int C) {
    Plan p;
    int o = 0, maxrows = 1, maxin = 1;
    for (int l = 0; l < kLayers; ++l) {
        const int rows = ceil_div(s.w[l + 1], C);
        p.wrow[l] = o;
        o += rows * odd(s.w[l]);
        p.brow[l] = o;
        o += rows;
        if (rows > maxrows) maxrows = rows;
        if (l > 0 && s.w[l] > maxin) maxin = s.w[l];
    }
    p.vshift = o;
    o *= 2;
    for (int l = 0; l < kLayers; ++l) {
        p.act[l] = o;
        o += batch * odd(s.w[l]);
    }
    p.drow = maxrows;
    p.delta[0] = o; o += batch * maxrows;
    p.delta[1] = o; o += batch * maxrows;
    p.part[0] = o; o += batch * odd(maxin);
    p.part[1] = o; o += batch * odd(maxin);
    p.pred = o; o += batch;
    p.yb = o; o += batch;
    p.idx = o; o += (batch + 1) / 2;
    p.total = o;
    return p;
}

struct TrainArgs {
    int f, n, epochs, batch, lr_step, C;
    const double* x;
    const double* y;
    const double* uniforms;
    const int* perms;
    double* params_out;
    double* epoch_loss_out;
    double weight_decay;
    long long max_steps;
    double lr[kMaxLrSteps];  // lr0 * gamma^k
    Shape S;                 // in the kernel's constant bank: indexing it by layer costs no local memory (a cluster barrier
    Plan P;                  // invalidates L1, so a stack copy would be re-fetched from L2 after every barrier)
};

// z[b][r] = sum_i W[r][i] a[b][i] + bias[r] for the rows r < rows of a weight block and the nb samples of the batch; one
// work item = one row x four samples (the weight is loaded once for four FMAs), shared by KS = 2^k <= 32 adjacent lanes: lane
// kl sums the terms i = kl, kl + KS, ... and a butterfly of shuffles adds the KS partial sums (the same bits in every lane).
// emit(b, r, z) consumes the result.  All threads of the block must call it (full-warp shuffles).
template <class Emit>
__device__ __forceinline__ void dense_rows(const double* __restrict__ W, int sw, const double* __restrict__ bias, int rows, int n_in,
                                           const double* __restrict__ a, int sa, int nb, int ks, Emit emit) {
    const int nbq = (nb + 3) >> 2, nitems = rows * nbq;
    const int group = threadIdx.x / ks, kl = threadIdx.x - group * ks, ngroups = blockDim.x / ks;
    for (int base = 0; base < nitems; base += ngroups) {
        const bool valid = base + group < nitems;
        const int item = valid ? base + group : nitems - 1;
        const int r = item / nbq, b0 = (item - r * nbq) * 4;
        const double* wr = W + (size_t)r * sw;
        const double* a0 = a + (size_t)b0 * sa;
        const double* a1 = a + (size_t)min(b0 + 1, nb - 1) * sa;
        const double* a2 = a + (size_t)min(b0 + 2, nb - 1) * sa;
        const double* a3 = a + (size_t)min(b0 + 3, nb - 1) * sa;
        double z0 = 0.0, z1 = 0.0, z2 = 0.0, z3 = 0.0;
        for (int i = kl; i < n_in; i += ks) {
            const double wv = wr[i];
            z0 = fma(wv, a0[i], z0);
            z1 = fma(wv, a1[i], z1);
            z2 = fma(wv, a2[i], z2);
            z3 = fma(wv, a3[i], z3);
        }
        for (int m = 1; m < ks; m <<= 1) {
            z0 += __shfl_xor_sync(0xffffffffu, z0, m);
            z1 += __shfl_xor_sync(0xffffffffu, z1, m);
            z2 += __shfl_xor_sync(0xffffffffu, z2, m);
            z3 += __shfl_xor_sync(0xffffffffu, z3, m);
        }
        if (!valid) continue;
        const double bv = bias[r];
        const int km = ks - 1;  // the four results are emitted by (up to) four different lanes of the group
        if ((0 & km) == kl) emit(b0, r, z0 + bv);
        if ((1 & km) == kl && b0 + 1 < nb) emit(b0 + 1, r, z1 + bv);
        if ((2 & km) == kl && b0 + 2 < nb) emit(b0 + 2, r, z2 + bv);
        if ((3 & km) == kl && b0 + 3 < nb) emit(b0 + 3, r, z3 + bv);
    }
}

// Lanes per work item of dense_rows in the training kernel: as many as keep 512 threads busy, at least 4 terms per lane.  A
// function of the layer and batch alone, NOT of the launch's block size, so that results do not depend on the latter.
__device__ __forceinline__ int lanes_per_item(int rows, int nb, int n_in) {
    const int nitems = rows * ((nb + 3) >> 2);
    int ks = 1;
    while (ks < 32 && nitems * ks * 2 <= 512 && ks * 8 <= n_in) ks *= 2;
    return ks;
}

// One RMSprop update (Reading R22), in the oracle's order of operations: g += wd p; v = 0.99 v + (0.01 g) g;
// p -= lr g / (sqrt(v) + 1e-8).  Explicit roundings: no FMA contraction.
__device__ __forceinline__ void rmsprop(double& p, double& v, double g, double lr, double wd) {
    g = __dadd_rn(g, __dmul_rn(wd, p));
    v = __dadd_rn(__dmul_rn(v, kAlpha), __dmul_rn(__dmul_rn(1.0 - kAlpha, g), g));
    p = __dsub_rn(p, __ddiv_rn(__dmul_rn(lr, g), __dadd_rn(__dsqrt_rn(v), kEps)));
}

__global__ void __launch_bounds__(kTrainMaxThreads, 1) costmodel_train_kernel(const TrainArgs A) {
    extern __shared__ double sm[];
    cg::cluster_group cluster = cg::this_cluster();
    const int C = A.C;
    const int rank = (int)cluster.block_rank();
    const int model = blockIdx.x / C;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const Shape& S = A.S;
    const Plan& P = A.P;
    __shared__ int lo[kLayers], rows[kLayers];  // the block's neurons of layer l: [lo, lo + rows)
    if (tid < kLayers) {
        lo[tid] = (int)(((long long)S.w[tid + 1] * rank) / C);
        rows[tid] = (int)(((long long)S.w[tid + 1] * (rank + 1)) / C) - lo[tid];
    }
    __syncthreads();
    const double* uni = A.uniforms + (size_t)model * S.nweight;
    const int* perms = A.perms + (size_t)model * A.epochs * A.n;
    int* idx = reinterpret_cast<int*>(sm + P.idx);
    const bool owner = rows[kLayers - 1] == 1;  // the block that holds the single output neuron (the last one of the cluster)
    const bool solo = C == 1;                   // a cluster of one block: block barriers do

    // Glorot uniform initialisation (Reading R21), biases and RMSprop accumulators 0
    for (int l = 0; l < kLayers; ++l) {
        const int n_in = S.w[l], sw = odd(n_in);
        const double bound = sqrt(6.0 / (double)(S.w[l] + S.w[l + 1]));
        for (int k = tid; k < rows[l] * sw; k += nthr) {
            const int r = k / sw, i = k - r * sw;
            double wv = 0.0;
            if (i < n_in) wv = __dmul_rn(__dsub_rn(__dmul_rn(2.0, uni[S.woff[l] + (size_t)(lo[l] + r) * n_in + i]), 1.0), bound);
            sm[P.wrow[l] + k] = wv;
            sm[P.wrow[l] + k + P.vshift] = 0.0;
        }
        for (int r = tid; r < rows[l]; r += nthr) {
            sm[P.brow[l] + r] = 0.0;
            sm[P.brow[l] + r + P.vshift] = 0.0;
        }
    }
    cluster.sync();

    long long steps = 0;
    for (int e = 0; e < A.epochs; ++e) {
        const double lr = A.lr[A.lr_step > 0 ? e / A.lr_step : 0];
        double loss_sum = 0.0;  // meaningful in thread 0 of the output neuron's block
        int nloss = 0;
        for (int s0 = 0; s0 < A.n; s0 += A.batch) {
            if (A.max_steps >= 0 && steps >= A.max_steps) break;
            const int nb = min(A.batch, A.n - s0);
            // ---- the mini-batch rows (every block keeps its own copy of a_0)
            if (tid < nb) {
                int r = perms[(size_t)e * A.n + s0 + tid];
                r = min(max(r, 0), A.n - 1);
                idx[tid] = r;
                if (owner) sm[P.yb + tid] = A.y[r];
            }
            __syncthreads();
            {
                const int sa = odd(A.f);
                for (int k = tid; k < nb * A.f; k += nthr) {
                    const int b = k / A.f, i = k - b * A.f;
                    sm[P.act[0] + b * sa + i] = A.x[(size_t)idx[b] * A.f + i];
                }
            }
            __syncthreads();
            // ---- forward: hidden layers broadcast their activations to every block of the cluster
            for (int l = 0; l < kLayers - 1; ++l) {
                const int sa_out = odd(S.w[l + 1]);
                double* out_local = sm + P.act[l + 1];
                const int lo_l = lo[l];
                dense_rows(sm + P.wrow[l], odd(S.w[l]), sm + P.brow[l], rows[l], S.w[l], sm + P.act[l], odd(S.w[l]), nb,
                           lanes_per_item(rows[l], nb, S.w[l]),
                           [&](int b, int r, double z) {
                               const double a = fmax(z, 0.0);  // ReLU (Reading R20)
                               double* dst = out_local + b * sa_out + lo_l + r;
                               for (int c = 0; c < C; ++c) *cluster.map_shared_rank(dst, c) = a;
                           });
                if (solo) __syncthreads(); else cluster.sync();
            }
            // ---- output layer (one neuron, owned by one block), loss (Eq. 2) and its derivative (Reading R23)
            dense_rows(sm + P.wrow[4], odd(S.w[4]), sm + P.brow[4], rows[4], S.w[4], sm + P.act[4], odd(S.w[4]), nb,
                       lanes_per_item(rows[4], nb, S.w[4]),
                       [&](int b, int, double z) { sm[P.pred + b] = z; });
            __syncthreads();
            if (owner && tid < 32) {
                double se = 0.0;
                for (int b = 0; b < nb; ++b) {
                    const double d = sm[P.pred + b] - sm[P.yb + b];
                    se = fma(d, d, se);
                }
                const double loss = sqrt(se / (double)nb);
                if (tid == 0) {
                    loss_sum += loss;
                    ++nloss;
                }
                for (int b = tid; b < nb; b += 32)
                    sm[P.delta[0] + b * P.drow] = (loss == 0.0) ? 0.0 : (sm[P.pred + b] - sm[P.yb + b]) / ((double)nb * loss);
            }
            __syncthreads();
            // ---- backward
            for (int l = kLayers - 1; l >= 0; --l) {
                const int n_in = S.w[l], sw = odd(n_in), sa = odd(n_in);
                const double* dl = sm + P.delta[l & 1];
                double* Wl = sm + P.wrow[l];
                const int nrow = rows[l];
                if (l > 0) {
                    // partial of delta_{l-1}: part[b][i] = sum_{own r} delta_l[b][r] W_l[r][i]; item = column i x four samples
                    double* part = sm + P.part[l & 1];
                    const int nbq = (nb + 3) >> 2;
                    for (int item = tid; item < n_in * nbq; item += nthr) {
                        const int q = item / n_in, i = item - q * n_in, b0 = q * 4;
                        const double* d0 = dl + b0 * P.drow;
                        const double* d1 = dl + min(b0 + 1, nb - 1) * P.drow;
                        const double* d2 = dl + min(b0 + 2, nb - 1) * P.drow;
                        const double* d3 = dl + min(b0 + 3, nb - 1) * P.drow;
                        double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
                        for (int r = 0; r < nrow; ++r) {
                            const double wv = Wl[r * sw + i];
                            p0 = fma(d0[r], wv, p0);
                            p1 = fma(d1[r], wv, p1);
                            p2 = fma(d2[r], wv, p2);
                            p3 = fma(d3[r], wv, p3);
                        }
                        part[b0 * sa + i] = p0;
                        if (b0 + 1 < nb) part[(b0 + 1) * sa + i] = p1;
                        if (b0 + 2 < nb) part[(b0 + 2) * sa + i] = p2;
                        if (b0 + 3 < nb) part[(b0 + 3) * sa + i] = p3;
                    }
                    __syncthreads();           // every thread has read the old W_l before anyone updates it
                    if (!solo) cluster.barrier_arrive();  // release: the partial is visible to the peers after their wait
                }
                // gradient of the own rows and RMSprop in place: g[r][i] = sum_b delta_l[b][r] a_l[b][i] (i == n_in: the bias)
                {
                    const double* al = sm + P.act[l];
                    double* bl = sm + P.brow[l];
                    for (int k = tid; k < nrow * (n_in + 1); k += nthr) {
                        const int r = k / (n_in + 1), i = k - r * (n_in + 1);
                        double g = 0.0;
                        if (i < n_in) {
                            for (int b = 0; b < nb; ++b) g = fma(dl[b * P.drow + r], al[b * sa + i], g);
                            double* p = Wl + r * sw + i;
                            rmsprop(p[0], p[P.vshift], g, lr, A.weight_decay);
                        } else {
                            for (int b = 0; b < nb; ++b) g += dl[b * P.drow + r];
                            double* p = bl + r;
                            rmsprop(p[0], p[P.vshift], g, lr, A.weight_decay);
                        }
                    }
                }
                if (l > 0) {
                    if (solo) __syncthreads(); else cluster.barrier_wait();  // acquire: all partials of this layer are complete
                    // delta of the own neurons of layer l-1: sum of the C partials in block order, times the ReLU mask
                    const double* part = sm + P.part[l & 1];
                    const double* al = sm + P.act[l];
                    double* dn = sm + P.delta[(l - 1) & 1];
                    const int lo_p = lo[l - 1], nrow_p = rows[l - 1];
                    for (int k = tid; k < nrow_p * nb; k += nthr) {
                        const int b = k / nrow_p, r = k - b * nrow_p;
                        const double* src = part + b * sa + lo_p + r;
                        double sum = 0.0;
                        for (int c = 0; c < C; ++c) sum += *cluster.map_shared_rank(src, c);
                        dn[b * P.drow + r] = (al[b * sa + lo_p + r] > 0.0) ? sum : 0.0;
                    }
                    __syncthreads();
                }
            }
            ++steps;
            if (solo) __syncthreads(); else cluster.sync();  // nobody overwrites activations / partials of this step while a peer still reads them
        }
        if (owner && tid == 0 && A.epoch_loss_out)
            A.epoch_loss_out[(size_t)model * A.epochs + e] = nloss ? loss_sum / (double)nloss : nan("");
    }

    // ---- final store in packing order
    double* out = A.params_out + (size_t)model * S.nparam;
    for (int l = 0; l < kLayers; ++l) {
        const int n_in = S.w[l], sw = odd(n_in);
        for (int k = tid; k < rows[l] * n_in; k += nthr) {
            const int r = k / n_in, i = k - r * n_in;
            out[S.poff[l] + (size_t)(lo[l] + r) * n_in + i] = sm[P.wrow[l] + r * sw + i];
        }
        for (int r = tid; r < rows[l]; r += nthr) out[S.poff[l] + (size_t)n_in * S.w[l + 1] + lo[l] + r] = sm[P.brow[l] + r];
    }
    cluster.sync();  // no block exits while a peer may still address its shared memory
}

// Inference: one block per group of up to 16 rows; weights straight from global memory (L2-resident, 177 KB for F = 33),
// activations ping-pong in shared memory.
constexpr int kPredRows = 16;

__global__ void __launch_bounds__(kThreads) costmodel_predict_kernel(int f, int n, const double* __restrict__ params, int n_models,
                                                                     const double* __restrict__ x, double* __restrict__ pred) {
    extern __shared__ double sm[];
    const Shape S = make_shape(f);
    const int sa = odd(4 * f);
    double* buf0 = sm;
    double* buf1 = sm + kPredRows * sa;
    const int groups = ceil_div(n, kPredRows);
    for (int work = blockIdx.x; work < groups * n_models; work += gridDim.x) {
        const int model = work / groups, r0 = (work - model * groups) * kPredRows;
        const int nb = min(kPredRows, n - r0);
        const double* P = params + (size_t)model * S.nparam;
        for (int k = threadIdx.x; k < nb * f; k += blockDim.x) {
            const int b = k / f, i = k - b * f;
            buf0[b * sa + i] = x[(size_t)(r0 + b) * f + i];
        }
        __syncthreads();
        double* in = buf0;
        double* out = buf1;
        for (int l = 0; l < kLayers; ++l) {
            const int n_in = S.w[l], n_out = S.w[l + 1];
            const double* W = P + S.poff[l];
            if (l < kLayers - 1) {
                dense_rows(W, n_in, W + (size_t)n_in * n_out, n_out, n_in, in, sa, nb, 1,
                           [&](int b, int r, double z) { out[b * sa + r] = fmax(z, 0.0); });
            } else {
                dense_rows(W, n_in, W + (size_t)n_in * n_out, n_out, n_in, in, sa, nb, 1,
                           [&](int b, int, double z) { pred[(size_t)model * n + r0 + b] = z; });
            }
            __syncthreads();
            double* t = in; in = out; out = t;
        }
    }
}

// Deterministic block reduction (fixed tree) of one value per thread; result valid in every thread.
template <class Op>
__device__ __forceinline__ double block_reduce(double v, double* scratch, Op op) {
    scratch[threadIdx.x] = v;
    __syncthreads();
    for (int s = blockDim.x >> 1; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) scratch[threadIdx.x] = op(scratch[threadIdx.x], scratch[threadIdx.x + s]);
        __syncthreads();
    }
    const double r = scratch[0];
    __syncthreads();
    return r;
}

// One block per column: mean, then the population deviation around it (two passes; Reading R25).
__global__ void __launch_bounds__(kThreads) costmodel_zscore_fit_kernel(int n, int cols, const double* __restrict__ a,
                                                                        double* __restrict__ mean, double* __restrict__ sd) {
    __shared__ double scratch[kThreads];
    const int c = blockIdx.x;
    auto add = [](double p, double q) { return p + q; };
    double s = 0.0;
    for (int r = threadIdx.x; r < n; r += blockDim.x) s += a[(size_t)r * cols + c];
    const double m = block_reduce(s, scratch, add) / (double)n;
    double q = 0.0;
    for (int r = threadIdx.x; r < n; r += blockDim.x) {
        const double d = a[(size_t)r * cols + c] - m;
        q = fma(d, d, q);
    }
    const double var = block_reduce(q, scratch, add) / (double)n;
    if (threadIdx.x == 0) {
        const double dev = sqrt(var);
        mean[c] = m;
        sd[c] = (dev == 0.0) ? 1.0 : dev;
    }
}

__global__ void __launch_bounds__(kThreads) costmodel_zscore_apply_kernel(long long total, int cols, const double* a,
                                                                          const double* __restrict__ mean,
                                                                          const double* __restrict__ sd, int inverse, double* out) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < total; k += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(k % cols);
        out[k] = inverse ? __dadd_rn(__dmul_rn(a[k], sd[c]), mean[c]) : __ddiv_rn(__dsub_rn(a[k], mean[c]), sd[c]);
    }
}

// One block: RMSE (Eq. 2) and NRMSE = RMSE / (y_max - y_min) (Eq. 3).
__global__ void __launch_bounds__(kThreads) costmodel_error_kernel(int n, const double* __restrict__ pred, const double* __restrict__ y,
                                                                   double* __restrict__ out) {
    __shared__ double scratch[kThreads];
    double se = 0.0, hi = -INFINITY, lo = INFINITY;
    for (int r = threadIdx.x; r < n; r += blockDim.x) {
        const double d = pred[r] - y[r];
        se = fma(d, d, se);
        hi = fmax(hi, y[r]);
        lo = fmin(lo, y[r]);
    }
    se = block_reduce(se, scratch, [](double p, double q) { return p + q; });
    hi = block_reduce(hi, scratch, [](double p, double q) { return fmax(p, q); });
    lo = block_reduce(lo, scratch, [](double p, double q) { return fmin(p, q); });
    if (threadIdx.x == 0) {
        const double rmse = sqrt(se / (double)n);
        out[0] = rmse;
        out[1] = rmse / (hi - lo);
    }
}

inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7u) != 0; }

}  // namespace

extern "C" {

size_t costmodel_param_count(int f) { return f < 1 ? 0 : (size_t)make_shape(f).nparam; }
size_t costmodel_weight_count(int f) { return f < 1 ? 0 : (size_t)make_shape(f).nweight; }

size_t costmodel_train_smem_bytes(int f, int batch, int cluster_size) {
    if (f < 1 || f > 4096 || batch < 1 || batch > kMaxBatch) return 0;
    if (cluster_size != 1 && cluster_size != 2 && cluster_size != 4 && cluster_size != 8) return 0;
    return (size_t)make_plan(make_shape(f), batch, cluster_size).total * sizeof(double);
}

int costmodel_set_option(int option, int value) {
    if (option != COSTMODEL_OPT_THREADS) return DSLASH_ERR_UNSUPPORTED;
    if (value != 0 && (value < 32 || value > kTrainMaxThreads || value % 32)) return DSLASH_ERR_UNSUPPORTED;
    g_train_threads.store(value);
    return DSLASH_OK;
}

int costmodel_last_cuda_error(void) { return g_last_cuda; }
long long costmodel_launch_count(void) { return g_launches.load(); }

int costmodel_train(int f, int n, const double* x, const double* y, const double* uniforms, const int* perms, int epochs, int batch,
                    double lr0, int lr_step, double lr_gamma, double weight_decay, long long max_steps, int n_models,
                    int cluster_size, double* params_out, double* epoch_loss_out, dslash_stream_t stream) {
    if (!x || !y || !uniforms || !params_out || (!perms && epochs > 0)) return DSLASH_ERR_NULL;
    if (f < 1 || f > 4096 || n < 1 || epochs < 0 || batch < 1 || batch > kMaxBatch || n_models < 1) return DSLASH_ERR_DIMS;
    if (misaligned(x) || misaligned(y) || misaligned(uniforms) || misaligned(params_out) || misaligned(epoch_loss_out) ||
        (reinterpret_cast<uintptr_t>(perms) & 3u))
        return DSLASH_ERR_ALIGN;
    if (cluster_size != 0 && cluster_size != 1 && cluster_size != 2 && cluster_size != 4 && cluster_size != 8)
        return DSLASH_ERR_UNSUPPORTED;
    const int nlr = (lr_step > 0 && epochs > 0) ? (epochs - 1) / lr_step + 1 : 1;
    if (nlr > kMaxLrSteps) return DSLASH_ERR_UNSUPPORTED;
    // Defaults by measurement (profiles/r02b_costmodel.md, one model, batch 16, us per update):
    //   F = 33: cluster 4 / 8 at 256 threads 44.8 / 34.6, at 512 threads 36.3 / 29.3, at 1024 threads 43.3 / 35.5
    //   F = 12: cluster 1 / 2 / 4 / 8 at 256 threads 27.6 / 23.5 / 19.1 / 17.5, at 512 threads 23.9 / 22.1 / 19.9 / 19.4
    // The update is a chain of ~25 short dependent phases, so more blocks per model shorten every phase even when a single
    // block could hold the model: a cluster of 8 whenever the launch's models still fit the device side by side.
    int threads = g_train_threads.load() > 0 ? g_train_threads.load() : 512;
    int C = cluster_size;
    if (C == 0) {
        if (n_models <= 16 && costmodel_train_smem_bytes(f, batch, 8) <= kMaxSmem) {
            C = 8;  // latency: 16 clusters of 8 are resident together on 148 SMs
        } else {
            // throughput (many models per launch): one block while the widest layer gives every thread at most one work
            // item, more blocks as the layers grow
            C = 1;
            while (C < 8 && (costmodel_train_smem_bytes(f, batch, C) > kMaxSmem || 4 * f * ((batch + 3) / 4) > threads * C)) C *= 2;
        }
    }
    if (g_train_threads.load() <= 0 && C == 8 && f <= 16 && batch <= 256) threads = 256;  // small layers spread over 8 blocks
    if (threads < batch) return DSLASH_ERR_UNSUPPORTED;  // the training kernel loads one mini-batch index per thread
    const size_t smem = costmodel_train_smem_bytes(f, batch, C);
    if (smem == 0 || smem > kMaxSmem) return DSLASH_ERR_UNSUPPORTED;

    TrainArgs A;
    A.f = f; A.n = n; A.epochs = epochs; A.batch = batch; A.lr_step = lr_step; A.C = C;
    A.x = x; A.y = y; A.uniforms = uniforms; A.perms = perms;
    A.params_out = params_out; A.epoch_loss_out = epoch_loss_out;
    A.weight_decay = weight_decay; A.max_steps = max_steps;
    for (int k = 0; k < kMaxLrSteps; ++k) A.lr[k] = lr0 * pow(lr_gamma, (double)k);
    A.S = make_shape(f);
    A.P = make_plan(A.S, batch, C);

    cudaError_t e = cudaFuncSetAttribute(costmodel_train_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(n_models * C), 1, 1);
    cfg.blockDim = dim3((unsigned)threads, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = (cudaStream_t)stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, costmodel_train_kernel, A);
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches += 1;
    return DSLASH_OK;
}

int costmodel_predict(int f, int n, const double* params, int n_models, const double* x, double* pred, dslash_stream_t stream) {
    if (!params || !x || !pred) return DSLASH_ERR_NULL;
    if (f < 1 || f > 4096 || n < 1 || n_models < 1) return DSLASH_ERR_DIMS;
    if (misaligned(params) || misaligned(x) || misaligned(pred)) return DSLASH_ERR_ALIGN;
    const size_t smem = (size_t)2 * kPredRows * odd(4 * f) * sizeof(double);
    if (smem > kMaxSmem) return DSLASH_ERR_UNSUPPORTED;
    cudaError_t e = cudaFuncSetAttribute(costmodel_predict_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e);
    const long long work = (long long)ceil_div(n, kPredRows) * n_models;
    const unsigned grid = (unsigned)(work < 148 * 8 ? work : 148 * 8);
    costmodel_predict_kernel<<<grid, kThreads, smem, (cudaStream_t)stream>>>(f, n, params, n_models, x, pred);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches += 1;
    return DSLASH_OK;
}

int costmodel_zscore_fit(int n, int cols, const double* a, double* mean, double* sd, dslash_stream_t stream) {
    if (!a || !mean || !sd) return DSLASH_ERR_NULL;
    if (n < 1 || cols < 1) return DSLASH_ERR_DIMS;
    if (misaligned(a) || misaligned(mean) || misaligned(sd)) return DSLASH_ERR_ALIGN;
    costmodel_zscore_fit_kernel<<<(unsigned)cols, kThreads, 0, (cudaStream_t)stream>>>(n, cols, a, mean, sd);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches += 1;
    return DSLASH_OK;
}

int costmodel_zscore_apply(int n, int cols, const double* a, const double* mean, const double* sd, int inverse, double* out,
                           dslash_stream_t stream) {
    if (!a || !mean || !sd || !out) return DSLASH_ERR_NULL;
    if (n < 1 || cols < 1) return DSLASH_ERR_DIMS;
    if (misaligned(a) || misaligned(mean) || misaligned(sd) || misaligned(out)) return DSLASH_ERR_ALIGN;
    const long long total = (long long)n * cols;
    const long long blocks = (total + kThreads - 1) / kThreads;
    costmodel_zscore_apply_kernel<<<(unsigned)(blocks < 148 * 8 ? blocks : 148 * 8), kThreads, 0, (cudaStream_t)stream>>>(
        total, cols, a, mean, sd, inverse, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches += 1;
    return DSLASH_OK;
}

int costmodel_error(int n, const double* pred, const double* y, double* out, dslash_stream_t stream) {
    if (!pred || !y || !out) return DSLASH_ERR_NULL;
    if (n < 1) return DSLASH_ERR_DIMS;
    if (misaligned(pred) || misaligned(y) || misaligned(out)) return DSLASH_ERR_ALIGN;
    costmodel_error_kernel<<<1, kThreads, 0, (cudaStream_t)stream>>>(n, pred, y, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches += 1;
    return DSLASH_OK;
}

}  // extern "C"

/*
 * advisor_costmodel.h -- C ABI of the Advisor's cost model on the B200 (part of libdslash_b200.so, sm_100a).
 *
 * What the paper fixes (PAPER.md:177-181 section 4.2, :303-321 section 5.3): a multi-layer perceptron with "one input layer,
 * four hidden layers, and one output layer" whose hidden widths are 2F, 4F, 2F, F for F input features (66, 132, 66, 33 for
 * F = 33); Glorot initialisation, bias 0; mini-batches of 16; RMSprop with initial learning rate 0.01 "stepped
 * down by a factor of 0.1 every 30 epochs", weight decay 1e-4, 150 epochs; RMSE loss (Eq. 2);
 * Z-score standardisation of the data; NRMSE = RMSE / (y_max - y_min) (Eq. 3), < 0.1 counts as success.
 * What it leaves open and how it is read here: DESIGN.md Readings R20-R25 (ReLU after each hidden layer; Glorot uniform with
 * the uniforms passed in; RMSprop smoothing 0.99, epsilon 1e-8 outside the root, weight decay as an L2 term on weights and
 * biases; RMSE per mini-batch with gradient 0 at RMSE == 0; the visiting order of every epoch passed in; Z-score with the
 * population deviation of the training rows, zero deviation -> 1).
 *
 * Arithmetic: float64 throughout (the paper does not state a precision; DESIGN.md Reading R26).
 *
 * Conventions
 *   - Every function that can fail returns an int status: DSLASH_OK (0) or a negative DSLASH_ERR_* code of dslash_b200.h.
 *     Nothing throws, aborts or prints.  The size queries return 0 for invalid arguments.
 *   - Every pointer is a DEVICE pointer (CUDA global memory of the current device), caller-owned, 8-byte aligned; the
 *     library never allocates, frees or keeps them.  All work is enqueued on `stream` (a cudaStream_t passed as an opaque
 *     pointer, NULL = legacy default stream); no call synchronises.
 *   - There is no CPU fallback: without a CUDA device the compute calls return DSLASH_ERR_CUDA.
 *
 * Parameter packing (params, params_out): for layer l = 0..4 with n_in = w[l], n_out = w[l+1], w = {F, 2F, 4F, 2F, F, 1}:
 *     W_l[n_out][n_in] row-major (y = W x + b), then b_l[n_out]; layers in order.  costmodel_param_count(F) doubles.
 *   uniforms: one u in [0,1) per WEIGHT in the same order without the biases (costmodel_weight_count(F) doubles per model);
 *     W = (2u - 1) * sqrt(6 / (n_in + n_out)).
 */
#ifndef ADVISOR_COSTMODEL_H
#define ADVISOR_COSTMODEL_H

#include <stddef.h>

#include "dslash_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of doubles of a packed parameter vector / number of weights (= uniforms consumed) for F features; 0 if F < 1. */
DSLASH_API size_t costmodel_param_count(int f);
DSLASH_API size_t costmodel_weight_count(int f);

/* Dynamic shared memory per thread block that costmodel_train() needs for (F, batch, cluster_size), in bytes; 0 for invalid
 * arguments.  A configuration is supported when this is <= 232448 (227 KB). */
DSLASH_API size_t costmodel_train_smem_bytes(int f, int batch, int cluster_size);

/*
 * Train n_models independent networks on the same standardised data, the whole protocol of PAPER.md:305-307 in ONE kernel
 * launch: one thread-block cluster per model; weights, biases, RMSprop state, activations and deltas live in the (distributed)
 * shared memory of the cluster for all epochs; global memory is read for the mini-batch rows and written once at the end.
 *
 *   x [n][F], y [n]                  standardised training rows (row-major)
 *   uniforms [n_models][costmodel_weight_count(F)]
 *   perms    [n_models][epochs][n]   int32: visiting order of each epoch (a permutation of 0..n-1 each; values are checked
 *                                    only for range on the device: an out-of-range index is clamped into 0..n-1)
 *   epochs >= 0; 1 <= batch <= 64; mini-batch s of an epoch = rows perms[e][s*batch .. min((s+1)*batch, n)) (last one may be short)
 *   learning rate of epoch e = lr0 * lr_gamma^(e / lr_step) (integer division; lr_step <= 0: constant lr0; at most 32 steps)
 *   weight_decay                     L2 coefficient added to every gradient (weights and biases)
 *   max_steps                        < 0: no limit; otherwise stop after that many updates in total (step-by-step comparisons)
 *   cluster_size                     1, 2, 4 or 8 thread blocks per model; 0 = the library chooses (8 while n_models <= 16, for
 *                                    latency: every phase of an update gets shorter with more blocks; else the fewest blocks that
 *                                    hold the model, for throughput).  The partial sums are added in block order, so the low bits
 *                                    of the result depend on the cluster size
 *   params_out     [n_models][costmodel_param_count(F)]
 *   epoch_loss_out [n_models][epochs]   mean mini-batch RMSE of each epoch (NaN for an epoch without updates); may be NULL
 *
 * Errors: DSLASH_ERR_NULL (a required pointer is NULL), DSLASH_ERR_DIMS (F < 1, n < 1, epochs < 0, batch outside 1..64,
 * n_models < 1), DSLASH_ERR_ALIGN, DSLASH_ERR_UNSUPPORTED (cluster_size not in {0,1,2,4,8}, shared memory does not fit,
 * more than 32 learning-rate steps), DSLASH_ERR_CUDA (launch failure; costmodel_last_cuda_error()).
 */
DSLASH_API int costmodel_train(int f, int n, const double *x, const double *y, const double *uniforms, const int *perms,
                               int epochs, int batch, double lr0, int lr_step, double lr_gamma, double weight_decay,
                               long long max_steps, int n_models, int cluster_size, double *params_out,
                               double *epoch_loss_out, dslash_stream_t stream);

/* pred[m][r] = network m (params [n_models][param_count]) applied to row r of x [n][F]; pred [n_models][n]. */
DSLASH_API int costmodel_predict(int f, int n, const double *params, int n_models, const double *x, double *pred,
                                 dslash_stream_t stream);

/* Z-score statistics of the columns of a [n][cols]: mean[c], and std[c] = population standard deviation (divisor n), with
 * std[c] = 1 where the deviation is exactly 0 (Reading R25).  Deterministic (fixed summation tree). */
DSLASH_API int costmodel_zscore_fit(int n, int cols, const double *a, double *mean, double *std, dslash_stream_t stream);

/* out = (a - mean) / std per column (inverse == 0) or out = a * std + mean (inverse != 0); out may be a itself. */
DSLASH_API int costmodel_zscore_apply(int n, int cols, const double *a, const double *mean, const double *std, int inverse,
                                      double *out, dslash_stream_t stream);

/* out[0] = RMSE(pred, y) (Eq. 2), out[1] = NRMSE = RMSE / (max y - min y) (Eq. 3; +inf if all y are equal and RMSE > 0,
 * NaN if RMSE == 0 as well), over n >= 1 values.  Deterministic. */
DSLASH_API int costmodel_error(int n, const double *pred, const double *y, double *out, dslash_stream_t stream);

/* Tuning knobs of costmodel_train() (process-wide).  COSTMODEL_OPT_THREADS: threads per block, a multiple of 32 in 32..1024,
 * 0 = the library's default.  Results do not depend on it bit for bit.  Anything else: DSLASH_ERR_UNSUPPORTED.
 * costmodel_train() returns DSLASH_ERR_UNSUPPORTED when it is smaller than the mini-batch size. */
#define COSTMODEL_OPT_THREADS 1
DSLASH_API int costmodel_set_option(int option, int value);

/* The cudaError_t of the last failed CUDA call of a costmodel_* function on this host thread's library (0 if none). */
DSLASH_API int costmodel_last_cuda_error(void);

/* Number of kernels the costmodel_* calls have launched since the library was loaded (bench.py's gpu_launches). */
DSLASH_API long long costmodel_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* ADVISOR_COSTMODEL_H */

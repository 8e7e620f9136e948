/*
 * dslash_b200_diag.h -- measurement aids of libdslash_b200.so.  NOT part of the operator's boundary (include/dslash_b200.h):
 * nothing here is on the Dslash path, and a caller of the operator never needs this header.  bench.py --probe and the
 * marching kernel's load-balance study use it.  Same conventions as dslash_b200.h (C ABI, int status codes, no torch types).
 */
#ifndef DSLASH_B200_DIAG_H
#define DSLASH_B200_DIAG_H

#include "dslash_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Where and how fast the blocks of the LAST DSLASH_KERNEL_MARCH launch of this ctx ran (a measurement aid: the kernel's work is
 * split statically, one block per SM, so the slowest SM sets the time).  stats (host, may be NULL to query *nblocks)
 * receives per block {SM id, SM clock cycles from block start to the last store of its first compute warp, low word of
 * %globaltimer (ns) when that warp began the middle step of its march}; capacity = its size in unsigned (>= 3 * *nblocks).
 * SYNCHRONISES the device.  Errors: NULL, UNSUPPORTED (capacity), CUDA.
 */
DSLASH_API int dslash_march_stats(dslash_ctx *ctx, unsigned *stats, size_t capacity, int *nblocks);

/*
 * Ceilings of the board at hand, measured with trivial kernels of this library (not on the Dslash
 * path).  Enqueues ONE kernel of `blocks` blocks of 256 threads on `stream`; the caller times it (bench.py --probe).
 *   DSLASH_PROBE_READ          reads n 16-byte units of src (dst: >= 8 bytes, never written)
 *   DSLASH_PROBE_WRITE         writes n units of dst
 *   DSLASH_PROBE_COPY          dst[i] = src[i], n units
 *   DSLASH_PROBE_READ4_WRITE1  dst[i] = src[i] + src[n+i] + src[2n+i] + src[3n+i]: Dslash's 4 : 1 read : write mix (src: 4n units)
 *   DSLASH_PROBE_DFMA          n iterations of 8 independent FP64 FMAs per thread in registers (dst: >= 8 bytes, never written)
 * dst, src: device pointers, 16-byte aligned.  Errors: DSLASH_ERR_NULL, _DIMS (n or blocks < 1), _ALIGN, _UNSUPPORTED, _CUDA.
 */
#define DSLASH_PROBE_READ 0
#define DSLASH_PROBE_WRITE 1
#define DSLASH_PROBE_COPY 2
#define DSLASH_PROBE_READ4_WRITE1 3
#define DSLASH_PROBE_DFMA 4
DSLASH_API int dslash_probe_launch(int kind, void *dst, const void *src, size_t n, int blocks, dslash_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* DSLASH_B200_DIAG_H */

/*
 * chase_filter_bench.h -- test and benchmark hooks of libchase_filter.so.  NOT part of the product ABI
 * (that is chase_filter.h: the filter of SURVEY 8(b) plus the 8(f) entry points): the functions here let
 * tests/ and bench.py look inside the library -- how one launch of the FP64 tensor kernel is decomposed,
 * how many kernels were launched, what the FP64 units reach on register-only code (csrc/peak_probe.cu, the
 * roofline denominator).  They may change between versions without notice.
 */
#ifndef CHASE_FILTER_BENCH_H
#define CHASE_FILTER_BENCH_H

#include "chase_filter.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Work decomposition the FP64 tensor step kernel (kernel path 1) uses for one launch on `n_active`
 * columns of an N x N problem on a GPU with `sms` SMs (host only, no CUDA call; for tests and inspection).
 * out (HOST int32[9]) = {row tiles of 128, column tiles, column tile width, data-parallel tiles, stream-K
 * CTAs, k-slabs per tile, CTAs launched (`grid`), data-parallel rounds, first stream-K CTA}.  The column
 * tiles cover [0, n_active) exactly once.  CTA b owns the whole tiles r * grid + b < data-parallel tiles
 * (r < rounds) in grouped raster order: by default persistent CTAs (grid = sms, first stream-K CTA = 0,
 * the producers kept in lock-step by a soft barrier); with CHASE_DMMA_LOCKSTEP=0 one tile per CTA (rounds = 1,
 * the stream-K CTAs follow them: first stream-K CTA = data-parallel tiles).  The remaining tiles are shared
 * by the CTAs first .. first + stream-K CTAs - 1 in contiguous k-slab ranges: sk_begin (HOST
 * int32[stream-K CTAs + 1], at most CHASE_MAX_SK_CTAS + 1; may be NULL) receives the range boundaries, slab s
 * being k-slab (s % slabs per tile) of tile (data-parallel tiles + s / slabs per tile).
 * Returns 0, CHASE_ERR_ARG or CHASE_ERR_DTYPE (not c128 / f64). */
#define CHASE_MAX_SK_CTAS 160
int chase_filter_step_plan(int64_t N, int64_t n_active, chase_dtype_t dtype, int32_t sms, int32_t *out,
                           int32_t *sk_begin);

/* Number of kernels launched by this library since load (all streams); for bench.py. */
int64_t chase_filter_launch_count(void);

/* Register-only FP64 peak probes on the current device (synchronous; for the roofline
 * denominator in bench.py).  kind 0: dependent-free DFMA chains, kind 1: mma.sync m8n8k4
 * f64 (SASS DMMA.8x8x4) chains.  Writes achieved GFLOP/s over `iters` inner iterations on
 * all SMs.  Returns 0 or a cudaError_t. */
int chase_fp64_peak_probe(int kind, int iters, double *gflops);

#ifdef __cplusplus
}
#endif
#endif /* CHASE_FILTER_BENCH_H */

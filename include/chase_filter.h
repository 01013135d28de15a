/*
 * chase_filter.h -- C ABI of the B200-native Chebyshev polynomial filter of ChASE
 * (arXiv 1805.10121).  Plain pointers and sizes only; no torch / C++ types.
 *
 * Operation (Alg. 4 "Chebyshev filter for optimized even degrees";
 * PAPER.md:311-313 Eq. (7); Eq. (5)):
 *
 *     V[:, j]  <-  p_{m_j}(H) V[:, j],     m_j = degrees[j],   j = 0 .. ncols-1
 *     p_m(x) = C_m((x - c)/e) / C_m((lambda1 - c)/e),  c = (a+b)/2,  e = (b-a)/2
 *
 * evaluated by the scaled three-term recurrence
 *     V_1     = (sigma_1/e) (H - cI) V_0
 *     V_{k+1} = (2 sigma_{k+1}/e) (H - cI) V_k - sigma_k sigma_{k+1} V_{k-1}
 *     sigma_1 = e/(lambda1 - c),  sigma_{k+1} = 1/(2/sigma_1 - sigma_k)
 * with a = mu_{nev+nex}, b = b_sup, lambda1 = mu_1.  Columns are sorted by
 * ascending degree (Alg. 1 l.15) so that step k works on the contiguous
 * suffix of columns with m_j >= k: one kernel launch, one pass over H per
 * step; shift (-c V_k), scaling and the V_{k-1} term are fused into the kernel epilogue
 * (replaces the paper's Shift + HEMM, Listing 1/2).
 *
 * Layouts (Listing 2): all matrices COLUMN-MAJOR, leading dimension N;
 * complex = interleaved (re, im) like std::complex<T>.  H is N x N, FULL Hermitian storage
 * (both triangles), EXACTLY Hermitian (H[i,j] == conj(H[j,i]) bitwise, real diagonal): a kernel may
 * read an entry from either triangle (the tcgen05 and streaming kernels read row m as the conjugate
 * of the contiguous column m).  H is never written.  V is N x ncols.
 *
 * Degrees: any m_j >= 0, non-decreasing.  0 leaves the column untouched, odd values are
 * accepted (the paper emits even ones only so that the result lands in V without a copy,
 * PAPER.md:393; here an odd-degree column costs one device copy of that column).
 *
 * All calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = legacy
 * default stream) unless stated otherwise.  The library never frees or retains caller
 * memory; `degrees` (HOST) is consumed before the call returns; H, V, workspace must stay
 * alive until `stream` has drained.
 *
 * Return codes: 0 success; negative = rejected before any launch (CHASE_ERR_*);
 * positive = a cudaError_t from a failed allocation / launch / copy.
 * ncols == 0 or max(degrees) == 0 is a success that launches nothing.
 */
#ifndef CHASE_FILTER_H
#define CHASE_FILTER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHASE_MAX_RANKS 16   /* most GPUs one row-sharded filter spans (chase_filter_rows_*) */
#define CHASE_MAX_DEGREE 4096 /* largest accepted degrees[j]; the paper's degrees are <= 36 (Table 1) */

typedef enum {
    CHASE_F32 = 0,  /* float,                 tcgen05 split-precision tensor path when N % 4 == 0, else FP32 FMA */
    CHASE_F64 = 1,  /* double,                FP64 (DMMA tensor path when N is even) */
    CHASE_C64 = 2,  /* interleaved float2,    tcgen05 split-precision tensor path when N % 2 == 0, else FP32 FMA */
    CHASE_C128 = 3  /* interleaved double2,   FP64 (DMMA tensor path for every N >= 16) */
} chase_dtype_t;

enum {
    CHASE_OK = 0,
    CHASE_ERR_ARG = -1,       /* null pointer, N <= 0, ncols < 0, N or ncols too large */
    CHASE_ERR_BOUNDS = -2,    /* not (lambda1 < a < b), or a non-finite bound (reading G8) */
    CHASE_ERR_DEGREES = -3,   /* a negative degree, one above CHASE_MAX_DEGREE, or degrees not non-decreasing (G7) */
    CHASE_ERR_DTYPE = -4,     /* unknown chase_dtype_t */
    CHASE_ERR_WORKSPACE = -5, /* workspace null or smaller than chase_filter_workspace_bytes */
    CHASE_ERR_ALIGN = -6,     /* H, V or workspace not aligned to 16 bytes */
    CHASE_ERR_TIMEOUT = -7,   /* row-sharded path: a peer rank did not reach an inter-GPU barrier in time
                                 (chase_rows_status), or the caller's host barrier reported a failure */
    CHASE_ERR_STATIC_LIMIT = -8 /* chase_residuals_static: the problem needs more scratch than the library's
                                 built-in CHASE_STATIC_SCRATCH_BYTES */
};

/* Bytes of device scratch chase_filter_ws needs: one N x ncols buffer of `dtype` (the W of
 * Alg. 4), rounded up to 256 bytes, plus -- see chase_filter_kernel_path -- 256 bytes on the tcgen05
 * 3xTF32 path (the counter of a soft barrier between the persistent CTAs) or about 20 MB on the FP64
 * tensor path (flags and partial accumulator tiles of the stream-K CTAs, chase_filter_step_plan).
 * 0 if an argument is invalid. */
size_t chase_filter_workspace_bytes(int64_t N, int64_t ncols, chase_dtype_t dtype);

/* The filter with caller-provided scratch.
 *   H          DEVICE, N x N column-major, ld = N, 16-byte aligned, read-only
 *   V          DEVICE, N x ncols column-major, ld = N, 16-byte aligned; in: V_0, out: result
 *   degrees    HOST, int32[ncols], non-decreasing, each >= 0
 *   a, b, lambda1   real bounds, lambda1 < a < b, finite (also for complex dtypes)
 *   workspace  DEVICE, >= chase_filter_workspace_bytes(...) bytes, 16-byte aligned; contents
 *              undefined on entry and exit
 *   stream     cudaStream_t
 * Enqueues exactly max(degrees) step kernels (plus one device copy per run of odd-degree
 * columns; on the 3xTF32 path a 4-byte memset before each kernel, on the FP64 tensor path one 1 KB
 * memset per call) and returns without synchronising. */
int chase_filter_ws(const void *H, int64_t N, void *V, int64_t ncols, const int32_t *degrees,
                    double a, double b, double lambda1, chase_dtype_t dtype,
                    void *workspace, size_t workspace_bytes, void *stream);

/* Same, scratch taken with cudaMallocAsync / cudaFreeAsync on `stream`. */
int chase_filter(const void *H, int64_t N, void *V, int64_t ncols, const int32_t *degrees,
                 double a, double b, double lambda1, chase_dtype_t dtype, void *stream);

/* End-to-end convenience for callers whose data lives on the HOST: H and V are HOST
 * pointers (pinned or pageable).  Allocates device buffers, copies V and H to the device,
 * runs the filter, copies V back, frees, and SYNCHRONISES before returning.  On the FP64 tensor
 * path H is uploaded in 8 row panels on a second stream and the first degree step runs panel by
 * panel as the rows arrive, so the upload of H hides behind that step.  For vector blocks of
 * 64 MB and more the result comes back column class by column class: the columns of degree k are
 * final after step k and are copied to V_host on a third stream while the later steps run (V_host
 * must not be read or written by the caller during the call; columns of degree 0 are not touched).
 * On an error return the contents of V_host are unspecified.  `device` is the CUDA device ordinal. */
int chase_filter_host(const void *H_host, int64_t N, void *V_host, int64_t ncols,
                      const int32_t *degrees, double a, double b, double lambda1,
                      chase_dtype_t dtype, int device);

/* chase_filter_host for a SEQUENCE of calls on one matrix.  The filter "is called hundreds of times" in a solve
 * and ChASE works on sequences of problems; chase_filter_host allocates, uploads and frees H
 * (N^2 elements: 25.6 GB at N = 40 000 complex128) on every call.  With a handle H goes up once:
 *   chase_filter_host_open   cudaSetDevice(device), allocates H, an N x max_ncols vector block and the workspace
 *                            of the widest call, uploads H_host (HOST, pinned or pageable; may be released after
 *                            the call) and SYNCHRONISES.  *handle_out (HOST) receives the handle.
 *   chase_filter_host_run    V_host (HOST, N x ncols, ncols <= max_ncols; in: V_0, out: result) goes up, the
 *                            filter of chase_filter_ws runs on the resident H, the result comes back; SYNCHRONISES.
 *                            Columns of degree 0 are not transferred.  Same validation and return codes as
 *                            chase_filter_host.  Calls on one handle must not overlap (one stream, one buffer set).
 *   chase_filter_host_close  waits for the handle's stream and frees everything.
 * A handle may be used from any host thread, one at a time. */
int chase_filter_host_open(const void *H_host, int64_t N, int64_t max_ncols, chase_dtype_t dtype, int device,
                           void **handle_out);
int chase_filter_host_run(void *handle, void *V_host, int64_t ncols, const int32_t *degrees, double a, double b,
                          double lambda1);
int chase_filter_host_close(void *handle);

/* Host-side pieces of Alg. 4, exposed for tests and callers that want to inspect the plan.
 * chase_filter_scalars: alpha[k], beta[k] (k = 1..m_max; entry 0 unused; arrays of m_max+1
 *   doubles, HOST) such that V_k = alpha[k] (H - cI) V_{k-1} + beta[k] V_{k-2}; *c = center.
 *   (Alg. 4 l.2-5, 8, 11.)  Returns 0 or CHASE_ERR_BOUNDS / CHASE_ERR_ARG.
 * chase_filter_schedule: offset[k] (k = 1..m_max, entry 0 unused; HOST int32[m_max+1]) =
 *   first active column of step k = #{j : degrees[j] < k} (Alg. 4 l.12-14).  Returns m_max
 *   (>= 0) or CHASE_ERR_DEGREES / CHASE_ERR_ARG; pass offset = NULL to only get m_max. */
int chase_filter_scalars(double a, double b, double lambda1, int32_t m_max,
                         double *alpha, double *beta, double *c);
int chase_filter_schedule(const int32_t *degrees, int64_t ncols, int32_t *offset);

/* Degree optimisation, host only (Alg. 5 "Degree Optimization"; Eq. (8),
 * PAPER.md:358) followed by the sort of Alg. 1 l.15.  For every column j:
 *     t = (ritzv[j] - c)/e,  c = (a+b)/2, e = (b-a)/2               (Alg. 5 l.2)
 *     rho = max(|t - sqrt(t^2-1)|, |t + sqrt(t^2-1)|)               (l.3; rho = 1 if |t| <= 1)
 *     deg = ceil(| ln(resid[j]/tol) / ln(rho) |)                    (l.4)
 *     deg = min(deg + deg_extra, deg_max)                           (l.5)
 *     deg = deg + (deg mod 2)                                       (l.6: even)
 * rho == 1 (Ritz value inside [a,b]) or a non-finite quotient gives deg_max before l.6.
 * degrees_out[i] (HOST int32[ncols]) receives the degrees sorted ascending, perm_out[i] (HOST
 * int64[ncols], may be NULL) the original index of the column that must move to position i
 * (stable sort), i.e. the permutation the caller applies to V, ritzv and resid before
 * chase_filter.  Returns 0, CHASE_ERR_ARG (null pointer, ncols < 0, tol <= 0, deg_extra < 0,
 * deg_max < 1, a resid <= 0 or non-finite) or CHASE_ERR_BOUNDS (not a < b, non-finite). */
int chase_degrees(int64_t ncols, const double *resid, const double *ritzv, double tol,
                  double a, double b, int32_t deg_extra, int32_t deg_max,
                  int32_t *degrees_out, int64_t *perm_out);

/* The other two HEMM call sites of ChASE, on the same step kernels.
 *
 * chase_hemm:  Y <- alpha (H - shift I) X + beta Y            (Listing 1 HEMM, PAPER.md:511;
 *   Rayleigh-Ritz A Q^, Alg. 2 l.2).  H, X, Y DEVICE, column-major, ld = N, 16-byte
 *   aligned, X and Y distinct N x ncols buffers; beta == 0 means Y is write-only.  Asynchronous.
 *
 * chase_residuals:  resid[j] = || H V[:,j] - ritzv[j] V[:,j] ||_2     (Alg. 1 l.8, PAPER.md:160;
 *   Listing 1 Resd).  One step kernel with a per-column shift in the epilogue
 *   (R = H V - V diag(ritzv) into the workspace) plus one column-norm kernel.  V DEVICE (read
 *   only), ritzv HOST double[ncols] (consumed before return), resid DEVICE double[ncols],
 *   workspace DEVICE >= chase_residuals_workspace_bytes(...).  Asynchronous on `stream`: ritzv is copied
 *   with one cudaMemcpyAsync, i.e. a PAGEABLE ritzv is consumed before return, a PINNED one must stay
 *   unchanged until `stream` has drained. */
int chase_hemm(const void *H, int64_t N, const void *X, void *Y, int64_t ncols,
               double alpha, double beta, double shift, chase_dtype_t dtype, void *stream);
size_t chase_residuals_workspace_bytes(int64_t N, int64_t ncols, chase_dtype_t dtype);
/* chase_hemm, chase_hemm_rows and the chase_filter_rows_* calls bring no workspace, so on the FP64 tensor path
 * their stream-K scratch (about 20 MB per launch in flight) comes from a process-wide cache of cudaMalloc'ed
 * buffers that is kept for reuse.  chase_scratch_cache_release gives those buffers back: it waits for the launch
 * each one last served, frees them, and the next such launch allocates afresh.  Returns 0, a cudaError_t, or
 * cudaErrorNotReady (600) when another host thread is inside such a launch at this moment (nothing freed). */
int chase_scratch_cache_release(void);
int chase_residuals(const void *H, int64_t N, const void *V, int64_t ncols, const double *ritzv,
                    double *resid, chase_dtype_t dtype, void *workspace, size_t workspace_bytes,
                    void *stream);

/* chase_residuals for callers that may not allocate device memory.
 *
 * Some users of this library live inside a memory budget they do not control: a plug-in of an application
 * whose own pool has already reserved the whole GPU, a process whose HBM share was fixed when the job
 * started, a latency-critical loop that must stay out of the driver's allocator (cudaMalloc and cudaFree
 * stall the whole device while they run).  Such a caller can neither pass a workspace to chase_residuals
 * nor let the library fetch one.  For them the library carries CHASE_STATIC_SCRATCH_BYTES of device memory
 * of its own, a static array inside the library image, and this one entry point uses it as the workspace:
 * same arguments as chase_residuals minus the workspace, same kernels, same results.  It calls no
 * cudaMalloc / cudaMallocAsync / cudaFree and no library routine that allocates.
 *
 *   H, V       DEVICE, read-only, as in chase_residuals, on the CURRENT device
 *   ritzv      HOST double[ncols]; resid  DEVICE double[ncols] (the only output)
 *   Limit: chase_residuals_workspace_bytes(N, ncols, dtype) <= CHASE_STATIC_SCRATCH_BYTES (48 MiB), i.e. a vector
 *          block N * ncols * sizeof(element) of just under 28 MiB on the FP64 tensor path (whose stream-K scratch
 *          takes 20 MiB of the array) and just under 48 MiB on the other paths; N = 3893, ncols = 282 complex128
 *          (the paper's NaCl problem) needs 36.8 MiB and fits.  Anything larger returns
 *          CHASE_ERR_STATIC_LIMIT before any CUDA call.
 *   Cost: a GPU holds the 48 MiB from the moment the CUDA module with the array is loaded on it (at the latest
 *          the first call of this entry point there; with eager module loading, as soon as the process has a
 *          context on it) until the process exits, whether or not the entry point is ever used again.
 *   First call on a device: looks up the array's device address (cudaGetSymbolAddress, which also makes the
 *          runtime load the module there); make that first call during set-up, before any stream capture
 *          and before the phase in which nothing may allocate.  Later calls only enqueue work.
 *   Sharing: all calls on one GPU use the SAME array.  It keeps the previous call's contents; the part that
 *          must start at zero (kernel flags / counters) is cleared in stream order by every call.  Two calls
 *          whose work can overlap on the GPU (different streams, or different host threads) RACE on it --
 *          keep them on one stream or order them with events.  chase_residuals has no such restriction.
 * Asynchronous on `stream` like chase_residuals; same return codes plus CHASE_ERR_STATIC_LIMIT. */
#define CHASE_STATIC_SCRATCH_BYTES (48u << 20)
int chase_residuals_static(const void *H, int64_t N, const void *V, int64_t ncols, const double *ritzv,
                           double *resid, chase_dtype_t dtype, void *stream);

/* Spectral estimates (Alg. 6 "Lanczos procedure for parameters estimates",
 * PAPER.md:421-475; Eq. (9)-(10)).
 *
 * chase_lanczos: `nruns` independent Lanczos runs of k steps each, advanced together so that the
 *   matrix-vector products of one step are ONE HEMM on an N x nruns block.  Run r
 *   starts from column r of V0 (DEVICE, N x nruns column-major, read only; the method's random start
 *   vectors are the caller's, they need not be normalised).  Every new Lanczos vector is
 *   re-orthogonalised against all previous ones of its run (two classical Gram-Schmidt passes).
 *   Output (HOST): alpha[r * k + j], beta[r * k + j], j = 0..k-1, with
 *       A U = U T_k + f_k e_k^T,  T_k = tridiag(beta[0..k-2]; alpha[0..k-1]; beta[0..k-2]),  beta[k-1] = ||f_k||_2.
 *   k <= N.  workspace DEVICE >= chase_lanczos_workspace_bytes(...), 16-byte aligned.  Enqueues on
 *   `stream` and SYNCHRONISES it before returning (the outputs are host arrays).
 *
 * chase_spectral_estimates (host only): from the coefficients of nruns = 1 + n_vec runs,
 *       b_sup = ||f_k||_2 + max Ritz value of run 0                                   (Alg. 6 l.3)
 *       mu_1  = smallest Ritz value over runs 1..n_vec                                (l.12)
 *       mu_ne = t with  int_{-inf}^{t} phi~ = nev_nex / N,                            (l.10-11)
 *       phi~(t) = 1/n_vec sum_j sum_i (Z^[j]_{1,i})^2 g_sigma(t - lambda~^[j]_i)      (Eq. 10)
 *   with g_sigma the Gaussian density of standard deviation sigma (paper default 0.25).
 *   nruns == 1 is the `approx` branch (l.4-5): only *b_sup is written (mu_1, mu_ne may be NULL).
 *   nev_nex is a double so that callers can aim between two eigenvalues; 0 < nev_nex < N.
 *   Returns 0 or CHASE_ERR_ARG (null pointer, bad size, non-finite / negative coefficient, sigma <= 0).
 *
 * chase_lanczos_ritz_vectors (Alg. 6 l.13, explained at :471: "Since ZQ are the approximate
 *   eigenvectors of A, we use those vectors corresponding to the Ritz values smaller than mu_{nev+nex} and
 *   intersperse them with random i.i.d. vectors in V^"): for run `run` (the paper uses the first of the
 *   n_vec runs, i.e. run = 1 when run 0 is the b_sup run), with T_k = Z^H diag(lam~) Z, writes the Ritz
 *   vector  x_i = U^[run] z_i  of every Ritz value lam~_i < mu_ne, in ascending order of lam~_i and at
 *   most max_vecs of them, into column dst_cols[i] of Vhat (DEVICE, N x ncols_vhat column-major) -- the
 *   caller picks the columns, which is the interspersing; the max_vecs entries of dst_cols must be distinct
 *   (CHASE_ERR_ARG otherwise).  The sign of x_i is fixed by Z_{1,i} >= 0.
 *   `workspace` is the one a chase_lanczos call with the same (N, nruns, k, dtype) left behind (the
 *   Lanczos vectors are still in it), alpha / beta that call's outputs (HOST [nruns * k]).
 *   *count (HOST) receives the number of vectors written, ritz_values (HOST [max_vecs], may be NULL)
 *   their Ritz values.  One N x k by k x count product in a small kernel; SYNCHRONISES `stream` after that
 *   kernel: Vhat is complete when the call returns. */
size_t chase_lanczos_workspace_bytes(int64_t N, int64_t nruns, int32_t k, chase_dtype_t dtype);
int chase_lanczos_ritz_vectors(const void *workspace, size_t workspace_bytes, int64_t N, int64_t nruns, int32_t k,
                               chase_dtype_t dtype, int64_t run, const double *alpha, const double *beta,
                               double mu_ne, void *Vhat, int64_t ncols_vhat, const int64_t *dst_cols,
                               int64_t max_vecs, int64_t *count, double *ritz_values, void *stream);
int chase_lanczos(const void *H, int64_t N, const void *V0, int64_t nruns, int32_t k, chase_dtype_t dtype,
                  double *alpha, double *beta, void *workspace, size_t workspace_bytes, void *stream);
int chase_spectral_estimates(int32_t k, int64_t nruns, const double *alpha, const double *beta, int64_t N,
                             double nev_nex, double sigma, double *b_sup, double *mu_1, double *mu_ne);

/* Row-sharded path for matrices that exceed one GPU (SURVEY 8(e) option 2; the paper's block
 * distribution of A, Fig. 3): one process per GPU, rank r owns the row block
 * [row0, row0 + nrows) of H as an nrows x N column-major matrix (ld = nrows) and a FULL N x ncols copy
 * of the vectors.  A step computes the rank's rows of the new iterate and its epilogue stores them into
 * the local copy AND, over NVLink peer memory, into every other rank's copy -- the all-gather of the
 * paper's HEMM ("gather") is fused into the kernel, tile by tile.  Only the FP64 tensor
 * kernels take this path: CHASE_C128 with N % 8 == 0 and nrows % 8 == 0, CHASE_F64 with % 16
 * (CHASE_ERR_ALIGN otherwise).  nranks <= CHASE_MAX_RANKS.
 *
 * chase_hemm_rows:  Y[rows, :] <- alpha (H_loc X - shift X[rows, :]) + beta Y[rows, :]  on this rank's
 *   rows, X and Y full N x ncols DEVICE buffers (ld = N), X complete on entry.  peer_Y: HOST array of
 *   npeers pointers valid ON THIS DEVICE to the other ranks' Y buffers (peer-mapped, e.g. through
 *   chase_ipc_open); the rows are pushed to each.  npeers = 0 is a plain local row-block HEMM.
 *   Asynchronous; no inter-GPU synchronisation (see chase_rows_barrier).
 *
 * chase_rows_barrier: all ranks' work enqueued so far on their streams has completed, including its
 *   peer stores.  flags: this rank's DEVICE uint32[nranks + 1], zeroed once by the caller -- entries
 *   [0, nranks) are the arrival slots, entry [nranks] is a STICKY status word; peer_flags: HOST
 *   array [nranks] of pointers valid on this device to every rank's flags array (entry [rank] = flags);
 *   seq: value strictly larger than any used before on these flags (same on all ranks).
 *   = chase_rows_signal (a kernel that release-stores seq, system scope, into flags[rank] of every rank)
 *   followed by chase_rows_wait (a kernel that polls the local slots until all nranks reach seq).
 *   The wait is bounded (30 s; environment CHASE_ROWS_TIMEOUT_MS overrides, read per call).  On a timeout
 *   it stores the failing seq into the status word and returns, and every later wait returns at once:
 *   the stream drains, the data are WRONG, and chase_rows_status says so.
 *
 * chase_rows_status: SYNCHRONISES `stream` and returns CHASE_ERR_TIMEOUT if any barrier enqueued on these
 *   flags timed out since they were zeroed, else 0.  Call it before using the result of a row-sharded
 *   filter.
 *
 * chase_filter_rows_ws: the filter of chase_filter_ws on a row-sharded H: per degree step one
 *   chase_hemm_rows launch on the active suffix and one chase_rows_barrier.  V (in: V_0 complete on
 *   every rank; out: result complete on every rank) and workspace as in chase_filter_ws; peer_V /
 *   peer_W: HOST arrays [nranks] of peer-mapped pointers to every rank's V / workspace (entry [rank]
 *   ignored); *seq (HOST, in/out) carries the barrier sequence across calls (start at 0).
 *   flags == NULL skips the barriers (single rank, or a caller that serialises the ranks itself).
 *
 * chase_filter_rows_hostsync_ws: same, for ranks that TIME-SHARE one GPU (several processes per device:
 *   their kernels are not guaranteed to run concurrently, so a spinning wait kernel could keep the peer's
 *   kernels off the GPU).  Every barrier becomes: signal kernel, cudaStreamSynchronize, host_barrier(ctx)
 *   (the caller's inter-process barrier, e.g. over gloo / MPI; non-zero return = failure ->
 *   CHASE_ERR_TIMEOUT), then the wait kernel, which finds every flag already set.  host_barrier == NULL is
 *   chase_filter_rows_ws.  Synchronises; not capturable. */
int chase_hemm_rows(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, const void *X, void *Y,
                    int64_t ncols, double alpha, double beta, double shift, chase_dtype_t dtype,
                    int32_t npeers, void *const *peer_Y, void *stream);
int chase_rows_barrier(uint32_t *flags, uint32_t *const *peer_flags, int32_t nranks, int32_t rank,
                       uint32_t seq, void *stream);
int chase_rows_signal(uint32_t *flags, uint32_t *const *peer_flags, int32_t nranks, int32_t rank,
                      uint32_t seq, void *stream);
int chase_rows_wait(uint32_t *flags, int32_t nranks, uint32_t seq, void *stream);
int chase_rows_status(const uint32_t *flags, int32_t nranks, void *stream);
int chase_filter_rows_ws(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, void *V, int64_t ncols,
                         const int32_t *degrees, double a, double b, double lambda1, chase_dtype_t dtype,
                         void *workspace, size_t workspace_bytes, int32_t nranks, int32_t rank,
                         void *const *peer_V, void *const *peer_W, uint32_t *flags,
                         uint32_t *const *peer_flags, uint32_t *seq, void *stream);
int chase_filter_rows_hostsync_ws(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, void *V, int64_t ncols,
                                  const int32_t *degrees, double a, double b, double lambda1, chase_dtype_t dtype,
                                  void *workspace, size_t workspace_bytes, int32_t nranks, int32_t rank,
                                  void *const *peer_V, void *const *peer_W, uint32_t *flags,
                                  uint32_t *const *peer_flags, uint32_t *seq, void *stream,
                                  int (*host_barrier)(void *), void *host_ctx);

/* CUDA IPC plumbing for the peer pointers above (one process per GPU).  chase_ipc_export: handle
 * (HOST, 64 bytes) of the allocation containing dev_ptr and dev_ptr's byte offset inside it.
 * chase_ipc_open: maps a handle received from another process, enabling peer access; *base_out is
 * the mapped allocation base (pass it to chase_ipc_close), the usable pointer is base + offset. */
int chase_ipc_export(const void *dev_ptr, void *handle64, int64_t *offset);
int chase_ipc_open(const void *handle64, void **base_out);
int chase_ipc_close(void *base);

/* Which kernel family chase_filter_ws would use: 1 = TMA + FP64 DMMA tensor kernel (c128 with
 * any N >= 16, f64 with even N), 2 = tcgen05 split-precision kernel (c64 with N % 2 == 0, f32 with
 * N % 4 == 0; every FP32 operand x is split on chip as hi + lo, hi*hi is a TF32 MMA and the two
 * cross terms are ONE BF16 MMA, FP32 accumulation; error vs an FP64 evaluation ~2e-5 at degree 16),
 * 0 = generic FMA kernel.  Environment (both read on every call; tests and bench.py use them to reach the FMA
 * kernels at TMA-legal sizes and to compare the two split schemes): CHASE_FILTER_FORCE_GENERIC=1 forces 0,
 * CHASE_TF32_MIXED=0 evaluates the cross terms as two TF32 MMAs (classic 3xTF32).  Negative = invalid arguments. */
int chase_filter_kernel_path(int64_t N, int64_t ncols, chase_dtype_t dtype);

const char *chase_filter_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* CHASE_FILTER_H */

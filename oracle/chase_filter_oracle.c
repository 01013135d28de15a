/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * Plain, slow, FP64 CPU evaluation of the ChASE Chebyshev filter (arXiv 1805.10121),
 * written from the paper alone.  It shares no code, header, table or helper with the
 * CUDA library under paper_1805_10121_b200/csrc and must never be linked into it.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.
 *
 * What it computes (Eq. (7); Alg. 4):
 *     out[:,j] = p_{m_j}(H) V0[:,j]         for every column j, m_j = degrees[j] >= 0
 * by the scaled three-term recurrence, in the paper's order and notation:
 *     c = (b_sup + mu_ne)/2, e = (b_sup - mu_ne)/2, sigma_1 = e/(mu_1 - c)   (Alg.4 l.2-3)
 *     W  <- (sigma_1/e) (H - cI) V                                           (l.4)
 *     sigma <- sigma_1                                                       (l.5)
 *     for i = 2 .. m_max:                                                    (l.7)
 *         tau <- 1/(2/sigma_1 - sigma)                                       (l.8)
 *         V[:,active] <- 2 (tau/e) (H - cI) W[:,active] - tau sigma V[:,active]   (l.9)
 *         V <-> W                                                            (l.10)
 *         sigma <- tau             (l.11: lost in PAPER.md, forced by PAPER.md:313; G1)
 *         drop columns with m_s <= i                                         (l.12-14)
 * "active" in the oracle is simply "columns with degrees[j] >= i" (no sortedness
 * needed here; readings G4/G5/G6 of DESIGN.md: degree 0 leaves the column untouched,
 * degree 1 stops after line 4, odd degrees allowed).  The result of column j is the
 * iterate of degree m_j and is returned in V.
 *
 * (H - cI) X is evaluated as the plain product H X, by the definition
 *     (H X)[i,j] = sum_{k=0}^{N-1} H[i,k] X[k,j]   (k ascending, real and imaginary
 * parts written out, full Hermitian storage read as a general matrix, reading G9),
 * followed by "- c X[i,j]".  No BLAS, no blocking of the k sum, no fusion of steps.
 * The only structure beyond the definition is the decomposition of the OUTPUT into
 * (row chunk) x (column chunk) pieces so that OpenMP threads own disjoint outputs and
 * H is streamed once per column chunk; every output element still sees exactly the
 * k-ascending sum above.
 *
 * Precision: always FP64.  For the single-precision GPU variants the caller passes
 * the FP32-rounded H (h_is_f32 = 1: H holds float / interleaved float pairs and is
 * upcast element by element inside the loop) and the FP32-rounded V0 upcast to FP64.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): spectral closed form P1, sigma
 * closed form P2, degree-1 brute force P3, gain invariants P4, H = cI / diagonal
 * special cases P5, reflector closed form P6, column independence P7, linearity P8,
 * uniform-vs-mixed degrees P9.  Nothing here is "parity unpinned".
 *
 * Layout: column-major, ld = N (Listing 2); complex = interleaved
 * (re, im) doubles.  Build: gcc -O2 -fopenmp -shared -fPIC (see oracle/__init__.py).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ROW_CHUNK 256 /* rows of the output owned by one task            */
#define COL_CHUNK 16  /* columns whose partial sums live in one task     */

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Alg. 4 lines 2, 3, 5, 8, 11 and the coefficients of lines 4 and 9.
 * On return, for k = 1..m_max (arrays indexed by k, entry 0 unused):
 *   sigma[k] = sigma_k, alpha[k] = coefficient of (H - cI) V_{k-1},
 *   beta[k]  = coefficient of V_{k-2}  (beta[1] = 0).
 * center/halfwidth receive c and e. */
void oracle_chase_scalars(double a, double b, double lambda1, int m_max,
                          double *sigma, double *alpha, double *beta,
                          double *center, double *halfwidth) {
    double c = (b + a) / 2.0;                 /* l.2 */
    double e = (b - a) / 2.0;                 /* l.2 */
    double sigma1 = e / (lambda1 - c);        /* l.3 */
    double sg = sigma1;                       /* l.5 */
    *center = c;
    *halfwidth = e;
    if (m_max >= 1) {
        sigma[1] = sigma1;
        alpha[1] = sigma1 / e;                /* l.4 */
        beta[1] = 0.0;
    }
    for (int i = 2; i <= m_max; ++i) {        /* l.7 */
        double tau = 1.0 / (2.0 / sigma1 - sg);   /* l.8 */
        alpha[i] = 2.0 * tau / e;             /* l.9 */
        beta[i] = -tau * sg;                  /* l.9 */
        sg = tau;                             /* l.11 */
        sigma[i] = sg;
    }
}

/* ------------------------------------------------------------------------------------
 * One recurrence step on a set of columns (Alg. 4 line 4 or line 9):
 *     dst_j[i] <- alpha * ( sum_k H[i,k] src_j[k]  -  c * src_j[i] )  +  beta * dst_j[i]
 * for every listed column j.  beta == 0 means "dst is not read" (line 4: W is
 * uninitialised).  src_j and dst_j are distinct buffers (V and W of Alg. 4).
 * ---------------------------------------------------------------------------------- */

static void step_complex(const void *Hv, int h_is_f32, int64_t N,
                         int ncol, double *const *src, double *const *dst,
                         double alpha, double beta, double c) {
    const double *Hd = (const double *)Hv;
    const float *Hf = (const float *)Hv;
    int64_t nrow_chunks = (N + ROW_CHUNK - 1) / ROW_CHUNK;
    int64_t ncol_chunks = (ncol + COL_CHUNK - 1) / COL_CHUNK;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int64_t cc = 0; cc < ncol_chunks; ++cc) {
        for (int64_t rc = 0; rc < nrow_chunks; ++rc) {
            int64_t i0 = rc * ROW_CHUNK, i1 = i0 + ROW_CHUNK < N ? i0 + ROW_CHUNK : N;
            int j0 = (int)(cc * COL_CHUNK), j1 = j0 + COL_CHUNK < ncol ? j0 + COL_CHUNK : ncol;
            double accr[COL_CHUNK][ROW_CHUNK], acci[COL_CHUNK][ROW_CHUNK];
            for (int j = j0; j < j1; ++j)
                for (int64_t i = i0; i < i1; ++i) { accr[j - j0][i - i0] = 0.0; acci[j - j0][i - i0] = 0.0; }
            for (int64_t k = 0; k < N; ++k) {              /* k ascending */
                for (int j = j0; j < j1; ++j) {
                    double xr = src[j][2 * k], xi = src[j][2 * k + 1];
                    double *ar = accr[j - j0], *ai = acci[j - j0];
                    if (h_is_f32) {
                        const float *col = Hf + 2 * (k * N);
                        for (int64_t i = i0; i < i1; ++i) {
                            double hr = (double)col[2 * i], hi = (double)col[2 * i + 1];
                            ar[i - i0] += hr * xr - hi * xi;
                            ai[i - i0] += hr * xi + hi * xr;
                        }
                    } else {
                        const double *col = Hd + 2 * (k * N);
                        for (int64_t i = i0; i < i1; ++i) {
                            double hr = col[2 * i], hi = col[2 * i + 1];
                            ar[i - i0] += hr * xr - hi * xi;
                            ai[i - i0] += hr * xi + hi * xr;
                        }
                    }
                }
            }
            for (int j = j0; j < j1; ++j) {
                for (int64_t i = i0; i < i1; ++i) {
                    double yr = alpha * (accr[j - j0][i - i0] - c * src[j][2 * i]);
                    double yi = alpha * (acci[j - j0][i - i0] - c * src[j][2 * i + 1]);
                    if (beta != 0.0) {
                        yr += beta * dst[j][2 * i];
                        yi += beta * dst[j][2 * i + 1];
                    }
                    dst[j][2 * i] = yr;
                    dst[j][2 * i + 1] = yi;
                }
            }
        }
    }
}

static void step_real(const void *Hv, int h_is_f32, int64_t N,
                      int ncol, double *const *src, double *const *dst,
                      double alpha, double beta, double c) {
    const double *Hd = (const double *)Hv;
    const float *Hf = (const float *)Hv;
    int64_t nrow_chunks = (N + ROW_CHUNK - 1) / ROW_CHUNK;
    int64_t ncol_chunks = (ncol + COL_CHUNK - 1) / COL_CHUNK;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int64_t cc = 0; cc < ncol_chunks; ++cc) {
        for (int64_t rc = 0; rc < nrow_chunks; ++rc) {
            int64_t i0 = rc * ROW_CHUNK, i1 = i0 + ROW_CHUNK < N ? i0 + ROW_CHUNK : N;
            int j0 = (int)(cc * COL_CHUNK), j1 = j0 + COL_CHUNK < ncol ? j0 + COL_CHUNK : ncol;
            double acc[COL_CHUNK][ROW_CHUNK];
            for (int j = j0; j < j1; ++j)
                for (int64_t i = i0; i < i1; ++i) acc[j - j0][i - i0] = 0.0;
            for (int64_t k = 0; k < N; ++k) {              /* k ascending */
                for (int j = j0; j < j1; ++j) {
                    double x = src[j][k];
                    double *ac = acc[j - j0];
                    if (h_is_f32) {
                        const float *col = Hf + k * N;
                        for (int64_t i = i0; i < i1; ++i) ac[i - i0] += (double)col[i] * x;
                    } else {
                        const double *col = Hd + k * N;
                        for (int64_t i = i0; i < i1; ++i) ac[i - i0] += col[i] * x;
                    }
                }
            }
            for (int j = j0; j < j1; ++j) {
                for (int64_t i = i0; i < i1; ++i) {
                    double y = alpha * (acc[j - j0][i - i0] - c * src[j][i]);
                    if (beta != 0.0) y += beta * dst[j][i];
                    dst[j][i] = y;
                }
            }
        }
    }
}

/* ------------------------------------------------------------------------------------
 * The filter (Alg. 4).  V: N x ncols (in: V0, out: result), W: scratch of the same size.
 * is_complex selects interleaved complex arithmetic.  Returns 0, or -1 on bad input /
 * allocation failure.  Host pointers only.
 * ---------------------------------------------------------------------------------- */
int oracle_chase_filter(const void *H, int h_is_f32, int is_complex, int64_t N,
                        double *V, double *W, int64_t ncols, const int32_t *degrees,
                        double a, double b, double lambda1) {
    if (!H || !V || !W || !degrees || N <= 0 || ncols < 0) return -1;
    int64_t ld = (is_complex ? 2 : 1) * N;          /* doubles per column */
    int m_max = 0;
    for (int64_t j = 0; j < ncols; ++j) {
        if (degrees[j] < 0) return -1;
        if (degrees[j] > m_max) m_max = degrees[j];
    }
    if (m_max == 0) return 0;

    double c = (b + a) / 2.0;                       /* l.2 */
    double e = (b - a) / 2.0;                       /* l.2 */
    double sigma1 = e / (lambda1 - c);              /* l.3 */
    double sigma = sigma1;                          /* l.5 */

    /* per-column roles: cur_j holds the newest iterate, oth_j the one before it */
    double **cur = (double **)malloc(sizeof(double *) * (size_t)ncols);
    double **oth = (double **)malloc(sizeof(double *) * (size_t)ncols);
    double **src = (double **)malloc(sizeof(double *) * (size_t)ncols);
    double **dst = (double **)malloc(sizeof(double *) * (size_t)ncols);
    if (!cur || !oth || !src || !dst) { free(cur); free(oth); free(src); free(dst); return -1; }
    for (int64_t j = 0; j < ncols; ++j) { cur[j] = V + j * ld; oth[j] = W + j * ld; }

    for (int i = 1; i <= m_max; ++i) {              /* l.4 (i = 1) and l.7 (i >= 2) */
        double alpha, beta;
        if (i == 1) {
            alpha = sigma1 / e;                     /* l.4 */
            beta = 0.0;
        } else {
            double tau = 1.0 / (2.0 / sigma1 - sigma);   /* l.8 */
            alpha = 2.0 * tau / e;                  /* l.9 */
            beta = -tau * sigma;                    /* l.9 */
            sigma = tau;                            /* l.11 (G1) */
        }
        int nact = 0;
        for (int64_t j = 0; j < ncols; ++j)         /* l.12-14: columns with m_j >= i */
            if (degrees[j] >= i) { src[nact] = cur[j]; dst[nact] = oth[j]; ++nact; }
        if (is_complex) step_complex(H, h_is_f32, N, nact, src, dst, alpha, beta, c);
        else            step_real(H, h_is_f32, N, nact, src, dst, alpha, beta, c);
        for (int64_t j = 0; j < ncols; ++j)         /* l.10: V <-> W for the active columns */
            if (degrees[j] >= i) { double *t = cur[j]; cur[j] = oth[j]; oth[j] = t; }
    }
    /* result of column j = its newest iterate; deliver it in V (G3) */
    for (int64_t j = 0; j < ncols; ++j)
        if (cur[j] != V + j * ld) memcpy(V + j * ld, cur[j], sizeof(double) * (size_t)ld);
    free(cur); free(oth); free(src); free(dst);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * The HEMM of Listing 1 as a general product, with a per-column shift:
 *     Y[:,j] <- alpha * ( H X[:,j] - shift[j] X[:,j] ) + beta * Y[:,j]
 * Used for Rayleigh-Ritz's A Q^ (Alg. 2 l.2: alpha=1, beta=0, shift=0) and for
 * the residual block H V - V diag(ritzv) (Alg. 1 l.8).  Same k-ascending sums
 * as the filter steps.  X, Y: N x ncols FP64 (interleaved if complex), distinct buffers.
 * ---------------------------------------------------------------------------------- */
int oracle_hemm(const void *H, int h_is_f32, int is_complex, int64_t N,
                const double *X, double *Y, int64_t ncols,
                double alpha, double beta, const double *shift) {
    if (!H || !X || !Y || !shift || N <= 0 || ncols < 0) return -1;
    int64_t ld = (is_complex ? 2 : 1) * N;
    for (int64_t j = 0; j < ncols; ++j) {       /* one column at a time: its own shift */
        double *src = (double *)(X + j * ld);
        double *dst = Y + j * ld;
        if (is_complex) step_complex(H, h_is_f32, N, 1, &src, &dst, alpha, beta, shift[j]);
        else            step_real(H, h_is_f32, N, 1, &src, &dst, alpha, beta, shift[j]);
    }
    return 0;
}

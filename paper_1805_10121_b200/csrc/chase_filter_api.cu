// Host orchestration of the Chebyshev filter (Alg. 4) behind the C ABI of
// include/chase_filter.h: validation, the sigma recurrence (l.2-5, 8, 11), the active-suffix
// schedule (l.12-14) and one fused step kernel per degree on one CUDA stream.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <exception>
#include <new>
#include <vector>

#include "chase_internal.h"

namespace chase {
static std::atomic<int64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

static size_t elem_bytes(chase_dtype_t dtype) {
    switch (dtype) {
        case CHASE_F32: return 4;
        case CHASE_F64: return 8;
        case CHASE_C64: return 8;
        case CHASE_C128: return 16;
        default: return 0;
    }
}
static const int64_t kMaxDim = (int64_t)1 << 30;   // keeps every index product inside int64
}  // namespace chase

using namespace chase;

extern "C" {

const char *chase_filter_strerror(int code) {
    switch (code) {
        case CHASE_OK: return "success";
        case CHASE_ERR_ARG: return "invalid argument (null pointer or bad size)";
        case CHASE_ERR_BOUNDS: return "bounds must satisfy lambda1 < a < b and be finite";
        case CHASE_ERR_DEGREES: return "degrees must be >= 0, <= CHASE_MAX_DEGREE and non-decreasing";
        case CHASE_ERR_DTYPE: return "unknown dtype";
        case CHASE_ERR_WORKSPACE: return "workspace missing or too small";
        case CHASE_ERR_ALIGN: return "H, V and workspace must be 16-byte aligned";
        case CHASE_ERR_TIMEOUT: return "a peer rank did not reach an inter-GPU barrier in time";
        case CHASE_ERR_STATIC_LIMIT:
            return "problem too large for the library's static scratch (CHASE_STATIC_SCRATCH_BYTES); use chase_residuals";
        default:
            if (code > 0) return cudaGetErrorString((cudaError_t)code);
            return "unknown error";
    }
}

int64_t chase_filter_launch_count(void) { return g_launches.load(); }

size_t chase_filter_workspace_bytes(int64_t N, int64_t ncols, chase_dtype_t dtype) {
    size_t w = elem_bytes(dtype);
    if (w == 0 || N <= 0 || ncols < 0 || N > kMaxDim || ncols > kMaxDim) return 0;
    size_t bytes = ((size_t)N * (size_t)ncols * w + 255) / 256 * 256;
    const int path = chase_filter_kernel_path(N, ncols, dtype);
    if (path == 2) bytes += 256;                         // tcgen05 path: soft grid barrier counter
    if (path == 1) bytes += dmma_sk_scratch_bytes();     // FP64 tensor path: stream-K flags + partial tiles
    return bytes;
}

int chase_filter_scalars(double a, double b, double lambda1, int32_t m_max,
                         double *alpha, double *beta, double *c_out) {
    if (m_max < 0 || (m_max > 0 && (!alpha || !beta))) return CHASE_ERR_ARG;
    if (!(std::isfinite(a) && std::isfinite(b) && std::isfinite(lambda1))) return CHASE_ERR_BOUNDS;
    if (!(lambda1 < a && a < b)) return CHASE_ERR_BOUNDS;
    const double c = 0.5 * (b + a);               // Alg. 4 l.2
    const double e = 0.5 * (b - a);               // l.2
    const double sigma1 = e / (lambda1 - c);      // l.3
    if (c_out) *c_out = c;
    double sigma = sigma1;                        // l.5
    if (m_max >= 1) {
        alpha[1] = sigma1 / e;                    // l.4
        beta[1] = 0.0;
    }
    for (int32_t k = 2; k <= m_max; ++k) {        // l.7
        const double tau = 1.0 / (2.0 / sigma1 - sigma);   // l.8
        alpha[k] = 2.0 * tau / e;                 // l.9
        beta[k] = -tau * sigma;                   // l.9
        sigma = tau;                              // l.11
    }
    return CHASE_OK;
}

int chase_filter_schedule(const int32_t *degrees, int64_t ncols, int32_t *offset) {
    if (ncols < 0 || ncols > kMaxDim || (ncols > 0 && !degrees)) return CHASE_ERR_ARG;
    int32_t prev = 0;
    for (int64_t j = 0; j < ncols; ++j) {
        if (degrees[j] < 0 || degrees[j] < prev || degrees[j] > CHASE_MAX_DEGREE) return CHASE_ERR_DEGREES;
        prev = degrees[j];
    }
    const int32_t m_max = ncols ? degrees[ncols - 1] : 0;
    if (offset) {
        int64_t s = 0;
        for (int32_t k = 1; k <= m_max; ++k) {    // l.12-14: drop columns whose degree is < k
            while (s < ncols && degrees[s] < k) ++s;
            offset[k] = (int32_t)s;
        }
    }
    return m_max;
}

int chase_degrees(int64_t ncols, const double *resid, const double *ritzv, double tol,
                  double a, double b, int32_t deg_extra, int32_t deg_max,
                  int32_t *degrees_out, int64_t *perm_out) {
    if (ncols < 0 || ncols > kMaxDim || !(tol > 0.0) || !std::isfinite(tol) || deg_extra < 0 || deg_max < 1)
        return CHASE_ERR_ARG;
    if (ncols > 0 && (!resid || !ritzv || !degrees_out)) return CHASE_ERR_ARG;
    if (!(std::isfinite(a) && std::isfinite(b)) || !(a < b)) return CHASE_ERR_BOUNDS;
    const double c = 0.5 * (b + a), e = 0.5 * (b - a);
    try {                                   // no C++ exception may cross the C ABI
    std::vector<int32_t> deg((size_t)ncols);
    for (int64_t j = 0; j < ncols; ++j) {
        if (!(resid[j] > 0.0) || !std::isfinite(resid[j]) || !std::isfinite(ritzv[j])) return CHASE_ERR_ARG;
        const double t = (ritzv[j] - c) / e;                                   // Alg. 5 l.2
        int32_t d = deg_max;
        if (std::fabs(t) > 1.0) {
            const double r = std::sqrt(t * t - 1.0);
            const double rho = std::fmax(std::fabs(t - r), std::fabs(t + r));   // l.3
            const double q = std::fabs(std::log(resid[j] / tol) / std::log(rho));   // l.4
            if (std::isfinite(q) && q < (double)deg_max) {
                const double dq = std::ceil(q) + (double)deg_extra;             // l.4, l.5
                d = dq < (double)deg_max ? (int32_t)dq : deg_max;
            }
        }
        deg[(size_t)j] = d + (d & 1);                                           // l.6
    }
    std::vector<int64_t> order((size_t)ncols);
    for (int64_t j = 0; j < ncols; ++j) order[(size_t)j] = j;
    std::stable_sort(order.begin(), order.end(),
                     [&](int64_t x, int64_t y) { return deg[(size_t)x] < deg[(size_t)y]; });   // Alg. 1 l.15
    for (int64_t i = 0; i < ncols; ++i) {
        degrees_out[i] = deg[(size_t)order[(size_t)i]];
        if (perm_out) perm_out[i] = order[(size_t)i];
    }
    } catch (const std::exception &) {
        return (int)cudaErrorMemoryAllocation;
    }
    return CHASE_OK;
}

}  // extern "C"

// One launch of the step kernel family: Y <- alpha (H X - c X) + beta Y with X, Y whole buffers.
namespace chase {
int launch_one_step(const void *H, int64_t N, const void *X, void *Y, int64_t ncols, double alpha,
                           double beta, double c, const double *c_col, int use_beta, chase_dtype_t dtype,
                           cudaStream_t stream, void *sk_scratch) {
    const int path = chase_filter_kernel_path(N, ncols, dtype);
    const char *force = std::getenv("CHASE_FILTER_FORCE_GENERIC");
    // A few vectors: one streaming pass over H (roofline: HBM).  Measured at c128, N = 40000 on the bulk-copy
    // streaming kernel: 7.2 TB/s (1-2 columns), 6.7 (5), 4.5 (8: FP64 FMA-bound) against 5.5 TB/s for the
    // stream-K narrow-tile tensor kernel, which therefore takes FP64 blocks of 7 and 8 columns.
    const bool fp64_tensor = path == 1 && ncols > 6;
    if (ncols <= kSkinnyMaxCols && !fp64_tensor && !(force && force[0] == '1')) {
        StepArgs sa;
        sa.H = H; sa.X = X; sa.Y = Y; sa.N = N; sa.n = ncols;
        sa.alpha = alpha; sa.beta = beta; sa.c = c; sa.c_col = c_col; sa.use_beta = use_beta;
        if (stream_supported(dtype, sa)) return (int)launch_step_stream(dtype, sa, stream);
        return (int)launch_step_skinny(dtype, sa, stream);
    }
    if (path == 1) {
        DmmaPlan plan;
        cudaError_t e = dmma_plan_create(&plan, dtype, H, N, const_cast<void *>(X), Y, ncols);
        if (e != cudaSuccess) return (int)e;
        plan.sk_scratch = sk_scratch;       // null: stream-ordered memory for this one launch
        e = dmma_launch_step(&plan, 0, 0, alpha, beta, c, use_beta, stream, c_col);
        return (int)e;
    }
    if (path == 2 && ncols >= 32) {   // a 128 x 128 (256) tensor tile only pays with enough columns
        Tf32Plan plan;
        cudaError_t e = tf32_plan_create(&plan, dtype, H, N, const_cast<void *>(X), Y, 0, ncols, stream);
        if (e != cudaSuccess) return (int)e;
        plan.sync_ctr = tf32_shared_sync_counter();     // may be null: the barrier is only a hint
        e = tf32_launch_step(&plan, 0, 0, alpha, beta, c, use_beta, stream, c_col);
        return (int)e;
    }
    StepArgs sa;
    sa.H = H; sa.X = X; sa.Y = Y; sa.N = N; sa.n = ncols;
    sa.alpha = alpha; sa.beta = beta; sa.c = c; sa.c_col = c_col; sa.use_beta = use_beta;
    return (int)launch_step_generic(dtype, sa, stream);
}
}  // namespace chase

extern "C" {

int chase_hemm(const void *H, int64_t N, const void *X, void *Y, int64_t ncols,
               double alpha, double beta, double shift, chase_dtype_t dtype, void *stream_) {
    if (elem_bytes(dtype) == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > kMaxDim || ncols > kMaxDim) return CHASE_ERR_ARG;
    if (!H || (ncols > 0 && (!X || !Y || X == Y))) return CHASE_ERR_ARG;
    if (!(std::isfinite(alpha) && std::isfinite(beta) && std::isfinite(shift))) return CHASE_ERR_ARG;
    if (ncols == 0) return CHASE_OK;
    if (((uintptr_t)H | (uintptr_t)X | (uintptr_t)Y) & 15) return CHASE_ERR_ALIGN;
    return launch_one_step(H, N, X, Y, ncols, alpha, beta, shift, nullptr, beta != 0.0, dtype,
                           (cudaStream_t)stream_);
}

int chase_scratch_cache_release(void) {
    try {
        return (int)dmma_sk_cache_clear();
    } catch (const std::exception &) {
        return (int)cudaErrorUnknown;
    }
}

size_t chase_residuals_workspace_bytes(int64_t N, int64_t ncols, chase_dtype_t dtype) {
    const size_t v = chase_filter_workspace_bytes(N, ncols, dtype);
    if (v == 0 && ncols != 0) return 0;
    return v + ((size_t)ncols * sizeof(double) + 255) / 256 * 256;
}

int chase_residuals(const void *H, int64_t N, const void *V, int64_t ncols, const double *ritzv,
                    double *resid, chase_dtype_t dtype, void *workspace, size_t workspace_bytes,
                    void *stream_) {
    cudaStream_t stream = (cudaStream_t)stream_;
    if (elem_bytes(dtype) == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > kMaxDim || ncols > kMaxDim) return CHASE_ERR_ARG;
    if (!H || (ncols > 0 && (!V || !ritzv || !resid))) return CHASE_ERR_ARG;
    if (ncols == 0) return CHASE_OK;
    for (int64_t j = 0; j < ncols; ++j)
        if (!std::isfinite(ritzv[j])) return CHASE_ERR_ARG;
    if (!workspace || workspace_bytes < chase_residuals_workspace_bytes(N, ncols, dtype)) return CHASE_ERR_WORKSPACE;
    if (((uintptr_t)H | (uintptr_t)V | (uintptr_t)workspace) & 15) return CHASE_ERR_ALIGN;
    const size_t r_bytes = chase_filter_workspace_bytes(N, ncols, dtype);
    double *d_shift = (double *)((char *)workspace + r_bytes);
    // A pageable source is staged by the runtime before cudaMemcpyAsync returns (consumed before return);
    // a pinned one is read in stream order (see the header): no synchronisation either way.
    cudaError_t e = cudaMemcpyAsync(d_shift, ritzv, (size_t)ncols * sizeof(double), cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) return (int)e;
    const size_t vb = ((size_t)N * (size_t)ncols * elem_bytes(dtype) + 255) / 256 * 256;
    void *sk = chase_filter_kernel_path(N, ncols, dtype) == 1 ? (char *)workspace + vb : nullptr;
    int rc = launch_one_step(H, N, V, workspace, ncols, 1.0, 0.0, 0.0, d_shift, 0, dtype, stream, sk);
    if (rc != CHASE_OK) return rc;
    return (int)launch_column_norms(dtype, workspace, N, ncols, resid, stream);
}

size_t chase_lanczos_workspace_bytes(int64_t N, int64_t nvec, int32_t k, chase_dtype_t dtype) {
    const size_t w = elem_bytes(dtype);
    if (w == 0 || N <= 0 || nvec <= 0 || k <= 0 || N > kMaxDim || nvec > 4096 || k > 4096 || k > N) return 0;
    return lanczos_workspace_bytes(N, nvec, k, w);
}

int chase_lanczos(const void *H, int64_t N, const void *V0, int64_t nvec, int32_t k, chase_dtype_t dtype,
                  double *alpha, double *beta, void *workspace, size_t workspace_bytes, void *stream_) {
    const size_t w = elem_bytes(dtype);
    if (w == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || nvec <= 0 || k <= 0 || N > kMaxDim || nvec > 4096 || k > 4096 || k > N) return CHASE_ERR_ARG;
    if (!H || !V0 || !alpha || !beta) return CHASE_ERR_ARG;
    if (!workspace || workspace_bytes < lanczos_workspace_bytes(N, nvec, k, w)) return CHASE_ERR_WORKSPACE;
    if (((uintptr_t)H | (uintptr_t)V0 | (uintptr_t)workspace) & 15) return CHASE_ERR_ALIGN;
    try {
        return (int)lanczos_run(H, N, V0, (int)nvec, k, dtype, w, workspace, alpha, beta, (cudaStream_t)stream_);
    } catch (const std::exception &) {
        return (int)cudaErrorMemoryAllocation;
    }
}

int chase_lanczos_ritz_vectors(const void *workspace, size_t workspace_bytes, int64_t N, int64_t nruns, int32_t k,
                               chase_dtype_t dtype, int64_t run, const double *alpha, const double *beta,
                               double mu_ne, void *Vhat, int64_t ncols_vhat, const int64_t *dst_cols,
                               int64_t max_vecs, int64_t *count, double *ritz_values, void *stream_) {
    const size_t w = elem_bytes(dtype);
    if (w == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || nruns <= 0 || k <= 0 || N > kMaxDim || nruns > 4096 || k > 4096 || k > N) return CHASE_ERR_ARG;
    if (run < 0 || run >= nruns || !alpha || !beta || !count || !std::isfinite(mu_ne)) return CHASE_ERR_ARG;
    if (max_vecs < 0 || ncols_vhat < 0 || ncols_vhat > kMaxDim || (max_vecs > 0 && (!Vhat || !dst_cols))) return CHASE_ERR_ARG;
    for (int64_t i = 0; i < max_vecs; ++i)
        if (dst_cols[i] < 0 || dst_cols[i] >= ncols_vhat) return CHASE_ERR_ARG;
    try {       // two Ritz vectors aimed at one column would race in the kernel: every destination at most once
        std::vector<int64_t> sorted_dst(dst_cols, dst_cols + max_vecs);
        std::sort(sorted_dst.begin(), sorted_dst.end());
        if (std::adjacent_find(sorted_dst.begin(), sorted_dst.end()) != sorted_dst.end()) return CHASE_ERR_ARG;
    } catch (const std::exception &) {
        return (int)cudaErrorMemoryAllocation;
    }
    for (int32_t j = 0; j < k; ++j) {
        const double al = alpha[run * k + j], be = beta[run * k + j];
        if (!std::isfinite(al) || !std::isfinite(be) || be < 0.0) return CHASE_ERR_ARG;
    }
    if (!workspace || workspace_bytes < lanczos_workspace_bytes(N, nruns, k, w)) return CHASE_ERR_WORKSPACE;
    if (((uintptr_t)workspace | (uintptr_t)Vhat) & 15) return CHASE_ERR_ALIGN;
    *count = 0;
    if (max_vecs == 0) return CHASE_OK;
    try {
        return (int)lanczos_ritz_vectors(workspace, N, (int)nruns, k, dtype, w, (int)run, alpha + run * k, beta + run * k,
                                         mu_ne, Vhat, dst_cols, std::min<int64_t>(max_vecs, k), count, ritz_values,
                                         (cudaStream_t)stream_);
    } catch (const std::exception &) {
        return (int)cudaErrorMemoryAllocation;
    }
}

int chase_spectral_estimates(int32_t k, int64_t nruns, const double *alpha, const double *beta, int64_t N,
                             double nev_nex, double sigma, double *b_sup, double *mu_1, double *mu_ne) {
    if (k <= 0 || nruns <= 0 || !alpha || !beta || !b_sup || N <= 0) return CHASE_ERR_ARG;
    for (int64_t i = 0; i < nruns * k; ++i)
        if (!std::isfinite(alpha[i]) || !std::isfinite(beta[i]) || beta[i] < 0.0) return CHASE_ERR_ARG;
    try {
    std::vector<double> lam, wt;
    if (!lanczos_ritz(k, alpha, beta, lam, wt)) return CHASE_ERR_ARG;
    *b_sup = beta[k - 1] + *std::max_element(lam.begin(), lam.end());          // Alg. 6 l.3
    if (nruns == 1) return CHASE_OK;                                            // l.4-5 (`approx`)
    if (!mu_1 || !mu_ne || !(sigma > 0.0) || !std::isfinite(sigma) || !(nev_nex > 0.0) || !(nev_nex < (double)N))
        return CHASE_ERR_ARG;
    std::vector<double> lams, wts;                                              // l.7-8: runs 1 .. n_vec
    double lo = 0.0, hi = 0.0, mu1 = 0.0;
    for (int64_t r = 1; r < nruns; ++r) {
        if (!lanczos_ritz(k, alpha + r * k, beta + r * k, lam, wt)) return CHASE_ERR_ARG;
        const double mn = *std::min_element(lam.begin(), lam.end()), mx = *std::max_element(lam.begin(), lam.end());
        if (r == 1 || mn < mu1) mu1 = mn;                                       // l.12
        if (r == 1 || mn < lo) lo = mn;
        if (r == 1 || mx > hi) hi = mx;
        lams.insert(lams.end(), lam.begin(), lam.end());
        wts.insert(wts.end(), wt.begin(), wt.end());
    }
    // l.10-11: the integral of phi~ (Eq. 10) up to t is sum_j w_j Phi((t - lam_j) / sigma) / n_vec; it is
    // strictly increasing in t, so the root is found by bisection.
    const double target = nev_nex / (double)N, inv = 1.0 / (sigma * std::sqrt(2.0)), nv = (double)(nruns - 1);
    auto integral = [&](double t) {
        double s = 0.0;
        for (size_t i = 0; i < lams.size(); ++i) s += wts[i] * 0.5 * std::erfc(-(t - lams[i]) * inv);
        return s / nv;
    };
    lo -= 40.0 * sigma;
    hi += 40.0 * sigma;
    for (int it = 0; it < 300 && hi - lo > 0.0; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (mid <= lo || mid >= hi) break;
        if (integral(mid) < target) lo = mid; else hi = mid;
    }
    *mu_ne = 0.5 * (lo + hi);
    *mu_1 = mu1;
    } catch (const std::exception &) {
        return (int)cudaErrorMemoryAllocation;
    }
    return CHASE_OK;
}

int chase_filter_kernel_path(int64_t N, int64_t ncols, chase_dtype_t dtype) {
    if (elem_bytes(dtype) == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0) return CHASE_ERR_ARG;
    const char *force = std::getenv("CHASE_FILTER_FORCE_GENERIC");
    if (force && force[0] == '1') return 0;
    if (dmma_supported(N, ncols, dtype)) return 1;
    if (tf32_supported(N, ncols, dtype)) return 2;
    return 0;
}

int chase_filter_step_plan(int64_t N, int64_t n_active, chase_dtype_t dtype, int32_t sms, int32_t *out,
                           int32_t *sk_begin) {
    if (elem_bytes(dtype) == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || n_active <= 0 || N > kMaxDim || n_active > kMaxDim || sms <= 0 || !out) return CHASE_ERR_ARG;
    if (dtype != CHASE_C128 && dtype != CHASE_F64) return CHASE_ERR_DTYPE;
    StepPlan pl;
    try {
        dmma_step_plan(N, n_active, dtype, sms, &pl);
    } catch (const std::exception &) {
        return (int)cudaErrorMemoryAllocation;
    }
    out[0] = pl.tiles_m; out[1] = pl.tiles_n; out[2] = pl.bn_w; out[3] = pl.dp_tiles; out[4] = pl.sk_ctas; out[5] = pl.KT;
    out[6] = pl.grid; out[7] = pl.dp_rounds; out[8] = pl.sk_first;
    if (sk_begin)
        for (int g = 0; g <= pl.sk_ctas; ++g) sk_begin[g] = pl.sk_begin[g];
    return CHASE_OK;
}

}  // extern "C"

namespace chase {
// H (device) is still empty on entry: it is filled from H_host panel by panel on copy_stream while the
// first step already runs on the panels that have arrived (chase_filter_host).
struct HostUpload {
    const void *H_host;
    cudaStream_t copy_stream;
    // result download, column class by column class: the columns of degree k are final after step k (later steps
    // only touch columns to their right, in either buffer), so they go back to the host while the remaining steps
    // run.  d2h_stream / done: a stream and a reusable event of the caller; V_host null = no early download.
    void *V_host;
    cudaStream_t d2h_stream;
    cudaEvent_t done;
};
static int filter_impl(const void *H, int64_t N, void *V, int64_t ncols, const int32_t *degrees,
                       double a, double b, double lambda1, chase_dtype_t dtype,
                       void *workspace, size_t workspace_bytes, void *stream_, const HostUpload *up);
}  // namespace chase

extern "C" {

int chase_filter_ws(const void *H, int64_t N, void *V, int64_t ncols, const int32_t *degrees,
                    double a, double b, double lambda1, chase_dtype_t dtype,
                    void *workspace, size_t workspace_bytes, void *stream_) {
    return filter_impl(H, N, V, ncols, degrees, a, b, lambda1, dtype, workspace, workspace_bytes, stream_, nullptr);
}

}  // extern "C"

static int chase::filter_impl(const void *H, int64_t N, void *V, int64_t ncols, const int32_t *degrees,
                              double a, double b, double lambda1, chase_dtype_t dtype,
                              void *workspace, size_t workspace_bytes, void *stream_, const HostUpload *up) {
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t w = elem_bytes(dtype);
    if (w == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > kMaxDim || ncols > kMaxDim) return CHASE_ERR_ARG;
    if (!H || (ncols > 0 && (!V || !degrees))) return CHASE_ERR_ARG;
    if (!(std::isfinite(a) && std::isfinite(b) && std::isfinite(lambda1))) return CHASE_ERR_BOUNDS;
    if (!(lambda1 < a && a < b)) return CHASE_ERR_BOUNDS;
    const int m_max = chase_filter_schedule(degrees, ncols, nullptr);
    if (m_max < 0) return m_max;
    if (ncols == 0 || m_max == 0) return CHASE_OK;
    if (!workspace || workspace_bytes < chase_filter_workspace_bytes(N, ncols, dtype))
        return CHASE_ERR_WORKSPACE;
    if (((uintptr_t)H | (uintptr_t)V | (uintptr_t)workspace) & 15) return CHASE_ERR_ALIGN;

    // m_max <= CHASE_MAX_DEGREE (chase_filter_schedule): fixed-size plans, no allocation that could throw
    int32_t offset[CHASE_MAX_DEGREE + 1];
    double alpha[CHASE_MAX_DEGREE + 1], beta[CHASE_MAX_DEGREE + 1];
    double c = 0.0;
    chase_filter_schedule(degrees, ncols, offset);
    int rc = chase_filter_scalars(a, b, lambda1, m_max, alpha, beta, &c);
    if (rc != CHASE_OK) return rc;

    // Two buffers, roles swapped after every step (Alg. 4 l.10; Listing 2):
    // V_k lives in buf[k & 1]; step k reads buf[(k-1)&1] and overwrites V_{k-2} in buf[k&1]
    // in place (V_{k-2} is an element-wise epilogue operand only, never a GEMM operand).
    void *buf[2] = {V, workspace};
    const size_t col_bytes = (size_t)N * w;

    const int path = chase_filter_kernel_path(N, ncols, dtype);
    const bool use_dmma = path == 1, use_tf32 = path == 2;
    DmmaPlan plan;
    Tf32Plan tplan;
    if (use_dmma) {
        cudaError_t e = dmma_plan_create(&plan, dtype, H, N, V, workspace, ncols);
        if (e != cudaSuccess) return (int)e;
        plan.sk_scratch = (char *)workspace + ((size_t)N * (size_t)ncols * w + 255) / 256 * 256;
    }
    if (use_tf32) {
        const size_t vb = ((size_t)N * (size_t)ncols * w + 255) / 256 * 256;
        cudaError_t e = tf32_plan_create(&tplan, dtype, H, N, V, workspace, vb, ncols, stream);
        if (e != cudaSuccess) return (int)e;
    }

    if (up && !use_dmma) {   // no panel-wise first step on this kernel family: plain upload, then the usual loop
        cudaError_t e = cudaMemcpyAsync(const_cast<void *>(H), up->H_host, (size_t)N * (size_t)N * w,
                                        cudaMemcpyHostToDevice, stream);
        if (e != cudaSuccess) return (int)e;
    }
    // chase_filter_host: the columns of degree k (final after step k, in buf[k & 1]) go back to the host behind an event
    const bool early_d2h = up && up->V_host;
    auto download_class = [&](int k) -> cudaError_t {
        if (!early_d2h) return cudaSuccess;
        const int64_t j0 = offset[k], j1 = k < m_max ? offset[k + 1] : ncols;
        if (j1 <= j0) return cudaSuccess;
        cudaError_t e = cudaEventRecord(up->done, stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(up->d2h_stream, up->done, 0);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync((char *)up->V_host + (size_t)j0 * col_bytes, (const char *)buf[k & 1] + (size_t)j0 * col_bytes,
                                (size_t)(j1 - j0) * col_bytes, cudaMemcpyDeviceToHost, up->d2h_stream);
        return e;
    };
    for (int k = 1; k <= m_max; ++k) {
        const int64_t s = offset[k];
        const int src = (k - 1) & 1;
        cudaError_t e;
        if (use_dmma && k == 1 && up) {
            // Step 1 row panel by row panel, each as soon as its rows of H have landed: the upload of H
            // (26 GB at cfg 4, ~0.5 s over PCIe) hides behind the first step (~0.7 s).
            const int64_t tiles = (N + 127) / 128;
            const int panels = (int)std::min<int64_t>(8, tiles);      // (16 panels measured no better: 15.86 vs 15.70 s)
            const int64_t rows_per = (tiles + panels - 1) / panels * 128;
            struct Events {                 // destroyed on every exit path
                cudaEvent_t ev[16];
                int n = 0;
                ~Events() { for (int i = 0; i < n; ++i) cudaEventDestroy(ev[i]); }
            } evs;
            cudaEvent_t *ev = evs.ev;
            for (int64_t r0 = 0; r0 < N; r0 += rows_per) {
                const int64_t rows = std::min(rows_per, N - r0);
                cudaEvent_t evp;
                if (evs.n >= 16) return CHASE_ERR_ARG;
                if ((e = cudaEventCreateWithFlags(&evp, cudaEventDisableTiming)) != cudaSuccess) return (int)e;
                ev[evs.n++] = evp;
                e = cudaMemcpy2DAsync((char *)const_cast<void *>(H) + (size_t)r0 * w, (size_t)N * w,
                                      (const char *)up->H_host + (size_t)r0 * w, (size_t)N * w, (size_t)rows * w,
                                      (size_t)N, cudaMemcpyHostToDevice, up->copy_stream);
                if (e == cudaSuccess) e = cudaEventRecord(evp, up->copy_stream);
                if (e != cudaSuccess) return (int)e;
            }
            int pi = 0;
            for (int64_t r0 = 0; r0 < N; r0 += rows_per, ++pi) {
                const int64_t rows = std::min(rows_per, N - r0);
                DmmaPlan pp;
                if ((e = cudaStreamWaitEvent(stream, ev[pi], 0)) != cudaSuccess) return (int)e;
                if ((e = dmma_plan_create_panel(&pp, dtype, H, N, r0, rows, V, workspace, ncols)) != cudaSuccess) return (int)e;
                // the panels run one after the other on `stream`: they share the workspace's stream-K scratch, with
                // the flag epoch and the soft-barrier count carried from panel to panel and on into the later steps
                pp.sk_scratch = plan.sk_scratch;
                pp.sk_epoch = plan.sk_epoch;
                pp.sync_count = plan.sync_count;
                e = dmma_launch_step(&pp, src, s, alpha[k], beta[k], c, 0, stream);
                plan.sk_epoch = pp.sk_epoch;
                plan.sync_count = pp.sync_count;
                if (e != cudaSuccess) return (int)e;
            }
            if ((e = download_class(k)) != cudaSuccess) return (int)e;
            continue;
        }
        // Few active columns left (the tail of a sorted-degree schedule): one streaming pass over H beats a
        // tensor tile that would be mostly padding (tcgen05 tiles are 128 / 256 columns wide; FP64: see
        // launch_one_step for the measured crossover).
        StepArgs ska;
        ska.H = H;
        ska.X = (const char *)buf[src] + (size_t)s * col_bytes;
        ska.Y = (char *)buf[src ^ 1] + (size_t)s * col_bytes;
        ska.N = N; ska.n = ncols - s;
        ska.alpha = alpha[k]; ska.beta = beta[k]; ska.c = c; ska.use_beta = k > 1;
        const bool few = ska.n <= (use_dmma ? 6 : kSkinnyMaxCols) && !(up && k == 1);
        if ((use_dmma || use_tf32) && few && stream_supported(dtype, ska)) {
            e = launch_step_stream(dtype, ska, stream);
        } else if (use_dmma) {
            e = dmma_launch_step(&plan, src, s, alpha[k], beta[k], c, k > 1, stream);
        } else if (use_tf32) {
            e = tf32_launch_step(&tplan, src, s, alpha[k], beta[k], c, k > 1, stream);
        } else {
            StepArgs sa;
            sa.H = H;
            sa.X = (const char *)buf[src] + (size_t)s * col_bytes;
            sa.Y = (char *)buf[src ^ 1] + (size_t)s * col_bytes;
            sa.N = N;
            sa.n = ncols - s;
            sa.alpha = alpha[k];
            sa.beta = beta[k];
            sa.c = c;
            sa.use_beta = k > 1;
            e = launch_step_generic(dtype, sa, stream);
        }
        if (e != cudaSuccess) return (int)e;
        if ((e = download_class(k)) != cudaSuccess) return (int)e;
    }
    if (early_d2h) return CHASE_OK;        // every column went to the host from the buffer it ended in

    // Result placement: V_{m_j} of an odd-degree column ended in the scratch
    // buffer; copy each contiguous run of odd-degree columns back (none for Alg. 5's degrees).
    for (int64_t j = 0; j < ncols;) {
        if ((degrees[j] & 1) == 0) { ++j; continue; }
        int64_t j1 = j;
        while (j1 < ncols && (degrees[j1] & 1)) ++j1;
        cudaError_t e = cudaMemcpyAsync((char *)V + (size_t)j * col_bytes,
                                        (const char *)workspace + (size_t)j * col_bytes,
                                        (size_t)(j1 - j) * col_bytes, cudaMemcpyDeviceToDevice, stream);
        if (e != cudaSuccess) return (int)e;
        j = j1;
    }
    return CHASE_OK;
}

extern "C" {

int chase_filter(const void *H, int64_t N, void *V, int64_t ncols, const int32_t *degrees,
                 double a, double b, double lambda1, chase_dtype_t dtype, void *stream_) {
    cudaStream_t stream = (cudaStream_t)stream_;
    if (chase::elem_bytes(dtype) == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > kMaxDim || ncols > kMaxDim) return CHASE_ERR_ARG;
    const int m_max = chase_filter_schedule(degrees, ncols, nullptr);
    if (m_max < 0) return m_max;
    if (ncols == 0 || m_max == 0) {
        // still validate the remaining arguments the same way chase_filter_ws does
        return chase_filter_ws(H, N, V, ncols, degrees, a, b, lambda1, dtype, nullptr, 0, stream_);
    }
    const size_t bytes = chase_filter_workspace_bytes(N, ncols, dtype);
    void *ws = nullptr;
    cudaError_t e = cudaMallocAsync(&ws, bytes, stream);
    if (e != cudaSuccess) return (int)e;
    int rc = chase_filter_ws(H, N, V, ncols, degrees, a, b, lambda1, dtype, ws, bytes, stream_);
    e = cudaFreeAsync(ws, stream);
    if (rc != CHASE_OK) return rc;
    return e == cudaSuccess ? CHASE_OK : (int)e;
}

int chase_filter_host(const void *H_host, int64_t N, void *V_host, int64_t ncols,
                      const int32_t *degrees, double a, double b, double lambda1,
                      chase_dtype_t dtype, int device) {
    const size_t w = chase::elem_bytes(dtype);
    if (w == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > kMaxDim || ncols > kMaxDim) return CHASE_ERR_ARG;
    if (!H_host || (ncols > 0 && (!V_host || !degrees))) return CHASE_ERR_ARG;
    if (!(std::isfinite(a) && std::isfinite(b) && std::isfinite(lambda1))) return CHASE_ERR_BOUNDS;
    if (!(lambda1 < a && a < b)) return CHASE_ERR_BOUNDS;
    const int m_max = chase_filter_schedule(degrees, ncols, nullptr);
    if (m_max < 0) return m_max;
    if (ncols == 0 || m_max == 0) return CHASE_OK;

    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return (int)e;
    const size_t hb = (size_t)N * (size_t)N * w, vb = (size_t)N * (size_t)ncols * w;
    const size_t wb = chase_filter_workspace_bytes(N, ncols, dtype);
    void *dH = nullptr, *dV = nullptr, *dW = nullptr;
    cudaStream_t st = nullptr;
    int rc = CHASE_OK;
    auto fail = [&](cudaError_t err) { rc = (int)err; };
    if ((e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking)) != cudaSuccess) return (int)e;
    if ((e = cudaMalloc(&dH, hb)) != cudaSuccess) fail(e);
    if (rc == CHASE_OK && (e = cudaMalloc(&dV, vb)) != cudaSuccess) fail(e);
    if (rc == CHASE_OK && (e = cudaMalloc(&dW, wb)) != cudaSuccess) fail(e);
    cudaStream_t cp = nullptr;
    if (rc == CHASE_OK && (e = cudaStreamCreateWithFlags(&cp, cudaStreamNonBlocking)) != cudaSuccess) fail(e);
    if (rc == CHASE_OK && (e = cudaMemcpyAsync(dV, V_host, vb, cudaMemcpyHostToDevice, st)) != cudaSuccess) fail(e);
    cudaStream_t dl = nullptr;
    cudaEvent_t done = nullptr;
    if (rc == CHASE_OK && (e = cudaStreamCreateWithFlags(&dl, cudaStreamNonBlocking)) != cudaSuccess) fail(e);
    if (rc == CHASE_OK && (e = cudaEventCreateWithFlags(&done, cudaEventDisableTiming)) != cudaSuccess) fail(e);
    if (rc == CHASE_OK) {   // H goes up inside the filter, overlapped with its first step; finished column classes
                            // go down while the remaining steps run (degree-0 columns never leave the host)
        // (only for large blocks: a copy into pageable memory blocks the host until the step before it has run,
        //  which would cost a latency-bound small call its launch overlap)
        const bool early = vb >= ((size_t)64 << 20);
        HostUpload up{H_host, cp, early ? V_host : nullptr, dl, done};
        rc = filter_impl(dH, N, dV, ncols, degrees, a, b, lambda1, dtype, dW, wb, (void *)st, &up);
        if (rc == CHASE_OK && !early &&
            (e = cudaMemcpyAsync(V_host, dV, vb, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
            fail(e);
    }
    (void)hb;
    e = cudaStreamSynchronize(st);
    if (rc == CHASE_OK && e != cudaSuccess) fail(e);
    if (dl) {
        e = cudaStreamSynchronize(dl);
        if (rc == CHASE_OK && e != cudaSuccess) fail(e);
        cudaStreamDestroy(dl);
    }
    if (done) cudaEventDestroy(done);
    cudaFree(dH);
    cudaFree(dV);
    cudaFree(dW);
    if (cp) {
        cudaStreamSynchronize(cp);
        cudaStreamDestroy(cp);
    }
    cudaStreamDestroy(st);
    return rc;
}


// ---- chase_filter_host with H kept on the device across calls (chase_filter_host_open / _run / _close) ----
namespace {
struct HostFilter {
    int device = 0;
    chase_dtype_t dtype = CHASE_C128;
    int64_t N = 0, max_ncols = 0;
    size_t ws_bytes = 0;
    void *dH = nullptr, *dV = nullptr, *dW = nullptr;
    cudaStream_t st = nullptr;
};
void host_filter_destroy(HostFilter *h) {
    if (!h) return;
    if (h->st) { cudaStreamSynchronize(h->st); cudaStreamDestroy(h->st); }
    cudaFree(h->dH);
    cudaFree(h->dV);
    cudaFree(h->dW);
    delete h;
}
}  // namespace

int chase_filter_host_open(const void *H_host, int64_t N, int64_t max_ncols, chase_dtype_t dtype, int device,
                           void **handle_out) {
    const size_t w = chase::elem_bytes(dtype);
    if (w == 0) return CHASE_ERR_DTYPE;
    if (!H_host || !handle_out || N <= 0 || max_ncols <= 0 || N > kMaxDim || max_ncols > kMaxDim) return CHASE_ERR_ARG;
    *handle_out = nullptr;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return (int)e;
    HostFilter *h = new (std::nothrow) HostFilter;
    if (!h) return (int)cudaErrorMemoryAllocation;
    h->device = device; h->dtype = dtype; h->N = N; h->max_ncols = max_ncols;
    // the scratch of the widest call serves every narrower one (same kernel family: it depends on N and dtype only)
    h->ws_bytes = chase_filter_workspace_bytes(N, max_ncols, dtype);
    const size_t hb = (size_t)N * (size_t)N * w;
    if ((e = cudaStreamCreateWithFlags(&h->st, cudaStreamNonBlocking)) == cudaSuccess &&
        (e = cudaMalloc(&h->dH, hb)) == cudaSuccess &&
        (e = cudaMalloc(&h->dV, (size_t)N * (size_t)max_ncols * w)) == cudaSuccess &&
        (e = cudaMalloc(&h->dW, h->ws_bytes)) == cudaSuccess &&
        (e = cudaMemcpyAsync(h->dH, H_host, hb, cudaMemcpyHostToDevice, h->st)) == cudaSuccess)
        e = cudaStreamSynchronize(h->st);
    if (e != cudaSuccess) {
        host_filter_destroy(h);
        return (int)e;
    }
    *handle_out = h;
    return CHASE_OK;
}

int chase_filter_host_run(void *handle, void *V_host, int64_t ncols, const int32_t *degrees, double a, double b,
                          double lambda1) {
    HostFilter *h = (HostFilter *)handle;
    if (!h || ncols < 0 || ncols > h->max_ncols || (ncols > 0 && (!V_host || !degrees))) return CHASE_ERR_ARG;
    const int m_max = chase_filter_schedule(degrees, ncols, nullptr);
    if (m_max < 0) return m_max;
    if (!(std::isfinite(a) && std::isfinite(b) && std::isfinite(lambda1))) return CHASE_ERR_BOUNDS;
    if (!(lambda1 < a && a < b)) return CHASE_ERR_BOUNDS;
    if (ncols == 0 || m_max == 0) return CHASE_OK;
    cudaError_t e = cudaSetDevice(h->device);
    if (e != cudaSuccess) return (int)e;
    const size_t w = chase::elem_bytes(h->dtype);
    int64_t j0 = 0;                                     // degree-0 columns never leave the host
    while (j0 < ncols && degrees[j0] == 0) ++j0;
    const size_t off = (size_t)j0 * (size_t)h->N * w, vb = (size_t)(ncols - j0) * (size_t)h->N * w;
    if ((e = cudaMemcpyAsync((char *)h->dV + off, (const char *)V_host + off, vb, cudaMemcpyHostToDevice, h->st)) != cudaSuccess)
        return (int)e;
    int rc = filter_impl(h->dH, h->N, h->dV, ncols, degrees, a, b, lambda1, h->dtype, h->dW, h->ws_bytes, (void *)h->st,
                         nullptr);
    if (rc == CHASE_OK &&
        (e = cudaMemcpyAsync((char *)V_host + off, (const char *)h->dV + off, vb, cudaMemcpyDeviceToHost, h->st)) != cudaSuccess)
        rc = (int)e;
    e = cudaStreamSynchronize(h->st);
    if (rc == CHASE_OK && e != cudaSuccess) rc = (int)e;
    return rc;
}

int chase_filter_host_close(void *handle) {
    if (!handle) return CHASE_ERR_ARG;
    HostFilter *h = (HostFilter *)handle;
    const cudaError_t e = cudaSetDevice(h->device);
    host_filter_destroy(h);
    return (int)e;
}

}  // extern "C"

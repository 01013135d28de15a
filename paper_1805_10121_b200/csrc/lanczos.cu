// Spectral estimates (Alg. 6 "Lanczos procedure for parameters estimates", PAPER.md:421-475;
// Eq. (9)-(10)): 1 + n_vec Lanczos runs of k steps advanced TOGETHER, so that the
// matrix-vector products of one step are a single HEMM on an N x (1 + n_vec) block ("the n_vec
// matrix-vector multiplications are coalesced into a single HEMM") -- the step kernel
// of the filter with alpha = 1, beta = 0, no shift.  Everything else of a step (Gram-Schmidt
// coefficients, vector updates, norms) runs in the small kernels below without leaving the device;
// the 2 k (1 + n_vec) Lanczos coefficients are copied to the host once at the end, where the
// tridiagonal eigenproblems, the DoS integral and b_sup are evaluated (chase_spectral_estimates).
//
// Reading G19: full re-orthogonalisation by two passes of classical Gram-Schmidt against
// all previous Lanczos vectors; alpha_j is the j-th coefficient of the first pass.
#include <algorithm>
#include <cmath>
#include <vector>

#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kBlock = 256;
constexpr int kRedBlock = 1024;   // the reductions run one block per (vector pair): wide blocks, 4 loads in flight per thread

__device__ __forceinline__ double2 ld(const float *p, int64_t i)   { return make_double2((double)p[i], 0.0); }
__device__ __forceinline__ double2 ld(const double *p, int64_t i)  { return make_double2(p[i], 0.0); }
__device__ __forceinline__ double2 ld(const float2 *p, int64_t i)  { const float2 v = p[i]; return make_double2(v.x, v.y); }
__device__ __forceinline__ double2 ld(const double2 *p, int64_t i) { return p[i]; }
__device__ __forceinline__ void st(float *p, int64_t i, double2 v)   { p[i] = (float)v.x; }
__device__ __forceinline__ void st(double *p, int64_t i, double2 v)  { p[i] = v.x; }
__device__ __forceinline__ void st(float2 *p, int64_t i, double2 v)  { p[i] = make_float2((float)v.x, (float)v.y); }
__device__ __forceinline__ void st(double2 *p, int64_t i, double2 v) { p[i] = v; }

// Sum of a double2 over the block (any block size that is a multiple of 32, up to 1024); result valid in thread 0.
__device__ __forceinline__ double2 block_sum(double2 v) {
    __shared__ double2 part[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_down_sync(0xffffffffu, v.x, o);
        v.y += __shfl_down_sync(0xffffffffu, v.y, o);
    }
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < (blockDim.x >> 5) ? part[threadIdx.x] : make_double2(0.0, 0.0);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            v.x += __shfl_down_sync(0xffffffffu, v.x, o);
            v.y += __shfl_down_sync(0xffffffffu, v.y, o);
        }
    }
    return v;
}

// h[i, c] = U_i[:, c]^H w[:, c]  for i = blockIdx.x <= j, run c = blockIdx.y.  U_i is block i of U
// (each block N x nvec, column-major).  pass 0 also records alpha_j[c] = Re h[j, c].
template <typename T>
__global__ void __launch_bounds__(kRedBlock) lz_project(const T *__restrict__ U, const T *__restrict__ w, int64_t N,
                                                        int nvec, int j, double2 *__restrict__ h,
                                                        double *__restrict__ alpha, int k, int pass) {
    const int i = blockIdx.x, c = blockIdx.y;
    const T *u = U + ((int64_t)i * nvec + c) * N;
    const T *x = w + (int64_t)c * N;
    double2 a4[4] = {};
    for (int64_t r0 = threadIdx.x; r0 < N; r0 += 4 * kRedBlock) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int64_t r = r0 + (int64_t)q * kRedBlock;
            if (r < N) {
                const double2 a = ld(u, r), b = ld(x, r);
                a4[q].x += a.x * b.x + a.y * b.y;          // conj(a) * b
                a4[q].y += a.x * b.y - a.y * b.x;
            }
        }
    }
    double2 acc = make_double2((a4[0].x + a4[1].x) + (a4[2].x + a4[3].x), (a4[0].y + a4[1].y) + (a4[2].y + a4[3].y));
    acc = block_sum(acc);
    if (threadIdx.x == 0) {
        h[(int64_t)i * nvec + c] = acc;
        if (pass == 0 && i == j) alpha[(int64_t)c * k + j] = acc.x;
    }
}

// w[:, c] -= sum_{i <= j} h[i, c] U_i[:, c]
template <typename T>
__global__ void __launch_bounds__(kBlock) lz_update(const T *__restrict__ U, T *__restrict__ w, int64_t N, int nvec,
                                                    int j, const double2 *__restrict__ h) {
    const int c = blockIdx.y;
    const int64_t r = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (r >= N) return;
    T *x = w + (int64_t)c * N;
    double2 v = ld(x, r);
    for (int i = 0; i <= j; ++i) {
        const double2 a = ld(U + ((int64_t)i * nvec + c) * N, r);
        const double2 g = h[(int64_t)i * nvec + c];
        v.x -= g.x * a.x - g.y * a.y;
        v.y -= g.x * a.y + g.y * a.x;
    }
    st(x, r, v);
}

// out[c * stride + idx] = || x[:, c] ||_2
template <typename T>
__global__ void __launch_bounds__(kRedBlock) lz_colnorm(const T *__restrict__ x, int64_t N, double *__restrict__ out,
                                                        int stride, int idx) {
    const int c = blockIdx.x;
    const T *p = x + (int64_t)c * N;
    double a4[4] = {};
    for (int64_t r0 = threadIdx.x; r0 < N; r0 += 4 * kRedBlock) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int64_t r = r0 + (int64_t)q * kRedBlock;
            if (r < N) {
                const double2 a = ld(p, r);
                a4[q] += a.x * a.x + a.y * a.y;
            }
        }
    }
    double2 acc = make_double2((a4[0] + a4[1]) + (a4[2] + a4[3]), 0.0);
    acc = block_sum(acc);
    if (threadIdx.x == 0) out[(int64_t)c * stride + idx] = sqrt(acc.x);
}

// y[:, c] = x[:, c] / nrm[c * stride + idx]
template <typename T>
__global__ void __launch_bounds__(kBlock) lz_scale(const T *__restrict__ x, T *__restrict__ y, int64_t N,
                                                   const double *__restrict__ nrm, int stride, int idx) {
    const int c = blockIdx.y;
    const int64_t r = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (r >= N) return;
    const double s = 1.0 / nrm[(int64_t)c * stride + idx];
    const double2 v = ld(x + (int64_t)c * N, r);
    st(y + (int64_t)c * N, r, make_double2(v.x * s, v.y * s));
}

size_t round256(size_t b) { return (b + 255) / 256 * 256; }

template <typename T>
cudaError_t run(const void *H, int64_t N, const void *V0, int nvec, int k, chase_dtype_t dtype, void *workspace,
                double *d_alpha, double *d_beta, double2 *d_h, cudaStream_t stream) {
    T *U = (T *)workspace;                                            // k blocks of N x nvec
    T *w = U + (size_t)k * N * nvec;                                  // N x nvec
    const dim3 grid_rows((unsigned)((N + kBlock - 1) / kBlock), (unsigned)nvec);
    // u_0 = v_0 / ||v_0||; the start norm is parked in beta[.., 0] and overwritten by step 0
    lz_colnorm<T><<<nvec, kRedBlock, 0, stream>>>((const T *)V0, N, d_beta, k, 0);
    lz_scale<T><<<grid_rows, kBlock, 0, stream>>>((const T *)V0, U, N, d_beta, k, 0);
    count_launch(); count_launch();
    for (int j = 0; j < k; ++j) {
        const T *uj = U + (size_t)j * N * nvec;
        int rc = launch_one_step(H, N, uj, w, nvec, 1.0, 0.0, 0.0, nullptr, 0, dtype, stream);   // w = A u_j, all runs
        if (rc != 0) return rc > 0 ? (cudaError_t)rc : cudaErrorInvalidValue;
        for (int pass = 0; pass < 2; ++pass) {
            lz_project<T><<<dim3(j + 1, nvec), kRedBlock, 0, stream>>>(U, w, N, nvec, j, d_h, d_alpha, k, pass);
            lz_update<T><<<grid_rows, kBlock, 0, stream>>>(U, w, N, nvec, j, d_h);
            count_launch(); count_launch();
        }
        lz_colnorm<T><<<nvec, kRedBlock, 0, stream>>>(w, N, d_beta, k, j);     // beta_j = ||w||; j = k-1: ||f_k||
        count_launch();
        if (j + 1 < k) {
            lz_scale<T><<<grid_rows, kBlock, 0, stream>>>(w, U + (size_t)(j + 1) * N * nvec, N, d_beta, k, j);
            count_launch();
        }
    }
    return cudaGetLastError();
}

// Eigenvalues of the symmetric tridiagonal T (diagonal d[0..n), off-diagonal e[0..n-1)) and the first
// `zrows` ROWS of its normalised eigenvector matrix, by the implicit-shift QL iteration with the
// rotations applied to those rows of the identity (zrows = 1: Golub-Welsch, only the first components;
// zrows = n: all eigenvectors, column i belonging to d[i]).  On return d holds the eigenvalues
// (unsorted), z (row-major zrows x n) the rows.  Returns false if an eigenvalue needs more than 60 sweeps.
bool tridiag_ql(int n, std::vector<double> &d, std::vector<double> &e, std::vector<double> &z, int zrows) {
    e.resize(n, 0.0);
    z.assign((size_t)zrows * n, 0.0);
    for (int r = 0; r < zrows; ++r) z[(size_t)r * n + r] = 1.0;
    const double eps = 2.220446049250313e-16;
    for (int l = 0; l < n; ++l) {
        int iter = 0, m;
        do {
            for (m = l; m < n - 1; ++m) {
                const double dd = std::fabs(d[m]) + std::fabs(d[m + 1]);
                if (std::fabs(e[m]) <= eps * dd) break;
            }
            if (m != l) {
                if (++iter > 60) return false;
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = std::hypot(g, 1.0);
                g = d[m] - d[l] + e[l] / (g + (g >= 0.0 ? std::fabs(r) : -std::fabs(r)));
                double s = 1.0, c = 1.0, p = 0.0;
                int i;
                for (i = m - 1; i >= l; --i) {
                    double f = s * e[i];
                    const double b = c * e[i];
                    r = std::hypot(f, g);
                    e[i + 1] = r;
                    if (r == 0.0) {
                        d[i + 1] -= p;
                        e[m] = 0.0;
                        break;
                    }
                    s = f / r;
                    c = g / r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - b;
                    for (int row = 0; row < zrows; ++row) {
                        double *zr = &z[(size_t)row * n];
                        f = zr[i + 1];
                        zr[i + 1] = s * zr[i] + c * f;
                        zr[i] = c * zr[i] - s * f;
                    }
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p;
                e[l] = g;
                e[m] = 0.0;
            }
        } while (m != l);
    }
    return true;
}

// Vhat[:, dst[i]] = sum_j U_j[:, run] S[j, i]: the Ritz vectors U^[run] z_i of Alg. 6 l.13 (S = the selected
// eigenvectors of T_k, k x cnt column-major, real).  One thread per (row, output vector).
template <typename T>
__global__ void __launch_bounds__(kBlock) lz_ritz_vectors(const T *__restrict__ U, int64_t N, int nvec, int run, int k,
                                                          const double *__restrict__ S, T *__restrict__ Vhat,
                                                          const int64_t *__restrict__ dst) {
    const int i = blockIdx.y;
    const int64_t r = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (r >= N) return;
    double2 acc = make_double2(0.0, 0.0);
    for (int j = 0; j < k; ++j) {
        const double2 u = ld(U + ((int64_t)j * nvec + run) * N, r);
        const double sji = S[(int64_t)i * k + j];
        acc.x = fma(sji, u.x, acc.x);
        acc.y = fma(sji, u.y, acc.y);
    }
    st(Vhat + dst[i] * N, r, acc);
}

}  // namespace

size_t lanczos_workspace_bytes(int64_t N, int64_t nvec, int32_t k, size_t elem) {
    const size_t vec = (size_t)N * (size_t)nvec * elem;
    return round256(vec * (size_t)k) + round256(vec)                      // U (k blocks), w
           + 2 * round256((size_t)nvec * k * sizeof(double))              // alpha, beta
           + round256((size_t)nvec * k * sizeof(double2))                 // Gram-Schmidt coefficients
           + round256((size_t)k * k * sizeof(double)) + round256((size_t)k * sizeof(int64_t));   // Ritz-vector coefficients, targets
}

cudaError_t lanczos_run(const void *H, int64_t N, const void *V0, int nvec, int k, chase_dtype_t dtype, size_t elem,
                        void *workspace, double *alpha_host, double *beta_host, cudaStream_t stream) {
    const size_t vec = (size_t)N * (size_t)nvec * elem;
    char *base = (char *)workspace;
    double *d_alpha = (double *)(base + round256(vec * (size_t)k) + round256(vec));
    double *d_beta = (double *)((char *)d_alpha + round256((size_t)nvec * k * sizeof(double)));
    double2 *d_h = (double2 *)((char *)d_beta + round256((size_t)nvec * k * sizeof(double)));
    cudaError_t e;
    switch (dtype) {
        case CHASE_F32:  e = run<float>(H, N, V0, nvec, k, dtype, workspace, d_alpha, d_beta, d_h, stream); break;
        case CHASE_F64:  e = run<double>(H, N, V0, nvec, k, dtype, workspace, d_alpha, d_beta, d_h, stream); break;
        case CHASE_C64:  e = run<float2>(H, N, V0, nvec, k, dtype, workspace, d_alpha, d_beta, d_h, stream); break;
        default:         e = run<double2>(H, N, V0, nvec, k, dtype, workspace, d_alpha, d_beta, d_h, stream); break;
    }
    if (e != cudaSuccess) return e;
    const size_t cb = (size_t)nvec * k * sizeof(double);
    if ((e = cudaMemcpyAsync(alpha_host, d_alpha, cb, cudaMemcpyDeviceToHost, stream)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(beta_host, d_beta, cb, cudaMemcpyDeviceToHost, stream)) != cudaSuccess) return e;
    return cudaStreamSynchronize(stream);
}

cudaError_t lanczos_ritz_vectors(const void *workspace, int64_t N, int nvec, int k, chase_dtype_t dtype, size_t elem,
                                 int run, const double *alpha_run, const double *beta_run, double mu_ne, void *Vhat,
                                 const int64_t *dst_cols, int64_t max_vecs, int64_t *count, double *ritz_values,
                                 cudaStream_t stream) {
    // T_k = Z^H diag(lam) Z on the host (k x k, negligible: PAPER.md:473)
    std::vector<double> d(alpha_run, alpha_run + k), e(beta_run, beta_run + (k > 0 ? k - 1 : 0)), z;
    if (!tridiag_ql(k, d, e, z, k)) return cudaErrorInvalidValue;
    std::vector<int> order(k);
    for (int i = 0; i < k; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int x, int y) { return d[x] < d[y]; });
    std::vector<double> S;
    int64_t cnt = 0;
    for (int oi = 0; oi < k && cnt < max_vecs; ++oi) {
        const int i = order[oi];
        if (!(d[i] < mu_ne)) break;                                       // l.13: Ritz values below mu_{nev+nex}
        const double sgn = z[(size_t)0 * k + i] < 0.0 ? -1.0 : 1.0;       // unique sign: first component >= 0
        for (int j = 0; j < k; ++j) S.push_back(sgn * z[(size_t)j * k + i]);
        if (ritz_values) ritz_values[cnt] = d[i];
        ++cnt;
    }
    *count = cnt;
    if (cnt == 0) return cudaSuccess;
    const size_t vec = (size_t)N * (size_t)nvec * elem;
    char *base = (char *)const_cast<void *>(workspace);
    char *p = base + round256(vec * (size_t)k) + round256(vec) + 2 * round256((size_t)nvec * k * sizeof(double)) +
              round256((size_t)nvec * k * sizeof(double2));
    double *d_S = (double *)p;
    int64_t *d_dst = (int64_t *)(p + round256((size_t)k * k * sizeof(double)));
    cudaError_t err;
    if ((err = cudaMemcpyAsync(d_S, S.data(), S.size() * sizeof(double), cudaMemcpyHostToDevice, stream)) != cudaSuccess) return err;
    if ((err = cudaMemcpyAsync(d_dst, dst_cols, (size_t)cnt * sizeof(int64_t), cudaMemcpyHostToDevice, stream)) != cudaSuccess) return err;
    const dim3 grid((unsigned)((N + kBlock - 1) / kBlock), (unsigned)cnt);
    switch (dtype) {
        case CHASE_F32:  lz_ritz_vectors<float><<<grid, kBlock, 0, stream>>>((const float *)workspace, N, nvec, run, k, d_S, (float *)Vhat, d_dst); break;
        case CHASE_F64:  lz_ritz_vectors<double><<<grid, kBlock, 0, stream>>>((const double *)workspace, N, nvec, run, k, d_S, (double *)Vhat, d_dst); break;
        case CHASE_C64:  lz_ritz_vectors<float2><<<grid, kBlock, 0, stream>>>((const float2 *)workspace, N, nvec, run, k, d_S, (float2 *)Vhat, d_dst); break;
        default:         lz_ritz_vectors<double2><<<grid, kBlock, 0, stream>>>((const double2 *)workspace, N, nvec, run, k, d_S, (double2 *)Vhat, d_dst); break;
    }
    count_launch();
    if ((err = cudaGetLastError()) != cudaSuccess) return err;
    // The documented contract: Vhat is complete when this returns.  (S is pageable, so the runtime staged it
    // before cudaMemcpyAsync returned; the caller's dst_cols may be pinned and is only safe to reuse from here on.)
    return cudaStreamSynchronize(stream);
}

bool lanczos_ritz(int k, const double *alpha, const double *beta, std::vector<double> &lam, std::vector<double> &w) {
    std::vector<double> d(alpha, alpha + k), e(beta, beta + (k > 0 ? k - 1 : 0)), z;
    if (!tridiag_ql(k, d, e, z, 1)) return false;
    lam = d;
    w.resize(k);
    for (int i = 0; i < k; ++i) w[i] = z[i] * z[i];
    return true;
}

}  // namespace chase

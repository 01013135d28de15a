// Generic FMA step kernel: any N, any number of active columns, all four dtypes.
//   Y[:, j] <- alpha * (H X[:, j] - c X[:, j]) + beta * Y[:, j]       (Alg. 4 l.4 / l.9)
// Shared-memory tiled GEMM on the FP32 / FP64 FMA pipes with the shift, scaling and V_{k-1}
// term fused into the epilogue.  It is the correctness path for the shapes neither tensor kernel takes
// -- their TMA views need columns that start on 16-byte boundaries: float64 / complex64 with odd N,
// float32 with N % 4 != 0 -- and for 9..31 active columns of a float32 / complex64 problem.
#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kThreads = 256;   // 16 x 16 thread grid; thread (tx, ty) owns rows tx+16i, cols ty+16j

template <typename R, bool CPLX, int TM, int TN, int BK>
__global__ void __launch_bounds__(kThreads)
step_generic_kernel(const R *__restrict__ H, const R *__restrict__ X, R *Y,
                    int64_t N, int64_t n, R alpha, R beta, R c0, const double *__restrict__ c_col, int use_beta) {
    constexpr int BM = 16 * TM, BN = 16 * TN;
    constexpr int NC = CPLX ? 2 : 1;
    __shared__ R As[NC][BK][BM];
    __shared__ R Bs[NC][BK][BN + 1];

    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const int64_t m0 = (int64_t)blockIdx.x * BM;
    const int64_t n0 = (int64_t)blockIdx.y * BN;

    R acc[NC][TM][TN];
#pragma unroll
    for (int q = 0; q < NC; ++q)
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
            for (int j = 0; j < TN; ++j) acc[q][i][j] = R(0);

    for (int64_t k0 = 0; k0 < N; k0 += BK) {
        // A tile: H[m0 + m, k0 + k], contiguous in m
        for (int idx = tid; idx < BM * BK; idx += kThreads) {
            const int m = idx % BM, k = idx / BM;
            const int64_t gm = m0 + m, gk = k0 + k;
            const bool ok = gm < N && gk < N;
            if (CPLX) {
                As[0][k][m] = ok ? H[2 * (gm + gk * N)] : R(0);
                As[NC - 1][k][m] = ok ? H[2 * (gm + gk * N) + 1] : R(0);
            } else {
                As[0][k][m] = ok ? H[gm + gk * N] : R(0);
            }
        }
        // B tile: X[k0 + k, n0 + j], contiguous in k
        for (int idx = tid; idx < BN * BK; idx += kThreads) {
            const int k = idx % BK, j = idx / BK;
            const int64_t gk = k0 + k, gj = n0 + j;
            const bool ok = gk < N && gj < n;
            if (CPLX) {
                Bs[0][k][j] = ok ? __ldcg(X + 2 * (gk + gj * N)) : R(0);
                Bs[NC - 1][k][j] = ok ? __ldcg(X + 2 * (gk + gj * N) + 1) : R(0);
            } else {
                Bs[0][k][j] = ok ? __ldcg(X + gk + gj * N) : R(0);
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            R ar[TM], ai[TM], br[TN], bi[TN];
#pragma unroll
            for (int i = 0; i < TM; ++i) {
                ar[i] = As[0][k][tx + 16 * i];
                ai[i] = CPLX ? As[NC - 1][k][tx + 16 * i] : R(0);
            }
#pragma unroll
            for (int j = 0; j < TN; ++j) {
                br[j] = Bs[0][k][ty + 16 * j];
                bi[j] = CPLX ? Bs[NC - 1][k][ty + 16 * j] : R(0);
            }
#pragma unroll
            for (int i = 0; i < TM; ++i)
#pragma unroll
                for (int j = 0; j < TN; ++j) {
                    if (CPLX) {
                        acc[0][i][j] = fma(ar[i], br[j], acc[0][i][j]);
                        acc[0][i][j] = fma(-ai[i], bi[j], acc[0][i][j]);
                        acc[NC - 1][i][j] = fma(ar[i], bi[j], acc[NC - 1][i][j]);
                        acc[NC - 1][i][j] = fma(ai[i], br[j], acc[NC - 1][i][j]);
                    } else {
                        acc[0][i][j] = fma(ar[i], br[j], acc[0][i][j]);
                    }
                }
        }
        __syncthreads();
    }

    // fused epilogue: shift, scaling, V_{k-1} term
#pragma unroll
    for (int j = 0; j < TN; ++j) {
        const int64_t gj = n0 + ty + 16 * j;
        if (gj >= n) continue;
        const R c = c_col ? (R)c_col[gj] : c0;
#pragma unroll
        for (int i = 0; i < TM; ++i) {
            const int64_t gm = m0 + tx + 16 * i;
            if (gm >= N) continue;
            const int64_t off = (gm + gj * N) * NC;
#pragma unroll
            for (int q = 0; q < NC; ++q) {
                R v = alpha * (acc[q][i][j] - c * __ldcg(X + off + q));
                if (use_beta) v = fma(beta, __ldcg(Y + off + q), v);
                Y[off + q] = v;
            }
        }
    }
}

template <typename R, bool CPLX, int TM, int TN, int BK>
cudaError_t launch(const StepArgs &a, cudaStream_t stream) {
    constexpr int BM = 16 * TM, BN = 16 * TN;
    dim3 grid((unsigned)((a.N + BM - 1) / BM), (unsigned)((a.n + BN - 1) / BN));
    if (grid.y > 65535) return cudaErrorInvalidConfiguration;
    step_generic_kernel<R, CPLX, TM, TN, BK><<<grid, kThreads, 0, stream>>>(
        (const R *)a.H, (const R *)a.X, (R *)a.Y, a.N, a.n, (R)a.alpha, (R)a.beta, (R)a.c, a.c_col, a.use_beta);
    count_launch();
    return cudaGetLastError();
}

}  // namespace

namespace {
// one CTA per column: sum of |r|^2 in FP64, then sqrt
template <typename R, int NC>
__global__ void __launch_bounds__(256) column_norms_kernel(const R *__restrict__ Rm, int64_t N, double *resid) {
    const R *col = Rm + (int64_t)blockIdx.x * N * NC;
    double s = 0.0;
    for (int64_t i = threadIdx.x; i < N * NC; i += blockDim.x) {
        const double v = (double)col[i];
        s = fma(v, v, s);
    }
    __shared__ double red[256];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) red[threadIdx.x] += red[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) resid[blockIdx.x] = sqrt(red[0]);
}
}  // namespace

cudaError_t launch_column_norms(chase_dtype_t dtype, const void *Rm, int64_t N, int64_t n, double *resid,
                                cudaStream_t stream) {
    if (n <= 0) return cudaSuccess;
    switch (dtype) {
        case CHASE_F32: column_norms_kernel<float, 1><<<(unsigned)n, 256, 0, stream>>>((const float *)Rm, N, resid); break;
        case CHASE_F64: column_norms_kernel<double, 1><<<(unsigned)n, 256, 0, stream>>>((const double *)Rm, N, resid); break;
        case CHASE_C64: column_norms_kernel<float, 2><<<(unsigned)n, 256, 0, stream>>>((const float *)Rm, N, resid); break;
        case CHASE_C128: column_norms_kernel<double, 2><<<(unsigned)n, 256, 0, stream>>>((const double *)Rm, N, resid); break;
        default: return cudaErrorInvalidValue;
    }
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_step_generic(chase_dtype_t dtype, const StepArgs &a, cudaStream_t stream) {
    if (a.n <= 0) return cudaSuccess;
    switch (dtype) {
        case CHASE_F32: return launch<float, false, 8, 8, 8>(a, stream);
        case CHASE_F64: return launch<double, false, 8, 4, 8>(a, stream);
        case CHASE_C64: return launch<float, true, 4, 4, 8>(a, stream);
        case CHASE_C128: return launch<double, true, 4, 2, 8>(a, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace chase

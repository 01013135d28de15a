// Tall-skinny step kernel: Y[:, j] <- alpha (H X[:, j] - c X[:, j]) + beta Y[:, j] for 1..8 columns,
// all four dtypes, any N.  With so few vectors the product is bound by ONE pass over H from HBM (the
// Lanczos runs of Alg. 6 coalesce 1 + n_vec = 5 vectors), so this is a streaming kernel:
// no tensor cores, no reuse of H, just wide coalesced loads and enough of them in flight.
//
// It uses that H is Hermitian (reading G9): (H x)[m] = sum_k conj(H[k, m]) x[k], and column m
// of the column-major H is contiguous -- every output row is a dot product over a contiguous stream,
// so no split-k atomics are needed.  A warp owns CM columns of H at a time and keeps CM x n partial sums
// per lane; every X value (read through L1, which all warps of an SM walk at the same pace) is reused
// for the CM columns, H itself is streamed past L1.
#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;
constexpr int CM = 4;             // columns of H (= output rows) per warp pass

template <typename T> struct Tr;
template <> struct Tr<float>   { using R = float; };
template <> struct Tr<double>  { using R = double; };
template <> struct Tr<float2>  { using R = float; };
template <> struct Tr<double2> { using R = double; };

// acc += conj(h) * x
__device__ __forceinline__ void cfma(float &a, float h, float x) { a = fmaf(h, x, a); }
__device__ __forceinline__ void cfma(double &a, double h, double x) { a = fma(h, x, a); }
__device__ __forceinline__ void cfma(float2 &a, float2 h, float2 x) {
    a.x = fmaf(h.x, x.x, a.x); a.x = fmaf(h.y, x.y, a.x);
    a.y = fmaf(h.x, x.y, a.y); a.y = fmaf(-h.y, x.x, a.y);
}
__device__ __forceinline__ void cfma(double2 &a, double2 h, double2 x) {
    a.x = fma(h.x, x.x, a.x); a.x = fma(h.y, x.y, a.x);
    a.y = fma(h.x, x.y, a.y); a.y = fma(-h.y, x.x, a.y);
}
__device__ __forceinline__ float zero(float) { return 0.f; }
__device__ __forceinline__ double zero(double) { return 0.0; }
__device__ __forceinline__ float2 zero(float2) { return make_float2(0.f, 0.f); }
__device__ __forceinline__ double2 zero(double2) { return make_double2(0.0, 0.0); }
__device__ __forceinline__ float shfl(float v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }
__device__ __forceinline__ double shfl(double v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }
__device__ __forceinline__ float2 shfl(float2 v, int o) { return make_float2(shfl(v.x, o), shfl(v.y, o)); }
__device__ __forceinline__ double2 shfl(double2 v, int o) { return make_double2(shfl(v.x, o), shfl(v.y, o)); }
__device__ __forceinline__ float add(float a, float b) { return a + b; }
__device__ __forceinline__ double add(double a, double b) { return a + b; }
__device__ __forceinline__ float2 add(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }

template <typename T, typename R>
__device__ __forceinline__ T epilogue(T acc, T x, T yold, R alpha, R beta, R c, int use_beta);
template <> __device__ __forceinline__ float epilogue(float acc, float x, float yold, float alpha, float beta, float c, int ub) {
    float y = alpha * (acc - c * x); return ub ? fmaf(beta, yold, y) : y;
}
template <> __device__ __forceinline__ double epilogue(double acc, double x, double yold, double alpha, double beta, double c, int ub) {
    double y = alpha * (acc - c * x); return ub ? fma(beta, yold, y) : y;
}
template <> __device__ __forceinline__ float2 epilogue(float2 acc, float2 x, float2 yold, float alpha, float beta, float c, int ub) {
    float2 y = make_float2(alpha * (acc.x - c * x.x), alpha * (acc.y - c * x.y));
    if (ub) { y.x = fmaf(beta, yold.x, y.x); y.y = fmaf(beta, yold.y, y.y); }
    return y;
}
template <> __device__ __forceinline__ double2 epilogue(double2 acc, double2 x, double2 yold, double alpha, double beta, double c, int ub) {
    double2 y = make_double2(alpha * (acc.x - c * x.x), alpha * (acc.y - c * x.y));
    if (ub) { y.x = fma(beta, yold.x, y.x); y.y = fma(beta, yold.y, y.y); }
    return y;
}

// VEC = elements of T per 16-byte load (1 = element-wise loads: any N and alignment).
template <typename T, int NV, int VEC>
__global__ void __launch_bounds__(kThreads) step_skinny_kernel(const T *__restrict__ H, const T *__restrict__ X,
                                                                T *__restrict__ Y, int64_t N, int n,
                                                                typename Tr<T>::R alpha, typename Tr<T>::R beta,
                                                                typename Tr<T>::R c, const double *__restrict__ c_col,
                                                                int use_beta) {
    using R = typename Tr<T>::R;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t m_base = ((int64_t)blockIdx.x * kWarps + warp) * CM;

    T acc[CM][NV];
#pragma unroll
    for (int cidx = 0; cidx < CM; ++cidx)
#pragma unroll
        for (int j = 0; j < NV; ++j) acc[cidx][j] = zero(T());
    const T *hcol[CM];
#pragma unroll
    for (int cidx = 0; cidx < CM; ++cidx) hcol[cidx] = H + min(m_base + cidx, N - 1) * N;   // clamp: loads stay legal

    // Two k-blocks per iteration: 2 * CM independent 16-byte loads of H in flight per lane.  H is
    // streamed past L1 (read once), X goes through L1 (every warp of the SM walks it at the same pace).
    constexpr int STEP = 32 * VEC;
    for (int64_t k = (int64_t)lane * VEC; k < N; k += 2 * STEP) {
        const bool second = k + STEP < N;
        T h[2][CM][VEC];
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int cidx = 0; cidx < CM; ++cidx) {
                const T *src = hcol[cidx] + k + (u ? (second ? STEP : 0) : 0);
                if (VEC == 1) {
                    h[u][cidx][0] = __ldcs(src);
                } else {   // one 16-byte load; N % VEC == 0, so a block is never entered half-way
                    const int4 raw = __ldcs(reinterpret_cast<const int4 *>(src));
                    *reinterpret_cast<int4 *>(&h[u][cidx][0]) = raw;
                }
            }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (u == 1 && !second) break;
#pragma unroll
            for (int v = 0; v < VEC; ++v)
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    const T xv = j < n ? __ldg(X + (int64_t)j * N + k + u * STEP + v) : zero(T());
#pragma unroll
                    for (int cidx = 0; cidx < CM; ++cidx) cfma(acc[cidx][j], h[u][cidx][v], xv);
                }
        }
    }

#pragma unroll
    for (int cidx = 0; cidx < CM; ++cidx)
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            T v = acc[cidx][j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v = add(v, shfl(v, o));
            acc[cidx][j] = v;
        }
    // lane (cidx * NV + j) writes output (row m_base + cidx, column j)
#pragma unroll
    for (int cidx = 0; cidx < CM; ++cidx)
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            if (lane == cidx * NV + j) {
                const int64_t m = m_base + cidx;
                if (m < N && j < n) {
                    const int64_t off = (int64_t)j * N + m;
                    const R cc = c_col ? (R)c_col[j] : c;
                    Y[off] = epilogue<T, R>(acc[cidx][j], __ldcg(X + off), use_beta ? __ldcg(Y + off) : zero(T()), alpha, beta, cc, use_beta);
                }
            }
        }
}

template <typename T, int NV>
cudaError_t launch_nv(const StepArgs &a, cudaStream_t stream) {
    using R = typename Tr<T>::R;
    constexpr int VEC = 16 / (int)sizeof(T);
    const unsigned grid = (unsigned)((a.N + kWarps * CM - 1) / (kWarps * CM));
    const bool vec_ok = VEC > 1 && a.N % VEC == 0 && ((uintptr_t)a.H & 15) == 0;
    if (vec_ok)
        step_skinny_kernel<T, NV, VEC><<<grid, kThreads, 0, stream>>>((const T *)a.H, (const T *)a.X, (T *)a.Y, a.N,
                                                                       (int)a.n, (R)a.alpha, (R)a.beta, (R)a.c,
                                                                       a.c_col, a.use_beta);
    else
        step_skinny_kernel<T, NV, 1><<<grid, kThreads, 0, stream>>>((const T *)a.H, (const T *)a.X, (T *)a.Y, a.N,
                                                                     (int)a.n, (R)a.alpha, (R)a.beta, (R)a.c,
                                                                     a.c_col, a.use_beta);
    count_launch();
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_t(const StepArgs &a, cudaStream_t stream) {
    if (a.n <= 2) return launch_nv<T, 2>(a, stream);
    if (a.n <= 4) return launch_nv<T, 4>(a, stream);
    if (a.n <= 6) return launch_nv<T, 6>(a, stream);
    return launch_nv<T, 8>(a, stream);
}

}  // namespace

cudaError_t launch_step_skinny(chase_dtype_t dtype, const StepArgs &a, cudaStream_t stream) {
    if (a.n <= 0) return cudaSuccess;
    if (a.n > kSkinnyMaxCols) return cudaErrorInvalidValue;
    switch (dtype) {
        case CHASE_F32: return launch_t<float>(a, stream);
        case CHASE_F64: return launch_t<double>(a, stream);
        case CHASE_C64: return launch_t<float2>(a, stream);
        default: return launch_t<double2>(a, stream);
    }
}

}  // namespace chase

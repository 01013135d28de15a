// Tall-skinny step kernel, bulk-copy version:  Y[:, j] <- alpha (H X[:, j] - c X[:, j]) + beta Y[:, j]
// for 1..8 columns, all four dtypes, every N whose columns start on 16-byte boundaries.
//
// With so few vectors the product is bound by ONE pass over H from HBM (the Lanczos runs of Alg. 6
// coalesce 1 + n_vec = 5 vectors): roofline = measured HBM copy bandwidth, algorithmic
// bytes = N^2 * sizeof(element).  It uses that H is Hermitian (reading G9):
// (H x)[m] = sum_k conj(H[k, m]) x[k], and column m of the column-major H is contiguous, so every
// output row is a dot product over a contiguous stream -- no split-k, no atomics.
//
// Structure: persistent CTAs (one per SM); a CTA takes blocks of CB = 16 columns of H and streams them
// -- together with the matching piece of X -- through a ring of shared-memory stages filled by TMA: per
// stage ONE 2-D box of H (2 KB of k x 16 columns; long sequential DRAM bursts, ~2400 streams chip-wide
// instead of one per warp) and one of X, issued by a producer thread and completed on mbarriers.
// (One 1-D bulk copy per column was issue-bound: ~125 clk per cp.async.bulk from a single thread.)
// H and X are viewed as matrices of 8-byte words (k along the rows), so one view serves all four
// dtypes; rows and columns past the matrix are zero-filled by TMA and need no masks.
// Eight consumer warps each own 4 columns x half of a stage; an X value is loaded once from shared
// memory and reused for the 4 columns; 4 x NV partial sums per lane live in registers across the
// whole k range; shuffle + shared-memory reduction and the fused epilogue close a block while the
// producer already streams the next one.
#include <cuda.h>

#include <mutex>

#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kConsumerWarps = 8;
constexpr int kThreads = (kConsumerWarps + 1) * 32;
constexpr int CB = 16;                  // columns of H (= output rows) per block
constexpr int CW = 4;                   // columns per consumer warp
constexpr int KCB = 2048;               // bytes of one column per stage
constexpr int kSmemBudget = 200 * 1024;

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

__device__ __forceinline__ float epi(float acc, float x, float yold, float alpha, float beta, float c, int ub) {
    float y = alpha * (acc - c * x); return ub ? fmaf(beta, yold, y) : y;
}
__device__ __forceinline__ double epi(double acc, double x, double yold, double alpha, double beta, double c, int ub) {
    double y = alpha * (acc - c * x); return ub ? fma(beta, yold, y) : y;
}
__device__ __forceinline__ float2 epi(float2 acc, float2 x, float2 yold, float alpha, float beta, float c, int ub) {
    float2 y = make_float2(alpha * (acc.x - c * x.x), alpha * (acc.y - c * x.y));
    if (ub) { y.x = fmaf(beta, yold.x, y.x); y.y = fmaf(beta, yold.y, y.y); }
    return y;
}
__device__ __forceinline__ double2 epi(double2 acc, double2 x, double2 yold, double alpha, double beta, double c, int ub) {
    double2 y = make_double2(alpha * (acc.x - c * x.x), alpha * (acc.y - c * x.y));
    if (ub) { y.x = fma(beta, yold.x, y.x); y.y = fma(beta, yold.y, y.y); }
    return y;
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n.reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n}\n"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}

template <int NV>
struct Geo {
    static constexpr int STAGE_BYTES = (CB + NV) * KCB;
    static constexpr int STAGES = (kSmemBudget / STAGE_BYTES) < 6 ? (kSmemBudget / STAGE_BYTES) : 6;
    static constexpr int RED_BYTES = 2 * kConsumerWarps * 32 * 16;     // two parities x warps x (CW x NV <= 32) elements
    static constexpr int TOTAL = STAGES * STAGE_BYTES + RED_BYTES + 128 /*barriers*/ + 128 /*align*/;
};

template <typename T, int NV>
__global__ void __launch_bounds__(kThreads, 1)
step_stream_kernel(const __grid_constant__ CUtensorMap tmapH, const __grid_constant__ CUtensorMap tmapX,
                   const T *__restrict__ X, T *__restrict__ Y, int64_t N, int n,
                   typename Tr<T>::R alpha, typename Tr<T>::R beta, typename Tr<T>::R c,
                   const double *__restrict__ c_col, int use_beta, int nblocks) {
    using R = typename Tr<T>::R;
    using G = Geo<NV>;
    constexpr int VEC = 16 / (int)sizeof(T);          // elements per 16-byte vector
    constexpr int EPC = KCB / (int)sizeof(T);         // elements of one column per stage
    static_assert(CW * NV <= 32, "one lane per (column, vector) result");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    const uint32_t smem_base = smem_u32(smem);
    T *red = reinterpret_cast<T *>(smem + G::STAGES * G::STAGE_BYTES);
    const uint32_t bar_base = smem_base + G::STAGES * G::STAGE_BYTES + G::RED_BYTES;   // full[STAGES], empty[STAGES]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nchunks = (int)((N + EPC - 1) / EPC);

    if (threadIdx.x == 0) {
        for (int s = 0; s < G::STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (G::STAGES + s), kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kConsumerWarps) {
        // ------------------------------------------------------------ producer: one lane issues the bulk copies
        if (lane == 0) {
            uint32_t it = 0;
            for (int blk = blockIdx.x; blk < nblocks; blk += gridDim.x) {
                const int m0 = blk * CB;
                for (int kc = 0; kc < nchunks; ++kc, ++it) {
                    const uint32_t slot = it % G::STAGES;
                    if (it >= (uint32_t)G::STAGES) mbar_wait(bar_base + 8 * (G::STAGES + slot), ((it / G::STAGES) - 1) & 1);
                    const uint32_t full = bar_base + 8 * slot;
                    const uint32_t dst = smem_base + slot * G::STAGE_BYTES;
                    mbar_expect_tx(full, (uint32_t)((CB + n) * KCB));       // whole boxes: TMA zero-fills out of bounds
                    tma_load_2d(dst, &tmapH, full, kc * (KCB / 8), m0);      // {2 KB of k as 8-byte words, 16 columns of H}
                    tma_load_2d(dst + CB * KCB, &tmapX, full, kc * (KCB / 8), 0);   // {same k, the n vectors}
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    const int cg = warp & 3, kh = warp >> 2;          // column group, k half of the stage
    uint32_t it = 0;
    int parity = 0;
    for (int blk = blockIdx.x; blk < nblocks; blk += gridDim.x, parity ^= 1) {
        T acc[CW][NV];
#pragma unroll
        for (int cidx = 0; cidx < CW; ++cidx)
#pragma unroll
            for (int j = 0; j < NV; ++j) acc[cidx][j] = zero(T());

        for (int kc = 0; kc < nchunks; ++kc, ++it) {
            const uint32_t slot = it % G::STAGES;
            mbar_wait(bar_base + 8 * slot, (it / G::STAGES) & 1);
            const unsigned char *st = smem + slot * G::STAGE_BYTES;
#pragma unroll
            for (int u = 0; u < KCB / 2 / 512; ++u) {
                const int off = kh * (KCB / 2) + u * 512 + lane * 16;
                {                                     // (k past N and columns past N arrive as zeros)
                    T h[CW][VEC], x[NV][VEC];
#pragma unroll
                    for (int cidx = 0; cidx < CW; ++cidx)
                        *reinterpret_cast<int4 *>(&h[cidx][0]) =
                            *reinterpret_cast<const int4 *>(st + (cg * CW + cidx) * KCB + off);
#pragma unroll
                    for (int j = 0; j < NV; ++j) {
                        if (j < n) {
                            *reinterpret_cast<int4 *>(&x[j][0]) = *reinterpret_cast<const int4 *>(st + (CB + j) * KCB + off);
                        } else {
#pragma unroll
                            for (int v = 0; v < VEC; ++v) x[j][v] = zero(T());
                        }
                    }
#pragma unroll
                    for (int v = 0; v < VEC; ++v)
#pragma unroll
                        for (int j = 0; j < NV; ++j)
#pragma unroll
                            for (int cidx = 0; cidx < CW; ++cidx) cfma(acc[cidx][j], h[cidx][v], x[j][v]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_base + 8 * (G::STAGES + slot));
        }

        // lanes -> one total per (column, vector); lane cidx * NV + j keeps it
        T mine = zero(T());
#pragma unroll
        for (int cidx = 0; cidx < CW; ++cidx)
#pragma unroll
            for (int j = 0; j < NV; ++j) {
                T v = acc[cidx][j];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v = add(v, shfl(v, o));
                if (lane == cidx * NV + j) mine = v;
            }
        T *r = red + (size_t)parity * kConsumerWarps * 32;
        r[warp * 32 + lane] = mine;
        asm volatile("bar.sync 1, %0;" ::"n"(kConsumerWarps * 32) : "memory");
        if (kh == 0 && lane < CW * NV) {
            const int cidx = lane / NV, j = lane % NV;
            const int64_t m = (int64_t)blk * CB + cg * CW + cidx;
            if (m < N && j < n) {
                const T total = add(r[warp * 32 + lane], r[(warp + 4) * 32 + lane]);
                const int64_t off = (int64_t)j * N + m;
                const R cc = c_col ? (R)c_col[j] : c;
                Y[off] = epi(total, __ldcg(X + off), use_beta ? __ldcg(Y + off) : zero(T()), alpha, beta, cc, use_beta);   // L2 only: step_dmma.cu
            }
        }
        // `red` alternates between two halves, and a warp can only get one block ahead of the slowest
        // (the bar.sync above), so the half it writes next was read two barriers ago.
    }
}

using EncodeTiledFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                   const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                   CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                   CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    });
    return fn;
}
// A column-major matrix with `col_bytes` bytes per column (a multiple of 16) and `cols` columns, viewed as
// 8-byte words: box = {KCB / 8 words of k, box_cols columns}, no swizzle -> smem image [column][2 KB].
cudaError_t encode_words(CUtensorMap *map, const void *base, size_t col_bytes, int64_t cols, int box_cols) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return cudaErrorNotSupported;
    cuuint64_t dims[2] = {(cuuint64_t)(col_bytes / 8), (cuuint64_t)cols};
    cuuint64_t strides[1] = {(cuuint64_t)col_bytes};
    cuuint32_t box[2] = {(cuuint32_t)(KCB / 8), (cuuint32_t)box_cols};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <typename T, int NV>
cudaError_t launch_nv(const StepArgs &a, cudaStream_t stream) {
    using R = typename Tr<T>::R;
    using G = Geo<NV>;
    static cudaError_t attr_err = cudaFuncSetAttribute(step_stream_kernel<T, NV>,
                                                       cudaFuncAttributeMaxDynamicSharedMemorySize, G::TOTAL);
    if (attr_err != cudaSuccess) return attr_err;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        sms = 148;
    alignas(64) CUtensorMap mapH, mapX;
    cudaError_t e;
    if ((e = encode_words(&mapH, a.H, (size_t)a.N * sizeof(T), a.N, CB)) != cudaSuccess) return e;
    if ((e = encode_words(&mapX, a.X, (size_t)a.N * sizeof(T), a.n, (int)a.n)) != cudaSuccess) return e;
    const int nblocks = (int)((a.N + CB - 1) / CB);
    const int grid = nblocks < sms ? nblocks : sms;
    step_stream_kernel<T, NV><<<grid, kThreads, G::TOTAL, stream>>>(mapH, mapX, (const T *)a.X, (T *)a.Y, a.N,
                                                                     (int)a.n, (R)a.alpha, (R)a.beta, (R)a.c, a.c_col,
                                                                     a.use_beta, nblocks);
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

size_t elem_size(chase_dtype_t dtype) {
    return dtype == CHASE_F32 ? 4 : dtype == CHASE_C128 ? 16 : 8;
}

}  // namespace

bool stream_supported(chase_dtype_t dtype, const StepArgs &a) {
    const size_t w = elem_size(dtype);
    return a.n >= 1 && a.n <= kSkinnyMaxCols && a.N >= 64 && ((size_t)a.N * w) % 16 == 0 &&
           (((uintptr_t)a.H | (uintptr_t)a.X) & 15) == 0;
}

cudaError_t launch_step_stream(chase_dtype_t dtype, const StepArgs &a, cudaStream_t stream) {
    if (a.n <= 0) return cudaSuccess;
    if (!stream_supported(dtype, a)) return cudaErrorInvalidValue;
    switch (dtype) {
        case CHASE_F32: return launch_t<float>(a, stream);
        case CHASE_F64: return launch_t<double>(a, stream);
        case CHASE_C64: return launch_t<float2>(a, stream);
        default: return launch_t<double2>(a, stream);
    }
}

}  // namespace chase

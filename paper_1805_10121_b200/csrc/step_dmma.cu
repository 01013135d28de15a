// TMA + FP64 tensor-core (DMMA) step kernel for complex128 and float64.
//
//   Y[:, j] <- alpha * (H X[:, j] - c X[:, j]) + beta * Y[:, j]     (Alg. 4 l.4 / l.9; Eq. 7)
//
// One kernel per degree step, one pass over H.  Structure:
//   * 1 producer warp: one elected lane issues TMA (cp.async.bulk.tensor) loads of an H tile and
//     an X tile per k-slab into a kStages-deep shared-memory ring, completion on mbarriers.
//   * 8 consumer warps: fragments by LDS from the 128B-swizzled tiles, mma.sync m8n8k4 f64
//     (SASS DMMA.8x8x4; sm_100a has no tcgen05 kind::f64), accumulators in registers,
//     complex as 4 real products on interleaved data (one sign flip per H fragment).
//   * fused epilogue in registers: -c X, alpha scaling, + beta Y (Y updated in place).
//
// Shared-memory tiles are rows of 128 bytes (8 complex / 16 real elements), TMA SWIZZLE_128B:
//   A (H tile, M-major as stored): row index = mgroup * BK + k, the 128B hold 8 (16) consecutive
//       matrix rows; loaded by ONE 3-D TMA box {16 doubles, BK, BM/rows_per_128B} from the view
//       (m_in_group, k, m_group) of the column-major H.
//   B (X tile, K-major as stored): row index = kgroup * BN + n, the 128B hold 8 (16) consecutive k.
// The k index each MMA lane slot consumes is a free permutation; it is chosen so that every
// fragment load is bank-conflict free under the swizzle (complex: k = 8q + 2t + a; real:
// k = {0,10,4,14}[t] ^ a with 16-byte loads shared by two MMAs), identically for A and B.
#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <mutex>
#include <vector>

#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kConsumerWarps = 8;
constexpr int kThreads = (kConsumerWarps + 4) * 32;   // 2 consumer warpgroups + 1 producer warpgroup

template <bool CPLX>
struct Cfg;
template <>
struct Cfg<true> {   // complex128: CTA tile 128 x 64, warp tile 32 x 32 (4 x 2 warps)
    static constexpr int BM = 128, BN = 64, WM = 32, WN = 32, WARPS_M = 4;
    static constexpr int ROWS128 = 8;       // matrix rows (or k) per 128-byte smem row
    static constexpr int ESZ = 16;
    static constexpr int BK = 16;           // k elements per pipeline stage (48 KB / stage)
    static constexpr int STAGES = 4;
    static constexpr int GROUP_N = 16;      // raster group: 16 column tiles x ~9 row tiles per wave
};
template <>
struct Cfg<false> {  // float64: CTA tile 128 x 128, warp tile 64 x 32 (2 x 4 warps)
    static constexpr int BM = 128, BN = 128, WM = 64, WN = 32, WARPS_M = 2;
    static constexpr int ROWS128 = 16;
    static constexpr int ESZ = 8;
#ifndef F64_BK
#define F64_BK 32
#define F64_STAGES 3
#endif
    static constexpr int BK = F64_BK;       // 32: 64 KB / stage, same DMMA count per stage as complex
    static constexpr int STAGES = F64_STAGES;
    static constexpr int GROUP_N = 12;
};

template <bool CPLX>
struct Smem {
    static constexpr int A_BYTES = Cfg<CPLX>::BM * Cfg<CPLX>::BK * Cfg<CPLX>::ESZ;
    static constexpr int B_BYTES = Cfg<CPLX>::BN * Cfg<CPLX>::BK * Cfg<CPLX>::ESZ;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int TOTAL = Cfg<CPLX>::STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
};

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
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
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------- the kernel
constexpr int kMaxPeers = CHASE_MAX_RANKS - 1;
struct StepParams {
    const double *X;     // source iterate V_k, first ACTIVE column (ld = N elements)
    double *Y;           // destination (holds V_{k-1}, becomes V_{k+1}), first active column
    int64_t N;           // matrix order = length of k = leading dimension of X, Y
    int64_t M;           // rows of H this launch owns (N unless row-sharded); H tile rows are local
    int64_t row0;        // global index of local row 0 (rows of X, Y touched by the epilogue: row0 + local)
    int a_2d;            // H view: 0 = one 3-D box per stage (M % ROWS128 == 0), 1 = BM / ROWS128 2-D boxes (any M)
    int npeers;          // row-sharded runs: the new rows are also stored into each peer GPU's copy of Y
    double *peer_Y[kMaxPeers];   // peer-mapped pointers, already offset to the first active column
    int n;               // active columns
    int col0;            // first active column in the full buffer (TMA coordinate offset)
    int tiles_m;
    int tiles_wide;      // column tiles of the full width BN, covering columns [0, tiles_wide * BN)
    int tiles_narrow;    // column tiles of width narrow_w covering the remaining columns
    int narrow_w;        // multiple of 8 * WARPS_N, <= BN
    double alpha, beta, c;
    const double *c_col;   // optional per-column shift (device, indexed by active column); overrides c
    int use_beta;
};

// Grouped rasterisation: consecutive CTAs cover kGroupN column tiles x a run of row tiles, so the
// CTAs resident at one time share both H row panels and X column panels in L2.  kGroupN is chosen
// so that a wave of 148 CTAs is roughly square in BYTES (rows*BM ~ cols*BN), which minimises the
// DRAM traffic of 148 register-resident output tiles.
template <int kGroupN>
__device__ __forceinline__ void tile_coords(int t, int tiles_m, int tiles_n, int &tm, int &tn) {
    const int per_group = kGroupN * tiles_m;
    const int grp = t / per_group;
    const int first_n = grp * kGroupN;
    const int gn = min(kGroupN, tiles_n - first_n);
    const int r = t - grp * per_group;
    tm = r / gn;
    tn = first_n + r % gn;
}

// The k loop of one consumer warp.  FULL = every 8-column block of the warp is valid (the common
// case: no per-block test, so the compiler schedules loads and MMAs across blocks); otherwise only
// the first jmax blocks are computed (ragged / narrow tiles).
template <bool CPLX, bool FULL>
__device__ __forceinline__ void mainloop(double (&acc)[CPLX ? 2 : 1][Cfg<CPLX>::WM / 8][Cfg<CPLX>::WN / 8][2],
                                         const unsigned char *smem, uint32_t bar_base, int KT, int lane, int warp,
                                         int jmax) {
    using C = Cfg<CPLX>;
    using S = Smem<CPLX>;
    constexpr int BN = C::BN, BK = C::BK, STAGES = C::STAGES;
    constexpr int MB = C::WM / 8, NB = C::WN / 8;
    constexpr int WARPS_N = kConsumerWarps / C::WARPS_M;
    const int g = lane >> 2, t = lane & 3;
    const int wm = warp % C::WARPS_M, wn = warp / C::WARPS_M;

    // float64: lane-dependent byte offsets of the fragment loads, hoisted out of the k loop.
    // MMA a of a 16-k group consumes, in lane slot t, k = {0,10,4,14}[t] ^ a.  One 16-byte load of A
    // yields matrix rows 2g and 2g+1 (the lane's "row g" of an even and an odd 8-row block), one 16-byte
    // load of B yields k and k^1, i.e. the operands of MMAs a and a^1: 24 LDS.128 per 128 MMAs, every
    // one conflict-free under the swizzle (k bits (1,2) and (2,3) both take 4 distinct values over t).
    int real_a_off[4], real_b_off[2];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const int kl = (10 * (t & 1) + 4 * (t >> 1)) ^ a;
        real_a_off[a] = kl * 128 + ((g ^ (kl & 7)) << 4);
        if ((a & 1) == 0) real_b_off[a >> 1] = g * 128 + ((((kl >> 1) & 7) ^ g) << 4);
    }

    for (int kt = 0; kt < KT; ++kt) {
        const int s = kt % STAGES;
        mbar_wait(bar_base + 8 * s, (kt / STAGES) & 1);
        const unsigned char *sa = smem + s * S::STAGE_BYTES;
        const unsigned char *sb = sa + S::A_BYTES;

        if (CPLX) {
            // 128B row = 8 complex.  A row index = mg*BK + k (mg = 8-row group), chunk = m ^ (k&7).
            //                        B row index = kg*BN + n (kg = 8-k group),  chunk = (k&7) ^ (n&7).
#pragma unroll
            for (int kq = 0; kq < BK / 8; ++kq) {
#pragma unroll
                for (int a = 0; a < 2; ++a) {
                    const int k7 = 2 * t + a;            // k & 7 of this lane's slot
                    const int k = kq * 8 + k7;
                    double ar[MB], ai[MB], nai[MB];
#pragma unroll
                    for (int i = 0; i < MB; ++i) {
                        const int mg = wm * (C::WM / 8) + i;
                        const double2 v = *reinterpret_cast<const double2 *>(
                            sa + (mg * BK + k) * 128 + ((g ^ k7) << 4));
                        ar[i] = v.x; ai[i] = v.y; nai[i] = -v.y;
                    }
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        if (!FULL && j >= jmax) break;
                        const int n = (j * WARPS_N + wn) * 8 + g;
                        const double2 b = *reinterpret_cast<const double2 *>(
                            sb + (kq * BN + n) * 128 + ((k7 ^ g) << 4));
#pragma unroll
                        for (int i = 0; i < MB; ++i) {
                            dmma884(acc[0][i][j][0], acc[0][i][j][1], ar[i], b.x);    // Cr += Ar Br
                            dmma884(acc[0][i][j][0], acc[0][i][j][1], nai[i], b.y);   // Cr -= Ai Bi
                            dmma884(acc[1][i][j][0], acc[1][i][j][1], ar[i], b.y);    // Ci += Ar Bi
                            dmma884(acc[1][i][j][0], acc[1][i][j][1], ai[i], b.x);    // Ci += Ai Br
                        }
                    }
                }
            }
        } else {
            // 128B row = 16 doubles.  A row index = mg*BK + k (mg = 16-row group), chunk = (m>>1) ^ (k&7);
            //                         B row index = kg*BN + n (kg = 16-k group),   chunk = (k>>1) ^ (n&7).
#pragma unroll
            for (int kq = 0; kq < BK / 16; ++kq) {
#pragma unroll
                for (int ap = 0; ap < 2; ++ap) {          // MMAs a = 2 ap and 2 ap + 1 share their B loads
                    double2 b2[NB];
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        if (!FULL && j >= jmax) break;
                        b2[j] = *reinterpret_cast<const double2 *>(
                            sb + (kq * BN + (j * WARPS_N + wn) * 8) * 128 + real_b_off[ap]);
                    }
#pragma unroll
                    for (int a1 = 0; a1 < 2; ++a1) {
                        double af[MB];
#pragma unroll
                        for (int i = 0; i < MB; i += 2) {
                            const int mg = wm * (C::WM / 16) + (i >> 1);
                            const double2 v = *reinterpret_cast<const double2 *>(
                                sa + (mg * BK + kq * 16) * 128 + real_a_off[2 * ap + a1]);
                            af[i] = v.x;          // matrix row 2g     of the 16-row group
                            af[i + 1] = v.y;      // matrix row 2g + 1
                        }
#pragma unroll
                        for (int j = 0; j < NB; ++j) {
                            if (!FULL && j >= jmax) break;
                            const double b = a1 ? b2[j].y : b2[j].x;
#pragma unroll
                            for (int i = 0; i < MB; ++i) dmma884(acc[0][i][j][0], acc[0][i][j][1], af[i], b);
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + s));
    }

}

template <bool CPLX>
__global__ void __launch_bounds__(kThreads, 1)
step_dmma_kernel(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB,
                 const StepParams p) {
    using C = Cfg<CPLX>;
    using S = Smem<CPLX>;
    constexpr int BM = C::BM, BN = C::BN, BK = C::BK, STAGES = C::STAGES;
    constexpr int MB = C::WM / 8, NB = C::WN / 8;   // 8x8 MMA blocks per warp tile

    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // 1024B alignment for SWIZZLE_128B; offset arithmetic keeps the pointer in the shared space
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t bar_base = smem_base + STAGES * S::STAGE_BYTES;   // full[STAGES], empty[STAGES]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // Column tiling (DESIGN.md 6.1 "ragged and narrow tiles"): tiles_wide tiles of BN columns first,
    // then tiles_narrow tiles of narrow_w columns (launched last, so that the tail of the launch is
    // made of short CTAs).  A tile with `ncols_tile` valid columns only computes its first
    // ceil(ncols_tile / 8) 8-column MMA blocks; block nb belongs to warp column nb % WARPS_N, so the
    // remaining work stays balanced over the warps and the tile's time is ~ ceil(nblk / WARPS_N).
    int tile_m, tile_n, n0, ncols_tile;
    {
        const int wide_ctas = p.tiles_m * p.tiles_wide;
        if ((int)blockIdx.x < wide_ctas) {
            tile_coords<C::GROUP_N>(blockIdx.x, p.tiles_m, p.tiles_wide, tile_m, tile_n);
            n0 = tile_n * BN;
            ncols_tile = min(BN, p.n - n0);
        } else {
            tile_coords<C::GROUP_N>(blockIdx.x - wide_ctas, p.tiles_m, p.tiles_narrow, tile_m, tile_n);
            n0 = p.tiles_wide * BN + tile_n * p.narrow_w;
            ncols_tile = min(p.narrow_w, p.n - n0);
        }
    }
    const int m0 = tile_m * BM;
    const int nblk = (ncols_tile + 7) >> 3;
    const int KT = (int)((p.N + BK - 1) / BK);

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);                          // full: producer's expect_tx arrive
            mbar_init(bar_base + 8 * (STAGES + s), kConsumerWarps);  // empty: one arrive per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= kConsumerWarps) {
        // ------------------------------------------------------------ producer warpgroup
        // gives its registers to the consumers (setmaxnreg is per warpgroup); one lane issues TMA
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == kConsumerWarps && lane == 0) {
            for (int kt = 0; kt < KT; ++kt) {
                const int s = kt % STAGES;
                const uint32_t full = bar_base + 8 * s, empty = bar_base + 8 * (STAGES + s);
                if (kt >= STAGES) mbar_wait(empty, ((kt / STAGES) - 1) & 1);
                const uint32_t sa = smem_base + s * S::STAGE_BYTES, sb = sa + S::A_BYTES;
                mbar_expect_tx(full, S::STAGE_BYTES);
                const int k0 = kt * BK;
                if (!p.a_2d) {
                    // A: view (16 doubles, k, m_group); one box {16, BK, BM / ROWS128}
                    tma_load_3d(sa, &tmapA, full, 0, k0, m0 / C::ROWS128);
                } else {
                    // A: view (doubles along m, k); one box {16, BK} per 128-byte row group -- the same
                    // shared-memory image, rows past M zero-filled (any M, e.g. the paper's odd sizes)
#pragma unroll 4
                    for (int gI = 0; gI < BM / C::ROWS128; ++gI)
                        tma_load_2d(sa + gI * BK * 128, &tmapA, full, (m0 + gI * C::ROWS128) * (CPLX ? 2 : 1), k0);
                }
                // B: (doubles along k, column); boxes {16 doubles, BN}
                if (CPLX) {
                    tma_load_2d(sb, &tmapB, full, 2 * k0, p.col0 + n0);
                    tma_load_2d(sb + BN * 128, &tmapB, full, 2 * k0 + 16, p.col0 + n0);
                } else {
#pragma unroll
                    for (int kq = 0; kq < BK / 16; ++kq)
                        tma_load_2d(sb + kq * BN * 128, &tmapB, full, k0 + 16 * kq, p.col0 + n0);
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumer warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    const int g = lane >> 2, t = lane & 3;
    constexpr int WARPS_N = kConsumerWarps / C::WARPS_M;
    static_assert(WARPS_N * C::WN == BN, "warp grid must cover the CTA tile");
    const int wm = warp % C::WARPS_M, wn = warp / C::WARPS_M;
    const int jmax = (nblk - wn + WARPS_N - 1) / WARPS_N;    // this warp owns blocks nb = j * WARPS_N + wn, j < jmax

    double acc[CPLX ? 2 : 1][MB][NB][2];
#pragma unroll
    for (int q = 0; q < (CPLX ? 2 : 1); ++q)
#pragma unroll
        for (int i = 0; i < MB; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) acc[q][i][j][0] = acc[q][i][j][1] = 0.0;

    if (jmax == NB) mainloop<CPLX, true>(acc, smem, bar_base, KT, lane, warp, jmax);
    else mainloop<CPLX, false>(acc, smem, bar_base, KT, lane, warp, jmax);

    // ---------------------------------------------------------------- fused epilogue
    // accumulator fragment: row g, columns 2t and 2t+1 of each 8x8 block
    const double alpha = p.alpha, beta = p.beta;
    constexpr int NC = CPLX ? 2 : 1;
#pragma unroll
    for (int j = 0; j < NB; ++j) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int cl = (j * WARPS_N + wn) * 8 + 2 * t + e;     // column inside the tile
            if (cl >= ncols_tile) continue;
            const int col = n0 + cl;
            const double c = p.c_col ? p.c_col[col] : p.c;
#pragma unroll
            for (int i = 0; i < MB; ++i) {
                int row;
                if (CPLX) row = m0 + wm * C::WM + i * 8 + g;
                else row = m0 + wm * C::WM + (i >> 1) * 16 + 2 * g + (i & 1);
                if (row >= p.M) continue;
                const int64_t off = ((int64_t)col * p.N + p.row0 + row) * NC;
                if (CPLX) {
                    const double2 x = *reinterpret_cast<const double2 *>(p.X + off);
                    double2 y;
                    y.x = alpha * (acc[0][i][j][e] - c * x.x);
                    y.y = alpha * (acc[NC - 1][i][j][e] - c * x.y);
                    if (p.use_beta) {
                        const double2 o = *reinterpret_cast<const double2 *>(p.Y + off);
                        y.x = fma(beta, o.x, y.x);
                        y.y = fma(beta, o.y, y.y);
                    }
                    *reinterpret_cast<double2 *>(p.Y + off) = y;
                    for (int q = 0; q < p.npeers; ++q)      // fused all-gather: push the row block over NVLink
                        *reinterpret_cast<double2 *>(p.peer_Y[q] + off) = y;
                } else {
                    double y = alpha * (acc[0][i][j][e] - c * p.X[off]);
                    if (p.use_beta) y = fma(beta, p.Y[off], y);
                    p.Y[off] = y;
                    for (int q = 0; q < p.npeers; ++q) p.peer_Y[q][off] = y;
                }
            }
        }
    }
}

// ---------------------------------------------------------------- host side
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

int sm_count() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        sms = 148;
    return sms;
}

template <bool CPLX>
cudaError_t encode_maps(DmmaPlan *plan) {
    using C = Cfg<CPLX>;
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return cudaErrorNotSupported;
    const cuuint64_t N = (cuuint64_t)plan->N;
    plan->a_2d = plan->M % C::ROWS128 != 0;
    if (plan->a_2d) {   // A: H viewed as (doubles along m, k): 2-D, rows past M are out of bounds -> zero fill
        cuuint64_t dims[2] = {(cuuint64_t)plan->M * (CPLX ? 2 : 1), N};
        cuuint64_t strides[1] = {(cuuint64_t)plan->ldh * C::ESZ};
        cuuint32_t box[2] = {16, (cuuint32_t)C::BK};
        cuuint32_t estr[2] = {1, 1};
        CUresult r = enc((CUtensorMap *)plan->tmap_H, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)plan->H, dims,
                         strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    } else {   // A: H (M x N, ld = ldh) viewed as (16 doubles, k, m_group)
        const cuuint64_t M = (cuuint64_t)plan->M;
        cuuint64_t dims[3] = {16, N, M / C::ROWS128};
        cuuint64_t strides[2] = {(cuuint64_t)plan->ldh * C::ESZ, 128};
        cuuint32_t box[3] = {16, (cuuint32_t)C::BK, (cuuint32_t)(C::BM / C::ROWS128)};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = enc((CUtensorMap *)plan->tmap_H, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)plan->H, dims,
                         strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    for (int b = 0; b < 2; ++b) {   // B: a vector buffer viewed as (doubles along k, column)
        cuuint64_t dims[2] = {N * (CPLX ? 2 : 1), (cuuint64_t)plan->ncols};
        cuuint64_t strides[1] = {N * C::ESZ};
        cuuint32_t box[2] = {16, (cuuint32_t)C::BN};
        cuuint32_t estr[2] = {1, 1};
        CUresult r = enc((CUtensorMap *)plan->tmap_B[b], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, plan->buf[b], dims,
                         strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    return cudaSuccess;
}

// Time of one launch in units of a "quarter" tile (8 * WARPS_N columns x BM rows over all of k) on `sms`
// SMs, one CTA per SM, CTAs dispatched in blockIdx order to the SM that frees first: `wide` CTAs of
// `wide_cost` quarters, then `narrow` CTAs of `narrow_cost`.  SM loads are kept as (load, count) levels.
struct Level { double load; int count; };
void assign(std::vector<Level> &lv, int64_t T, double cost) {
    while (T > 0) {
        if (lv.size() == 1 && T >= lv[0].count) {          // whole rounds at once
            const int64_t rounds = T / lv[0].count;
            lv[0].load += (double)rounds * cost;
            T -= rounds * lv[0].count;
            continue;
        }
        const Level lo = lv.front();                          // levels are sorted by ascending load
        const int m = (int)std::min<int64_t>(lo.count, T);
        lv.front().count -= m;
        if (lv.front().count == 0) lv.erase(lv.begin());
        const double nl = lo.load + cost;
        size_t i = 0;
        while (i < lv.size() && lv[i].load < nl - 1e-9) ++i;
        if (i < lv.size() && std::fabs(lv[i].load - nl) <= 1e-9) lv[i].count += m;
        else lv.insert(lv.begin() + i, Level{nl, m});
        T -= m;
    }
}
double makespan(int sms, int64_t wide, double wide_cost, int64_t narrow, double narrow_cost) {
    std::vector<Level> lv{Level{0.0, sms}};
    assign(lv, wide, wide_cost);
    assign(lv, narrow, narrow_cost);
    return lv.back().load;
}

// Chooses the column tiling of one launch: `wide` tiles of BN columns, then tiles of `narrow_w` columns
// (a multiple of the quarter width Q = 8 * WARPS_N) over the rest, minimising the modelled makespan.
template <bool CPLX>
void choose_tiling(int64_t n, int tiles_m, int sms, int &tiles_wide, int &tiles_narrow, int &narrow_w) {
    using C = Cfg<CPLX>;
    constexpr int Q = 8 * (kConsumerWarps / C::WARPS_M);      // columns per quarter tile
    constexpr int QPT = C::BN / Q;                            // quarters per full tile (4)
    constexpr double kNarrowOverhead = 0.06;                  // per-CTA cost of a narrow tile beyond its quarters
    const int full_tiles = (int)(n / C::BN);
    double best = 1e300;
    tiles_wide = full_tiles; tiles_narrow = 0; narrow_w = C::BN;
    const int backs[4] = {0, 1, 2, full_tiles};                         // full tiles handed to the narrow region
    for (int bi = 0; bi < 4; ++bi) {
        const int back = backs[bi];
        if (back > full_tiles || (bi == 3 && back <= 2)) continue;
        const int wide = full_tiles - back;
        const int64_t rest = n - (int64_t)wide * C::BN;
        if (rest == 0) {
            const double t = makespan(sms, (int64_t)wide * tiles_m, QPT, 0, 0.0);
            if (t < best) { best = t; tiles_wide = wide; tiles_narrow = 0; narrow_w = C::BN; }
            continue;
        }
        for (int wq = 1; wq <= QPT; ++wq) {
            const int w = wq * Q;
            const int64_t nt = (rest + w - 1) / w;
            // cost of the narrow tiles: all but the last have wq quarters; model the last one the same
            const double t = makespan(sms, (int64_t)wide * tiles_m, QPT, nt * tiles_m, wq + kNarrowOverhead);
            // total work also matters when the launch is shorter than one wave: prefer fewer, wider tiles on ties
            if (t < best - 1e-9) { best = t; tiles_wide = wide; tiles_narrow = (int)nt; narrow_w = w; }
        }
    }
}

template <bool CPLX>
cudaError_t launch(const DmmaPlan *plan, int src, int64_t s, double alpha, double beta, double c, int use_beta,
                   cudaStream_t stream, const double *c_col) {
    using C = Cfg<CPLX>;
    static std::once_flag once;
    static cudaError_t attr_err = cudaSuccess;
    std::call_once(once, [] {
        attr_err = cudaFuncSetAttribute(step_dmma_kernel<CPLX>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        Smem<CPLX>::TOTAL);
    });
    if (attr_err != cudaSuccess) return attr_err;
    const int64_t n = plan->ncols - s;
    if (n <= 0) return cudaSuccess;
    StepParams p;
    const size_t col_doubles = (size_t)plan->N * (CPLX ? 2 : 1);
    p.X = (const double *)plan->buf[src] + (size_t)s * col_doubles;
    p.Y = (double *)plan->buf[src ^ 1] + (size_t)s * col_doubles;
    p.N = plan->N;
    p.M = plan->M;
    p.row0 = plan->row0;
    p.a_2d = plan->a_2d;
    p.npeers = plan->npeers;
    for (int q = 0; q < plan->npeers; ++q)
        p.peer_Y[q] = (double *)plan->peer_buf[src ^ 1][q] + (size_t)s * col_doubles;
    p.n = (int)n;
    p.col0 = (int)s;
    p.tiles_m = (int)((plan->M + C::BM - 1) / C::BM);
    choose_tiling<CPLX>(n, p.tiles_m, sm_count(), p.tiles_wide, p.tiles_narrow, p.narrow_w);
    p.alpha = alpha;
    p.beta = beta;
    p.c = c;
    p.c_col = c_col;
    p.use_beta = use_beta;
    const CUtensorMap *mA = (const CUtensorMap *)plan->tmap_H;
    const CUtensorMap *mB = (const CUtensorMap *)plan->tmap_B[src];
    step_dmma_kernel<CPLX><<<(unsigned)(p.tiles_m * (p.tiles_wide + p.tiles_narrow)), kThreads, Smem<CPLX>::TOTAL, stream>>>(*mA, *mB, p);
    count_launch();
    return cudaGetLastError();
}

}  // namespace

void dmma_plan_tiling(int64_t N, int64_t n, chase_dtype_t dtype, int sms, int32_t out[4]) {
    int tw = 0, tn = 0, nw = 0;
    const int tiles_m = (int)((N + 127) / 128);
    if (dtype == CHASE_C128) choose_tiling<true>(n, tiles_m, sms, tw, tn, nw);
    else choose_tiling<false>(n, tiles_m, sms, tw, tn, nw);
    out[0] = tiles_m; out[1] = tw; out[2] = tn; out[3] = nw;
}

bool dmma_supported(int64_t N, int64_t ncols, chase_dtype_t dtype) {
    if (ncols < 1 || N < 16 || N > (1 << 28) || ncols > (1 << 28)) return false;
    if (dtype == CHASE_C128) return true;           // column stride N * 16 bytes: always a TMA-legal stride
    if (dtype == CHASE_F64) return N % 2 == 0;      // TMA strides must be multiples of 16 bytes
    return false;
}

cudaError_t dmma_plan_create(DmmaPlan *plan, chase_dtype_t dtype, const void *H, int64_t N, void *V, void *W,
                             int64_t ncols) {
    return dmma_plan_create_rows(plan, dtype, H, N, 0, N, V, W, ncols);
}

cudaError_t dmma_plan_create_rows(DmmaPlan *plan, chase_dtype_t dtype, const void *H_loc, int64_t N, int64_t row0,
                                  int64_t nrows, void *V, void *W, int64_t ncols) {
    plan->dtype = dtype;
    plan->N = N;
    plan->M = nrows;
    plan->ldh = nrows;
    plan->row0 = row0;
    plan->npeers = 0;
    plan->ncols = ncols;
    plan->H = H_loc;
    plan->buf[0] = V;
    plan->buf[1] = W;
    return dtype == CHASE_C128 ? encode_maps<true>(plan) : encode_maps<false>(plan);
}

cudaError_t dmma_plan_create_panel(DmmaPlan *plan, chase_dtype_t dtype, const void *H_full, int64_t N, int64_t row0,
                                   int64_t nrows, void *V, void *W, int64_t ncols) {
    const size_t esz = dtype == CHASE_C128 ? 16 : 8;
    plan->dtype = dtype;
    plan->N = N;
    plan->M = nrows;
    plan->ldh = N;
    plan->row0 = row0;
    plan->npeers = 0;
    plan->ncols = ncols;
    plan->H = (const char *)H_full + (size_t)row0 * esz;
    plan->buf[0] = V;
    plan->buf[1] = W;
    return dtype == CHASE_C128 ? encode_maps<true>(plan) : encode_maps<false>(plan);
}

cudaError_t dmma_launch_step(const DmmaPlan *plan, int src, int64_t s, double alpha, double beta, double c,
                             int use_beta, cudaStream_t stream, const double *c_col) {
    return plan->dtype == CHASE_C128 ? launch<true>(plan, src, s, alpha, beta, c, use_beta, stream, c_col)
                                     : launch<false>(plan, src, s, alpha, beta, c, use_beta, stream, c_col);
}

}  // namespace chase

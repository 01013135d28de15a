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
//
// Work decomposition of one launch (DESIGN.md 6.1 "stream-K tail").  Default (lock-step): persistent CTAs, one
// per SM; CTA b owns the whole output tiles b, b + grid, ... of the first `dp_tiles` tiles (grouped raster), and
// the producers of all CTAs keep within a window of 64 k-slabs of each other through a soft barrier, so that
// they hit each other's H / X tiles in L2 (cfg 4: 153 instead of 325 GB of DRAM reads per step, 27 W less, same
// speed).  CHASE_DMMA_LOCKSTEP=0: one CTA per whole tile, dispatched to whichever SM frees first.
// In both modes `sk_ctas` CTAs then share the remaining
// tiles' k-slabs in equal-TIME contiguous ranges (stream-K): a CTA whose range ends inside a tile
// leaves its partial accumulators in the scratch buffer and raises a flag -- first thing, because it
// walks its range from the top down --, the CTA that holds the tile's last slab adds the partials of
// the lower-numbered CTAs and runs the fused epilogue.  A CTA only ever waits on CTAs with a smaller
// blockIdx, which were dispatched before it and parked their partial at the start of their life.
// Launched with programmatic stream serialisation: prologue and the first H loads of step k+1
// overlap the tail of step k (griddepcontrol).
#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <exception>
#include <functional>
#include <mutex>
#include <queue>
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
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kPartBytes = 128 * 1024;     // one partial accumulator tile: 256 threads x 64 doubles (both dtypes)

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
    int tiles_m, tiles_n;
    int ragged_last;     // raster variant (tile_coords)
    int bn_w;            // column tile width of this launch: a multiple of 8 * WARPS_N, <= BN
    int dp_tiles;        // tiles [0, dp_tiles) in raster order: whole tiles, tile r * gridDim.x + b belongs to CTA b
    int dp_rounds;       // data-parallel rounds per CTA
    int sk_first;        // first stream-K CTA: 0 (persistent CTAs: whole tiles first, then a stream-K range) or
                         // dp_tiles (one CTA per whole tile, dispatched first; the stream-K CTAs follow)
    int sk_ctas;         // CTAs [sk_first, sk_first + sk_ctas) share the k-slabs of tiles [dp_tiles, tiles_m * tiles_n)
    unsigned *sync_ctr;  // soft barrier of the producers during the data-parallel rounds (or null)
    unsigned sync_base;  // value of *sync_ctr before this launch
    uint32_t epoch;      // value the stream-K flags take in this launch
    unsigned char *sk_part;   // sk_ctas partial tiles of kPartBytes
    uint32_t *sk_flag;        // sk_ctas flags
    double alpha, beta, c;
    const double *c_col;   // optional per-column shift (device, indexed by active column); overrides c
    int use_beta;
    int sk_begin[kMaxSkCtas + 1];   // CTA g owns the slabs [sk_begin[g], sk_begin[g+1]) of the stream-K region,
                                    // slab s = k-slab (s % KT) of tile dp_tiles + s / KT
};

// Grouped rasterisation: consecutive tiles cover kGroupN column tiles x a run of row tiles, so the
// CTAs working at one time share both H row panels and X column panels in L2.  kGroupN is chosen
// so that a round of 148 tiles is roughly square in BYTES (rows*BM ~ cols*BN), which minimises the
// DRAM traffic of 148 register-resident output tiles.
// ragged_last (lock-step mode): the last tile column -- the only one that can be ragged, i.e. cheaper --
// comes after all the others, so that the whole-tile rounds consist of equal-cost tiles that can walk along
// k in step (with static ownership, interleaved cheap tiles would leave their owners idle at the barrier).
// Without lock-step the ragged tiles stay interleaved: their H panels are then shared with the neighbours in
// L2 and their bandwidth appetite (same H bytes for a quarter of the MMAs) is diluted among full tiles.
template <int kGroupN>
__host__ __device__ __forceinline__ void tile_coords(int t, int tiles_m, int tiles_n, int ragged_last, int &tm,
                                                     int &tn) {
    const int body_n = ragged_last ? tiles_n - 1 : tiles_n;
    const int body = body_n * tiles_m;
    if (t >= body) {
        tm = t - body;
        tn = body_n;
        return;
    }
    const int per_group = kGroupN * tiles_m;
    const int grp = t / per_group;
    const int first_n = grp * kGroupN;
    const int gn = (body_n - first_n) < kGroupN ? (body_n - first_n) : kGroupN;
    const int r = t - grp * per_group;
    tm = r / gn;
    tn = first_n + r % gn;
}

// The k loop of one consumer warp over `len` slabs, ring position `it` onwards.  FULL = every 8-column
// block of the warp is valid (the common case: no per-block test, so the compiler schedules loads and
// MMAs across blocks); otherwise only the first jmax blocks are computed (ragged / narrow tiles).
template <bool CPLX, bool FULL>
__device__ __forceinline__ void mainloop(double (&acc)[CPLX ? 2 : 1][Cfg<CPLX>::WM / 8][Cfg<CPLX>::WN / 8][2],
                                         const unsigned char *smem, uint32_t bar_base, uint32_t it, int len, int lane,
                                         int warp, int jmax) {
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

    uint32_t s = it % STAGES, ph = (it / STAGES) & 1;
    for (int kt = 0; kt < len; ++kt) {
        mbar_wait(bar_base + 8 * s, ph);
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
        if (++s == STAGES) { s = 0; ph ^= 1; }
    }
}

// One unit of a CTA's work: k-slabs [k0, k1) of output tile `tile` (raster index).
struct Segment {
    int tile, k0, k1;
};
// Iterator over the segments of this CTA: first its whole tiles (one per data-parallel round), then its
// stream-K range.  The stream-K range [s_begin, s_end) is walked from the TOP DOWN: the head of the last tile
// it touches comes first -- it is parked at once for the higher-numbered CTA that holds that tile's tail --
// and the tail of the first tile comes last, when the partial sums of the lower-numbered CTAs that hold
// its head have long been parked.  (Bottom-up, every CTA would wait for the END of its predecessor.)
struct WorkIter {
    int round, s_begin, s_end;
};
__device__ __forceinline__ WorkIter work_begin(const StepParams &p) {
    WorkIter w;
    w.round = 0;
    w.s_begin = w.s_end = 0;
    const int g = (int)blockIdx.x - p.sk_first;
    if (g >= 0 && g < p.sk_ctas) { w.s_begin = p.sk_begin[g]; w.s_end = p.sk_begin[g + 1]; }
    return w;
}
// false when the CTA's work is exhausted; `dp_round` = the round of a whole-tile segment, -1 for stream-K
__device__ __forceinline__ bool next_segment(const StepParams &p, int KT, WorkIter &w, Segment &seg, int &dp_round) {
    while (w.round < p.dp_rounds) {
        const int t = w.round * (int)gridDim.x + (int)blockIdx.x;
        dp_round = w.round++;
        if (t < p.dp_tiles) {
            seg.tile = t; seg.k0 = 0; seg.k1 = KT;
            return true;
        }
    }
    dp_round = -1;
    if (w.s_end <= w.s_begin) return false;
    const int tr = (w.s_end - 1) / KT;
    const int tile_first = tr * KT;
    seg.tile = p.dp_tiles + tr;
    seg.k1 = w.s_end - tile_first;
    seg.k0 = max(w.s_begin, tile_first) - tile_first;
    w.s_end = tile_first + seg.k0;
    return true;
}

// Soft barrier between the TMA producers of all CTAs (a performance hint, never needed for correctness):
// arrive on a global counter, then poll until `target` arrivals for a bounded time.  Returns false when
// the wait timed out; the caller then stops polling but keeps arriving, so the counts stay consistent.
constexpr int kSyncSlabs = 32;
__device__ __forceinline__ bool soft_grid_sync(unsigned *ctr, unsigned target, bool poll) {
    atomicAdd(ctr, 1u);
    if (!poll) return false;
    for (int i = 0; i < 4096; ++i) {
        unsigned v;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        if ((int)(v - target) >= 0) return true;
        __nanosleep(32);
    }
    return false;
}

template <bool CPLX>
__global__ void __launch_bounds__(kThreads, 1)
step_dmma_kernel(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB,
                 const __grid_constant__ StepParams p) {
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
    const int KT = (int)((p.N + BK - 1) / BK);
    const int sk_g = (int)blockIdx.x - p.sk_first;    // index among the stream-K CTAs
    WorkIter work = work_begin(p);

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);                          // full: producer's expect_tx arrive
            mbar_init(bar_base + 8 * (STAGES + s), kConsumerWarps);  // empty: one arrive per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // Programmatic dependent launch: the next step's CTAs may be dispatched as soon as every CTA of this
    // launch has got here (they then run their prologue and first H loads while this launch drains).
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    if (warp >= kConsumerWarps) {
        // ------------------------------------------------------------ producer warpgroup
        // gives its registers to the consumers (setmaxnreg is per warpgroup); one lane issues TMA
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == kConsumerWarps && lane == 0) {
            // H is never written, so its first tiles may be fetched before the previous launch (which
            // produces this step's X) has finished; X loads and everything after wait for it.
            bool dep_waited = false, sync_poll = true;
            const int spt = (KT + kSyncSlabs - 1) / kSyncSlabs;      // soft-barrier points per whole tile
            uint32_t it = 0;
            Segment seg;
            int dp_round;
            while (next_segment(p, KT, work, seg, dp_round)) {
                int tile_m, tile_n;
                tile_coords<C::GROUP_N>(seg.tile, p.tiles_m, p.tiles_n, p.ragged_last, tile_m, tile_n);
                const int m0 = tile_m * BM, n0 = tile_n * p.bn_w;
                // data-parallel rounds: every kSyncSlabs slabs a producer checks in and waits (bounded) until ALL
                // producers have passed the PREVIOUS check-in: nobody runs more than 2 * kSyncSlabs slabs ahead
                // of the slowest CTA -- the union stream of that window (~35 MB) stays in L2 -- and nobody stalls
                // unless it is a full window ahead.  (Meeting at every check-in cost 0.7 % of cfg 4.)
                auto sync_point = [&](int kt) {
                    if (dp_round >= 0 && p.sync_ctr && kt % kSyncSlabs == 0) {
                        const unsigned q = (unsigned)(dp_round * spt + kt / kSyncSlabs);
                        sync_poll = soft_grid_sync(p.sync_ctr, p.sync_base + gridDim.x * q, sync_poll);
                    }
                };
                auto load_A = [&](uint32_t slot, int kt) {
                    const uint32_t full = bar_base + 8 * slot;
                    const uint32_t sa = smem_base + slot * S::STAGE_BYTES;
                    const int k0 = kt * BK;
                    mbar_expect_tx(full, S::STAGE_BYTES);
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
                };
                auto load_B = [&](uint32_t slot, int kt) {
                    const uint32_t full = bar_base + 8 * slot;
                    const uint32_t sb = smem_base + slot * S::STAGE_BYTES + S::A_BYTES;
                    const int k0 = kt * BK;
                    // B: (doubles along k, column); boxes {16 doubles, BN}
                    if (CPLX) {
                        tma_load_2d(sb, &tmapB, full, 2 * k0, p.col0 + n0);
                        tma_load_2d(sb + BN * 128, &tmapB, full, 2 * k0 + 16, p.col0 + n0);
                    } else {
#pragma unroll
                        for (int kq = 0; kq < BK / 16; ++kq)
                            tma_load_2d(sb + kq * BN * 128, &tmapB, full, k0 + 16 * kq, p.col0 + n0);
                    }
                };
                int kt = seg.k0;
                if (!dep_waited) {
                    const int pre = min(STAGES, seg.k1 - seg.k0);       // ring is empty: no empty-wait needed
                    for (int i = 0; i < pre; ++i) { sync_point(kt + i); load_A(i, kt + i); }
                    asm volatile("griddepcontrol.wait;" ::: "memory");
                    for (int i = 0; i < pre; ++i) load_B(i, kt + i);
                    dep_waited = true;
                    kt += pre;
                    it += pre;
                }
                for (; kt < seg.k1; ++kt, ++it) {
                    sync_point(kt);
                    const uint32_t slot = it % STAGES;
                    if (it >= (uint32_t)STAGES) mbar_wait(bar_base + 8 * (STAGES + slot), ((it / STAGES) - 1) & 1);
                    load_A(slot, kt);
                    load_B(slot, kt);
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumer warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    asm volatile("griddepcontrol.wait;" ::: "memory");     // X, Y and the stream-K scratch belong to the previous launch until here
    const int g = lane >> 2, t = lane & 3;
    constexpr int WARPS_N = kConsumerWarps / C::WARPS_M;
    static_assert(WARPS_N * C::WN == BN, "warp grid must cover the CTA tile");
    static_assert((CPLX ? 2 : 1) * MB * NB * 16 * kConsumerThreads == kPartBytes, "partial tile size");
    const int wm = warp % C::WARPS_M, wn = warp / C::WARPS_M;
    const int tid = threadIdx.x;                           // 0 .. kConsumerThreads-1 here
    constexpr int NC = CPLX ? 2 : 1;

    uint32_t it = 0;
    Segment seg;
    int dp_round;
    while (next_segment(p, KT, work, seg, dp_round)) {
        // Column tiling: tiles of bn_w columns; a tile with `ncols_tile` valid columns only
        // computes its first ceil(ncols_tile / 8) 8-column MMA blocks; block nb belongs to warp column
        // nb % WARPS_N, so the work stays balanced over the warps and the tile's time is ~ ceil(nblk / WARPS_N).
        int tile_m, tile_n;
        tile_coords<C::GROUP_N>(seg.tile, p.tiles_m, p.tiles_n, p.ragged_last, tile_m, tile_n);
        const int m0 = tile_m * BM, n0 = tile_n * p.bn_w;
        const int ncols_tile = min(p.bn_w, p.n - n0);
        const int nblk = (ncols_tile + 7) >> 3;
        const int jmax = (nblk - wn + WARPS_N - 1) / WARPS_N;    // this warp owns blocks nb = j * WARPS_N + wn, j < jmax

        double acc[NC][MB][NB][2];
#pragma unroll
        for (int q = 0; q < NC; ++q)
#pragma unroll
            for (int i = 0; i < MB; ++i)
#pragma unroll
                for (int j = 0; j < NB; ++j) acc[q][i][j][0] = acc[q][i][j][1] = 0.0;

        const int len = seg.k1 - seg.k0;
        if (jmax == NB) mainloop<CPLX, true>(acc, smem, bar_base, it, len, lane, warp, jmax);
        else mainloop<CPLX, false>(acc, smem, bar_base, it, len, lane, warp, jmax);
        it += (uint32_t)len;

        if (seg.k1 < KT) {
            // ---- stream-K: this CTA stops inside the tile: park the partial sums, raise the flag
            unsigned char *part = p.sk_part + (size_t)sk_g * kPartBytes;
#pragma unroll
            for (int q = 0; q < NC; ++q)
#pragma unroll
                for (int i = 0; i < MB; ++i)
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        if (j >= jmax) break;
                        const int pr = (q * MB + i) * NB + j;
                        *reinterpret_cast<double2 *>(part + ((size_t)pr * kConsumerThreads + tid) * 16) =
                            make_double2(acc[q][i][j][0], acc[q][i][j][1]);
                    }
            __threadfence();
            asm volatile("bar.sync 1, %0;" ::"n"(kConsumerThreads) : "memory");
            if (tid == 0)
                asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p.sk_flag + sk_g), "r"(p.epoch) : "memory");
            continue;
        }
        if (seg.k0 > 0) {
            // ---- stream-K: this CTA finishes a tile that lower-numbered CTAs started: add their partials.
            // Contributors are the CTAs [c_lo, sk_g) with a non-empty range (CTA c_lo holds the tile's slab 0).
            const int tile_first = (seg.tile - p.dp_tiles) * KT;       // slab index of the tile's k-slab 0
            int c_lo = sk_g;
            while (c_lo > 0) {
                --c_lo;
                if (p.sk_begin[c_lo] <= tile_first) break;
            }
            // all flags at once: thread t polls contributor c_lo + t (at most kMaxSkCtas < kConsumerThreads of them)
            {
                const int c = c_lo + tid;
                if (c < sk_g && p.sk_begin[c + 1] > p.sk_begin[c]) {
                    uint32_t v;
                    unsigned long long t0 = 0;
                    for (uint32_t spins = 0;; ++spins) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p.sk_flag + c) : "memory");
                        if (v == p.epoch) break;
                        if ((spins & 1023u) == 1023u) {            // a lost partial must not pass silently:
                            unsigned long long now;                // trap after 20 s without the flag
                            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
                            if (t0 == 0) t0 = now;
                            else if (now - t0 > 20000000000ull) __trap();
                        }
                        __nanosleep(32);
                    }
                }
                __syncwarp();
                asm volatile("bar.sync 1, %0;" ::"n"(kConsumerThreads) : "memory");
            }
            if (sk_g - c_lo >= 3) {
                // many small partials (a tile split among many CTAs: tiny launches): keep the loads of four
                // contributors in flight at a time, one 8-column block after the other
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    if (j >= jmax) break;
                    for (int c = c_lo; c < sk_g; c += 4) {
                        double2 v[4][NC][MB];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const int cc = c + u;
                            const bool ok = cc < sk_g && p.sk_begin[cc + 1] > p.sk_begin[cc];
                            const unsigned char *part = p.sk_part + (size_t)(ok ? cc : c) * kPartBytes;
#pragma unroll
                            for (int q = 0; q < NC; ++q)
#pragma unroll
                                for (int i = 0; i < MB; ++i) {
                                    const int pr = (q * MB + i) * NB + j;
                                    v[u][q][i] = ok ? __ldcg(reinterpret_cast<const double2 *>(
                                                          part + ((size_t)pr * kConsumerThreads + tid) * 16))
                                                    : make_double2(0.0, 0.0);
                                }
                        }
#pragma unroll
                        for (int u = 0; u < 4; ++u)
#pragma unroll
                            for (int q = 0; q < NC; ++q)
#pragma unroll
                                for (int i = 0; i < MB; ++i) {
                                    acc[q][i][j][0] += v[u][q][i].x;
                                    acc[q][i][j][1] += v[u][q][i].y;
                                }
                    }
                }
            } else {
                for (int c = sk_g - 1; c >= c_lo; --c) {
                    if (p.sk_begin[c + 1] <= p.sk_begin[c]) continue;      // (an empty CTA parks nothing)
                    const unsigned char *part = p.sk_part + (size_t)c * kPartBytes;
#pragma unroll
                    for (int q = 0; q < NC; ++q)
#pragma unroll
                        for (int i = 0; i < MB; ++i)
#pragma unroll
                            for (int j = 0; j < NB; ++j) {
                                if (j >= jmax) break;
                                const int pr = (q * MB + i) * NB + j;
                                const double2 v = __ldcg(reinterpret_cast<const double2 *>(
                                    part + ((size_t)pr * kConsumerThreads + tid) * 16));
                                acc[q][i][j][0] += v.x;
                                acc[q][i][j][1] += v.y;
                            }
                }
            }
        }

        // ---------------------------------------------------------------- fused epilogue
        // accumulator fragment: row g, columns 2t and 2t+1 of each 8x8 block.  Per 8-column block all loads of
        // X (and Y) are issued before the first store: Y may alias nothing the loads need, but the compiler cannot
        // know, and a load-store-load chain pays one L2 round trip per element (32 per tile: ~10 us, most of a
        // small launch).
        const double alpha = p.alpha, beta = p.beta;
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            if (j >= jmax) break;
            constexpr int EB = CPLX ? 2 : 1;       // columns of the fragment per batch (float64: 8 row blocks per column)
#pragma unroll
            for (int e0 = 0; e0 < 2; e0 += EB) {
            double2 xv[2][MB], ov[2][MB];
            double cc[2];
            bool colok[2];
#pragma unroll
            for (int e = e0; e < e0 + EB; ++e) {
                const int cl = (j * WARPS_N + wn) * 8 + 2 * t + e;     // column inside the tile
                colok[e] = cl < ncols_tile;
                const int col = n0 + cl;
                cc[e] = colok[e] ? (p.c_col ? p.c_col[col] : p.c) : 0.0;
#pragma unroll
                for (int i = 0; i < MB; ++i) {
                    int row;
                    if (CPLX) row = m0 + wm * C::WM + i * 8 + g;
                    else row = m0 + wm * C::WM + (i >> 1) * 16 + 2 * g + (i & 1);
                    const bool ok = colok[e] && row < p.M;
                    const int64_t off = ((int64_t)col * p.N + p.row0 + row) * NC;
                    xv[e][i] = make_double2(0.0, 0.0);
                    ov[e][i] = make_double2(0.0, 0.0);
                    if (ok) {
                        // ld.global.cg: the vector buffers are rewritten by OTHER SMs from one launch to the next, and
                        // the (non-coherent) L1 was seen to serve lines of an earlier iterate to these batched loads
                        // (rare 32 x 8 patches of V_{k-2} in place of V_k; bypassing L1 removes them)
                        if (CPLX) {
                            xv[e][i] = __ldcg(reinterpret_cast<const double2 *>(p.X + off));
                            if (p.use_beta) ov[e][i] = __ldcg(reinterpret_cast<const double2 *>(p.Y + off));
                        } else {
                            xv[e][i].x = __ldcg(p.X + off);
                            if (p.use_beta) ov[e][i].x = __ldcg(p.Y + off);
                        }
                    }
                }
            }
#pragma unroll
            for (int e = e0; e < e0 + EB; ++e) {
                const int cl = (j * WARPS_N + wn) * 8 + 2 * t + e;
                const int col = n0 + cl;
                const double c = cc[e];
#pragma unroll
                for (int i = 0; i < MB; ++i) {
                    int row;
                    if (CPLX) row = m0 + wm * C::WM + i * 8 + g;
                    else row = m0 + wm * C::WM + (i >> 1) * 16 + 2 * g + (i & 1);
                    if (!colok[e] || row >= p.M) continue;
                    const int64_t off = ((int64_t)col * p.N + p.row0 + row) * NC;
                    if (CPLX) {
                        double2 y;
                        y.x = alpha * (acc[0][i][j][e] - c * xv[e][i].x);
                        y.y = alpha * (acc[NC - 1][i][j][e] - c * xv[e][i].y);
                        if (p.use_beta) {
                            y.x = fma(beta, ov[e][i].x, y.x);
                            y.y = fma(beta, ov[e][i].y, y.y);
                        }
                        *reinterpret_cast<double2 *>(p.Y + off) = y;
                        for (int q = 0; q < p.npeers; ++q)      // fused all-gather: push the row block over NVLink
                            *reinterpret_cast<double2 *>(p.peer_Y[q] + off) = y;
                    } else {
                        double y = alpha * (acc[0][i][j][e] - c * xv[e][i].x);
                        if (p.use_beta) y = fma(beta, ov[e][i].x, y);
                        p.Y[off] = y;
                        for (int q = 0; q < p.npeers; ++q) p.peer_Y[q][off] = y;
                    }
                }
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
    static int cached = 0;                  // one device kind per process is assumed for the plan heuristics
    if (cached > 0) return cached;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        return 148;
    cached = sms;
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

// ---------------------------------------------------------------- the launch plan (host, no CUDA call)
// Cost unit: one "quarter slab" = the MMAs of one k-slab on 8 * WARPS_N columns x BM rows; a tile with v valid
// columns costs ceil(ceil(v / 8) / WARPS_N) quarters per slab (measured: DESIGN.md 6.1).
template <bool CPLX>
void make_plan(int64_t M, int64_t N, int64_t n, int sms, bool allow_sk, StepPlan &pl) {
    using C = Cfg<CPLX>;
    constexpr int WARPS_N = kConsumerWarps / C::WARPS_M;
    constexpr int Q = 8 * WARPS_N;                            // columns per quarter tile
    constexpr int QPT = C::BN / Q;                            // quarters per full tile (4)
    constexpr int kMinWork = 4;                               // quarter slabs a stream-K CTA should at least get
    const int KT = (int)((N + C::BK - 1) / C::BK);
    const int tiles_m = (int)((M + C::BM - 1) / C::BM);
    sms = std::max(1, std::min(sms, kMaxSkCtas));
    // Column tile width: the full BN unless that leaves so few tiles that a tile would be split among
    // more than ~6 stream-K CTAs (its finisher adds their partial tiles one after the other); then narrower.
    int w = C::BN;
    if (allow_sk) {
        const int cand[3] = {C::BN, 2 * Q, Q};
        for (int ci = 0; ci < 3; ++ci) {
            w = cand[ci];
            const int64_t T = (int64_t)tiles_m * ((n + w - 1) / w);
            if (T * 6 >= sms) break;
        }
    }
    const int tiles_n = (int)((n + w - 1) / w);
    const int64_t T = (int64_t)tiles_m * tiles_n;
    auto quarters_of_col_tile = [&](int tn) {
        const int v = (int)std::min<int64_t>(w, n - (int64_t)tn * w);
        const int nblk = (v + 7) / 8;
        return (nblk + WARPS_N - 1) / WARPS_N;
    };
    const int q_full = quarters_of_col_tile(0), q_last = quarters_of_col_tile(tiles_n - 1);
    static const bool lockstep_env = [] {          // default on; CHASE_DMMA_LOCKSTEP=0 selects one CTA per whole tile
        const char *env = std::getenv("CHASE_DMMA_LOCKSTEP");
        return !(env && env[0] == '0');
    }();
    // lock-step only pays (and only applies) when there are whole-tile rounds: same condition as D > 0 below
    const bool lockstep = lockstep_env && allow_sk && T >= 2 * (int64_t)sms;
    auto quarters_of_tile = [&](int64_t t) {
        int tm, tn;
        tile_coords<C::GROUP_N>((int)t, tiles_m, tiles_n, lockstep ? 1 : 0, tm, tn);
        return tn == tiles_n - 1 ? q_last : q_full;
    };
    pl.KT = KT; pl.tiles_m = tiles_m; pl.tiles_n = tiles_n; pl.bn_w = w; pl.ragged_last = lockstep ? 1 : 0;
    pl.dp_tiles = (int)T; pl.sk_ctas = 0; pl.sk_begin[0] = 0;
    pl.grid = (int)T; pl.dp_rounds = 1; pl.sk_first = 0;      // default: one CTA per tile
    (void)QPT;
    if (!allow_sk || T <= 0) return;

    // Data-parallel region: whole rounds of `sms` tiles, all but the last one-to-two rounds' worth of tiles.
    int64_t D = 0;
    if (T >= 2 * (int64_t)sms) D = (T / sms - 1) * sms;
    // Stream-K region: tiles [D, T); work in quarter slabs.  It must hold at least one round's worth of full
    // tiles, or the CTAs could not all be made to finish together (the cheap ragged tiles come last).
    double work = 0.0;
    for (int64_t t = D; t < T; ++t) work += (double)quarters_of_tile(t) * KT;
    while (D > 0 && work < (double)sms * q_full * KT) {
        for (int64_t t = D - sms; t < D; ++t) work += (double)quarters_of_tile(t) * KT;
        D -= sms;
    }
    // Time (quarter slabs) at which the SM that runs stream-K CTA g has finished its whole tiles.
    //   lock-step: CTA b owns the tiles b, b + sms, ... and continues with stream-K range b;
    //   default:   tiles go to whichever SM frees first (list scheduling in blockIdx order), and the g-th
    //              stream-K CTA, the (D + g)-th CTA of the grid, starts on the g-th SM to become free.
    std::vector<double> free_at((size_t)sms, 0.0);
    if (lockstep) {
        for (int64_t t = 0; t < D; ++t) free_at[(size_t)(t % sms)] += (double)quarters_of_tile(t) * KT;
    } else if (D > 0) {
        if (q_last == q_full) {                                               // all whole tiles cost the same
            std::fill(free_at.begin(), free_at.end(), (double)(D / sms) * q_full * KT);
        } else {
            std::priority_queue<double, std::vector<double>, std::greater<double>> heap;
            for (int i = 0; i < sms; ++i) heap.push(0.0);
            for (int64_t t = 0; t < D; ++t) {
                const double f = heap.top();
                heap.pop();
                heap.push(f + (double)quarters_of_tile(t) * KT);
            }
            for (int i = 0; i < sms; ++i) { free_at[(size_t)i] = heap.top(); heap.pop(); }
        }
    }
    int G = sms;
    if (work < (double)G * kMinWork) G = (int)std::max(1.0, work / kMinWork);
    const int64_t R = T - D;
    if (R < G && (int64_t)KT * q_full < 32 * (int64_t)(G / R)) {
        // tiny launch: align the split with the tile boundaries (every CTA inside ONE tile)
        G = (int)(R * (G / R));
    }
    if (D == 0 && G <= 1) return;                              // too little work to split: one CTA per tile
    if (D == 0 && R == G && q_last == q_full) return;          // one whole tile per CTA already: nothing to balance
    if (D > 0) G = sms;
    // Water-filling: finish time F with sum_b max(0, F - free_at[b]) = work over the CTAs 0 .. G-1.
    double F = 0.0;
    {
        std::vector<double> f(free_at.begin(), free_at.begin() + G);
        std::sort(f.begin(), f.end());
        double acc_f = 0.0;
        for (int i = 0; i < G; ++i) {                         // ascending: try using the i + 1 earliest CTAs
            acc_f += f[(size_t)i];
            F = (work + acc_f) / (i + 1);
            if (i + 1 == G || F <= f[(size_t)i + 1]) break;
        }
    }
    pl.dp_tiles = (int)D;
    pl.sk_ctas = G;
    if (lockstep || D == 0) {
        pl.grid = D > 0 ? sms : G;
        pl.dp_rounds = (int)(D / sms);
        pl.sk_first = 0;
    } else {
        pl.grid = (int)D + G;
        pl.dp_rounds = 1;
        pl.sk_first = (int)D;
    }
    // Boundaries: walk the region's tiles, cutting where the cumulative cost reaches each CTA's share.
    const int64_t total_slabs = R * KT;
    double target = 0.0, cum = 0.0;            // cost before the current tile
    int64_t t = D;
    int qt = quarters_of_tile(t);
    pl.sk_begin[0] = 0;
    for (int gI = 0; gI < G; ++gI) {
        target += std::max(0.0, F - free_at[(size_t)gI]);
        // advance to the tile containing `target`
        while (t < T - 1 && cum + (double)qt * KT <= target) {
            cum += (double)qt * KT;
            ++t;
            qt = quarters_of_tile(t);
        }
        int64_t slab = (t - D) * KT + (int64_t)std::llround((target - cum) / qt);
        slab = std::max<int64_t>(slab, pl.sk_begin[gI]);
        slab = std::min<int64_t>(slab, total_slabs);
        pl.sk_begin[gI + 1] = (int)slab;
    }
    pl.sk_begin[G] = (int)total_slabs;
}

// Stream-K scratch for launches that bring none (chase_hemm, chase_residuals, the row-sharded path): a small
// per-process cache of device buffers.  A buffer is handed to one launch at a time: it becomes free again
// when the event recorded behind that launch has completed, so launches on different streams never share
// one, and nothing is allocated or freed in steady state.  (Not meant for stream capture: a captured event
// record does not mark real completion.  chase_filter_ws uses the caller's workspace and is capturable.)
struct SkSlot {
    void *ptr;
    cudaEvent_t ev;
    int dev;
    bool held;          // between acquire and release on some host thread
    uint32_t epoch;
    unsigned sync_count;   // arrivals the soft-barrier counter in this buffer has seen so far
};
std::mutex g_sk_mu;
std::vector<SkSlot> g_sk_slots;

// `stream`: the stream the launch that takes the buffer goes to.  A fresh buffer's flag block is zeroed ON THAT
// STREAM: a plain cudaMemset runs on the legacy default stream, which a non-blocking stream (chase_filter_host's,
// any torch side stream) does not wait for, so the kernel could otherwise meet uninitialised flags.
cudaError_t sk_cache_acquire(int *slot, void **ptr, uint32_t *epoch, unsigned *sync_base, unsigned sync_arrivals,
                             cudaStream_t stream) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(g_sk_mu);
    for (size_t i = 0; i < g_sk_slots.size(); ++i) {
        SkSlot &sl = g_sk_slots[i];
        if (sl.dev != dev || sl.held) continue;
        const cudaError_t q = cudaEventQuery(sl.ev);
        if (q == cudaErrorNotReady) continue;
        if (q != cudaSuccess) return q;
        sl.held = true;
        *slot = (int)i; *ptr = sl.ptr; *epoch = ++sl.epoch;
        *sync_base = sl.sync_count;
        sl.sync_count += sync_arrivals;
        return cudaSuccess;
    }
    SkSlot sl{};
    sl.dev = dev; sl.held = true; sl.epoch = 1; sl.sync_count = sync_arrivals;
    *sync_base = 0;
    if ((e = cudaMalloc(&sl.ptr, dmma_sk_scratch_bytes())) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(sl.ptr, 0, kSkFlagBytes, stream)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&sl.ev, cudaEventDisableTiming)) != cudaSuccess) {
        cudaFree(sl.ptr);
        return e;
    }
    try {
        g_sk_slots.push_back(sl);
    } catch (const std::exception &) {
        cudaEventDestroy(sl.ev);
        cudaFree(sl.ptr);
        return cudaErrorMemoryAllocation;
    }
    *slot = (int)g_sk_slots.size() - 1; *ptr = sl.ptr; *epoch = 1;
    return cudaSuccess;
}

cudaError_t sk_cache_release(int slot, cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g_sk_mu);
    SkSlot &sl = g_sk_slots[(size_t)slot];
    const cudaError_t e = cudaEventRecord(sl.ev, stream);
    sl.held = false;
    return e;
}

// Gives the cached buffers back to the driver (chase_scratch_cache_release): waits for the launch each one last
// served, frees it, forgets it.  A buffer some host thread holds at this moment stays.
cudaError_t sk_cache_clear() {
    std::lock_guard<std::mutex> lock(g_sk_mu);
    cudaError_t first = cudaSuccess;
    for (SkSlot &sl : g_sk_slots) {
        if (sl.held) {
            // indices of held slots must stay valid for their sk_cache_release: only a cache without held slots shrinks
            return cudaErrorNotReady;
        }
    }
    for (SkSlot &sl : g_sk_slots) {
        cudaError_t e = cudaEventSynchronize(sl.ev);
        if (e == cudaSuccess) e = cudaFree(sl.ptr);
        const cudaError_t e2 = cudaEventDestroy(sl.ev);
        if (first == cudaSuccess) first = e != cudaSuccess ? e : e2;
    }
    g_sk_slots.clear();
    return first;
}

template <bool CPLX>
cudaError_t launch(DmmaPlan *plan, int src, int64_t s, double alpha, double beta, double c, int use_beta,
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

    // The plan only depends on the active width: reuse it across the steps of one filter call.
    if (plan->step_plan_n != n) {
        try {
            make_plan<CPLX>(plan->M, plan->N, n, sm_count(), true, plan->step_plan);
        } catch (const std::exception &) {
            return cudaErrorMemoryAllocation;
        }
        plan->step_plan_n = n;
    }
    const StepPlan &pl = plan->step_plan;

    // Scratch (stream-K flags and partial tiles, soft-barrier counter): the caller's (chase_filter_ws: part of
    // the workspace), else one of the library's cached buffers, handed out in stream order (sk_cache_*).
    unsigned char *scratch = (unsigned char *)plan->sk_scratch;
    int cache_slot = -1;
    uint32_t epoch = 0;
    unsigned sync_base = 0;
    const bool want_sync = pl.dp_rounds >= 1 && pl.sk_ctas > 0 && pl.sk_first == 0;   // persistent CTAs with whole-tile rounds
    const unsigned sync_arrivals =
        want_sync ? (unsigned)pl.grid * (unsigned)pl.dp_rounds * (unsigned)((pl.KT + kSyncSlabs - 1) / kSyncSlabs) : 0u;
    cudaError_t e;
    if (pl.sk_ctas > 0) {
        if (!scratch) {
            if ((e = sk_cache_acquire(&cache_slot, (void **)&scratch, &epoch, &sync_base, sync_arrivals, stream)) != cudaSuccess)
                return e;
        } else {
            if (plan->sk_epoch == 0) {                                     // flags and counter start at 0, epochs at 1
                if ((e = cudaMemsetAsync(scratch, 0, kSkFlagBytes, stream)) != cudaSuccess) return e;
                plan->sync_count = 0;
            }
            epoch = ++plan->sk_epoch;
            sync_base = plan->sync_count;
            plan->sync_count += sync_arrivals;
        }
    }

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
    p.tiles_m = pl.tiles_m;
    p.tiles_n = pl.tiles_n;
    p.ragged_last = pl.ragged_last;
    p.bn_w = pl.bn_w;
    p.dp_tiles = pl.dp_tiles;
    p.dp_rounds = pl.dp_rounds;
    p.sk_first = pl.sk_first;
    p.sk_ctas = pl.sk_ctas;
    p.sync_ctr = want_sync && scratch ? (unsigned *)(scratch + kSkSyncOffset) : nullptr;
    p.sync_base = sync_base;
    p.epoch = epoch;
    p.sk_flag = (uint32_t *)scratch;
    p.sk_part = scratch ? scratch + kSkFlagBytes : nullptr;
    p.alpha = alpha;
    p.beta = beta;
    p.c = c;
    p.c_col = c_col;
    p.use_beta = use_beta;
    std::memcpy(p.sk_begin, pl.sk_begin, sizeof(int) * (size_t)(pl.sk_ctas + 1));
    const CUtensorMap *mA = (const CUtensorMap *)plan->tmap_H;
    const CUtensorMap *mB = (const CUtensorMap *)plan->tmap_B[src];

    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)pl.grid);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = Smem<CPLX>::TOTAL;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, step_dmma_kernel<CPLX>, *mA, *mB, p);
    count_launch();
    if (cache_slot >= 0) {
        const cudaError_t e2 = sk_cache_release(cache_slot, stream);
        if (e == cudaSuccess) e = e2;
    }
    return e;
}

}  // namespace

size_t dmma_sk_scratch_bytes() { return kSkFlagBytes + (size_t)kMaxSkCtas * kPartBytes; }

cudaError_t dmma_sk_cache_clear() { return sk_cache_clear(); }

void dmma_step_plan(int64_t N, int64_t n, chase_dtype_t dtype, int sms, StepPlan *out) {
    if (dtype == CHASE_C128) make_plan<true>(N, N, n, sms, true, *out);
    else make_plan<false>(N, N, n, sms, true, *out);
}

bool dmma_supported(int64_t N, int64_t ncols, chase_dtype_t dtype) {
    if (ncols < 1 || N < 16 || N > (1 << 28) || ncols > (1 << 28)) return false;
    if (dtype == CHASE_C128) return true;           // column stride N * 16 bytes: always a TMA-legal stride
    if (dtype == CHASE_F64) return N % 2 == 0;      // TMA strides must be multiples of 16 bytes
    return false;
}

static void plan_common(DmmaPlan *plan, chase_dtype_t dtype, const void *H, int64_t N, int64_t row0, int64_t nrows,
                        int64_t ldh, void *V, void *W, int64_t ncols) {
    plan->dtype = dtype;
    plan->N = N;
    plan->M = nrows;
    plan->ldh = ldh;
    plan->row0 = row0;
    plan->npeers = 0;
    plan->ncols = ncols;
    plan->H = H;
    plan->buf[0] = V;
    plan->buf[1] = W;
    plan->sk_scratch = nullptr;
    plan->sk_epoch = 0;
    plan->sync_count = 0;
    plan->step_plan_n = -1;
}

cudaError_t dmma_plan_create(DmmaPlan *plan, chase_dtype_t dtype, const void *H, int64_t N, void *V, void *W,
                             int64_t ncols) {
    return dmma_plan_create_rows(plan, dtype, H, N, 0, N, V, W, ncols);
}

cudaError_t dmma_plan_create_rows(DmmaPlan *plan, chase_dtype_t dtype, const void *H_loc, int64_t N, int64_t row0,
                                  int64_t nrows, void *V, void *W, int64_t ncols) {
    plan_common(plan, dtype, H_loc, N, row0, nrows, nrows, V, W, ncols);
    return dtype == CHASE_C128 ? encode_maps<true>(plan) : encode_maps<false>(plan);
}

cudaError_t dmma_plan_create_panel(DmmaPlan *plan, chase_dtype_t dtype, const void *H_full, int64_t N, int64_t row0,
                                   int64_t nrows, void *V, void *W, int64_t ncols) {
    const size_t esz = dtype == CHASE_C128 ? 16 : 8;
    plan_common(plan, dtype, (const char *)H_full + (size_t)row0 * esz, N, row0, nrows, N, V, W, ncols);
    return dtype == CHASE_C128 ? encode_maps<true>(plan) : encode_maps<false>(plan);
}

cudaError_t dmma_launch_step(DmmaPlan *plan, int src, int64_t s, double alpha, double beta, double c,
                             int use_beta, cudaStream_t stream, const double *c_col) {
    return plan->dtype == CHASE_C128 ? launch<true>(plan, src, s, alpha, beta, c, use_beta, stream, c_col)
                                     : launch<false>(plan, src, s, alpha, beta, c, use_beta, stream, c_col);
}

}  // namespace chase

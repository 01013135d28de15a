// tcgen05 (5th-gen tensor core) step kernel for float32 / complex64: split-precision products on CTA pairs with
// FP32 accumulation in TMEM.
//
//   Y[:, j] <- alpha * (H X[:, j] - c X[:, j]) + beta * Y[:, j]     (Alg. 4 l.4 / l.9; Eq. 7)
//
// ONE kernel: step_tf32_pair_kernel<CPLX, MIXED>, 512 threads per CTA, two CTAs of a cluster (the two SMs of a
// TPC) on one 256 x 256 tile through tcgen05.mma.cta_group::2 (the section "CTA-pair variant" below has the
// roles, the rings and the barriers).
//
// Every fp32 operand x is split as x = hi + lo, hi = x with the low 13 mantissa bits cleared (what kind::tf32
// reads from an fp32 word), lo = x - hi (exact in fp32).  A product is hi*hi + (hi*lo + lo*hi); lo*lo ~ 2^-22
// relative is dropped.  hi*hi is a kind::tf32 MMA on the raw tiles.  The cross terms are
//   MIXED = true (default): ONE kind::f16 MMA on BF16 "pair tiles" over a doubled K (pack_pair below): 2 MMA units
//                           per product, error vs an FP64 evaluation ~2e-5 at degree 16;
//   MIXED = false (CHASE_TF32_MIXED=0): two more kind::tf32 MMAs on lo tiles -- classic 3xTF32, 3 units.
// All of them accumulate into one fp32 accumulator in tensor memory; plain single-pass TF32 (2^-11 per operand)
// would not meet the 1e-4 bound.
//
// Only the fp32 data itself crosses L2: TMA brings the raw H and X tiles (they serve as the hi operands, the tensor
// core ignores the low mantissa bits) and the converter warps derive the second tiles (lo or BF16 pair) -- and for
// complex64 the rotated tile -i X -- in shared memory.  The split is element-wise and the rotation stays inside a
// 16-byte chunk, so both are oblivious of the 64-byte swizzle.
//
// Both operands are K-major.  For A this uses that H is Hermitian (reading G9): row m of
// H along k is the conjugate of column m, which is contiguous in the column-major storage.
//   float32:   A[m][k] = H[k][m] (column m read along k); B = X as stored.
//   complex64: a REAL GEMM over the interleaved index kk = 2k + {0, 1}:
//     A2[m][kk]  = column m of H as floats    = (Re A[m,k], -Im A[m,k])      (conjugate of H[k,m])
//     B1[kk][j]  = column j of X as floats    = (Re x, Im x)
//     B2[kk][j]  = column j of -i X           = (Im x, -Re x)
//     A2 . B1 = Re(A x),  A2 . B2 = Im(A x):  D = complex rows x [128 Re | 128 Im] columns.
//
// The MMA issuer accumulates CHUNK stages into one of two TMEM buffers; the accumulator warps add each finished
// chunk into fp32 registers (round to nearest) while the tensor core fills the other buffer, then run the fused
// epilogue.  Shared-memory operand tiles are the canonical K-major SWIZZLE_64B UMMA layout written directly by
// TMA: [row][16 floats of k] (64-byte rows, 8-row groups 512 B apart); one TF32 UMMA consumes 8 k.
#include <cuda.h>

#include <algorithm>
#include <cstdlib>
#include <mutex>

#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kFirstAccWarp = 4;   // multiple of 4: TMEM lane quarter = warp % 4
constexpr int kAccWarps = 8;       // accumulator / epilogue warps: 4 TMEM lane quarters x 2 column halves
constexpr int KS = 16;            // floats of k per pipeline stage (two UMMA K = 8 slices)
constexpr int TM = 128;           // (complex or real) rows per CTA tile = TMEM lanes
constexpr int TN = 256;           // real B columns per CTA tile = TMEM columns
#ifndef TF32_CHUNK
#define TF32_CHUNK 8
#endif
constexpr int CHUNK = TF32_CHUNK;            // pipeline stages accumulated in TMEM before the sum moves to registers
constexpr int A_BYTES = TM * KS * 4;          // 8 KB

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
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
// Wait of a warp that expects to wait LONG (accumulator warps on a chunk, the producer on a free stage): back off
// between polls, so that the idle roles do not burn issue slots and power next to the converter warps.
#ifndef TF32_WAIT_SLEEP_NS
#define TF32_WAIT_SLEEP_NS 200
#endif
__device__ __forceinline__ void mbar_wait_long(uint32_t bar, uint32_t parity) {
    uint32_t done;
    for (;;) {
        asm volatile(
            "{\n.reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n}\n"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) break;
        if (TF32_WAIT_SLEEP_NS > 0) __nanosleep(TF32_WAIT_SLEEP_NS);
    }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}

__device__ __forceinline__ void tma_prefetch_2d(const CUtensorMap *map, int c0, int c1) {
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global [%0, {%1, %2}];" ::"l"(map), "r"(c0), "r"(c1) : "memory");
}

// UMMA shared-memory matrix descriptor (sm_100): start address, leading / stride byte offsets
// (all >> 4), version = 1, layout type in bits 61..63 (2 = SWIZZLE_128B, 4 = SWIZZLE_64B).
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout) {
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46) | ((uint64_t)layout << 61);
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, float4 v) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float4 split_lo(float4 v) {
    return make_float4(v.x - tf32_hi(v.x), v.y - tf32_hi(v.y), v.z - tf32_hi(v.z), v.w - tf32_hi(v.w));
}
// Mixed scheme (DESIGN.md 6.4 "TF32 + BF16 cross terms"): the two small products hi*lo + lo*hi of a k-slice are
// ONE kind::f16 MMA over a doubled K: the 16-byte chunk that holds the fp32 values x0..x3 (k .. k+3) becomes the
// 16-byte chunk of 8 BF16 values [x0 x1 x2 x3 | l0 l1 l2 l3] for A and [l0 l1 l2 l3 | x0 x1 x2 x3] for B
// (l = x - tf32_hi(x), both rounded to nearest BF16), so slot s of A meets slot s of B: sum_k xA lB + lA xB.
// Element-wise per chunk, hence at the same (swizzled) position as the raw chunk.
__device__ __forceinline__ uint32_t bf16x2(float lo_elem, float hi_elem) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi_elem), "f"(lo_elem));   // first source -> upper half
    return r;
}
template <bool B_SIDE>
__device__ __forceinline__ float4 pack_pair(float4 v) {
    const float4 l = make_float4(v.x - tf32_hi(v.x), v.y - tf32_hi(v.y), v.z - tf32_hi(v.z), v.w - tf32_hi(v.w));
    const float x01 = __uint_as_float(bf16x2(v.x, v.y)), x23 = __uint_as_float(bf16x2(v.z, v.w));
    const float l01 = __uint_as_float(bf16x2(l.x, l.y)), l23 = __uint_as_float(bf16x2(l.z, l.w));
    return B_SIDE ? make_float4(l01, l23, x01, x23) : make_float4(x01, x23, l01, l23);
}
// the second tile of an operand: its lo part (3xTF32) or its BF16 pair tile (mixed scheme)
template <bool B_SIDE>
__device__ __forceinline__ float4 second_tile(float4 v, int mixed) {
    return mixed ? pack_pair<B_SIDE>(v) : split_lo(v);
}
__device__ __forceinline__ float4 rot_mi(float4 v) { return make_float4(v.y, -v.x, v.w, -v.z); }   // -i (x + iy) pairs


struct Tf32Params {
    const float *X;                     // source iterate, first active column
    float *Y;                           // destination iterate (holds V_{k-1}, becomes V_{k+1}), first active column
    int64_t N;                          // matrix order
    int64_t KF;                         // floats along k per column: 2N (complex) or N (real)
    int n;                              // active columns
    int col0;                           // first active column in the full buffers (TMA coordinate offset)
    int tiles_m, tiles_n;
    float alpha, beta, c;
    const double *c_col;
    int use_beta;
    unsigned *sync_ctr;                 // soft grid barrier counter (zeroed before the launch) or nullptr
    int mixed;                          // 1: hi*hi in TF32 + one BF16 MMA for the cross terms; 0: classic 3xTF32
};

#ifndef TF32_SYNC_STAGES
#define TF32_SYNC_STAGES 64
#endif
constexpr int kSyncStages = TF32_SYNC_STAGES;   // producers meet every this many pipeline stages
constexpr int kSyncMaxPolls = 512;              // bounded wait (~50 us): the barrier is only a hint
constexpr int kGroupN = 8;
__device__ __forceinline__ void tile_coords(int t, int tiles_m, int tiles_n, int &tm, int &tn) {
    const int per_group = kGroupN * tiles_m;
    const int grp = t / per_group;
    const int first_n = grp * kGroupN;
    const int gn = min(kGroupN, tiles_n - first_n);
    const int r = t - grp * per_group;
    tm = r / gn;
    tn = first_n + r % gn;
}

// Soft grid barrier between the TMA producers of all CTAs (a performance hint, never needed for
// correctness): arrive on a global counter and poll until `target` arrivals, for a bounded time.
// Returns false if the wait timed out (the caller then stops syncing: some CTA is not running alongside).
__device__ __forceinline__ bool soft_grid_sync(unsigned *ctr, unsigned target) {
    atomicAdd(ctr, 1u);
    for (int i = 0; i < kSyncMaxPolls; ++i) {
        unsigned v;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        if ((int)(v - target) >= 0) return true;
        __nanosleep(64);
    }
    return false;
}

// Persistent: CTA b processes tiles b, b + gridDim.x, ... of the grouped raster (round r = the tiles
// r * gridDim.x .. (r+1) * gridDim.x - 1, i.e. ~8 column tiles x ~18 row tiles that share H row panels and
// X column panels in L2).  The resident CTAs only share those panels if they walk along k TOGETHER: the
// L2 holds ~18 pipeline stages of the union stream, a tile lasts ~7500 stages.  So the producers meet at
// a soft barrier at the start of every tile and every kSyncStages stages.
// ---------------------------------------------------------------- CTA-pair variant (cta_group::2)
// Two CTAs of a cluster (the two SMs of a TPC) share one 256 x 256 tile: tcgen05.mma.cta_group::2 with
// M = 256 takes 128 rows of A from each CTA's shared memory and HALF of B (128 of the 256 real columns)
// from each, and leaves each CTA's 128 x 256 accumulator rows in its own TMEM.  Per CTA and stage the
// tensor core then reads 48 KB of operands instead of 72 KB and the converter warps derive the lo (and,
// complex, the rotated -iX) tiles of only 8 KB of B instead of 16 KB: the shared-memory port, which
// bounded the single-CTA kernel at ~72 % tensor activity, drops below the MMA time.
//   complex64: CTA 0 holds X (-> real parts), CTA 1 holds -iX (-> imaginary parts), both from the same
//              raw X tile (CTA 1 rotates it in place); float32: each CTA holds its 128 columns of X.
// Synchronisation: every CTA has its own TMA / empty / accumulator-full barriers (tcgen05.commit is
// multicast to both); the barriers that gate the single MMA issuer (CTA 0) -- "converted" and
// "accumulator drained" -- live in CTA 0 and take remote arrivals from CTA 1 (mapa + cluster-scope
// release / acquire).
// Thread layout of the pair kernel (4 warpgroups, registers rebalanced with setmaxnreg): warpgroup 0 = TMA producer,
// MMA issuer, two idle warps (40 registers); warpgroups 1-2 = accumulator / epilogue warps (184); warpgroup 3 =
// converter warps (104).  The converters form kConvGroups2 groups of kConvWpg2 warps; group g derives the second
// tiles of the stages it % kConvGroups2 == g, so the fixed latencies of consecutive stages (barrier wait, LDS
// round trip, fence.proxy.async) overlap.  Measured: with two converter warps that serial chain,
// not the tensor core, set the stage time (1320 clk against an MMA floor of 512-768).
#ifndef TF32_CONV_GROUPS
#define TF32_CONV_GROUPS 2
#endif
#ifndef TF32_CONV_WARPS
#define TF32_CONV_WARPS 4          // 8 (two converter warpgroups) measured slower: more power, same stage time
#endif
constexpr int kConvWarps2 = TF32_CONV_WARPS;
constexpr int kConvGroups2 = TF32_CONV_GROUPS;
constexpr int kConvWpg2 = kConvWarps2 / kConvGroups2;
constexpr int kFirstConvWarp2 = kFirstAccWarp + kAccWarps;     // 12
constexpr int kThreads2 = (kFirstConvWarp2 + kConvWarps2) * 32;   // 640
// registers per thread after setmaxnreg: 128 x 40 (warpgroup 0) + 256 x kAccRegs2 + 32 kConvWarps2 x kConvRegs2 <= 65536
// setmaxnreg moves registers inside the CTA's OWN allocation (threads x the launch count ptxas reports: 128 for
// 512 threads, 96 for 640), so the counts after rebalancing must fit in that, or the .inc never returns.
constexpr int kLaunchRegs2 = kConvWarps2 == 8 ? 96 : 128;
constexpr int kConvRegs2 = kConvWarps2 == 8 ? 64 : 104;
constexpr int kAccRegs2 = kConvWarps2 == 8 ? 152 : 184;
static_assert(kConvWarps2 == 4 || kConvWarps2 == 8, "whole converter warpgroups");
static_assert(128 * 40 + 256 * kAccRegs2 + 32 * kConvWarps2 * kConvRegs2 <= kThreads2 * kLaunchRegs2,
              "registers of one CTA");
static_assert(kConvGroups2 * kConvWpg2 == kConvWarps2, "converter groups must tile the converter warps");
// Two rings: the RAW tiles [A | B] written by TMA live from the load to the retirement of the
// stage's MMAs, the SECOND tiles [A' | B'] written by the converters only from the conversion on.  With one
// 32 KB ring of 6 stages the ~3000-clock TMA round trip alone capped the rate at 6 stages per round trip
// (measured: 521 clk per stage with neither conversion nor MMAs); a deep raw ring and a short second ring keep
// 10 loads in flight in the same shared memory.
#ifndef TF32_RAW_STAGES
#define TF32_RAW_STAGES 10
#endif
#ifndef TF32_PAIR_STAGES
#define TF32_PAIR_STAGES 3
#endif
#ifndef TF32_PREFETCH
#define TF32_PREFETCH 0           // stages the producer prefetches into L2 ahead of its loads (0: off; 12 measured
                                  // 3 % SLOWER: the lock-step CTAs already find each other's lines in L2)
#endif
constexpr int RAW2 = TF32_RAW_STAGES, SEC2 = TF32_PAIR_STAGES, kPrefetch2 = TF32_PREFETCH;
static_assert(SEC2 < RAW2, "the second ring must be shorter than the raw ring (see the converter's slot-free wait)");
constexpr int BH = TN / 2;                       // real B columns held by one CTA of a pair
constexpr int B2_BYTES = BH * KS * 4;            // 8 KB
constexpr int RAW2_BYTES = A_BYTES + B2_BYTES;   // A raw | B raw (complex, CTA 1: rotated in place) : 16 KB
constexpr int SEC2_BYTES = A_BYTES + B2_BYTES;   // A' | B' (lo parts or BF16 pair tiles)             : 16 KB
constexpr int SMEM2_TOTAL = RAW2 * RAW2_BYTES + SEC2 * SEC2_BYTES + 1024 + 512;
static_assert(SMEM2_TOTAL <= 232448, "shared memory of one CTA");
constexpr uint32_t kInstrDesc2 = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TN >> 3) << 17) |
                                 ((uint32_t)((2 * TM) >> 4) << 24);

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// Arrive on a barrier of the peer CTA.  Default (CTA-scope release) semantics, as for a local arrive: the
// cluster-scope forms cost a MEMBAR.ALL.GPU per arrive and an L1 invalidation per wait (measured: 2000
// instead of 830 clk per stage).  What the arrive publishes here is shared memory already fenced for the
// async proxy (converters) or the completion of TMEM loads (accumulator warps), not global memory.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) { mbar_wait(bar, parity); }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void umma_tf32_pair(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n}\n"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(kInstrDesc2), "r"(accumulate) : "memory");
}
constexpr uint32_t kInstrDescBf16Pair = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TN >> 3) << 17) |
                                        ((uint32_t)((2 * TM) >> 4) << 24);
__device__ __forceinline__ void umma_bf16_pair(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n}\n"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(kInstrDescBf16Pair), "r"(accumulate) : "memory");
}
// arrives (once the MMAs issued so far have retired) on the barrier at this offset in BOTH CTAs of the pair
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(bar), "h"((uint16_t)3) : "memory");
}

template <bool CPLX, bool MIXED>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads2, 1)
step_tf32_pair_kernel(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB,
                      const Tf32Params p) {
    constexpr int COLS = CPLX ? TN / 2 : TN;      // (complex or real) columns per pair tile
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t sec_base = smem_base + RAW2 * RAW2_BYTES;
    const uint32_t bar_base = sec_base + SEC2 * SEC2_BYTES;   // full[RAW2], empty[RAW2], conv[SEC2], tfull[2], tempty[2], tmem slot
    const uint32_t bar_empty = bar_base + 8 * RAW2;
    const uint32_t bar_conv = bar_base + 8 * (2 * RAW2);
    const uint32_t bar_tfull = bar_conv + 8 * SEC2;
    const uint32_t bar_tempty = bar_tfull + 16;
    const uint32_t tmem_slot = bar_tempty + 16;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();              // 0: leader (issues the MMAs), 1: peer
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
    const int total_tiles = p.tiles_m * p.tiles_n;        // tiles of 256 rows
    const int KT = (int)((p.KF + KS - 1) / KS);
    const int NCH = (KT + CHUNK - 1) / CHUNK;

    if (threadIdx.x == 0) {
        for (int s = 0; s < RAW2; ++s) {
            mbar_init(bar_base + 8 * s, 1);                       // full: this CTA's producer (expect_tx)
            mbar_init(bar_empty + 8 * s, 1);                      // empty: one multicast tcgen05.commit
        }
        for (int s = 0; s < SEC2; ++s)
            mbar_init(bar_conv + 8 * s, 2 * kConvWpg2);           // conv (used in CTA 0): one converter group of both CTAs
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_tfull + 8 * b, 1);                      // chunk accumulator complete (multicast commit)
            mbar_init(bar_tempty + 8 * b, 2 * kAccWarps);         // (used in CTA 0): drained by both CTAs' accumulator warps
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {   // all of TMEM in both CTAs: two 256-column fp32 accumulators (ping-pong between chunks)
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(2 * TN) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();                                     // barriers of both CTAs initialised before any remote arrive
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot) : "memory");

    if (warp < kFirstAccWarp) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");

    if (warp == 0) {
        // ------------------------------------------------------------------ TMA producer (both CTAs)
        if (lane == 0) {
            const int syncs_per_tile = (KT + kSyncStages - 1) / kSyncStages;
            unsigned it = 0;
            unsigned *sync_ctr = p.sync_ctr;
            int round = 0;
            // L2 prefetch cursor: runs kPrefetch2 stages ahead of the loads (through tile boundaries), so that the
            // loads that fill shared memory find their lines in L2 instead of paying the DRAM round trip.
            int pf_tile = pair, pf_kt = 0, pf_m0 = 0, pf_nb0 = 0;
            auto pf_coords = [&]() {
                int tm, tn;
                tile_coords(pf_tile, p.tiles_m, p.tiles_n, tm, tn);
                pf_m0 = tm * (2 * TM) + (int)rank * TM;
                pf_nb0 = p.col0 + tn * COLS + (CPLX ? 0 : (int)rank * BH);
            };
            auto prefetch_next = [&]() {
                if (kPrefetch2 == 0 || pf_tile >= total_tiles) return;
                tma_prefetch_2d(&tmapA, pf_kt * KS, pf_m0);
                if (!CPLX || rank == 0) tma_prefetch_2d(&tmapB, pf_kt * KS, pf_nb0);   // complex: the pair shares one X tile
                if (++pf_kt == KT) {
                    pf_kt = 0;
                    pf_tile += npairs;
                    if (pf_tile < total_tiles) pf_coords();
                }
            };
            if (kPrefetch2 > 0 && pf_tile < total_tiles) {
                pf_coords();
                for (int i = 0; i < kPrefetch2; ++i) prefetch_next();
            }
            for (int tile = pair; tile < total_tiles; tile += npairs, ++round) {
                int tile_m, tile_n;
                tile_coords(tile, p.tiles_m, p.tiles_n, tile_m, tile_n);
                const int m0 = tile_m * (2 * TM) + (int)rank * TM, n0 = tile_n * COLS;
                const int nb0 = p.col0 + n0 + (CPLX ? 0 : (int)rank * BH);   // complex: both CTAs take the same raw X tile
                const unsigned active = 2u * (unsigned)min(npairs, total_tiles - round * npairs);
                const unsigned sync_base = (unsigned)round * gridDim.x * (unsigned)syncs_per_tile;
                for (int kt = 0; kt < KT; ++kt, ++it) {
                    if (sync_ctr && kt % kSyncStages == 0 &&
                        !soft_grid_sync(sync_ctr, sync_base + active * (unsigned)(kt / kSyncStages + 1)))
                        sync_ctr = nullptr;
                    prefetch_next();
                    const int s = it % RAW2;
                    const uint32_t full = bar_base + 8 * s, empty = bar_empty + 8 * s;
                    if (it >= RAW2) mbar_wait_long(empty, ((it / RAW2) - 1) & 1);
                    const uint32_t sa = smem_base + s * RAW2_BYTES, sb = sa + A_BYTES;
                    const int k0 = kt * KS;
                    mbar_expect_tx(full, A_BYTES + B2_BYTES);
                    tma_load_2d(sa, &tmapA, full, k0, m0);
                    tma_load_2d(sb, &tmapB, full, k0, nb0);
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (leader CTA only)
        if (lane == 0 && rank == 0) {
            unsigned it = 0, gc = 0;
            for (int tile = pair; tile < total_tiles; tile += npairs) {
                int kt = 0;
                for (int ch = 0; ch < NCH; ++ch, ++gc) {
                    const int b = gc & 1;
                    if (gc >= 2) {   // the accumulator warps of BOTH CTAs must have drained this buffer's previous chunk
                        mbar_wait_cluster(bar_tempty + 8 * b, ((gc >> 1) - 1) & 1);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    }
                    const uint32_t d = tmem_base + b * TN;
                    const int kt_end = min(KT, kt + CHUNK);
                    for (bool first = true; kt < kt_end; ++kt, ++it) {
                        const int s = it % RAW2, s2 = it % SEC2;
                        mbar_wait(bar_base + 8 * s, (it / RAW2) & 1);             // this CTA's TMA tiles landed
                        mbar_wait_cluster(bar_conv + 8 * s2, (it / SEC2) & 1);    // second tiles written in both CTAs
                                                                                  // (the peer's converters saw its TMA tiles)
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t sa_hi = smem_base + s * RAW2_BYTES, sb_hi = sa_hi + A_BYTES;
                        const uint32_t sa_lo = sec_base + s2 * SEC2_BYTES, sb_lo = sa_lo + A_BYTES;
#pragma unroll
                        for (int ks = 0; ks < KS / 8; ++ks) {
                            const uint64_t ah = umma_desc(sa_hi + ks * 32, 16, 512, 4);
                            const uint64_t al = umma_desc(sa_lo + ks * 32, 16, 512, 4);
                            const uint64_t bh = umma_desc(sb_hi + ks * 32, 16, 512, 4);
                            const uint64_t bl = umma_desc(sb_lo + ks * 32, 16, 512, 4);
                            if (MIXED) {
                                umma_bf16_pair(d, al, bl, first ? 0u : 1u);    // x_b * lo_b + lo_b * x_b (pair tiles, K = 16)
                            } else {
                                umma_tf32_pair(d, ah, bl, first ? 0u : 1u);    // hi * lo  (first MMA of a chunk overwrites)
                                umma_tf32_pair(d, al, bh, 1u);                 // lo * hi
                            }
                            umma_tf32_pair(d, ah, bh, 1u);                     // hi * hi
                            first = false;
                        }
                        umma_commit_pair(bar_empty + 8 * s);              // frees the stage in both CTAs when these MMAs retire
                    }
                    umma_commit_pair(bar_tfull + 8 * b);                  // this chunk's accumulator is complete (both CTAs)
                }
            }
        }
    } else if (warp >= kFirstConvWarp2) {
        // ------------------------------------------------------------------ converter warps (both CTAs)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kConvRegs2));
        constexpr int CT = kConvWpg2 * 32;                       // threads that share one stage
        constexpr int NA = A_BYTES / 16 / CT, NBV = B2_BYTES / 16 / CT;
        constexpr int BATCH = NA < 8 ? NA : 8;                   // 16-byte chunks of A (and of B) in flight per thread
        const int grp = (warp - kFirstConvWarp2) / kConvWpg2;
        const int ct = ((warp - kFirstConvWarp2) % kConvWpg2) * 32 + lane;
        const uint32_t leader_conv = mapa_shared(bar_conv, 0);
        unsigned it = 0;
        for (int tile = pair; tile < total_tiles; tile += npairs) {
            for (int kt = 0; kt < KT; ++kt, ++it) {
                if ((int)(it % kConvGroups2) != grp) continue;
                const int s = it % RAW2, s2 = it % SEC2;
                mbar_wait(bar_base + 8 * s, (it / RAW2) & 1);
                // slot s2 of the second ring is free once the MMAs of stage it - SEC2 have retired, which is what the
                // raw ring's empty barrier of that stage reports (it cannot be a whole phase further: the in-order
                // MMA issuer has not seen stage `it` converted yet, and SEC2 < RAW2)
                if (it >= (unsigned)SEC2) mbar_wait(bar_empty + 8 * ((it - SEC2) % RAW2), ((it - SEC2) / RAW2) & 1);
                const uint32_t sa_hi = smem_base + s * RAW2_BYTES, sb_hi = sa_hi + A_BYTES;
                const uint32_t sa_lo = sec_base + s2 * SEC2_BYTES, sb_lo = sa_lo + A_BYTES;
#pragma unroll
                for (int b0 = 0; b0 < NA; b0 += BATCH) {
                    float4 va[BATCH], vb[BATCH];
#pragma unroll
                    for (int i = 0; i < BATCH; ++i) va[i] = lds128(sa_hi + (uint32_t)(ct + (b0 + i) * CT) * 16);
#pragma unroll
                    for (int i = 0; i < BATCH; ++i) vb[i] = lds128(sb_hi + (uint32_t)(ct + (b0 + i) * CT) * 16);
#pragma unroll
                    for (int i = 0; i < BATCH; ++i)
                        sts128(sa_lo + (uint32_t)(ct + (b0 + i) * CT) * 16, second_tile<false>(va[i], MIXED));
                    if (CPLX && rank == 1) {
                        // this CTA supplies -iX: rotate the raw tile in place (a thread rewrites the chunk it read)
#pragma unroll
                        for (int i = 0; i < BATCH; ++i) {
                            const uint32_t off = (uint32_t)(ct + (b0 + i) * CT) * 16;
                            const float4 r = rot_mi(vb[i]);
                            sts128(sb_hi + off, r);
                            sts128(sb_lo + off, second_tile<true>(r, MIXED));
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < BATCH; ++i)
                            sts128(sb_lo + (uint32_t)(ct + (b0 + i) * CT) * 16, second_tile<true>(vb[i], MIXED));
                    }
                }
                static_assert(NA == NBV && NA % BATCH == 0, "A and B halves of a stage have the same size");
                // generic-proxy writes -> visible to the tensor core's async-proxy reads
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(leader_conv + 8 * s2);
            }
        }
    } else if (warp >= kFirstAccWarp && warp < kFirstConvWarp2) {
        // ------------------------------------------------------------------ accumulator / epilogue warps (both CTAs)
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kAccRegs2));
        const int quarter = warp & 3;
        const int half = (warp - kFirstAccWarp) >> 2;
        const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + half * (TN / 2);
        const uint32_t leader_tempty = mapa_shared(bar_tempty, 0);
        const float alpha = p.alpha, beta = p.beta;
        unsigned gc = 0;
        for (int tile = pair; tile < total_tiles; tile += npairs) {
            int tile_m, tile_n;
            tile_coords(tile, p.tiles_m, p.tiles_n, tile_m, tile_n);
            const int m0 = tile_m * (2 * TM) + (int)rank * TM, n0 = tile_n * COLS;
            float racc[TN / 2];
#pragma unroll
            for (int i = 0; i < TN / 2; ++i) racc[i] = 0.f;
            for (int ch = 0; ch < NCH; ++ch, ++gc) {
                const int b = gc & 1;
                mbar_wait_long(bar_tfull + 8 * b, (gc >> 1) & 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int j = 0; j < TN / 2 / 16; ++j) {      // 16 columns at a time: the 128 sums leave few registers
                    float t[16];
                    tmem_ld16(taddr + b * TN + j * 16, t);
#pragma unroll
                    for (int i = 0; i < 16; ++i) racc[j * 16 + i] += t[i];
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(leader_tempty + 8 * b);
            }

            const int64_t row = (int64_t)m0 + quarter * 32 + lane;
            const bool row_ok = row < p.N;
#pragma unroll
            for (int i = 0; i < TN / 2; ++i) {
                // complex: half 0 owns the real parts, half 1 the imaginary parts of columns n0 .. n0+127
                const int col = CPLX ? n0 + i : n0 + half * (TN / 2) + i;
                if (col < p.n && row_ok) {
                    const float c = p.c_col ? (float)p.c_col[col] : p.c;
                    const int64_t off = CPLX ? ((int64_t)col * p.N + row) * 2 + half : (int64_t)col * p.N + row;
                    float y = alpha * (racc[i] - c * __ldcg(p.X + off));   // L2 only: see step_dmma.cu
                    if (p.use_beta) y = fmaf(beta, __ldcg(p.Y + off), y);
                    p.Y[off] = y;
                }
            }
        }
    }

    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();                                     // no CTA frees TMEM or exits while its peer may still signal it
    if (warp == 1) {
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(2 * TN) : "memory");
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

// A column-major float matrix (KF floats per column, `cols` columns) viewed K-major:
// box = 16 floats of k x `box_rows` columns, SWIZZLE_64B.
cudaError_t encode_kmajor(CUtensorMap *map, const void *base, int64_t KF, int64_t cols, int box_rows) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return cudaErrorNotSupported;
    cuuint64_t dims[2] = {(cuuint64_t)KF, (cuuint64_t)cols};
    cuuint64_t strides[1] = {(cuuint64_t)KF * 4};
    cuuint32_t box[2] = {16, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

int sm_count() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        sms = 148;
    return sms;
}

template <bool CPLX>
cudaError_t launch(const Tf32Plan *plan, int src, int64_t s, double alpha, double beta, double c, int use_beta,
                   cudaStream_t stream, const double *c_col) {
    static std::once_flag once;
    static cudaError_t attr_err = cudaSuccess;
    std::call_once(once, [] {
        attr_err = cudaFuncSetAttribute(step_tf32_pair_kernel<CPLX, true>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM2_TOTAL);
        if (attr_err == cudaSuccess)
            attr_err = cudaFuncSetAttribute(step_tf32_pair_kernel<CPLX, false>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM2_TOTAL);
    });
    if (attr_err != cudaSuccess) return attr_err;
    const int64_t n = plan->ncols - s;
    if (n <= 0) return cudaSuccess;
    constexpr int COLS = CPLX ? TN / 2 : TN;
    constexpr int FL = CPLX ? 2 : 1;
    const size_t col_floats = (size_t)plan->N * FL;
    const int dst = src ^ 1;
    Tf32Params p;
    p.X = (const float *)plan->buf[src] + (size_t)s * col_floats;
    p.Y = (float *)plan->buf[dst] + (size_t)s * col_floats;
    p.N = plan->N;
    p.KF = plan->N * FL;
    p.n = (int)n;
    p.col0 = (int)s;
    p.tiles_m = (int)((plan->N + 2 * TM - 1) / (2 * TM));           // 256 rows per CTA pair
    p.tiles_n = (int)((n + COLS - 1) / COLS);
    p.alpha = (float)alpha;
    p.beta = (float)beta;
    p.c = (float)c;
    p.c_col = c_col;
    p.use_beta = use_beta;
    p.sync_ctr = (unsigned *)plan->sync_ctr;
    p.mixed = plan->mixed;
    const int total_tiles = p.tiles_m * p.tiles_n;
    if (p.sync_ctr) {
        cudaError_t e = cudaMemsetAsync(p.sync_ctr, 0, sizeof(unsigned), stream);
        if (e != cudaSuccess) return e;
    }
    // persistent CTA pairs: one cluster of 2 per TPC
    const int grid = 2 * std::min(total_tiles, std::max(1, sm_count() / 2));
    if (plan->mixed)
        step_tf32_pair_kernel<CPLX, true><<<(unsigned)grid, kThreads2, SMEM2_TOTAL, stream>>>(
            *(const CUtensorMap *)plan->tmap_A, *(const CUtensorMap *)plan->tmap_B[src], p);
    else
        step_tf32_pair_kernel<CPLX, false><<<(unsigned)grid, kThreads2, SMEM2_TOTAL, stream>>>(
            *(const CUtensorMap *)plan->tmap_A, *(const CUtensorMap *)plan->tmap_B[src], p);
    count_launch();
    return cudaGetLastError();
}

}  // namespace

bool tf32_supported(int64_t N, int64_t ncols, chase_dtype_t dtype) {
    if (ncols < 1 || N < 16 || N > (1 << 28) || ncols > (1 << 28)) return false;
    if (dtype == CHASE_C64) return N % 2 == 0;     // TMA: column stride must be a multiple of 16 bytes
    if (dtype == CHASE_F32) return N % 4 == 0;
    return false;
}

// Workspace layout: [W (one N x ncols block, vb bytes) | 256 bytes holding the soft-barrier counter].
int tf32_vector_blocks(chase_dtype_t) { return 1; }

cudaError_t tf32_plan_create(Tf32Plan *plan, chase_dtype_t dtype, const void *H, int64_t N, void *V,
                             void *workspace, size_t vb, int64_t ncols, cudaStream_t) {
    const bool cplx = dtype == CHASE_C64;
    const int64_t KF = N * (cplx ? 2 : 1);
    plan->dtype = dtype;
    plan->N = N;
    plan->ncols = ncols;
    plan->buf[0] = V;
    plan->buf[1] = workspace;
    plan->sync_ctr = (workspace && vb) ? (char *)workspace + vb : nullptr;
    // cross terms hi*lo + lo*hi as ONE BF16 MMA (2 MMA units per product) unless CHASE_TF32_MIXED=0 (classic 3xTF32)
    const char *mixed_env = std::getenv("CHASE_TF32_MIXED");
    plan->mixed = !(mixed_env && mixed_env[0] == '0');
    cudaError_t e;
    if ((e = encode_kmajor((CUtensorMap *)plan->tmap_A, H, KF, N, TM)) != cudaSuccess) return e;
    const int b_box = TN / 2;                                          // B columns one TMA box brings (one CTA's half)
    for (int i = 0; i < 2; ++i)
        if (plan->buf[i] &&
            (e = encode_kmajor((CUtensorMap *)plan->tmap_B[i], plan->buf[i], KF, ncols, b_box)) != cudaSuccess)
            return e;
    return cudaSuccess;
}

void *tf32_shared_sync_counter() {
    // one small buffer per device (a process may drive several GPUs), allocated on first use
    static std::mutex mu;
    static void *buf[64] = {};
    static bool tried[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (!tried[dev]) {
        tried[dev] = true;
        if (cudaMalloc(&buf[dev], 256) != cudaSuccess) {
            buf[dev] = nullptr;
            (void)cudaGetLastError();
        }
    }
    return buf[dev];
}

cudaError_t tf32_launch_step(const Tf32Plan *plan, int src, int64_t s, double alpha, double beta, double c,
                             int use_beta, cudaStream_t stream, const double *c_col) {
    return plan->dtype == CHASE_C64 ? launch<true>(plan, src, s, alpha, beta, c, use_beta, stream, c_col)
                                    : launch<false>(plan, src, s, alpha, beta, c, use_beta, stream, c_col);
}

}  // namespace chase

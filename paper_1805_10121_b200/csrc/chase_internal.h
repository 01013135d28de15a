// Internal declarations shared by the translation units of libchase_filter.so.
// Not part of the public ABI (that is include/chase_filter.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "chase_filter.h"
#include "chase_filter_bench.h"

namespace chase {

// One recurrence step (Alg. 4 line 4 / line 9) on `n` active columns:
//   Y[:, j] <- alpha * (H X[:, j] - c X[:, j]) + beta * Y[:, j],   j = 0..n-1
// X, Y are device pointers already offset to the first active column (ld = N).
// use_beta == 0: Y is write-only (first step: the scratch buffer is uninitialised).
struct StepArgs {
    const void *H;
    const void *X;
    void *Y;
    int64_t N;
    int64_t n;
    double alpha, beta, c;
    const double *c_col = nullptr;   // optional per-column shift (device double[n]); overrides c
    int use_beta;
};

// Generic FMA kernels: any N, any n, all four dtypes.
cudaError_t launch_step_generic(chase_dtype_t dtype, const StepArgs &a, cudaStream_t stream);

// Tall-skinny streaming kernel (csrc/step_skinny.cu): 1..kSkinnyMaxCols columns, all dtypes, any N;
// bound by one pass over H from HBM.  Uses that H is Hermitian.
constexpr int kSkinnyMaxCols = 8;
cudaError_t launch_step_skinny(chase_dtype_t dtype, const StepArgs &a, cudaStream_t stream);
// Same operation through a ring of bulk copies (csrc/step_stream.cu): persistent CTAs, long sequential
// DRAM bursts.  Needs 16-byte aligned H, X and columns (N * sizeof(element) % 16 == 0), N >= 64.
bool stream_supported(chase_dtype_t dtype, const StepArgs &a);
cudaError_t launch_step_stream(chase_dtype_t dtype, const StepArgs &a, cudaStream_t stream);

// TMA + DMMA tensor kernels (CHASE_C128 with any N >= 16, CHASE_F64 with even N).
// Work decomposition of one launch on `n` active columns (csrc/step_dmma.cu): tiles of
// 128 rows x bn_w columns in grouped raster order; `grid` persistent CTAs; CTA b owns the whole tiles
// r * grid + b (r < dp_rounds) of the first dp_tiles tiles, then CTAs 0 .. sk_ctas-1 share the k-slabs of the
// remaining tiles: CTA g owns slabs [sk_begin[g], sk_begin[g+1]) of that region, slab s = k-slab (s % KT) of
// tile dp_tiles + s / KT.
constexpr int kMaxSkCtas = 160;                 // >= SM count of any sm_100 part
constexpr size_t kSkFlagBytes = 1024;           // kMaxSkCtas uint32 flags + the soft-barrier counter, padded
constexpr size_t kSkSyncOffset = 800;           // byte offset of the soft-barrier counter inside the flag block
struct StepPlan {
    int KT, tiles_m, tiles_n, bn_w, dp_tiles, sk_ctas;
    int grid, dp_rounds;                        // CTAs launched; whole-tile rounds per CTA (tile r * grid + b)
    int ragged_last;                            // raster variant: the last tile column after all others (lock-step mode)
    int sk_first;                               // blockIdx of stream-K CTA 0 (0: persistent CTAs; dp_tiles: one CTA per whole tile)
    int sk_begin[kMaxSkCtas + 1];
};
// Bytes of device scratch the stream-K CTAs need (flags + one partial accumulator tile per CTA).
size_t dmma_sk_scratch_bytes();
// Frees the library's cached stream-K buffers (those launches without a caller workspace take); cudaErrorNotReady
// if a launch on another host thread holds one right now.
cudaError_t dmma_sk_cache_clear();
void dmma_step_plan(int64_t N, int64_t n, chase_dtype_t dtype, int sms, StepPlan *out);

// A plan holds the three tensor maps (H, and both vector buffers) of one chase_filter call.
struct DmmaPlan {
    alignas(64) unsigned char tmap_H[128];
    alignas(64) unsigned char tmap_B[2][128];   // [0]: buffer V, [1]: buffer W
    chase_dtype_t dtype;
    int64_t N, ncols;
    int64_t M, row0;                            // row block of H this launch owns (M = N, row0 = 0 unless row-sharded)
    int a_2d;                                   // set by the plan: 2-D H view (M not a multiple of the 128-byte row group)
    int64_t ldh;                                // leading dimension of the H view (M for a packed row block, N for a panel of the full H)
    const void *H;
    void *buf[2];
    int npeers;                                 // row-sharded: peer-mapped copies of buf[0], buf[1] on the other GPUs
    void *peer_buf[2][CHASE_MAX_RANKS - 1];
    void *sk_scratch;                           // dmma_sk_scratch_bytes() of device memory, or null: every launch that
                                                // needs it then takes stream-ordered memory (cudaMallocAsync)
    uint32_t sk_epoch;                          // flag value of the last stream-K launch on sk_scratch (0: flags not yet zeroed)
    unsigned sync_count;                        // arrivals the soft-barrier counter in sk_scratch has seen so far
    int64_t step_plan_n;                        // active width step_plan was made for (-1: none)
    StepPlan step_plan;
};
bool dmma_supported(int64_t N, int64_t ncols, chase_dtype_t dtype);
// Returns cudaSuccess or the error of the tensor-map encoding (reported to the caller; there is no
// silent fallback to another kernel family).
cudaError_t dmma_plan_create(DmmaPlan *plan, chase_dtype_t dtype, const void *H, int64_t N,
                             void *V, void *W, int64_t ncols);
// Row-sharded variant: H_loc is the nrows x N row block [row0, row0 + nrows) of H, column-major, ld = nrows.
cudaError_t dmma_plan_create_rows(DmmaPlan *plan, chase_dtype_t dtype, const void *H_loc, int64_t N, int64_t row0,
                                  int64_t nrows, void *V, void *W, int64_t ncols);
// Row panel [row0, row0 + nrows) of the FULL N x N matrix (ld = N): used to start the first step while H is
// still being uploaded panel by panel (chase_filter_host).
cudaError_t dmma_plan_create_panel(DmmaPlan *plan, chase_dtype_t dtype, const void *H_full, int64_t N, int64_t row0,
                                   int64_t nrows, void *V, void *W, int64_t ncols);
// Step reading buffer `src` (0/1) and writing buffer 1-src, active columns [s, ncols).
cudaError_t dmma_launch_step(DmmaPlan *plan, int src, int64_t s, double alpha, double beta,
                             double c, int use_beta, cudaStream_t stream, const double *c_col = nullptr);

// tcgen05 split-precision CTA-pair kernels (CHASE_C64 with N % 2 == 0, CHASE_F32 with N % 4 == 0).
struct Tf32Plan {
    alignas(64) unsigned char tmap_A[128];      // H viewed K-major (Hermitian: row m along k = conj of column m)
    alignas(64) unsigned char tmap_B[2][128];   // [0]: the caller's V, [1]: the workspace W
    chase_dtype_t dtype;
    int64_t N, ncols;
    void *buf[2];
    void *sync_ctr;                             // 4-byte counter of the producers' soft grid barrier
    int mixed;                                  // 1: TF32 hi*hi + one BF16 MMA for both cross terms, 0: classic 3xTF32
};
bool tf32_supported(int64_t N, int64_t ncols, chase_dtype_t dtype);
int tf32_vector_blocks(chase_dtype_t dtype);    // vector-sized blocks in the workspace besides H_lo
// Encodes the tensor maps.  vb = bytes of one N x ncols block rounded up to 256; the 256 bytes after
// it hold the soft-barrier counter.
cudaError_t tf32_plan_create(Tf32Plan *plan, chase_dtype_t dtype, const void *H, int64_t N, void *V,
                             void *workspace, size_t vb, int64_t ncols, cudaStream_t stream);
// A process-wide 256-byte device buffer for the soft barrier of launches that have no workspace
// (chase_hemm, chase_residuals, chase_lanczos); nullptr if it cannot be allocated.
void *tf32_shared_sync_counter();
cudaError_t tf32_launch_step(const Tf32Plan *plan, int src, int64_t s, double alpha, double beta, double c,
                             int use_beta, cudaStream_t stream, const double *c_col = nullptr);

// resid[j] = || R[:, j] ||_2 for an N x n column-major block R (device), resid device double[n].
cudaError_t launch_column_norms(chase_dtype_t dtype, const void *R, int64_t N, int64_t n, double *resid,
                                cudaStream_t stream);

// One launch of the step kernel family on whole buffers: Y <- alpha (H X - c X) + beta Y (c_col: optional
// per-column shift).  Returns 0, a negative CHASE_ERR_* or a positive cudaError_t.
int launch_one_step(const void *H, int64_t N, const void *X, void *Y, int64_t ncols, double alpha, double beta,
                    double c, const double *c_col, int use_beta, chase_dtype_t dtype, cudaStream_t stream,
                    void *sk_scratch = nullptr);

// Alg. 6: 1 + n_vec coalesced Lanczos runs (csrc/lanczos.cu).  alpha_host / beta_host: HOST [nvec * k],
// run r at offset r * k.  Synchronises `stream`.
size_t lanczos_workspace_bytes(int64_t N, int64_t nvec, int32_t k, size_t elem);
cudaError_t lanczos_run(const void *H, int64_t N, const void *V0, int nvec, int k, chase_dtype_t dtype, size_t elem,
                        void *workspace, double *alpha_host, double *beta_host, cudaStream_t stream);
// Alg. 6 l.13: Ritz vectors U^[run] z_i of the run's Ritz values below mu_ne (ascending, at most max_vecs) into
// columns dst_cols[i] of Vhat; `workspace` is the one lanczos_run left behind.  Synchronises `stream`.
cudaError_t lanczos_ritz_vectors(const void *workspace, int64_t N, int nvec, int k, chase_dtype_t dtype, size_t elem,
                                 int run, const double *alpha_run, const double *beta_run, double mu_ne, void *Vhat,
                                 const int64_t *dst_cols, int64_t max_vecs, int64_t *count, double *ritz_values,
                                 cudaStream_t stream);
// Ritz values (unsorted) and squared first eigenvector components of T_k; false = QL did not converge.
bool lanczos_ritz(int k, const double *alpha, const double *beta, std::vector<double> &lam, std::vector<double> &w);

void count_launch();

}  // namespace chase

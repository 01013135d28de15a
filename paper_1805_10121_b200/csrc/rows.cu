// Row-sharded filter across GPUs (SURVEY 8(e) option 2; Fig. 3): rank r owns a
// row block of H and a full copy of the vectors; the step kernel's epilogue pushes the rank's rows of
// the new iterate into every peer's copy over NVLink peer memory (csrc/step_dmma.cu), so the
// all-gather of the paper's distributed HEMM costs no extra pass.  This file holds the inter-GPU
// barrier (flags in peer memory), the CUDA IPC plumbing and the host loop of Alg. 4 for this layout.
#include <cuda.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "chase_internal.h"

namespace chase {
namespace {

struct PeerFlags {
    uint32_t *p[CHASE_MAX_RANKS];
};

// Release-store `seq` into slot `rank` of every rank's flag array (own included).
__global__ void rows_signal_kernel(PeerFlags peers, int nranks, int rank, uint32_t seq) {
    if ((int)threadIdx.x < nranks) {
        __threadfence_system();
        asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(peers.p[threadIdx.x] + rank), "r"(seq) : "memory");
    }
}

__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// Wait until every slot of the local flag array has reached `seq`.  A dead or slow peer must neither
// hang the GPU nor go unnoticed: after `timeout_ns` of polling the kernel stores `seq` into the STICKY
// status word flags[nranks] (first failure wins) and returns; once the word is set, later waits return
// at once, so a failed exchange costs one timeout, and chase_rows_status reports it to the host.
__global__ void rows_wait_kernel(uint32_t *flags, int nranks, uint32_t seq, unsigned long long timeout_ns) {
    uint32_t *status = flags + nranks;
    if ((int)threadIdx.x < nranks) {
        const unsigned long long t0 = global_ns();
        for (;;) {
            uint32_t v;
            asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(flags + threadIdx.x) : "memory");
            if ((int)(v - seq) >= 0) break;
            if (*(volatile uint32_t *)status != 0u) break;                 // an earlier barrier already failed
            if (global_ns() - t0 > timeout_ns) {
                atomicCAS(status, 0u, seq ? seq : 0xFFFFFFFFu);
                break;
            }
            __nanosleep(200);
        }
    }
    __syncthreads();
}

unsigned long long rows_timeout_ns() {
    const char *env = std::getenv("CHASE_ROWS_TIMEOUT_MS");
    long long ms = 30000;
    if (env && env[0]) {
        char *end = nullptr;
        const long long v = std::strtoll(env, &end, 10);
        if (end != env && v > 0) ms = v;
    }
    return (unsigned long long)ms * 1000000ull;
}

size_t elem_size(chase_dtype_t dtype) { return dtype == CHASE_C128 ? 16 : 8; }

bool rows_supported(int64_t N, int64_t nrows, chase_dtype_t dtype) {
    const int64_t g = dtype == CHASE_C128 ? 8 : 16;
    return (dtype == CHASE_C128 || dtype == CHASE_F64) && N % g == 0 && nrows % g == 0 && N >= 16;
}

int check_rows_args(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, int64_t ncols, chase_dtype_t dtype) {
    if (dtype != CHASE_F32 && dtype != CHASE_F64 && dtype != CHASE_C64 && dtype != CHASE_C128) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > ((int64_t)1 << 28) || ncols > ((int64_t)1 << 28)) return CHASE_ERR_ARG;
    if (row0 < 0 || nrows <= 0 || row0 + nrows > N || !H_loc) return CHASE_ERR_ARG;
    if (!rows_supported(N, nrows, dtype)) return CHASE_ERR_ALIGN;
    return CHASE_OK;
}

}  // namespace
}  // namespace chase

using namespace chase;

extern "C" {

int chase_hemm_rows(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, const void *X, void *Y,
                    int64_t ncols, double alpha, double beta, double shift, chase_dtype_t dtype,
                    int32_t npeers, void *const *peer_Y, void *stream_) {
    int rc = check_rows_args(H_loc, N, row0, nrows, ncols, dtype);
    if (rc != CHASE_OK) return rc;
    if (npeers < 0 || npeers > CHASE_MAX_RANKS - 1 || (npeers > 0 && !peer_Y)) return CHASE_ERR_ARG;
    if (ncols > 0 && (!X || !Y || X == Y)) return CHASE_ERR_ARG;
    if (!(std::isfinite(alpha) && std::isfinite(beta) && std::isfinite(shift))) return CHASE_ERR_ARG;
    if (ncols == 0) return CHASE_OK;
    if (((uintptr_t)H_loc | (uintptr_t)X | (uintptr_t)Y) & 15) return CHASE_ERR_ALIGN;
    DmmaPlan plan;
    cudaError_t e = dmma_plan_create_rows(&plan, dtype, H_loc, N, row0, nrows, const_cast<void *>(X), Y, ncols);
    if (e != cudaSuccess) return (int)e;
    plan.npeers = npeers;
    for (int q = 0; q < npeers; ++q) {
        if (!peer_Y[q] || ((uintptr_t)peer_Y[q] & 15)) return CHASE_ERR_ARG;
        plan.peer_buf[1][q] = peer_Y[q];      // the step writes buffer 1 (src = 0)
        plan.peer_buf[0][q] = nullptr;
    }
    return (int)dmma_launch_step(&plan, 0, 0, alpha, beta, shift, beta != 0.0, (cudaStream_t)stream_);
}

static int fill_peer_flags(PeerFlags &pf, uint32_t *flags, uint32_t *const *peer_flags, int32_t nranks, int32_t rank) {
    if (!flags || !peer_flags || nranks < 1 || nranks > CHASE_MAX_RANKS || rank < 0 || rank >= nranks)
        return CHASE_ERR_ARG;
    for (int q = 0; q < nranks; ++q) {
        pf.p[q] = q == rank ? flags : peer_flags[q];
        if (!pf.p[q]) return CHASE_ERR_ARG;
    }
    return CHASE_OK;
}

int chase_rows_signal(uint32_t *flags, uint32_t *const *peer_flags, int32_t nranks, int32_t rank, uint32_t seq,
                      void *stream_) {
    PeerFlags pf;
    int rc = fill_peer_flags(pf, flags, peer_flags, nranks, rank);
    if (rc != CHASE_OK) return rc;
    rows_signal_kernel<<<1, 32, 0, (cudaStream_t)stream_>>>(pf, nranks, rank, seq);
    count_launch();
    return (int)cudaGetLastError();
}

int chase_rows_wait(uint32_t *flags, int32_t nranks, uint32_t seq, void *stream_) {
    if (!flags || nranks < 1 || nranks > CHASE_MAX_RANKS) return CHASE_ERR_ARG;
    rows_wait_kernel<<<1, 32, 0, (cudaStream_t)stream_>>>(flags, nranks, seq, rows_timeout_ns());
    count_launch();
    return (int)cudaGetLastError();
}

int chase_rows_barrier(uint32_t *flags, uint32_t *const *peer_flags, int32_t nranks, int32_t rank, uint32_t seq,
                       void *stream_) {
    int rc = chase_rows_signal(flags, peer_flags, nranks, rank, seq, stream_);
    if (rc != CHASE_OK) return rc;
    return chase_rows_wait(flags, nranks, seq, stream_);
}

int chase_rows_status(const uint32_t *flags, int32_t nranks, void *stream_) {
    if (!flags || nranks < 1 || nranks > CHASE_MAX_RANKS) return CHASE_ERR_ARG;
    cudaStream_t stream = (cudaStream_t)stream_;
    uint32_t status = 0;
    cudaError_t e = cudaMemcpyAsync(&status, flags + nranks, sizeof(status), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return (int)e;
    return status == 0 ? CHASE_OK : CHASE_ERR_TIMEOUT;
}

int chase_filter_rows_hostsync_ws(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, void *V, int64_t ncols,
                                  const int32_t *degrees, double a, double b, double lambda1, chase_dtype_t dtype,
                                  void *workspace, size_t workspace_bytes, int32_t nranks, int32_t rank,
                                  void *const *peer_V, void *const *peer_W, uint32_t *flags,
                                  uint32_t *const *peer_flags, uint32_t *seq, void *stream_,
                                  int (*host_barrier)(void *), void *host_ctx) {
    cudaStream_t stream = (cudaStream_t)stream_;
    int rc = check_rows_args(H_loc, N, row0, nrows, ncols, dtype);
    if (rc != CHASE_OK) return rc;
    if (nranks < 1 || nranks > CHASE_MAX_RANKS || rank < 0 || rank >= nranks) return CHASE_ERR_ARG;
    if (nranks > 1 && (!peer_V || !peer_W)) return CHASE_ERR_ARG;
    if (flags && (!peer_flags || !seq)) return CHASE_ERR_ARG;
    if (host_barrier && !flags) return CHASE_ERR_ARG;
    if (ncols > 0 && (!V || !degrees)) return CHASE_ERR_ARG;
    if (!(std::isfinite(a) && std::isfinite(b) && std::isfinite(lambda1))) return CHASE_ERR_BOUNDS;
    if (!(lambda1 < a && a < b)) return CHASE_ERR_BOUNDS;
    const int m_max = chase_filter_schedule(degrees, ncols, nullptr);
    if (m_max < 0) return m_max;
    if (ncols == 0 || m_max == 0) return CHASE_OK;
    const size_t w = elem_size(dtype);
    if (!workspace || workspace_bytes < (size_t)N * (size_t)ncols * w) return CHASE_ERR_WORKSPACE;   // one vector block
    if (((uintptr_t)H_loc | (uintptr_t)V | (uintptr_t)workspace) & 15) return CHASE_ERR_ALIGN;

    int32_t offset[CHASE_MAX_DEGREE + 1];
    double alpha[CHASE_MAX_DEGREE + 1], beta[CHASE_MAX_DEGREE + 1];
    double c = 0.0;
    chase_filter_schedule(degrees, ncols, offset);
    rc = chase_filter_scalars(a, b, lambda1, m_max, alpha, beta, &c);
    if (rc != CHASE_OK) return rc;

    DmmaPlan plan;
    cudaError_t e = dmma_plan_create_rows(&plan, dtype, H_loc, N, row0, nrows, V, workspace, ncols);
    if (e != cudaSuccess) return (int)e;
    plan.npeers = nranks - 1;
    for (int q = 0, i = 0; q < nranks; ++q) {
        if (q == rank) continue;
        if (!peer_V[q] || !peer_W[q] || (((uintptr_t)peer_V[q] | (uintptr_t)peer_W[q]) & 15)) return CHASE_ERR_ARG;
        plan.peer_buf[0][i] = peer_V[q];
        plan.peer_buf[1][i] = peer_W[q];
        ++i;
    }
    // One inter-GPU barrier: signal on the stream; then either the device-side wait (one GPU per rank, the
    // ranks' kernels run concurrently) or, with a host barrier (ranks that time-share a GPU, where a
    // spinning wait kernel would keep the peer's kernels from running): drain the stream, meet the other
    // ranks on the host, and enqueue the wait, which then finds every flag already set.
    auto sync_ranks = [&]() -> int {
        if (!flags) return CHASE_OK;
        const uint32_t s = ++*seq;
        int r = chase_rows_signal(flags, peer_flags, nranks, rank, s, stream_);
        if (r != CHASE_OK) return r;
        if (host_barrier) {
            cudaError_t es = cudaStreamSynchronize(stream);
            if (es != cudaSuccess) return (int)es;
            if (host_barrier(host_ctx) != 0) return CHASE_ERR_TIMEOUT;
        }
        return chase_rows_wait(flags, nranks, s, stream_);
    };
    // Before step 1 overwrites the peers' scratch rows, every rank must have entered the call
    // (its previous use of the scratch buffer is over) -- and after each step k every rank must have
    // finished it: all rows of V_k have landed everywhere and nobody still reads V_{k-1}.
    if ((rc = sync_ranks()) != CHASE_OK) return rc;
    for (int k = 1; k <= m_max; ++k) {
        e = dmma_launch_step(&plan, (k - 1) & 1, offset[k], alpha[k], beta[k], c, k > 1, stream);
        if (e != cudaSuccess) return (int)e;
        if ((rc = sync_ranks()) != CHASE_OK) return rc;
    }
    // odd-degree columns ended in the scratch buffer, which is complete on every rank: local copy back
    const size_t col_bytes = (size_t)N * w;
    for (int64_t j = 0; j < ncols;) {
        if ((degrees[j] & 1) == 0) { ++j; continue; }
        int64_t j1 = j;
        while (j1 < ncols && (degrees[j1] & 1)) ++j1;
        e = cudaMemcpyAsync((char *)V + (size_t)j * col_bytes, (const char *)workspace + (size_t)j * col_bytes,
                            (size_t)(j1 - j) * col_bytes, cudaMemcpyDeviceToDevice, stream);
        if (e != cudaSuccess) return (int)e;
        j = j1;
    }
    return CHASE_OK;
}

int chase_filter_rows_ws(const void *H_loc, int64_t N, int64_t row0, int64_t nrows, void *V, int64_t ncols,
                         const int32_t *degrees, double a, double b, double lambda1, chase_dtype_t dtype,
                         void *workspace, size_t workspace_bytes, int32_t nranks, int32_t rank,
                         void *const *peer_V, void *const *peer_W, uint32_t *flags,
                         uint32_t *const *peer_flags, uint32_t *seq, void *stream_) {
    return chase_filter_rows_hostsync_ws(H_loc, N, row0, nrows, V, ncols, degrees, a, b, lambda1, dtype, workspace,
                                         workspace_bytes, nranks, rank, peer_V, peer_W, flags, peer_flags, seq,
                                         stream_, nullptr, nullptr);
}

int chase_ipc_export(const void *dev_ptr, void *handle64, int64_t *offset) {
    if (!dev_ptr || !handle64 || !offset) return CHASE_ERR_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
    void *base = nullptr;
    size_t size = 0;
    // cudaIpcGetMemHandle refers to the whole allocation; find where dev_ptr sits inside it
    CUresult (*get_range)(CUdeviceptr_v2 *, size_t *, CUdeviceptr_v2) = nullptr;
    cudaDriverEntryPointQueryResult q;
    void *fn = nullptr;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return (int)cudaErrorNotSupported;
    get_range = (decltype(get_range))fn;
    CUdeviceptr_v2 b = 0;
    if (get_range(&b, &size, (CUdeviceptr_v2)(uintptr_t)dev_ptr) != CUDA_SUCCESS) return (int)cudaErrorInvalidValue;
    base = (void *)(uintptr_t)b;
    cudaIpcMemHandle_t h;
    cudaError_t e = cudaIpcGetMemHandle(&h, base);
    if (e != cudaSuccess) return (int)e;
    std::memcpy(handle64, &h, 64);
    *offset = (int64_t)((const char *)dev_ptr - (const char *)base);
    return CHASE_OK;
}

int chase_ipc_open(const void *handle64, void **base_out) {
    if (!handle64 || !base_out) return CHASE_ERR_ARG;
    cudaIpcMemHandle_t h;
    std::memcpy(&h, handle64, 64);
    return (int)cudaIpcOpenMemHandle(base_out, h, cudaIpcMemLazyEnablePeerAccess);
}

int chase_ipc_close(void *base) {
    if (!base) return CHASE_ERR_ARG;
    return (int)cudaIpcCloseMemHandle(base);
}

}  // extern "C"

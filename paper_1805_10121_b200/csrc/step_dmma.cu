// placeholder until the TMA + DMMA kernel lands
#include "chase_internal.h"
namespace chase {
bool dmma_supported(int64_t, int64_t, chase_dtype_t) { return false; }
cudaError_t dmma_plan_create(DmmaPlan *, chase_dtype_t, const void *, int64_t, void *, void *, int64_t) { return cudaErrorNotSupported; }
cudaError_t dmma_launch_step(const DmmaPlan *, int, int64_t, double, double, double, int, cudaStream_t) { return cudaErrorNotSupported; }
}

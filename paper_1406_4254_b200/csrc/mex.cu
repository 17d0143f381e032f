// mex.cu — MEX half of the hot path (placeholder until the kernels land; returns cudaErrorNotSupported).
#include "etics_common.cuh"

namespace etics {
cudaError_t mex_init_constants() { return cudaSuccess; }
size_t mex_workspace(long long, int) { return 256; }
cudaError_t mex_sort_launch(const double*, long long, unsigned long long*, unsigned int*, void*, cudaStream_t) { return cudaErrorNotSupported; }
cudaError_t mex_force_launch(const double*, const double*, long long, int, double*, double*, void*, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace etics

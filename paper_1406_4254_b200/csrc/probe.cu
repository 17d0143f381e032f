// probe.cu — roofline probes (measurement support; MEASURED_PEAKS.json has no fp64 entry,
// so a register-resident DFMA loop supplies the fp64 denominator).  Not part of the method.
#include "etics_common.cuh"

namespace etics {

constexpr int kProbeThreads = 256;
constexpr int kProbeChains = 16;     // independent FMA chains per thread
constexpr int kProbeBlocksPerSM = 4;

__global__ void __launch_bounds__(kProbeThreads)
probe_dfma_kernel(int iters, double* __restrict__ sink) {
    double v[kProbeChains];
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * blockIdx.x;
#pragma unroll
    for (int i = 0; i < kProbeChains; ++i) v[i] = 0.5 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kProbeChains; ++i) v[i] = fma(v[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kProbeChains; ++i) s += v[i];
    if (s == 123.456) sink[0] = s;   // never true; keeps the chains alive
}

cudaError_t probe_dfma_launch(int iters, double* sink, double* flops_out, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const int blocks = sms * kProbeBlocksPerSM;
    if (flops_out) *flops_out = 2.0 * (double)iters * kProbeChains * kProbeThreads * blocks;
    probe_dfma_kernel<<<blocks, kProbeThreads, 0, st>>>(iters, sink);
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256)
probe_copy_kernel(const double2* __restrict__ src, double2* __restrict__ dst, size_t n) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = src[i];
}

cudaError_t probe_copy_launch(void* dst, const void* src, size_t bytes, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    probe_copy_kernel<<<sms * 16, 256, 0, st>>>(static_cast<const double2*>(src), static_cast<double2*>(dst), bytes / 16);
    return cudaGetLastError();
}

}  // namespace etics

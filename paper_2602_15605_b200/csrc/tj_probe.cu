// tj_probe.cu -- DFMA-chain microbenchmark: the measured denominator of the FP64 roofline.
// 16 independent dependent-chains per thread keep the FP64 pipe full from registers alone.
#include "tj_internal.cuh"

namespace tj {
namespace {

__global__ void __launch_bounds__(256) fp64_probe_kernel(int iters, double *sink)
{
    double x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = 1.0 + 1e-9 * (double)(threadIdx.x + k);
    const double m = 0.9999999, b = 1e-7;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) x[k] = __fma_rn(x[k], m, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

cudaError_t launch_fp64_probe(int iters, double *d_sink, int blocks, int threads, cudaStream_t st)
{
    fp64_probe_kernel<<<blocks, threads, 0, st>>>(iters, d_sink);
    return cudaGetLastError();
}

}  // namespace tj

// bench_gpu/fp64_probe.cu -- BENCH-ONLY: DFMA-chain microbenchmark, the measured denominator of the FP64 roofline
// ("the build must measure it with a register-resident DFMA-chain microbenchmark, >= 1 s").
// Not part of libtj: bench.py is its only caller.  16 independent dependent chains per thread keep the FP64 pipe full
// from registers alone; 256 threads per CTA, 4 CTAs per SM (32 warps/SM).
#include <cuda_runtime.h>

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

// Runs `iters` loop iterations (16 DFMA each, per thread) on every SM of the current device, on `cuda_stream`
// (cudaStream_t as void*), after a warm-up launch of iters/8; synchronous, CUDA-event timed.
// *h_thread_instr_per_s = achieved FP64 thread-instructions per second.  Returns 0, or the cudaError_t that failed.
extern "C" int probe_fp64(int iters, void *cuda_stream, double *h_thread_instr_per_s)
{
    if (iters <= 0 || !h_thread_instr_per_s) return (int)cudaErrorInvalidValue;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    const int threads = 256, blocks = sms * 4;
    double *sink = nullptr;
    e = cudaMalloc((void **)&sink, sizeof(double) * (size_t)blocks * threads);
    if (e != cudaSuccess) return (int)e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    fp64_probe_kernel<<<blocks, threads, 0, st>>>(iters / 8 + 1, sink);   // warm-up
    cudaEventRecord(e0, st);
    fp64_probe_kernel<<<blocks, threads, 0, st>>>(iters, sink);
    e = cudaGetLastError();
    cudaEventRecord(e1, st);
    cudaError_t es = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return (int)e;
    if (es != cudaSuccess) return (int)es;
    *h_thread_instr_per_s = 16.0 * (double)iters * (double)blocks * (double)threads / ((double)ms * 1e-3);
    return 0;
}

// bench_kernels.cu -- measurement aid: sustained FP64 FMA throughput of the device (register-only
// DFMA chains, 8 independent chains per thread, 32 warps per SM), the denominator of the "alu"
// roofline bench.py reports.  Not part of the ERI path.
#include "../../include/rcg.h"
#include <cuda_runtime.h>
#include "rcg_internal.h"

__global__ void __launch_bounds__(256) rcg_dfma_kernel(double *out, int iters, double a, double b)
{
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 123.456) out[0] = s;
}

extern "C" rcg_status rcg_fp64_peak_tflops(double *tflops, void *stream)
{
    if (!tflops) return RCG_ERR_INVALID_ARG;
    int dev = 0, nsm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    double *d = nullptr;
    if (e == cudaSuccess) e = cudaMalloc((void **)&d, 64);
    if (e != cudaSuccess) return rcg_cuda_fail(e);
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 20000, blocks = nsm * 4, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        rcg_dfma_kernel<<<blocks, threads, 0, st>>>(d, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        double tf = 2.0 * 8 * iters * (double)blocks * threads / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    if (e != cudaSuccess) return rcg_cuda_fail(e);
    *tflops = best;
    return RCG_OK;
}

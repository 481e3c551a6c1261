// fma_peak.cu -- heget_fma_peak: measured non-tensor FMA rate of the device, the roofline
// denominator for the amplitude kernels (product code; MEASURED_PEAKS.json holds only HBM and
// tensor-core figures).  Every thread runs 16 independent FMA chains so that neither the FMA
// latency nor register-bank conflicts limit the issue rate; enough CTAs to fill every SM.
#include "heget_internal.cuh"

namespace {

template <typename T>
__global__ void __launch_bounds__(256)
fma_peak_kernel(T* __restrict__ sink, int iters, T a, T b)
{
    T x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = (T)(threadIdx.x + k) * (T)1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep)
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = x[k] * a + b;
    }
    T s = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    if (s == (T)12345.678) sink[0] = s;  // never true; keeps the chains alive
}

template <typename T>
cudaError_t run(const heget_ctx* ctx, double* flops_per_s, int* launches)
{
    T* sink = nullptr;
    cudaError_t err = cudaMalloc(&sink, sizeof(T));
    if (err != cudaSuccess) return err;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = ctx->sm_count * 8, threads = 256;
    const int iters = (sizeof(T) == 4) ? 16384 : 8192;
    double best = 0.0;
    for (int trial = 0; trial < 4; ++trial) {
        cudaEventRecord(t0, 0);
        fma_peak_kernel<T><<<blocks, threads>>>(sink, iters, (T)0.999, (T)1e-3);
        cudaEventRecord(t1, 0);
        err = cudaEventSynchronize(t1);
        ++*launches;
        if (err != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        const double flops = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;
        const double rate = flops / (ms * 1e-3);
        if (trial > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    *flops_per_s = best;
    return err;
}

}  // namespace

cudaError_t heget_run_fma_peak(const heget_ctx* ctx, int precision, double* flops_per_s, int* launches)
{
    *launches = 0;
    if (precision == HEGET_FP32) return run<float>(ctx, flops_per_s, launches);
    return run<double>(ctx, flops_per_s, launches);
}

// fma_peak.cu -- heget_fma_peak: measured non-tensor FMA rate of the device, the roofline
// denominator for the amplitude kernels (product code; MEASURED_PEAKS.json holds only HBM and
// tensor-core figures).  Every thread runs 16 independent FMA chains so that the FMA latency
// does not limit the issue rate; enough CTAs to fill every SM.  Three operand patterns:
//   0  x = x*a + b with a, b kernel arguments (constant-bank operands): the pipe's own peak;
//   1  x = y*z + x with three distinct register operands and no operand shared by consecutive
//      FMAs: what the register file sustains (measured 2/3 of pattern 0 in fp32 on B200);
//   2  the fvixx0 node of amp2.cu (psi' = P (E' psi), 16 FMA + 4 MUL) on register-held
//      operands: the practical ceiling of the amplitude kernels' own instruction mix.
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
__global__ void __launch_bounds__(256)
fma_3reg_kernel(T* __restrict__ sink, const T* __restrict__ in, int iters)
{
    T x[16], y[16], z[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        x[k] = in[threadIdx.x + k];
        y[k] = in[threadIdx.x + 16 + k];
        z[k] = in[threadIdx.x + 32 + k];
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep)
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = fma(y[k], z[(k + rep) & 15], x[k]);
    }
    T s = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    if (s == (T)12345.678) sink[0] = s;
}

template <typename T>
__global__ void __launch_bounds__(256)
fma_node_kernel(T* __restrict__ sink, const T* __restrict__ in, int iters)
{
    T e[4][4], p[4][4], f[4];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            e[m][c] = in[threadIdx.x + 4 * m + c];
            p[m][c] = in[threadIdx.x + 64 + 4 * m + c];
        }
#pragma unroll
    for (int c = 0; c < 4; ++c) f[c] = in[threadIdx.x + 128 + c];
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const T w0r = fma(-e[m][2], f[2], fma(e[m][3], f[3], -f[0]));
            const T w0i = fma(-e[m][2], f[3], fma(-e[m][3], f[2], -f[1]));
            const T w1r = fma(e[m][0], f[0], fma(-e[m][1], f[1], f[2]));
            const T w1i = fma(e[m][0], f[1], fma(e[m][1], f[0], f[3]));
            f[0] = fma(p[m][0], w0r, fma(p[m][2], w1r, p[m][3] * w1i));
            f[1] = fma(p[m][0], w0i, fma(p[m][2], w1i, -(p[m][3] * w1r)));
            f[2] = fma(p[m][1], w1r, fma(p[m][2], w0r, -(p[m][3] * w0i)));
            f[3] = fma(p[m][1], w1i, fma(p[m][2], w0i, p[m][3] * w0r));
        }
    }
    const T s = f[0] + f[1] + f[2] + f[3];
    if (s == (T)12345.678) sink[0] = s;
}

template <typename T>
cudaError_t run(const heget_ctx* ctx, int pattern, double* flops_per_s, int* launches)
{
    T* sink = nullptr;
    cudaError_t err = cudaMalloc(&sink, sizeof(T) * 1024);
    if (err != cudaSuccess) return err;
    {   // operands of patterns 1, 2: non-trivial values of order one (all-zero data would toggle fewer bits,
        // draw less power and could clock higher than real operands do), contracting so the chains stay finite
        T host[1024];
        for (int i = 0; i < 1024; ++i) host[i] = (T)(0.25 + 0.5 * ((i * 2654435761u) % 1000) / 1000.0) * ((i & 1) ? (T)1 : (T)-1);
        err = cudaMemcpy(sink, host, sizeof(host), cudaMemcpyHostToDevice);
        if (err != cudaSuccess) { cudaFree(sink); return err; }
    }
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = ctx->sm_count * 8, threads = 256;
    const int iters = (sizeof(T) == 4) ? 16384 : 8192;
    double best = 0.0;
    for (int trial = 0; trial < 4; ++trial) {
        cudaEventRecord(t0, 0);
        if (pattern == 0)
            fma_peak_kernel<T><<<blocks, threads>>>(sink, iters, (T)0.999, (T)1e-3);
        else if (pattern == 1)
            fma_3reg_kernel<T><<<blocks, threads>>>(sink, sink, iters);
        else
            fma_node_kernel<T><<<blocks, threads>>>(sink, sink, iters);
        cudaEventRecord(t1, 0);
        err = cudaEventSynchronize(t1);
        ++*launches;
        if (err != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        // flops per thread and iteration: 64 FMA (patterns 0, 1); 4 nodes x (16 FMA + 4 MUL) (pattern 2)
        const double per_iter = (pattern == 2) ? 4.0 * 36.0 : 2.0 * 64.0;
        const double flops = per_iter * (double)iters * (double)blocks * (double)threads;
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

cudaError_t heget_run_fma_peak(const heget_ctx* ctx, int precision, int pattern, double* flops_per_s, int* launches)
{
    *launches = 0;
    if (precision == HEGET_FP32) return run<float>(ctx, pattern, flops_per_s, launches);
    return run<double>(ctx, pattern, flops_per_s, launches);
}

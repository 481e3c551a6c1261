// reduce.cu -- heget_xsec_reduce: step 6 of PAPER.md:141 on the device (product code).
// x_e = weight[e] * amp2[e] * (1/4)(1/9)(1/n!)  (eq. 2; 0 where weight[e] == 0);
// out3 = {sum x, sum x^2, #(weight != 0)}.  Fixed reduction tree (grid-stride partials, warp shuffles, one final CTA):
// bit-reproducible from run to run, no floating-point atomics.
#include "heget_internal.cuh"

namespace {

constexpr double kSpinAverage = 1.0 / 4.0;   // 1/2^2 of eq. (2)
constexpr double kColourFactor = 1.0 / 9.0;  // eq. (2)'s garbled 1/3^2 factors, R1

__device__ __forceinline__ void warp_sum3(double& a, double& b, double& c)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, off);
        b += __shfl_xor_sync(0xffffffffu, b, off);
        c += __shfl_xor_sync(0xffffffffu, c, off);
    }
}

__device__ __forceinline__ void block_sum3(double& a, double& b, double& c, double (*sm)[3])
{
    warp_sum3(a, b, c);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sm[warp][0] = a; sm[warp][1] = b; sm[warp][2] = c; }
    __syncthreads();
    if (warp == 0) {
        const int nw = blockDim.x >> 5;
        a = lane < nw ? sm[lane][0] : 0.0;
        b = lane < nw ? sm[lane][1] : 0.0;
        c = lane < nw ? sm[lane][2] : 0.0;
        warp_sum3(a, b, c);
    }
}

__global__ void __launch_bounds__(256)
reduce_partial_kernel(const double* __restrict__ amp2, const double* __restrict__ weight, int64_t n_events,
                      double factor, double* __restrict__ partials)
{
    __shared__ double sm[8][3];
    double s1 = 0.0, s2 = 0.0, cnt = 0.0;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_events;
         e += (int64_t)gridDim.x * blockDim.x) {
        const double w = weight[e];
        // an event that failed the cuts contributes exactly 0 whatever its amp2 holds (R26:
        // a forward photon outside the cuts may have driven amp2 to Inf or NaN, fp32 range included)
        const double x = (w != 0.0) ? w * amp2[e] * factor : 0.0;
        s1 += x;
        s2 += x * x;
        cnt += (w != 0.0) ? 1.0 : 0.0;
    }
    block_sum3(s1, s2, cnt, sm);
    if (threadIdx.x == 0) {
        partials[3 * blockIdx.x + 0] = s1;
        partials[3 * blockIdx.x + 1] = s2;
        partials[3 * blockIdx.x + 2] = cnt;
    }
}

__global__ void __launch_bounds__(256)
reduce_final_kernel(const double* __restrict__ partials, int n_partials, double* __restrict__ out3)
{
    __shared__ double sm[8][3];
    double s1 = 0.0, s2 = 0.0, cnt = 0.0;
    for (int i = threadIdx.x; i < n_partials; i += blockDim.x) {
        s1 += partials[3 * i + 0];
        s2 += partials[3 * i + 1];
        cnt += partials[3 * i + 2];
    }
    block_sum3(s1, s2, cnt, sm);
    if (threadIdx.x == 0) { out3[0] = s1; out3[1] = s2; out3[2] = cnt; }
}

// ---- no-allocation variant (heget_xsec_reduce_noalloc) ---------------------------------------------------------
// For callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it) and do not
// want a context-owned buffer either: the block partials live in a file-scope device array.  One block per chunk
// of kNoAllocChunk events (no grid stride), one partial triple per block, so the scratch bounds the batch:
// HEGET_NOALLOC_MAX_EVENTS = kNoAllocMaxBlocks * kNoAllocChunk.  Every GPU that loads the library holds the
// 96 KB until exit.  All calls share the array and it keeps the last call's contents: a call writes partials
// [0, blocks) before its final kernel reads exactly those, so nothing has to start at zero -- but two calls
// that overlap on the GPU (different streams, or graphs launched concurrently) race on it.
constexpr int kNoAllocChunk = 256 * 16;                                          // events per block
constexpr int kNoAllocMaxBlocks = (int)(HEGET_NOALLOC_MAX_EVENTS / kNoAllocChunk);  // 4096
static_assert((int64_t)kNoAllocMaxBlocks * kNoAllocChunk == HEGET_NOALLOC_MAX_EVENTS, "the maximum is a whole number of chunks");
static __device__ __align__(256) double g_noalloc_partials[kNoAllocMaxBlocks * 3];

__global__ void __launch_bounds__(256)
reduce_partial_noalloc_kernel(const double* __restrict__ amp2, const double* __restrict__ weight, int64_t n_events,
                              double factor, double* __restrict__ partials)
{
    __shared__ double sm[8][3];
    double s1 = 0.0, s2 = 0.0, cnt = 0.0;
    const int64_t lo = (int64_t)blockIdx.x * kNoAllocChunk;
#pragma unroll 4
    for (int k = 0; k < kNoAllocChunk / 256; ++k) {
        const int64_t e = lo + k * 256 + threadIdx.x;
        if (e < n_events) {
            const double w = weight[e];
            const double x = (w != 0.0) ? w * amp2[e] * factor : 0.0;   // DESIGN.md R26, as reduce_partial_kernel
            s1 += x;
            s2 += x * x;
            cnt += (w != 0.0) ? 1.0 : 0.0;
        }
    }
    block_sum3(s1, s2, cnt, sm);
    if (threadIdx.x == 0) {
        partials[3 * blockIdx.x + 0] = s1;
        partials[3 * blockIdx.x + 1] = s2;
        partials[3 * blockIdx.x + 2] = cnt;
    }
}

// In host code `g_noalloc_partials` is a host-side stand-in, not a device address: the address a kernel can use
// comes from cudaGetSymbolAddress, resolved once per device with that device current.
constexpr int kMaxDevices = 64;
double* g_noalloc_addr[kMaxDevices] = {};

}  // namespace

cudaError_t heget_launch_reduce_noalloc(int device, const double* amp2, const double* weight, int n, int64_t N,
                                        double* out3, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    double* partials = g_noalloc_addr[device];
    if (!partials) {   // set-up, once per device (the caller made `device` current); benign if two threads race: same value
        void* p = nullptr;
        const cudaError_t err = cudaGetSymbolAddress(&p, g_noalloc_partials);
        if (err != cudaSuccess) return err;
        g_noalloc_addr[device] = partials = static_cast<double*>(p);
    }
    double nfact = 1.0;
    for (int i = 2; i <= n; ++i) nfact *= (double)i;
    const double factor = kSpinAverage * kColourFactor / nfact;
    const int blocks = (int)((N + kNoAllocChunk - 1) / kNoAllocChunk);   // <= kNoAllocMaxBlocks, checked by the caller
    if (blocks > 0) {
        reduce_partial_noalloc_kernel<<<blocks, 256, 0, stream>>>(amp2, weight, N, factor, partials);
        const cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
        ++*launches;
    }
    reduce_final_kernel<<<1, 256, 0, stream>>>(partials, blocks, out3);   // blocks = 0: writes {0, 0, 0}
    ++*launches;
    return cudaGetLastError();
}

cudaError_t heget_launch_reduce(double* partials, const double* amp2, const double* weight, int n,
                                int64_t N, double* out3, cudaStream_t stream, int* launches)
{
    double nfact = 1.0;
    for (int i = 2; i <= n; ++i) nfact *= (double)i;
    const double factor = kSpinAverage * kColourFactor / nfact;
    *launches = 2;
    reduce_partial_kernel<<<kReduceBlocks, 256, 0, stream>>>(amp2, weight, N, factor, partials);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    reduce_final_kernel<<<1, 256, 0, stream>>>(partials, kReduceBlocks, out3);
    return cudaGetLastError();
}

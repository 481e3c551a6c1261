// hist.cu -- heget_histogram: the kinematical distributions of Fig. 2 on the
// device (product code).  The paper sums "the total cross section and
// distributions on the CPU" (step 6); here the weighted histograms of the maximum
// photon pT and of the Delta R separation of eq. (10) are filled where the
// momenta and weights already are.
//
// One thread per event; the CTA accumulates into a shared-memory histogram with fp64 atomics and
// flushes its non-empty bins to the output with global fp64 atomics.  The order of the atomic
// additions is not fixed, so two runs may differ in the last bits of a bin (relative ~1e-16 per
// addition); bin ASSIGNMENT is deterministic.  Binning convention: DESIGN.md R23.
#include "heget_internal.cuh"

namespace {

__device__ __forceinline__ int bin_of(double x, double lo, double hi, int nbins)
{
    // slot 0 = underflow, 1..nbins = bins on [lo, hi), nbins + 1 = overflow (also NaN)
    if (x < lo) return 0;
    if (!(x < hi)) return nbins + 1;
    int b = (int)floor((x - lo) / (hi - lo) * nbins);
    if (b >= nbins) b = nbins - 1;
    return 1 + b;
}

__global__ void __launch_bounds__(256)
hist_kernel(const double* __restrict__ momenta, const double* __restrict__ value, int n, int64_t n_events,
            int observable, double lo, double hi, int nbins, double* __restrict__ hist)
{
    extern __shared__ double s_hist[];
    const double pi = 3.14159265358979323846;
    for (int b = threadIdx.x; b < nbins + 2; b += blockDim.x) s_hist[b] = 0.0;
    __syncthreads();
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_events;
         e += (int64_t)gridDim.x * blockDim.x) {
        const double v = value[e];
        if (v == 0.0) continue;  // events that failed the cuts carry no weight
        const double2* k = reinterpret_cast<const double2*>(momenta + e * 4 * (n + 2) + 8);
        double pt[8], eta[8], phi[8];
        double ptmax = 0.0;
        for (int i = 0; i < n; ++i) {
            const double2 a = k[2 * i], b = k[2 * i + 1];  // (E, px), (py, pz)
            pt[i] = sqrt(a.y * a.y + b.x * b.x);
            eta[i] = asinh(b.y / pt[i]);
            phi[i] = atan2(b.x, a.y);
            ptmax = fmax(ptmax, pt[i]);
        }
        if (observable == HEGET_OBS_PT_MAX) {
            atomicAdd(&s_hist[bin_of(ptmax, lo, hi, nbins)], v);
        } else {
            double best = INFINITY;
            for (int i = 0; i < n; ++i)
                for (int j = i + 1; j < n; ++j) {
                    const double deta = eta[i] - eta[j];
                    double dphi = fabs(phi[i] - phi[j]);
                    if (dphi > pi) dphi = 2.0 * pi - dphi;
                    const double dr = sqrt(deta * deta + dphi * dphi);
                    if (observable == HEGET_OBS_DR_ALL) atomicAdd(&s_hist[bin_of(dr, lo, hi, nbins)], v);
                    best = fmin(best, dr);
                }
            if (observable == HEGET_OBS_DR_MIN) atomicAdd(&s_hist[bin_of(best, lo, hi, nbins)], v);
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins + 2; b += blockDim.x)
        if (s_hist[b] != 0.0) atomicAdd(&hist[b], s_hist[b]);
}

}  // namespace

cudaError_t heget_launch_histogram(const heget_ctx* ctx, const double* momenta, const double* value, int n,
                                   int64_t N, int observable, double lo, double hi, int nbins, double* hist,
                                   cudaStream_t stream, int* launches)
{
    *launches = 0;
    cudaError_t err = cudaMemsetAsync(hist, 0, sizeof(double) * (size_t)(nbins + 2), stream);
    if (err != cudaSuccess || N == 0) return err;
    int64_t blocks = (N + 255) / 256;
    const int64_t cap = (int64_t)ctx->sm_count * 8;  // grid-stride beyond 8 CTAs per SM
    if (blocks > cap) blocks = cap;
    hist_kernel<<<(unsigned)blocks, 256, sizeof(double) * (size_t)(nbins + 2), stream>>>(momenta, value, n, N, observable,
                                                                                         lo, hi, nbins, hist);
    *launches = 1;
    return cudaGetLastError();
}

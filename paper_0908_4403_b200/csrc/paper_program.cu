// paper_program.cu -- heget_list2: the paper's OWN amplitude program, List 2,
// generalised from 3 to n photons and run as the paper runs it (product code; the design this
// library is measured against on the same GPU):
//   * one THREAD per event ("a unit program, called a thread, ... calculates the amplitudes for
//     one event"), 256 threads per block (the paper's best block size);
//   * one helicity assignment per event, drawn from random numbers -- the same
//     Philox draw as heget_amp2_sampled, so the two return the same estimator 4*2^n*|M(h)|^2;
//   * 4-component HEGET functions on cmplx w[6] (helas.cuh): ixxxx1 for u, oxxxx2 (nSF = -1) for
//     ubar, vxxxx0 for every photon, then for every permutation n-1 fvoxx0 chained from the ubar
//     line and one iovxxx, ampsum += amp, with iPNext stepping through the n! orderings
//     (lexicographic; the paper does not state the order, R9);
//   * no prefix reuse, no propagator table, no two-component form.
// One deviation, forced by fp32's range (|M|^2 ~ s_hat^(2-n) leaves it for n >= 7):
// the fp32 instantiation divides the momenta by sqrt(s_hat) on load and restores s_hat^(2-n) in
// fp64 at the store, as the other fp32 kernels of this library do.
#include "helas.cuh"
#include "heget_internal.cuh"
#include "philox.cuh"

namespace {

constexpr uint32_t kHelicitySlot = 15u;  // as amp2_sampled.cu (R21)

// next permutation in lexicographic order; false after the last one (iPNext)
template <int N>
__device__ __forceinline__ bool ipnext(int* a)
{
    int i = N - 2;
    while (i >= 0 && a[i] > a[i + 1]) --i;
    if (i < 0) return false;
    int j = N - 1;
    while (a[j] < a[i]) --j;
    int t = a[i]; a[i] = a[j]; a[j] = t;
    for (int l = i + 1, r = N - 1; l < r; ++l, --r) { t = a[l]; a[l] = a[r]; a[r] = t; }
    return true;
}

// List 2 for one event and one helicity assignment `bits` (bit k: particle k in the order u,
// ubar, gamma_1..gamma_n; 1 -> +1): returns |ampsum|^2 in the units of p.
template <int N, typename T>
__device__ __forceinline__ double list2_program(const T (&p)[N + 2][4], uint32_t bits, T gau)
{
    cmplx<T> w[N + 2][6];
#pragma unroll
    for (int k = 0; k < N + 2; ++k) {
        const int nh = ((bits >> k) & 1u) ? +1 : -1;
        if (k == 0) ixxxx1(p[0], nh, +1, w[0]);
        else if (k == 1) oxxxx2(p[1], nh, -1, w[1]);
        else vxxxx0(p[k], nh, +1, w[k]);
    }
    cmplx<T> ampsum = mkcmplx((T)0, (T)0);
    int a[N];
#pragma unroll
    for (int k = 0; k < N; ++k) a[k] = 2 + k;
    do {
        cmplx<T> wa[6], wb[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) wa[c] = w[1][c];
        for (int l = 0; l < N - 1; ++l) {       // n-1 off-shell fermions chained from the ubar line
            fvoxx0(wa, w[a[l]], gau, wb);
#pragma unroll
            for (int c = 0; c < 6; ++c) wa[c] = wb[c];
        }
        ampsum = ampsum + iovxxx(w[0], wa, w[a[N - 1]], gau);
    } while (ipnext<N>(a));
    return (double)ampsum.re * (double)ampsum.re + (double)ampsum.im * (double)ampsum.im;
}

// SUM = false: one drawn helicity assignment per event (the paper's loop), out = 4 2^n |M(h)|^2.
// SUM = true: the same program called for every one of the 4 2^n assignments, out = sum |M|^2 --
// the paper's arithmetic (SURVEY 8(d) model A) for the quantity heget_amp2 returns.
template <int N, typename T, bool SUM>
__global__ void __launch_bounds__(256)
list2_kernel(const double* __restrict__ momenta, uint64_t seed, uint64_t first_event, double* __restrict__ out,
             int32_t* __restrict__ out_hel, int64_t n_events, double g)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_events) return;
    const double* mom = momenta + e * 4 * (N + 2);
    const double shat = 4.0 * mom[0] * mom[4];
    const double unit = (sizeof(T) == 4) ? 1.0 / sqrt(shat) : 1.0;
    T p[N + 2][4];
#pragma unroll
    for (int k = 0; k < N + 2; ++k)
#pragma unroll
        for (int c = 0; c < 4; ++c) p[k][c] = (T)(mom[4 * k + c] * unit);

    double r;
    uint32_t bits = 0u;
    if constexpr (SUM) {
        r = 0.0;
        for (uint32_t h = 0; h < (4u << N); ++h) r += list2_program<N, T>(p, h, (T)g);
    } else {
        uint32_t x[4];
        const uint64_t gev = first_event + (uint64_t)e;
        philox4x32_10((uint32_t)gev, (uint32_t)(gev >> 32), kHelicitySlot, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), x);
        bits = x[0] & ((1u << (N + 2)) - 1u);
        r = 4.0 * (double)(1 << N) * list2_program<N, T>(p, bits, (T)g);
    }
    if (sizeof(T) == 4) {
        // amplitude ~ (energy)^(2-n): |M|^2 in units of sqrt(s_hat) times s_hat^(2-n)
        const double inv = 1.0 / shat;
#pragma unroll
        for (int i = 0; i < N - 2; ++i) r *= inv;
    }
    out[e] = r;
    if (!SUM && out_hel) out_hel[e] = (int32_t)bits;
}

template <int N, typename T>
cudaError_t launch_one(const double* momenta, uint64_t seed, uint64_t first_event, double* out, int32_t* out_hel,
                       int64_t n_events, double g, bool sum, cudaStream_t stream)
{
    const int64_t blocks = (n_events + 255) / 256;
    if (sum)
        list2_kernel<N, T, true><<<(unsigned)blocks, 256, 0, stream>>>(momenta, seed, first_event, out, out_hel, n_events, g);
    else
        list2_kernel<N, T, false><<<(unsigned)blocks, 256, 0, stream>>>(momenta, seed, first_event, out, out_hel, n_events, g);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_n(int n, const double* momenta, uint64_t seed, uint64_t first_event, double* out,
                     int32_t* out_hel, int64_t n_events, double g, bool sum, cudaStream_t stream)
{
    switch (n) {
        case 2: return launch_one<2, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        case 3: return launch_one<3, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        case 4: return launch_one<4, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        case 5: return launch_one<5, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        case 6: return launch_one<6, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        case 7: return launch_one<7, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        case 8: return launch_one<8, T>(momenta, seed, first_event, out, out_hel, n_events, g, sum, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t heget_launch_list2(const heget_ctx* ctx, uint64_t seed, uint64_t first_event, const double* momenta,
                               int n, int precision, double* out_amp2, int32_t* out_hel, int64_t N, bool sum,
                               cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    if (precision == HEGET_FP32)
        return launch_n<float>(n, momenta, seed, first_event, out_amp2, out_hel, N, ctx->g, sum, stream);
    return launch_n<double>(n, momenta, seed, first_event, out_amp2, out_hel, N, ctx->g, sum, stream);
}

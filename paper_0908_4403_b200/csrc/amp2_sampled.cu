// amp2_sampled.cu -- heget_amp2_sampled: the paper's own event loop (product
// code).  Instead of summing all helicities, every event draws ONE helicity assignment
// (sigma_1, sigma_2, lambda_1..lambda_n) from random numbers ("generate helicities and momenta
// ... using random numbers, and compute squared amplitudes", step 4 of PAPER.md:116-122) and
// returns the unbiased estimator 4 * 2^n * |M(h)|^2 of the helicity sum of eq. (2)
// (PAPER.md:37), together with the bits that were drawn (step 5).
//
// Readings (R21, R22): Philox4x32-10, key = seed, counter = (event_lo, event_hi, 15, 0);
// bit b of the first output word is the helicity of particle b in the order u, ubar,
// gamma_1..gamma_n (1 -> +1).  sigma_1 = sigma_2 gives exactly 0 (helicity conservation on the
// massless line); sigma_1 = -1 is evaluated through parity, |M(-s,-l)| = |M(s,l)|.
//
// Mapping: one WARP per event (the paper's thread-per-event mapping would need the 2^n-entry
// propagator table per thread).  The warp builds the event's E' and P tables in shared memory
// (lanes stride over the 2^n - 2 subsets), then its lanes share the permutation tree of
// eq. (6) by ordered prefixes of length D = min(n-1, 3): n!/(n-D)! units, each lane
// walks the subtrees below its units with the same Walk / Bottom code as amp2.cu (prefix reuse
// inside a subtree), and a warp shuffle adds the partial ampsums before squaring.
#include "amp2_tree.cuh"
#include "philox.cuh"

namespace {

constexpr uint32_t kHelicitySlot = 15u;
// events (warps) per CTA: the P tables of a CTA's events must fit 48 KB of static shared memory
template <int N>
constexpr int kWarpsPerCta = (N >= 8) ? 4 : 8;

__host__ __device__ constexpr int falling_factorial(int n, int d)
{
    int r = 1;
    for (int i = 0; i < d; ++i) r *= (n - i);
    return r;
}

// position of the k-th (0-based) set bit of mask
__device__ __forceinline__ int kth_set_bit(unsigned mask, int k)
{
    for (int t = 0; t < k; ++t) mask &= mask - 1u;
    return __ffs(mask) - 1;
}

template <int N, typename T>
__global__ void __launch_bounds__(kWarpsPerCta<N> * 32)
amp2_sampled_kernel(const double* __restrict__ momenta, uint64_t seed, uint64_t first_event,
                    double* __restrict__ out, int32_t* __restrict__ out_hel, int64_t n_events, double g)
{
    constexpr int L = 1 << N;
    constexpr int MOM = 4 * (N + 2);
    constexpr int EPB = kWarpsPerCta<N>;
    constexpr int D = (N - 1 < 3) ? N - 1 : 3;          // prefix length that defines a unit
    constexpr int UNITS = falling_factorial(N, D);
    constexpr int KB = (N - D < HEGET_KB) ? N - D : HEGET_KB;
    __shared__ __align__(16) double s_mom[EPB * MOM];
    __shared__ PEntry<T> s_P[EPB * L];
    __shared__ EEntry<T> s_E[EPB * 2 * N];
    __shared__ double s_s2[EPB * N];
    constexpr int NP = N * (N - 1) / 2;
    __shared__ Spinor<T> s_W[EPB * NP];  // pair closing table of the drawn helicities (amp2_tree.cuh, CLOSE = 3)

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int64_t ev0 = (int64_t)blockIdx.x * EPB;
    {
        const double2* src = reinterpret_cast<const double2*>(momenta);
        double2* dst = reinterpret_cast<double2*>(s_mom);
        for (int idx = tid; idx < EPB * MOM / 2; idx += EPB * 32) {
            int64_t e = ev0 + idx / (MOM / 2);
            if (e >= n_events) e = n_events - 1;
            dst[idx] = src[e * (MOM / 2) + idx % (MOM / 2)];
        }
    }
    __syncthreads();

    const double* mom = s_mom + w * MOM;
    const double shat = 4.0 * mom[0] * mom[4];
    const double scale = (sizeof(T) == 4) ? sqrt(shat) : 1.0;
    PEntry<T>* P = s_P + w * L;
    EEntry<T>* E = s_E + w * 2 * N;
    if (lane < N) s_s2[w * N + lane] = make_photon_entries<T>(mom + 4 * (2 + lane), &E[2 * lane + 1], &E[2 * lane]);
    for (unsigned S = 1u + lane; S <= (unsigned)(L - 2); S += 32u) {
        if constexpr (sizeof(T) == 4)
            make_subset_entry_plain<N>(mom, S, g, scale, &P[S]);
        else
            make_subset_entry<N, T>(mom, S, g, scale, &P[S]);
    }
    __syncthreads();

    const int64_t e = ev0 + w;
    const uint64_t gev = first_event + (uint64_t)(e < n_events ? e : n_events - 1);
    uint32_t x[4];
    philox4x32_10((uint32_t)gev, (uint32_t)(gev >> 32), kHelicitySlot, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), x);
    const uint32_t bits = x[0] & ((1u << (N + 2)) - 1u);
    const bool s1 = bits & 1u, s2 = (bits >> 1) & 1u;
    const unsigned lam = (bits >> 2) & (unsigned)(L - 1);
    const unsigned hel = s1 ? lam : (~lam & (unsigned)(L - 1));   // parity image for sigma_1 = -1

    // W_ab = U_b E'_a + U_a E'_b for the drawn helicities of a < b (build_pair_table, amp2_common.cuh)
    if (lane < NP) {
        unsigned b = 1;
        while ((b + 1) * b / 2 <= (unsigned)lane) ++b;
        const unsigned a = (unsigned)lane - b * (b - 1) / 2;
        const EEntry<T> ea = E[2 * a + ((hel >> a) & 1u)], eb = E[2 * b + ((hel >> b) & 1u)];
        Spinor<T> wab = {(T)0, (T)0, (T)0, (T)0};
        accumulate_row_times_vertex(closing_entry(eb, P[(L - 1) ^ (1 << b)]), ea, wab);
        accumulate_row_times_vertex(closing_entry(ea, P[(L - 1) ^ (1 << a)]), eb, wab);
        s_W[w * NP + lane] = wab;
    }
    __syncthreads();

    T ar = 0, ai = 0;
    if (s1 != s2) {                                                // warp-uniform
        for (int u = lane; u < UNITS; u += 32) {
            Spinor<T> f = {(T)1, (T)0, (T)0, (T)0};
            unsigned used = 0u;
            int rest = u;
#pragma unroll
            for (int d = 0; d < D; ++d) {
                const int stride = falling_factorial(N - d - 1, D - d - 1);
                const int idx = rest / stride;
                rest -= idx * stride;
                const int i = kth_set_bit(((unsigned)L - 1u) & ~used, idx);
                used |= 1u << i;
                f = fvixx0_weyl(P[used], E[2 * i + ((hel >> i) & 1u)], f);
            }
            Walk<N, D, KB, T, 0, (KB >= 2) ? 3 : 0>::run(P, E, hel, used, f, ar, ai, s_W + w * NP);
        }
    }
    double dr = (double)ar, di = (double)ai;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        dr += __shfl_xor_sync(0xffffffffu, dr, off);
        di += __shfl_xor_sync(0xffffffffu, di, off);
    }
    if (lane == 0 && e < n_events) {
        // |M(h)|^2 = g^2 s_hat 2^-N prod s_i^2 |ampsum|^2 (fp32: in units of sqrt(s_hat));
        // estimator = 4 * 2^N * |M(h)|^2
        double fct = 4.0 * g * g * shat;
#pragma unroll
        for (int i = 0; i < N; ++i) fct *= s_s2[w * N + i];
        if (sizeof(T) == 4) {
            const double inv = 1.0 / shat;
#pragma unroll
            for (int i = 0; i < N - 1; ++i) fct *= inv;
        }
        out[e] = fct * (dr * dr + di * di);
        if (out_hel) out_hel[e] = (int32_t)bits;
    }
}

// Small n: the whole event fits one THREAD (the paper's own mapping): its 2^N - 2
// propagator entries and 2N polarisation entries live in thread-local arrays (L1-resident), the
// tables are built with the same functions as everywhere else and the same Walk / Bottom code
// walks the tree.  For small N a warp per event is mostly idle lanes in the table phase; measured
// on B200 (2^20 events, fp64, warp -> thread per event): 2 gamma 0.54 -> 0.08 ms, 3 gamma 0.68 -> 0.11,
// 4 gamma 0.78 -> 0.23, 5 gamma 1.28 -> 0.73; 6 gamma 4.5 -> 10.1 ms (the 62-entry table and the
// deeper tree no longer fit the registers), so the switch is at N = 5.
#ifndef HEGET_SAMPLED_THREAD_MAXN
#define HEGET_SAMPLED_THREAD_MAXN 5
#endif
#ifndef HEGET_SAMPLED_PAIR_MINN
#define HEGET_SAMPLED_PAIR_MINN 4   // thread kernel: pair closing table from this N on
#endif

template <int N, typename T>
__global__ void __launch_bounds__(128)
amp2_sampled_thread_kernel(const double* __restrict__ momenta, uint64_t seed, uint64_t first_event,
                           double* __restrict__ out, int32_t* __restrict__ out_hel, int64_t n_events, double g)
{
    constexpr int L = 1 << N;
    constexpr int MOM = 4 * (N + 2);
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_events) return;
    double mom[MOM];
    {
        const double2* src = reinterpret_cast<const double2*>(momenta + e * MOM);
#pragma unroll
        for (int k = 0; k < MOM / 2; ++k) {
            const double2 v = src[k];
            mom[2 * k] = v.x;
            mom[2 * k + 1] = v.y;
        }
    }
    const uint64_t gev = first_event + (uint64_t)e;
    uint32_t x[4];
    philox4x32_10((uint32_t)gev, (uint32_t)(gev >> 32), kHelicitySlot, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), x);
    const uint32_t bits = x[0] & ((1u << (N + 2)) - 1u);
    const bool s1 = bits & 1u, s2 = (bits >> 1) & 1u;
    double result = 0.0;
    if (s1 != s2) {
        const unsigned lam = (bits >> 2) & (unsigned)(L - 1);
        const unsigned hel = s1 ? lam : (~lam & (unsigned)(L - 1));   // parity image for sigma_1 = -1
        const double shat = 4.0 * mom[0] * mom[4];
        const double scale = (sizeof(T) == 4) ? sqrt(shat) : 1.0;
        PEntry<T> P[L];
        EEntry<T> E[2 * N];
        double fct = 4.0 * g * g * shat;
#pragma unroll
        for (int i = 0; i < N; ++i) fct *= make_photon_entries<T>(mom + 4 * (2 + i), &E[2 * i + 1], &E[2 * i]);
#pragma unroll 1
        for (unsigned S = 1; S <= (unsigned)(L - 2); ++S) {
            if constexpr (sizeof(T) == 4)
                make_subset_entry_plain<N>(mom, S, g, scale, &P[S]);
            else
                make_subset_entry<N, T>(mom, S, g, scale, &P[S]);
        }
        T ar = 0, ai = 0;
        const Spinor<T> f0 = {(T)1, (T)0, (T)0, (T)0};
        if constexpr (N >= HEGET_SAMPLED_PAIR_MINN) {
            // pair closing table of the drawn helicities (amp2_tree.cuh, CLOSE = 3)
            Spinor<T> W[N * (N - 1) / 2];
#pragma unroll
            for (int b = 1; b < N; ++b)
#pragma unroll
                for (int a = 0; a < b; ++a) {
                    const EEntry<T> ea = E[2 * a + ((hel >> a) & 1u)], eb = E[2 * b + ((hel >> b) & 1u)];
                    Spinor<T> wab = {(T)0, (T)0, (T)0, (T)0};
                    accumulate_row_times_vertex(closing_entry(eb, P[(L - 1) ^ (1 << b)]), ea, wab);
                    accumulate_row_times_vertex(closing_entry(ea, P[(L - 1) ^ (1 << a)]), eb, wab);
                    W[b * (b - 1) / 2 + a] = wab;
                }
            Walk<N, 0, N, T, 0, 3>::run(P, E, hel, 0u, f0, ar, ai, W);
        } else {
            Spinor<T> U[2 * N];
#pragma unroll
            for (int q = 0; q < 2 * N; ++q) U[q] = closing_entry(E[q], P[(L - 1) ^ (1 << (q >> 1))]);
            Walk<N, 0, N, T, 0, 1>::run(P, E, hel, 0u, f0, ar, ai, U);
        }
        if (sizeof(T) == 4) {
            const double inv = 1.0 / shat;
#pragma unroll
            for (int i = 0; i < N - 1; ++i) fct *= inv;
        }
        result = fct * ((double)ar * (double)ar + (double)ai * (double)ai);
    }
    out[e] = result;
    if (out_hel) out_hel[e] = (int32_t)bits;
}

template <int N, typename T>
cudaError_t launch_one(const double* momenta, uint64_t seed, uint64_t first_event, double* out, int32_t* out_hel,
                       int64_t n_events, double g, cudaStream_t stream)
{
    if constexpr (N <= HEGET_SAMPLED_THREAD_MAXN) {
        amp2_sampled_thread_kernel<N, T><<<(unsigned)((n_events + 127) / 128), 128, 0, stream>>>(
            momenta, seed, first_event, out, out_hel, n_events, g);
        return cudaGetLastError();
    }
    const int64_t blocks = (n_events + kWarpsPerCta<N> - 1) / kWarpsPerCta<N>;
    amp2_sampled_kernel<N, T><<<(unsigned)blocks, kWarpsPerCta<N> * 32, 0, stream>>>(momenta, seed, first_event, out,
                                                                                  out_hel, n_events, g);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_n(int n, const double* momenta, uint64_t seed, uint64_t first_event, double* out,
                     int32_t* out_hel, int64_t n_events, double g, cudaStream_t stream)
{
    switch (n) {
        case 2: return launch_one<2, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        case 3: return launch_one<3, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        case 4: return launch_one<4, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        case 5: return launch_one<5, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        case 6: return launch_one<6, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        case 7: return launch_one<7, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        case 8: return launch_one<8, T>(momenta, seed, first_event, out, out_hel, n_events, g, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t heget_launch_amp2_sampled(const heget_ctx* ctx, uint64_t seed, uint64_t first_event,
                                      const double* momenta, int n, int precision, double* out_amp2,
                                      int32_t* out_hel, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    if (precision == HEGET_FP32)
        return launch_n<float>(n, momenta, seed, first_event, out_amp2, out_hel, N, ctx->g, stream);
    return launch_n<double>(n, momenta, seed, first_event, out_amp2, out_hel, N, ctx->g, stream);
}

// amp2.cu -- heget_amp2: summed squared helicity amplitude of u ubar -> n gamma (product code).
//
// Mapping: one lane per photon-helicity configuration (2^N lanes per event), 256-thread CTAs
// holding 256/2^N events.  All lanes of a CTA walk the SAME permutation tree in lockstep
// (no divergence); they differ only in which helicity entry of the per-photon E table they
// read.  Per event the CTA first builds, in shared memory,
//   - the E table (vxxxx0 for both helicities of every photon) and
//   - the subset table P[S] = -g/t_S * (p1 - K_S)-slash block for every photon subset S,
// then every lane runs the depth-first walk of eq. (6)'s n! orderings: each
// ordered prefix (tree node) is one fvixx0 computed once, each leaf one
// iovxxx accumulated into ampsum (List 2).
// Only sigma_1 = +1, sigma_2 = -1 is evaluated: sigma_1 = sigma_2 vanishes identically and
// |M(-sigma,-lambda)| = |M(sigma,lambda)|, so the helicity sum is twice the sum over lambda.
#include "amp2_common.cuh"

#ifndef HEGET_KB
#define HEGET_KB 4          // unrolled bottom levels of the permutation tree
#endif
#ifndef HEGET_E_BY_PTR
#define HEGET_E_BY_PTR 0    // 1: Bottom<K> re-reads E' entries from shared memory instead of holding them
#endif
#ifndef HEGET_MINB32
#define HEGET_MINB32 1      // __launch_bounds__ min CTAs per SM, fp32 / fp64 kernels
#endif
#ifndef HEGET_MINB64
#define HEGET_MINB64 2
#endif

namespace {

// fvixx0 in Weyl form: psi' = P_S * (E'_i * psi), 20 FMA-pipe instructions.
template <typename T>
__device__ __forceinline__ Spinor<T> fvixx0_weyl(const PEntry<T>& P, const EEntry<T>& E, const Spinor<T>& f)
{
    // w = E' f,  E' = [[-1, -b], [a, 1]]
    const T w0r = fma(-E.br, f.r1, fma(E.bi, f.i1, -f.r0));
    const T w0i = fma(-E.br, f.i1, fma(-E.bi, f.r1, -f.i0));
    const T w1r = fma(E.ar, f.r0, fma(-E.ai, f.i0, f.r1));
    const T w1i = fma(E.ar, f.i0, fma(E.ai, f.r0, f.i1));
    // psi' = P w,  P = [[pp, px - i py], [px + i py, pm]]
    Spinor<T> o;
    o.r0 = fma(P.pp, w0r, fma(P.px, w1r, P.py * w1i));
    o.i0 = fma(P.pp, w0i, fma(P.px, w1i, -(P.py * w1r)));
    o.r1 = fma(P.pm, w1r, fma(P.px, w0r, -(P.py * w0i)));
    o.i1 = fma(P.pm, w1i, fma(P.px, w0i, P.py * w0r));
    return o;
}

// iovxxx in Weyl form: vbar (oxxxx2) has the single component 1 of the (0,1)
// pair, so amp = row 1 of E'_j times psi = a psi0 + psi1 (constant factors applied at the end).
template <typename T>
__device__ __forceinline__ void iovxxx_weyl(const EEntry<T>& E, const Spinor<T>& f, T& ar, T& ai)
{
    ar += fma(E.ar, f.r0, fma(-E.ai, f.i0, f.r1));
    ai += fma(E.ar, f.i0, fma(E.ai, f.r0, f.i1));
}

// Bottom K levels of the permutation tree, fully unrolled.  The K photons still to attach are
// held as compile-time-indexed register arrays (bit[] = their subset-index bits, e[] = this
// lane's E' entries), so choosing a child is register renaming, not bit arithmetic: the code
// of a subtree is straight-line FMAs plus one P-entry load per node.
template <typename T> __device__ __forceinline__ const EEntry<T>& eload(const EEntry<T>& e) { return e; }
template <typename T> __device__ __forceinline__ EEntry<T> eload(const EEntry<T>* e) { return *e; }

template <int K, typename T, typename EA>
struct Bottom {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ PS, const int (&bit)[K],
                                               const EA (&e)[K], const Spinor<T>& f, T& ar, T& ai)
    {
#pragma unroll
        for (int i = 0; i < K; ++i) {
            int sub_bit[K - 1];
            EA sub_e[K - 1];
#pragma unroll
            for (int m = 0; m < K - 1; ++m) {
                sub_bit[m] = bit[m + (m >= i ? 1 : 0)];
                sub_e[m] = e[m + (m >= i ? 1 : 0)];
            }
            const PEntry<T>* Pn = PS + bit[i];
            const Spinor<T> fn = fvixx0_weyl(*Pn, eload<T>(e[i]), f);
            Bottom<K - 1, T, EA>::run(Pn, sub_bit, sub_e, fn, ar, ai);
        }
    }
};

template <typename T, typename EA>
struct Bottom<1, T, EA> {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__, const int (&)[1],
                                               const EA (&e)[1], const Spinor<T>& f, T& ar, T& ai)
    {
        iovxxx_weyl(eload<T>(e[0]), f, ar, ai);
    }
};

// Depth-first walk of the upper levels.  `used` = set of photons already attached (uniform
// over the CTA); when KB photons remain the unrolled Bottom<KB> takes over.
template <int N, int DEPTH, int KB, typename T>
struct Walk {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                               unsigned hel, unsigned used, const Spinor<T>& f, T& ar, T& ai)
    {
        unsigned avail = ((1u << N) - 1u) & ~used;
        if constexpr (N - DEPTH == KB) {
            int bit[KB];
#if HEGET_E_BY_PTR
            using EA = const EEntry<T>*;
#else
            using EA = EEntry<T>;
#endif
            EA e[KB];
#pragma unroll
            for (int m = 0; m < KB; ++m) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                bit[m] = 1 << i;
#if HEGET_E_BY_PTR
                e[m] = &E[2 * i + ((hel >> i) & 1u)];
#else
                e[m] = E[2 * i + ((hel >> i) & 1u)];
#endif
            }
            Bottom<KB, T, EA>::run(P + used, bit, e, f, ar, ai);
        } else {
            while (avail) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                const unsigned S = used | (1u << i);
                const Spinor<T> fn = fvixx0_weyl(P[S], E[2 * i + ((hel >> i) & 1u)], f);
                Walk<N, DEPTH + 1, KB, T>::run(P, E, hel, S, fn, ar, ai);
            }
        }
    }
};

template <int N>
constexpr int kBottom = (N < HEGET_KB) ? N : HEGET_KB;  // unrolled bottom levels of the tree

template <int N, typename T>
__global__ void __launch_bounds__(Geometry<N>::THREADS, (sizeof(T) == 4) ? HEGET_MINB32 : HEGET_MINB64)
amp2_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    using G = Geometry<N>;
    constexpr int MOM = 4 * (N + 2);
    __shared__ __align__(16) double s_mom[G::EPB * MOM];
    __shared__ PEntry<T> s_P[G::EPB * G::L];
    __shared__ EEntry<T> s_E[G::EPB * 2 * N];
    __shared__ double s_red[G::THREADS / 32];
    __shared__ double s_s2[G::EPB * N];  // s_i^2 = (pT/w)^2 taken out of photon i's E entries

    const int ev_local = threadIdx.x / G::L;
    const unsigned hel = threadIdx.x % G::L;

    // a1, a4, a5: momenta -> shared memory, E' and P tables of the CTA's events
    build_event_tables<N, T>(momenta, n_events, g, s_mom, s_P, s_E, s_s2);

    // a2, a6, a7: psi_0 = u(p1,+)/sqrt(2E1) = (1,0); walk the permutation tree
    T ar = 0, ai = 0;
    const Spinor<T> f0 = {(T)1, (T)0, (T)0, (T)0};
    Walk<N, 0, kBottom<N>, T>::run(s_P + ev_local * G::L, s_E + ev_local * 2 * N, hel, 0u, f0, ar, ai);

    // a8: |ampsum|^2 summed over the event's 2^N lanes, constant factors, store
    finish_event<N, T>(ar, ai, s_mom, s_s2, s_red, g, out, n_events);
}

template <int N, typename T>
cudaError_t launch_one(const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    using G = Geometry<N>;
    const int64_t blocks = (n_events + G::EPB - 1) / G::EPB;
    amp2_kernel<N, T><<<(unsigned)blocks, G::THREADS, 0, stream>>>(momenta, out, n_events, g);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_n(int n, const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    switch (n) {
        case 2: return launch_one<2, T>(momenta, out, n_events, g, stream);
        case 3: return launch_one<3, T>(momenta, out, n_events, g, stream);
        case 4: return launch_one<4, T>(momenta, out, n_events, g, stream);
        case 5: return launch_one<5, T>(momenta, out, n_events, g, stream);
        case 6: return launch_one<6, T>(momenta, out, n_events, g, stream);
        case 7: return launch_one<7, T>(momenta, out, n_events, g, stream);
        case 8: return launch_one<8, T>(momenta, out, n_events, g, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t heget_launch_amp2(const heget_ctx* ctx, const double* momenta, int n, int precision,
                              double* out_amp2, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    if (precision == HEGET_FP32) return launch_n<float>(n, momenta, out_amp2, N, ctx->g, stream);
    return launch_n<double>(n, momenta, out_amp2, N, ctx->g, stream);
}

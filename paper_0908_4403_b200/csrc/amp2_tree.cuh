// amp2_tree.cuh -- the depth-first permutation tree of eq. (6): fvixx0 node,
// iovxxx leaf, the looped upper levels and the unrolled bottom levels (product code).  Used by
// amp2.cu (all helicities, one lane per helicity configuration) and amp2_sampled.cu (one drawn
// helicity configuration per event, lanes split the top of the tree).
#pragma once
#include "amp2_common.cuh"

#ifndef HEGET_KB
#define HEGET_KB 4          // unrolled bottom levels of the permutation tree
#endif
#ifndef HEGET_E_BY_PTR
#define HEGET_E_BY_PTR 0    // 1: Bottom<K> re-reads E' entries from shared memory instead of holding them
#endif

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


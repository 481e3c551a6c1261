// amp2_tree.cuh -- the depth-first permutation tree of eq. (6): fvixx0 node,
// iovxxx leaf, the looped upper levels and the unrolled bottom levels (product code).  Used by
// amp2.cu (all helicities, one lane per helicity configuration) and amp2_sampled.cu (one drawn
// helicity configuration per event, lanes split the top of the tree).
#pragma once
#include <type_traits>

#include "amp2_common.cuh"

#ifndef HEGET_KB
#define HEGET_KB 4          // unrolled bottom levels of the permutation tree
#endif
#ifndef HEGET_SHARE_BY_PTR
#define HEGET_SHARE_BY_PTR 1  // lane-sharing kernels keep E' entries as pointers (one select instead of eight)
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

// The FFV vertex alone, w = E' psi (8 FMA-pipe instructions), and the closing of a branch whose
// last propagator has been contracted into the closing vertex:
//   <vbar| E'_b P_{all \ b} (E'_a psi) = U_b . (E'_a psi),   U_b = <vbar| E'_b P_{all \ b}
// (the last propagator of EVERY ordering that ends with photon b belongs to the set "all but b",
// so U_b is one row vector per photon and helicity: build_closing_table, amp2_common.cuh).
// The product of the last three factors of a diagram is merely associated differently:
// 8 + 8 instructions for the last fvixx0 + iovxxx of a branch instead of 20 + 6.
template <typename T>
__device__ __forceinline__ Spinor<T> vertex_weyl(const EEntry<T>& E, const Spinor<T>& f)
{
    Spinor<T> w;
    w.r0 = fma(-E.br, f.r1, fma(E.bi, f.i1, -f.r0));
    w.i0 = fma(-E.br, f.i1, fma(-E.bi, f.r1, -f.i0));
    w.r1 = fma(E.ar, f.r0, fma(-E.ai, f.i0, f.r1));
    w.i1 = fma(E.ar, f.i0, fma(E.ai, f.r0, f.i1));
    return w;
}

template <typename T>
__device__ __forceinline__ void close_weyl(const Spinor<T>& U, const Spinor<T>& w, T& ar, T& ai)
{
    ar += fma(U.r0, w.r0, fma(-U.i0, w.i0, fma(U.r1, w.r1, -(U.i1 * w.i1))));
    ai += fma(U.r0, w.i0, fma(U.i0, w.r0, fma(U.r1, w.i1, U.i1 * w.r1)));
}

// Bottom K levels of the permutation tree, fully unrolled.  The K photons still to attach are
// held as compile-time-indexed register arrays (bit[] = their subset-index bits, e[] = this
// lane's E' entries), so choosing a child is register renaming, not bit arithmetic: the code
// of a subtree is straight-line FMAs plus one P-entry load per node.
template <typename T> __device__ __forceinline__ const EEntry<T>& eload(const EEntry<T>& e) { return e; }
template <typename T> __device__ __forceinline__ EEntry<T> eload(const EEntry<T>* e) { return *e; }
template <typename T>
__device__ __forceinline__ EEntry<T> eselect(bool c, const EEntry<T>& a, const EEntry<T>& b)
{
    EEntry<T> r;
    r.ar = c ? a.ar : b.ar; r.ai = c ? a.ai : b.ai; r.br = c ? a.br : b.br; r.bi = c ? a.bi : b.bi;
    return r;
}
template <typename T>
__device__ __forceinline__ EEntry<T> eselect(bool c, const EEntry<T>* a, const EEntry<T>* b) { return *(c ? a : b); }

// SHARE = 1 (amp2.cu, fp64): at the last level the two lanes that differ only in the helicity of
// the photon still to be closed need the SAME off-shell spinor (a prefix's spinor depends on the
// helicities of the photons in the prefix only).  With two photons a, b left, a lane whose
// helicity bits of a and b are equal computes psi(.., a) and receives psi(.., b) from the lane
// with bit a flipped; a lane whose bits differ computes psi(.., b) and receives psi(.., a) from the
// lane with bit b flipped -- one fvixx0 (20 FP64 instructions) and 8 shuffles per lane instead of
// two fvixx0.  Every lane still executes the same instruction stream (per-lane operand selects).
// Needs both photons' lane bits inside the warp (photon index < 5); otherwise, and always for
// SHARE = 0 (fp32, where the shuffles would cost what they save; amp2_sampled.cu, whose lanes are
// not helicity configurations), both nodes are computed.  hb[] = this lane's helicity bits.
// CLOSE = 1: the last fvixx0 + iovxxx of every branch are evaluated as vertex + close_weyl with
// the closing table (u[] = this lane's U entries of the remaining photons).
// CLOSE = 2: the last TWO orderings of every prefix of n-2 photons are one dot product with the
// pair closing table (build_pair_table, amp2_common.cuh): idx[] = positions of the remaining
// photons in the list Bottom<KB> started from, w[] = this lane's W entries of the KP = KB(KB-1)/2
// pairs of that list (position pair p < q at q(q-1)/2 + p); u[] is unused.  CLOSE = 3: the same
// with a table that holds ONE helicity assignment, W[b(b-1)/2 + a] (amp2_sampled.cu).
template <int K, typename T, typename EA, int SHARE = 0, int CLOSE = 0, int KP = 1>
struct Bottom {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ PS, const int (&bit)[K],
                                               const EA (&e)[K], const unsigned (&hb)[K],
                                               const Spinor<T>* const (&u)[K], const int (&idx)[K],
                                               const Spinor<T>* const (&w)[KP], const Spinor<T>& f, T& ar, T& ai)
    {
        static_assert(!(SHARE == 1 && CLOSE >= 2), "lane sharing and the pair table are alternatives");
        if constexpr (K == 2 && CLOSE >= 2) {
            close_weyl(*w[idx[1] * (idx[1] - 1) / 2 + idx[0]], f, ar, ai);
            return;
        }
        if constexpr (K == 2 && CLOSE == 1) {
            if constexpr (SHARE == 1) {
                if ((bit[0] | bit[1]) < 32) {  // uniform over the CTA
                    // w_a = E'_a psi does not depend on the helicity of b (and vice versa): each lane
                    // evaluates one of the two vertices and fetches the other one by shuffle
                    const bool odd = (hb[0] ^ hb[1]) != 0u;
                    const EEntry<T> em = eselect<T>(odd, e[1], e[0]);
                    const int bm = odd ? bit[1] : bit[0];
                    const Spinor<T> wm = vertex_weyl(em, f);
                    Spinor<T> wo;
                    wo.r0 = __shfl_xor_sync(0xffffffffu, wm.r0, bm);
                    wo.i0 = __shfl_xor_sync(0xffffffffu, wm.i0, bm);
                    wo.r1 = __shfl_xor_sync(0xffffffffu, wm.r1, bm);
                    wo.i1 = __shfl_xor_sync(0xffffffffu, wm.i1, bm);
                    close_weyl(*(odd ? u[0] : u[1]), wm, ar, ai);  // my vertex closes with the other photon
                    close_weyl(*(odd ? u[1] : u[0]), wo, ar, ai);  // the received one closes with mine
                    return;
                }
            }
            close_weyl(*u[1], vertex_weyl(eload<T>(e[0]), f), ar, ai);
            close_weyl(*u[0], vertex_weyl(eload<T>(e[1]), f), ar, ai);
            return;
        }
        if constexpr (K == 2 && SHARE == 1) {
            if ((bit[0] | bit[1]) < 32) {  // uniform over the CTA
                const bool odd = (hb[0] ^ hb[1]) != 0u;
                // mine: the photon this lane attaches; other: the one it closes with.  With
                // pointer lists the choice is one select and a shared-memory load per entry.
                const EEntry<T> em = eselect<T>(odd, e[1], e[0]);
                const EEntry<T> eo = eselect<T>(odd, e[0], e[1]);
                const int bm = odd ? bit[1] : bit[0];
                const Spinor<T> fm = fvixx0_weyl(PS[bm], em, f);
                Spinor<T> fo;
                fo.r0 = __shfl_xor_sync(0xffffffffu, fm.r0, bm);
                fo.i0 = __shfl_xor_sync(0xffffffffu, fm.i0, bm);
                fo.r1 = __shfl_xor_sync(0xffffffffu, fm.r1, bm);
                fo.i1 = __shfl_xor_sync(0xffffffffu, fm.i1, bm);
                iovxxx_weyl(eo, fm, ar, ai);  // my node closes with the other photon
                iovxxx_weyl(em, fo, ar, ai);  // the received node closes with my photon
                return;
            }
        }
#pragma unroll
        for (int i = 0; i < K; ++i) {
            int sub_bit[K - 1];
            EA sub_e[K - 1];
            unsigned sub_hb[K - 1];
            const Spinor<T>* sub_u[K - 1];
            int sub_idx[K - 1];
#pragma unroll
            for (int m = 0; m < K - 1; ++m) {
                sub_bit[m] = bit[m + (m >= i ? 1 : 0)];
                sub_e[m] = e[m + (m >= i ? 1 : 0)];
                sub_hb[m] = hb[m + (m >= i ? 1 : 0)];
                sub_u[m] = u[m + (m >= i ? 1 : 0)];
                sub_idx[m] = idx[m + (m >= i ? 1 : 0)];
            }
            const PEntry<T>* Pn = PS + bit[i];
            const Spinor<T> fn = fvixx0_weyl(*Pn, eload<T>(e[i]), f);
            Bottom<K - 1, T, EA, SHARE, CLOSE, KP>::run(Pn, sub_bit, sub_e, sub_hb, sub_u, sub_idx, w, fn, ar, ai);
        }
    }
};

template <typename T, typename EA, int SHARE, int CLOSE, int KP>
struct Bottom<1, T, EA, SHARE, CLOSE, KP> {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__, const int (&)[1],
                                               const EA (&e)[1], const unsigned (&)[1],
                                               const Spinor<T>* const (&)[1], const int (&)[1],
                                               const Spinor<T>* const (&)[KP], const Spinor<T>& f, T& ar, T& ai)
    {
        iovxxx_weyl(eload<T>(e[0]), f, ar, ai);
    }
};

// Depth-first walk of the upper levels.  `used` = set of photons already attached (uniform
// over the CTA); when KB photons remain the unrolled Bottom<KB> takes over.
template <int N, int DEPTH, int KB, typename T, int SHARE = 0, int CLOSE = 0>
struct Walk {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                               unsigned hel, unsigned used, const Spinor<T>& f, T& ar, T& ai,
                                               const Spinor<T>* __restrict__ U = nullptr)
    {
        static_assert(CLOSE == 0 || KB >= 2, "the closing tables replace the last TWO levels");
        unsigned avail = ((1u << N) - 1u) & ~used;
        if constexpr (N - DEPTH == KB) {
            int bit[KB];
            unsigned hb[KB];
            // entries held in registers, or (HEGET_E_BY_PTR, and the lane-sharing fp64 kernels)
            // pointers into the shared-memory table that are dereferenced at each use
            constexpr bool BY_PTR = (HEGET_E_BY_PTR != 0) || (SHARE == 1 && HEGET_SHARE_BY_PTR != 0);
            using EA = std::conditional_t<BY_PTR, const EEntry<T>*, EEntry<T>>;
            EA e[KB];
            const Spinor<T>* u[KB];
            int idx[KB], photon[KB];
#pragma unroll
            for (int m = 0; m < KB; ++m) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                bit[m] = 1 << i;
                hb[m] = (hel >> i) & 1u;
                u[m] = (CLOSE >= 2) ? nullptr : U + 2 * i + hb[m];
                idx[m] = m;
                photon[m] = i;
                if constexpr (BY_PTR)
                    e[m] = &E[2 * i + hb[m]];
                else
                    e[m] = E[2 * i + hb[m]];
            }
            constexpr int KP = (CLOSE >= 2) ? KB * (KB - 1) / 2 : 1;
            const Spinor<T>* w[KP];
            if constexpr (CLOSE >= 2) {  // U is the pair closing table; photon[] is increasing
#pragma unroll
                for (int q = 1; q < KB; ++q)
#pragma unroll
                    for (int p = 0; p < q; ++p) {
                        const int pair = photon[q] * (photon[q] - 1) / 2 + photon[p];
                        w[q * (q - 1) / 2 + p] = (CLOSE == 2) ? U + 4 * pair + 2 * hb[p] + hb[q] : U + pair;
                    }
            } else {
                w[0] = nullptr;
            }
            Bottom<KB, T, EA, SHARE, CLOSE, KP>::run(P + used, bit, e, hb, u, idx, w, f, ar, ai);
        } else {
            while (avail) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                const unsigned S = used | (1u << i);
                const Spinor<T> fn = fvixx0_weyl(P[S], E[2 * i + ((hel >> i) & 1u)], f);
                Walk<N, DEPTH + 1, KB, T, SHARE, CLOSE>::run(P, E, hel, S, fn, ar, ai, U);
            }
        }
    }
};

// amp2_chain.cuh -- the permutation tree of eq. (6) with every off-shell spinor held
// in factorised form (product code, v9; amp2.cu uses it for n >= 5).
//
// For a massless photon of definite helicity the chiral block of eps-slash has rank one
// (eps-slash^2 = eps.eps = 0): in the normalisation of amp2_tables.cuh, a b = 1 and
//     E' = [[-1, -b], [a, 1]] = (-1, a)^T (1, b),   E' psi = (psi_0 + b psi_1) (-1, a)^T.
// So fvixx0, psi' = P_S E'_i psi, is a complex NUMBER times a vector that does not
// depend on the prefix's order or on psi:
//     psi' = (psi_0 + b_i psi_1) v,   v = v(S, i, h_i) = P_S (-1, a_i)^T.
// Every node of the tree is therefore psi = z v with z one complex number; a child j of the node is
//     rho = v_0 + b_j v_1,  z' = z rho          (4 + 4 FMA-pipe instructions)
//     v'  = P_{S+j} (-1, a_j)^T                  (6 instructions; only if the child has children)
// instead of the 20 instructions of fvixx0_weyl.  Each ordered prefix is still ONE node computed once
// by the depth-first walk and all n! orderings are visited; no ordering-summed quantity is
// tabulated beyond the pair closing table W of v8 (amp2_common.cuh).  A node of n-2 photons closes
// its two remaining orderings with W_ab . psi = z (W_ab . v): the dot product depends on the event
// only, so it is tabulated per event (build_chain_table),
//     K[(pair(a,b) N + j) 8 + 4 h_j + 2 h_a + h_b] = W_ab(h_a,h_b) . v(all \ {a,b}, j, h_j),
// and the closing is z' K: 4 instructions instead of 8.  The walk does not carry z down: z is a
// common factor of everything below a node, so each node RETURNS the sum of its subtree without it,
//     A(node of n-2 photons) = K,   A(node) = sum over children j of rho_j A(child j),   ampsum = A(root)
// (distributivity only; every ordering is still one term).  Per node: 14 instructions
// (rho 4, v' 6, rho A 4; levels 1..n-3) or 8 (level n-2) instead of 20 and 28.
#pragma once
#include "amp2_common.cuh"

#ifndef HEGET_CHAIN_LEAN_MAXN
#define HEGET_CHAIN_LEAN_MAXN 6   // build_chain_table: one work item per (pair, j, h_j) up to this N
#endif

template <typename T>
struct alignas(2 * sizeof(T)) Cx {
    T r, i;
};

// v = P (-1, a)^T,  P = [[pp, px - i py], [px + i py, pm]]
template <typename T>
__device__ __forceinline__ Spinor<T> chain_vector(const PEntry<T>& P, const EEntry<T>& E)
{
    Spinor<T> v;
    v.r0 = fma(E.ar, P.px, fma(E.ai, P.py, -P.pp));
    v.i0 = fma(E.ai, P.px, -(E.ar * P.py));
    v.r1 = fma(E.ar, P.pm, -P.px);
    v.i1 = fma(E.ai, P.pm, -P.py);
    return v;
}

// rho = v_0 + b v_1
template <typename T>
__device__ __forceinline__ void chain_rho(const Spinor<T>& v, const EEntry<T>& E, T& rr, T& ri)
{
    rr = fma(E.br, v.r1, fma(-E.bi, v.i1, v.r0));
    ri = fma(E.br, v.i1, fma(E.bi, v.r1, v.i0));
}

// s += rho a
template <typename T>
__device__ __forceinline__ void chain_acc(T rr, T ri, T xr, T xi, T& sr, T& si)
{
    sr = fma(rr, xr, fma(-ri, xi, sr));
    si = fma(rr, xi, fma(ri, xr, si));
}

// Reads s_P, s_E and the pair closing table s_W (barrier before), ends with a barrier.
template <int N, typename T, typename G = Geometry<N>>
__device__ __forceinline__ void build_chain_table(const PEntry<T>* s_P, const EEntry<T>* s_E, const Spinor<T>* s_W,
                                                  Cx<T>* s_K)
{
    constexpr unsigned NP = N * (N - 1) / 2, ENTRIES = NP * N * 8u;
    // one work item per (pair, j not in the pair, h_j): the vector v once, then its dot products with
    // the four W entries of the pair (the K entries with j in {a, b} are holes and stay unwritten)
    constexpr unsigned ITEMS = NP * (N - 2) * 2u;
    const int ev_local = threadIdx.x / G::L;
    const unsigned lane = threadIdx.x % G::L;
    const PEntry<T>* P = s_P + ev_local * G::L;
    const EEntry<T>* E = s_E + ev_local * 2 * N;
    const Spinor<T>* W = s_W + ev_local * 4 * NP;
    Cx<T>* K = s_K + ev_local * ENTRIES;
    if constexpr (N <= HEGET_CHAIN_LEAN_MAXN) {
        for (unsigned q = lane; q < ITEMS; q += G::L) {
            const unsigned hj = q & 1u, t = q >> 1, jr = t % (N - 2), pair = t / (N - 2);
            unsigned b = 1;
            while ((b + 1) * b / 2 <= pair) ++b;
            const unsigned a = pair - b * (b - 1) / 2;
            unsigned j = jr;   // the jr-th photon outside {a, b}, a < b
            if (j >= a) ++j;
            if (j >= b) ++j;
            const Spinor<T> v = chain_vector(P[(G::L - 1) ^ (1u << a) ^ (1u << b)], E[2 * j + hj]);
    #pragma unroll
            for (unsigned h = 0; h < 4; ++h) {
                const Spinor<T> w = W[4 * pair + h];
                Cx<T> k;
                k.r = fma(w.r0, v.r0, fma(-w.i0, v.i0, fma(w.r1, v.r1, -(w.i1 * v.i1))));
                k.i = fma(w.r0, v.i0, fma(w.i0, v.r0, fma(w.r1, v.i1, w.i1 * v.r1)));
                K[(pair * N + j) * 8u + 4u * hj + h] = k;
            }
        }
    } else {
        // one entry per work item (the holes skipped).  From 7 photons on the table is < 1 % of the
        // kernel either way, and ptxas allocates the unrolled tree below better after this form
        // (8 gamma fp32: 223 ms against 232 ms with the loop above)
        for (unsigned q = lane; q < ENTRIES; q += G::L) {
            const unsigned h = q & 7u, pj = q >> 3, j = pj % N, pair = pj / N;
            unsigned b = 1;
            while ((b + 1) * b / 2 <= pair) ++b;
            const unsigned a = pair - b * (b - 1) / 2;
            if (j == a || j == b) continue;
            const Spinor<T> v = chain_vector(P[(G::L - 1) ^ (1u << a) ^ (1u << b)], E[2 * j + (h >> 2)]);
            const Spinor<T> w = W[4 * pair + (h & 3u)];
            Cx<T> k;
            k.r = fma(w.r0, v.r0, fma(-w.i0, v.i0, fma(w.r1, v.r1, -(w.i1 * v.i1))));
            k.i = fma(w.r0, v.i0, fma(w.i0, v.r0, fma(w.r1, v.i1, w.i1 * v.r1)));
            K[q] = k;
        }
    }
    __syncthreads();
}

// Bottom levels, fully unrolled (as Bottom<K> of amp2_tree.cuh: the K photons still to attach are
// compile-time-indexed register arrays, choosing a child is register renaming).  idx[] = positions
// of the remaining photons in the list of KB photons the unrolled part started from, kp[] = this
// lane's K-table base of each position pair p < q (at q(q-1)/2 + p), jo[] = offset of (j, h_j)
// for each position.  Ends at K = 3: the children are the nodes of n-2 photons, closed with K.
template <int K, int KB, typename T>
struct ChainBottom {
    static constexpr int KP = KB * (KB - 1) / 2;
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ PS, const int (&bit)[K],
                                               const EEntry<T> (&e)[K], const int (&idx)[K],
                                               const Cx<T>* const (&kp)[KP], const int (&jo)[KB],
                                               const Spinor<T>& v, T& ar, T& ai)
    {
        static_assert(K >= 3, "the K table closes the nodes of n-2 photons");
        T sr = 0, si = 0;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            T rr, ri;
            chain_rho(v, e[i], rr, ri);
            if constexpr (K == 3) {
                const int p = idx[i == 0 ? 1 : 0], q = idx[i == 2 ? 1 : 2];
                const Cx<T> k = kp[q * (q - 1) / 2 + p][jo[idx[i]]];
                chain_acc(rr, ri, k.r, k.i, sr, si);
            } else {
                int sub_bit[K - 1];
                EEntry<T> sub_e[K - 1];
                int sub_idx[K - 1];
#pragma unroll
                for (int m = 0; m < K - 1; ++m) {
                    sub_bit[m] = bit[m + (m >= i ? 1 : 0)];
                    sub_e[m] = e[m + (m >= i ? 1 : 0)];
                    sub_idx[m] = idx[m + (m >= i ? 1 : 0)];
                }
                const PEntry<T>* Pn = PS + bit[i];
                const Spinor<T> vc = chain_vector(*Pn, e[i]);
                T cr, ci;
                ChainBottom<K - 1, KB, T>::run(Pn, sub_bit, sub_e, sub_idx, kp, jo, vc, cr, ci);
                chain_acc(rr, ri, cr, ci, sr, si);
            }
        }
        ar = sr;
        ai = si;
    }
};

// Depth-first walk of the upper levels (`used` = photons already attached, uniform over the CTA;
// returns A(node) in ar, ai);
// when KB photons remain the unrolled ChainBottom<KB> takes over.  Needs N - KB >= 0 and KB >= 3.
template <int N, int DEPTH, int KB, typename T>
struct WalkChain {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                               unsigned hel, unsigned used, const Spinor<T>& v, T& ar, T& ai,
                                               const Cx<T>* __restrict__ Kt)
    {
        unsigned avail = ((1u << N) - 1u) & ~used;
        if constexpr (N - DEPTH == KB) {
            constexpr int KP = KB * (KB - 1) / 2;
            int bit[KB], idx[KB], photon[KB], jo[KB];
            unsigned hb[KB];
            EEntry<T> e[KB];
#pragma unroll
            for (int m = 0; m < KB; ++m) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                bit[m] = 1 << i;
                hb[m] = (hel >> i) & 1u;
                e[m] = E[2 * i + hb[m]];
                idx[m] = m;
                photon[m] = i;
                jo[m] = 8 * i + 4 * (int)hb[m];
            }
            const Cx<T>* kp[KP];
#pragma unroll
            for (int q = 1; q < KB; ++q)
#pragma unroll
                for (int p = 0; p < q; ++p) {  // photon[] is increasing
                    const int pair = photon[q] * (photon[q] - 1) / 2 + photon[p];
                    kp[q * (q - 1) / 2 + p] = Kt + pair * (N * 8) + 2 * hb[p] + hb[q];
                }
            ChainBottom<KB, KB, T>::run(P + used, bit, e, idx, kp, jo, v, ar, ai);
        } else {
            T sr = 0, si = 0;
            while (avail) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                const unsigned S = used | (1u << i);
                const EEntry<T> e = E[2 * i + ((hel >> i) & 1u)];
                T rr, ri, cr, ci;
                chain_rho(v, e, rr, ri);
                const Spinor<T> vc = chain_vector(P[S], e);
                WalkChain<N, DEPTH + 1, KB, T>::run(P, E, hel, S, vc, cr, ci, Kt);
                chain_acc(rr, ri, cr, ci, sr, si);
            }
            ar = sr;
            ai = si;
        }
    }
};

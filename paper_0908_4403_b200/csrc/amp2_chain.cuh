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
//
// rho table (round 2).  The rho of the LAST attachment -- photon j below a node of n-3 photons --
//     R[(T, i, h_i, j, h_j)] = v(S, i, h_i)_0 + b_j(h_j) v(S, i, h_i)_1,   S = all \ T, i in S, j in T,
// depends on the event only (T = the three photons still to attach), so it is tabulated per event:
// C(n,3) 12 (n-3) complex entries (3 360 at n = 8; build_rho_table).  A node of n-3 photons then needs no
// vector of its own -- its three children are R K, one complex FMA each -- and costs 8 instructions
// (rho, rho A) + 3 x 4 instead of 14 + 3 x 8: per lane 163 k instead of 284 k FMA-pipe instructions
// at n = 8.  Nothing summed over orderings is tabulated: R and K are per-node factors, every ordered
// prefix of up to n-2 photons is still one term of the walk.
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

// Table reads of the unrolled walk go through 32-bit shared-memory addresses: every address is a sum
// of per-photon byte offsets held in registers (one IADD per load instead of a 64-bit LEA pair).
__device__ __forceinline__ Cx<float> lds_cx(unsigned addr, float)
{
    Cx<float> c;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(c.r), "=f"(c.i) : "r"(addr));
    return c;
}
__device__ __forceinline__ Cx<double> lds_cx(unsigned addr, double)
{
    Cx<double> c;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(c.r), "=d"(c.i) : "r"(addr));
    return c;
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

// rho table entries per event: [triple T (colex rank)][i: rank of i in all \ T][h_i][j: rank in T][h_j]
template <int N>
constexpr int kRhoEntries = (N * (N - 1) * (N - 2) / 6) * 12 * (N - 3);

// Reads s_P and s_E (barrier before), ends with a barrier.  One work item per (T, i, h_i): the vector
// v(all \ T, i, h_i) once, then its six rho (j in T, h_j).
template <int N, typename T, typename G = Geometry<N>>
__device__ __forceinline__ void build_rho_table(const PEntry<T>* s_P, const EEntry<T>* s_E, Cx<T>* s_R)
{
    constexpr unsigned NT = N * (N - 1) * (N - 2) / 6, ITEMS = NT * (N - 3) * 2u;
    const int ev_local = threadIdx.x / G::L;
    const unsigned lane = threadIdx.x % G::L;
    const PEntry<T>* P = s_P + ev_local * G::L;
    const EEntry<T>* E = s_E + ev_local * 2 * N;
    Cx<T>* R = s_R + ev_local * kRhoEntries<N>;
    for (unsigned q = lane; q < ITEMS; q += G::L) {
        const unsigned hi = q & 1u, t = q >> 1, islot = t % (N - 3), tr = t / (N - 3);
        // unrank the triple x < y < z: tr = C(z,3) + C(y,2) + x
        unsigned z = 2;
        while ((z + 1) * z * (z - 1) / 6 <= tr) ++z;
        unsigned rem = tr - z * (z - 1) * (z - 2) / 6, y = 1;
        while ((y + 1) * y / 2 <= rem) ++y;
        const unsigned x = rem - y * (y - 1) / 2;
        unsigned i = islot;   // the islot-th photon outside {x, y, z}
        if (i >= x) ++i;
        if (i >= y) ++i;
        if (i >= z) ++i;
        const Spinor<T> v = chain_vector(P[(G::L - 1) ^ (1u << x) ^ (1u << y) ^ (1u << z)], E[2 * i + hi]);
        const unsigned js[3] = {x, y, z};
#pragma unroll
        for (unsigned jslot = 0; jslot < 3; ++jslot)
#pragma unroll
            for (unsigned hj = 0; hj < 2; ++hj) {
                Cx<T> r;
                chain_rho(v, E[2 * js[jslot] + hj], r.r, r.i);
                R[((tr * (N - 3) + islot) * 2 + hi) * 6 + jslot * 2 + hj] = r;
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
    static constexpr int KP = KB * (KB - 1) / 2, KT = KB * (KB - 1) * (KB - 2) / 6;
    // All table addresses are 32-bit shared-memory BYTE addresses / offsets:
    // kp[] = this lane's K-table base of each position pair, jo[] = offset of (j, h_j) per position;
    // rp[] = rho-table base of each position triple p < q < r (at C(r,3) + C(q,2) + p), io[] = offset of
    // (i, h_i) in a triple's block per position (photon id x 12 + h_i x 6 entries; the members of T below
    // i are subtracted at compile time), hb[] = this lane's helicity bit per position x one entry
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ PS, const int (&bit)[K],
                                               const EEntry<T> (&e)[K], const int (&idx)[K],
                                               const unsigned (&kp)[KP], const unsigned (&rp)[KT],
                                               const unsigned (&jo)[KB], const unsigned (&io)[KB], const unsigned (&hb)[KB],
                                               const Spinor<T>& v, T& ar, T& ai)
    {
        static_assert(K >= 4, "a node of n-4 photons attaches i; the tables close the three levels below it");
        T sr = 0, si = 0;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            T rr, ri;
            chain_rho(v, e[i], rr, ri);
            T cr = 0, ci = 0;
            if constexpr (K == 4) {
                // the child holds n-3 photons; T = the other three positions p < q < r
                const int p = idx[i == 0 ? 1 : 0], q = idx[i <= 1 ? 2 : 1], r = idx[i == 3 ? 2 : 3];
                const int below = (p < idx[i]) + (q < idx[i]) + (r < idx[i]);
                constexpr unsigned EB = sizeof(Cx<T>);
                const unsigned R = rp[r * (r - 1) * (r - 2) / 6 + q * (q - 1) / 2 + p] + io[idx[i]] - 12 * EB * below;
                const Cx<T> r0 = lds_cx(R + hb[p], T()), r1 = lds_cx(R + hb[q] + 2 * EB, T()),
                            r2 = lds_cx(R + hb[r] + 4 * EB, T());
                const Cx<T> k0 = lds_cx(kp[r * (r - 1) / 2 + q] + jo[p], T()), k1 = lds_cx(kp[r * (r - 1) / 2 + p] + jo[q], T()),
                            k2 = lds_cx(kp[q * (q - 1) / 2 + p] + jo[r], T());
                chain_acc(r0.r, r0.i, k0.r, k0.i, cr, ci);
                chain_acc(r1.r, r1.i, k1.r, k1.i, cr, ci);
                chain_acc(r2.r, r2.i, k2.r, k2.i, cr, ci);
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
                ChainBottom<K - 1, KB, T>::run(Pn, sub_bit, sub_e, sub_idx, kp, rp, jo, io, hb, vc, cr, ci);
            }
            chain_acc(rr, ri, cr, ci, sr, si);
        }
        ar = sr;
        ai = si;
    }
};

// Depth-first walk of the upper levels (`used` = photons already attached, uniform over the CTA;
// returns A(node) in ar, ai);
// when KB photons remain the unrolled ChainBottom<KB> takes over.  Needs N - KB >= 0 and KB >= 4.
template <int N, int DEPTH, int KB, typename T>
struct WalkChain {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                               unsigned hel, unsigned used, const Spinor<T>& v, T& ar, T& ai,
                                               const Cx<T>* __restrict__ Kt, const Cx<T>* __restrict__ Rt)
    {
        unsigned avail = ((1u << N) - 1u) & ~used;
        if constexpr (N - DEPTH == KB) {
            constexpr int KP = KB * (KB - 1) / 2, KT = KB * (KB - 1) * (KB - 2) / 6;
            constexpr unsigned EB = sizeof(Cx<T>);
            int bit[KB], idx[KB], photon[KB];
            unsigned jo[KB], io[KB], hb[KB], hbit[KB];
            EEntry<T> e[KB];
#pragma unroll
            for (int m = 0; m < KB; ++m) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                bit[m] = 1 << i;
                hbit[m] = (hel >> i) & 1u;
                e[m] = E[2 * i + hbit[m]];
                idx[m] = m;
                photon[m] = i;
                hb[m] = EB * hbit[m];
                jo[m] = EB * (8 * i + 4 * hbit[m]);
                io[m] = EB * (12 * i + 6 * hbit[m]);
            }
            const unsigned k_base = (unsigned)__cvta_generic_to_shared(Kt), r_base = (unsigned)__cvta_generic_to_shared(Rt);
            unsigned kp[KP];
#pragma unroll
            for (int q = 1; q < KB; ++q)
#pragma unroll
                for (int p = 0; p < q; ++p) {  // photon[] is increasing
                    const int pair = photon[q] * (photon[q] - 1) / 2 + photon[p];
                    kp[q * (q - 1) / 2 + p] = k_base + EB * (pair * (N * 8) + 2 * hbit[p] + hbit[q]);
                }
            unsigned rp[KT];
#pragma unroll
            for (int r = 2; r < KB; ++r)
#pragma unroll
                for (int q = 1; q < r; ++q)
#pragma unroll
                    for (int p = 0; p < q; ++p) {  // colex rank of the photon triple
                        const int tr = photon[r] * (photon[r] - 1) * (photon[r] - 2) / 6 + photon[q] * (photon[q] - 1) / 2 + photon[p];
                        rp[r * (r - 1) * (r - 2) / 6 + q * (q - 1) / 2 + p] = r_base + EB * (tr * (12 * (N - 3)));
                    }
            ChainBottom<KB, KB, T>::run(P + used, bit, e, idx, kp, rp, jo, io, hb, v, ar, ai);
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
                WalkChain<N, DEPTH + 1, KB, T>::run(P, E, hel, S, vc, cr, ci, Kt, Rt);
                chain_acc(rr, ri, cr, ci, sr, si);
            }
            ar = sr;
            ai = si;
        }
    }
};

// amp2_chain.cuh -- the permutation tree of eq. (6) with every off-shell spinor held
// in factorised form (product code, v9; amp2.cu uses it for n >= 6; amp2_thread.cu borrows its node helpers).
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
// only, so it is tabulated per event (build_chain_table), indexed by the triple T = {j, a, b} of the
// photons not in the node's parent, x < y < z, their helicities and which of them is j,
//     K[(rank(T) 3 + slot(j)) 8 + 4 h_x + 2 h_y + h_z] = W_ab(h_a,h_b) . v(all \ {a,b}, j, h_j),
// so that the three entries a node of n-3 photons needs (j = x, y, z) sit at ONE lane-dependent address
// plus constants, and the 8 helicity combinations a warp reads at once are adjacent (one wavefront),
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
#include <type_traits>

#include "amp2_common.cuh"


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
// the three K entries of one node: the same lane-dependent address plus 0, 8 and 16 entries
__device__ __forceinline__ void lds_cx3(unsigned addr, Cx<float>& a, Cx<float>& b, Cx<float>& c)
{
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(a.r), "=f"(a.i) : "r"(addr));
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+64];" : "=f"(b.r), "=f"(b.i) : "r"(addr));
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+128];" : "=f"(c.r), "=f"(c.i) : "r"(addr));
}
__device__ __forceinline__ void lds_cx3(unsigned addr, Cx<double>& a, Cx<double>& b, Cx<double>& c)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a.r), "=d"(a.i) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+128];" : "=d"(b.r), "=d"(b.i) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+256];" : "=d"(c.r), "=d"(c.i) : "r"(addr));
}

// fp32 "packed" layout (HEGET_CHAIN_PACKED32): the three entries a node of n-3 photons reads from the K table,
// and the three it reads from the rho table, are ADJACENT (one 16-byte and one 8-byte load at constant offsets
// from one lane-dependent address) instead of three loads at three lane-dependent addresses: a row holds, for
// each of the 8 helicity assignments h_T = 4 h_x + 2 h_y + h_z of the triple, a chunk of 4 entries (3 used);
// the chunks of h_T >= 4 are shifted by 2 entries so that the 8 chunks a warp reads at once fall into distinct
// banks.  The rho table grows 4x (the rho of photon j is stored under every assignment of the other two), which
// fp32 can afford (n = 8: 152 KB) and fp64 cannot.
#ifndef HEGET_CHAIN_PACKED32
#define HEGET_CHAIN_PACKED32 1
#endif
template <typename T>
constexpr bool kPacked = (sizeof(T) == 4) && (HEGET_CHAIN_PACKED32 != 0);
constexpr unsigned kPackRow = 8 * 4 + 2;                                   // entries per row
__host__ __device__ constexpr unsigned pack_off(unsigned ht) { return 4u * ht + (ht >= 4u ? 2u : 0u); }

// packed fp32: three adjacent entries
__device__ __forceinline__ void lds_cx3_packed(unsigned addr, Cx<float>& a, Cx<float>& b, Cx<float>& c)
{
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(a.r), "=f"(a.i), "=f"(b.r), "=f"(b.i) : "r"(addr));
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+16];" : "=f"(c.r), "=f"(c.i) : "r"(addr));
}
__device__ __forceinline__ void lds_cx3_packed(unsigned, Cx<double>&, Cx<double>&, Cx<double>&) {}   // never used

// K table entries per event: [triple T (colex rank)][slot of j in T][4 h_x + 2 h_y + h_z]; packed: [T][h_T chunk][slot]
template <int N, typename T>
constexpr int kChainEntries = (N * (N - 1) * (N - 2) / 6) * (kPacked<T> ? (int)kPackRow : 24);

// unrank a photon triple x < y < z from its colex rank tr = C(z,3) + C(y,2) + x
__device__ __forceinline__ void unrank_triple(unsigned tr, unsigned& x, unsigned& y, unsigned& z)
{
    z = 2;
    while ((z + 1) * z * (z - 1) / 6 <= tr) ++z;
    const unsigned rem = tr - z * (z - 1) * (z - 2) / 6;
    y = 1;
    while ((y + 1) * y / 2 <= rem) ++y;
    x = rem - y * (y - 1) / 2;
}

// Reads s_P, s_E and the pair closing table s_W (barrier before), ends with a barrier.  One work item
// per (T, j in T, h_j): the vector v(all \ {a,b}, j, h_j) once, then its dot products with the four W
// rows of the pair {a, b} = T \ j.
template <int N, typename T, typename G = Geometry<N>>
__device__ __forceinline__ void build_chain_table(const PEntry<T>* s_P, const EEntry<T>* s_E, const Spinor<T>* s_W,
                                                  Cx<T>* s_K)
{
    constexpr unsigned NT = N * (N - 1) * (N - 2) / 6, ITEMS = NT * 6u;
    const int ev_local = threadIdx.x / G::L;
    const unsigned lane = threadIdx.x % G::L;
    const PEntry<T>* P = s_P + ev_local * G::L;
    const EEntry<T>* E = s_E + ev_local * 2 * N;
    const Spinor<T>* W = s_W + ev_local * 4 * (N * (N - 1) / 2);
    Cx<T>* K = s_K + ev_local * kChainEntries<N, T>;
    for (unsigned q = lane; q < ITEMS; q += G::L) {
        const unsigned hj = q & 1u, t = q >> 1, slot = t % 3u, tr = t / 3u;
        unsigned x, y, z;
        unrank_triple(tr, x, y, z);
        const unsigned j = slot == 0 ? x : (slot == 1 ? y : z);
        const unsigned a = slot == 0 ? y : x, b = slot == 2 ? y : z;   // a < b: the pair that closes
        const Spinor<T> v = chain_vector(P[(G::L - 1) ^ (1u << a) ^ (1u << b)], E[2 * j + hj]);
        const unsigned pair = b * (b - 1) / 2 + a;
        // bit weight of h_j, h_a, h_b in 4 h_x + 2 h_y + h_z
        const unsigned wj = 4u >> slot, wa = slot == 0 ? 2u : 4u, wb = slot == 2 ? 2u : 1u;
#pragma unroll
        for (unsigned h = 0; h < 4; ++h) {   // h = 2 h_a + h_b
            const Spinor<T> w = W[4 * pair + h];
            Cx<T> k;
            k.r = fma(w.r0, v.r0, fma(-w.i0, v.i0, fma(w.r1, v.r1, -(w.i1 * v.i1))));
            k.i = fma(w.r0, v.i0, fma(w.i0, v.r0, fma(w.r1, v.i1, w.i1 * v.r1)));
            const unsigned ht = wj * hj + wa * (h >> 1) + wb * (h & 1u);
            if constexpr (kPacked<T>)
                K[tr * kPackRow + pack_off(ht) + slot] = k;
            else
                K[(tr * 3u + slot) * 8u + ht] = k;
        }
    }
    __syncthreads();
}

// rho table entries per event: [triple T (colex rank)][i: rank of i in all \ T][h_i][j: rank in T][h_j];
// packed: [T][i][h_i] rows of [h_T chunk][j]
template <int N, typename T>
constexpr int kRhoEntries = (N * (N - 1) * (N - 2) / 6) * (N - 3) * (kPacked<T> ? 2 * (int)kPackRow : 12);

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
    Cx<T>* R = s_R + ev_local * kRhoEntries<N, T>;
    for (unsigned q = lane; q < ITEMS; q += G::L) {
        const unsigned hi = q & 1u, t = q >> 1, islot = t % (N - 3), tr = t / (N - 3);
        unsigned x, y, z;
        unrank_triple(tr, x, y, z);
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
                if constexpr (kPacked<T>) {
                    const unsigned row = (tr * (N - 3) + islot) * 2 + hi, w = 4u >> jslot;   // bit of h_j in h_T
#pragma unroll
                    for (unsigned ht = 0; ht < 8; ++ht)
                        if (((ht / w) & 1u) == hj) R[row * kPackRow + pack_off(ht) + jslot] = r;
                } else {
                    R[((tr * (N - 3) + islot) * 2 + hi) * 6 + jslot * 2 + hj] = r;
                }
            }
    }
    __syncthreads();
}

// Bottom levels, fully unrolled (as Bottom<K> of amp2_tree.cuh: the K photons still to attach are
// compile-time-indexed register arrays, choosing a child is register renaming).  idx[] = positions
// of the remaining photons in the list of KB photons the unrolled part started from, kp[] = this
// lane's K-table base of each position pair p < q (at q(q-1)/2 + p), jo[] = offset of (j, h_j)
// for each position.  Ends at K = 3: the children are the nodes of n-2 photons, closed with K.
// EA = EEntry<T> (the list's E' entries held in registers) or unsigned (their 32-bit shared-memory address;
// a and b are re-read where they are used: 4 T registers less per remaining photon, which is what lets six
// levels nearly fit in fp64)
template <typename T> __device__ __forceinline__ Cx<T> chain_ea(const EEntry<T>& e) { return {e.ar, e.ai}; }
template <typename T> __device__ __forceinline__ Cx<T> chain_eb(const EEntry<T>& e) { return {e.br, e.bi}; }
template <typename T> __device__ __forceinline__ Cx<T> chain_ea(unsigned e) { return lds_cx(e, T()); }
template <typename T> __device__ __forceinline__ Cx<T> chain_eb(unsigned e) { return lds_cx(e + (unsigned)sizeof(Cx<T>), T()); }

template <int K, int KB, typename T, typename EA = EEntry<T>>
struct ChainBottom {
    static constexpr int KT = KB * (KB - 1) * (KB - 2) / 6;
    // All table addresses are 32-bit shared-memory BYTE addresses / offsets, per position triple p < q < r
    // of the list (at C(r,3) + C(q,2) + p): kt[] = address of this lane's three K entries (the lane's
    // helicities of the triple folded in), rp[] = rho-table base of the triple; io[] = offset of (i, h_i) in
    // a triple's rho block per position (photon id x 12 + h_i x 6 entries; the members of T below i are
    // subtracted at compile time), hb[] = this lane's helicity bit per position x one entry
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ PS, const int (&bit)[K],
                                               const EA (&e)[K], const int (&idx)[K],
                                               const unsigned (&kt)[KT], const unsigned (&rp)[KT],
                                               const unsigned (&io)[KB], const unsigned (&hb)[KB],
                                               const Spinor<T>& v, T& ar, T& ai)
    {
        static_assert(K >= 4, "a node of n-4 photons attaches i; the tables close the three levels below it");
        T sr = 0, si = 0;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            T rr, ri;
            EEntry<T> ei;
            {
                const Cx<T> b = chain_eb<T>(e[i]);
                ei.br = b.r;
                ei.bi = b.i;
            }
            chain_rho(v, ei, rr, ri);
            T cr = 0, ci = 0;
            if constexpr (K == 4) {
                // the child holds n-3 photons; T = the other three positions p < q < r
                const int p = idx[i == 0 ? 1 : 0], q = idx[i <= 1 ? 2 : 1], r = idx[i == 3 ? 2 : 3];
                const int below = (p < idx[i]) + (q < idx[i]) + (r < idx[i]);
                constexpr unsigned EB = sizeof(Cx<T>);
                const int t = r * (r - 1) * (r - 2) / 6 + q * (q - 1) / 2 + p;
                Cx<T> r0, r1, r2, k0, k1, k2;
                if constexpr (kPacked<T>) {
                    lds_cx3_packed(rp[t] + io[idx[i]] - 2 * kPackRow * EB * below, r0, r1, r2);
                    lds_cx3_packed(kt[t], k0, k1, k2);
                } else {
                    const unsigned R = rp[t] + io[idx[i]] - 12 * EB * below;
                    r0 = lds_cx(R + hb[p], T());
                    r1 = lds_cx(R + hb[q] + 2 * EB, T());
                    r2 = lds_cx(R + hb[r] + 4 * EB, T());
                    lds_cx3(kt[t], k0, k1, k2);
                }
                chain_acc(r0.r, r0.i, k0.r, k0.i, cr, ci);
                chain_acc(r1.r, r1.i, k1.r, k1.i, cr, ci);
                chain_acc(r2.r, r2.i, k2.r, k2.i, cr, ci);
            } else {
                int sub_bit[K - 1];
                EA sub_e[K - 1];
                int sub_idx[K - 1];
#pragma unroll
                for (int m = 0; m < K - 1; ++m) {
                    sub_bit[m] = bit[m + (m >= i ? 1 : 0)];
                    sub_e[m] = e[m + (m >= i ? 1 : 0)];
                    sub_idx[m] = idx[m + (m >= i ? 1 : 0)];
                }
                const PEntry<T>* Pn = PS + bit[i];
                {
                    const Cx<T> a = chain_ea<T>(e[i]);
                    ei.ar = a.r;
                    ei.ai = a.i;
                }
                const Spinor<T> vc = chain_vector(*Pn, ei);
                ChainBottom<K - 1, KB, T, EA>::run(Pn, sub_bit, sub_e, sub_idx, kt, rp, io, hb, vc, cr, ci);
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
template <int N, int DEPTH, int KB, typename T, bool E_BY_PTR = false>
struct WalkChain {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                               unsigned hel, unsigned used, const Spinor<T>& v, T& ar, T& ai,
                                               const Cx<T>* __restrict__ Kt, const Cx<T>* __restrict__ Rt)
    {
        unsigned avail = ((1u << N) - 1u) & ~used;
        if constexpr (N - DEPTH == KB) {
            constexpr int KT = KB * (KB - 1) * (KB - 2) / 6;
            constexpr unsigned EB = sizeof(Cx<T>);
            int bit[KB], idx[KB], photon[KB];
            unsigned io[KB], hb[KB], hbit[KB];
            using EA = std::conditional_t<E_BY_PTR, unsigned, EEntry<T>>;
            EA e[KB];
#pragma unroll
            for (int m = 0; m < KB; ++m) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                bit[m] = 1 << i;
                hbit[m] = (hel >> i) & 1u;
                if constexpr (E_BY_PTR)
                    e[m] = (unsigned)__cvta_generic_to_shared(&E[2 * i + hbit[m]]);
                else
                    e[m] = E[2 * i + hbit[m]];
                idx[m] = m;
                photon[m] = i;
                hb[m] = EB * hbit[m];
                io[m] = kPacked<T> ? EB * kPackRow * (2 * i + hbit[m]) : EB * (12 * i + 6 * hbit[m]);
            }
            const unsigned k_base = (unsigned)__cvta_generic_to_shared(Kt), r_base = (unsigned)__cvta_generic_to_shared(Rt);
            unsigned rp[KT], kt[KT];
#pragma unroll
            for (int r = 2; r < KB; ++r)
#pragma unroll
                for (int q = 1; q < r; ++q)
#pragma unroll
                    for (int p = 0; p < q; ++p) {  // colex rank of the photon triple
                        const int tr = photon[r] * (photon[r] - 1) * (photon[r] - 2) / 6 + photon[q] * (photon[q] - 1) / 2 + photon[p];
                        const int t = r * (r - 1) * (r - 2) / 6 + q * (q - 1) / 2 + p;
                        if constexpr (kPacked<T>) {
                            // chunk of this lane's h_T = 4 h_p + 2 h_q + h_r: pack_off is additive in the three bits
                            const unsigned hoff = EB * (pack_off(4) * hbit[p] + pack_off(2) * hbit[q] + pack_off(1) * hbit[r]);
                            rp[t] = r_base + EB * (tr * (2 * kPackRow * (N - 3))) + hoff;
                            kt[t] = k_base + EB * (tr * kPackRow) + hoff;
                        } else {
                            rp[t] = r_base + EB * (tr * (12 * (N - 3)));
                            kt[t] = k_base + EB * (tr * 24 + 4 * hbit[p] + 2 * hbit[q] + hbit[r]);
                        }
                    }
            ChainBottom<KB, KB, T, EA>::run(P + used, bit, e, idx, kt, rp, io, hb, v, ar, ai);
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
                WalkChain<N, DEPTH + 1, KB, T, E_BY_PTR>::run(P, E, hel, S, vc, cr, ci, Kt, Rt);
                chain_acc(rr, ri, cr, ci, sr, si);
            }
            ar = sr;
            ai = si;
        }
    }
};

// amp2_thread.cu -- heget_amp2 for n = 2 .. 6: one THREAD per event (n = 6: two or four lanes) (product code).
//
// This is the paper's own mapping (one phase-space point per thread) applied to the
// permutation tree of eq. (6) in the two-component, factorised form of amp2_tables.cuh
// and amp2_chain.cuh.  For n <= 4 an event's whole tree, for ALL 2^n photon-helicity assignments, fits
// one thread's registers (2^n complex accumulators) plus a few per-thread columns of shared memory
// (n = 5, further down: the 32 accumulators live in the column too),
// and the thread never idles: the lane-per-helicity kernel of amp2.cu spends most of a 4-photon event
// in table phases that occupy 4, 6 or 14 of an event's 16 lanes and in the index arithmetic of its
// work-item loops, which here is all folded at compile time.
//
// Per event (sigma_1 = +1 only; parity doubles it, sigma_1 = sigma_2 vanishes):
//   a1  the thread reads its event's (n+2) four-vectors with 16-byte loads;
//   a4  vxxxx0 of every photon, both helicities: E' entries (a, b) (make_photon_entries);
//   a5  every non-empty proper subset S: P_S = -g/t_S (p1 - K_S)-slash block.  The components are
//       light-cone sums in plain fp64; t_S of eq. (8) is exact on the fp64 inputs as
//       given (reading R10) from per-event invariants held as unevaluated double-double sums,
//           t_S = sum_{i in S} (k_i.k_i - 2 p1.k_i) + sum_{i<j in S} 2 k_i.k_j ,
//       n(n+3)/2 Minkowski products per event instead of a double-double four-vector per subset
//       (the fp32 kernel takes t_S = p+ p- - pT^2 in plain fp64);
//   a6  fvixx0 nodes in factorised form psi = z v: v(S, i, h_i) = P_S (-1, a_i)^T, rho = v_0 + b_j v_1;
//       every ordered prefix of up to n-2 photons is one node, computed once per helicity
//       assignment OF THE PREFIX (2^|S| values, not 2^n);
//   a7  the two orderings below a prefix of n-2 photons close with the pair closing row
//       W_ab = U_b E'_a + U_a E'_b (U_b = <vbar| E'_b P_{all\b}); with the rank-one form of E',
//       row . E' = (-u_0 + a u_1) (1, b).  For n = 4 the two ordered prefixes (i,j), (j,i) of a pair close
//       with the same rows: ampsum(h) += W_ab(h_a,h_b) . [psi_2(i,j) + psi_2(j,i)](h_i,h_j);
//   a8  sum_h |ampsum(h)|^2 and the constant factors, one 8-byte store.
// Shared memory (n = 4 only): the thread's 8 vectors v({i}, i, h), 8 closing rows U_b(h) and 6 pair
// entries P_{ij}, as columns [word][thread] (conflict-free 16-byte / 8-byte accesses).
#include "amp2_chain.cuh"

namespace {

#ifndef HEGET_THREAD_CTA
#define HEGET_THREAD_CTA 64        // threads (= events) per CTA
#endif
#ifndef HEGET_THREAD_MINB64_N4
#define HEGET_THREAD_MINB64_N4 4   // __launch_bounds__ min CTAs per SM: fp64 4 photons (255 registers)
#endif
#ifndef HEGET_THREAD_MINB32_N4
#define HEGET_THREAD_MINB32_N4 8   // fp32 4 photons: 128 registers (16-48 B of spills): 0.152 -> 0.139 ms against 6 (168 registers)
#endif
#ifndef HEGET_THREAD_MINB_SMALL
#define HEGET_THREAD_MINB_SMALL 6  // n = 2, 3
#endif

// unevaluated sum hi + lo; not normalised (lo may be comparable to hi after cancellation)
__device__ __forceinline__ void dd_add_to(dd& a, const dd& b)
{
    const dd s = dd_two_sum(a.hi, b.hi);
    a.hi = s.hi;
    a.lo = __dadd_rn(a.lo, __dadd_rn(s.lo, b.lo));
}

// a.b = a0 b0 - a1 b1 - a2 b2 - a3 b3 as an unevaluated sum: exact products (FMA), the high parts
// summed error-free, every rounding error collected in lo.  For two massless vectors (photons) the running sum
// dominates the next term -- a0 b0 - a1 b1 >= |a2 b2| + |a3 b3| and a0 b0 - a1 b1 - a2 b2 >= |a3 b3| by
// Cauchy-Schwarz on (|a1|,|a2|,|a3|).(|b1|,|b2|,|b3|) <= a0 b0 -- so the three additions are Dekker's
// FastTwoSum (3 operations) instead of Knuth's TwoSum (6); an ulp-level violation from the rounding of the
// running sum only moves a second-order error
__device__ __forceinline__ dd dd_minkowski(const double (&a)[4], const double (&b)[4])
{
    const dd p0 = dd_two_prod(a[0], b[0]), p1 = dd_two_prod(a[1], b[1]), p2 = dd_two_prod(a[2], b[2]),
             p3 = dd_two_prod(a[3], b[3]);
    const dd s1 = dd_fast_two_sum(p0.hi, -p1.hi), s2 = dd_fast_two_sum(s1.hi, -p2.hi), s3 = dd_fast_two_sum(s2.hi, -p3.hi);
    const double lo = __dadd_rn(__dadd_rn(__dsub_rn(__dsub_rn(__dsub_rn(p0.lo, p1.lo), p2.lo), p3.lo), s1.lo),
                                __dadd_rn(s2.lo, s3.lo));
    return {s3.hi, lo};
}

template <typename T>
__device__ __forceinline__ Cx<T> cx_mul(const Cx<T>& a, const Cx<T>& b)
{
    return {fma(a.r, b.r, -(a.i * b.i)), fma(a.r, b.i, a.i * b.r)};
}

// -u_0 + a u_1 for a row u = (u_0, u_1): the scalar of row . E' = (-u_0 + a u_1) (1, b)
template <typename T>
__device__ __forceinline__ Cx<T> row_scalar(const Spinor<T>& u, const EEntry<T>& e)
{
    return {fma(e.ar, u.r1, fma(-e.ai, u.i1, -u.r0)), fma(e.ar, u.i1, fma(e.ai, u.r1, -u.i0))};
}

// W . v (two-component dot product, no conjugation)
template <typename T>
__device__ __forceinline__ Cx<T> row_dot(const Spinor<T>& w, const Spinor<T>& v)
{
    return {fma(w.r0, v.r0, fma(-w.i0, v.i0, fma(w.r1, v.r1, -(w.i1 * v.i1)))),
            fma(w.r0, v.i0, fma(w.i0, v.r0, fma(w.r1, v.i1, w.i1 * v.r1)))};
}

// Per-event kinematics shared by all subsets: light-cone components of every photon and, for the
// fp64 kernel, the invariants c_i = k_i.k_i - 2 p1.k_i and d_ij = 2 k_i.k_j as double-doubles.
template <int N, bool EXACT>
struct Kinematics {
    double kp[N], km[N], kx[N], ky[N];
    double two_e1, coupling;   // 2 E1; -g * scale
    dd c[EXACT ? N : 1];
    dd d[EXACT ? N * (N - 1) / 2 : 1];   // pair i < j at j (j - 1) / 2 + i

    __device__ __forceinline__ void init(const double (&k)[N][4], double e1, double g, double scale)
    {
        two_e1 = 2.0 * e1;
        coupling = -g * scale;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            kp[i] = k[i][0] + k[i][3];
            km[i] = k[i][0] - k[i][3];
            kx[i] = k[i][1];
            ky[i] = k[i][2];
        }
        if constexpr (EXACT) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
                // p1 = (E1, 0, 0, E1): 2 p1.k_i = 2 E1 (w_i - kz_i), the difference by TwoSum
                const dd u = dd_two_sum(k[i][0], -k[i][3]);
                dd q = dd_two_prod(two_e1, u.hi);
                q.lo = __fma_rn(two_e1, u.lo, q.lo);
                c[i] = dd_minkowski(k[i], k[i]);
                dd_add_to(c[i], dd_neg(q));
            }
#pragma unroll
            for (int j = 1; j < N; ++j)
#pragma unroll
                for (int i = 0; i < j; ++i) {
                    const dd m = dd_minkowski(k[i], k[j]);
                    d[j * (j - 1) / 2 + i] = {2.0 * m.hi, 2.0 * m.lo};
                }
        }
    }

    // P entry of subset S (compile-time constant after unrolling)
    template <typename T>
    __device__ __forceinline__ PEntry<T> subset(unsigned S) const
    {
        double skp = 0.0, skm = 0.0, skx = 0.0, sky = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i)
            if ((S >> i) & 1u) {
                skp += kp[i];
                skm += km[i];
                skx += kx[i];
                sky += ky[i];
            }
        const double pp = two_e1 - skp;
        double t;
        if constexpr (EXACT) {
            dd acc = {0.0, 0.0};
            bool first = true;
#pragma unroll
            for (int i = 0; i < N; ++i)
                if ((S >> i) & 1u) {
                    if (first) acc = c[i]; else dd_add_to(acc, c[i]);
                    first = false;
                }
#pragma unroll
            for (int j = 1; j < N; ++j)
#pragma unroll
                for (int i = 0; i < j; ++i)
                    if (((S >> i) & 1u) && ((S >> j) & 1u)) dd_add_to(acc, d[j * (j - 1) / 2 + i]);
            t = __dadd_rn(acc.hi, acc.lo);
        } else {
            t = -fma(pp, skm, fma(skx, skx, sky * sky));   // p+ p- - pT^2, both terms <= 0
        }
        const double f = coupling * fast_rcp(t);
        PEntry<T> out;
        out.pp = (T)(f * pp);
        out.pm = (T)(-f * skm);
        out.px = (T)(-f * skx);
        out.py = (T)(-f * sky);
        return out;
    }
};

// per-thread column store in shared memory: word w of this thread at col[w * CTA]
template <typename T>
__device__ __forceinline__ void put(Cx<T>* col, int w, const Spinor<T>& s)
{
    col[(2 * w) * HEGET_THREAD_CTA] = {s.r0, s.i0};
    col[(2 * w + 1) * HEGET_THREAD_CTA] = {s.r1, s.i1};
}
template <typename T>
__device__ __forceinline__ Spinor<T> get(const Cx<T>* col, int w)
{
    const Cx<T> a = col[(2 * w) * HEGET_THREAD_CTA], b = col[(2 * w + 1) * HEGET_THREAD_CTA];
    return {a.r, a.i, b.r, b.i};
}
template <typename T>
__device__ __forceinline__ void put(Cx<T>* col, int w, const PEntry<T>& p)
{
    col[(2 * w) * HEGET_THREAD_CTA] = {p.pp, p.pm};
    col[(2 * w + 1) * HEGET_THREAD_CTA] = {p.px, p.py};
}
template <typename T>
__device__ __forceinline__ PEntry<T> get_p(const Cx<T>* col, int w)
{
    const Cx<T> a = col[(2 * w) * HEGET_THREAD_CTA], b = col[(2 * w + 1) * HEGET_THREAD_CTA];
    return {a.r, a.i, b.r, b.i};
}

// pair closing row W_ab(h_a, h_b) = U_b(h_b) E'_a(h_a) + U_a(h_a) E'_b(h_b), rank-one form of E'
template <typename T>
__device__ __forceinline__ Spinor<T> pair_row(const Spinor<T>& ua, const Spinor<T>& ub, const EEntry<T>& ea,
                                              const EEntry<T>& eb)
{
    const Cx<T> sba = row_scalar(ub, ea), sab = row_scalar(ua, eb);
    const Cx<T> ba = {ea.br, ea.bi}, bb = {eb.br, eb.bi};
    const Cx<T> x = cx_mul(sba, ba);
    Spinor<T> w;
    w.r0 = sba.r + sab.r;
    w.i0 = sba.i + sab.i;
    w.r1 = fma(sab.r, bb.r, fma(-sab.i, bb.i, x.r));
    w.i1 = fma(sab.r, bb.i, fma(sab.i, bb.r, x.i));
    return w;
}

constexpr int kColumnWords4 = 2 * (8 + 8 + 6);   // Cx words per thread, n = 4: v1[8], U[8], P_ij[6]

template <int N, typename T>
constexpr int kMinBlocks = (N == 4) ? ((sizeof(T) == 8) ? HEGET_THREAD_MINB64_N4 : HEGET_THREAD_MINB32_N4)
                                    : HEGET_THREAD_MINB_SMALL;

template <int N, typename T>
__global__ void __launch_bounds__(HEGET_THREAD_CTA, kMinBlocks<N, T>)
amp2_thread_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    static_assert(N >= 2 && N <= 4, "one thread per event holds 2^N accumulators: n <= 4");
    constexpr int L = 1 << N;
    constexpr unsigned ALL = L - 1;
    __shared__ Cx<T> s_col[(N == 4) ? kColumnWords4 * HEGET_THREAD_CTA : 1];

    int64_t ev = (int64_t)blockIdx.x * HEGET_THREAD_CTA + threadIdx.x;
    const bool live = ev < n_events;
    if (!live) ev = n_events - 1;

    // a1: (n+2) four-vectors, 16-byte loads
    double e1, e2, k[N][4];
    {
        const double2* src = reinterpret_cast<const double2*>(momenta) + ev * (2 * (N + 2));
        e1 = __ldg(src).x;
        e2 = __ldg(src + 2).x;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const double2 a = __ldg(src + 4 + 2 * i), b = __ldg(src + 5 + 2 * i);
            k[i][0] = a.x; k[i][1] = a.y; k[i][2] = b.x; k[i][3] = b.y;
        }
    }
    const double shat = 4.0 * e1 * e2;
    const double scale = (sizeof(T) == 4) ? sqrt(shat) : 1.0;   // fp32 works in units of sqrt(s_hat)

    // a4: E' entries e[i][h], h = 1: lambda = +1
    EEntry<T> e[N][2];
    double norm = 2.0 * g * g * shat;   // 2 (parity) g^2 (closing vertex) s_hat (spinor norms) prod s_i^2 / 2
#pragma unroll
    for (int i = 0; i < N; ++i) norm *= 0.5 * make_photon_entries<T>(k[i], &e[i][1], &e[i][0]);
    if constexpr (sizeof(T) == 4) {
        const double inv = 1.0 / shat;
#pragma unroll
        for (int i = 0; i < N - 1; ++i) norm *= inv;
    }

    // a5: kinematic invariants of the event
    Kinematics<N, sizeof(T) == 8> kin;
    kin.init(k, e1, g, scale);

    Cx<T> amp[L];
#pragma unroll
    for (int h = 0; h < L; ++h) amp[h] = {(T)0, (T)0};

    if constexpr (N == 2) {
        // ampsum(h) = W_01(h_0, h_1) . (1, 0): the two diagrams
        Spinor<T> u[2][2];
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const PEntry<T> p = kin.template subset<T>(ALL ^ (1u << b));
#pragma unroll
            for (int h = 0; h < 2; ++h) u[b][h] = closing_entry(e[b][h], p);
        }
#pragma unroll
        for (int h0 = 0; h0 < 2; ++h0)
#pragma unroll
            for (int h1 = 0; h1 < 2; ++h1) {
                const Spinor<T> w = pair_row(u[0][h0], u[1][h1], e[0][h0], e[1][h1]);
                amp[h0 | (h1 << 1)] = {w.r0, w.i0};
            }
    } else if constexpr (N == 3) {
        Spinor<T> u[3][2];
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const PEntry<T> p = kin.template subset<T>(ALL ^ (1u << b));
#pragma unroll
            for (int h = 0; h < 2; ++h) u[b][h] = closing_entry(e[b][h], p);
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const int a = (i == 0) ? 1 : 0, b = (i == 2) ? 1 : 2;   // the other two, a < b
            const PEntry<T> p = kin.template subset<T>(1u << i);
            Spinor<T> v[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) v[h] = chain_vector(p, e[i][h]);
#pragma unroll
            for (int ha = 0; ha < 2; ++ha)
#pragma unroll
                for (int hb = 0; hb < 2; ++hb) {
                    const Spinor<T> w = pair_row(u[a][ha], u[b][hb], e[a][ha], e[b][hb]);
#pragma unroll
                    for (int hi = 0; hi < 2; ++hi) {
                        const Cx<T> kk = row_dot(w, v[hi]);
                        const int h = (hi << i) | (ha << a) | (hb << b);
                        amp[h].r += kk.r;
                        amp[h].i += kk.i;
                    }
                }
        }
    } else {
        Cx<T>* col = s_col + threadIdx.x;
        // tables: v1[2 i + h] = v({i}, i, h), U[2 b + h], P_ij at pair index j (j - 1) / 2 + i
        constexpr int V1 = 0, UU = 8, PP = 16;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const PEntry<T> p1 = kin.template subset<T>(1u << i);
            const PEntry<T> p3 = kin.template subset<T>(ALL ^ (1u << i));
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                put(col, V1 + 2 * i + h, chain_vector(p1, e[i][h]));
                put(col, UU + 2 * i + h, closing_entry(e[i][h], p3));
            }
        }
#pragma unroll
        for (int j = 1; j < 4; ++j)
#pragma unroll
            for (int i = 0; i < j; ++i)
                put(col, PP + j * (j - 1) / 2 + i, kin.template subset<T>((1u << i) | (1u << j)));
        // the columns are private to the thread; the fence only keeps the compiler from forwarding the
        // stored values through registers (which spills) instead of reloading them where they are used
        __syncwarp();

        // the 12 ordered prefixes (i, j), grouped by the unordered pair: both close with W_ab, {a,b} the rest
#pragma unroll
        for (int j = 1; j < 4; ++j)
#pragma unroll
            for (int i = 0; i < j; ++i) {
                const unsigned rest = ALL ^ (1u << i) ^ (1u << j);   // {a < b}: folded after unrolling
                const int a = (rest & 1u) ? 0 : ((rest & 2u) ? 1 : 2);
                const int b = (rest & 8u) ? 3 : ((rest & 4u) ? 2 : 1);
                // Psi(h_i, h_j) = psi_2(i, j) + psi_2(j, i): the two ordered prefixes of {i, j}, each
                // rho(f -> l) v({i,j}, l), close with the same rows W_ab (distributivity)
                const PEntry<T> pij = get_p(col, PP + j * (j - 1) / 2 + i);
                Spinor<T> psi[2][2];   // [h_i][h_j]
                {
                    Spinor<T> v2i[2], v2j[2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        v2i[h] = chain_vector(pij, e[i][h]);
                        v2j[h] = chain_vector(pij, e[j][h]);
                    }
#pragma unroll
                    for (int hi = 0; hi < 2; ++hi) {
                        const Spinor<T> v1i = get(col, V1 + 2 * i + hi);
#pragma unroll
                        for (int hj = 0; hj < 2; ++hj) {
                            Cx<T> r;
                            chain_rho(v1i, e[j][hj], r.r, r.i);
                            psi[hi][hj].r0 = fma(r.r, v2j[hj].r0, -(r.i * v2j[hj].i0));
                            psi[hi][hj].i0 = fma(r.r, v2j[hj].i0, r.i * v2j[hj].r0);
                            psi[hi][hj].r1 = fma(r.r, v2j[hj].r1, -(r.i * v2j[hj].i1));
                            psi[hi][hj].i1 = fma(r.r, v2j[hj].i1, r.i * v2j[hj].r1);
                        }
                    }
#pragma unroll
                    for (int hj = 0; hj < 2; ++hj) {
                        const Spinor<T> v1j = get(col, V1 + 2 * j + hj);
#pragma unroll
                        for (int hi = 0; hi < 2; ++hi) {
                            Cx<T> r;
                            chain_rho(v1j, e[i][hi], r.r, r.i);
                            psi[hi][hj].r0 = fma(r.r, v2i[hi].r0, fma(-r.i, v2i[hi].i0, psi[hi][hj].r0));
                            psi[hi][hj].i0 = fma(r.r, v2i[hi].i0, fma(r.i, v2i[hi].r0, psi[hi][hj].i0));
                            psi[hi][hj].r1 = fma(r.r, v2i[hi].r1, fma(-r.i, v2i[hi].i1, psi[hi][hj].r1));
                            psi[hi][hj].i1 = fma(r.r, v2i[hi].i1, fma(r.i, v2i[hi].r1, psi[hi][hj].i1));
                        }
                    }
                }
#pragma unroll
                for (int ha = 0; ha < 2; ++ha) {
                    const Spinor<T> ua = get(col, UU + 2 * a + ha);
#pragma unroll
                    for (int hb = 0; hb < 2; ++hb) {
                        const Spinor<T> w = pair_row(ua, get(col, UU + 2 * b + hb), e[a][ha], e[b][hb]);
#pragma unroll
                        for (int hi = 0; hi < 2; ++hi)
#pragma unroll
                            for (int hj = 0; hj < 2; ++hj) {
                                const int h = (hi << i) | (hj << j) | (ha << a) | (hb << b);
                                const Cx<T> kk = row_dot(w, psi[hi][hj]);
                                amp[h].r += kk.r;
                                amp[h].i += kk.i;
                            }
                    }
                }
            }
    }

    // a8
    double m2 = 0.0;
#pragma unroll
    for (int h = 0; h < L; ++h) m2 += (double)amp[h].r * (double)amp[h].r + (double)amp[h].i * (double)amp[h].i;
    if (live) out[ev] = norm * m2;
}

// ---- n = 5: one thread per event with the 32 accumulators in the thread's shared-memory column --------------
//
// Same mathematics; the unit of work is an unordered triple T3 = {i,j,k} of photons with the pair {a,b} left
// over: Psi_T3(h_i,h_j,h_k) = sum over the 6 ordered prefixes (p,q,r) of T3 of rho(p->q) rho(q->r) v(T3, r, h_r)
// (each ordered prefix one node, evaluated once per helicity assignment of ITS photons), closed by the pair rows:
// ampsum(h) += W_ab(h_a,h_b) . Psi_T3(h_i,h_j,h_k).  2^5 complex accumulators do not fit the register file
// beside Psi, so they live in the column and are read-modified-written once per triple.
#ifndef HEGET_THREAD5_CTA
#define HEGET_THREAD5_CTA 32
#endif
#ifndef HEGET_THREAD5_MINB64
#define HEGET_THREAD5_MINB64 4
#endif
#ifndef HEGET_THREAD5_MINB32
#define HEGET_THREAD5_MINB32 8
#endif
#ifndef HEGET_THREAD5_LEAN
#define HEGET_THREAD5_LEAN 1   // fp64: the column holds P_{i} and P_{all\i} (5 + 5 entries) and the vectors v({i}, i, h) and
                               // rows U_i(h) are recomputed where used (6 FMAs each): 1 632 instead of 1 952 B per thread,
                               // i.e. 4 instead of 3 CTAs per SM: measured 1.60 -> 1.21 ms.  fp32 is not limited by shared
                               // memory (0.613 -> 0.627 ms) and keeps the 10 + 10 vectors and rows themselves
#endif
// layout of the thread's column: spinor-sized slots (two Cx words each), then the 32 accumulators
template <typename T>
struct Col5 {
    static constexpr bool LEAN = (HEGET_THREAD5_LEAN != 0) && (sizeof(T) == 8);
    static constexpr int V1 = 0, U = LEAN ? 5 : 10, P2 = LEAN ? 10 : 20, P3 = P2 + 10, E = P3 + 10, AMP = 2 * (E + 5);
    static constexpr int WORDS = AMP + 32;   // Cx words per thread
};

// v({i}, i, h) and U_i(h): read from the column, or rebuilt from the P entry kept there
template <int CTA, typename T>
__device__ __forceinline__ Spinor<T> v1_5(const Cx<T>* col, int i, int h, const EEntry<T>& e)
{
    if constexpr (Col5<T>::LEAN) {
        const Cx<T> a = col[(2 * (Col5<T>::V1 + i)) * CTA], b = col[(2 * (Col5<T>::V1 + i) + 1) * CTA];
        return chain_vector(PEntry<T>{a.r, a.i, b.r, b.i}, e);
    } else {
        const Cx<T> a = col[(2 * (Col5<T>::V1 + 2 * i + h)) * CTA], b = col[(2 * (Col5<T>::V1 + 2 * i + h) + 1) * CTA];
        return {a.r, a.i, b.r, b.i};
    }
}
template <int CTA, typename T>
__device__ __forceinline__ Spinor<T> u_5(const Cx<T>* col, int i, int h, const EEntry<T>& e)
{
    if constexpr (Col5<T>::LEAN) {
        const Cx<T> a = col[(2 * (Col5<T>::U + i)) * CTA], b = col[(2 * (Col5<T>::U + i) + 1) * CTA];
        return closing_entry(e, PEntry<T>{a.r, a.i, b.r, b.i});
    } else {
        const Cx<T> a = col[(2 * (Col5<T>::U + 2 * i + h)) * CTA], b = col[(2 * (Col5<T>::U + 2 * i + h) + 1) * CTA];
        return {a.r, a.i, b.r, b.i};
    }
}

// the 10 units of work: triple {i < j < k} in colex order and the pair {a < b} left over
struct Triple5 { unsigned char i, j, k, a, b; };
__constant__ Triple5 c_triples5[10] = {{0, 1, 2, 3, 4}, {0, 1, 3, 2, 4}, {0, 2, 3, 1, 4}, {1, 2, 3, 0, 4}, {0, 1, 4, 2, 3},
                                       {0, 2, 4, 1, 3}, {1, 2, 4, 0, 3}, {0, 3, 4, 1, 2}, {1, 3, 4, 0, 2}, {2, 3, 4, 0, 1}};

// E' entry of photon `ph` and helicity h (compile-time) from the lambda = +1 entry kept in the column:
// lambda = -1 is a' = -conj(b), b' = -conj(a) (amp2_tables.cuh)
template <int CTA, int H, typename T>
__device__ __forceinline__ EEntry<T> e5(const Cx<T>* col, int ph)
{
    const Cx<T> a = col[(2 * (Col5<T>::E + ph)) * CTA], b = col[(2 * (Col5<T>::E + ph) + 1) * CTA];
    if constexpr (H == 1) return {a.r, a.i, b.r, b.i};
    return {-b.r, b.i, -a.r, a.i};
}

template <int CTA, typename T>
__device__ __forceinline__ void put5(Cx<T>* col, int w, T a, T b, T c, T d)
{
    col[(2 * w) * CTA] = {a, b};
    col[(2 * w + 1) * CTA] = {c, d};
}
template <int CTA, typename T>
__device__ __forceinline__ Spinor<T> get5(const Cx<T>* col, int w)
{
    const Cx<T> a = col[(2 * w) * CTA], b = col[(2 * w + 1) * CTA];
    return {a.r, a.i, b.r, b.i};
}
template <int CTA, typename T>
__device__ __forceinline__ PEntry<T> get5p(const Cx<T>* col, int w)
{
    const Cx<T> a = col[(2 * w) * CTA], b = col[(2 * w + 1) * CTA];
    return {a.r, a.i, b.r, b.i};
}

template <typename T>
__global__ void __launch_bounds__(HEGET_THREAD5_CTA, (sizeof(T) == 8) ? HEGET_THREAD5_MINB64 : HEGET_THREAD5_MINB32)
amp2_thread5_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    constexpr int N = 5, CTA = HEGET_THREAD5_CTA;
    constexpr unsigned ALL = 31u;
    extern __shared__ __align__(16) unsigned char s_dyn5[];
    Cx<T>* col = reinterpret_cast<Cx<T>*>(s_dyn5) + threadIdx.x;

    int64_t ev = (int64_t)blockIdx.x * CTA + threadIdx.x;
    const bool live = ev < n_events;
    if (!live) ev = n_events - 1;

    double e1, e2, k[N][4];
    {
        const double2* src = reinterpret_cast<const double2*>(momenta) + ev * (2 * (N + 2));
        e1 = __ldg(src).x;
        e2 = __ldg(src + 2).x;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const double2 a = __ldg(src + 4 + 2 * i), b = __ldg(src + 5 + 2 * i);
            k[i][0] = a.x; k[i][1] = a.y; k[i][2] = b.x; k[i][3] = b.y;
        }
    }
    const double shat = 4.0 * e1 * e2;
    const double scale = (sizeof(T) == 4) ? sqrt(shat) : 1.0;

    EEntry<T> e[N][2];
    double norm = 2.0 * g * g * shat;
#pragma unroll
    for (int i = 0; i < N; ++i) norm *= 0.5 * make_photon_entries<T>(k[i], &e[i][1], &e[i][0]);
    if constexpr (sizeof(T) == 4) {
        const double inv = 1.0 / shat;
#pragma unroll
        for (int i = 0; i < N - 1; ++i) norm *= inv;
    }

    {   // tables: v1[2 i + h], U[2 b + h], P_ij at j (j-1)/2 + i, P_ijk at the colex rank of the triple
        Kinematics<N, sizeof(T) == 8> kin;
        kin.init(k, e1, g, scale);
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const PEntry<T> p1 = kin.template subset<T>(1u << i);
            const PEntry<T> p4 = kin.template subset<T>(ALL ^ (1u << i));
            if constexpr (Col5<T>::LEAN) {
                put5<CTA>(col, Col5<T>::V1 + i, p1.pp, p1.pm, p1.px, p1.py);
                put5<CTA>(col, Col5<T>::U + i, p4.pp, p4.pm, p4.px, p4.py);
            } else {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const Spinor<T> v = chain_vector(p1, e[i][h]), u = closing_entry(e[i][h], p4);
                    put5<CTA>(col, Col5<T>::V1 + 2 * i + h, v.r0, v.i0, v.r1, v.i1);
                    put5<CTA>(col, Col5<T>::U + 2 * i + h, u.r0, u.i0, u.r1, u.i1);
                }
            }
        }
#pragma unroll
        for (int j = 1; j < N; ++j)
#pragma unroll
            for (int i = 0; i < j; ++i) {
                const PEntry<T> p = kin.template subset<T>((1u << i) | (1u << j));
                put5<CTA>(col, Col5<T>::P2 + j * (j - 1) / 2 + i, p.pp, p.pm, p.px, p.py);
            }
#pragma unroll
        for (int kk = 2; kk < N; ++kk)
#pragma unroll
            for (int j = 1; j < kk; ++j)
#pragma unroll
                for (int i = 0; i < j; ++i) {
                    const PEntry<T> p = kin.template subset<T>((1u << i) | (1u << j) | (1u << kk));
                    put5<CTA>(col, Col5<T>::P3 + kk * (kk - 1) * (kk - 2) / 6 + j * (j - 1) / 2 + i, p.pp, p.pm, p.px, p.py);
                }
#pragma unroll
        for (int i = 0; i < N; ++i) put5<CTA>(col, Col5<T>::E + i, e[i][1].ar, e[i][1].ai, e[i][1].br, e[i][1].bi);
#pragma unroll
        for (int h = 0; h < 32; ++h) col[(Col5<T>::AMP + h) * CTA] = {(T)0, (T)0};
    }
    __syncwarp();   // keeps the compiler from forwarding the column through registers (it would spill)

    // A rolled loop over the 10 triples (the photon indices are run-time values read from constant memory, the
    // E' entries come from the column): fully unrolled, the kernel was 225 KB of straight-line code and its few
    // warps per SM waited for instructions more than for anything else (ncu: no_instruction 3.4 per issue).
#pragma unroll 1
    for (int t = 0; t < 10; ++t) {
        const int t3[3] = {c_triples5[t].i, c_triples5[t].j, c_triples5[t].k};
        const int a = c_triples5[t].a, b = c_triples5[t].b;
        const PEntry<T> p3 = get5p<CTA>(col, Col5<T>::P3 + t);
        Spinor<T> psi[8];   // index 4 h_i + 2 h_j + h_k
#pragma unroll
        for (int rr = 0; rr < 3; ++rr) {
            // last photon r of the prefix; p < q the other two: orderings (p, q, r) and (q, p, r)
            const int r = t3[2 - rr], p = t3[rr == 2 ? 1 : 0], q = t3[rr == 0 ? 1 : 2];
            const int sr = rr, sp = (rr == 2) ? 1 : 2, sq = (rr == 0) ? 1 : 0;   // bit of h_r, h_p, h_q in psi's index
            const PEntry<T> p2 = get5p<CTA>(col, Col5<T>::P2 + q * (q - 1) / 2 + p);
            const EEntry<T> ep[2] = {e5<CTA, 0>(col, p), e5<CTA, 1>(col, p)}, eq[2] = {e5<CTA, 0>(col, q), e5<CTA, 1>(col, q)},
                            er[2] = {e5<CTA, 0>(col, r), e5<CTA, 1>(col, r)};
            Cx<T> A[2][2], B[2][2], C[2][2], D[2][2];   // rho(p->q)[hp][hq], rho(q->r)[hq][hr], rho(q->p)[hq][hp], rho(p->r)[hp][hr]
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const Spinor<T> v1p = v1_5<CTA>(col, p, h, ep[h]), v1q = v1_5<CTA>(col, q, h, eq[h]);
                const Spinor<T> v2q = chain_vector(p2, eq[h]), v2p = chain_vector(p2, ep[h]);   // last = q / p, helicity h
#pragma unroll
                for (int g2 = 0; g2 < 2; ++g2) {
                    chain_rho(v1p, eq[g2], A[h][g2].r, A[h][g2].i);
                    chain_rho(v1q, ep[g2], C[h][g2].r, C[h][g2].i);
                    chain_rho(v2q, er[g2], B[h][g2].r, B[h][g2].i);
                    chain_rho(v2p, er[g2], D[h][g2].r, D[h][g2].i);
                }
            }
#pragma unroll
            for (int hr = 0; hr < 2; ++hr) {
                const Spinor<T> v3 = chain_vector(p3, er[hr]);
#pragma unroll
                for (int hp = 0; hp < 2; ++hp)
#pragma unroll
                    for (int hq = 0; hq < 2; ++hq) {
                        Cx<T> z = cx_mul(A[hp][hq], B[hq][hr]);
                        chain_acc(C[hq][hp].r, C[hq][hp].i, D[hp][hr].r, D[hp][hr].i, z.r, z.i);
                        Spinor<T>& ps = psi[(hr << sr) | (hp << sp) | (hq << sq)];
                        if (rr == 0) {
                            ps.r0 = fma(z.r, v3.r0, -(z.i * v3.i0));
                            ps.i0 = fma(z.r, v3.i0, z.i * v3.r0);
                            ps.r1 = fma(z.r, v3.r1, -(z.i * v3.i1));
                            ps.i1 = fma(z.r, v3.i1, z.i * v3.r1);
                        } else {
                            chain_acc(z.r, z.i, v3.r0, v3.i0, ps.r0, ps.i0);
                            chain_acc(z.r, z.i, v3.r1, v3.i1, ps.r1, ps.i1);
                        }
                    }
            }
        }
        const EEntry<T> ea[2] = {e5<CTA, 0>(col, a), e5<CTA, 1>(col, a)}, eb[2] = {e5<CTA, 0>(col, b), e5<CTA, 1>(col, b)};
        // accumulator of assignment h sits at word h: bits of the triple's and the pair's photons, as byte offsets
        Cx<T>* amp = col + Col5<T>::AMP * CTA;
#pragma unroll
        for (int ha = 0; ha < 2; ++ha) {
            const Spinor<T> ua = u_5<CTA>(col, a, ha, ea[ha]);
#pragma unroll
            for (int hb = 0; hb < 2; ++hb) {
                const Spinor<T> w = pair_row(ua, u_5<CTA>(col, b, hb, eb[hb]), ea[ha], eb[hb]);
                const int hab = (ha << a) | (hb << b);
                // eight accumulators at a time: all loads, then all stores (the compiler must keep a load behind an
                // earlier store it cannot tell apart, which would make the 32 updates of a triple one serial chain)
                Cx<T> acc[8];
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    acc[c] = amp[((((c >> 2) & 1) << t3[0]) | (((c >> 1) & 1) << t3[1]) | ((c & 1) << t3[2]) | hab) * CTA];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const Cx<T> dot = row_dot(w, psi[c]);
                    acc[c].r += dot.r;
                    acc[c].i += dot.i;
                }
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    amp[((((c >> 2) & 1) << t3[0]) | (((c >> 1) & 1) << t3[1]) | ((c & 1) << t3[2]) | hab) * CTA] = acc[c];
            }
        }
    }
    __syncwarp();

    double m2 = 0.0;
#pragma unroll
    for (int h = 0; h < 32; ++h) {
        const Cx<T> acc = col[(Col5<T>::AMP + h) * CTA];
        m2 += (double)acc.r * (double)acc.r + (double)acc.i * (double)acc.i;
    }
    if (live) out[ev] = norm * m2;
}

template <typename T>
cudaError_t launch_thread5(const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    constexpr size_t dyn = sizeof(Cx<T>) * Col5<T>::WORDS * HEGET_THREAD5_CTA;
    const cudaError_t attr = cudaFuncSetAttribute(amp2_thread5_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    if (attr != cudaSuccess) return attr;
    const int64_t blocks = (n_events + HEGET_THREAD5_CTA - 1) / HEGET_THREAD5_CTA;
    amp2_thread5_kernel<T><<<(unsigned)blocks, HEGET_THREAD5_CTA, dyn, stream>>>(momenta, out, n_events, g);
    return cudaGetLastError();
}

template <int N, typename T>
cudaError_t launch_thread(const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    const int64_t blocks = (n_events + HEGET_THREAD_CTA - 1) / HEGET_THREAD_CTA;
    amp2_thread_kernel<N, T><<<(unsigned)blocks, HEGET_THREAD_CTA, 0, stream>>>(momenta, out, n_events, g);
    return cudaGetLastError();
}

// ---- n = 6: TWO (fp32) or FOUR (fp64) adjacent lanes per event ------------------------------------------------------------------------
//
// The unit of work is a quadruple T4 = {t0 < t1 < t2 < t3} of photons with the pair {a, b} left over:
//     Psi_T4(h) = sum over s in T4 of Y4(s; h) v(T4, s, h_s),
//     Y4(s; h)  = sum over r in T4\s of [ z(p,q,r) + z(q,p,r) ] rho_s(v(T4\s, r, h_r)),   {p,q} = T4 \ {s,r},
//     z(p,q,r)  = rho_q(v({p},p,h_p)) rho_r(v({p,q},q,h_q))      (every ordered prefix one product, as for n = 5)
// closed by the pair rows: ampsum(h) += W_ab(h_a,h_b) . Psi_T4.  An event's 2^FIX lanes take the helicities of the
// last FIX members of the quadruple (FIX = 1: t3; FIX = 2: t2 and t3): a lane holds Psi for the 2^(4-FIX)
// assignments of the others and updates the 64 / 2^FIX accumulators with its helicities of the fixed ones.
// fp64 uses FIX = 2: half the registers per lane (Psi, Y4 and the rho tables shrink) and twice the warps per SM.
// Tables (the P entry of every subset, E' of lambda = +1) and the 64 accumulators live in ONE column per event
// that all its lanes address; which lane owns which accumulators changes from one quadruple to the next, hence
// the __syncwarp() at the end of the loop body (a CTA is one warp).
#ifndef HEGET_THREAD6_CTA
#define HEGET_THREAD6_CTA 32   // threads per CTA = one warp (__syncwarp is the only synchronisation)
#endif
#ifndef HEGET_THREAD6_FIX32
#define HEGET_THREAD6_FIX32 1  // lanes per event = 2^FIX
#endif
#ifndef HEGET_THREAD6_FIX64
#define HEGET_THREAD6_FIX64 2  // fp64: measured 2^20 events: FIX = 1: 14.6 ms (255 registers, 750 B of spills, 4 warps per SM: the
                               // column is 3 200 B per event), FIX = 2: 14.4 ms (254 registers, no spills, 8 warps per SM,
                               // 1.4x the instructions: what does not depend on the fixed helicities is computed by every
                               // lane).  Splitting the quadruples between two lane groups at FIX = 1 (own accumulators
                               // each) was slower (18.7 ms), a register-lean order of the inner block no faster (15.0 ms)
#endif
#ifndef HEGET_THREAD6_MINB32
#define HEGET_THREAD6_MINB32 8
#endif
#ifndef HEGET_THREAD6_MINB64
#define HEGET_THREAD6_MINB64 8
#endif
struct Col6 {   // spinor-sized slots (two Cx words each), then the 64 accumulators
    static constexpr int E = 0, P1 = 6, P5 = 12, P2 = 18, P3 = 33, P4 = 53, AMP = 2 * 68;   // followed by the 64 accumulators
};
struct Quad6 { unsigned char t[4], a, b; };   // at pair rank b (b - 1) / 2 + a: the complement of {a < b}
__constant__ Quad6 c_quads6[15] = {{{2, 3, 4, 5}, 0, 1}, {{1, 3, 4, 5}, 0, 2}, {{0, 3, 4, 5}, 1, 2}, {{1, 2, 4, 5}, 0, 3}, {{0, 2, 4, 5}, 1, 3},
                                   {{0, 1, 4, 5}, 2, 3}, {{1, 2, 3, 5}, 0, 4}, {{0, 2, 3, 5}, 1, 4}, {{0, 1, 3, 5}, 2, 4}, {{0, 1, 2, 5}, 3, 4},
                                   {{1, 2, 3, 4}, 0, 5}, {{0, 2, 3, 4}, 1, 5}, {{0, 1, 3, 4}, 2, 5}, {{0, 1, 2, 4}, 3, 5}, {{0, 1, 2, 3}, 4, 5}};

// positions 0..3 inside a quadruple: the last FIX positions have ONE helicity per lane and no bit in the index of Psi
__host__ __device__ constexpr bool fixed6(int pos, int FIX) { return pos >= 4 - FIX; }
__host__ __device__ constexpr int hc6(int pos, int FIX) { return fixed6(pos, FIX) ? 1 : 2; }
__host__ __device__ constexpr int wt6(int pos, int FIX) { return fixed6(pos, FIX) ? 0 : (1 << (3 - FIX - pos)); }
__host__ __device__ constexpr int wt6nz(int pos, int FIX) { return fixed6(pos, FIX) ? 1 : (1 << (3 - FIX - pos)); }
__host__ __device__ constexpr int other6(int s, int k) { return k + (k >= s ? 1 : 0); }   // k-th position of T4 \ s

template <int EV, typename T>
__device__ __forceinline__ void put6(Cx<T>* col, int w, T a, T b, T c, T d)
{
    col[(2 * w) * EV] = {a, b};
    col[(2 * w + 1) * EV] = {c, d};
}
template <int EV, typename T>
__device__ __forceinline__ PEntry<T> getp6(const Cx<T>* col, int w)
{
    const Cx<T> a = col[(2 * w) * EV], b = col[(2 * w + 1) * EV];
    return {a.r, a.i, b.r, b.i};
}
// E' entry of photon ph and helicity h (run time or folded) from the lambda = +1 entry in the column
template <int EV, typename T>
__device__ __forceinline__ EEntry<T> e6(const Cx<T>* col, int ph, int h)
{
    const Cx<T> a = col[(2 * (Col6::E + ph)) * EV], b = col[(2 * (Col6::E + ph) + 1) * EV];
    return h ? EEntry<T>{a.r, a.i, b.r, b.i} : EEntry<T>{-b.r, b.i, -a.r, a.i};
}

template <typename T>
constexpr int kFix6 = (sizeof(T) == 8) ? HEGET_THREAD6_FIX64 : HEGET_THREAD6_FIX32;

template <typename T>
__global__ void __launch_bounds__(HEGET_THREAD6_CTA, (sizeof(T) == 8) ? HEGET_THREAD6_MINB64 : HEGET_THREAD6_MINB32)
amp2_thread6_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    constexpr int N = 6, FIX = kFix6<T>, LANES = 1 << FIX, EV = HEGET_THREAD6_CTA / LANES, NC = 1 << (4 - FIX);
    static_assert(HEGET_THREAD6_CTA == 32 && (FIX == 1 || FIX == 2), "a CTA is one warp: __syncwarp() is the only synchronisation");
    constexpr unsigned ALL = 63u;
    extern __shared__ __align__(16) unsigned char s_dyn6[];
    Cx<T>* col = reinterpret_cast<Cx<T>*>(s_dyn6) + (threadIdx.x / LANES);
    const int lane = threadIdx.x % LANES;   // bit 0: this lane's helicity of t3; bit 1 (FIX = 2): of t2
    auto fixed_h = [lane](int pos) { return (lane >> (3 - pos)) & 1; };   // helicity of a fixed position

    int64_t ev = (int64_t)blockIdx.x * EV + (threadIdx.x / LANES);
    const bool live = ev < n_events;
    if (!live) ev = n_events - 1;

    double norm;
    {   // prologue: both lanes of an event compute the tables (7 % of the kernel), each stores half of them
        double e1, e2, k[N][4];
        const double2* src = reinterpret_cast<const double2*>(momenta) + ev * (2 * (N + 2));
        e1 = __ldg(src).x;
        e2 = __ldg(src + 2).x;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const double2 a = __ldg(src + 4 + 2 * i), b = __ldg(src + 5 + 2 * i);
            k[i][0] = a.x; k[i][1] = a.y; k[i][2] = b.x; k[i][3] = b.y;
        }
        const double shat = 4.0 * e1 * e2;
        const double scale = (sizeof(T) == 4) ? sqrt(shat) : 1.0;
        norm = 2.0 * g * g * shat;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            EEntry<T> ep, em;
            norm *= 0.5 * make_photon_entries<T>(k[i], &ep, &em);
            if (lane == (i % LANES)) put6<EV>(col, Col6::E + i, ep.ar, ep.ai, ep.br, ep.bi);
        }
        if constexpr (sizeof(T) == 4) {
            const double inv = 1.0 / shat;
#pragma unroll
            for (int i = 0; i < N - 1; ++i) norm *= inv;
        }
        Kinematics<N, sizeof(T) == 8> kin;
        kin.init(k, e1, g, scale);
#pragma unroll
        for (unsigned S = 1; S < ALL; ++S) {
            const int m = __popc(S);
            // slot of subset S: singles and their complements by photon, pairs and quadruples by the rank of
            // the (complementary) pair, triples by colex rank
            int x = -1, y = -1, z = -1, cnt = 0;
            const unsigned Q = (m <= 3) ? S : (ALL ^ S);   // the set that is ranked (at most 3 members)
#pragma unroll
            for (int i = 0; i < N; ++i)
                if ((Q >> i) & 1u) { if (cnt == 0) x = i; else if (cnt == 1) y = i; else z = i; ++cnt; }
            const int slot = (m == 1) ? Col6::P1 + x : (m == 5) ? Col6::P5 + x
                           : (m == 2) ? Col6::P2 + y * (y - 1) / 2 + x : (m == 4) ? Col6::P4 + y * (y - 1) / 2 + x
                           : Col6::P3 + z * (z - 1) * (z - 2) / 6 + y * (y - 1) / 2 + x;
            const PEntry<T> pe = kin.template subset<T>(S);
            if (lane == (int)(S % LANES)) put6<EV>(col, slot, pe.pp, pe.pm, pe.px, pe.py);
        }
#pragma unroll
        for (int h = 0; h < 64 / LANES; ++h) col[(Col6::AMP + LANES * h + lane) * EV] = {(T)0, (T)0};
    }
    __syncwarp();

#pragma unroll 1
    for (int t = 0; t < 15; ++t) {
        const int ph[4] = {c_quads6[t].t[0], c_quads6[t].t[1], c_quads6[t].t[2], c_quads6[t].t[3]};
        const int a = c_quads6[t].a, b = c_quads6[t].b;
        const PEntry<T> p4 = getp6<EV>(col, Col6::P4 + t);
        Spinor<T> psi[NC];   // index: the helicities of the free positions, t0 most significant
#pragma unroll
        for (int sp = 0; sp < 4; ++sp) {   // s = last photon of the prefix, at position sp of the quadruple
            const int x = ph[other6(sp, 0)], y = ph[other6(sp, 1)], z = ph[other6(sp, 2)];   // T4 \ s, increasing
            const PEntry<T> p3 = getp6<EV>(col, Col6::P3 + z * (z - 1) * (z - 2) / 6 + y * (y - 1) / 2 + x);
            const EEntry<T> es[2] = {e6<EV>(col, ph[sp], fixed6(sp, FIX) ? fixed_h(sp) : 0), e6<EV>(col, ph[sp], 1)};
            Cx<T> y4[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) y4[c] = {(T)0, (T)0};
#pragma unroll
            for (int rk = 0; rk < 3; ++rk) {   // r = third photon; p < q the first two, in both orders
                const int rp = other6(sp, rk), pp = other6(sp, rk == 0 ? 1 : 0), qp = other6(sp, rk == 2 ? 1 : 2);
                const int r = ph[rp], p = ph[pp], q = ph[qp];
                const EEntry<T> er[2] = {e6<EV>(col, r, fixed6(rp, FIX) ? fixed_h(rp) : 0), e6<EV>(col, r, 1)};
                const EEntry<T> ep[2] = {e6<EV>(col, p, fixed6(pp, FIX) ? fixed_h(pp) : 0), e6<EV>(col, p, 1)};
                const EEntry<T> eq[2] = {e6<EV>(col, q, fixed6(qp, FIX) ? fixed_h(qp) : 0), e6<EV>(col, q, 1)};
                const PEntry<T> p2 = getp6<EV>(col, Col6::P2 + q * (q - 1) / 2 + p);
                const PEntry<T> p1p = getp6<EV>(col, Col6::P1 + p), p1q = getp6<EV>(col, Col6::P1 + q);
                Cx<T> A[2][2], B[2][2], C[2][2], D[2][2], R3[2][2];
                // A = rho(p->q)[hp][hq], C = rho(q->p)[hq][hp], B = rho(q->r)[hq][hr], D = rho(p->r)[hp][hr], R3 = rho(r->s)[hr][hs]
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    if (h < hc6(pp, FIX)) {
                        const Spinor<T> v1p = chain_vector(p1p, ep[h]), v2p = chain_vector(p2, ep[h]);
#pragma unroll
                        for (int g2 = 0; g2 < 2; ++g2) {
                            if (g2 < hc6(qp, FIX)) chain_rho(v1p, eq[g2], A[h][g2].r, A[h][g2].i);
                            if (g2 < hc6(rp, FIX)) chain_rho(v2p, er[g2], D[h][g2].r, D[h][g2].i);
                        }
                    }
                    if (h < hc6(qp, FIX)) {
                        const Spinor<T> v1q = chain_vector(p1q, eq[h]), v2q = chain_vector(p2, eq[h]);
#pragma unroll
                        for (int g2 = 0; g2 < 2; ++g2) {
                            if (g2 < hc6(pp, FIX)) chain_rho(v1q, ep[g2], C[h][g2].r, C[h][g2].i);
                            if (g2 < hc6(rp, FIX)) chain_rho(v2q, er[g2], B[h][g2].r, B[h][g2].i);
                        }
                    }
                    if (h < hc6(rp, FIX)) {
                        const Spinor<T> v3 = chain_vector(p3, er[h]);
#pragma unroll
                        for (int g2 = 0; g2 < 2; ++g2)
                            if (g2 < hc6(sp, FIX)) chain_rho(v3, es[g2], R3[h][g2].r, R3[h][g2].i);
                    }
                }
#pragma unroll
                for (int hp = 0; hp < hc6(pp, FIX); ++hp)
#pragma unroll
                    for (int hq = 0; hq < hc6(qp, FIX); ++hq)
#pragma unroll
                        for (int hr = 0; hr < hc6(rp, FIX); ++hr) {
                            Cx<T> zz = cx_mul(A[hp][hq], B[hq][hr]);                                         // (p, q, r)
                            chain_acc(C[hq][hp].r, C[hq][hp].i, D[hp][hr].r, D[hp][hr].i, zz.r, zz.i);      // (q, p, r)
#pragma unroll
                            for (int hs = 0; hs < hc6(sp, FIX); ++hs) {
                                Cx<T>& yy = y4[hp * wt6(pp, FIX) + hq * wt6(qp, FIX) + hr * wt6(rp, FIX) + hs * wt6(sp, FIX)];
                                chain_acc(zz.r, zz.i, R3[hr][hs].r, R3[hr][hs].i, yy.r, yy.i);              // (.., r, s)
                            }
                        }
            }
#pragma unroll
            for (int hs = 0; hs < hc6(sp, FIX); ++hs) {
                const Spinor<T> v4 = chain_vector(p4, es[hs]);
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    if (!fixed6(sp, FIX) && ((c / wt6nz(sp, FIX)) & 1) != hs) continue;   // c carries h_s unless s is fixed
                    if (sp == 0) {
                        psi[c].r0 = fma(y4[c].r, v4.r0, -(y4[c].i * v4.i0));
                        psi[c].i0 = fma(y4[c].r, v4.i0, y4[c].i * v4.r0);
                        psi[c].r1 = fma(y4[c].r, v4.r1, -(y4[c].i * v4.i1));
                        psi[c].i1 = fma(y4[c].r, v4.i1, y4[c].i * v4.r1);
                    } else {
                        chain_acc(y4[c].r, y4[c].i, v4.r0, v4.i0, psi[c].r0, psi[c].i0);
                        chain_acc(y4[c].r, y4[c].i, v4.r1, v4.i1, psi[c].r1, psi[c].i1);
                    }
                }
            }
        }
        // close with the pair rows W_ab(h_a, h_b); this lane owns the accumulators with its helicities of the fixed positions
        const EEntry<T> ea[2] = {e6<EV>(col, a, 0), e6<EV>(col, a, 1)}, eb[2] = {e6<EV>(col, b, 0), e6<EV>(col, b, 1)};
        const PEntry<T> p5a = getp6<EV>(col, Col6::P5 + a), p5b = getp6<EV>(col, Col6::P5 + b);
        Cx<T>* amp = col + Col6::AMP * EV;
        int hfix = 0;
#pragma unroll
        for (int pos = 4 - FIX; pos < 4; ++pos) hfix |= fixed_h(pos) << ph[pos];
        int hfree[NC];   // accumulator bits of the free positions for every index of Psi
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            hfree[c] = 0;
#pragma unroll
            for (int pos = 0; pos < 4 - FIX; ++pos) hfree[c] |= ((c / wt6nz(pos, FIX)) & 1) << ph[pos];
        }
#pragma unroll
        for (int ha = 0; ha < 2; ++ha) {
            const Spinor<T> ua = closing_entry(ea[ha], p5a);
#pragma unroll
            for (int hb = 0; hb < 2; ++hb) {
                const Spinor<T> w = pair_row(ua, closing_entry(eb[hb], p5b), ea[ha], eb[hb]);
                const int hab = (ha << a) | (hb << b) | hfix;
                Cx<T> acc[NC];   // all loads, then all stores (see amp2_thread5_kernel)
#pragma unroll
                for (int c = 0; c < NC; ++c) acc[c] = amp[(hfree[c] | hab) * EV];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const Cx<T> dot = row_dot(w, psi[c]);
                    acc[c].r += dot.r;
                    acc[c].i += dot.i;
                }
#pragma unroll
                for (int c = 0; c < NC; ++c) amp[(hfree[c] | hab) * EV] = acc[c];
            }
        }
        __syncwarp();   // the next quadruple splits the accumulators between the lanes differently
    }

    double m2 = 0.0;
#pragma unroll
    for (int h = lane; h < 64; h += LANES) {
        const Cx<T> acc = col[(Col6::AMP + h) * EV];
        m2 += (double)acc.r * (double)acc.r + (double)acc.i * (double)acc.i;
    }
#pragma unroll
    for (int off = 1; off < LANES; off <<= 1) m2 += __shfl_xor_sync(0xffffffffu, m2, off);
    if (live && lane == 0) out[ev] = norm * m2;
}

template <typename T>
cudaError_t launch_thread6(const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    constexpr int EV = HEGET_THREAD6_CTA >> kFix6<T>;
    constexpr size_t dyn = sizeof(Cx<T>) * (Col6::AMP + 64) * EV;
    const cudaError_t attr = cudaFuncSetAttribute(amp2_thread6_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    if (attr != cudaSuccess) return attr;
    const int64_t blocks = (n_events + EV - 1) / EV;
    amp2_thread6_kernel<T><<<(unsigned)blocks, HEGET_THREAD6_CTA, dyn, stream>>>(momenta, out, n_events, g);
    return cudaGetLastError();
}

}  // namespace

cudaError_t heget_launch_amp2_thread(const heget_ctx* ctx, const double* momenta, int n, int precision,
                                     double* out_amp2, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    const bool f32 = precision == HEGET_FP32;
    switch (n) {
        case 2: return f32 ? launch_thread<2, float>(momenta, out_amp2, N, ctx->g, stream)
                           : launch_thread<2, double>(momenta, out_amp2, N, ctx->g, stream);
        case 3: return f32 ? launch_thread<3, float>(momenta, out_amp2, N, ctx->g, stream)
                           : launch_thread<3, double>(momenta, out_amp2, N, ctx->g, stream);
        case 4: return f32 ? launch_thread<4, float>(momenta, out_amp2, N, ctx->g, stream)
                           : launch_thread<4, double>(momenta, out_amp2, N, ctx->g, stream);
        case 5: return f32 ? launch_thread5<float>(momenta, out_amp2, N, ctx->g, stream)
                           : launch_thread5<double>(momenta, out_amp2, N, ctx->g, stream);
        case 6: return f32 ? launch_thread6<float>(momenta, out_amp2, N, ctx->g, stream)
                           : launch_thread6<double>(momenta, out_amp2, N, ctx->g, stream);
        default: return cudaErrorInvalidValue;
    }
}

// amp2_common.cuh -- what the amplitude kernels (amp2.cu: permutation tree; amp2_subset.cu:
// subset recursion) share: thread geometry, the per-event prologue that fills the E' and P
// tables in shared memory, and the epilogue that squares, sums over helicities and stores
// (product code).
#pragma once
#include "amp2_tables.cuh"
#include "heget_internal.cuh"

#ifndef HEGET_CTA_THREADS
#define HEGET_CTA_THREADS 256   // default CTA size (at least one event's 2^N lanes)
#endif
#ifndef HEGET_UNIFORM_TABLES
#define HEGET_UNIFORM_TABLES 1
#endif

template <typename T>
struct alignas(16) Spinor {
    T r0, i0, r1, i1;  // two complex components
};

// One lane per photon-helicity configuration: 2^N lanes per event, CTAs of CTA threads (or one
// event's lanes if that is more).
template <int N, int CTA = HEGET_CTA_THREADS>
struct Geometry {
    static constexpr int L = 1 << N;                       // lanes (helicity configurations) per event
    static constexpr int THREADS = (L > CTA) ? L : CTA;
    static constexpr int EPB = THREADS / L;                // events per CTA
};

// a1: the CTA's momenta as double2 words, PF words per thread: global -> registers
// (events past the end re-read the last event) and registers -> shared memory.  Split in two
// so that a persistent CTA can have the next batch's loads in flight while it computes.
template <int N, typename G = Geometry<N>>
struct MomentaTile {
    static constexpr int MOM = 4 * (N + 2);
    static constexpr int WORDS = G::EPB * MOM / 2;
    static constexpr int PF = (WORDS + G::THREADS - 1) / G::THREADS;

    static __device__ __forceinline__ void load(const double* __restrict__ momenta, int64_t ev0, int64_t n_events,
                                                double2 (&r)[PF])
    {
        const double2* src = reinterpret_cast<const double2*>(momenta);
#pragma unroll
        for (int k = 0; k < PF; ++k) {
            const int idx = threadIdx.x + k * G::THREADS;
            if (idx < WORDS) {
                int64_t e = ev0 + idx / (MOM / 2);
                if (e >= n_events) e = n_events - 1;
                r[k] = src[e * (MOM / 2) + idx % (MOM / 2)];
            }
        }
    }
    static __device__ __forceinline__ void store(double* s_mom, const double2 (&r)[PF])
    {
        double2* dst = reinterpret_cast<double2*>(s_mom);
#pragma unroll
        for (int k = 0; k < PF; ++k) {
            const int idx = threadIdx.x + k * G::THREADS;
            if (idx < WORDS) dst[idx] = r[k];
        }
    }
};

// a4: vxxxx0 for both helicities of photon `hel` (lanes 0..N-1 of each event);
// a5: subset kinematics, one subset per lane.  Reads s_mom (barrier before), ends with a barrier.
template <int N, typename T, typename G = Geometry<N>>
__device__ __forceinline__ void build_tables(double g, const double* s_mom, PEntry<T>* s_P, EEntry<T>* s_E,
                                             double* s_s2)
{
    constexpr int MOM = 4 * (N + 2);
    const int ev_local = threadIdx.x / G::L;
    const unsigned hel = threadIdx.x % G::L;
    const double* mom = s_mom + ev_local * MOM;
    const double shat = 4.0 * mom[0] * mom[4];  // (p1+p2)^2 for p1 || +z, p2 || -z
    const double scale = (sizeof(T) == 4) ? sqrt(shat) : 1.0;
    if constexpr (HEGET_UNIFORM_TABLES != 0 && N >= 4) {  // measured: 4 gamma fp64 -2.5 %, 3 gamma +12 %
        // branch-free form: every lane evaluates a photon (its own, or the last one) and a subset
        // (its own, or the nearest proper one) in ONE instruction stream -- no reconvergence points,
        // and the two independent dependency chains interleave; only the stores are predicated
        const unsigned ph = hel < (unsigned)N ? hel : (unsigned)(N - 1);
        const unsigned S = hel < 1u ? 1u : (hel > (unsigned)(G::L - 2) ? (unsigned)(G::L - 2) : hel);
        EEntry<T> ep, em;
        PEntry<T> pe;
        const double s2 = make_photon_entries<T>(mom + 4 * (2 + ph), &ep, &em);
        if constexpr (sizeof(T) == 4)
            make_subset_entry_plain<N>(mom, S, g, scale, &pe);
        else
            make_subset_entry<N, T>(mom, S, g, scale, &pe);
        if (hel < (unsigned)N) {
            s_s2[ev_local * N + hel] = s2;
            s_E[(ev_local * N + hel) * 2 + 1] = ep;
            s_E[(ev_local * N + hel) * 2 + 0] = em;
        }
        if (S == hel) s_P[ev_local * G::L + hel] = pe;
    } else {
        if (hel < (unsigned)N)
            s_s2[ev_local * N + hel] = make_photon_entries<T>(mom + 4 * (2 + hel), &s_E[(ev_local * N + hel) * 2 + 1],
                                                              &s_E[(ev_local * N + hel) * 2 + 0]);
        if (hel >= 1u && hel <= (unsigned)(G::L - 2)) {
            if constexpr (sizeof(T) == 4)
                make_subset_entry_plain<N>(mom, hel, g, scale, &s_P[ev_local * G::L + hel]);
            else
                make_subset_entry<N, T>(mom, hel, g, scale, &s_P[ev_local * G::L + hel]);
        }
    }
    __syncthreads();
}

// Closing row U_b(h) = <vbar| E'_b(h) P_{all \ b} = (a pp + q, a qbar + pm), one row vector per photon
// and helicity (amp2_tree.cuh, close_weyl).
template <typename T>
__device__ __forceinline__ Spinor<T> closing_entry(const EEntry<T>& e, const PEntry<T>& p)
{
    Spinor<T> u;  // (a, 1) . [[pp, px - i py], [px + i py, pm]]
    u.r0 = fma(e.ar, p.pp, p.px);
    u.i0 = fma(e.ai, p.pp, p.py);
    u.r1 = fma(e.ar, p.px, fma(e.ai, p.py, p.pm));
    u.i1 = fma(e.ai, p.px, -(e.ar * p.py));
    return u;
}

// Pair closing table: the two orderings that share a prefix of n-2 photons end with (a, b) or
// (b, a), and both close on the same spinor psi of that prefix:
//   <vbar|E'_b P_{all\b} E'_a psi + <vbar|E'_a P_{all\a} E'_b psi = (U_b E'_a + U_a E'_b) . psi = W_ab . psi,
// one row vector per unordered pair a < b and per helicity of a and b,
//   W[4 (b(b-1)/2 + a) + 2 h_a + h_b],   (u0, u1) E' = (-u0 + a u1, -b u0 + u1).
template <typename T>
__device__ __forceinline__ void accumulate_row_times_vertex(const Spinor<T>& u, const EEntry<T>& e, Spinor<T>& r)
{
    r.r0 += fma(e.ar, u.r1, fma(-e.ai, u.i1, -u.r0));
    r.i0 += fma(e.ar, u.i1, fma(e.ai, u.r1, -u.i0));
    r.r1 += fma(-e.br, u.r0, fma(e.bi, u.i0, u.r1));
    r.i1 += fma(-e.br, u.i0, fma(-e.bi, u.r0, u.i1));
}

// Built straight from the P and E tables (the closing rows U_a, U_b of an item are evaluated in place).
// Reads s_P and s_E (barrier before); ends with a barrier unless SYNC = false.
template <int N, typename T, typename G = Geometry<N>, bool SYNC = true>
__device__ __forceinline__ void build_pair_table_direct(const PEntry<T>* s_P, const EEntry<T>* s_E, Spinor<T>* s_W)
{
    constexpr unsigned ITEMS = 4u * (N * (N - 1) / 2);
    const int ev_local = threadIdx.x / G::L;
    const unsigned lane = threadIdx.x % G::L;
    const PEntry<T>* P = s_P + ev_local * G::L;
    const EEntry<T>* E = s_E + ev_local * 2 * N;
    for (unsigned q = lane; q < ITEMS; q += G::L) {
        const unsigned pair = q >> 2, ha = (q >> 1) & 1u, hb = q & 1u;
        unsigned b = 1;
        while ((b + 1) * b / 2 <= pair) ++b;
        const unsigned a = pair - b * (b - 1) / 2;
        const EEntry<T> ea = E[2 * a + ha], eb = E[2 * b + hb];
        Spinor<T> w = {(T)0, (T)0, (T)0, (T)0};
        accumulate_row_times_vertex(closing_entry(eb, P[(G::L - 1) ^ (1u << b)]), ea, w);
        accumulate_row_times_vertex(closing_entry(ea, P[(G::L - 1) ^ (1u << a)]), eb, w);
        s_W[ev_local * ITEMS + q] = w;
    }
    if constexpr (SYNC) __syncthreads();
}

// a1 + a4 + a5 for the batch of events starting at ev0 (one-shot form).
template <int N, typename T, typename G = Geometry<N>>
__device__ __forceinline__ void build_event_tables(const double* __restrict__ momenta, int64_t ev0, int64_t n_events,
                                                   double g, double* s_mom, PEntry<T>* s_P, EEntry<T>* s_E,
                                                   double* s_s2)
{
    double2 r[MomentaTile<N, G>::PF];
    MomentaTile<N, G>::load(momenta, ev0, n_events, r);
    MomentaTile<N, G>::store(s_mom, r);
    __syncthreads();
    build_tables<N, T, G>(g, s_mom, s_P, s_E, s_s2);
}

// a8: |ampsum|^2 summed over the event's 2^N lanes (warp shuffles, one shared-memory pass for
// N > 5), times the constant factors, one store per event.
template <int N, typename T, typename G = Geometry<N>>
__device__ __forceinline__ void finish_event(T ar, T ai, const double* s_mom, const double* s_s2, double* s_red,
                                             double g, double* __restrict__ out, int64_t ev0, int64_t n_events)
{
    constexpr int MOM = 4 * (N + 2);
    const int tid = threadIdx.x;
    const int ev_local = tid / G::L;
    const unsigned hel = tid % G::L;
    double m2 = (double)ar * (double)ar + (double)ai * (double)ai;
    constexpr int WL = (G::L < 32) ? G::L : 32;
#pragma unroll
    for (int off = WL / 2; off > 0; off >>= 1) m2 += __shfl_xor_sync(0xffffffffu, m2, off);
    if constexpr (G::L > 32) {
        if ((tid & 31) == 0) s_red[tid >> 5] = m2;
        __syncthreads();
        if (hel == 0) {
            m2 = 0.0;
#pragma unroll
            for (int w = 0; w < G::L / 32; ++w) m2 += s_red[ev_local * (G::L / 32) + w];
        }
    }
    if (hel == 0 && ev0 + ev_local < n_events) {
        // constants: 2 (parity) * g^2 (closing vertex) * 2E1*2E2 = s_hat (spinor norms) * 2^-N
        // (the sqrt(2) of every polarisation vector) * prod s_i^2 (E' normalisation);
        // fp32 worked in units of sqrt(s_hat)
        const double* mom = s_mom + ev_local * MOM;
        const double shat = 4.0 * mom[0] * mom[4];
        double f = 2.0 * g * g * shat;
#pragma unroll
        for (int i = 0; i < N; ++i) f *= 0.5 * s_s2[ev_local * N + i];
        if (sizeof(T) == 4) {
            const double inv = 1.0 / shat;
#pragma unroll
            for (int i = 0; i < N - 1; ++i) f *= inv;
        }
        out[ev0 + ev_local] = f * m2;
    }
}

// amp2_twosided.cu -- HEGET_ALGO_TREE2: two-sided chaining (product code).
//
// List 2 of the paper chains the off-shell line from the ubar end with fvoxx0 (PAPER.md:449-450,
// 642-656) while eq. (7) chains it from the u end with fvixx0: the same
// n! diagrams.  Here both ends are used and meet in the middle, which is the reuse of off-shell
// lines that makes the MadGraph-generated code faster than the permutation code:
//   * from the ubar end, the row vectors
//         L_1[j]   = <vbar| E'_j                                        (closing vertex, no propagator)
//         L_m+1[T] = sum_{x in T} ( L_m[T \ x] P_{all \ (T \ x)} ) E'_x    (fvoxx0 summed over orderings)
//     are tabulated in shared memory for all sets T of up to KS = min(n, 4) photons and all
//     helicities of T (C(n,2) 4 + C(n,3) 8 + C(n,4) 16 entries; n = 8: 1 680);
//   * from the u end, the depth-first permutation tree of amp2.cu is walked only to depth n - KS
//     (each ordered prefix once), and every node at that depth closes with ONE dot product
//         ampsum += L_KS[remaining photons] . psi
//     instead of the KS! orderings below it (the propagator of that last u-side node is folded into
//     the table entry, L'[T] = L[T] P_{all \\ T}, so the node itself is only its vertex).
// Per helicity configuration: sum_{l=1}^{n-KS} n!/(n-l)! fvixx0 nodes and n!/KS! closings
// (n = 8: 2 080 + 1 680 against 69 280 + 40 320 in the one-sided tree).  Same E' / P tables,
// parity shortcut, lane mapping (one lane per helicity configuration) and epilogue as amp2.cu.
#include "amp2_tree.cuh"
#include "subset_index.cuh"

// CTA size ("CTA size"): measured on B200, 256 -> 64 threads: 4 gamma fp64 1.04 -> 0.91 ms, 6 gamma fp64 14.2 -> 12.2 ms
#ifndef HEGET_TS_CTA_THREADS
#define HEGET_TS_CTA_THREADS 64
#endif
template <int N>
using KGeometry = Geometry<N, HEGET_TS_CTA_THREADS>;

namespace {

#ifndef HEGET_KSUFFIX
#define HEGET_KSUFFIX 4
#endif
template <int N>
constexpr int kSuffix = (N < HEGET_KSUFFIX) ? N : HEGET_KSUFFIX;  // KS: photons attached from the ubar end

// row vector times the propagator block, r' = r P,  P = [[pp, px - i py], [px + i py, pm]]
template <typename T>
__device__ __forceinline__ Spinor<T> row_times_P(const Spinor<T>& r, const PEntry<T>& P)
{
    Spinor<T> o;
    o.r0 = fma(P.pp, r.r0, fma(P.px, r.r1, -(P.py * r.i1)));
    o.i0 = fma(P.pp, r.i0, fma(P.px, r.i1, P.py * r.r1));
    o.r1 = fma(P.pm, r.r1, fma(P.px, r.r0, P.py * r.i0));
    o.i1 = fma(P.pm, r.i1, fma(P.px, r.i0, -(P.py * r.r0)));
    return o;
}

// acc += r E',  E' = [[-1, -b], [a, 1]]:  (r0, r1) E' = (-r0 + a r1, -b r0 + r1)
template <typename T>
__device__ __forceinline__ void accumulate_row_times_E(const Spinor<T>& r, const EEntry<T>& E, Spinor<T>& acc)
{
    acc.r0 += fma(E.ar, r.r1, fma(-E.ai, r.i1, -r.r0));
    acc.i0 += fma(E.ar, r.i1, fma(E.ai, r.r1, -r.i0));
    acc.r1 += fma(-E.br, r.r0, fma(E.bi, r.i0, r.r1));
    acc.i1 += fma(-E.br, r.i0, fma(-E.bi, r.r0, r.i1));
}

// Level M >= 2 of the ubar-side table from level M - 1 (M = 2: from L_1[j] = (a_j, 1)).
// Entry q = rank(T) * 2^M + h, h compact: bit j of h = helicity of the j-th lowest photon of T.
// FOLD: multiply the finished row vector by the propagator of the complementary set,
// L'[T] = L[T] P_{all \ T}; used for the last level when a u-side tree remains (KS < N), whose
// last fvixx0 then reduces to its vertex (the same re-association as the closing table of amp2.cu).
template <int N, int M, typename T, bool FOLD = false>
__device__ __forceinline__ void build_suffix_level(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                                   const unsigned char* __restrict__ s_rank,
                                                   const unsigned char* __restrict__ s_list,
                                                   const Spinor<T>* __restrict__ prev, Spinor<T>* __restrict__ cur,
                                                   unsigned lane)
{
    constexpr int L = 1 << N;
    constexpr unsigned FULL = (1u << N) - 1u;
    constexpr int ITEMS = binom(N, M) << M;
    for (int q = (int)lane; q < ITEMS; q += L) {
        const unsigned h = (unsigned)q & ((1u << M) - 1u);
        const unsigned Tset = s_list[M * 72 + (q >> M)];
        Spinor<T> acc = {(T)0, (T)0, (T)0, (T)0};
        unsigned rem = Tset;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            const int x = __ffs(rem) - 1;
            rem &= rem - 1u;
            const unsigned child = Tset ^ (1u << x);
            const unsigned hc = (h & ((1u << j) - 1u)) | ((h >> (j + 1)) << j);  // h without bit j
            Spinor<T> r;
            if constexpr (M == 2) {
                const int y = __ffs(child) - 1;
                const EEntry<T> ey = E[2 * y + (hc & 1u)];
                r = {ey.ar, ey.ai, (T)1, (T)0};  // L_1[y] = <vbar| E'_y
            } else {
                r = prev[((unsigned)s_rank[child] << (M - 1)) + hc];
            }
            const Spinor<T> rp = row_times_P(r, P[FULL ^ child]);
            accumulate_row_times_E(rp, E[2 * x + ((h >> j) & 1u)], acc);
        }
        if constexpr (FOLD) acc = row_times_P(acc, P[FULL ^ Tset]);
        cur[q] = acc;
    }
}

// Unrolled levels of the u-side tree from R remaining photons down to KS, where the branch
// closes with the tabulated ubar-side row vector.  The remaining photons are compile-time-indexed
// register lists in ascending photon order: bit[] = subset-index bits, e[] = this lane's E'
// entry pointers, hb[] = this lane's helicity bits.
template <int R, int KS, typename T, bool FOLD = false>
struct Close {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ PS, const int (&bit)[R],
                                               const EEntry<T>* const (&e)[R], const unsigned (&hb)[R],
                                               const Spinor<T>& f, const Spinor<T>* __restrict__ Ltab,
                                               const unsigned char* __restrict__ s_rank, T& ar, T& ai)
    {
        if constexpr (R == KS) {
            unsigned Tset = 0u, h = 0u;
#pragma unroll
            for (int m = 0; m < R; ++m) {
                Tset |= (unsigned)bit[m];
                h |= hb[m] << m;
            }
            const Spinor<T> r = Ltab[((unsigned)s_rank[Tset] << KS) + h];
            ar += fma(r.r0, f.r0, fma(-r.i0, f.i0, fma(r.r1, f.r1, -(r.i1 * f.i1))));
            ai += fma(r.r0, f.i0, fma(r.i0, f.r0, fma(r.r1, f.i1, r.i1 * f.r1)));
        } else {
#pragma unroll
            for (int i = 0; i < R; ++i) {
                int sub_bit[R - 1];
                const EEntry<T>* sub_e[R - 1];
                unsigned sub_hb[R - 1];
#pragma unroll
                for (int m = 0; m < R - 1; ++m) {
                    sub_bit[m] = bit[m + (m >= i ? 1 : 0)];
                    sub_e[m] = e[m + (m >= i ? 1 : 0)];
                    sub_hb[m] = hb[m + (m >= i ? 1 : 0)];
                }
                if constexpr (FOLD && R == KS + 1) {
                    // last u-side photon: its propagator is already in the table entry
                    unsigned Tset = 0u, h = 0u;
#pragma unroll
                    for (int m = 0; m < R - 1; ++m) {
                        Tset |= (unsigned)sub_bit[m];
                        h |= sub_hb[m] << m;
                    }
                    close_weyl(Ltab[((unsigned)s_rank[Tset] << KS) + h], vertex_weyl(*e[i], f), ar, ai);
                } else {
                    const PEntry<T>* Pn = PS + bit[i];
                    const Spinor<T> fn = fvixx0_weyl(*Pn, *e[i], f);
                    Close<R - 1, KS, T, FOLD>::run(Pn, sub_bit, sub_e, sub_hb, fn, Ltab, s_rank, ar, ai);
                }
            }
        }
    }
};

// Looped upper levels; when RB photons remain the unrolled Close<RB, KS> takes over.
template <int N, int DEPTH, int RB, int KS, typename T, bool FOLD = false>
struct Walk2 {
    static __device__ __forceinline__ void run(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                               unsigned hel, unsigned used, const Spinor<T>& f,
                                               const Spinor<T>* __restrict__ Ltab,
                                               const unsigned char* __restrict__ s_rank, T& ar, T& ai)
    {
        unsigned avail = ((1u << N) - 1u) & ~used;
        if constexpr (N - DEPTH == RB) {
            int bit[RB];
            const EEntry<T>* e[RB];
            unsigned hb[RB];
#pragma unroll
            for (int m = 0; m < RB; ++m) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                bit[m] = 1 << i;
                hb[m] = (hel >> i) & 1u;
                e[m] = &E[2 * i + hb[m]];
            }
            Close<RB, KS, T, FOLD>::run(P + used, bit, e, hb, f, Ltab, s_rank, ar, ai);
        } else {
            while (avail) {
                const int i = __ffs(avail) - 1;
                avail &= avail - 1u;
                const unsigned S = used | (1u << i);
                const Spinor<T> fn = fvixx0_weyl(P[S], E[2 * i + ((hel >> i) & 1u)], f);
                Walk2<N, DEPTH + 1, RB, KS, T, FOLD>::run(P, E, hel, S, fn, Ltab, s_rank, ar, ai);
            }
        }
    }
};

template <int N, typename T>
struct TwoSidedSmem {
    using G = KGeometry<N>;
    static constexpr int KS = kSuffix<N>;
    static constexpr int MOM = 4 * (N + 2);
    static constexpr int L2 = binom(N, 2) << 2;                 // entries of level 2
    static constexpr int L3 = (KS >= 3) ? (binom(N, 3) << 3) : 0;  // entries of level 3
    static constexpr int L4 = (KS >= 4) ? (binom(N, 4) << 4) : 0;  // entries of level 4
    static constexpr size_t off_l2 = 0;
    static constexpr size_t off_l3 = off_l2 + sizeof(Spinor<T>) * G::EPB * L2;
    static constexpr size_t off_l4 = off_l3 + sizeof(Spinor<T>) * G::EPB * L3;
    static constexpr size_t off_P = off_l4 + sizeof(Spinor<T>) * G::EPB * L4;
    static constexpr size_t off_E = off_P + sizeof(PEntry<T>) * G::EPB * G::L;
    static constexpr size_t off_mom = off_E + sizeof(EEntry<T>) * G::EPB * 2 * N;
    static constexpr size_t off_s2 = off_mom + sizeof(double) * G::EPB * MOM;
    static constexpr size_t off_red = off_s2 + sizeof(double) * G::EPB * N;
    static constexpr size_t off_rank = off_red + sizeof(double) * (G::THREADS / 32);
    static constexpr size_t off_list = off_rank + 256;
    static constexpr size_t bytes = off_list + (N + 1) * 72;
};

#ifndef HEGET_TS_MINB32
#define HEGET_TS_MINB32 2   // 128 registers, two CTAs per SM: 6 gamma 9.8 -> 7.0 ms, 7 gamma 14.8 -> 12.5 ms
#endif
#ifndef HEGET_TS_MINB64
#define HEGET_TS_MINB64 1
#endif
template <int N, typename T>
__global__ void __launch_bounds__(KGeometry<N>::THREADS,
                                  ((sizeof(T) == 4) ? HEGET_TS_MINB32 : HEGET_TS_MINB64) * 256 / KGeometry<N>::THREADS)
amp2_twosided_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    using G = KGeometry<N>;
    using SM = TwoSidedSmem<N, T>;
    constexpr int KS = SM::KS;
    constexpr int RB = (N < KS + 2) ? N : KS + 2;  // remaining photons where unrolling starts
    extern __shared__ __align__(32) unsigned char smem[];
    Spinor<T>* s_l2 = reinterpret_cast<Spinor<T>*>(smem + SM::off_l2);
    Spinor<T>* s_l3 = reinterpret_cast<Spinor<T>*>(smem + SM::off_l3);
    Spinor<T>* s_l4 = reinterpret_cast<Spinor<T>*>(smem + SM::off_l4);
    PEntry<T>* s_P = reinterpret_cast<PEntry<T>*>(smem + SM::off_P);
    EEntry<T>* s_E = reinterpret_cast<EEntry<T>*>(smem + SM::off_E);
    double* s_mom = reinterpret_cast<double*>(smem + SM::off_mom);
    double* s_s2 = reinterpret_cast<double*>(smem + SM::off_s2);
    double* s_red = reinterpret_cast<double*>(smem + SM::off_red);
    unsigned char* s_rank = smem + SM::off_rank;
    unsigned char* s_list = smem + SM::off_list;

    const int ev_local = threadIdx.x / G::L;
    const unsigned hel = threadIdx.x % G::L;
    const int64_t ev0 = (int64_t)blockIdx.x * G::EPB;

    load_subset_index<N, G::THREADS>(s_rank, s_list);
    build_event_tables<N, T, G>(momenta, ev0, n_events, g, s_mom, s_P, s_E, s_s2);  // ends with a barrier

    const PEntry<T>* P = s_P + ev_local * G::L;
    const EEntry<T>* E = s_E + ev_local * 2 * N;
    Spinor<T>* l2 = s_l2 + ev_local * SM::L2;
    Spinor<T>* l3 = s_l3 + ev_local * SM::L3;
    Spinor<T>* l4 = s_l4 + ev_local * SM::L4;
    constexpr bool FOLD = (KS < N);  // a u-side tree remains: fold its last propagator into the table
    build_suffix_level<N, 2, T, FOLD && KS == 2>(P, E, s_rank, s_list, nullptr, l2, hel);
    __syncthreads();
    if constexpr (KS >= 3) {
        build_suffix_level<N, 3, T, FOLD && KS == 3>(P, E, s_rank, s_list, l2, l3, hel);
        __syncthreads();
    }
    if constexpr (KS >= 4) {
        build_suffix_level<N, 4, T, FOLD && KS == 4>(P, E, s_rank, s_list, l3, l4, hel);
        __syncthreads();
    }
    const Spinor<T>* Ltab = (KS >= 4) ? l4 : (KS >= 3) ? l3 : l2;

    T ar = 0, ai = 0;
    const Spinor<T> f0 = {(T)1, (T)0, (T)0, (T)0};
    Walk2<N, 0, RB, KS, T, FOLD>::run(P, E, hel, 0u, f0, Ltab, s_rank, ar, ai);
    finish_event<N, T, G>(ar, ai, s_mom, s_s2, s_red, g, out, ev0, n_events);
}

template <int N, typename T>
cudaError_t launch_one(const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    using G = KGeometry<N>;
    constexpr size_t bytes = TwoSidedSmem<N, T>::bytes;
    if (bytes > 48 * 1024) {
        cudaError_t err = cudaFuncSetAttribute(amp2_twosided_kernel<N, T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)bytes);
        if (err != cudaSuccess) return err;
    }
    const int64_t blocks = (n_events + G::EPB - 1) / G::EPB;
    amp2_twosided_kernel<N, T><<<(unsigned)blocks, G::THREADS, bytes, stream>>>(momenta, out, n_events, g);
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

cudaError_t heget_launch_amp2_twosided(const heget_ctx* ctx, const double* momenta, int n, int precision,
                                       double* out_amp2, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    if (precision == HEGET_FP32) return launch_n<float>(n, momenta, out_amp2, N, ctx->g, stream);
    return launch_n<double>(n, momenta, out_amp2, N, ctx->g, stream);
}

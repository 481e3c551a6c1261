// amp2_subset.cu -- HEGET_ALGO_SUBSET: the permutation sum of eq. (6) reorganised as
// a recursion over photon SUBSETS instead of a walk over ordered prefixes (product code).
//
// The propagator (p1 - K_l)/t_l of eqs. (7),(8) depends only on the SET of
// photons attached so far, so the sum of the fvixx0 chains over all orderings
// of a set S,
//     Psi(S) = sum_{orderings of S} prod_l [ -g (p1-K_l)-slash / t_l  eps-slash_{pi(l)} ] u(p1),
// obeys
//     Psi(S) = P_S * sum_{i in S} E'_i Psi(S \ i),      Psi({}) = u(p1),
// and the amplitude is ampsum = sum_j <vbar| E'_j Psi(all \ j) (iovxxx).
// Psi(S) depends on the helicities of the photons in S only, so level m (|S| = m) holds
// C(n,m) 2^m two-component spinors; the whole event needs 3^n - 1 of them instead of the
// 2^n * sum_l n!/(n-l)! nodes of the permutation tree (n = 8: 6.6e3 against 1.8e7).  This is the
// paper's remark that reusing off-shell lines is what makes the MadGraph code faster than the
// permutation code taken to its end; it is NOT the permutation-tree method and is
// therefore a separately named algorithm of heget_amp2_algo.  Same tables, same E'
// normalisation, same sigma_1 = +1 parity shortcut and the same epilogue as amp2.cu.
//
// Mapping: 2^N lanes per event as in amp2.cu; at level m the event's lanes stride over the
// C(N,m) 2^m items (S, helicities of S); levels are separated by CTA barriers and ping-pong
// between two shared-memory buffers.
#include "amp2_common.cuh"
#include "subset_index.cuh"

// CTA size ("CTA size"): measured on B200, 256 -> 128 threads: 4 gamma 0.449 -> 0.436 ms fp32, 5 gamma 1.50 -> 1.43 ms
#ifndef HEGET_SUBSET_CTA_THREADS
#define HEGET_SUBSET_CTA_THREADS 128
#endif
template <int N>
using KGeometry = Geometry<N, HEGET_SUBSET_CTA_THREADS>;

namespace {

template <int N>
__host__ __device__ constexpr int max_level_items()
{
    int best = 0;
    for (int m = 1; m < N; ++m) {
        const int c = binom(N, m) << m;
        if (c > best) best = c;
    }
    return best;
}

// sum_i E'_i psi_i accumulated into (a0, a1):  E' = [[-1, -b], [a, 1]]
template <typename T>
__device__ __forceinline__ void accumulate_vertex(const EEntry<T>& E, const Spinor<T>& f, Spinor<T>& acc)
{
    acc.r0 = fma(-E.br, f.r1, fma(E.bi, f.i1, acc.r0 - f.r0));
    acc.i0 = fma(-E.br, f.i1, fma(-E.bi, f.r1, acc.i0 - f.i0));
    acc.r1 = fma(E.ar, f.r0, fma(-E.ai, f.i0, acc.r1 + f.r1));
    acc.i1 = fma(E.ar, f.i0, fma(E.ai, f.r0, acc.i1 + f.i1));
}

template <typename T>
__device__ __forceinline__ Spinor<T> apply_propagator(const PEntry<T>& P, const Spinor<T>& w)
{
    Spinor<T> o;
    o.r0 = fma(P.pp, w.r0, fma(P.px, w.r1, P.py * w.i1));
    o.i0 = fma(P.pp, w.i0, fma(P.px, w.i1, -(P.py * w.r1)));
    o.r1 = fma(P.pm, w.r1, fma(P.px, w.r0, -(P.py * w.i0)));
    o.i1 = fma(P.pm, w.i1, fma(P.px, w.i0, P.py * w.r0));
    return o;
}

// Level M (1 <= M < N): Psi(S, h) for all |S| = M and all helicity assignments h of S.
// h is stored compactly: bit j of h is the helicity of the j-th lowest photon of S.
//
// When 2^M >= 32 (and an event owns whole warps, N >= 5) the 32 lanes of a warp work on 32
// helicity assignments of ONE subset S, so everything derived from S -- its members, the ranks of
// its children, the P entry -- is warp-uniform: the warp index is broadcast with a shuffle so that
// the compiler keeps that arithmetic on the uniform datapath and reads the index tables from
// constant memory; only the helicity bits stay per lane.  These levels hold most of the work
// (N = 8: levels 5-7 are 27 000 of the 33 000 vertex terms).
template <int N, int M, typename T>
__device__ __forceinline__ void run_level(const PEntry<T>* __restrict__ P, const EEntry<T>* __restrict__ E,
                                          const unsigned char* __restrict__ s_rank,
                                          const unsigned char* __restrict__ s_list, const Spinor<T>* __restrict__ prev,
                                          Spinor<T>* __restrict__ cur, unsigned lane)
{
    constexpr int L = 1 << N;
    constexpr int ITEMS = binom(N, M) << M;
    if constexpr (M >= 5 && N >= 5 && sizeof(T) == 8) {  // measured: +3..10 % in fp64, -5..+1 % in fp32
        const unsigned warp_q = __shfl_sync(0xffffffffu, lane & ~31u, 0);  // first item of this warp, uniform
        const unsigned lane_id = lane & 31u;
        for (unsigned q0 = warp_q; q0 < (unsigned)ITEMS; q0 += L) {
            const unsigned h = (q0 & ((1u << M) - 1u)) | lane_id;
            const unsigned S = c_index.list[M][q0 >> M];
            Spinor<T> acc = {(T)0, (T)0, (T)0, (T)0};
            unsigned rem = S;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                const int i = __ffs(rem) - 1;
                rem &= rem - 1u;
                const unsigned child_base = (unsigned)c_index.rank[S ^ (1u << i)] << (M - 1);
                const unsigned hc = (h & ((1u << j) - 1u)) | ((h >> (j + 1)) << j);  // h without bit j
                accumulate_vertex(E[2 * i + ((h >> j) & 1u)], prev[child_base + hc], acc);
            }
            cur[q0 + lane_id] = apply_propagator(P[S], acc);
        }
    } else {
        for (int q = (int)lane; q < ITEMS; q += L) {
            const unsigned h = (unsigned)q & ((1u << M) - 1u);
            const unsigned S = s_list[M * 72 + (q >> M)];
            Spinor<T> acc = {(T)0, (T)0, (T)0, (T)0};
            unsigned rem = S;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                const int i = __ffs(rem) - 1;
                rem &= rem - 1u;
                const EEntry<T> e = E[2 * i + ((h >> j) & 1u)];
                Spinor<T> f;
                if constexpr (M == 1) {
                    f = {(T)1, (T)0, (T)0, (T)0};  // u(p1,+) / sqrt(2 E1)
                } else {
                    const unsigned hc = (h & ((1u << j) - 1u)) | ((h >> (j + 1)) << j);  // h without bit j
                    f = prev[((unsigned)s_rank[S ^ (1u << i)] << (M - 1)) + hc];
                }
                accumulate_vertex(e, f, acc);
            }
            cur[q] = apply_propagator(P[S], acc);
        }
    }
}

template <int N, int M, typename T>
struct Levels {
    static __device__ __forceinline__ void run(const PEntry<T>* P, const EEntry<T>* E, const unsigned char* s_rank,
                                               const unsigned char* s_list, Spinor<T>* buf0, Spinor<T>* buf1,
                                               unsigned lane)
    {
        Spinor<T>* cur = (M & 1) ? buf1 : buf0;
        const Spinor<T>* prev = (M & 1) ? buf0 : buf1;
        run_level<N, M, T>(P, E, s_rank, s_list, prev, cur, lane);
        __syncthreads();
        if constexpr (M + 1 < N) Levels<N, M + 1, T>::run(P, E, s_rank, s_list, buf0, buf1, lane);
    }
};

template <int N, typename T>
struct SubsetSmem {
    using G = KGeometry<N>;
    static constexpr int MOM = 4 * (N + 2);
    static constexpr int LVL = max_level_items<N>();
    // byte offsets, every array 16-byte aligned (32 for the double spinors)
    static constexpr size_t off_psi0 = 0;
    static constexpr size_t off_psi1 = off_psi0 + sizeof(Spinor<T>) * G::EPB * LVL;
    static constexpr size_t off_P = off_psi1 + sizeof(Spinor<T>) * G::EPB * LVL;
    static constexpr size_t off_E = off_P + sizeof(PEntry<T>) * G::EPB * G::L;
    static constexpr size_t off_mom = off_E + sizeof(EEntry<T>) * G::EPB * 2 * N;
    static constexpr size_t off_s2 = off_mom + sizeof(double) * G::EPB * MOM;
    static constexpr size_t off_red = off_s2 + sizeof(double) * G::EPB * N;
    static constexpr size_t off_rank = off_red + sizeof(double) * (G::THREADS / 32);
    static constexpr size_t off_list = off_rank + 256;
    static constexpr size_t bytes = off_list + (N + 1) * 72;
};

template <int N, typename T>
__global__ void __launch_bounds__(KGeometry<N>::THREADS)
amp2_subset_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    using G = KGeometry<N>;
    using SM = SubsetSmem<N, T>;
    extern __shared__ __align__(32) unsigned char smem[];
    Spinor<T>* s_psi0 = reinterpret_cast<Spinor<T>*>(smem + SM::off_psi0);
    Spinor<T>* s_psi1 = reinterpret_cast<Spinor<T>*>(smem + SM::off_psi1);
    PEntry<T>* s_P = reinterpret_cast<PEntry<T>*>(smem + SM::off_P);
    EEntry<T>* s_E = reinterpret_cast<EEntry<T>*>(smem + SM::off_E);
    double* s_mom = reinterpret_cast<double*>(smem + SM::off_mom);
    double* s_s2 = reinterpret_cast<double*>(smem + SM::off_s2);
    double* s_red = reinterpret_cast<double*>(smem + SM::off_red);
    unsigned char* s_rank = smem + SM::off_rank;
    unsigned char* s_list = smem + SM::off_list;

    const int ev_local = threadIdx.x / G::L;
    const unsigned hel = threadIdx.x % G::L;

    load_subset_index<N, G::THREADS>(s_rank, s_list);
    build_event_tables<N, T, G>(momenta, (int64_t)blockIdx.x * G::EPB, n_events, g, s_mom, s_P, s_E, s_s2);  // ends with a barrier

    const PEntry<T>* P = s_P + ev_local * G::L;
    const EEntry<T>* E = s_E + ev_local * 2 * N;
    Spinor<T>* buf0 = s_psi0 + ev_local * SM::LVL;
    Spinor<T>* buf1 = s_psi1 + ev_local * SM::LVL;
    Levels<N, 1, T>::run(P, E, s_rank, s_list, buf0, buf1, hel);

    // closing vertex (iovxxx): ampsum(hel) = sum_j [ a_j psi0 + psi1 ](all \ j, hel without j)
    const Spinor<T>* last = ((N - 1) & 1) ? buf1 : buf0;
    T ar = 0, ai = 0;
#pragma unroll
    for (int j = 0; j < N; ++j) {
        const EEntry<T> e = E[2 * j + ((hel >> j) & 1u)];
        const unsigned hc = (hel & ((1u << j) - 1u)) | ((hel >> (j + 1)) << j);
        // the (N-1)-photon sets in increasing numeric order are "all but photon N-1", ..., "all but 0"
        const Spinor<T> f = last[((unsigned)(N - 1 - j) << (N - 1)) + hc];
        ar += fma(e.ar, f.r0, fma(-e.ai, f.i0, f.r1));
        ai += fma(e.ar, f.i0, fma(e.ai, f.r0, f.i1));
    }
    finish_event<N, T, G>(ar, ai, s_mom, s_s2, s_red, g, out, (int64_t)blockIdx.x * G::EPB, n_events);
}

template <int N, typename T>
cudaError_t launch_one(const double* momenta, double* out, int64_t n_events, double g, cudaStream_t stream)
{
    using G = KGeometry<N>;
    constexpr size_t bytes = SubsetSmem<N, T>::bytes;
    if (bytes > 48 * 1024) {  // opt in to large dynamic shared memory (per device, cheap to repeat)
        cudaError_t err = cudaFuncSetAttribute(amp2_subset_kernel<N, T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)bytes);
        if (err != cudaSuccess) return err;
    }
    const int64_t blocks = (n_events + G::EPB - 1) / G::EPB;
    amp2_subset_kernel<N, T><<<(unsigned)blocks, G::THREADS, bytes, stream>>>(momenta, out, n_events, g);
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

cudaError_t heget_launch_amp2_subset(const heget_ctx* ctx, const double* momenta, int n, int precision,
                                     double* out_amp2, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    if (precision == HEGET_FP32) return launch_n<float>(n, momenta, out_amp2, N, ctx->g, stream);
    return launch_n<double>(n, momenta, out_amp2, N, ctx->g, stream);
}

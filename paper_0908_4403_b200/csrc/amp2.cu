// amp2.cu -- heget_amp2: summed squared helicity amplitude of u ubar -> n gamma (product code).
//
// Mapping: one lane per photon-helicity configuration (2^N lanes per event), CTAs of
// max(64, 2^N) threads holding 64/2^N events (one event from n = 6 on).  All lanes of a CTA walk the SAME permutation tree in lockstep
// (no divergence); they differ only in which helicity entry of the per-photon E table they
// read.  Per event the CTA first builds, in shared memory,
//   - the E table (vxxxx0 for both helicities of every photon) and
//   - the subset table P[S] = -g/t_S * (p1 - K_S)-slash block for every photon subset S,
// then every lane runs the depth-first walk of eq. (6)'s n! orderings: each
// ordered prefix (tree node) is one fvixx0 computed once, each leaf one
// iovxxx accumulated into ampsum (List 2).  For n >= 4 the two
// orderings below a prefix of n-2 photons close through a per-event pair table (amp2_common.cuh);
// for n >= 5 the nodes are evaluated in factorised form psi = z v (amp2_chain.cuh).
// Only sigma_1 = +1, sigma_2 = -1 is evaluated: sigma_1 = sigma_2 vanishes identically and
// |M(-sigma,-lambda)| = |M(sigma,lambda)|, so the helicity sum is twice the sum over lambda.
#include "amp2_tree.cuh"
#include "amp2_chain.cuh"

#ifndef HEGET_MINB32
#define HEGET_MINB32 1      // __launch_bounds__ min CTAs per SM, fp32 / fp64 kernels
#endif
#ifndef HEGET_MINB64
#define HEGET_MINB64 1      // fp64 (n = 2, 3 and n >= 6): 1 = no register cap.  The v2-v8 tree kernels ran best at 2
                            // (128 registers, 16 warps per SM); the factorised walk with five unrolled levels
                            // (HEGET_CHAIN_KB64) needs 160-185 registers and is 13-15 % faster uncapped
#endif
#ifndef HEGET_MINW64
#define HEGET_MINW64 (HEGET_MINB64 * 8)   // fp64: minimum resident warps per SM the register cap is set for
#endif
#ifndef HEGET_MINW32_N4
#define HEGET_MINW32_N4 8                 // fp32 4-photon kernel: minimum resident warps per SM; 8 = no cap (110 registers).
                                          // Measured: 24 (80 registers) 0.521 ms, 32 (64 registers) 0.525 ms against 0.502 ms
                                          // uncapped (no spills in any of them): the persistent fp32 kernel prefers registers
#endif
#ifndef HEGET_MINW64_N5
#define HEGET_MINW64_N5 24                // ... of the 5-photon kernel (124 -> 78 registers, no spills: 5.02 -> 4.63 ms;
                                          // the same cap leaves 6 gamma unchanged and costs 1-3 % at 7 and 8 gamma)
#endif
#ifndef HEGET_MINW64_N4
#define HEGET_MINW64_N4 32                // ... of the 4-photon kernel (95 -> 80 registers: 0.768 -> 0.746 ms in v8; v9 with
                                          // the one-phase pair table: 80 -> 72 -> 64 registers, no spills, 16 CTAs per SM:
                                          // 0.713 -> 0.704 -> 0.701 ms; for n >= 6 such caps spill and are 15-30 % slower)
#endif

// CTA size of the tree kernels.  Small CTAs (64 threads: 4 events at n = 4) put more CTAs, each in
// its own phase (load / tables / tree), on an SM at the same number of warps, which overlaps the
// latency-bound phases better: measured on B200, 256 -> 64 threads: 4 gamma fp64 1.114 -> 1.012 ms,
// fp32 0.748 -> 0.731 ms, 3 gamma fp64 0.256 -> 0.238 ms, 5-7 gamma 1-2 %.  (The subset and two-sided
// kernels keep 256: they copy index tables per CTA and lose up to 2x at 64.)
#ifndef HEGET_TREE_CTA_THREADS
#define HEGET_TREE_CTA_THREADS 64
#endif
template <int N>
using TreeGeometry = Geometry<N, HEGET_TREE_CTA_THREADS>;

// n <= HEGET_THREAD_MAXN runs one thread per event (amp2_thread.cu); the lane-per-helicity kernel below
// serves the larger n
#ifndef HEGET_THREAD_MAXN
#define HEGET_THREAD_MAXN 4
#endif

namespace {

#ifndef HEGET_SHARE32_MAXN
#define HEGET_SHARE32_MAXN 0   // fp32: lane sharing of the last level for N up to this; 0 = off (measured: no gain,
                               // 3 gamma -6 %, 4 gamma +4 %, 5-7 gamma +-1 %: the shuffles cost the issue slots they save)
#endif
#ifndef HEGET_CLOSE
#define HEGET_CLOSE 2   // 1: last fvixx0 + iovxxx of a branch as vertex + closing-table dot (amp2_tree.cuh, v7)
                        // 2: the two orderings below a prefix of n-2 photons as ONE dot with the pair closing
                        //    table (v8).  Measured on B200, 1 -> 2: 4 gamma 0.633 -> 0.549 ms fp32, 1.024 ->
                        //    0.762 ms fp64; 8 gamma 841 -> 575 ms fp32, 1584 -> 951 ms fp64; 2 and 3 gamma
                        //    4-14 % slower (the table costs more than it saves), so those stay on 1 (kClose)
#endif
template <int N>
constexpr int kClose = (HEGET_CLOSE == 2 && N < 4) ? 1 : HEGET_CLOSE;
#ifndef HEGET_SHARE64_MAXN
#define HEGET_SHARE64_MAXN 7
#endif
#ifndef HEGET_SHARE64
#define HEGET_SHARE64 0   // fp64: share the last vertex of a branch between the two helicity lanes that need it
                          // (v4: -8 % at 4 gamma; since the closing table (HEGET_CLOSE) halves that level's work
                          // it costs 1-3 % at 5-7 gamma and gains < 1 % at 4 gamma: off)
#endif
template <int N, typename T>
constexpr int kShare = (sizeof(T) == 8) ? ((N <= HEGET_SHARE64_MAXN) ? HEGET_SHARE64 : 0) : ((N <= HEGET_SHARE32_MAXN) ? 1 : 0);  // N = 8: too few in-warp pairs, 2 % slower

// Small N: the spinors of the first two tree levels depend on two photons' helicities only, so
// the 2^N lanes of an event would each recompute the same N(N-1)*4 values (N = 4: 30 % of a
// lane's tree).  With kTopShare the event's lanes compute each psi_2(i, j; h_i, h_j) once into
// shared memory and every lane starts its N(N-1) subtrees from there.
// Measured on B200 (2^20 events): 4 gamma fp64 1.350 -> 1.204 ms (v4); fp32 unchanged then, 0.554 ->
// 0.526 ms since the pair closing table made the rest of the lane's tree cheap (v8); 5 gamma slower
// in both precisions (the subtrees below depth 2 then start from three photons instead of the
// four that Bottom<4> unrolls), so it is on for the 4-photon kernels only.
#ifndef HEGET_TOPSHARE32
#define HEGET_TOPSHARE32 1
#endif
#ifndef HEGET_PAIR_DIRECT
#define HEGET_PAIR_DIRECT 1   // pair closing table in one phase (build_pair_table_direct, amp2_common.cuh)
#endif
#ifndef HEGET_TOP_FACTORISED
#define HEGET_TOP_FACTORISED 1
#endif
template <int N, typename T>
constexpr bool kTopShare = (N == 4 && (sizeof(T) == 8 || HEGET_TOPSHARE32 != 0));

// v9: factorised nodes psi = z v (amp2_chain.cuh) on top of the pair closing table.  Measured on
// B200 see DESIGN.md section 6.1; n = 4 keeps the v8 form (its tree is 12 dots per lane on top of the
// shared first two levels; the K table would cost more than it saves).
#ifndef HEGET_CHAIN
#define HEGET_CHAIN 1
#endif
#ifndef HEGET_CHAIN_MINN
#define HEGET_CHAIN_MINN 5
#endif
#ifndef HEGET_CHAIN_KB32
#define HEGET_CHAIN_KB32 5   // unrolled bottom levels of the factorised walk, fp32 / fp64
#endif
#ifndef HEGET_CHAIN_KB64
#define HEGET_CHAIN_KB64 5   // n >= 6, with the register cap lifted (HEGET_MINB64 = 1: 160-185 registers, 8-12 warps per
                             // SM, no spills).  Measured against four levels under the 128-register cap (16 warps):
                             // 6 gamma 34.1 -> 29.5 ms, 7 gamma 110.8 -> 96.6 ms, 8 gamma 440 -> 375 ms; five levels
                             // UNDER the cap spill 800 B
#endif
template <int N, typename T>
constexpr int kChainBottom = (sizeof(T) == 4) ? ((N < HEGET_CHAIN_KB32) ? N : HEGET_CHAIN_KB32)
                                              : ((N < 6) ? ((N < 4) ? N : 4) : HEGET_CHAIN_KB64);  // 5 gamma: capped at 80 registers
template <int N>
constexpr bool kChain = (HEGET_CHAIN != 0) && (kClose<N> == 2) && (N >= HEGET_CHAIN_MINN) && (N > HEGET_KB - 1) && (HEGET_KB >= 3);

template <int N>
constexpr int kBottom = (N < HEGET_KB) ? N : HEGET_KB;  // unrolled bottom levels of the tree

// A CTA's batch (256 / 2^N events) lasts only a few microseconds for small N, so the DRAM latency
// of its momenta is a visible fraction of it.  Where it pays, the grid is sized to the number of
// resident CTAs and each CTA loops over batches with the next batch's loads in flight
// (registers) while it computes the current one.  Measured on B200 (2^20 events): fp32 4 gamma
// 0.862 -> 0.755 ms, 5 gamma 6.48 -> 6.39 ms; fp32 3 gamma and every fp64 kernel are 1-6 % SLOWER
// that way (two 128-register CTAs per SM overlap their phases better when CTAs turn over), so
// those keep one batch per CTA.
#ifndef HEGET_PERSIST32
#define HEGET_PERSIST32 1
#endif
#ifndef HEGET_PERSIST64_N4
#define HEGET_PERSIST64_N4 0
#endif
template <int N, typename T>
constexpr bool kPersistent = (HEGET_PERSIST32 != 0 && (sizeof(T) == 4) && (N == 4 || N == 5)) || (HEGET_PERSIST64_N4 != 0 && sizeof(T) == 8 && N == 4);

template <int N, typename T>
__global__ void __launch_bounds__(TreeGeometry<N>::THREADS,
                                  ((sizeof(T) == 4) ? ((N == 4) ? HEGET_MINW32_N4 * 32 : HEGET_MINB32 * 256) : (N == 4 ? HEGET_MINW64_N4 : (N == 5 ? HEGET_MINW64_N5 : HEGET_MINW64)) * 32) /
                                      TreeGeometry<N>::THREADS)
amp2_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g,
            int64_t n_batches)
{
    using G = TreeGeometry<N>;
    using Tile = MomentaTile<N, G>;
    constexpr int MOM = 4 * (N + 2);
    __shared__ __align__(16) double s_mom[G::EPB * MOM];
    __shared__ PEntry<T> s_P[G::EPB * G::L];
    __shared__ EEntry<T> s_E[G::EPB * 2 * N];
    __shared__ double s_red[G::THREADS / 32];
    __shared__ double s_s2[G::EPB * N];  // s_i^2 = (pT/w)^2 taken out of photon i's E entries
    __shared__ Spinor<T> s_U[(kClose<N> == 2 && HEGET_PAIR_DIRECT != 0) ? 1 : G::EPB * 2 * N];  // closing table (amp2_tree.cuh, close_weyl)
    constexpr int NW = (kClose<N> == 2) ? 4 * (N * (N - 1) / 2) : 1;  // pair closing table entries per event
    __shared__ Spinor<T> s_W[(kClose<N> == 2) ? G::EPB * NW : 1];
    constexpr int TOP = kTopShare<N, T> ? N * (N - 1) * 4 : 1;  // psi_2 entries per event
    __shared__ Spinor<T> s_top[kTopShare<N, T> ? G::EPB * TOP : 1];
    constexpr int NK = kChain<N> ? (N * (N - 1) / 2) * N * 8 : 1;  // K table entries per event (amp2_chain.cuh)
    __shared__ Cx<T> s_K[kChain<N> ? G::EPB * NK : 1];

    const int ev_local = threadIdx.x / G::L;
    const unsigned hel = threadIdx.x % G::L;

    double2 pf[Tile::PF];
    int64_t batch = blockIdx.x;
    Tile::load(momenta, batch * G::EPB, n_events, pf);                       // a1
    do {  // one pass unless kPersistent (grid = number of batches)
        Tile::store(s_mom, pf);
        __syncthreads();
        if constexpr (kPersistent<N, T>) {
            if (batch + gridDim.x < n_batches) Tile::load(momenta, (batch + gridDim.x) * G::EPB, n_events, pf);
        }
        build_tables<N, T, G>(g, s_mom, s_P, s_E, s_s2);                        // a4, a5 (ends with a barrier)
        if constexpr (kClose<N> == 2 && HEGET_PAIR_DIRECT != 0) {
            // W straight from P and E; with kTopShare the barrier is the one after the top table below
            build_pair_table_direct<N, T, G, !kTopShare<N, T>>(s_P, s_E, s_W);
        } else {
            if constexpr (kClose<N> != 0) build_closing_table<N, T, G>(s_P, s_E, s_U);
            if constexpr (kClose<N> == 2) build_pair_table<N, T, G>(s_U, s_E, s_W);
        }
        if constexpr (kChain<N>) build_chain_table<N, T, G>(s_P, s_E, s_W, s_K);
        const Spinor<T>* closing = (kClose<N> == 2) ? s_W + ev_local * NW : s_U + ev_local * 2 * N;

        // a2, a6, a7: psi_0 = u(p1,+)/sqrt(2E1) = (1,0); walk the permutation tree
        T ar = 0, ai = 0;
        const Spinor<T> f0 = {(T)1, (T)0, (T)0, (T)0};
        const PEntry<T>* P = s_P + ev_local * G::L;
        const EEntry<T>* E = s_E + ev_local * 2 * N;
        if constexpr (kTopShare<N, T>) {
            // entry q = ((i * (N-1) + jj) * 4 + 2 h_i + h_j), j = jj + (jj >= i): psi_2 = node(node(u, i), j)
            Spinor<T>* top = s_top + ev_local * TOP;
            for (int q = (int)hel; q < TOP; q += G::L) {
                const int pair = q >> 2, i = pair / (N - 1), jj = pair % (N - 1), j = jj + (jj >= i ? 1 : 0);
#if HEGET_TOP_FACTORISED
                // factorised form (amp2_chain.cuh): psi_1 = v({i}, i), psi_2 = (v_0 + b_j v_1) v({i,j}, j),
                // 24 instead of 40 instructions per entry
                const EEntry<T> ej = E[2 * j + (q & 1)];
                T rr, ri;
                chain_rho(chain_vector(P[1u << i], E[2 * i + ((q >> 1) & 1)]), ej, rr, ri);
                const Spinor<T> v2 = chain_vector(P[(1u << i) | (1u << j)], ej);
                Spinor<T> f2;
                f2.r0 = fma(rr, v2.r0, -(ri * v2.i0));
                f2.i0 = fma(rr, v2.i0, ri * v2.r0);
                f2.r1 = fma(rr, v2.r1, -(ri * v2.i1));
                f2.i1 = fma(rr, v2.i1, ri * v2.r1);
                top[q] = f2;
#else
                const Spinor<T> f1 = fvixx0_weyl(P[1u << i], E[2 * i + ((q >> 1) & 1)], f0);
                top[q] = fvixx0_weyl(P[(1u << i) | (1u << j)], E[2 * j + (q & 1)], f1);
#endif
            }
            __syncthreads();
#pragma unroll
            for (int i = 0; i < N; ++i)
#pragma unroll
                for (int jj = 0; jj < N - 1; ++jj) {
                    const int j = jj + (jj >= i ? 1 : 0);
                    const Spinor<T> f2 = top[(i * (N - 1) + jj) * 4 + 2 * ((hel >> i) & 1u) + ((hel >> j) & 1u)];
                    Walk<N, 2, N - 2, T, kShare<N, T>, kClose<N>>::run(P, E, hel, (1u << i) | (1u << j), f2, ar, ai,
                                                                        closing);
                }
        } else if constexpr (kChain<N>) {
            // the root is v = (1, 0): rho = v_0 + b v_1 = 1 for every first photon; ampsum = A(root)
            WalkChain<N, 0, kChainBottom<N, T>, T>::run(P, E, hel, 0u, f0, ar, ai, s_K + ev_local * NK);
        } else {
            Walk<N, 0, kBottom<N>, T, kShare<N, T>, kClose<N>>::run(P, E, hel, 0u, f0, ar, ai, closing);
        }

        // a8: |ampsum|^2 summed over the event's 2^N lanes, constant factors, store
        finish_event<N, T, G>(ar, ai, s_mom, s_s2, s_red, g, out, batch * G::EPB, n_events);
        if constexpr (kPersistent<N, T>) __syncthreads();                    // tables are rewritten next round
    } while (kPersistent<N, T> && (batch += gridDim.x) < n_batches);
}

template <int N, typename T>
cudaError_t launch_one(const heget_ctx* ctx, const double* momenta, double* out, int64_t n_events, double g,
                       cudaStream_t stream)
{
    using G = TreeGeometry<N>;
    const int64_t n_batches = (n_events + G::EPB - 1) / G::EPB;
    int64_t blocks = n_batches;
    if (kPersistent<N, T>) {
        int per_sm = 0;
        cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, amp2_kernel<N, T>, G::THREADS, 0);
        if (err != cudaSuccess) return err;
        const int64_t resident = (int64_t)ctx->sm_count * (per_sm > 0 ? per_sm : 1);
        if (blocks > resident) blocks = resident;
    }
    amp2_kernel<N, T><<<(unsigned)blocks, G::THREADS, 0, stream>>>(momenta, out, n_events, g, n_batches);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_n(const heget_ctx* ctx, int n, const double* momenta, double* out, int64_t n_events, double g,
                     cudaStream_t stream)
{
    switch (n) {
        case 2: return launch_one<2, T>(ctx, momenta, out, n_events, g, stream);
        case 3: return launch_one<3, T>(ctx, momenta, out, n_events, g, stream);
        case 4: return launch_one<4, T>(ctx, momenta, out, n_events, g, stream);
        case 5: return launch_one<5, T>(ctx, momenta, out, n_events, g, stream);
        case 6: return launch_one<6, T>(ctx, momenta, out, n_events, g, stream);
        case 7: return launch_one<7, T>(ctx, momenta, out, n_events, g, stream);
        case 8: return launch_one<8, T>(ctx, momenta, out, n_events, g, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t heget_launch_amp2(const heget_ctx* ctx, const double* momenta, int n, int precision,
                              double* out_amp2, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    if (n <= HEGET_THREAD_MAXN) return heget_launch_amp2_thread(ctx, momenta, n, precision, out_amp2, N, stream, launches);
    *launches = 1;
    if (precision == HEGET_FP32) return launch_n<float>(ctx, n, momenta, out_amp2, N, ctx->g, stream);
    return launch_n<double>(ctx, n, momenta, out_amp2, N, ctx->g, stream);
}

// amp2.cu -- heget_amp2: summed squared helicity amplitude of u ubar -> n gamma (product code).
//
// n <= 6 runs in amp2_thread.cu (one thread, at n = 6 two or four lanes, per event).  This file is the kernel for
// n >= 7 (it is instantiated for n = 6 too: HEGET_THREAD_MAXN = 5 puts 6 photons back on it):
// one lane per photon-helicity configuration (2^N lanes per event), one event per CTA of 2^N
// threads.  All lanes of a CTA walk the SAME
// permutation tree in lockstep (no divergence); they differ only in which helicity entry of the
// per-photon and per-subset tables they read.  Per event the CTA first builds, in shared memory,
//   - the E table (vxxxx0 for both helicities of every photon),
//   - the subset table P[S] = -g/t_S * (p1 - K_S)-slash block for every photon subset S,
//   - the pair closing table W, the table of closing dots K and the rho table R (amp2_chain.cuh),
// then every lane runs the depth-first walk of eq. (6)'s n! orderings: each ordered
// prefix (tree node) is one fvixx0 in factorised form psi = z v, computed once;
// the two orderings below a prefix of n-2 photons close through the per-event tables (iovxxx,
// PAPER.md:592-620; List 2).
// Only sigma_1 = +1, sigma_2 = -1 is evaluated: sigma_1 = sigma_2 vanishes identically and
// |M(-sigma,-lambda)| = |M(sigma,lambda)|, so the helicity sum is twice the sum over lambda.
#include "amp2_chain.cuh"

#ifndef HEGET_THREAD_MAXN
#define HEGET_THREAD_MAXN 6   // n up to this runs in amp2_thread.cu (5: 6 photons stay on the lane kernel below)
#endif
#ifndef HEGET_MINB32
#define HEGET_MINB32 1      // fp32, n >= 6: __launch_bounds__ min CTAs of 256 threads per SM; 1 = no register cap (the six
                            // unrolled levels take 250 registers; capped at 128 they spill 600 B: 8 gamma 132 against 102 ms)
#endif
#ifndef HEGET_MINW64
#define HEGET_MINW64 12     // fp64, n = 6: minimum resident warps per SM the register cap is set for (168 registers, no
                            // spills; measured 8 -> 12: 24.0 -> 21.6 ms); n >= 7 run uncapped (six unrolled levels)
#endif

// CTA size: at least 64 threads; from 6 photons on an event's 2^N lanes are one CTA.
#ifndef HEGET_TREE_CTA_THREADS
#define HEGET_TREE_CTA_THREADS 64
#endif
template <int N>
using TreeGeometry = Geometry<N, HEGET_TREE_CTA_THREADS>;

namespace {

#ifndef HEGET_CHAIN_KB32
#define HEGET_CHAIN_KB32 6   // unrolled bottom levels of the factorised walk, fp32 / fp64.  With nodes as cheap as the rho
                             // table makes them, the per-lane address lists set up at the top of the unrolled part
                             // must be amortised over many nodes: measured 5 (128 registers, 2 CTAs per SM) -> 6
                             // (250 registers, 1 CTA): 6 gamma 14.8 -> 12.2 ms, 7 gamma 41.9 -> 29.4, 8 gamma 167 -> 102
#endif
#ifndef HEGET_CHAIN_KB64
#define HEGET_CHAIN_KB64 6   // fp64, n >= 7 (n = 6: five levels).  Six levels need the
                             // E' entries of the list re-read from shared memory (kEByPtr) and still spill 0.7-1 KB at 255
                             // registers, but win: measured 5 -> 6: 7 gamma 63.7 -> 56.8 ms, 8 gamma 257 -> 194 ms
                             // (6 gamma 21.0 -> 23.8: stays at five)
#endif
template <int N, typename T>
constexpr int kChainBottom = (sizeof(T) == 4) ? HEGET_CHAIN_KB32 : ((N == 6) ? 5 : HEGET_CHAIN_KB64);

#ifndef HEGET_CHAIN_E_BY_PTR64
#define HEGET_CHAIN_E_BY_PTR64 1   // fp64, six unrolled levels: re-read the E' entries of the list from shared memory
#endif
template <int N, typename T>
constexpr bool kEByPtr = (sizeof(T) == 8) && (HEGET_CHAIN_E_BY_PTR64 != 0) && (kChainBottom<N, T> >= 6);

// per-event entries of the tables of the factorised walk (dynamic shared memory of amp2_kernel)
template <int N, typename T>
struct ChainTables {
    static constexpr int NW = 4 * (N * (N - 1) / 2);          // pair closing rows W
    static constexpr int NK = kChainEntries<N, T>;            // closing dots K
    static constexpr int NR = kRhoEntries<N, T>;              // rho of the last attachment
    static constexpr size_t BYTES = (size_t)TreeGeometry<N>::EPB * (NK + NR) * sizeof(Cx<T>);
};

template <int N, typename T>
constexpr int kMinBlocks = ((sizeof(T) == 4) ? HEGET_MINB32 * 256 : ((N == 6) ? HEGET_MINW64 : 8) * 32) / TreeGeometry<N>::THREADS;

template <int N, typename T>
__global__ void __launch_bounds__(TreeGeometry<N>::THREADS, kMinBlocks<N, T>)
amp2_kernel(const double* __restrict__ momenta, double* __restrict__ out, int64_t n_events, double g)
{
    using G = TreeGeometry<N>;
    using Tile = MomentaTile<N, G>;
    using Tab = ChainTables<N, T>;
    constexpr int MOM = 4 * (N + 2);
    __shared__ __align__(16) double s_mom[G::EPB * MOM];
    __shared__ PEntry<T> s_P[G::EPB * G::L];
    __shared__ EEntry<T> s_E[G::EPB * 2 * N];
    __shared__ double s_red[G::THREADS / 32];
    __shared__ double s_s2[G::EPB * N];  // s_i^2 = (pT/w)^2 taken out of photon i's E entries
    __shared__ Spinor<T> s_W[G::EPB * Tab::NW];
    // K and rho tables: opt-in dynamic shared memory (n = 8 fp64: 28 + 54 KB)
    extern __shared__ __align__(16) unsigned char s_dyn[];
    Cx<T>* s_K = reinterpret_cast<Cx<T>*>(s_dyn);
    Cx<T>* s_R = s_K + G::EPB * Tab::NK;

    const int ev_local = threadIdx.x / G::L;
    const unsigned hel = threadIdx.x % G::L;

    const int64_t ev0 = (int64_t)blockIdx.x * G::EPB;
    double2 pf[Tile::PF];
    Tile::load(momenta, ev0, n_events, pf);                                  // a1
    Tile::store(s_mom, pf);
    __syncthreads();
    build_tables<N, T, G>(g, s_mom, s_P, s_E, s_s2);                            // a4, a5 (every build_* ends with a barrier)
    build_pair_table_direct<N, T, G>(s_P, s_E, s_W);
    build_chain_table<N, T, G>(s_P, s_E, s_W, s_K);
    build_rho_table<N, T, G>(s_P, s_E, s_R);

    // a2, a6, a7: psi_0 = u(p1,+)/sqrt(2E1) = (1,0) is the root vector (rho = v_0 + b v_1 = 1 for every
    // first photon); ampsum = A(root)
    T ar = 0, ai = 0;
    const Spinor<T> f0 = {(T)1, (T)0, (T)0, (T)0};
    WalkChain<N, 0, kChainBottom<N, T>, T, kEByPtr<N, T>>::run(s_P + ev_local * G::L, s_E + ev_local * 2 * N, hel, 0u, f0, ar, ai,
                                                 s_K + ev_local * Tab::NK, s_R + ev_local * Tab::NR);

    // a8: |ampsum|^2 summed over the event's 2^N lanes, constant factors, store
    finish_event<N, T, G>(ar, ai, s_mom, s_s2, s_red, g, out, ev0, n_events);
}

template <int N, typename T>
cudaError_t launch_one(const heget_ctx* ctx, const double* momenta, double* out, int64_t n_events, double g,
                       cudaStream_t stream)
{
    using G = TreeGeometry<N>;
    constexpr size_t dyn = ChainTables<N, T>::BYTES;
    // more than the 48 KB a kernel gets without asking (n = 8).  Set on every launch: the attribute belongs to the
    // current device, and a process may hold contexts on several
    const cudaError_t attr =
        cudaFuncSetAttribute(amp2_kernel<N, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    if (attr != cudaSuccess) return attr;
    const int64_t blocks = (n_events + G::EPB - 1) / G::EPB;
    amp2_kernel<N, T><<<(unsigned)blocks, G::THREADS, dyn, stream>>>(momenta, out, n_events, g);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_n(const heget_ctx* ctx, int n, const double* momenta, double* out, int64_t n_events, double g,
                     cudaStream_t stream)
{
    switch (n) {
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

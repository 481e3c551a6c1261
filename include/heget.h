/* heget.h -- C ABI of libheget.so: B200 (sm_100a) evaluation of the summed squared
 * helicity amplitude of u ubar -> n gamma, n = 2..8 (arXiv 0908.4403, "HEGET").
 *
 * Citations are PAPER.md line numbers of the paper text this library was written from.
 *
 * Conventions common to all calls
 *  - every function returns 0 (HEGET_OK) or a negative HEGET_E* code; nothing aborts and
 *    nothing throws across this boundary; heget_strerror() gives the text, and for
 *    HEGET_ECUDA heget_last_cuda_error() gives the CUDA runtime's message;
 *  - pointers marked [dev] are device pointers on the context's device, owned by the
 *    caller (e.g. a torch tensor's data_ptr()); pointers marked [host] are host pointers
 *    (pinned or pageable).  The library allocates nothing per call for the [dev] entry
 *    points; the *_host entry points use staging buffers owned by the context;
 *  - [dev] calls are asynchronous on `stream` (a cudaStream_t passed as void*, NULL = the
 *    legacy default stream) and do not synchronise the host; *_host calls return after
 *    the result is in the host buffer;
 *  - a context is not thread-safe: host calls on the SAME heget_ctx must not overlap in time
 *    (different contexts, e.g. one per GPU or per host thread, are independent).  [dev] calls
 *    of one context may be issued on DIFFERENT streams and run concurrently; the only scratch a
 *    [dev] call uses is heget_xsec_reduce's block partials, a ring of HEGET_REDUCE_SLOTS
 *    buffers used round-robin, so at most HEGET_REDUCE_SLOTS reductions of one context may be
 *    in flight at the same time (heget_xsec_host has staging and partials of its own);
 *  - momenta layout: double[N][n+2][4], four-vectors (E,px,py,pz) (PAPER.md:474-477,
 *    553-554), particle order u, ubar, gamma_1..gamma_n (p1..p5 of List 2);
 *    the base pointer must be 16-byte aligned.
 *  - preconditions (documented, not checked on the hot path; PAPER.md:203-205 makes the
 *    same assumptions by choosing ixxxx1 / oxxxx2 / branch-free vxxxx0):
 *    p1 = (E1,0,0,+E1), p2 = (E2,0,0,-E2), photons massless to rounding with pT > 0.
 */
#ifndef HEGET_H
#define HEGET_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct heget_ctx heget_ctx; /* opaque; owned by the library */

enum { HEGET_FP32 = 0, HEGET_FP64 = 1 };

enum {
    HEGET_OK = 0,
    HEGET_EINVAL = -1, /* n outside [2,8], N < 0 or > HEGET_MAX_EVENTS, null pointer, bad precision/mode */
    HEGET_ECUDA = -2,  /* a CUDA runtime call or launch failed */
    HEGET_ENOMEM = -3, /* host or device allocation failed */
    HEGET_ETOOBIG = -4 /* N exceeds the fixed scratch of a no-allocation entry point */
};

/* Largest N (events, or items of the heget_helas_* calls) one call accepts: the kernels that give
 * an event a CTA of its own (n >= 6) are launched on a grid of N blocks and CUDA's grid limit is
 * 2^31 - 1.  A larger batch is cut by the caller (per-event results do not depend on the cut);
 * at 32 (n + 2) bytes of momenta per event such a batch does not fit one B200 anyway. */
#define HEGET_MAX_EVENTS 2147483647LL

/* heget_xsec_reduce calls of one context that may be in flight on different streams at once. */
#define HEGET_REDUCE_SLOTS 8

/* Event-generation modes of heget_gen_events ("input recipe"). */
enum {
    HEGET_GEN_FIXED = 0,      /* sqrt_s_hat = a, y = 0 */
    HEGET_GEN_LOGUNIFORM = 1, /* sqrt_s_hat = a (b/a)^u log-uniform in [a,b], y uniform in [-y_max,y_max] */
    HEGET_GEN_TOYPDF = 2      /* pp at sqrt(s) = a with f(x) = x^-0.5 (1-x)^3 for both partons */
};

typedef struct heget_gen_cfg {
    int mode;       /* HEGET_GEN_* */
    int apply_cuts; /* 0: weight never zeroed; 1: eq. (9) cuts from the context */
    double a;       /* see mode */
    double b;       /* see mode */
    double y_max;   /* HEGET_GEN_LOGUNIFORM only */
} heget_gen_cfg;

/* Create a context on CUDA device `device`.
 *   alpha, q_charge : fine-structure constant and quark charge; the FFV coupling is
 *                     gal[0] = gal[1] = -e Q_q, e = sqrt(4 pi alpha) (eq. 26)
 *   pt_cut, eta_cut, dr_cut : final-state cuts of eq. (9); finite and >= 0
 * alpha <= 0 or a non-finite argument gives HEGET_EINVAL.
 * *out is written on success only and must be released with heget_destroy. */
int heget_init(int device, double alpha, double q_charge, double pt_cut, double eta_cut,
               double dr_cut, heget_ctx** out);
void heget_destroy(heget_ctx* ctx);
const char* heget_strerror(int code);
const char* heget_last_cuda_error(const heget_ctx* ctx);

/* Phase space generation from random numbers, step 4 of PAPER.md:116-122 ("generates a
 * phase space point and computes a Jacobian") with device-side Philox4x32-10
 * and RAMBO (neither is named by the paper; BASELINE.json fixes them, R6/R7).
 * heget_rambo is the north-star form: fixed sqrt_s_hat, partonic rest frame, u along +z,
 * ubar along -z, no cuts.  Event e uses Philox counter (e, slot) with key `seed`.
 *   momenta [dev] double[N][n+2][4], written. */
int heget_rambo(heget_ctx* ctx, uint64_t seed, int n, double sqrt_s_hat, int64_t N,
                double* momenta, void* stream);

/* General form: per-event sqrt_s_hat and boost rapidity y according to cfg, cuts of eq. (9)
 * evaluated in the boosted frame, and the event weight
 *   w = [cuts] * Phi_n(s_hat) / (2 s_hat) * (TOYPDF: Jacobian * 2 f(x1) f(x2))
 * (eqs. 1-4).  Global event index = first_event + local index, so any
 * contiguous shard of a run reproduces the same events (multi-GPU: shard by index range).
 * HEGET_GEN_TOYPDF needs tau_min = (n pt_cut)^2 / a^2 inside (0, 1) (the context's pt_cut > 0),
 * else HEGET_EINVAL; weight must not be NULL.
 *   momenta [dev] double[N][n+2][4], weight [dev] double[N]; both written. */
int heget_gen_events(heget_ctx* ctx, uint64_t seed, int n, const heget_gen_cfg* cfg,
                     uint64_t first_event, int64_t N, double* momenta, double* weight,
                     void* stream);

/* The hot path.  For each event: external wavefunctions (ixxxx1, oxxxx2, vxxxx0;
 * PAPER.md:435-439), the fvixx0 chain through the propagators (p1 - K_l)/t_l of eqs. (7),(8)
 * over all n! photon orderings of eq. (6), walked
 * as a depth-first permutation tree with every prefix computed once, closed by iovxxx
 * (the two orderings below a prefix of n-2 photons are closed together
 * through a per-event table built from the ubar side; each fvixx0 of the walk is evaluated in
 * factorised form, a complex number times a per-(subset, photon) vector, which the rank-one
 * polarisation blocks of massless photons allow; n <= 5: one thread per event, n = 6: two or
 * four lanes per event, n >= 7: one lane per photon-helicity assignment), squared and
 * summed over all 4*2^n helicities:
 *   out_amp2[e] = sum_{sigma1,sigma2,lambda_1..lambda_n} |M|^2   (the sum in eq. 2,
 *   PAPER.md:37, WITHOUT 1/(2 s_hat), spin/colour average and 1/n!).
 * precision selects the arithmetic of the tree walk (separate fp32 and fp64 kernels);
 * input and output buffers are fp64 in both cases (the fp32 kernel rescales each event to
 * unit s_hat internally because |M|^2 ~ s_hat^(2-n) leaves the fp32 range).
 *   momenta [dev] const double[N][n+2][4]; out_amp2 [dev] double[N], written. */
int heget_amp2(heget_ctx* ctx, const double* momenta, int n, int precision, double* out_amp2,
               int64_t N, void* stream);

/* The same quantity with a selectable organisation of the permutation sum:
 *   HEGET_ALGO_TREE    depth-first permutation tree with prefix reuse (= heget_amp2; the method
 *                      of eq. 6 / List 2)
 *   HEGET_ALGO_SUBSET  recursion over photon subsets: Psi(S) = P_S sum_{i in S} E_i Psi(S\i); the
 *                      propagators of eq. (8) depend on the set S only, so the n! orderings
 *                      collapse onto 2^n sets (3^n - 1 spinors per event including helicities).
 *                      Same result up to rounding order; NOT the permutation-tree method, hence a
 *                      separately named mode (reuse of off-shell lines).
 *   HEGET_ALGO_TREE2   two-sided chaining: the permutation tree from the u end (fvixx0) is walked
 *                      to depth n - KS only, KS = min(n,4), and every branch closes with one dot product
 *                      against row vectors chained from the ubar end (fvoxx0 of List 2,
 *                      PAPER.md:449-450, 642-656) and tabulated per photon set: the same n!
 *                      diagrams with the off-shell lines near the ubar end shared.
 * Arguments, layout and errors as heget_amp2; algo outside the enum gives HEGET_EINVAL. */
enum { HEGET_ALGO_TREE = 0, HEGET_ALGO_SUBSET = 1, HEGET_ALGO_TREE2 = 2 };
int heget_amp2_algo(heget_ctx* ctx, const double* momenta, int n, int precision, int algo,
                    double* out_amp2, int64_t N, void* stream);

/* The paper's own event loop (step 4 of PAPER.md:116-122): ONE random helicity assignment per
 * event instead of the explicit helicity sum.  Event e (global index first_event + e) draws
 * Philox4x32-10 with key `seed` and counter (event_lo, event_hi, 15, 0); bit b of the first
 * output word is the helicity of particle b in the order u, ubar, gamma_1..gamma_n (1 -> +1,
 * 0 -> -1).  out_amp2[e] = 4 * 2^n * |M(h_e)|^2, whose mean over h is the helicity sum that
 * heget_amp2 returns (exactly 0 for sigma_1 = sigma_2); out_hel[e] = the n+2 bits drawn
 * (step 5), or pass NULL.  Permutation tree as heget_amp2, one warp per event.
 *   momenta [dev] const double[N][n+2][4]; out_amp2 [dev] double[N]; out_hel [dev] int32[N]. */
int heget_amp2_sampled(heget_ctx* ctx, uint64_t seed, uint64_t first_event, const double* momenta,
                       int n, int precision, double* out_amp2, int32_t* out_hel, int64_t N,
                       void* stream);

/* Kinematical distributions of Fig. 2 as weighted histograms, filled on the
 * device: event e adds value[e] (e.g. weight * amp2; 0 = event failed the cuts, skipped) at
 *   HEGET_OBS_PT_MAX  max_i pT(gamma_i)                         (eq. 9)
 *   HEGET_OBS_DR_MIN  min_{i<j} Delta R_ij                      (eq. 10)
 *   HEGET_OBS_DR_ALL  every Delta R_ij (n(n-1)/2 entries per event)
 * with eta = asinh(pz/pT) and Delta phi wrapped to [0, pi].  nbins equal bins on [lo, hi):
 * hist[0] = underflow (x < lo), hist[1..nbins], hist[nbins+1] = overflow (x >= hi or NaN).
 * hist is zeroed by the call.  1 <= nbins <= HEGET_HIST_MAX_BINS, hi > lo, else HEGET_EINVAL.
 * Additions are fp64 atomics: bin assignment is deterministic, the summation order is not.
 *   momenta [dev] const double[N][n+2][4]; value [dev] const double[N];
 *   hist [dev] double[nbins+2], written. */
enum { HEGET_OBS_PT_MAX = 0, HEGET_OBS_DR_MIN = 1, HEGET_OBS_DR_ALL = 2 };
#define HEGET_HIST_MAX_BINS 4094
int heget_histogram(heget_ctx* ctx, const double* momenta, const double* value, int n, int64_t N,
                    int observable, double lo, double hi, int nbins, double* hist, void* stream);

/* The complete HEGET function set of Tables 3 and 4, batched: one call evaluates
 * one function on N inputs.  A wavefunction is cmplx w[6] = double[6][2]: components 0..3 the
 * 4-spinor / 4-vector, w[4] = (p0, p3) * nS and w[5] = (p1, p2) * nS the flowing momentum
 * (PAPER.md:553-554).  Massless, branch-free; "0" = generic direction (spinors: p0 + p3 > 0;
 * vectors: pT > 0), "1" = momentum along +z, "2" = along -z (only p[0] is read).
 *   heget_helas_wavefunction: fn = HEGET_FN_*; p [dev] const double[N][4] = (E,px,py,pz);
 *     nhel = +-1 (twice the helicity / the helicity), ns = nSF or nSV = +-1 (PAPER.md:474-487,
 *     eqs. 11-13); w [dev] double[N][6][2], written.
 *   heget_helas_vertex: fn = HEGET_VTX_*; gal[0] = gal[1] = g (eq. 26);
 *     IOVXXX(fi,fo,vc) -> out [dev] double[N][2], the amplitude g <fo|vc-slash|fi>
 *     FVIXX0(fi,vc)    -> out [dev] double[N][6][2], -g pf-slash vc-slash |fi> / pf^2, pf = p_fi - p_vc
 *     FVOXX0(fo,vc)    -> out [dev] double[N][6][2], -g <fo| vc-slash pf-slash / pf^2, pf = p_fo + p_vc
 *     JIOXX0(fi,fo)    -> out [dev] double[N][6][2], g <fo|gamma^mu|fi> / q^2, q = p_fo - p_fi
 *     (PAPER.md:622-672); the argument a function does not take may be NULL.
 * precision selects the arithmetic; all pointers 16-byte aligned; errors as for heget_amp2. */
enum {
    HEGET_FN_IXXXX0 = 0, HEGET_FN_IXXXX1 = 1, HEGET_FN_IXXXX2 = 2,
    HEGET_FN_OXXXX0 = 3, HEGET_FN_OXXXX1 = 4, HEGET_FN_OXXXX2 = 5,
    HEGET_FN_VXXXX0 = 6, HEGET_FN_VXXXX1 = 7, HEGET_FN_VXXXX2 = 8
};
enum { HEGET_VTX_IOVXXX = 0, HEGET_VTX_FVIXX0 = 1, HEGET_VTX_FVOXX0 = 2, HEGET_VTX_JIOXX0 = 3 };
int heget_helas_wavefunction(heget_ctx* ctx, int fn, int precision, const double* p, int nhel, int ns,
                             double* w, int64_t N, void* stream);
int heget_helas_vertex(heget_ctx* ctx, int fn, int precision, const double* fi, const double* fo,
                       const double* vc, double g, double* out, int64_t N, void* stream);

/* Step 6 of PAPER.md:141 on the device: with x_e = weight[e] * amp2[e] * (1/4)(1/9)(1/n!)
 * (helicity average, colour factor and identical-photon factor of eq. 2, PAPER.md:37;
 * DESIGN.md R1 for the colour factor),
 *   out3 = { sum_e x_e, sum_e x_e^2, #(weight[e] != 0) }   accumulated in fp64.
 * An event with weight[e] == 0 (failed the cuts) contributes exactly 0 whatever amp2[e] holds, NaN
 * and Inf included (R26: such events are what the cuts remove).
 * The result is deterministic (fixed reduction tree, no floating-point atomics).
 *   amp2, weight [dev] const double[N]; out3 [dev] double[3], written. */
int heget_xsec_reduce(heget_ctx* ctx, const double* amp2, const double* weight, int n, int64_t N,
                      double* out3, void* stream);

/* heget_xsec_reduce for callers that cannot allocate and must not touch allocator-owned scratch: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same arguments and result
 * ({sum x, sum x^2, count}; a different, equally fixed reduction tree, so sums agree with heget_xsec_reduce to
 * rounding, ~1e-15, and are bit-reproducible from call to call).  The block partials live in a file-scope
 * `static __device__` array inside the library: 96 KB that every GPU which loads libheget.so holds until exit.
 * It bounds the batch: N > HEGET_NOALLOC_MAX_EVENTS (2^24) returns HEGET_ETOOBIG (heget_last_cuda_error has
 * the text).  The call launches two kernels on `stream` and calls no cudaMalloc / cudaFree / allocating
 * routine; the first call on a device resolves the array's device address (cudaGetSymbolAddress, once per
 * device) -- make one call before starting a graph capture.  All calls, from every context, share that one
 * array and it keeps the last call's contents (nothing in it needs clearing: a call overwrites what it
 * reads): calls that OVERLAP ON THE GPU -- different streams, concurrent graph launches -- race on it;
 * order them on one stream or with events.
 *   amp2, weight [dev] const double[N]; out3 [dev] double[3], written. */
#define HEGET_NOALLOC_MAX_EVENTS 16777216LL
int heget_xsec_reduce_noalloc(heget_ctx* ctx, const double* amp2, const double* weight, int n, int64_t N,
                              double* out3, void* stream);

/* End-to-end form of the same path with host buffers: copies momenta and weight to the
 * device, runs heget_amp2 and heget_xsec_reduce, copies out_amp2 (if non-NULL) and out3
 * back, and returns when they are in host memory.
 *   momenta [host] const double[N][n+2][4]; weight [host] const double[N];
 *   out_amp2 [host] double[N] or NULL; out3 [host] double[3]. */
int heget_xsec_host(heget_ctx* ctx, const double* momenta, const double* weight, int n,
                    int precision, int64_t N, double* out_amp2, double* out3);

#ifdef __cplusplus
}
#endif
#endif /* HEGET_H */

/* oracle/heget_oracle.c -- TEST INFRASTRUCTURE, not product code.
 *
 * CPU oracle for the summed squared helicity amplitude of u ubar -> n gamma
 * (arXiv 0908.4403, eqs. 2, 5-8).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this library.  It shares no code with the CUDA path.
 *
 * The arithmetic lives in amp_body.inc, instantiated in double (suffix _d, the
 * oracle proper and the timed CPU baseline) and in long double (suffix _ld, x87
 * 80-bit, used to certify the double result and as the parity reference where a
 * 1e-12 gate would otherwise be decided by the oracle's own rounding; pin P8 in
 * DESIGN.md).
 *
 * Exported entry points take and return plain double arrays on the host:
 *   momenta : [N][n+2][4]  (E,px,py,pz), particle order u, ubar, gamma_1..gamma_n
 *   nhel    : [n+2] entries +-1, same order
 *   g       : gal[0] = gal[1] = -e Q_q of eq. (26)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REAL double
#define SFX _d
#define SQRT sqrt
#define CREAL creal
#define CIMAG cimag
#include "amp_body.inc"
#undef REAL
#undef SFX
#undef SQRT
#undef CREAL
#undef CIMAG

#define REAL long double
#define SFX _ld
#define SQRT sqrtl
#define CREAL creall
#define CIMAG cimagl
#include "amp_body.inc"
#undef REAL
#undef SFX
#undef SQRT
#undef CREAL
#undef CIMAG

int heget_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* One helicity amplitude ampsum (List 2) for one event.
 * out[0] = Re, out[1] = Im.  gauge_idx >= 0: eps(k_gauge_idx) -> k_gauge_idx. */
void heget_oracle_amp_d(const double *mom, int n, const int *nhel, double g, int gauge_idx, double *out)
{
    const double _Complex m = amp_one_helicity_d(mom, n, nhel, g, gauge_idx);
    out[0] = creal(m);
    out[1] = cimag(m);
}

void heget_oracle_amp_ld(const double *mom, int n, const int *nhel, double g, int gauge_idx, double *out)
{
    long double lm[40];
    for (int i = 0; i < 4 * (n + 2); ++i) lm[i] = (long double)mom[i];
    const long double _Complex m = amp_one_helicity_ld(lm, n, nhel, (long double)g, gauge_idx);
    out[0] = (double)creall(m);
    out[1] = (double)cimagl(m);
}

/* Sum over all 4*2^n helicity assignments of |ampsum|^2 for each of N events
 * (the sum in eq. 2; no flux, average, colour or 1/n! factor).
 * Events (and, when there are few events, helicity assignments) are spread over
 * OpenMP threads; each event's sum runs in fixed helicity order, so the result does
 * not depend on the thread count. */
#define DEFINE_AMP2(SFX_, REAL_, CREAL_, CIMAG_)                                                   \
    void heget_oracle_amp2##SFX_(const double *momenta, int n, int64_t N, double g, double *out)  \
    {                                                                                              \
        const int np = n + 2, ncfg = 1 << (n + 2);                                                 \
        int nthreads = heget_oracle_num_threads();                                                 \
        if (N >= 4 * (int64_t)nthreads) {                                                          \
            _Pragma("omp parallel for schedule(dynamic, 1)")                                       \
            for (int64_t e = 0; e < N; ++e) {                                                      \
                REAL_ lm[40];                                                                      \
                for (int i = 0; i < 4 * np; ++i) lm[i] = (REAL_)momenta[e * 4 * np + i];           \
                out[e] = (double)amp2_event##SFX_(lm, n, (REAL_)g);                                \
            }                                                                                      \
        } else {                                                                                   \
            REAL_ *part = (REAL_ *)malloc(sizeof(REAL_) * (size_t)N * ncfg);                       \
            _Pragma("omp parallel for collapse(2) schedule(dynamic, 1)")                           \
            for (int64_t e = 0; e < N; ++e)                                                        \
                for (int h = 0; h < ncfg; ++h) {                                                   \
                    REAL_ lm[40];                                                                  \
                    int nhel[10];                                                                  \
                    for (int i = 0; i < 4 * np; ++i) lm[i] = (REAL_)momenta[e * 4 * np + i];       \
                    for (int b = 0; b < np; ++b) nhel[b] = ((h >> b) & 1) ? +1 : -1;               \
                    const REAL_ _Complex m = amp_one_helicity##SFX_(lm, n, nhel, (REAL_)g, -1);    \
                    part[e * ncfg + h] = CREAL_(m) * CREAL_(m) + CIMAG_(m) * CIMAG_(m);            \
                }                                                                                  \
            for (int64_t e = 0; e < N; ++e) {                                                      \
                REAL_ total = 0;                                                                   \
                for (int h = 0; h < ncfg; ++h) total += part[e * ncfg + h];                        \
                out[e] = (double)total;                                                            \
            }                                                                                      \
            free(part);                                                                            \
        }                                                                                          \
    }

DEFINE_AMP2(_d, double, creal, cimag)
DEFINE_AMP2(_ld, long double, creall, cimagl)

/* ---- hooks for the pin tests (tests/test_oracle_pins.py) ------------------ */

/* gamma^mu as 16 (re,im) pairs, row-major. */
void heget_oracle_gamma(int mu, double *out32)
{
    double _Complex G[4][4];
    gamma_mu_d(mu, G);
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) {
            out32[2 * (4 * r + c)] = creal(G[r][c]);
            out32[2 * (4 * r + c) + 1] = cimag(G[r][c]);
        }
}

/* which: 0 = ixxxx0, 1 = oxxxx0, 2 = vxxxx0 (ns = nSF or nSV); out8 = 4 (re,im) pairs. */
void heget_oracle_wavefunction(int which, const double *p, int nhel, int ns, double *out8)
{
    double _Complex w[4];
    if (which == 0) ixxxx0_d(p, nhel, ns, w);
    else if (which == 1) oxxxx0_d(p, nhel, ns, w);
    else vxxxx0_d(p, nhel, ns, w);
    for (int a = 0; a < 4; ++a) {
        out8[2 * a] = creal(w[a]);
        out8[2 * a + 1] = cimag(w[a]);
    }
}

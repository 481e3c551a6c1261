/* oracle/heget_oracle_next1.c -- TEST INFRASTRUCTURE, not product code.
 *
 * Oracle for the paper's own event loop: one random helicity
 * assignment per event instead of the explicit helicity sum ("generate helicities and
 * momenta ... using random numbers, and compute squared amplitudes", step 4 of
 * PAPER.md:116-122), and the kinematical distributions of Fig. 2:
 * the maximum transverse momentum and the Delta R separation (eq. 10) of the
 * final-state photons, as weighted histograms.
 *
 * Readings (R21-R23; the paper gives neither the random-number layout nor the
 * binning):
 *   R21 helicity draw: Philox4x32-10, key = seed, counter = (event_lo, event_hi, 15, 0);
 *       bit b of the first output word is the helicity of particle b in the order
 *       u, ubar, gamma_1..gamma_n (1 -> +1, 0 -> -1);
 *   R22 estimator: 4 * 2^n * |M(h)|^2, whose mean over h is the helicity sum of eq. (2);
 *   R23 histograms: nbins equal bins on [lo, hi); bin = floor((x - lo) / (hi - lo) * nbins)
 *       computed in fp64; x < lo -> underflow, x >= hi or NaN -> overflow; entries are
 *       added with the event's value (weight * amplitude); observables: 0 = max_i pT_i,
 *       1 = min_{i<j} Delta R_ij, 2 = every Delta R_ij (n(n-1)/2 entries per event).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA path.
 */
#include <math.h>
#include <stdint.h>

void heget_oracle_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]);
void heget_oracle_amp_d(const double *mom, int n, const int *nhel, double g, int gauge_idx, double *out);
void heget_oracle_amp_ld(const double *mom, int n, const int *nhel, double g, int gauge_idx, double *out);

#define HELICITY_SLOT 15u

/* R21: the n+2 helicity bits of one event. */
uint32_t heget_oracle_helicity_bits(uint64_t seed, uint64_t event, int n)
{
    const uint32_t ctr[4] = {(uint32_t)event, (uint32_t)(event >> 32), HELICITY_SLOT, 0u};
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t x[4];
    heget_oracle_philox4x32_10(ctr, key, x);
    return x[0] & ((1u << (n + 2)) - 1u);
}

/* R22: out[e] = 4 * 2^n * |ampsum(h_e)|^2, hel[e] = the bits used.  extended != 0 evaluates
 * the amplitude in long double. */
void heget_oracle_amp2_sampled(uint64_t seed, uint64_t first_event, const double *momenta, int n,
                               int64_t N, double g, int extended, double *out, int32_t *hel)
{
    const int np = n + 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t e = 0; e < N; ++e) {
        const uint32_t bits = heget_oracle_helicity_bits(seed, first_event + (uint64_t)e, n);
        int nhel[10];
        for (int b = 0; b < np; ++b) nhel[b] = ((bits >> b) & 1u) ? +1 : -1;
        double m[2];
        if (extended)
            heget_oracle_amp_ld(momenta + e * 4 * np, n, nhel, g, -1, m);
        else
            heget_oracle_amp_d(momenta + e * 4 * np, n, nhel, g, -1, m);
        out[e] = (double)(4 << n) * (m[0] * m[0] + m[1] * m[1]);
        hel[e] = (int32_t)bits;
    }
}

static double photon_pt(const double *k) { return sqrt(k[1] * k[1] + k[2] * k[2]); }

/* eq. (10), with eta = asinh(pz / pT) (massless photons, R8) and
 * Delta phi wrapped to [0, pi]. */
static double delta_r(const double *a, const double *b)
{
    const double pi = 3.14159265358979323846;
    const double eta_a = asinh(a[3] / photon_pt(a)), eta_b = asinh(b[3] / photon_pt(b));
    double dphi = fabs(atan2(a[2], a[1]) - atan2(b[2], b[1]));
    if (dphi > pi) dphi = 2.0 * pi - dphi;
    const double deta = eta_a - eta_b;
    return sqrt(deta * deta + dphi * dphi);
}

static void fill(double *hist, int nbins, double lo, double hi, double x, double v)
{
    /* hist[0] = underflow, hist[1..nbins] = bins, hist[nbins+1] = overflow */
    if (x < lo) {
        hist[0] += v;
    } else if (!(x < hi)) {
        hist[nbins + 1] += v;
    } else {
        int b = (int)floor((x - lo) / (hi - lo) * nbins);
        if (b >= nbins) b = nbins - 1; /* rounding at the upper edge */
        hist[1 + b] += v;
    }
}

/* R23: hist[nbins + 2], zeroed here, filled in event order. */
void heget_oracle_histogram(const double *momenta, const double *value, int n, int64_t N,
                            int observable, double lo, double hi, int nbins, double *hist)
{
    const int np = n + 2;
    for (int b = 0; b < nbins + 2; ++b) hist[b] = 0.0;
    for (int64_t e = 0; e < N; ++e) {
        const double *k = momenta + e * 4 * np + 8; /* photons */
        const double v = value[e];
        if (v == 0.0) continue; /* events that failed the cuts carry no weight */
        if (observable == 0) {
            double best = 0.0;
            for (int i = 0; i < n; ++i) {
                const double pt = photon_pt(k + 4 * i);
                if (pt > best) best = pt;
            }
            fill(hist, nbins, lo, hi, best, v);
        } else {
            double best = INFINITY;
            for (int i = 0; i < n; ++i)
                for (int j = i + 1; j < n; ++j) {
                    const double dr = delta_r(k + 4 * i, k + 4 * j);
                    if (observable == 2) fill(hist, nbins, lo, hi, dr, v);
                    if (dr < best) best = dr;
                }
            if (observable == 1) fill(hist, nbins, lo, hi, best, v);
        }
    }
}

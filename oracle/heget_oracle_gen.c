/* oracle/heget_oracle_gen.c -- TEST INFRASTRUCTURE, not product code.
 *
 * CPU oracle for the event generation step of arXiv 0908.4403: "if the program is
 * given a set of random numbers, it generates a phase space point and computes a
 * Jacobian" (step 4 at PAPER.md:121), the final-state cuts of eq. (9)
 * and the per-event weight built from eqs. (1)-(4),
 * plus the sum of step 6.
 *
 * The paper names neither the random number generator nor the phase-space algorithm
 * (readings R6, R7); BASELINE.json fixes them as Philox4x32-10 and RAMBO.
 * Both are restated here from their published definitions (Salmon et al., SC'11;
 * Kleiss, Stirling, Ellis, CPC 40 (1986) 359) step by step.  The CUDA path has its
 * own, separately written implementation; the two share no code.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this library.
 */
#include <math.h>
#include <stdint.h>

/* ---- Philox4x32-10 ------------------------------------------------------- */

static void mulhilo32(uint32_t a, uint32_t b, uint32_t *hi, uint32_t *lo)
{
    const uint64_t p = (uint64_t)a * (uint64_t)b;
    *hi = (uint32_t)(p >> 32);
    *lo = (uint32_t)p;
}

/* ctr[4], key[2] -> out[4]; ten rounds, the key bumped by the Weyl constants
 * between rounds. */
void heget_oracle_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4])
{
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        uint32_t hi0, lo0, hi1, lo1;
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        mulhilo32(0xD2511F53u, c0, &hi0, &lo0);
        mulhilo32(0xCD9E8D57u, c2, &hi1, &lo1);
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Four uniforms in (0,1) for (seed, global event index, slot): key = (seed_lo,
 * seed_hi), counter = (event_lo, event_hi, slot, 0); u = (x + 0.5) * 2^-32.
 * slot 0: event-level numbers (u_a, u_b, unused, unused); slot j = 1..n: photon j. */
void heget_oracle_uniforms(uint64_t seed, uint64_t event, uint32_t slot, double u[4])
{
    uint32_t ctr[4] = {(uint32_t)event, (uint32_t)(event >> 32), slot, 0u};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t x[4];
    heget_oracle_philox4x32_10(ctr, key, x);
    for (int i = 0; i < 4; ++i) u[i] = ((double)x[i] + 0.5) * (1.0 / 4294967296.0);
}

/* ---- n-body massless phase space volume ---------------------------------- */

/* Integral of eq. (4) for massless particles at invariant mass^2 = s:
 * Phi_n(s) = (2 pi)^(4-3n) (pi/2)^(n-1) s^(n-2) / ((n-1)! (n-2)!).  RAMBO's weight
 * is this constant for every event. */
double heget_oracle_phase_space_volume(int n, double s)
{
    const double pi = 3.14159265358979323846;
    double fact1 = 1.0, fact2 = 1.0;
    for (int i = 2; i <= n - 1; ++i) fact1 *= (double)i;
    for (int i = 2; i <= n - 2; ++i) fact2 *= (double)i;
    return pow(2.0 * pi, 4.0 - 3.0 * n) * pow(pi / 2.0, n - 1.0) * pow(s, n - 2.0) / (fact1 * fact2);
}

/* ---- RAMBO --------------------------------------------------------------- */

/* n massless momenta k[n][4] = (E,px,py,pz) in the rest frame of total mass w,
 * from 4n uniforms u[n][4].  Step 1: isotropic massless q_i with energy
 * distribution q0 exp(-q0).  Step 2: conformal boost + rescale so that sum k = (w,0). */
static void rambo(int n, double w, const double u[][4], double k[][4])
{
    const double twopi = 6.28318530717958647692;
    double q[8][4], Q[4] = {0, 0, 0, 0};
    for (int i = 0; i < n; ++i) {
        const double c = 2.0 * u[i][0] - 1.0;
        const double s = sqrt(1.0 - c * c);
        const double f = twopi * u[i][1];
        const double q0 = -log(u[i][2] * u[i][3]);
        q[i][0] = q0;
        q[i][1] = q0 * s * cos(f);
        q[i][2] = q0 * s * sin(f);
        q[i][3] = q0 * c;
        for (int mu = 0; mu < 4; ++mu) Q[mu] += q[i][mu];
    }
    const double M = sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
    const double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
    const double gam = Q[0] / M;
    const double a = 1.0 / (1.0 + gam);
    const double x = w / M;
    for (int i = 0; i < n; ++i) {
        const double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
        k[i][0] = x * (gam * q[i][0] + bq);
        for (int j = 0; j < 3; ++j) k[i][1 + j] = x * (q[i][1 + j] + b[j] * q[i][0] + a * bq * b[j]);
    }
}

/* ---- cuts, eq. (9) -------------------------------------------------------- */

/* 1 if every photon has pT > pt_cut, |eta| < eta_cut and every pair has
 * Delta R > dr_cut (strict inequalities; eta = rapidity = pseudorapidity for a
 * massless photon; Delta R of eq. 10, with Delta phi
 * wrapped into [0, pi]); reading R8. */
static int passes_cuts(int n, const double k[][4], double pt_cut, double eta_cut, double dr_cut)
{
    const double pi = 3.14159265358979323846;
    double eta[8], phi[8];
    for (int i = 0; i < n; ++i) {
        const double pt = sqrt(k[i][1] * k[i][1] + k[i][2] * k[i][2]);
        if (!(pt > pt_cut)) return 0;
        eta[i] = asinh(k[i][3] / pt);
        if (!(fabs(eta[i]) < eta_cut)) return 0;
        phi[i] = atan2(k[i][2], k[i][1]);
    }
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j) {
            const double deta = eta[i] - eta[j];
            double dphi = fabs(phi[i] - phi[j]);
            if (dphi > pi) dphi = 2.0 * pi - dphi;
            const double dr = sqrt(deta * deta + dphi * dphi);
            if (!(dr > dr_cut)) return 0;
        }
    return 1;
}

/* ---- event generation ----------------------------------------------------- */

/* mode 0: sqrt_s_hat = a fixed, y = 0 (the north-star heget_rambo form);
 * mode 1: sqrt_s_hat = a (b/a)^u_a log-uniform in [a,b], y = y_max (2 u_b - 1);
 * mode 2: toy parton densities at collider energy sqrt_s = a: tau = x1 x2
 *         log-uniform in [tau_min, 1], tau_min = (n pt_cut)^2 / s,
 *         y uniform in [ln(tau)/2, -ln(tau)/2], x1,2 = sqrt(tau) exp(+-y),
 *         s_hat = tau s (eq. 3); Jacobian tau ln(1/tau_min) ln(1/tau);
 *         parton luminosity 2 f(x1) f(x2), f(x) = x^-0.5 (1-x)^3 (eq. 1, PAPER.md:33,
 *         both terms equal for one common toy density; reading R16).
 * Every event: RAMBO in the u ubar rest frame, boost by y along z,
 *   p1 = (sqrt_s_hat/2) e^y (1,0,0,1), p2 = (sqrt_s_hat/2) e^-y (1,0,0,-1),
 *   weight = [cuts] * Phi_n(s_hat) / (2 s_hat) * (mode 2: Jacobian * luminosity).
 * The spin/colour average and 1/n! of eq. (2) are applied by the reduction.
 * momenta: [N][n+2][4]; weight: [N]; event index = first_event + local index. */
void heget_oracle_gen_events(uint64_t seed, int n, int mode, double a, double b, double y_max,
                             int apply_cuts, double pt_cut, double eta_cut, double dr_cut,
                             uint64_t first_event, int64_t N, double *momenta, double *weight)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        const uint64_t ev = first_event + (uint64_t)e;
        double u0[4], u[8][4], k[8][4];
        heget_oracle_uniforms(seed, ev, 0u, u0);
        for (int i = 0; i < n; ++i) heget_oracle_uniforms(seed, ev, (uint32_t)(i + 1), u[i]);
        double rs, y, extra = 1.0;
        if (mode == 0) {
            rs = a;
            y = 0.0;
        } else if (mode == 1) {
            rs = a * pow(b / a, u0[0]);
            y = y_max * (2.0 * u0[1] - 1.0);
        } else {
            const double s = a * a;
            const double tau_min = (n * pt_cut) * (n * pt_cut) / s;
            const double ln_tau_min = log(tau_min);
            const double ln_tau = (1.0 - u0[0]) * ln_tau_min;
            const double tau = exp(ln_tau);
            y = (2.0 * u0[1] - 1.0) * (-0.5 * ln_tau);
            const double x1 = sqrt(tau) * exp(y), x2 = sqrt(tau) * exp(-y);
            const double f1 = pow(1.0 - x1, 3.0) / sqrt(x1), f2 = pow(1.0 - x2, 3.0) / sqrt(x2);
            rs = sqrt(tau * s);
            extra = tau * (-ln_tau_min) * (-ln_tau) * 2.0 * f1 * f2;
        }
        rambo(n, rs, (const double(*)[4])u, k);
        const double ch = cosh(y), sh = sinh(y);
        double *out = momenta + e * 4 * (n + 2);
        const double e1 = 0.5 * rs * exp(y), e2 = 0.5 * rs * exp(-y);
        out[0] = e1; out[1] = 0.0; out[2] = 0.0; out[3] = e1;
        out[4] = e2; out[5] = 0.0; out[6] = 0.0; out[7] = -e2;
        for (int i = 0; i < n; ++i) {
            const double E = k[i][0] * ch + k[i][3] * sh;
            const double pz = k[i][3] * ch + k[i][0] * sh;
            k[i][0] = E;
            k[i][3] = pz;
            for (int mu = 0; mu < 4; ++mu) out[4 * (2 + i) + mu] = k[i][mu];
        }
        const double shat = rs * rs;
        double w = heget_oracle_phase_space_volume(n, shat) / (2.0 * shat) * extra;
        if (apply_cuts && !passes_cuts(n, (const double(*)[4])k, pt_cut, eta_cut, dr_cut)) w = 0.0;
        weight[e] = w;
    }
}

/* Step 6: out3 = { sum x, sum x^2, #(weight != 0) } with
 * x = weight * amp2 * (1/4)(1/9)(1/n!) -- the helicity average 1/2^2, the colour
 * factor and the identical-photon factor of eq. (2) (the colour factor
 * is garbled there, reading R1).  Plain sequential sums in long double. */
void heget_oracle_xsec_reduce(const double *amp2, const double *weight, int64_t N, int n, double *out3)
{
    double nfact = 1.0;
    for (int i = 2; i <= n; ++i) nfact *= (double)i;
    const long double cf = (long double)(1.0 / 4.0) * (1.0L / 9.0L) / (long double)nfact;
    long double s1 = 0, s2 = 0;
    int64_t cnt = 0;
    for (int64_t e = 0; e < N; ++e) {
        /* weight 0 = the event failed the cuts of eq. (9) and is not part of the
         * integral: it contributes 0 whatever amp2 holds (reading R26) */
        if (weight[e] == 0.0) continue;
        const long double x = (long double)weight[e] * (long double)amp2[e] * cf;
        s1 += x;
        s2 += x * x;
        ++cnt;
    }
    out3[0] = (double)s1;
    out3[1] = (double)s2;
    out3[2] = (double)cnt;
}

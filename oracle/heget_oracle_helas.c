/* oracle/heget_oracle_helas.c -- TEST INFRASTRUCTURE, not product code.
 *
 * Oracle for the full HEGET function set of Tables 3 and 4 (SURVEY 8(f)
 * NEXT-4) in the paper's own data layout: a wavefunction is cmplx w[6], components 0..3 the
 * 4-spinor or 4-vector, w[4] = (p0, p3) * nS and w[5] = (p1, p2) * nS as complex numbers
 * ("flowing" momentum).  Everything is evaluated with explicit 4x4 gamma
 * matrices (amp_body.inc), one matrix-vector product per slash, as in heget_oracle.c.
 *
 * Definitions (the bodies of Lists 3-8, 11-15 are missing from PAPER.md; R3, R24):
 *   ixxxx0/oxxxx0/vxxxx0  eqs. (11)-(15), generic direction (amp_body.inc);
 *   ixxxx1, oxxxx1, vxxxx1  the same for p along +z, ixxxx2, oxxxx2, vxxxx2 for p along -z
 *                         (PAPER.md:203-205); here they ARE the generic formula evaluated at
 *                         (|p|,0,0,+-|p|), whose pT = 0 branches carry the HELAS conventions and,
 *                         for nSV = -1, reproduce Lists 9/10;
 *   iovxxx(fi,fo,vc)      g <fo| vc-slash |fi>
 *   fvixx0(fi,vc)         -g pf-slash vc-slash |fi> / pf^2, pf = p_fi - p_vc
 *   fvoxx0(fo,vc)         -g <fo| vc-slash pf-slash / pf^2, pf = p_fo + p_vc
 *   jioxx0(fi,fo)         g <fo| gamma^mu |fi> / q^2, q = p_fo - p_fi, Feynman gauge
 *
 * with gal[0] = gal[1] = g (eq. 26).  The signs of the two propagators follow from
 * HELAS leaving out one factor i per vertex and per propagator: i(p-slash)/p^2 between two
 * vertices gives -1, -i g_{mu nu}/q^2 gives +1.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code with the CUDA path.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>

#define REAL double
#define SFX _h
#define SQRT sqrt
#define CREAL creal
#define CIMAG cimag
#include "amp_body.inc"

typedef double _Complex cplx;

static void unpack(const double *w12, cplx w[6])
{
    for (int a = 0; a < 6; ++a) w[a] = w12[2 * a] + I * w12[2 * a + 1];
}

static void pack(const cplx w[6], double *w12)
{
    for (int a = 0; a < 6; ++a) {
        w12[2 * a] = creal(w[a]);
        w12[2 * a + 1] = cimag(w[a]);
    }
}

/* flowing momentum stored in w[4], w[5] */
static void momentum_of(const cplx w[6], double p[4])
{
    p[0] = creal(w[4]);
    p[3] = cimag(w[4]);
    p[1] = creal(w[5]);
    p[2] = cimag(w[5]);
}

/* fn: 0,1,2 = ixxxx0,1,2; 3,4,5 = oxxxx0,1,2; 6,7,8 = vxxxx0,1,2.  For the "1" / "2" forms only
 * |p| = p[0] is used and the direction is +z / -z by definition. */
void heget_oracle_helas_wavefunction(int fn, const double *p_in, int nhel, int ns, double *w12)
{
    double p[4] = {p_in[0], p_in[1], p_in[2], p_in[3]};
    const int kind = fn / 3, dir = fn % 3;
    if (dir == 1) { p[1] = 0; p[2] = 0; p[3] = p[0]; }
    if (dir == 2) { p[1] = 0; p[2] = 0; p[3] = -p[0]; }
    cplx w[6];
    if (kind == 0) ixxxx0_h(p, nhel, ns, w);
    else if (kind == 1) oxxxx0_h(p, nhel, ns, w);
    else vxxxx0_h(p, nhel, ns, w);
    w[4] = (p[0] + I * p[3]) * (double)ns;
    w[5] = (p[1] + I * p[2]) * (double)ns;
    pack(w, w12);
}

/* fn: 0 = iovxxx(a=fi, b=fo, c=vc) -> out12[0..1] = amplitude, rest 0
 *     1 = fvixx0(a=fi, c=vc) -> fvi[6];  2 = fvoxx0(b=fo, c=vc) -> fvo[6]
 *     3 = jioxx0(a=fi, b=fo) -> jio[6] */
void heget_oracle_helas_vertex(int fn, const double *a12, const double *b12, const double *c12, double g,
                               double *out12)
{
    cplx fi[6], fo[6], vc[6], out[6] = {0, 0, 0, 0, 0, 0};
    cplx V[4][4], P[4][4], tmp[4];
    double pf[4];
    if (a12) unpack(a12, fi);
    if (b12) unpack(b12, fo);
    if (c12) unpack(c12, vc);
    if (fn == 0) {
        slash_h(vc, V);
        out[0] = iovxxx_h(fi, fo, V, g);
    } else if (fn == 1) {
        out[4] = fi[4] - vc[4];
        out[5] = fi[5] - vc[5];
        momentum_of(out, pf);
        const double pf2 = pf[0] * pf[0] - pf[1] * pf[1] - pf[2] * pf[2] - pf[3] * pf[3];
        slash_h(vc, V);
        slash_real_h(pf, P);
        matvec_h(V, fi, tmp);
        matvec_h(P, tmp, out);
        for (int k = 0; k < 4; ++k) out[k] *= -g / pf2;
    } else if (fn == 2) {
        out[4] = fo[4] + vc[4];
        out[5] = fo[5] + vc[5];
        momentum_of(out, pf);
        const double pf2 = pf[0] * pf[0] - pf[1] * pf[1] - pf[2] * pf[2] - pf[3] * pf[3];
        slash_h(vc, V);
        slash_real_h(pf, P);
        /* row vector times matrices: (fo V) P */
        for (int c = 0; c < 4; ++c) {
            tmp[c] = 0;
            for (int r = 0; r < 4; ++r) tmp[c] += fo[r] * V[r][c];
        }
        for (int c = 0; c < 4; ++c) {
            out[c] = 0;
            for (int r = 0; r < 4; ++r) out[c] += tmp[r] * P[r][c];
            out[c] *= -g / pf2;
        }
    } else {
        out[4] = fo[4] - fi[4];
        out[5] = fo[5] - fi[5];
        momentum_of(out, pf);
        const double q2 = pf[0] * pf[0] - pf[1] * pf[1] - pf[2] * pf[2] - pf[3] * pf[3];
        for (int mu = 0; mu < 4; ++mu) {
            cplx G[4][4];
            gamma_mu_h(mu, G);
            matvec_h(G, fi, tmp);
            cplx acc = 0;
            for (int r = 0; r < 4; ++r) acc += fo[r] * tmp[r];
            out[mu] = g * acc / q2;
        }
    }
    pack(out, out12);
}

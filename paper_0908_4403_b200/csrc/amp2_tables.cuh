// amp2_tables.cuh -- per-event tables of the amplitude kernel (product code).
//
// Two-component (Weyl) form of the HELAS objects for a massless quark line, chiral
// representation with components (0,1) left- and (2,3) right-handed (eq. 16):
//   a-slash = [[0, a0 - a.sigma], [a0 + a.sigma, 0]].
// For sigma_1 = +1 the u spinor (ixxxx1) is (0,0,sqrt(2E1),0); the photon
// vertex maps (2,3) -> (0,1) through the upper-right block of eps-slash and the propagator
// maps (0,1) -> (2,3) through the lower-left block of (p1-K)-slash, so the whole fvixx0
// chain lives in two complex components.  The paper keeps 4-spinors
// (the gain "never exceeds a factor of two"); here that factor is taken.
//
// E table, per photon i and helicity lambda (vxxxx0, eqs. 13-15, nSV=+1),
// upper-right block of eps-slash times sqrt(2):
//     lambda=+1: [[-s, -B], [A, s]],  s = pT/w, A = (1+c) e^{i phi}, B = (1-c) e^{-i phi}
//     lambda=-1: same form with s -> -s, A -> conj(B), B -> conj(A)   (eps(-l) = -eps(l)^*)
// P table, per non-empty proper subset S of photons (eq. 8), lower-left block of
// (p1 - K_S)-slash times the propagator factor -g/t_S of fvixx0:
//     (-g/t_S) * [[p+, px - i py], [px + i py, p-]],  p+- = p0 +- p3 of p1 - K_S.
#pragma once
#include "dd.cuh"

template <typename T>
struct alignas(16) EEntry {
    T s, ar, ai, br;
    T bi, pad0, pad1, pad2;
};

template <typename T>
struct alignas(16) PEntry {
    T pp, pm, px, py;
};

// Photon i's two E entries from its four-momentum k = (w, kx, ky, kz), in fp64.
template <typename T>
__device__ __forceinline__ void make_photon_entries(const double* k, EEntry<T>* e_plus, EEntry<T>* e_minus)
{
    const double w = k[0], kx = k[1], ky = k[2], kz = k[3];
    const double pt = sqrt(kx * kx + ky * ky);
    const double inv_w = 1.0 / w, inv_pt = 1.0 / pt;
    const double opc = (w + kz) * inv_w;  // 1 + cos(theta)
    const double omc = (w - kz) * inv_w;  // 1 - cos(theta): one rounded subtraction, no 1 - c
    const double s = pt * inv_w;
    const double cf = kx * inv_pt, sf = ky * inv_pt;
    const double ar = opc * cf, ai = opc * sf;   // A = (1+c) e^{+i phi}
    const double br = omc * cf, bi = -omc * sf;  // B = (1-c) e^{-i phi}
    e_plus->s = (T)s;   e_plus->ar = (T)ar;  e_plus->ai = (T)ai;   e_plus->br = (T)br;  e_plus->bi = (T)bi;
    e_minus->s = (T)-s; e_minus->ar = (T)br; e_minus->ai = (T)-bi; e_minus->br = (T)ar; e_minus->bi = (T)-ai;
}

// P entry of subset S (bit i set = photon i attached).  mom: the event's (n+2) four-vectors.
// Accumulated in double-double and rounded once; `scale` multiplies the entry (sqrt(s_hat)
// for the fp32 kernel, which works in units of sqrt(s_hat); 1 for fp64).
template <int N, typename T>
__device__ __forceinline__ void make_subset_entry(const double* mom, unsigned S, double g, double scale,
                                                  PEntry<T>* out)
{
    const double e1 = mom[0];
    dd pe = {e1, 0.0}, pz = {mom[3], 0.0}, px = {mom[1], 0.0}, py = {mom[2], 0.0};
#pragma unroll
    for (int i = 0; i < N; ++i) {
        if ((S >> i) & 1u) {
            const double* k = mom + 4 * (2 + i);
            pe = dd_add_d(pe, -k[0]);
            px = dd_add_d(px, -k[1]);
            py = dd_add_d(py, -k[2]);
            pz = dd_add_d(pz, -k[3]);
        }
    }
    const dd pp = dd_add(pe, pz);
    const dd pm = dd_add(pe, dd_neg(pz));
    dd t = dd_mul(pp, pm);
    t = dd_add(t, dd_neg(dd_mul(px, px)));
    t = dd_add(t, dd_neg(dd_mul(py, py)));
    const double c = -g / dd_to_double(t) * scale;
    out->pp = (T)(c * dd_to_double(pp));
    out->pm = (T)(c * dd_to_double(pm));
    out->px = (T)(c * dd_to_double(px));
    out->py = (T)(c * dd_to_double(py));
}

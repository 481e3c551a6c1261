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
// E table, per photon i and helicity lambda (vxxxx0, eqs. 13-15, nSV=+1):
// the upper-right block of eps-slash times sqrt(2) is, with s = pT/w = sin(theta),
//     lambda=+1: [[-s, -B], [A, s]],  A = (1+c) e^{i phi}, B = (1-c) e^{-i phi}
//     lambda=-1: same form with s -> -s, A -> conj(B), B -> conj(A)   (eps(-l) = -eps(l)^*)
// Every diagram of a helicity configuration contains each photon exactly once, so a factor
// common to all four elements of photon i's block is a factor of ampsum.  The table stores
// the block divided by +s (lambda=+1) or -s (lambda=-1),
//     E' = [[-1, -b], [a, 1]],   a = A/s, b = B/s   (lambda=-1: a = -conj(B)/s, b = -conj(A)/s)
// i.e. four reals per entry and no multiplications by s in the tree; |ampsum|^2 is multiplied
// by prod_i s_i^2 (helicity independent) once per event, in fp64.
// P table, per non-empty proper subset S of photons (eq. 8), lower-left block of
// (p1 - K_S)-slash times the propagator factor -g/t_S of fvixx0:
//     (-g/t_S) * [[p+, px - i py], [px + i py, p-]],  p+- = p0 +- p3 of p1 - K_S.
#pragma once
#include "dd.cuh"

template <typename T>
struct alignas(16) EEntry {
    T ar, ai, br, bi;
};

template <typename T>
struct alignas(16) PEntry {
    T pp, pm, px, py;
};

// 1/x for a normal, finite double: hardware approximation (>= 20 bits) and two Newton steps,
// without the slow path of the IEEE division (the tables never see 0, inf or subnormals for
// inputs that satisfy the preconditions of include/heget.h).  Relative error ~1 ulp.
__device__ __forceinline__ double fast_rcp(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(r, fma(-x, r, 1.0), r);
    r = fma(r, fma(-x, r, 1.0), r);
    return r;
}

// Photon i's two E' entries from its four-momentum k = (w, kx, ky, kz), in fp64.
// Returns s^2 = (pT/w)^2, the factor taken out of |ampsum|^2.
template <typename T>
__device__ __forceinline__ double make_photon_entries(const double* k, EEntry<T>* e_plus, EEntry<T>* e_minus)
{
    const double w = k[0], kx = k[1], ky = k[2], kz = k[3];
    const double pt2 = kx * kx + ky * ky;
    const double w2 = w * w;
    const double r = fast_rcp(pt2 * w2);  // one reciprocal serves 1/pT^2 and pT^2/w^2
    const double inv_pt2 = r * w2;
    const double ca = (w + kz) * inv_pt2;  // (1+c)/s / pT
    const double cb = (w - kz) * inv_pt2;  // (1-c)/s / pT: one rounded subtraction, no 1 - c
    const double ar = ca * kx, ai = ca * ky;    // a = (1+c)/s e^{+i phi}
    const double br = cb * kx, bi = -cb * ky;   // b = (1-c)/s e^{-i phi}
    e_plus->ar = (T)ar;   e_plus->ai = (T)ai;  e_plus->br = (T)br;   e_plus->bi = (T)bi;
    e_minus->ar = (T)-br; e_minus->ai = (T)bi; e_minus->br = (T)-ar; e_minus->bi = (T)ai;
    return pt2 * pt2 * r;
}

// P entry of subset S for the fp32 kernel, in plain fp64 and rounded to fp32 once: light-cone
// components k+- = w +- kz of each photon (one rounded operation each), p+ = 2 E1 - sum k+,
// p- = -sum k-, t_S = p+ p- - px^2 - py^2 (both terms <= 0, no cancellation between them).
// Error ~1e-13 relative on cut-passing events, far below fp32's 6e-8.
template <int N>
__device__ __forceinline__ void make_subset_entry_plain(const double* mom, unsigned S, double g, double scale,
                                                        PEntry<float>* out)
{
    double kp = 0.0, km = 0.0, kx = 0.0, ky = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        if ((S >> i) & 1u) {
            const double* k = mom + 4 * (2 + i);
            kp += k[0] + k[3];
            km += k[0] - k[3];
            kx += k[1];
            ky += k[2];
        }
    }
    const double pp = 2.0 * mom[0] - kp;
    const double t = -fma(pp, km, fma(kx, kx, ky * ky));
    const double c = -g * scale * fast_rcp(t);
    out->pp = (float)(c * pp);
    out->pm = (float)(-c * km);
    out->px = (float)(-c * kx);
    out->py = (float)(-c * ky);
}

// P entry of subset S (bit i set = photon i attached).  mom: the event's (n+2) four-vectors.
// Accumulated in double-double and rounded once; `scale` multiplies the entry (sqrt(s_hat)
// for the fp32 kernel, which works in units of sqrt(s_hat); 1 for fp64).
template <int N, typename T>
__device__ __forceinline__ void make_subset_entry(const double* mom, unsigned S, double g, double scale,
                                                  PEntry<T>* out)
{
    // p1 = (E1, 0, 0, E1) (precondition of include/heget.h): the transverse sums start from the
    // first member exactly, the others from p1.  A proper subset has 1..N-1 members: one
    // unconditional round and N-2 rounds over "the next member of S" instead of N rounds over all
    // photons (lanes with fewer members idle in the last rounds).
    unsigned rem = S;
    const double* k0 = mom + 4 * (2 + (__ffs(rem) - 1));
    rem &= rem - 1u;
    dd pe = {mom[0], 0.0}, pz = {mom[3], 0.0}, px = {-k0[1], 0.0}, py = {-k0[2], 0.0};
    dd_acc(pe, -k0[0]);
    dd_acc(pz, -k0[3]);
#pragma unroll
    for (int j = 1; j < N - 1; ++j) {
        if (rem) {
            const double* k = mom + 4 * (2 + (__ffs(rem) - 1));
            rem &= rem - 1u;
            dd_acc(pe, -k[0]);
            dd_acc(px, -k[1]);
            dd_acc(py, -k[2]);
            dd_acc(pz, -k[3]);
        }
    }
    // p+- = pe +- pz: high parts by TwoSum, low parts added
    dd pp = dd_two_sum(pe.hi, pz.hi), pm = dd_two_sum(pe.hi, -pz.hi);
    pp.lo = __dadd_rn(pp.lo, __dadd_rn(pe.lo, pz.lo));
    pm.lo = __dadd_rn(pm.lo, __dsub_rn(pe.lo, pz.lo));
    // t = p+ p- - px^2 - py^2: exact products of the high parts, first-order low parts
    dd a = dd_two_prod(pp.hi, pm.hi), bx = dd_two_prod(px.hi, px.hi), by = dd_two_prod(py.hi, py.hi);
    a.lo = __fma_rn(pp.hi, pm.lo, __fma_rn(pp.lo, pm.hi, a.lo));
    bx.lo = __fma_rn(2.0 * px.hi, px.lo, bx.lo);
    by.lo = __fma_rn(2.0 * py.hi, py.lo, by.lo);
    const dd s1 = dd_two_sum(a.hi, -bx.hi), s2 = dd_two_sum(s1.hi, -by.hi);
    const dd t = {s2.hi, __dadd_rn(__dadd_rn(s2.lo, s1.lo), __dsub_rn(__dsub_rn(a.lo, bx.lo), by.lo))};
    const double c = -g * scale * fast_rcp(dd_to_double(t));
    out->pp = (T)(c * dd_to_double(pp));
    out->pm = (T)(c * dd_to_double(pm));
    out->px = (T)(c * dd_to_double(px));
    out->py = (T)(c * dd_to_double(py));
}

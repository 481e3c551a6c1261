// helas.cuh -- the HEGET function set of Tables 3 and 4 as device functions
// in the paper's own form (product code): massless only, branch-free
// ("conditional branches ... eliminated as much as possible"), three direction
// variants per external line (0 generic, 1 = +z, 2 = -z), 4-component spinors and
// vectors in cmplx w[6] with the flowing momentum packed into w[4] = (p0, p3) nS and
// w[5] = (p1, p2) nS.  Templated on the real type: fp32 as in the paper, fp64
// as its double-precision build.
//
// The hot kernels (amp2*.cu) do NOT call these: they use the two-component reduction of the
// same objects (amp2_tables.cuh).  These are the general-purpose building blocks for other
// processes, evaluated and parity-tested through heget_helas_wavefunction / heget_helas_vertex.
//
// Conventions (the bodies of Lists 3-8, 11-15 are missing from PAPER.md; R3, R24):
// metric (+,-,-,-); chiral representation, gamma^0 = [[0,1],[1,0]], gamma^i = [[0,s^i],[-s^i,0]],
// so a-slash = [[0, a0 - a.s], [a0 + a.s, 0]] with a.s = [[a3, a1 - i a2], [a1 + i a2, -a3]];
// components 0,1 left-handed, 2,3 right-handed (eq. 16).
#pragma once

template <typename T>
struct cmplx {
    T re, im;
};

template <typename T> __device__ __forceinline__ cmplx<T> mkcmplx(T re, T im) { return {re, im}; }
template <typename T> __device__ __forceinline__ cmplx<T> operator+(cmplx<T> a, cmplx<T> b) { return {a.re + b.re, a.im + b.im}; }
template <typename T> __device__ __forceinline__ cmplx<T> operator-(cmplx<T> a, cmplx<T> b) { return {a.re - b.re, a.im - b.im}; }
template <typename T> __device__ __forceinline__ cmplx<T> operator-(cmplx<T> a) { return {-a.re, -a.im}; }
template <typename T> __device__ __forceinline__ cmplx<T> operator*(cmplx<T> a, cmplx<T> b)
{
    return {fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re)};
}
template <typename T> __device__ __forceinline__ cmplx<T> operator*(T a, cmplx<T> b) { return {a * b.re, a * b.im}; }
template <typename T> __device__ __forceinline__ cmplx<T> times_i(cmplx<T> a) { return {-a.im, a.re}; }

// ---- external fermions (Appendix B.1) ---------------------------------------
// |fi> = u(p, nHEL/2) (nSF = +1) or v(p, nHEL/2) (nSF = -1), eqs. (11a,b).
// With nh = nHEL nSF, sq = nSF sqrt(p0 + p3):  chi = (sq, (nh p1 + i p2) / sq);
// nh = +1 -> (0, 0, chi0, chi1), nh = -1 -> (chi1, chi0, 0, 0).  Precondition p0 + p3 > 0
// (use ixxxx2 on the -z axis).  The helicity selection is arithmetic, not a branch.
template <typename T>
__device__ __forceinline__ void helas_place_in(int nh, cmplx<T> chi0, cmplx<T> chi1, cmplx<T>* fi)
{
    const T up = (T)(nh == 1), dn = (T)(nh == -1);
    fi[0] = dn * chi1;
    fi[1] = dn * chi0;
    fi[2] = up * chi0;
    fi[3] = up * chi1;
}

template <typename T>
__device__ __forceinline__ void ixxxx0(const T* p, int nHEL, int nSF, cmplx<T>* fi)
{
    const int nh = nHEL * nSF;
    const T sq = (T)nSF * sqrt(p[0] + p[3]);
    const T inv = (T)1 / sq;
    helas_place_in(nh, mkcmplx(sq, (T)0), mkcmplx((T)nh * p[1] * inv, p[2] * inv), fi);
    fi[4] = mkcmplx((T)nSF * p[0], (T)nSF * p[3]);
    fi[5] = mkcmplx((T)nSF * p[1], (T)nSF * p[2]);
}

// p along +z: chi = (nSF sqrt(2 p0), 0)
template <typename T>
__device__ __forceinline__ void ixxxx1(const T* p, int nHEL, int nSF, cmplx<T>* fi)
{
    helas_place_in(nHEL * nSF, mkcmplx((T)nSF * sqrt((T)2 * p[0]), (T)0), mkcmplx((T)0, (T)0), fi);
    fi[4] = mkcmplx((T)nSF * p[0], (T)nSF * p[0]);
    fi[5] = mkcmplx((T)0, (T)0);
}

// p along -z (p0 + p3 = 0): the HELAS singular-direction value chi = (0, -nHEL sqrt(2 p0))
template <typename T>
__device__ __forceinline__ void ixxxx2(const T* p, int nHEL, int nSF, cmplx<T>* fi)
{
    helas_place_in(nHEL * nSF, mkcmplx((T)0, (T)0), mkcmplx(-(T)nHEL * sqrt((T)2 * p[0]), (T)0), fi);
    fi[4] = mkcmplx((T)nSF * p[0], -(T)nSF * p[0]);
    fi[5] = mkcmplx((T)0, (T)0);
}

// <fo| = ubar(p, nHEL/2) (nSF = +1) or vbar(p, nHEL/2) (nSF = -1), eqs. (12a,b), PAPER.md:221-225;
// chi = (sq, (nh p1 - i p2) / sq); slot pattern of the List 8 fragment:
// nh = +1 -> (chi0, chi1, 0, 0), nh = -1 -> (0, 0, chi1, chi0).
template <typename T>
__device__ __forceinline__ void helas_place_out(int nh, cmplx<T> chi0, cmplx<T> chi1, cmplx<T>* fo)
{
    const T up = (T)(nh == 1), dn = (T)(nh == -1);
    fo[0] = up * chi0;
    fo[1] = up * chi1;
    fo[2] = dn * chi1;
    fo[3] = dn * chi0;
}

template <typename T>
__device__ __forceinline__ void oxxxx0(const T* p, int nHEL, int nSF, cmplx<T>* fo)
{
    const int nh = nHEL * nSF;
    const T sq = (T)nSF * sqrt(p[0] + p[3]);
    const T inv = (T)1 / sq;
    helas_place_out(nh, mkcmplx(sq, (T)0), mkcmplx((T)nh * p[1] * inv, -p[2] * inv), fo);
    fo[4] = mkcmplx((T)nSF * p[0], (T)nSF * p[3]);
    fo[5] = mkcmplx((T)nSF * p[1], (T)nSF * p[2]);
}

template <typename T>
__device__ __forceinline__ void oxxxx1(const T* p, int nHEL, int nSF, cmplx<T>* fo)
{
    helas_place_out(nHEL * nSF, mkcmplx((T)nSF * sqrt((T)2 * p[0]), (T)0), mkcmplx((T)0, (T)0), fo);
    fo[4] = mkcmplx((T)nSF * p[0], (T)nSF * p[0]);
    fo[5] = mkcmplx((T)0, (T)0);
}

template <typename T>
__device__ __forceinline__ void oxxxx2(const T* p, int nHEL, int nSF, cmplx<T>* fo)
{
    helas_place_out(nHEL * nSF, mkcmplx((T)0, (T)0), mkcmplx(-(T)nHEL * sqrt((T)2 * p[0]), (T)0), fo);
    fo[4] = mkcmplx((T)nSF * p[0], -(T)nSF * p[0]);
    fo[5] = mkcmplx((T)0, (T)0);
}

// ---- external vector bosons (Appendix B.2) ----------------------------------
// vc = eps(p, nHEL)^* (nSV = +1, final) or eps(p, nHEL) (nSV = -1, initial), eqs. (13a,b), in the
// light-cone gauge of eqs. (14), (15): eps^0 = 0, eps.p = 0.  With pT = sqrt(p1^2 + p2^2):
//   eps^3 = nHEL pT / (|p| sqrt2),  eps^1 = -nHEL p1 p3 / (|p| pT sqrt2) - i nSV p2 / (pT sqrt2),
//   eps^2 = -nHEL p2 p3 / (|p| pT sqrt2) + i nSV p1 / (pT sqrt2).     Precondition pT > 0.
template <typename T>
__device__ __forceinline__ void vxxxx0(const T* p, int nHEL, int nSV, cmplx<T>* vc)
{
    const T rsqrt2 = (T)0.70710678118654752440;
    const T hel = (T)nHEL, sv = (T)nSV;
    const T pt = sqrt(p[1] * p[1] + p[2] * p[2]);
    const T ipt = rsqrt2 / pt, ipp = (T)1 / p[0];
    const T pzpt = hel * p[3] * ipp * ipt;
    vc[0] = mkcmplx((T)0, (T)0);
    vc[1] = mkcmplx(-p[1] * pzpt, -sv * p[2] * ipt);
    vc[2] = mkcmplx(-p[2] * pzpt, sv * p[1] * ipt);
    vc[3] = mkcmplx(hel * pt * ipp * rsqrt2, (T)0);
    vc[4] = mkcmplx(sv * p[0], sv * p[3]);
    vc[5] = mkcmplx(sv * p[1], sv * p[2]);
}

// p along +z: Lists 9 is this with nSV = -1
template <typename T>
__device__ __forceinline__ void vxxxx1(const T* p, int nHEL, int nSV, cmplx<T>* vc)
{
    const T rsqrt2 = (T)0.70710678118654752440;
    vc[0] = mkcmplx((T)0, (T)0);
    vc[1] = mkcmplx(-(T)nHEL * rsqrt2, (T)0);
    vc[2] = mkcmplx((T)0, (T)nSV * rsqrt2);
    vc[3] = mkcmplx((T)0, (T)0);
    vc[4] = mkcmplx((T)nSV * p[0], (T)nSV * p[0]);
    vc[5] = mkcmplx((T)0, (T)0);
}

// p along -z: List 10 is this with nSV = -1
template <typename T>
__device__ __forceinline__ void vxxxx2(const T* p, int nHEL, int nSV, cmplx<T>* vc)
{
    const T rsqrt2 = (T)0.70710678118654752440;
    vc[0] = mkcmplx((T)0, (T)0);
    vc[1] = mkcmplx(-(T)nHEL * rsqrt2, (T)0);
    vc[2] = mkcmplx((T)0, -(T)nSV * rsqrt2);
    vc[3] = mkcmplx((T)0, (T)0);
    vc[4] = mkcmplx((T)nSV * p[0], -(T)nSV * p[0]);
    vc[5] = mkcmplx((T)0, (T)0);
}

// ---- FFV vertex (Appendix B.3), gal[0] = gal[1] = g (eq. 26) ----------------
// 2x2 blocks of a-slash for a complex four-vector a: Vm = a0 - a.s, Vp = a0 + a.s
template <typename T>
struct SlashBlocks {
    cmplx<T> m00, m01, m10, m11;  // Vm
    cmplx<T> p00, p01, p10, p11;  // Vp
};

template <typename T>
__device__ __forceinline__ SlashBlocks<T> slash_blocks(const cmplx<T>* a)
{
    const cmplx<T> a12m = a[1] - times_i(a[2]);  // a1 - i a2
    const cmplx<T> a12p = a[1] + times_i(a[2]);  // a1 + i a2
    SlashBlocks<T> s;
    s.m00 = a[0] - a[3]; s.m01 = -a12m; s.m10 = -a12p; s.m11 = a[0] + a[3];
    s.p00 = a[0] + a[3]; s.p01 = a12m;  s.p10 = a12p;  s.p11 = a[0] - a[3];
    return s;
}

// the same for the real momentum stored in w[4], w[5]
template <typename T>
__device__ __forceinline__ SlashBlocks<T> slash_blocks_momentum(cmplx<T> w4, cmplx<T> w5, T& p2)
{
    const T p0 = w4.re, p3 = w4.im, p1 = w5.re, pim = w5.im;
    p2 = fma(p0 - p3, p0 + p3, -fma(p1, p1, pim * pim));  // Minkowski square, eq. (8)
    SlashBlocks<T> s;
    s.m00 = mkcmplx(p0 - p3, (T)0); s.m01 = mkcmplx(-p1, pim);  s.m10 = mkcmplx(-p1, -pim); s.m11 = mkcmplx(p0 + p3, (T)0);
    s.p00 = mkcmplx(p0 + p3, (T)0); s.p01 = mkcmplx(p1, -pim);  s.p10 = mkcmplx(p1, pim);   s.p11 = mkcmplx(p0 - p3, (T)0);
    return s;
}

// column: out = a-slash psi;  row: out = phi a-slash
template <typename T>
__device__ __forceinline__ void slash_times_column(const SlashBlocks<T>& s, const cmplx<T>* psi, cmplx<T>* out)
{
    out[0] = s.m00 * psi[2] + s.m01 * psi[3];
    out[1] = s.m10 * psi[2] + s.m11 * psi[3];
    out[2] = s.p00 * psi[0] + s.p01 * psi[1];
    out[3] = s.p10 * psi[0] + s.p11 * psi[1];
}

template <typename T>
__device__ __forceinline__ void row_times_slash(const cmplx<T>* phi, const SlashBlocks<T>& s, cmplx<T>* out)
{
    out[0] = phi[2] * s.p00 + phi[3] * s.p10;
    out[1] = phi[2] * s.p01 + phi[3] * s.p11;
    out[2] = phi[0] * s.m00 + phi[1] * s.m10;
    out[3] = phi[0] * s.m01 + phi[1] * s.m11;
}

// iovxxx: amplitude g <fo| vc-slash |fi>  (List 12)
template <typename T>
__device__ __forceinline__ cmplx<T> iovxxx(const cmplx<T>* fi, const cmplx<T>* fo, const cmplx<T>* vc, T g)
{
    cmplx<T> w[4];
    slash_times_column(slash_blocks(vc), fi, w);
    return g * (fo[0] * w[0] + fo[1] * w[1] + fo[2] * w[2] + fo[3] * w[3]);
}

// fvixx0: off-shell flowing-in fermion -g pf-slash vc-slash |fi> / pf^2, pf = p_fi - p_vc
// (List 13)
template <typename T>
__device__ __forceinline__ void fvixx0(const cmplx<T>* fi, const cmplx<T>* vc, T g, cmplx<T>* fvi)
{
    fvi[4] = fi[4] - vc[4];
    fvi[5] = fi[5] - vc[5];
    T pf2;
    const SlashBlocks<T> P = slash_blocks_momentum(fvi[4], fvi[5], pf2);
    cmplx<T> w[4], o[4];
    slash_times_column(slash_blocks(vc), fi, w);
    slash_times_column(P, w, o);
    const T d = -g / pf2;
#pragma unroll
    for (int a = 0; a < 4; ++a) fvi[a] = d * o[a];
}

// fvoxx0: off-shell flowing-out fermion -g <fo| vc-slash pf-slash / pf^2, pf = p_fo + p_vc
// (List 14)
template <typename T>
__device__ __forceinline__ void fvoxx0(const cmplx<T>* fo, const cmplx<T>* vc, T g, cmplx<T>* fvo)
{
    fvo[4] = fo[4] + vc[4];
    fvo[5] = fo[5] + vc[5];
    T pf2;
    const SlashBlocks<T> P = slash_blocks_momentum(fvo[4], fvo[5], pf2);
    cmplx<T> w[4], o[4];
    row_times_slash(fo, slash_blocks(vc), w);
    row_times_slash(w, P, o);
    const T d = -g / pf2;
#pragma unroll
    for (int a = 0; a < 4; ++a) fvo[a] = d * o[a];
}

// jioxx0: off-shell vector current g <fo| gamma^mu |fi> / q^2 in the Feynman gauge,
// q = p_fo - p_fi (List 15)
template <typename T>
__device__ __forceinline__ void jioxx0(const cmplx<T>* fi, const cmplx<T>* fo, T g, cmplx<T>* jio)
{
    jio[4] = fo[4] - fi[4];
    jio[5] = fo[5] - fi[5];
    const T q0 = jio[4].re, q3 = jio[4].im, q1 = jio[5].re, q2c = jio[5].im;
    const T q2 = fma(q0 - q3, q0 + q3, -fma(q1, q1, q2c * q2c));
    const T d = g / q2;
    // fo_u s^i fi_l - fo_l s^i fi_u for i = 1..3, fo_u fi_l + fo_l fi_u for mu = 0
    const cmplx<T> a00 = fo[0] * fi[2], a01 = fo[0] * fi[3], a10 = fo[1] * fi[2], a11 = fo[1] * fi[3];
    const cmplx<T> b00 = fo[2] * fi[0], b01 = fo[2] * fi[1], b10 = fo[3] * fi[0], b11 = fo[3] * fi[1];
    jio[0] = d * (a00 + a11 + b00 + b11);
    jio[1] = d * ((a01 + a10) - (b01 + b10));
    jio[2] = d * (times_i(a10 - a01) - times_i(b10 - b01));
    jio[3] = d * ((a00 - a11) - (b00 - b11));
}

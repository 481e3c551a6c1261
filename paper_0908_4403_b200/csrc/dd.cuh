// dd.cuh -- double-double ("compensated") arithmetic for the subset kinematics table.
//
// t_S = (p1 - K_S)^2 of eq. (8) cancels catastrophically for forward photons;
// the table is therefore accumulated as unevaluated sums hi+lo of two doubles (error-free
// transformations of Knuth / Dekker, products via FMA) and rounded once.  Explicit _rn
// intrinsics keep the compiler from contracting or re-associating the sequences.
#pragma once

struct dd {
    double hi, lo;
};

__device__ __forceinline__ dd dd_two_sum(double a, double b)
{
    const double s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    const double e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
    return {s, e};
}

__device__ __forceinline__ dd dd_fast_two_sum(double a, double b)  // |a| >= |b|
{
    const double s = __dadd_rn(a, b);
    const double e = __dsub_rn(b, __dsub_rn(s, a));
    return {s, e};
}

__device__ __forceinline__ dd dd_two_prod(double a, double b)
{
    const double p = __dmul_rn(a, b);
    const double e = __fma_rn(a, b, -p);
    return {p, e};
}

// a += b without renormalising: the high part by TwoSum, its rounding error collected in the
// low part (exact to ~2^-106 of the largest intermediate for the handful of terms summed here)
__device__ __forceinline__ void dd_acc(dd& a, double b)
{
    const dd s = dd_two_sum(a.hi, b);
    a.hi = s.hi;
    a.lo = __dadd_rn(a.lo, s.lo);
}

__device__ __forceinline__ dd dd_add_d(dd a, double b)
{
    dd s = dd_two_sum(a.hi, b);
    s.lo = __dadd_rn(s.lo, a.lo);
    return dd_fast_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = dd_two_sum(a.hi, b.hi);
    dd t = dd_two_sum(a.lo, b.lo);
    s.lo = __dadd_rn(s.lo, t.hi);
    s = dd_fast_two_sum(s.hi, s.lo);
    s.lo = __dadd_rn(s.lo, t.lo);
    return dd_fast_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_neg(dd a) { return {-a.hi, -a.lo}; }

__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    dd p = dd_two_prod(a.hi, b.hi);
    p.lo = __dadd_rn(p.lo, __dadd_rn(__dmul_rn(a.hi, b.lo), __dmul_rn(a.lo, b.hi)));
    return dd_fast_two_sum(p.hi, p.lo);
}

__device__ __forceinline__ double dd_to_double(dd a) { return __dadd_rn(a.hi, a.lo); }

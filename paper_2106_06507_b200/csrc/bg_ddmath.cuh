// Double-double instantiation of the vertex algebra of bg_math.cuh, for the program interpreter's re-evaluation of
// events whose FP64 result is flagged as ill-conditioned (the colour-flow amplitude of
// Eq. 19 / 28-32, has near-zeros where FP64 round-off exceeds 1e-11).
// Same formulas, same (unscaled) conventions and the same function names as bg_math.cuh, so that one interpreter body
// serves cx (complex FP64), double (real FP64) and cxd (complex double-double) currents.
// The multiply-accumulate is fused: acc += a*b costs one two-product (FMA), two cross terms and one two-sum, without
// renormalising the accumulator (11 FP64 instructions; dd_renorm once per vertex); ~106-bit significands are far more than the re-evaluation
// needs (cancellations down to 1e-9 of the terms at a 1e-11 target), so the cheaper "sloppy" addition is used.
#pragma once
#include "bg_dd.cuh"
#include "bg_math.cuh"

namespace bg {

using cxd = cxt<dd>;


// acc += a*b.  (The leading product is formed with __dmul_rn: a plain a.hi * b.hi could be contracted with the
// following addition into one FMA, and the two-sum below is error-free only for the rounded product.)
__device__ __forceinline__ void dd_fma(dd& acc, dd a, dd b) {
    const double p = __dmul_rn(a.hi, b.hi);
    double e = fma(a.hi, b.hi, -p);
    e = fma(a.hi, b.lo, e);
    e = fma(a.lo, b.hi, e);
    const double s = acc.hi + p;
    const double bb = s - acc.hi;
    const double err = (acc.hi - (s - bb)) + (p - bb);
    // the accumulator is NOT renormalised here: hi takes the rounded sum, lo collects the exact error terms.  A chain
    // of multiply-adds into one accumulator then depends on the previous one through a single addition instead of
    // ten dependent operations, and costs 11 instead of 15 instructions; dd_renorm() at the end of a vertex.
    acc.lo += err + e;
    acc.hi = s;
}
// (hi, lo) -> the same value with |lo| <= ulp(hi)/2 (two-sum: |hi| >= |lo| is not guaranteed after cancellation)
__device__ __forceinline__ void dd_renorm(dd& a) {
    const double s = a.hi + a.lo, bb = s - a.hi;
    a.lo = (a.hi - (s - bb)) + (a.lo - bb);
    a.hi = s;
}
__device__ __forceinline__ dd dd_neg(dd a) { return mkdd(-a.hi, -a.lo); }
// a + b without the second renormalisation (error 2^-104 relative to |a| + |b|)
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    const double s = a.hi + b.hi;
    const double bb = s - a.hi;
    const double err = (a.hi - (s - bb)) + (b.hi - bb);
    const double lo = err + (a.lo + b.lo);
    const double hi = s + lo;
    return mkdd(hi, lo - (hi - s));
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    const double p = __dmul_rn(a.hi, b.hi);
    double e = fma(a.hi, b.hi, -p);
    e = fma(a.hi, b.lo, e);
    e = fma(a.lo, b.hi, e);
    const double hi = p + e;
    return mkdd(hi, e - (hi - p));
}
__device__ __forceinline__ dd dd_twice(dd a) { return mkdd(2.0 * a.hi, 2.0 * a.lo); }

// ---- complex double-double ------------------------------------------------------------------------------
__device__ __forceinline__ cxd mkd(dd re, dd im) { cxd r; r.re = re; r.im = im; return r; }
__device__ __forceinline__ cxd cxd_add(cxd a, cxd b) { return mkd(dd_add(a.re, b.re), dd_add(a.im, b.im)); }
__device__ __forceinline__ cxd cxd_neg(cxd a) { return mkd(dd_neg(a.re), dd_neg(a.im)); }
// (Tried: cfma as a real function to shrink the ~10k-instruction kernel body, which stalls on instruction fetch -
// the argument moves cost as many instructions as the body saves; 20 % slower.  DESIGN.md 9.)
__device__ __forceinline__ void cfma(cxd& acc, cxd a, cxd b) {
    dd_fma(acc.re, a.re, b.re);
    dd_fma(acc.re, dd_neg(a.im), b.im);
    dd_fma(acc.im, a.re, b.im);
    dd_fma(acc.im, a.im, b.re);
}
__device__ __forceinline__ void cfms(cxd& acc, cxd a, cxd b) { cfma(acc, cxd_neg(a), b); }
__device__ __forceinline__ void rfma(cxd& acc, dd s, cxd a) {
    dd_fma(acc.re, s, a.re);
    dd_fma(acc.im, s, a.im);
}
__device__ __forceinline__ cxd cxd_mul(cxd a, cxd b) {
    cxd r = mkd(dd_mul(a.re, b.re), dd_mul(a.re, b.im));
    dd_fma(r.re, dd_neg(a.im), b.im);
    dd_fma(r.im, a.im, b.re);
    dd_renorm(r.re);
    dd_renorm(r.im);
    return r;
}
__device__ __forceinline__ void cxd_renorm(cxd& a) { dd_renorm(a.re); dd_renorm(a.im); }
__device__ __forceinline__ cxd cxd_scale(dd s, cxd a) { return mkd(dd_mul(s, a.re), dd_mul(s, a.im)); }

// Minkowski products (no complex conjugation)
__device__ __forceinline__ cxd mdot(const cxd* a, const cxd* b) {
    cxd r = cxd_mul(a[0], b[0]);
    cfms(r, a[1], b[1]);
    cfms(r, a[2], b[2]);
    cfms(r, a[3], b[3]);
    cxd_renorm(r);
    return r;
}
__device__ __forceinline__ cxd mdot(const dd* p, const cxd* a) {
    cxd r = cxd_scale(p[0], a[0]);
    rfma(r, dd_neg(p[1]), a[1]);
    rfma(r, dd_neg(p[2]), a[2]);
    rfma(r, dd_neg(p[3]), a[3]);
    cxd_renorm(r);
    return r;
}
__device__ __forceinline__ dd mdot(const dd* p, const dd* q) {
    dd r = dd_mul(p[0], q[0]);
    dd_fma(r, dd_neg(p[1]), q[1]);
    dd_fma(r, dd_neg(p[2]), q[2]);
    dd_fma(r, dd_neg(p[3]), q[3]);
    dd_renorm(r);
    return r;
}

// acc += sign * sqrt2 * V3(p,q;a,b)   [Eq. 21 first line, as bg_math.cuh]
__device__ __forceinline__ void v3_acc(cxd* acc, const dd* p, const dd* q, const cxd* a, const cxd* b, double sign) {
    dd tqp[4], tpq[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        tqp[mu] = dd_add(dd_twice(q[mu]), p[mu]);
        tpq[mu] = dd_add(dd_twice(p[mu]), q[mu]);
    }
    cxd ab = mdot(a, b), qa = mdot(tqp, a), pb = mdot(tpq, b);
    if (sign < 0.0) { ab = cxd_neg(ab); qa = cxd_neg(qa); pb = cxd_neg(pb); }
#pragma unroll
    for (int nu = 0; nu < 4; nu++) {
        rfma(acc[nu], dd_sub(p[nu], q[nu]), ab);
        cfma(acc[nu], qa, b[nu]);
        cfms(acc[nu], pb, a[nu]);
        cxd_renorm(acc[nu]);
    }
}
// acc^nu += sign * T^{nu beta} v_beta ; T[0..5] = T^{01}, T^{02}, T^{03}, T^{12}, T^{13}, T^{23}
__device__ __forceinline__ void tcontract_acc(cxd* acc, const cxd* T, const cxd* v, double sign) {
    cxd v0 = v[0], v1 = v[1], v2 = v[2], v3 = v[3];
    if (sign < 0.0) { v0 = cxd_neg(v0); v1 = cxd_neg(v1); v2 = cxd_neg(v2); v3 = cxd_neg(v3); }
    cfms(acc[0], T[0], v1); cfms(acc[0], T[1], v2); cfms(acc[0], T[2], v3);
    cfms(acc[1], T[0], v0); cfms(acc[1], T[3], v2); cfms(acc[1], T[4], v3);
    cfms(acc[2], T[1], v0); cfma(acc[2], T[3], v1); cfms(acc[2], T[5], v3);
    cfms(acc[3], T[2], v0); cfma(acc[3], T[4], v1); cfma(acc[3], T[5], v2);
#pragma unroll
    for (int nu = 0; nu < 4; nu++) cxd_renorm(acc[nu]);
}
// tacc += sign * (a^alpha b^beta - a^beta b^alpha)
__device__ __forceinline__ void tbuild_acc(cxd* tacc, const cxd* a, const cxd* b, double sign) {
    cxd b0 = b[0], b1 = b[1], b2 = b[2], b3 = b[3];
    if (sign < 0.0) { b0 = cxd_neg(b0); b1 = cxd_neg(b1); b2 = cxd_neg(b2); b3 = cxd_neg(b3); }
    cfma(tacc[0], a[0], b1); cfms(tacc[0], a[1], b0);
    cfma(tacc[1], a[0], b2); cfms(tacc[1], a[2], b0);
    cfma(tacc[2], a[0], b3); cfms(tacc[2], a[3], b0);
    cfma(tacc[3], a[1], b2); cfms(tacc[3], a[2], b1);
    cfma(tacc[4], a[1], b3); cfms(tacc[4], a[3], b1);
    cfma(tacc[5], a[2], b3); cfms(tacc[5], a[3], b2);
#pragma unroll
    for (int c = 0; c < 6; c++) cxd_renorm(tacc[c]);
}

template <> __device__ __forceinline__ cxd s_zero<cxd>() { return mkd(mkdd(0.0), mkdd(0.0)); }
template <> __device__ __forceinline__ cxd s_real<cxd>(double x) { return mkd(mkdd(x), mkdd(0.0)); }
__device__ __forceinline__ double s_norm2(cxd a) {
    dd r = dd_mul(a.re, a.re);
    dd_fma(r, a.im, a.im);
    return r.hi + r.lo;
}

}  // namespace bg

// Double-double arithmetic (two FP64 words, ~106-bit significand) and the complex Lorentz algebra of
// bg_math.cuh written for a generic real type.  Used only by the refinement path that re-evaluates ill-conditioned
// events; the FP64 kernels keep their hand-scheduled versions in bg_math.cuh.
// Error-free transformations: Knuth two-sum, FMA two-product (Dekker / Hida-Li-Bailey "QD" algorithms, restated).
#pragma once
#include <cuda_runtime.h>

namespace bg {

struct dd {
    double hi, lo;
};

__device__ __forceinline__ dd mkdd(double hi, double lo = 0.0) { dd r; r.hi = hi; r.lo = lo; return r; }
__device__ __forceinline__ dd quick_two_sum(double a, double b) {   // |a| >= |b|
    const double s = a + b;
    return mkdd(s, b - (s - a));
}
__device__ __forceinline__ dd two_sum(double a, double b) {
    const double s = a + b, bb = s - a;
    return mkdd(s, (a - (s - bb)) + (b - bb));
}
__device__ __forceinline__ dd two_prod(double a, double b) {
    const double p = __dmul_rn(a, b);   // never contracted into an FMA with a later addition
    return mkdd(p, fma(a, b, -p));
}
__device__ __forceinline__ dd operator+(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    const dd t = two_sum(a.lo, b.lo);
    s.lo += t.hi;
    s = quick_two_sum(s.hi, s.lo);
    s.lo += t.lo;
    return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd operator-(dd a) { return mkdd(-a.hi, -a.lo); }
__device__ __forceinline__ dd operator-(dd a, dd b) { return a + (-b); }
__device__ __forceinline__ dd operator*(dd a, dd b) {
    dd p = two_prod(a.hi, b.hi);
    p.lo += a.hi * b.lo + a.lo * b.hi;
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd operator/(dd a, dd b) {
    const double q1 = a.hi / b.hi;
    dd r = a - b * mkdd(q1);
    const double q2 = r.hi / b.hi;
    r = r - b * mkdd(q2);
    const double q3 = r.hi / b.hi;
    dd q = quick_two_sum(q1, q2);
    return q + mkdd(q3);
}
__device__ __forceinline__ dd sqrt(dd a) {
    if (a.hi <= 0.0) return mkdd(0.0);
    const double x = 1.0 / ::sqrt(a.hi), ax = a.hi * x;
    const dd e = a - two_prod(ax, ax);
    return two_sum(ax, e.hi * (x * 0.5));
}
__device__ __forceinline__ bool operator<(dd a, dd b) { return a.hi < b.hi || (a.hi == b.hi && a.lo < b.lo); }

// conversions shared by the generic code below
__device__ __forceinline__ double to_double(double x) { return x; }
__device__ __forceinline__ double to_double(dd x) { return x.hi + x.lo; }
template <class R> __device__ __forceinline__ R from_double(double x);
template <> __device__ __forceinline__ double from_double<double>(double x) { return x; }
template <> __device__ __forceinline__ dd from_double<dd>(double x) { return mkdd(x); }

// ---- complex numbers and Lorentz algebra over a generic real type R ------------------------------------
template <class R>
struct cxt {
    R re, im;
};
template <class R> __device__ __forceinline__ cxt<R> mkc(R re, R im) { cxt<R> r; r.re = re; r.im = im; return r; }
template <class R> __device__ __forceinline__ cxt<R> operator+(cxt<R> a, cxt<R> b) { return mkc<R>(a.re + b.re, a.im + b.im); }
template <class R> __device__ __forceinline__ cxt<R> operator-(cxt<R> a, cxt<R> b) { return mkc<R>(a.re - b.re, a.im - b.im); }
template <class R> __device__ __forceinline__ cxt<R> operator*(cxt<R> a, cxt<R> b) {
    return mkc<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <class R> __device__ __forceinline__ cxt<R> operator*(R s, cxt<R> a) { return mkc<R>(s * a.re, s * a.im); }


// Minkowski products (no conjugation)
template <class R> __device__ __forceinline__ cxt<R> mdot_t(const cxt<R>* a, const cxt<R>* b) {
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
}
template <class R> __device__ __forceinline__ cxt<R> mdot_t(const R* p, const cxt<R>* a) {
    return p[0] * a[0] - p[1] * a[1] - p[2] * a[2] - p[3] * a[3];
}
template <class R> __device__ __forceinline__ R mdot_t(const R* p, const R* q) {
    return p[0] * q[0] - p[1] * q[1] - p[2] * q[2] - p[3] * q[3];
}

// eps^lambda(p), Eq. 3, gauge of DESIGN.md readings g2/g3 - same formula as bg_math.cuh
template <class R> __device__ __forceinline__ void polarisation_t(const R* p, int lambda, cxt<R>* eps) {
    const R zero = from_double<R>(0.0), one = from_double<R>(1.0);
    const bool flip = to_double(p[0]) < 0.0;
    const R qx = flip ? zero - p[1] : p[1], qy = flip ? zero - p[2] : p[2], qz = flip ? zero - p[3] : p[3];
    const R qt2 = qx * qx + qy * qy;
    const R qt = sqrt(qt2), qa = sqrt(qt2 + qz * qz);
    R e1x, e1y, e1z, e2x, e2y;
    if (to_double(qt) < 1e-9 * to_double(qa)) {
        e1x = one; e1y = zero; e1z = zero;
        e2x = zero; e2y = to_double(qz) < 0.0 ? zero - one : one;
    } else {
        e1x = qx * qz / (qa * qt); e1y = qy * qz / (qa * qt); e1z = zero - qt / qa;
        e2x = zero - qy / qt; e2y = qx / qt;
    }
    const R is2 = one / sqrt(from_double<R>(2.0));
    const R l = lambda > 0 ? zero - is2 : is2;
    eps[0] = mkc<R>(zero, zero);
    eps[1] = mkc<R>(l * e1x, zero - is2 * e2x);
    eps[2] = mkc<R>(l * e1y, zero - is2 * e2y);
    eps[3] = mkc<R>(l * e1z, zero);
}

// acc += sign * sqrt2 * V3(p,q;a,b)   (Eq. 21 first line, unscaled as in bg_math.cuh)
template <class R>
__device__ __forceinline__ void v3_acc_t(cxt<R>* acc, const R* p, const R* q, const cxt<R>* a, const cxt<R>* b, bool neg) {
    const R two = from_double<R>(2.0);
    R tqp[4], tpq[4];
    for (int mu = 0; mu < 4; mu++) { tqp[mu] = two * q[mu] + p[mu]; tpq[mu] = two * p[mu] + q[mu]; }
    const cxt<R> ab = mdot_t(a, b), qa = mdot_t(tqp, a), pb = mdot_t(tpq, b);
    for (int nu = 0; nu < 4; nu++) {
        const cxt<R> t = (p[nu] - q[nu]) * ab + qa * b[nu] - pb * a[nu];
        acc[nu] = neg ? acc[nu] - t : acc[nu] + t;
    }
}
// acc^nu += sign * T^{nu beta} v_beta ; T[0..5] = T^{01}, T^{02}, T^{03}, T^{12}, T^{13}, T^{23}
template <class R>
__device__ __forceinline__ void tcontract_acc_t(cxt<R>* acc, const cxt<R>* T, const cxt<R>* v, bool neg) {
    cxt<R> t[4];
    const cxt<R> z = mkc<R>(from_double<R>(0.0), from_double<R>(0.0));
    t[0] = z - T[0] * v[1] - T[1] * v[2] - T[2] * v[3];
    t[1] = z - T[0] * v[0] - T[3] * v[2] - T[4] * v[3];
    t[2] = z - T[1] * v[0] + T[3] * v[1] - T[5] * v[3];
    t[3] = z - T[2] * v[0] + T[4] * v[1] + T[5] * v[2];
    for (int nu = 0; nu < 4; nu++) acc[nu] = neg ? acc[nu] - t[nu] : acc[nu] + t[nu];
}
// tacc += sign * (a^alpha b^beta - a^beta b^alpha)
template <class R>
__device__ __forceinline__ void tbuild_acc_t(cxt<R>* tacc, const cxt<R>* a, const cxt<R>* b, bool neg) {
    cxt<R> t[6];
    t[0] = a[0] * b[1] - a[1] * b[0]; t[1] = a[0] * b[2] - a[2] * b[0]; t[2] = a[0] * b[3] - a[3] * b[0];
    t[3] = a[1] * b[2] - a[2] * b[1]; t[4] = a[1] * b[3] - a[3] * b[1]; t[5] = a[2] * b[3] - a[3] * b[2];
    for (int c = 0; c < 6; c++) tacc[c] = neg ? tacc[c] - t[c] : tacc[c] + t[c];
}

}  // namespace bg

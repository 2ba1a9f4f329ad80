// Device-side FP64 complex Lorentz arithmetic for the Berends-Giele kernels (sm_100a).
// Formulas follow PAPER.md Eq. 3 (polarisation vectors), Eq. 21 (three- and four-gluon vertices) and
// Eq. 23-26 (tensor pseudo-particle) with g_s = 1 and the factors of i multiplied out; the common factor
// 1/sqrt2 of V3, V_T and of the tensor current is NOT applied here: callers accumulate unscaled sums and
// multiply once when a current is finalised.
#pragma once
#include <cuda_runtime.h>

namespace bg {

constexpr double kInvSqrt2 = 0.70710678118654752440;

struct cx {
    double re, im;
};

__device__ __forceinline__ cx mk(double re, double im) { cx r; r.re = re; r.im = im; return r; }
__device__ __forceinline__ cx operator+(cx a, cx b) { return mk(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ cx operator-(cx a, cx b) { return mk(a.re - b.re, a.im - b.im); }
__device__ __forceinline__ cx operator*(cx a, cx b) {
    return mk(fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re));
}
__device__ __forceinline__ cx operator*(double s, cx a) { return mk(s * a.re, s * a.im); }
// acc += a*b
__device__ __forceinline__ void cfma(cx& acc, cx a, cx b) {
    acc.re = fma(a.re, b.re, acc.re);
    acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im);
    acc.im = fma(a.im, b.re, acc.im);
}
// acc -= a*b
__device__ __forceinline__ void cfms(cx& acc, cx a, cx b) {
    acc.re = fma(-a.re, b.re, acc.re);
    acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(-a.re, b.im, acc.im);
    acc.im = fma(-a.im, b.re, acc.im);
}
// acc += s*a (s real)
__device__ __forceinline__ void rfma(cx& acc, double s, cx a) {
    acc.re = fma(s, a.re, acc.re);
    acc.im = fma(s, a.im, acc.im);
}

// Minkowski product, no complex conjugation
__device__ __forceinline__ cx mdot(const cx* a, const cx* b) {
    cx r = a[0] * b[0];
    cfms(r, a[1], b[1]);
    cfms(r, a[2], b[2]);
    cfms(r, a[3], b[3]);
    return r;
}
__device__ __forceinline__ cx mdot(const double* p, const cx* a) {
    cx r = mk(p[0] * a[0].re, p[0] * a[0].im);
    rfma(r, -p[1], a[1]);
    rfma(r, -p[2], a[2]);
    rfma(r, -p[3], a[3]);
    return r;
}
__device__ __forceinline__ double mdot(const double* p, const double* q) {
    return fma(p[0], q[0], -fma(p[1], q[1], fma(p[2], q[2], p[3] * q[3])));
}

// Helicity eigenvector eps^lambda(p), Eq. 3 in the light-cone gauge k = (q0, -q) of DESIGN.md
// reading g2/g3 (q = p for outgoing, -p for incoming legs; same lambda).  eps^0 = 0.
__device__ __forceinline__ void polarisation(const double* p, int lambda, cx* eps) {
    const double s = p[0] < 0.0 ? -1.0 : 1.0;
    const double qx = s * p[1], qy = s * p[2], qz = s * p[3];
    const double qt2 = qx * qx + qy * qy;
    const double qt = ::sqrt(qt2), qa = ::sqrt(qt2 + qz * qz);
    double e1x, e1y, e1z, e2x, e2y;
    if (qt < 1e-9 * qa) {
        e1x = 1.0; e1y = 0.0; e1z = 0.0;
        e2x = 0.0; e2y = qz < 0.0 ? -1.0 : 1.0;
    } else {
        const double inv = 1.0 / (qa * qt), invt = 1.0 / qt;
        e1x = qx * qz * inv; e1y = qy * qz * inv; e1z = -qt / qa;
        e2x = -qy * invt; e2y = qx * invt;
    }
    const double l = -(double)lambda * kInvSqrt2;
    eps[0] = mk(0.0, 0.0);
    eps[1] = mk(l * e1x, -kInvSqrt2 * e2x);
    eps[2] = mk(l * e1y, -kInvSqrt2 * e2y);
    eps[3] = mk(l * e1z, 0.0);
}

// The same event in another frame (second stage of the precision cascade).
// rotate_frame: the spatial components of a momentum rotated by a fixed rotation (axis (1,2,3), angle 1 rad).  The
// polarisation vectors of Eq. 3 in the gauge k = (q0, -q) rotate with the momenta, so every Lorentz product of the
// recursion keeps its value and |A|^2 is the same number - computed from different components, i.e. with independent
// round-off: the difference of the two results samples the FP64 error of the event.
__device__ __forceinline__ void rotate_frame(double* pk) {
    const double x = pk[1], y = pk[2], z = pk[3];
    pk[1] = fma(0.5731378554489869, x, fma(-0.6090066421373933, y, 0.5482918096085999 * z));
    pk[2] = fma(0.740348840460782, x, fma(0.6716445041915284, y, -0.027879282947946255 * z));
    pk[3] = fma(-0.35127851212351696, x, fma(0.4219058779181122, y, 0.8358222520957642 * z));
}
// boost_frame: that rotation followed by a boost (beta = (0.3, -0.2, 0.25)).  Helicities of massless particles are
// Lorentz invariant; the polarisation vectors built from the transformed momenta differ from the transformed vectors by
// a phase and a gauge shift, so |A|^2 is again the same number - now with the energies changed too.  A rotation leaves
// the energies, and with them half of the round-off of every P^2 = E^2 - |p|^2, as they were: in the colour-ordered
// path events whose two results agreed to 5e-13 while both were off by 1.5e-11 turned up once per 2 - 4 million with
// the rotation and not at all with the boost (4.2e6 / 2.1e6 events at n = 6 / 7).  The colour-dressed path keeps the
// rotation: there the boost left the misses as they were (unflagged events) and raised the share of
// events the second stage rejects from 2.6 to 3.1 % at n = 6.
__device__ __forceinline__ void boost_frame(double* pk) {
    const double e = pk[0], x = pk[1], y = pk[2], z = pk[3];
    pk[0] = fma(1.1128297681493144, e, fma(0.07116328195741217, x, fma(0.23542406061087687, y, -0.4217835841587401 * z)));
    pk[1] = fma(-0.3338489304447943, e, fma(0.5618933217309517, x, fma(-0.6462060758166889, y, 0.6149379732386724 * z)));
    pk[2] = fma(0.2225659536298629, e, fma(0.7478451962728053, x, fma(0.696444126644392, y, -0.0723100587013279 * z)));
    pk[3] = fma(-0.2782074420373286, e, fma(-0.36064895688854626, x, fma(0.3909063498520326, y, 0.8913607217874913 * z)));
}

// Real polarisation vector of the continuous sampling, Eq. 7: e(p, phi) = cos(phi) e1 + sin(phi) e2
// with the unit vectors e1, e2 of the same gauge as `polarisation` (eps^lambda = (-lambda e1 - i e2)/sqrt2).
__device__ __forceinline__ void polarisation_real(const double* p, double phi, double* e) {
    const double s = p[0] < 0.0 ? -1.0 : 1.0;
    const double qx = s * p[1], qy = s * p[2], qz = s * p[3];
    const double qt2 = qx * qx + qy * qy;
    const double qt = ::sqrt(qt2), qa = ::sqrt(qt2 + qz * qz);
    double e1x, e1y, e1z, e2x, e2y;
    if (qt < 1e-9 * qa) {
        e1x = 1.0; e1y = 0.0; e1z = 0.0;
        e2x = 0.0; e2y = qz < 0.0 ? -1.0 : 1.0;
    } else {
        const double inv = 1.0 / (qa * qt), invt = 1.0 / qt;
        e1x = qx * qz * inv; e1y = qy * qz * inv; e1z = -qt / qa;
        e2x = -qy * invt; e2y = qx * invt;
    }
    double sn, cs;
    sincos(phi, &sn, &cs);
    e[0] = 0.0;
    e[1] = cs * e1x + sn * e2x;
    e[2] = cs * e1y + sn * e2y;
    e[3] = cs * e1z;
}

// acc += sign * sqrt2 * V3(p,q;a,b)   [Eq. 21 first line: (a.b)(p-q) + ((2q+p).a) b - ((2p+q).b) a]
__device__ __forceinline__ void v3_acc(cx* acc, const double* p, const double* q, const cx* a, const cx* b,
                                       double sign) {
    double tqp[4], tpq[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        tqp[mu] = fma(2.0, q[mu], p[mu]);
        tpq[mu] = fma(2.0, p[mu], q[mu]);
    }
    cx ab = mdot(a, b), qa = mdot(tqp, a), pb = mdot(tpq, b);
    ab = sign * ab; qa = sign * qa; pb = sign * pb;
#pragma unroll
    for (int nu = 0; nu < 4; nu++) {
        rfma(acc[nu], p[nu] - q[nu], ab);
        cfma(acc[nu], qa, b[nu]);
        cfms(acc[nu], pb, a[nu]);
    }
}

// Tensor components are stored as T[0..5] = T^{01}, T^{02}, T^{03}, T^{12}, T^{13}, T^{23} (antisymmetric).
// acc^nu += sign * T^{nu beta} v_beta (index lowered with the metric)
__device__ __forceinline__ void tcontract_acc(cx* acc, const cx* T, const cx* v, double sign) {
    const cx v0 = sign * v[0], v1 = sign * v[1], v2 = sign * v[2], v3 = sign * v[3];
    cfms(acc[0], T[0], v1); cfms(acc[0], T[1], v2); cfms(acc[0], T[2], v3);
    cfms(acc[1], T[0], v0); cfms(acc[1], T[3], v2); cfms(acc[1], T[4], v3);
    cfms(acc[2], T[1], v0); cfma(acc[2], T[3], v1); cfms(acc[2], T[5], v3);
    cfms(acc[3], T[2], v0); cfma(acc[3], T[4], v1); cfma(acc[3], T[5], v2);
}

// tacc += sign * (a^alpha b^beta - a^beta b^alpha)   [Eq. 25, unscaled]
__device__ __forceinline__ void tbuild_acc(cx* tacc, const cx* a, const cx* b, double sign) {
    const cx b0 = sign * b[0], b1 = sign * b[1], b2 = sign * b[2], b3 = sign * b[3];
    cfma(tacc[0], a[0], b1); cfms(tacc[0], a[1], b0);
    cfma(tacc[1], a[0], b2); cfms(tacc[1], a[2], b0);
    cfma(tacc[2], a[0], b3); cfms(tacc[2], a[3], b0);
    cfma(tacc[3], a[1], b2); cfms(tacc[3], a[2], b1);
    cfma(tacc[4], a[1], b3); cfms(tacc[4], a[3], b1);
    cfma(tacc[5], a[2], b3); cfms(tacc[5], a[3], b2);
}

// acc += sign * 2 * V4(a,b,c)   [Eq. 21 second line: 2(a.c) b - (a.b) c - (b.c) a]
__device__ __forceinline__ void v4_acc(cx* acc, const cx* a, const cx* b, const cx* c) {
    cx ac = mdot(a, c), ab = mdot(a, b), bc = mdot(b, c);
    ac = 2.0 * ac;
#pragma unroll
    for (int nu = 0; nu < 4; nu++) {
        cfma(acc[nu], ac, b[nu]);
        cfms(acc[nu], ab, c[nu]);
        cfms(acc[nu], bc, a[nu]);
    }
}

// ---- the same vertex algebra for REAL currents (continuous states with real polarisations, Eq. 7: "real valued
// amplitudes for the gluon-only case") --------------------------------------------------------
__device__ __forceinline__ void v3_acc(double* acc, const double* p, const double* q, const double* a, const double* b,
                                       double sign) {
    double tqp[4], tpq[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        tqp[mu] = fma(2.0, q[mu], p[mu]);
        tpq[mu] = fma(2.0, p[mu], q[mu]);
    }
    const double ab = sign * mdot(a, b), qa = sign * mdot(tqp, a), pb = sign * mdot(tpq, b);
#pragma unroll
    for (int nu = 0; nu < 4; nu++) {
        acc[nu] = fma(p[nu] - q[nu], ab, acc[nu]);
        acc[nu] = fma(qa, b[nu], acc[nu]);
        acc[nu] = fma(-pb, a[nu], acc[nu]);
    }
}
__device__ __forceinline__ void tcontract_acc(double* acc, const double* T, const double* v, double sign) {
    const double v0 = sign * v[0], v1 = sign * v[1], v2 = sign * v[2], v3 = sign * v[3];
    acc[0] = fma(-T[0], v1, acc[0]); acc[0] = fma(-T[1], v2, acc[0]); acc[0] = fma(-T[2], v3, acc[0]);
    acc[1] = fma(-T[0], v0, acc[1]); acc[1] = fma(-T[3], v2, acc[1]); acc[1] = fma(-T[4], v3, acc[1]);
    acc[2] = fma(-T[1], v0, acc[2]); acc[2] = fma(T[3], v1, acc[2]);  acc[2] = fma(-T[5], v3, acc[2]);
    acc[3] = fma(-T[2], v0, acc[3]); acc[3] = fma(T[4], v1, acc[3]);  acc[3] = fma(T[5], v2, acc[3]);
}
__device__ __forceinline__ void tbuild_acc(double* tacc, const double* a, const double* b, double sign) {
    const double b0 = sign * b[0], b1 = sign * b[1], b2 = sign * b[2], b3 = sign * b[3];
    tacc[0] = fma(a[0], b1, tacc[0]); tacc[0] = fma(-a[1], b0, tacc[0]);
    tacc[1] = fma(a[0], b2, tacc[1]); tacc[1] = fma(-a[2], b0, tacc[1]);
    tacc[2] = fma(a[0], b3, tacc[2]); tacc[2] = fma(-a[3], b0, tacc[2]);
    tacc[3] = fma(a[1], b2, tacc[3]); tacc[3] = fma(-a[2], b1, tacc[3]);
    tacc[4] = fma(a[1], b3, tacc[4]); tacc[4] = fma(-a[3], b1, tacc[4]);
    tacc[5] = fma(a[2], b3, tacc[5]); tacc[5] = fma(-a[3], b2, tacc[5]);
}

// scalar-type helpers so that one interpreter body serves complex (cx) and real (double) currents
template <class S> __device__ __forceinline__ S s_zero();
template <> __device__ __forceinline__ cx s_zero<cx>() { return mk(0.0, 0.0); }
template <> __device__ __forceinline__ double s_zero<double>() { return 0.0; }
template <class S> __device__ __forceinline__ S s_real(double x);
template <> __device__ __forceinline__ cx s_real<cx>(double x) { return mk(x, 0.0); }
template <> __device__ __forceinline__ double s_real<double>(double x) { return x; }
__device__ __forceinline__ double s_norm2(cx a) { return fma(a.re, a.re, a.im * a.im); }
__device__ __forceinline__ double s_norm2(double a) { return a * a; }

}  // namespace bg

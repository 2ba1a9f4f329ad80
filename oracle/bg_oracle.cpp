// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, literal CPU implementation of what the hot path of
// arxiv 2106.06507 computes, written from /root/reference/PAPER.md (citations "PAPER.md:L<line>").
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
// It shares no code with paper_2106_06507_b200/csrc (the CUDA path) and neither includes the other.
//
// Conventions: n gluons, all-outgoing momenta, metric (+,-,-,-),
// N_c = 3, g_s = 1, generators normalised Tr(T^a T^b) = delta^ab ("conventions of [64]").
// The factors of i in Eq. 20/21 multiply out: (-i from the propagator) x (i from the vertex) = 1.
//
// Every function is a template on the real type R; the extern "C" entry points instantiate R = double
// (first-line comparison and timed CPU baseline) and R = long double (x87 80-bit: the "truth" for the
// round-off protocol).  No blocking, fusion or reordering beyond the formulas as printed; the only shortcut is
// skipping terms whose input current is identically zero, which cannot change any result.
//
// Pins (tests/test_oracle_pins_cobg.py, test_oracle_pins_colour.py, test_oracle_pins_continuous.py): Parke-Taylor MHV moduli, vanishing all-plus / single-minus amplitudes,
// cyclicity, reflection, U(1) decoupling, gauge invariance (eps -> eps + z p, eps -> p), V4 form == tensor
// form, closed-form gg->gg, hand-derivable colour-matrix entries, Eq. 33 exactness at n = 4,5, colour-dressed
// == Eq. 19 brute force, sum over all 9^n colour flows == A^dagger C A; general external states (continuous
// colour / polarisation, Eq. 7-14): elementary X == discrete CDBG, multilinearity in colour and helicity, real
// inputs give real amplitudes, trace part of X decouples, Monte-Carlo normalisation of Eq. 13.  Parity unpinned: nothing exported here.
//
// Build: g++ -O2 -std=c++17 -fopenmp -shared -fPIC bg_oracle.cpp -o libbgoracle.so
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#include <omp.h>

namespace {

constexpr int MAXN = 13;
inline int omp_get_max_threads_wrapper() { return omp_get_max_threads(); }

template <class R> using cx = std::complex<R>;
template <class R> struct V4c { cx<R> v[4]; };          // complex Lorentz vector, upper index
template <class R> struct V4r { R v[4]; };              // real Lorentz vector, upper index
template <class R> struct T6c { cx<R> t[4][4]; };       // antisymmetric tensor, upper indices (full 4x4 kept)

template <class R> inline R sqrt_half() { return R(1) / std::sqrt(R(2)); }

// Minkowski product without complex conjugation
template <class R> inline cx<R> mdot(const V4c<R>& a, const V4c<R>& b) {
    return a.v[0] * b.v[0] - a.v[1] * b.v[1] - a.v[2] * b.v[2] - a.v[3] * b.v[3];
}
template <class R> inline cx<R> mdot(const V4r<R>& p, const V4c<R>& b) {
    return p.v[0] * b.v[0] - p.v[1] * b.v[1] - p.v[2] * b.v[2] - p.v[3] * b.v[3];
}
template <class R> inline R mdot(const V4r<R>& p, const V4r<R>& q) {
    return p.v[0] * q.v[0] - p.v[1] * q.v[1] - p.v[2] * q.v[2] - p.v[3] * q.v[3];
}
template <class R> inline R metric(int mu) { return mu == 0 ? R(1) : R(-1); }

// ---- External currents: helicity eigenvectors, Eq. 3 -----------------------------------
// The paper never prints eps^{+-}(p,k) (k "arbitrary", L44).  DESIGN.md reading g2: for q = +-p with q0 > 0,
//   e1 = (0, qx qz/(|q| qT), qy qz/(|q| qT), -qT/|q|),  e2 = (0, -qy/qT, qx/qT, 0),
//   [qT < 1e-9 |q|: e1 = (0,1,0,0), e2 = (0,0,sgn qz,0)],   eps^lambda = (-lambda e1 - i e2)/sqrt2.
// Reading g3: a negative-energy (incoming) leg uses q = -p with the same lambda.
template <class R> void polarisation(const V4r<R>& p, int lambda, V4c<R>& eps) {
    R s = p.v[0] < 0 ? R(-1) : R(1);
    R qx = s * p.v[1], qy = s * p.v[2], qz = s * p.v[3];
    R qt = std::sqrt(qx * qx + qy * qy);
    R qa = std::sqrt(qx * qx + qy * qy + qz * qz);
    R e1[4], e2[4];
    if (qt < R(1e-9) * qa) {
        e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0;
        e2[0] = 0; e2[1] = 0; e2[2] = qz < 0 ? R(-1) : R(1); e2[3] = 0;
    } else {
        e1[0] = 0; e1[1] = qx * qz / (qa * qt); e1[2] = qy * qz / (qa * qt); e1[3] = -qt / qa;
        e2[0] = 0; e2[1] = -qy / qt; e2[2] = qx / qt; e2[3] = 0;
    }
    R l = R(lambda);
    for (int mu = 0; mu < 4; mu++) eps.v[mu] = cx<R>(-l * e1[mu], -e2[mu]) * sqrt_half<R>();
}

// ---- Vertices, Eq. 21 with g_s = 1 and the i's multiplied out ----------------------
// V3^{nu kappa lambda}(p,q) a_kappa b_lambda = (1/sqrt2)[(a.b)(p-q)^nu + ((2q+p).a) b^nu - ((2p+q).b) a^nu]
template <class R>
void V3(const V4r<R>& p, const V4r<R>& q, const V4c<R>& a, const V4c<R>& b, V4c<R>& out) {
    V4r<R> pmq, tqp, tpq;
    for (int mu = 0; mu < 4; mu++) {
        pmq.v[mu] = p.v[mu] - q.v[mu];
        tqp.v[mu] = R(2) * q.v[mu] + p.v[mu];
        tpq.v[mu] = R(2) * p.v[mu] + q.v[mu];
    }
    cx<R> ab = mdot(a, b), qa = mdot(tqp, a), pb = mdot(tpq, b);
    for (int nu = 0; nu < 4; nu++)
        out.v[nu] = sqrt_half<R>() * (ab * pmq.v[nu] + qa * b.v[nu] - pb * a.v[nu]);
}
// V4^{nu rho kappa lambda} a_rho b_kappa c_lambda = (1/2)[2 (a.c) b^nu - (a.b) c^nu - (b.c) a^nu]
template <class R> void V4(const V4c<R>& a, const V4c<R>& b, const V4c<R>& c, V4c<R>& out) {
    cx<R> ac = mdot(a, c), ab = mdot(a, b), bc = mdot(b, c);
    for (int nu = 0; nu < 4; nu++) out.v[nu] = R(0.5) * (R(2) * ac * b.v[nu] - ab * c.v[nu] - bc * a.v[nu]);
}
// Tensor pseudo-particle, Eq. 23-26, literal reduction (reading c-2):
//   T^{alpha beta}(1..n) = (1/sqrt2) sum_k [J^alpha(1..k) J^beta(k+1..n) - (alpha <-> beta)]      (Eq. 25)
//   extra terms in Eq. 24 per split: (1/sqrt2) T(right)^{nu beta} J(left)_beta + (1/sqrt2) T(left)^{lambda nu} J(right)_lambda
template <class R> void tensor_build_add(const V4c<R>& a, const V4c<R>& b, T6c<R>& T) {
    for (int al = 0; al < 4; al++)
        for (int be = 0; be < 4; be++) T.t[al][be] += sqrt_half<R>() * (a.v[al] * b.v[be] - a.v[be] * b.v[al]);
}
template <class R>
void VT_add(const V4c<R>& left, const T6c<R>& Tleft, const V4c<R>& right, const T6c<R>& Tright, V4c<R>& out) {
    for (int nu = 0; nu < 4; nu++) {
        cx<R> s(0, 0);
        for (int be = 0; be < 4; be++) s += Tright.t[nu][be] * (metric<R>(be) * left.v[be]);
        for (int la = 0; la < 4; la++) s += Tleft.t[la][nu] * (metric<R>(la) * right.v[la]);
        out.v[nu] += sqrt_half<R>() * s;
    }
}

// ---- COBG: colour-ordered Berends-Giele recursion, Eq. 20 (V4 form) or Eq. 24-25 (tensor form), closed by
// Eq. 22.  mom[k], ext[k] are given IN THE ORDER of the colour ordering (k = 0..n-1).
// Reading g1: Eq. 22's "p^2_{1,n}" is the inverse propagator of the (n-1)-current: the last current is not
// divided by its P^2. -------------------------------------------------------------------------------------
template <class R>
cx<R> cobg_amplitude(int n, const V4r<R>* mom, const V4c<R>* ext, bool tensor_form) {
    const int m = n - 1;  // currents over legs 0..m-1
    static thread_local V4c<R> J[MAXN][MAXN];
    static thread_local T6c<R> T[MAXN][MAXN];
    static thread_local V4r<R> P[MAXN][MAXN];
    for (int i = 0; i < m; i++) {
        J[i][i] = ext[i];
        P[i][i] = mom[i];
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) T[i][i].t[a][b] = cx<R>(0, 0);
    }
    for (int len = 2; len <= m; len++)
        for (int i = 0; i + len <= m; i++) {
            int j = i + len - 1;
            for (int mu = 0; mu < 4; mu++) P[i][j].v[mu] = P[i][j - 1].v[mu] + mom[j].v[mu];
            V4c<R> acc;
            for (int mu = 0; mu < 4; mu++) acc.v[mu] = cx<R>(0, 0);
            T6c<R> tacc;
            for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) tacc.t[a][b] = cx<R>(0, 0);
            for (int k = i; k < j; k++) {
                V4c<R> t;
                V3(P[i][k], P[k + 1][j], J[i][k], J[k + 1][j], t);
                for (int mu = 0; mu < 4; mu++) acc.v[mu] += t.v[mu];
                if (tensor_form) {
                    VT_add(J[i][k], T[i][k], J[k + 1][j], T[k + 1][j], acc);
                    tensor_build_add(J[i][k], J[k + 1][j], tacc);
                }
            }
            if (!tensor_form)
                for (int k = i; k < j; k++)
                    for (int l = k + 1; l < j; l++) {
                        V4c<R> t;
                        V4(J[i][k], J[k + 1][l], J[l + 1][j], t);
                        for (int mu = 0; mu < 4; mu++) acc.v[mu] += t.v[mu];
                    }
            if (len < m) {
                R P2 = mdot(P[i][j], P[i][j]);
                for (int mu = 0; mu < 4; mu++) acc.v[mu] /= P2;
            }
            J[i][j] = acc;
            T[i][j] = tacc;
        }
    return mdot(ext[n - 1], J[0][m - 1]);
}

// amplitude for labels order[0..n-1] (0-based gluon labels) with helicity eigenvectors as external currents
template <class R>
cx<R> cobg_ordered(int n, const V4r<R>* mom, const int8_t* hel, const int* order, bool tensor_form) {
    V4r<R> pm[MAXN];
    V4c<R> ex[MAXN];
    for (int k = 0; k < n; k++) {
        pm[k] = mom[order[k]];
        polarisation(pm[k], hel[order[k]], ex[k]);
    }
    return cobg_amplitude(n, pm, ex, tensor_form);
}

// ---- Colour matrix, Eq. 17, literally from the definition ---------------------------
// Generators T^a = lambda^a/sqrt2 (Gell-Mann), so Tr(T^a T^b) = delta^ab; [T^a,T^b] = i f^{abc} T^c gives
// f^{abc} = -i Tr([T^a,T^b] T^c); F^a_{bc} = i f^{abc} (L117).  Orderings sigma run over the permutations of
// gluons 2..n-1 in lexicographic order.  (F..F) = i^{n-2} (f..f) with f real, and |i^{n-2}|^2 = 1, so the
// Gram matrix of the real products equals Eq. 17.
void structure_constants(double f[8][8][8]) {
    typedef std::complex<double> C;
    C lam[8][3][3];
    for (auto& l : lam) for (auto& r : l) for (auto& x : r) x = 0;
    const C I(0, 1);
    lam[0][0][1] = lam[0][1][0] = 1;
    lam[1][0][1] = -I; lam[1][1][0] = I;
    lam[2][0][0] = 1; lam[2][1][1] = -1;
    lam[3][0][2] = lam[3][2][0] = 1;
    lam[4][0][2] = -I; lam[4][2][0] = I;
    lam[5][1][2] = lam[5][2][1] = 1;
    lam[6][1][2] = -I; lam[6][2][1] = I;
    lam[7][0][0] = lam[7][1][1] = 1 / std::sqrt(3.0); lam[7][2][2] = -2 / std::sqrt(3.0);
    const double s = 1 / std::sqrt(2.0);
    for (int a = 0; a < 8; a++)
        for (int b = 0; b < 8; b++)
            for (int c = 0; c < 8; c++) {
                C tr = 0;
                for (int i = 0; i < 3; i++)
                    for (int j = 0; j < 3; j++)
                        for (int k = 0; k < 3; k++)
                            tr += (lam[a][i][j] * lam[b][j][k] - lam[b][i][j] * lam[a][j][k]) * lam[c][k][i];
                f[a][b][c] = (-I * tr * s * s * s).real();
            }
}

// C[(n-2)!][(n-2)!] row-major
void colour_matrix(int n, double* Cout) {
    double f[8][8][8];
    structure_constants(f);
    const int m = n - 2;
    std::vector<std::vector<int>> perms;
    std::vector<int> p(m);
    std::iota(p.begin(), p.end(), 0);
    do perms.push_back(p); while (std::next_permutation(p.begin(), p.end()));
    const int np = (int)perms.size();
    long long nassign = 1;
    for (int i = 0; i < m; i++) nassign *= 8;
    std::vector<double> Cacc((size_t)np * np, 0.0);
#pragma omp parallel
    {
        std::vector<double> Cloc((size_t)np * np, 0.0);
        std::vector<double> M((size_t)np * 64);
#pragma omp for schedule(dynamic, 16)
        for (long long as = 0; as < nassign; as++) {
            int a[MAXN];
            long long t = as;
            for (int i = 0; i < m; i++) { a[i] = (int)(t % 8); t /= 8; }
            for (int s = 0; s < np; s++) {
                // (f^{a_s0} f^{a_s1} ... )_{a1 an}: matrices (f^a)_{bc} = f[a][b][c]
                double cur[8][8], nxt[8][8];
                for (int b = 0; b < 8; b++) for (int c = 0; c < 8; c++) cur[b][c] = f[a[perms[s][0]]][b][c];
                for (int i = 1; i < m; i++) {
                    const int ai = a[perms[s][i]];
                    for (int b = 0; b < 8; b++)
                        for (int c = 0; c < 8; c++) {
                            double x = 0;
                            for (int d = 0; d < 8; d++) x += cur[b][d] * f[ai][d][c];
                            nxt[b][c] = x;
                        }
                    std::memcpy(cur, nxt, sizeof(cur));
                }
                std::memcpy(&M[(size_t)s * 64], cur, sizeof(cur));
            }
            for (int s = 0; s < np; s++)
                for (int s2 = 0; s2 < np; s2++) {
                    double x = 0;
                    for (int q = 0; q < 64; q++) x += M[(size_t)s * 64 + q] * M[(size_t)s2 * 64 + q];
                    Cloc[(size_t)s * np + s2] += x;
                }
        }
#pragma omp critical
        for (size_t i = 0; i < Cacc.size(); i++) Cacc[i] += Cloc[i];
    }
    for (size_t i = 0; i < Cacc.size(); i++) Cout[i] = Cacc[i];
}

// ---- Full-colour assembly, Eq. 15/16: A_sigma = A(1, sigma_2..sigma_{n-1}, n),
// w = sum_{sigma sigma'} C_{sigma sigma'} A_sigma A_sigma'^* for ONE helicity assignment -------------------
template <class R>
R cobg_full_colour(int n, const V4r<R>* mom, const int8_t* hel, const double* C, bool tensor_form,
                   cx<R>* amps_out /* may be null */) {
    const int m = n - 2;
    std::vector<int> p(m);
    std::iota(p.begin(), p.end(), 1);
    std::vector<cx<R>> A;
    do {
        int order[MAXN];
        order[0] = 0;
        for (int i = 0; i < m; i++) order[i + 1] = p[i];
        order[n - 1] = n - 1;
        A.push_back(cobg_ordered(n, mom, hel, order, tensor_form));
    } while (std::next_permutation(p.begin(), p.end()));
    const int np = (int)A.size();
    cx<R> w(0, 0);
    for (int s = 0; s < np; s++)
        for (int s2 = 0; s2 < np; s2++) w += R(C[(size_t)s * np + s2]) * A[s] * std::conj(A[s2]);
    if (amps_out) for (int s = 0; s < np; s++) amps_out[s] = A[s];
    return w.real();
}

// helicity sum, Eq. 4 / Eq. 16: all 2^n assignments
template <class R> R cobg_full_colour_helsum(int n, const V4r<R>* mom, const double* C, bool tensor_form) {
    R w = 0;
    for (int h = 0; h < (1 << n); h++) {
        int8_t hel[MAXN];
        for (int k = 0; k < n; k++) hel[k] = (h >> k) & 1 ? 1 : -1;
        w += cobg_full_colour(n, mom, hel, C, tensor_form, (cx<R>*)nullptr);
    }
    return w;
}

// ---- CDBG: colour-dressed recursion, Eq. 28-32, reading c-5: 3x3-matrix
// valued currents over subsets pi of {1..n-1}, ordered 2-splits, colour matrices multiplied in split order.
//   |pi|=1: J(pi)_{hg} = eps_k [h==i_k][g==j_k], T = 0
//   else  : J(pi)_{hg} += V3(P1,P2; J(pi1)_{hk}, J(pi2)_{kg}) + (1/sqrt2) T(pi2)_{kg}^{nu b} J(pi1)_{hk,b}
//                         + (1/sqrt2) T(pi1)_{hk}^{l nu} J(pi2)_{kg,l};   T(pi)_{hg} += (1/sqrt2)[J^a J^b - J^b J^a]
//           J(pi) /= P_pi^2 unless pi = {1..n-1}
//   A = sum_{hg} (eps_n . J({1..n-1})_{hg}) [g==i_n][h==j_n];  out = |A|^2
template <class R>
cx<R> cdbg_amplitude(int n, const V4r<R>* mom, const V4c<R>* ext, const int8_t* col /* [n][2], 1..3 */,
                     long long* live_splits /* may be null: counts (split, h,k,g) terms evaluated */,
                     R* cancel /* may be null: rho = |A| / sum over top-level ordered-split terms |eps_n . term| */) {
    const int m = n - 1;
    const int nsub = 1 << m;
    const int in = col[2 * (n - 1)] - 1, jn = col[2 * (n - 1) + 1] - 1;
    R sumabs = 0;
    struct Cur { V4c<R> J[3][3]; T6c<R> T[3][3]; bool nzJ[3][3]; bool nzT[3][3]; V4r<R> P; };
    std::vector<Cur> cur(nsub);
    long long live = 0;
    for (int pi = 1; pi < nsub; pi++) {
        Cur& c = cur[pi];
        for (int h = 0; h < 3; h++)
            for (int g = 0; g < 3; g++) {
                for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] = cx<R>(0, 0);
                for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) c.T[h][g].t[a][b] = cx<R>(0, 0);
                c.nzJ[h][g] = c.nzT[h][g] = false;
            }
        for (int mu = 0; mu < 4; mu++) c.P.v[mu] = 0;
        for (int k = 0; k < m; k++)
            if (pi >> k & 1) for (int mu = 0; mu < 4; mu++) c.P.v[mu] += mom[k].v[mu];
        if ((pi & (pi - 1)) == 0) {
            int k = __builtin_ctz(pi);
            c.J[col[2 * k] - 1][col[2 * k + 1] - 1] = ext[k];
            c.nzJ[col[2 * k] - 1][col[2 * k + 1] - 1] = true;
            continue;
        }
        // ordered splits pi = pi1 + pi2
        for (int p1 = (pi - 1) & pi; p1 > 0; p1 = (p1 - 1) & pi) {
            const int p2 = pi ^ p1;
            const Cur& c1 = cur[p1];
            const Cur& c2 = cur[p2];
            for (int h = 0; h < 3; h++)
                for (int k = 0; k < 3; k++)
                    for (int g = 0; g < 3; g++) {
                        if (!c1.nzJ[h][k] || !c2.nzJ[k][g]) continue;  // a zero input current gives a zero term
                        live++;
                        V4c<R> t;
                        V3(c1.P, c2.P, c1.J[h][k], c2.J[k][g], t);
                        VT_add(c1.J[h][k], c1.T[h][k], c2.J[k][g], c2.T[k][g], t);
                        for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] += t.v[mu];
                        if (pi == nsub - 1 && h == jn && g == in) sumabs += std::abs(mdot(ext[n - 1], t));
                        tensor_build_add(c1.J[h][k], c2.J[k][g], c.T[h][g]);
                        c.nzJ[h][g] = c.nzT[h][g] = true;
                    }
        }
        if (pi != nsub - 1) {
            R P2 = mdot(c.P, c.P);
            for (int h = 0; h < 3; h++)
                for (int g = 0; g < 3; g++)
                    if (c.nzJ[h][g]) for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] /= P2;
        }
    }
    if (live_splits) *live_splits = live;
    const cx<R> A = mdot(ext[n - 1], cur[nsub - 1].J[jn][in]);
    if (cancel) *cancel = sumabs > 0 ? std::abs(A) / sumabs : R(1);
    return A;
}

// ---- CDBG with general external states: the same recursion Eq. 28-32 with arbitrary external
// polarisation vectors ext[k] and arbitrary external 3x3 colour matrices X[k] (Eq. 14: the
// colour-helicity sub-amplitude is the amplitude contracted with one polarisation and one colour state per gluon).
//   |pi|=1: J({k})_{hg} = ext[k] X[k]_{hg};   closure: A = sum_{hg} (ext[n-1] . J({1..n-1})_{hg}) X[n-1]_{gh}
// Continuous sampling (Eq. 7, 9, 12): ext = cos(phi) e1 + sin(phi) e2, X_{hg} = etabar_h eta_g (the trace part of
// eta_i T^a_ij etabar_j T^a_hg = eta_g etabar_h - delta_hg (eta.etabar)/3 decouples - pinned).  Discrete colour flow
// (i_k, j_k) is X = e_{i_k j_k}, which must reproduce cdbg_amplitude - pinned.
template <class R>
cx<R> cdbg_amplitude_general(int n, const V4r<R>* mom, const V4c<R>* ext, const cx<R> (*X)[3][3]) {
    const int m = n - 1;
    const int nsub = 1 << m;
    struct Cur { V4c<R> J[3][3]; T6c<R> T[3][3]; V4r<R> P; };
    std::vector<Cur> cur(nsub);
    for (int pi = 1; pi < nsub; pi++) {
        Cur& c = cur[pi];
        for (int h = 0; h < 3; h++)
            for (int g = 0; g < 3; g++) {
                for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] = cx<R>(0, 0);
                for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) c.T[h][g].t[a][b] = cx<R>(0, 0);
            }
        for (int mu = 0; mu < 4; mu++) c.P.v[mu] = 0;
        for (int k = 0; k < m; k++)
            if (pi >> k & 1) for (int mu = 0; mu < 4; mu++) c.P.v[mu] += mom[k].v[mu];
        if ((pi & (pi - 1)) == 0) {
            const int k = __builtin_ctz(pi);
            for (int h = 0; h < 3; h++)
                for (int g = 0; g < 3; g++)
                    for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] = ext[k].v[mu] * X[k][h][g];
            continue;
        }
        for (int p1 = (pi - 1) & pi; p1 > 0; p1 = (p1 - 1) & pi) {   // ordered splits
            const int p2 = pi ^ p1;
            const Cur& c1 = cur[p1];
            const Cur& c2 = cur[p2];
            for (int h = 0; h < 3; h++)
                for (int k = 0; k < 3; k++)
                    for (int g = 0; g < 3; g++) {
                        V4c<R> t;
                        V3(c1.P, c2.P, c1.J[h][k], c2.J[k][g], t);
                        VT_add(c1.J[h][k], c1.T[h][k], c2.J[k][g], c2.T[k][g], t);
                        for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] += t.v[mu];
                        tensor_build_add(c1.J[h][k], c2.J[k][g], c.T[h][g]);
                    }
        }
        if (pi != nsub - 1) {
            const R P2 = mdot(c.P, c.P);
            for (int h = 0; h < 3; h++)
                for (int g = 0; g < 3; g++)
                    for (int mu = 0; mu < 4; mu++) c.J[h][g].v[mu] /= P2;
        }
    }
    cx<R> A(0, 0);
    for (int h = 0; h < 3; h++)
        for (int g = 0; g < 3; g++) A += mdot(ext[n - 1], cur[nsub - 1].J[h][g]) * X[n - 1][g][h];
    return A;
}

template <class R>
R cdbg_me2(int n, const V4r<R>* mom, const int8_t* hel, const int8_t* col, long long* live, double* rho) {
    V4c<R> ex[MAXN];
    for (int k = 0; k < n; k++) polarisation(mom[k], hel[k], ex[k]);
    R cancel = 1;
    const R r = std::norm(cdbg_amplitude(n, mom, ex, col, live, &cancel));
    if (rho) *rho = (double)cancel;
    return r;
}

// ---- Colour-flow decomposition, Eq. 19: the definition CDBG must equal.  Matrix-product
// convention (reading g5): an ordering (s_1..s_{n-1}, n) contributes when j_n = i_{s_1},
// j_{s_1} = i_{s_2}, ..., j_{s_{n-1}} = i_n.  Depth-first search over colour-connected orderings. ----------
template <class R>
void colour_flow_dfs(int n, const V4r<R>* mom, const int8_t* hel, const int8_t* col, int depth, int* order,
                     unsigned used, int last, cx<R>& sum, R& sumabs, long long& count) {
    const int m = n - 1;
    if (depth == m) {
        if (col[2 * last + 1] != col[2 * (n - 1)]) return;   // j_last = i_n
        order[m] = n - 1;
        const cx<R> a = cobg_ordered(n, mom, hel, order, false);
        sum += a;
        sumabs += std::abs(a);
        count++;
        return;
    }
    for (int k = 0; k < m; k++) {
        if (used >> k & 1) continue;
        if (col[2 * last + 1] != col[2 * k]) continue;       // j_prev = i_k
        order[depth] = k;
        colour_flow_dfs(n, mom, hel, col, depth + 1, order, used | (1u << k), k, sum, sumabs, count);
    }
}
template <class R>
R colour_flow_me2(int n, const V4r<R>* mom, const int8_t* hel, const int8_t* col, long long* cnt, double* rho) {
    cx<R> sum(0, 0);
    R sumabs = 0;
    long long count = 0;
    int order[MAXN];
    colour_flow_dfs(n, mom, hel, col, 0, order, 0u, n - 1, sum, sumabs, count);
    if (cnt) *cnt = count;
    if (rho) *rho = sumabs > 0 ? (double)(std::abs(sum) / sumabs) : 1.0;   // |sum_s A_s| / sum_s |A_s|
    return std::norm(sum);
}

template <class R> void load_mom(int n, const double* mom, V4r<R>* out) {
    for (int k = 0; k < n; k++) for (int mu = 0; mu < 4; mu++) out[k].v[mu] = R(mom[4 * k + mu]);
}

}  // namespace

// ======================================= C entry points (ctypes) ==========================================
// Arrays: mom[N][n][4] doubles (E,px,py,pz), hel[N][n] int8 (+1/-1), col[N][n][2] int8 in {1,2,3}; AoS.
// prec: 0 = double, 1 = long double.  All return 0 on success, -1 on bad arguments.
// Batched CDBG amplitude with general external states: ext [N][n][4][2] (re, im), X [N][n][3][3][2]; amp [N][2].
template <class R>
static void cdbg_general_one(int n, const double* mom, const double* ext, const double* X, double* amp) {
    V4r<R> pm[MAXN]; load_mom(n, mom, pm);
    V4c<R> ex[MAXN];
    cx<R> Xm[MAXN][3][3];
    for (int k = 0; k < n; k++) {
        for (int mu = 0; mu < 4; mu++) ex[k].v[mu] = cx<R>(ext[(k * 4 + mu) * 2], ext[(k * 4 + mu) * 2 + 1]);
        for (int h = 0; h < 3; h++)
            for (int g = 0; g < 3; g++) Xm[k][h][g] = cx<R>(X[((k * 3 + h) * 3 + g) * 2], X[((k * 3 + h) * 3 + g) * 2 + 1]);
    }
    const cx<R> A = cdbg_amplitude_general<R>(n, pm, ex, Xm);
    amp[0] = (double)A.real();
    amp[1] = (double)A.imag();
}

extern "C" {

int bgo_polarisation(const double* p, int lambda, double* eps_re_im /* [4][2] */) {
    V4r<double> pp;
    V4c<double> e;
    for (int mu = 0; mu < 4; mu++) pp.v[mu] = p[mu];
    polarisation(pp, lambda, e);
    for (int mu = 0; mu < 4; mu++) { eps_re_im[2 * mu] = e.v[mu].real(); eps_re_im[2 * mu + 1] = e.v[mu].imag(); }
    return 0;
}

// One colour-ordered amplitude for explicit external currents ext[n][4][2] (re,im), momenta in ordering order.
int bgo_cobg_amp_ext(int n, const double* mom, const double* ext, int tensor_form, int prec, double* out2) {
    if (n < 3 || n >= MAXN) return -1;
    if (prec == 0) {
        V4r<double> pm[MAXN]; V4c<double> ex[MAXN];
        load_mom(n, mom, pm);
        for (int k = 0; k < n; k++) for (int mu = 0; mu < 4; mu++) ex[k].v[mu] = {ext[(k * 4 + mu) * 2], ext[(k * 4 + mu) * 2 + 1]};
        auto a = cobg_amplitude(n, pm, ex, tensor_form != 0);
        out2[0] = a.real(); out2[1] = a.imag();
    } else {
        V4r<long double> pm[MAXN]; V4c<long double> ex[MAXN];
        load_mom(n, mom, pm);
        for (int k = 0; k < n; k++) for (int mu = 0; mu < 4; mu++) ex[k].v[mu] = {(long double)ext[(k * 4 + mu) * 2], (long double)ext[(k * 4 + mu) * 2 + 1]};
        auto a = cobg_amplitude(n, pm, ex, tensor_form != 0);
        out2[0] = (double)a.real(); out2[1] = (double)a.imag();
    }
    return 0;
}

// One colour-ordered helicity amplitude A(order[0],...,order[n-1]) (0-based labels) for one event.
int bgo_cobg_amp(int n, const double* mom, const signed char* hel, const int* order, int tensor_form, int prec,
                 double* out2) {
    if (n < 3 || n >= MAXN) return -1;
    if (prec == 0) {
        V4r<double> pm[MAXN]; load_mom(n, mom, pm);
        auto a = cobg_ordered(n, pm, (const int8_t*)hel, order, tensor_form != 0);
        out2[0] = a.real(); out2[1] = a.imag();
    } else {
        V4r<long double> pm[MAXN]; load_mom(n, mom, pm);
        auto a = cobg_ordered(n, pm, (const int8_t*)hel, order, tensor_form != 0);
        out2[0] = (double)a.real(); out2[1] = (double)a.imag();
    }
    return 0;
}

int bgo_colour_matrix(int n, double* C) {
    if (n < 4 || n > 8) return -1;
    colour_matrix(n, C);
    return 0;
}

// Batched full-colour |M|^2 (COBG + Eq. 16).  hel == NULL: helicity-summed.  amps (may be NULL):
// [N][(n-2)!][2] partial amplitudes (only for given helicities).  threads <= 0: OpenMP default.
int bgo_cobg_full_colour(int n, long long N, const double* mom, const signed char* hel, const double* C,
                         int tensor_form, int prec, int threads, double* out, double* amps) {
    if (n < 4 || n > 9) return -1;
    int np = 1;
    for (int i = 2; i <= n - 2; i++) np *= i;
#pragma omp parallel for schedule(dynamic, 4) num_threads(threads > 0 ? threads : omp_get_max_threads_wrapper())
    for (long long e = 0; e < N; e++) {
        if (prec == 0) {
            V4r<double> pm[MAXN]; load_mom(n, mom + (size_t)e * n * 4, pm);
            if (hel) {
                std::vector<cx<double>> A(np);
                out[e] = cobg_full_colour(n, pm, (const int8_t*)hel + (size_t)e * n, C, tensor_form != 0, A.data());
                if (amps) for (int s = 0; s < np; s++) { amps[((size_t)e * np + s) * 2] = A[s].real(); amps[((size_t)e * np + s) * 2 + 1] = A[s].imag(); }
            } else out[e] = cobg_full_colour_helsum(n, pm, C, tensor_form != 0);
        } else {
            V4r<long double> pm[MAXN]; load_mom(n, mom + (size_t)e * n * 4, pm);
            if (hel) {
                std::vector<cx<long double>> A(np);
                out[e] = (double)cobg_full_colour(n, pm, (const int8_t*)hel + (size_t)e * n, C, tensor_form != 0, A.data());
                if (amps) for (int s = 0; s < np; s++) { amps[((size_t)e * np + s) * 2] = (double)A[s].real(); amps[((size_t)e * np + s) * 2 + 1] = (double)A[s].imag(); }
            } else out[e] = (double)cobg_full_colour_helsum(n, pm, C, tensor_form != 0);
        }
    }
    return 0;
}

// Batched colour-dressed |A|^2 (CDBG).  live (may be NULL): [N] number of non-zero (split,h,k,g) terms.
int bgo_cdbg(int n, long long N, const double* mom, const signed char* hel, const signed char* col, int prec,
             int threads, double* out, long long* live, double* rho /* may be NULL: [N] cancellation ratio */) {
    if (n < 3 || n >= MAXN) return -1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(threads > 0 ? threads : omp_get_max_threads_wrapper())
    for (long long e = 0; e < N; e++) {
        long long lv = 0;
        if (prec == 0) {
            V4r<double> pm[MAXN]; load_mom(n, mom + (size_t)e * n * 4, pm);
            out[e] = cdbg_me2(n, pm, (const int8_t*)hel + (size_t)e * n, (const int8_t*)col + (size_t)e * n * 2, &lv, rho ? rho + e : nullptr);
        } else {
            V4r<long double> pm[MAXN]; load_mom(n, mom + (size_t)e * n * 4, pm);
            out[e] = (double)cdbg_me2(n, pm, (const int8_t*)hel + (size_t)e * n, (const int8_t*)col + (size_t)e * n * 2, &lv, rho ? rho + e : nullptr);
        }
        if (live) live[e] = lv;
    }
    return 0;
}

// Batched Eq. 19 brute force.  count (may be NULL): [N] number of colour-connected orderings.
int bgo_colour_flow(int n, long long N, const double* mom, const signed char* hel, const signed char* col,
                    int prec, int threads, double* out, long long* count,
                    double* rho /* may be NULL: [N] |sum A_sigma| / sum |A_sigma| over connected orderings */) {
    if (n < 3 || n >= MAXN) return -1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 0 ? threads : omp_get_max_threads_wrapper())
    for (long long e = 0; e < N; e++) {
        long long c = 0;
        if (prec == 0) {
            V4r<double> pm[MAXN]; load_mom(n, mom + (size_t)e * n * 4, pm);
            out[e] = colour_flow_me2(n, pm, (const int8_t*)hel + (size_t)e * n, (const int8_t*)col + (size_t)e * n * 2, &c, rho ? rho + e : nullptr);
        } else {
            V4r<long double> pm[MAXN]; load_mom(n, mom + (size_t)e * n * 4, pm);
            out[e] = (double)colour_flow_me2(n, pm, (const int8_t*)hel + (size_t)e * n, (const int8_t*)col + (size_t)e * n * 2, &c, rho ? rho + e : nullptr);
        }
        if (count) count[e] = c;
    }
    return 0;
}

int bgo_cdbg_general(int n, long long N, const double* mom, const double* ext, const double* X, int prec, int threads,
                     double* amp) {
    if (n < 3 || n >= MAXN) return -1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(threads > 0 ? threads : omp_get_max_threads_wrapper())
    for (long long e = 0; e < N; e++) {
        if (prec == 0) cdbg_general_one<double>(n, mom + (size_t)e * n * 4, ext + (size_t)e * n * 8, X + (size_t)e * n * 18, amp + 2 * e);
        else cdbg_general_one<long double>(n, mom + (size_t)e * n * 4, ext + (size_t)e * n * 8, X + (size_t)e * n * 18, amp + 2 * e);
    }
    return 0;
}

int bgo_max_threads(void) { return omp_get_max_threads_wrapper(); }

}  // extern "C"

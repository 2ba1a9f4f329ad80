// Generic kernels: one thread per event, runtime n (4..12), currents in global scratch (event-interleaved so
// that a warp's accesses to the same slot coalesce).  These are the first-correct path and the fallback for
// shapes the on-chip kernels do not cover; they mirror the paper's "all quantities in global memory" layout
// and are not the performance path.
#include "bg_internal.h"
#include "bg_math.cuh"

namespace bg {

// ---------------------------------------------------------------------------------------------------------
// CDBG, Eq. 28-32, colour-flow basis with discrete (i_k, j_k).
//
// A product of elementary matrices e_{ij} is a single elementary matrix, so the 3x3 colour matrix of a subset
// current J(pi) has at most one off-diagonal entry or up to three diagonal entries; which one follows from
// d_c = #{k in pi: i_k = c} - #{k in pi: j_k = c}:  d = e_h - e_g -> entry (h,g);  d = 0 -> diagonal; else dead.
// The pair of ordered splits (pi1,pi2), (pi2,pi1) of Eq. 29 shares one vertex value X(a,b) (V3 and the tensor
// terms are antisymmetric under exchange of the two legs): +X goes to entry (h1,g2) if g1 == h2 and -X to
// (h2,g1) if g2 == h1.
//
// type byte of a subset: 0x40 dead | 0x80|mask diagonal with live entries mask | (h<<2)|g single off-diagonal.
// slot of entry (h,g) of subset pi: pi*3 + (h == g ? h : 0); 20 doubles per slot (4 cx vector + 6 cx tensor).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool has_entry(unsigned t, int h, int g) {
    if (t & 0x80u) return h == g && ((t >> h) & 1u);
    if (t & 0x40u) return false;
    return t == (unsigned)((h << 2) | g);
}

struct GScratch {
    double* cur;     // [nsub*3][20][NC]
    double* P;       // [nsub][4][NC]
    uint8_t* type;   // [nsub][NC]
    long long NC;
};

__device__ __forceinline__ void load_entry(const GScratch& w, long long e, int slot, bool tensor, cx* J, cx* T) {
    const double* b = w.cur + (size_t)slot * 20 * w.NC + e;
#pragma unroll
    for (int c = 0; c < 4; c++) J[c] = mk(b[(size_t)(2 * c) * w.NC], b[(size_t)(2 * c + 1) * w.NC]);
    if (tensor) {
#pragma unroll
        for (int c = 0; c < 6; c++) T[c] = mk(b[(size_t)(8 + 2 * c) * w.NC], b[(size_t)(9 + 2 * c) * w.NC]);
    }
}

__global__ void __launch_bounds__(128)
cdbg_generic_kernel(int n, int helsum, long long N, long long first, long long count, const double* __restrict__ mom,
                    const signed char* __restrict__ hel, const signed char* __restrict__ col, double* __restrict__ out,
                    GScratch w) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= count) return;
    const long long ge = first + e;
    const int m = n - 1, nsub = 1 << m, full = nsub - 1;

    int ci[12], cj[12];
    int wk[12];
    for (int k = 0; k < n; k++) {
        ci[k] = col[(size_t)(2 * k) * N + ge] - 1;
        cj[k] = col[(size_t)(2 * k + 1) * N + ge] - 1;
        wk[k] = (1 << (8 * ci[k])) - (1 << (8 * cj[k]));
    }
    double pn[4];
    for (int c = 0; c < 4; c++) pn[c] = mom[(size_t)((n - 1) * 4 + c) * N + ge];

    double total = 0.0;
    const int nhel = helsum ? (1 << n) : 1;
    for (int hc = 0; hc < nhel; hc++) {
        // external currents
        for (int k = 0; k < m; k++) {
            double p[4];
            for (int c = 0; c < 4; c++) p[c] = mom[(size_t)(k * 4 + c) * N + ge];
            const int lam = helsum ? (((hc >> k) & 1) ? 1 : -1) : (int)hel[(size_t)k * N + ge];
            cx eps[4];
            polarisation(p, lam, eps);
            const int pi = 1 << k;
            const bool diag = ci[k] == cj[k];
            const int slot = pi * 3 + (diag ? ci[k] : 0);
            double* b = w.cur + (size_t)slot * 20 * w.NC + e;
            for (int c = 0; c < 4; c++) {
                b[(size_t)(2 * c) * w.NC] = eps[c].re;
                b[(size_t)(2 * c + 1) * w.NC] = eps[c].im;
                w.P[(size_t)(pi * 4 + c) * w.NC + e] = p[c];
            }
            w.type[(size_t)pi * w.NC + e] = diag ? (uint8_t)(0x80u | (1u << ci[k])) : (uint8_t)((ci[k] << 2) | cj[k]);
        }
        cx epsn[4];
        {
            const int lam = helsum ? (((hc >> (n - 1)) & 1) ? 1 : -1) : (int)hel[(size_t)(n - 1) * N + ge];
            polarisation(pn, lam, epsn);
        }
        cx amp = mk(0.0, 0.0);

        for (int pi = 3; pi <= full; pi++) {
            if ((pi & (pi - 1)) == 0) continue;
            const int low = pi & -pi, rest = pi ^ low;
            // momentum and colour charge of the subset
            double P[4];
            for (int c = 0; c < 4; c++) {
                P[c] = w.P[(size_t)(rest * 4 + c) * w.NC + e] + w.P[(size_t)(low * 4 + c) * w.NC + e];
                w.P[(size_t)(pi * 4 + c) * w.NC + e] = P[c];
            }
            int D = 0;
            for (int k = 0; k < m; k++)
                if ((pi >> k) & 1) D += wk[k];
            // candidate entries
            int cand_h[3], cand_g[3], ncand = 0;
            bool diag = false;
            if (D == 0) {
                diag = true;
                for (int h = 0; h < 3; h++) { cand_h[ncand] = h; cand_g[ncand] = h; ncand++; }
            } else {
                for (int h = 0; h < 3; h++)
                    for (int g = 0; g < 3; g++)
                        if (h != g && D == (1 << (8 * h)) - (1 << (8 * g))) { cand_h[0] = h; cand_g[0] = g; ncand = 1; }
            }
            if (pi == full) {
                // closure, Eq. 22: only the entry contracted with X_n = e_{i_n j_n} is needed
                const int h = cj[n - 1], g = ci[n - 1];
                bool ok = false;
                for (int c = 0; c < ncand; c++) ok = ok || (cand_h[c] == h && cand_g[c] == g);
                ncand = 0;
                if (ok) { cand_h[0] = h; cand_g[0] = g; ncand = 1; }
            }
            unsigned livemask = 0;
            for (int cd = 0; cd < ncand; cd++) {
                const int h = cand_h[cd], g = cand_g[cd];
                cx acc[4], tacc[6];
                for (int c = 0; c < 4; c++) acc[c] = mk(0.0, 0.0);
                for (int c = 0; c < 6; c++) tacc[c] = mk(0.0, 0.0);
                bool any = false;
                // unordered splits: pi1 contains the lowest gluon of pi
                for (int sub = (rest - 1) & rest;; sub = (sub - 1) & rest) {
                    const int p1 = low | sub, p2 = pi ^ p1;
                    const unsigned t1 = w.type[(size_t)p1 * w.NC + e], t2 = w.type[(size_t)p2 * w.NC + e];
                    {
                        if (!((t1 | t2) & 0x40u)) {
                            const bool ten1 = (p1 & (p1 - 1)) != 0, ten2 = (p2 & (p2 - 1)) != 0;
                            for (int k = 0; k < 3; k++) {
                                const bool fwd = has_entry(t1, h, k) && has_entry(t2, k, g);   // a=(h,k) in pi1, b=(k,g) in pi2
                                const bool bwd = has_entry(t2, h, k) && has_entry(t1, k, g);   // b=(h,k) in pi2, a=(k,g) in pi1
                                if (fwd && bwd && h == k && k == g) continue;                  // +X - X
                                for (int dir = 0; dir < 2; dir++) {
                                    if (dir == 0 ? !fwd : !bwd) continue;
                                    const int ah = dir == 0 ? h : k, ag = dir == 0 ? k : g;
                                    const int bh = dir == 0 ? k : h, bgc = dir == 0 ? g : k;
                                    const double sign = dir == 0 ? 1.0 : -1.0;
                                    cx a[4], b[4], Ta[6], Tb[6];
                                    load_entry(w, e, p1 * 3 + (ah == ag ? ah : 0), ten1, a, Ta);
                                    load_entry(w, e, p2 * 3 + (bh == bgc ? bh : 0), ten2, b, Tb);
                                    double P1[4], P2[4];
                                    for (int c = 0; c < 4; c++) {
                                        P1[c] = w.P[(size_t)(p1 * 4 + c) * w.NC + e];
                                        P2[c] = P[c] - P1[c];
                                    }
                                    v3_acc(acc, P1, P2, a, b, sign);
                                    if (ten2) tcontract_acc(acc, Tb, a, sign);
                                    if (ten1) tcontract_acc(acc, Ta, b, -sign);
                                    if (pi != full) tbuild_acc(tacc, a, b, sign);
                                    any = true;
                                }
                            }
                        }
                    }
                    if (sub == 0) break;
                }
                if (!any) continue;
                if (pi == full) {
                    amp = kInvSqrt2 * mdot(epsn, acc);
                } else {
                    const double f = kInvSqrt2 / mdot(P, P);
                    const int slot = pi * 3 + (h == g ? h : 0);
                    double* b = w.cur + (size_t)slot * 20 * w.NC + e;
                    for (int c = 0; c < 4; c++) {
                        b[(size_t)(2 * c) * w.NC] = f * acc[c].re;
                        b[(size_t)(2 * c + 1) * w.NC] = f * acc[c].im;
                    }
                    for (int c = 0; c < 6; c++) {
                        b[(size_t)(8 + 2 * c) * w.NC] = kInvSqrt2 * tacc[c].re;
                        b[(size_t)(9 + 2 * c) * w.NC] = kInvSqrt2 * tacc[c].im;
                    }
                    livemask |= diag ? (1u << h) : 1u;
                }
            }
            if (pi != full) {
                uint8_t t = 0x40u;
                if (livemask) t = diag ? (uint8_t)(0x80u | livemask) : (uint8_t)((cand_h[0] << 2) | cand_g[0]);
                w.type[(size_t)pi * w.NC + e] = t;
            }
        }
        total += amp.re * amp.re + amp.im * amp.im;
    }
    out[ge] = total;
}

size_t cdbg_generic_scratch_per_event(int n) {
    const size_t nsub = (size_t)1 << (n - 1);
    return nsub * 3 * 20 * sizeof(double) + nsub * 4 * sizeof(double) + nsub;
}

cudaError_t cdbg_generic_launch(cudaStream_t s, int n, bool helsum, long long N, long long first, long long count,
                                const double* mom, const signed char* hel, const signed char* col, double* out,
                                void* scratch) {
    const size_t nsub = (size_t)1 << (n - 1);
    GScratch w;
    w.NC = count;
    w.cur = (double*)scratch;
    w.P = w.cur + nsub * 3 * 20 * (size_t)count;
    w.type = (uint8_t*)(w.P + nsub * 4 * (size_t)count);
    const int threads = 128;
    const unsigned blocks = (unsigned)((count + threads - 1) / threads);
    cdbg_generic_kernel<<<blocks, threads, 0, s>>>(n, helsum ? 1 : 0, N, first, count, mom, hel, col, out, w);
    return cudaGetLastError();
}

}  // namespace bg

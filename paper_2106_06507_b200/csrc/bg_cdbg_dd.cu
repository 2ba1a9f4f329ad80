// Colour-dressed recursion (CDBG, Eq. 28-32, closed with Eq. 22) in double-double arithmetic:
// one thread per event, currents in global scratch, the same subset walk and colour bookkeeping as
// bg_generic.cu.  This is the precision reference on the GPU (BG_OPT_PRECISION = 1): single-colour-flow amplitudes
// have near-zeros by cancellation where FP64 round-off exceeds 1e-11; evaluated with
// ~106-bit significands the same inputs reproduce the extended-precision oracle on every event, which shows that
// what is left in the FP64 kernels is rounding, not arithmetic.  Not a performance path.
#include <algorithm>

#include "bg_ddmath.cuh"
#include "bg_internal.h"

namespace bg {

namespace {

__device__ __forceinline__ bool has_entry_dd(unsigned t, int h, int g) {
    if (t & 0x80u) return h == g && ((t >> h) & 1u);
    if (t & 0x40u) return false;
    return t == (unsigned)((h << 2) | g);
}

using C = cxt<dd>;

struct DScratch {
    double2* cur;    // [nsub*3][20][NC]  (hi, lo)
    double2* P;      // [nsub][4][NC]
    uint8_t* type;   // [nsub][NC]
    long long NC;
};

__device__ __forceinline__ dd ld_dd(const double2* p) { const double2 v = *p; return mkdd(v.x, v.y); }
__device__ __forceinline__ void st_dd(double2* p, dd v) { *p = make_double2(v.hi, v.lo); }

__device__ __forceinline__ void load_entry_dd(const DScratch& w, long long e, int slot, bool tensor, C* J, C* T) {
    const double2* b = w.cur + (size_t)slot * 20 * w.NC + e;
    for (int c = 0; c < 4; c++) J[c] = mkc<dd>(ld_dd(b + (size_t)(2 * c) * w.NC), ld_dd(b + (size_t)(2 * c + 1) * w.NC));
    if (tensor)
        for (int c = 0; c < 6; c++)
            T[c] = mkc<dd>(ld_dd(b + (size_t)(8 + 2 * c) * w.NC), ld_dd(b + (size_t)(9 + 2 * c) * w.NC));
}

}  // namespace

__global__ void __launch_bounds__(128)
cdbg_dd_kernel(int n, long long N, long long first, long long count, const double* __restrict__ mom,
               const signed char* __restrict__ hel, const signed char* __restrict__ col, double* __restrict__ out,
               DScratch w) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= count) return;
    const long long ge = first + e;
    const int m = n - 1, nsub = 1 << m, full = nsub - 1;
    const dd zero = mkdd(0.0);
    const dd inv_sqrt2 = mkdd(1.0) / sqrt(mkdd(2.0));

    int ci[12], cj[12], wk[12];
    for (int k = 0; k < n; k++) {
        ci[k] = col[(size_t)(2 * k) * N + ge] - 1;
        cj[k] = col[(size_t)(2 * k + 1) * N + ge] - 1;
        wk[k] = (1 << (8 * ci[k])) - (1 << (8 * cj[k]));
    }
    // external currents
    for (int k = 0; k < m; k++) {
        dd p[4];
        for (int c = 0; c < 4; c++) p[c] = mkdd(mom[(size_t)(k * 4 + c) * N + ge]);
        C eps[4];
        polarisation_t<dd>(p, (int)hel[(size_t)k * N + ge], eps);
        const int pi = 1 << k;
        const bool diag = ci[k] == cj[k];
        const int slot = pi * 3 + (diag ? ci[k] : 0);
        double2* b = w.cur + (size_t)slot * 20 * w.NC + e;
        for (int c = 0; c < 4; c++) {
            st_dd(b + (size_t)(2 * c) * w.NC, eps[c].re);
            st_dd(b + (size_t)(2 * c + 1) * w.NC, eps[c].im);
            st_dd(w.P + (size_t)(pi * 4 + c) * w.NC + e, p[c]);
        }
        w.type[(size_t)pi * w.NC + e] = diag ? (uint8_t)(0x80u | (1u << ci[k])) : (uint8_t)((ci[k] << 2) | cj[k]);
    }
    C epsn[4];
    {
        dd pn[4];
        for (int c = 0; c < 4; c++) pn[c] = mkdd(mom[(size_t)((n - 1) * 4 + c) * N + ge]);
        polarisation_t<dd>(pn, (int)hel[(size_t)(n - 1) * N + ge], epsn);
    }
    C amp = mkc<dd>(zero, zero);

    for (int pi = 3; pi <= full; pi++) {
        if ((pi & (pi - 1)) == 0) continue;
        const int low = pi & -pi, rest = pi ^ low;
        dd P[4];
        for (int c = 0; c < 4; c++) {
            P[c] = ld_dd(w.P + (size_t)(rest * 4 + c) * w.NC + e) + ld_dd(w.P + (size_t)(low * 4 + c) * w.NC + e);
            st_dd(w.P + (size_t)(pi * 4 + c) * w.NC + e, P[c]);
        }
        int D = 0;
        for (int k = 0; k < m; k++)
            if ((pi >> k) & 1) D += wk[k];
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
            const int h = cj[n - 1], g = ci[n - 1];
            bool ok = false;
            for (int c = 0; c < ncand; c++) ok = ok || (cand_h[c] == h && cand_g[c] == g);
            ncand = 0;
            if (ok) { cand_h[0] = h; cand_g[0] = g; ncand = 1; }
        }
        unsigned livemask = 0;
        for (int cd = 0; cd < ncand; cd++) {
            const int h = cand_h[cd], g = cand_g[cd];
            C acc[4], tacc[6];
            for (int c = 0; c < 4; c++) acc[c] = mkc<dd>(zero, zero);
            for (int c = 0; c < 6; c++) tacc[c] = mkc<dd>(zero, zero);
            bool any = false;
            for (int sub = (rest - 1) & rest;; sub = (sub - 1) & rest) {
                const int p1 = low | sub, p2 = pi ^ p1;
                const unsigned t1 = w.type[(size_t)p1 * w.NC + e], t2 = w.type[(size_t)p2 * w.NC + e];
                if (!((t1 | t2) & 0x40u)) {
                    const bool ten1 = (p1 & (p1 - 1)) != 0, ten2 = (p2 & (p2 - 1)) != 0;
                    for (int k = 0; k < 3; k++) {
                        const bool fwd = has_entry_dd(t1, h, k) && has_entry_dd(t2, k, g);
                        const bool bwd = has_entry_dd(t2, h, k) && has_entry_dd(t1, k, g);
                        if (fwd && bwd && h == k && k == g) continue;   // +X - X
                        for (int dir = 0; dir < 2; dir++) {
                            if (dir == 0 ? !fwd : !bwd) continue;
                            const int ah = dir == 0 ? h : k, ag = dir == 0 ? k : g;
                            const int bh = dir == 0 ? k : h, bgc = dir == 0 ? g : k;
                            const bool neg = dir == 1;
                            C a[4], b[4], Ta[6], Tb[6];
                            load_entry_dd(w, e, p1 * 3 + (ah == ag ? ah : 0), ten1, a, Ta);
                            load_entry_dd(w, e, p2 * 3 + (bh == bgc ? bh : 0), ten2, b, Tb);
                            dd P1[4], P2[4];
                            for (int c = 0; c < 4; c++) {
                                P1[c] = ld_dd(w.P + (size_t)(p1 * 4 + c) * w.NC + e);
                                P2[c] = P[c] - P1[c];
                            }
                            v3_acc_t<dd>(acc, P1, P2, a, b, neg);
                            if (ten2) tcontract_acc_t<dd>(acc, Tb, a, neg);
                            if (ten1) tcontract_acc_t<dd>(acc, Ta, b, !neg);
                            if (pi != full) tbuild_acc_t<dd>(tacc, a, b, neg);
                            any = true;
                        }
                    }
                }
                if (sub == 0) break;
            }
            if (!any) continue;
            if (pi == full) {
                amp = inv_sqrt2 * mdot_t<dd>(epsn, acc);
            } else {
                const dd f = inv_sqrt2 / mdot_t<dd>(P, P);
                const int slot = pi * 3 + (h == g ? h : 0);
                double2* b = w.cur + (size_t)slot * 20 * w.NC + e;
                for (int c = 0; c < 4; c++) {
                    st_dd(b + (size_t)(2 * c) * w.NC, f * acc[c].re);
                    st_dd(b + (size_t)(2 * c + 1) * w.NC, f * acc[c].im);
                }
                for (int c = 0; c < 6; c++) {
                    st_dd(b + (size_t)(8 + 2 * c) * w.NC, inv_sqrt2 * tacc[c].re);
                    st_dd(b + (size_t)(9 + 2 * c) * w.NC, inv_sqrt2 * tacc[c].im);
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
    out[ge] = to_double(amp.re * amp.re + amp.im * amp.im);
}

size_t cdbg_dd_scratch_per_event(int n) {
    const size_t nsub = (size_t)1 << (n - 1);
    return nsub * 3 * 20 * sizeof(double2) + nsub * 4 * sizeof(double2) + nsub;
}

cudaError_t cdbg_dd_launch(cudaStream_t s, int n, long long N, long long first, long long count, const double* mom,
                           const signed char* hel, const signed char* col, double* out, void* scratch) {
    const size_t nsub = (size_t)1 << (n - 1);
    DScratch w;
    w.NC = count;
    w.cur = (double2*)scratch;
    w.P = w.cur + nsub * 3 * 20 * (size_t)count;
    w.type = (uint8_t*)(w.P + nsub * 4 * (size_t)count);
    const int threads = 128;
    const unsigned blocks = (unsigned)((count + threads - 1) / threads);
    cdbg_dd_kernel<<<blocks, threads, 0, s>>>(n, N, first, count, mom, hel, col, out, w);
    return cudaGetLastError();
}

}  // namespace bg

// ---------------------------------------------------------------------------------------------------------
// Colour-ordered recursion (Eq. 20-22) and full-colour form (Eq. 16) in double-double:
// kernel 1 - one thread per (event, helicity assignment, ordering): triangular current table, A_sigma to scratch;
// kernel 2 - one thread per event: sum over helicity assignments of  sum_{s s'} C_{s s'} A_s A_s'^*.
// ---------------------------------------------------------------------------------------------------------
namespace bg {

namespace {
constexpr int kDdMaxN = 8;
__device__ __forceinline__ int tri_dd(int i, int j) { return j * (j + 1) / 2 + i; }   // i <= j
}  // namespace

// A(1, sigma_s(2..n-1), n) of event e in double-double arithmetic (Eq. 20 + 22); hc >= 0: helicity assignment from
// the bits of hc, else from hel.
__device__ C cobg_dd_amplitude(int n, int nperm, int s, int hc, long long N, long long e, const double* __restrict__ mom,
                               const signed char* __restrict__ hel) {
    const int m = n - 1, mm = n - 2;
    // s-th permutation of gluons 2..n-1 (0-based labels 1..n-2) in lexicographic order
    int avail[kDdMaxN], order[kDdMaxN];
    for (int i = 0; i < mm; i++) avail[i] = i + 1;
    int rem = s, fact = nperm;
    order[0] = 0;
    for (int i = 0; i < mm; i++) {
        fact /= (mm - i);
        const int d = rem / fact;
        rem -= d * fact;
        order[i + 1] = avail[d];
        for (int q = d; q < mm - i - 1; q++) avail[q] = avail[q + 1];
    }
    order[n - 1] = n - 1;
    C J[kDdMaxN * (kDdMaxN - 1) / 2][4];
    dd P[kDdMaxN * (kDdMaxN - 1) / 2][4];
    C epsn[4];
    for (int i = 0; i < n; i++) {
        const int g = order[i];
        dd p[4];
        for (int c = 0; c < 4; c++) p[c] = mkdd(mom[(size_t)(g * 4 + c) * N + e]);
        const int lam = hc >= 0 ? (((hc >> g) & 1) ? 1 : -1) : (int)hel[(size_t)g * N + e];
        if (i < m) {
            polarisation_t<dd>(p, lam, J[tri_dd(i, i)]);
            for (int c = 0; c < 4; c++) P[tri_dd(i, i)][c] = p[c];
        } else {
            polarisation_t<dd>(p, lam, epsn);
        }
    }
    const dd inv_sqrt2 = mkdd(1.0) / sqrt(mkdd(2.0)), half = mkdd(0.5), zero = mkdd(0.0), two = mkdd(2.0);
    for (int len = 2; len <= m; len++)
        for (int i = 0; i + len <= m; i++) {
            const int j = i + len - 1;
            for (int c = 0; c < 4; c++) P[tri_dd(i, j)][c] = dd_add(P[tri_dd(i, j - 1)][c], P[tri_dd(j, j)][c]);
            C s3[4], s4[4];
            for (int c = 0; c < 4; c++) { s3[c] = mkc<dd>(zero, zero); s4[c] = mkc<dd>(zero, zero); }
            for (int k = i; k < j; k++) {
                const C* a = J[tri_dd(i, k)];
                v3_acc(s3, P[tri_dd(i, k)], P[tri_dd(k + 1, j)], a, J[tri_dd(k + 1, j)], 1.0);   // fused dd multiply-adds (bg_ddmath.cuh)
                for (int l = k + 1; l < j; l++) {
                    // 2 V4(a,b,c) = 2 (a.c) b - (a.b) c - (b.c) a   (Eq. 21, second line)
                    const C* b = J[tri_dd(k + 1, l)];
                    const C* c3 = J[tri_dd(l + 1, j)];
                    const C ac = cxd_scale(two, mdot(a, c3)), ab = mdot(a, b), bc = mdot(b, c3);
                    for (int nu = 0; nu < 4; nu++) {
                        cfma(s4[nu], ac, b[nu]);
                        cfms(s4[nu], ab, c3[nu]);
                        cfms(s4[nu], bc, a[nu]);
                    }
                }
            }
            for (int nu = 0; nu < 4; nu++) cxd_renorm(s4[nu]);      // (multiply-adds leave their accumulator unnormalised)
            dd f3 = inv_sqrt2, f4 = half;
            if (len < m) {
                const dd ip2 = mkdd(1.0) / mdot(P[tri_dd(i, j)], P[tri_dd(i, j)]);
                f3 = dd_mul(f3, ip2); f4 = dd_mul(f4, ip2);
            }
            for (int c = 0; c < 4; c++) J[tri_dd(i, j)][c] = cxd_add(cxd_scale(f3, s3[c]), cxd_scale(f4, s4[c]));
        }
    return mdot(epsn, J[tri_dd(0, m - 1)]);
}

__global__ void __launch_bounds__(64)
cobg_dd_amp_kernel(int n, int nhel, int nperm, long long N, long long first, long long count,
                   const double* __restrict__ mom, const signed char* __restrict__ hel, double2* __restrict__ amps) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= count * nhel * nperm) return;
    const int s = (int)(idx % nperm);
    const int hc = (int)((idx / nperm) % nhel);
    const long long e = first + idx / ((long long)nperm * nhel);
    const C A = cobg_dd_amplitude(n, nperm, s, nhel > 1 ? hc : -1, N, e, mom, hel);
    double2* o = amps + idx * 2;
    o[0] = make_double2(A.re.hi, A.re.lo);
    o[1] = make_double2(A.im.hi, A.im.lo);
}

// Re-evaluation of the events the FP64 kernel flagged (BG_OPT_PRECISION = 2, given helicities): one block per listed
// event, one thread per ordering; the amplitudes stay in shared memory and thread s takes row s of Eq. 16.
__global__ void __launch_bounds__(128)
cobg_dd_flagged_kernel(int n, int nperm, long long N, const uint32_t* __restrict__ list, const uint32_t* __restrict__ count,
                       const double* __restrict__ mom, const signed char* __restrict__ hel, const double* __restrict__ Cm,
                       double* __restrict__ out) {
    extern __shared__ double2 sh_amp[];   // [nperm][2]: (re.hi, re.lo), (im.hi, im.lo); reused for the row sums
    const uint32_t total = *count;
    for (uint32_t it = blockIdx.x; it < total; it += gridDim.x) {
        const long long e = list[it];
        __syncthreads();
        for (int s = threadIdx.x; s < nperm; s += blockDim.x) {       // (n = 8: 720 orderings in rounds of 128)
            const C A = cobg_dd_amplitude(n, nperm, s, -1, N, e, mom, hel);
            sh_amp[2 * s] = make_double2(A.re.hi, A.re.lo);
            sh_amp[2 * s + 1] = make_double2(A.im.hi, A.im.lo);
        }
        __syncthreads();
        dd mine = mkdd(0.0);
        for (int s = threadIdx.x; s < nperm; s += blockDim.x) {
            dd tr = mkdd(0.0), ti = mkdd(0.0);
            for (int s2 = 0; s2 < nperm; s2++) {
                const dd c = mkdd(Cm[(size_t)s * nperm + s2]);
                dd_fma(tr, c, mkdd(sh_amp[2 * s2].x, sh_amp[2 * s2].y));
                dd_fma(ti, c, mkdd(sh_amp[2 * s2 + 1].x, sh_amp[2 * s2 + 1].y));
            }
            dd_renorm(tr);
            dd_renorm(ti);
            dd_fma(mine, mkdd(sh_amp[2 * s].x, sh_amp[2 * s].y), tr);
            dd_fma(mine, mkdd(sh_amp[2 * s + 1].x, sh_amp[2 * s + 1].y), ti);
        }
        dd_renorm(mine);
        __syncthreads();
        sh_amp[threadIdx.x] = make_double2(mine.hi, mine.lo);
        __syncthreads();
        if (threadIdx.x == 0) {
            dd sum = mkdd(0.0);
            for (int s2 = 0; s2 < (int)blockDim.x; s2++) sum = sum + mkdd(sh_amp[s2].x, sh_amp[s2].y);
            out[e] = to_double(sum);
        }
    }
}

__global__ void __launch_bounds__(64)
cobg_dd_colour_kernel(int nhel, int nperm, long long first, long long count, const double* __restrict__ Cm,
                      const double2* __restrict__ amps, double* __restrict__ out) {
    const long long el = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (el >= count) return;
    dd total = mkdd(0.0);
    for (int hc = 0; hc < nhel; hc++) {
        const double2* a = amps + (el * nhel + hc) * (long long)nperm * 2;
        for (int s = 0; s < nperm; s++) {
            dd tr = mkdd(0.0), ti = mkdd(0.0);
            for (int s2 = 0; s2 < nperm; s2++) {
                const dd c = mkdd(Cm[(size_t)s * nperm + s2]);
                tr = tr + c * mkdd(a[2 * s2].x, a[2 * s2].y);
                ti = ti + c * mkdd(a[2 * s2 + 1].x, a[2 * s2 + 1].y);
            }
            total = total + mkdd(a[2 * s].x, a[2 * s].y) * tr + mkdd(a[2 * s + 1].x, a[2 * s + 1].y) * ti;
        }
    }
    out[first + el] = to_double(total);
}

cudaError_t cobg_dd_flagged_launch(cudaStream_t s, int n, int nperm, const double* dC, long long N, const uint32_t* list,
                                   const uint32_t* count, int blocks, const double* mom, const signed char* hel, double* out) {
    const int threads = std::min(128, (nperm + 31) / 32 * 32);
    cobg_dd_flagged_kernel<<<blocks, threads, (size_t)std::max(nperm * 2, threads) * sizeof(double2), s>>>(n, nperm, N, list, count, mom, hel, dC, out);
    return cudaGetLastError();
}

size_t cobg_dd_scratch_per_event(int n, bool helsum) {
    size_t np = 1;
    for (int i = 2; i <= n - 2; i++) np *= i;
    return np * (helsum ? ((size_t)1 << n) : 1) * 2 * sizeof(double2);
}

cudaError_t cobg_dd_launch(cudaStream_t s, int n, bool helsum, int nperm, const double* dC, long long N, long long first,
                           long long count, const double* mom, const signed char* hel, double* out, void* scratch) {
    const int nhel = helsum ? (1 << n) : 1;
    const long long threads = count * nhel * nperm;
    cobg_dd_amp_kernel<<<(unsigned)((threads + 63) / 64), 64, 0, s>>>(n, nhel, nperm, N, first, count, mom, hel,
                                                                      (double2*)scratch);
    cobg_dd_colour_kernel<<<(unsigned)((count + 63) / 64), 64, 0, s>>>(nhel, nperm, first, count, dC, (const double2*)scratch,
                                                                       out);
    return cudaGetLastError();
}

}  // namespace bg

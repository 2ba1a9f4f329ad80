// Colour-ordered recursion (COBG, Eq. 20-22) for all (n-2)! orderings A(1, sigma, n) of one
// event, followed by the full-colour quadratic form of Eq. 16 (L119-127) - the performance path of BASELINE
// configs 1 and 3.
//
// The (n-2)! orderings of one event share their short sub-currents: J(g_i .. g_j) depends only on the ordered
// sequence of gluons, not on the ordering it sits in (651 distinct sequences against 120 x 21 = 2520 ranges at
// n = 7).  A group of TPE threads works on one event:
//   * "shared" currents - sequences of length <= n-3 - are computed once, one thread per sequence, level by level,
//     into shared memory (291 x 64 B = 18.2 KB at n = 7);
//   * the two currents of length n-2 and the final one of length n-1 of every ordering are used by that ordering
//     only, so thread sigma computes them in registers (13 V3 + 22 V4 at n = 7) from the shared ones and closes
//     with eps_n (Eq. 22: the last current keeps no propagator);
//   * A_sigma goes to shared memory and thread sigma takes row sigma of  w = a_r^T C a_r + a_i^T C a_i  (C of
//     Eq. 17 is real and symmetric, so consecutive threads read consecutive addresses of a column).
// The amplitudes never leave the SM.  Which sequence lives in which slot is tabulated on the host at bg_init
// (integer bookkeeping, same for every event).
#include <algorithm>
#include <cstring>
#include <map>
#include <new>
#include <numeric>
#include <vector>

#include "bg_internal.h"
#include "bg_math.cuh"

namespace bg {

constexpr int kCobgMaxM = 7;   // n - 1 <= 7: n = 4..8
constexpr int kCobgMaxVals = 64;   // distinct entries of the colour matrix held in shared memory (16 at n = 7, 38 at n = 8)

struct CobgTable {
    int n, np, nslots;
    int level_begin[kCobgMaxM + 2];   // level L (sequence length) occupies lower[level_begin[L] .. level_begin[L+1])
    uint16_t* d_slot;                 // [np][m][m] slot of range (i..j) of ordering sigma; 0xFFFF if longer than n-3
    uint8_t* d_ord;                   // [np][m] gluon at position i of (1, sigma)  (0-based labels, position 0 = gluon 0)
    uint32_t* d_lower;                // representatives of the shared sequences: sigma << 8 | i << 4 | j
    uint32_t* d_cidx4;                // compressed colour matrix: [ceil(np/4)][np] words, byte u = index of C[4q+u][sigma] in cval
    int nval;                         // number of distinct entries of C (0: no compressed form)
    double cval[kCobgMaxVals];
};

struct CobgParams {
    int n, np, nslots, helsum;
    double lc_factor;                 // N_c^(n-2) (N_c^2 - 1)
    int lc;                           // leading colour (Eq. 33): sum |A|^2 over all (n-1)! orderings, no colour matrix
    long long N;
    const double* mom;
    const signed char* hel;
    const double* C;
    double* out;
    const uint16_t* slot;
    const uint8_t* ord;
    const uint32_t* lower;
    int level_begin[kCobgMaxM + 2];
    const uint32_t* cidx4;            // compressed colour matrix (nval > 0), else C is read as doubles
    int nval;
    double cval[kCobgMaxVals];
    // conditioning flag (given helicities, full colour; BG_OPT_PRECISION = 2): Ward residual of the closing currents
    double tau2;                      // 0: off; < 0: diagnostic, `out` receives the residual
    uint32_t* flag_list;              // [N] event ids
    uint32_t* flag_count;             // [1]
    // cascade (as the colour-dressed path): events whose residual lies between tau and tau_twin are evaluated
    // once more in FP64 in the rotated frame (twin bit 0) and compared with out[e] (twin bit 1)
    int twin;
    double tw2, td;                   // tau_twin^2 for the residuals, tau_twin for |w - w'| / w
    uint32_t* soft_list;              // [N] first stage: events for the second stage
    uint32_t* soft_count;             // [1]
    const uint32_t* list;             // second stage: the events to evaluate (nullptr: all N)
    const uint32_t* list_count;
};


// ---------------------------------------------------------------------------------------------------------
// device side
// ---------------------------------------------------------------------------------------------------------
constexpr int kSlotStride = 5;   // complex doubles between slots: 4 of data + 1 of padding (odd: spreads the bank groups)

__device__ __forceinline__ void lds_cur(const double* cur, int slot, cx* v) {
    const double2* p = reinterpret_cast<const double2*>(cur + (size_t)slot * (2 * kSlotStride));
#pragma unroll
    for (int c = 0; c < 4; c++) { const double2 t = p[c]; v[c] = mk(t.x, t.y); }
}
__device__ __forceinline__ void sts_cur(double* cur, int slot, const cx* v) {
    double2* p = reinterpret_cast<double2*>(cur + (size_t)slot * (2 * kSlotStride));
#pragma unroll
    for (int c = 0; c < 4; c++) p[c] = make_double2(v[c].re, v[c].im);
}

// Per-ordering view used by the register-resident top of the recursion: sl[i*M+j] = shared slot of range (i..j),
// pm[k] = OR of the gluon bits at positions 0..k-1, JA / JB = the two currents of length M-1 (positions 1..M-1 and
// 0..M-2) once they exist.
template <int NG>
struct TopView {
    static constexpr int M = NG - 1, LS = NG - 3;
    const double* cur;
    const double* P;
    uint16_t sl[M * M];
    unsigned pm[M + 1];
    cx JA[4], JB[4];

    template <int I, int J>
    __device__ __forceinline__ void fetch(cx* v) const {
        if (J - I + 1 <= LS) {
            lds_cur(cur, sl[I * M + J], v);
        } else if (I == 0) {
#pragma unroll
            for (int c = 0; c < 4; c++) v[c] = JB[c];
        } else {
#pragma unroll
            for (int c = 0; c < 4; c++) v[c] = JA[c];
        }
    }
    template <int I, int J>
    __device__ __forceinline__ const double* mom() const { return P + 4 * (pm[J + 1] ^ pm[I]); }

    template <int I, int K, int L, int J>
    __device__ __forceinline__ void v4_inner(cx* s4, const cx* a) const {
        if constexpr (L < J) {
            asm volatile("" ::: "memory");   // keep the operand loads of later vertices from being hoisted (registers)
            cx b[4], c[4];
            fetch<K + 1, L>(b);
            fetch<L + 1, J>(c);
            v4_acc(s4, a, b, c);
            v4_inner<I, K, L + 1, J>(s4, a);
        }
    }
    template <int I, int K, int J>
    __device__ __forceinline__ void splits(cx* s3, cx* s4) const {
        if constexpr (K < J) {
            asm volatile("" ::: "memory");
            cx a[4], b[4];
            fetch<I, K>(a);
            fetch<K + 1, J>(b);
            v3_acc(s3, mom<I, K>(), mom<K + 1, J>(), a, b, 1.0);
            v4_inner<I, K, K + 1, J>(s4, a);
            splits<I, K + 1, J>(s3, s4);
        }
    }
    // Eq. 20 for the range (I..J); PROP = false keeps the inverse propagator (last current, Eq. 22)
    template <int I, int J, bool PROP>
    __device__ __forceinline__ void range(cx* out) const {
        cx s3[4], s4[4];
#pragma unroll
        for (int c = 0; c < 4; c++) { s3[c] = mk(0.0, 0.0); s4[c] = mk(0.0, 0.0); }
        splits<I, I, J>(s3, s4);
        double f3 = kInvSqrt2, f4 = 0.5;
        if (PROP) {
            const double* Pr = mom<I, J>();
            const double ip2 = 1.0 / mdot(Pr, Pr);
            f3 *= ip2; f4 *= ip2;
        }
#pragma unroll
        for (int c = 0; c < 4; c++) out[c] = f3 * s3[c] + f4 * s4[c];
    }
};

// TPE threads per event in blocks of max(128, TPE) threads; with more orderings than threads (n = 8: 720 orderings,
// 256 threads) a thread takes the orderings t, t + TPE, .. in rounds.
template <int NG, int TPE, bool LC>
__global__ void __launch_bounds__(TPE > 128 ? TPE : 128, TPE > 128 ? 1 : 4) cobg_shared_kernel(const CobgParams p) {
    constexpr int BLOCK = TPE > 128 ? TPE : 128;
    constexpr int M = NG - 1, LS = NG - 3, EPB = BLOCK / TPE, NSUB = 1 << M;
    extern __shared__ double smem_d[];
    const int evl = threadIdx.x / TPE, t = threadIdx.x % TPE;
    const int np = p.np;
    // per-event shared block: currents | subset momenta | eps_n | amplitudes | reduction scratch
    const int ev_doubles = p.nslots * 2 * kSlotStride + NSUB * 4 + 8 + np * 2 + 16;
    double* cur = smem_d + (size_t)evl * ev_doubles;
    double* P = cur + p.nslots * 2 * kSlotStride;
    double* epsn = P + NSUB * 4;
    double* A = epsn + 8;
    double* red = A + np * 2;
    // Eq. 17's matrix has few distinct entries (C_ss' = C_{e, s^-1 s'}: those of one row; 16 at n = 7): the form
    // below reads one byte per entry (four per load, one L1 line per row of C instead of eight) and looks the value
    // up here - 32 doubles span the 32 banks once, so any mix of indices is conflict-free
    __shared__ double cv[kCobgMaxVals];
    if (p.nval) {
#pragma unroll
        for (int i = 0; i < kCobgMaxVals; i++)
            if (threadIdx.x == i) cv[i] = p.cval[i];
    }
    const long long N = p.N;
    // given helicities: the EPB thread groups of a block take EPB events.  Summed helicities: the block takes one
    // event and its groups share the 2^n assignments (group evl takes hc = evl, evl + EPB, ..)
    // (list launches: the grid is sized without knowing the count, a block takes tasks blockIdx.x, + gridDim.x, ..)
    const long long nev = p.list ? (long long)*p.list_count : N;
    const long long ntask = p.helsum ? nev : (nev + EPB - 1) / EPB;
    for (long long task = blockIdx.x; task < ntask; task += gridDim.x) {
    const long long e_raw = p.helsum ? task : task * EPB + evl;
    const bool active = e_raw < nev;
    const long long e = active ? (p.list ? (long long)p.list[e_raw] : e_raw) : 0;
    auto load_momentum = [&](int g, double* pg) {
#pragma unroll
        for (int c = 0; c < 4; c++) pg[c] = p.mom[(size_t)(g * 4 + c) * N + e];
        if (p.twin & 1) boost_frame(pg);
    };

    double total = 0.0;
    // Leading colour (Eq. 33) needs A(1, sigma) for all (n-1)! orderings of gluons 2..n: for each
    // choice `last` of the gluon that closes the amplitude the (n-2)! orderings of the others are the same
    // computation with gluon labels `last` and n exchanged.  Full colour: one pass, last = n.
    for (int last = M; last >= (LC ? 1 : M); last--) {
    auto relabel = [&](int g) { return !LC ? g : (g == M ? last : (g == last ? M : g)); };
    __syncthreads();   // the previous pass is done with P and the currents
    // subset momenta P[mask] = sum of p_g over the bits of mask (gluons 0..M-1), the same for all helicities
    for (int mask = t; mask < NSUB; mask += TPE) {
        double ps[4] = {0.0, 0.0, 0.0, 0.0};
        for (int g = 0; g < M; g++)
            if ((mask >> g) & 1) {
                double pg[4];
                load_momentum(relabel(g), pg);
#pragma unroll
                for (int c = 0; c < 4; c++) ps[c] += pg[c];
            }
#pragma unroll
        for (int c = 0; c < 4; c++) P[mask * 4 + c] = ps[c];
    }

    TopView<NG> tv;
    tv.cur = cur;
    tv.P = P;
    const bool top = t < np;
    auto load_view = [&](int sig) {
        tv.pm[0] = 0;
#pragma unroll
        for (int i = 0; i < M; i++) {
            tv.pm[i + 1] = tv.pm[i] | (1u << p.ord[sig * M + i]);
#pragma unroll
            for (int j = 0; j < M; j++) tv.sl[i * M + j] = p.slot[(sig * M + i) * M + j];
        }
    };
    load_view(top ? t : 0);

    const int nhel = p.helsum ? (1 << NG) : 1;
    const int hc_step = p.helsum ? EPB : 1;
    static_assert((1 << NG) % EPB == 0, "every group runs the same number of helicity assignments (block barriers)");
    for (int hc = p.helsum ? evl : 0; hc < nhel; hc += hc_step) {
        __syncthreads();   // previous helicity's reads are done; P is visible
        // level 1: external currents eps^lambda(p_g), Eq. 3, and eps_n
        for (int idx = t; idx <= M; idx += TPE) {
            int g = M, slot = -1;
            if (idx < M) {
                const uint32_t rep = p.lower[p.level_begin[1] + idx];
                const int sig = rep >> 8, i = (rep >> 4) & 0xF;
                g = p.ord[sig * M + i];
                slot = p.slot[(sig * M + i) * M + i];
            }
            double pg[4];
            load_momentum(relabel(g), pg);
            const int lam = p.helsum ? (((hc >> relabel(g)) & 1) ? 1 : -1) : (int)p.hel[(size_t)relabel(g) * N + e];
            cx eps[4];
            polarisation(pg, lam, eps);
            if (slot >= 0) sts_cur(cur, slot, eps);
            else sts_cur(epsn, 0, eps);
        }
        __syncthreads();
        // shared levels 2 .. n-3: one thread per distinct gluon sequence
        for (int L = 2; L <= LS; L++) {
            for (int idx = p.level_begin[L] + t; idx < p.level_begin[L + 1]; idx += TPE) {
                const uint32_t rep = p.lower[idx];
                const int sig = rep >> 8, i = (rep >> 4) & 0xF, j = rep & 0xF;
                const uint16_t* sl = p.slot + (size_t)sig * M * M;
                const uint8_t* og = p.ord + sig * M;
                cx s3[4], s4[4];
#pragma unroll
                for (int c = 0; c < 4; c++) { s3[c] = mk(0.0, 0.0); s4[c] = mk(0.0, 0.0); }
                unsigned mall = 0;
                for (int k = i; k <= j; k++) mall |= 1u << og[k];
                unsigned ma = 0;
                for (int k = i; k < j; k++) {
                    ma |= 1u << og[k];
                    cx a[4], b[4];
                    lds_cur(cur, sl[i * M + k], a);
                    lds_cur(cur, sl[(k + 1) * M + j], b);
                    v3_acc(s3, P + 4 * ma, P + 4 * (mall ^ ma), a, b, 1.0);
                    for (int l = k + 1; l < j; l++) {
                        cx b2[4], c2[4];
                        lds_cur(cur, sl[(k + 1) * M + l], b2);
                        lds_cur(cur, sl[(l + 1) * M + j], c2);
                        v4_acc(s4, a, b2, c2);
                    }
                }
                const double ip2 = 1.0 / mdot(P + 4 * mall, P + 4 * mall);
                cx J[4];
#pragma unroll
                for (int c = 0; c < 4; c++) J[c] = (kInvSqrt2 * ip2) * s3[c] + (0.5 * ip2) * s4[c];
                sts_cur(cur, sl[i * M + j], J);
            }
            __syncthreads();
        }
        // register-resident top: thread sigma builds the two (n-2)-gluon currents and the final one of its ordering
        double ward2 = 0.0, amp2 = 0.0;
        for (int sig = t; sig < np; sig += TPE) {
            if (sig != t || np > TPE) load_view(sig);      // (one ordering per thread: the view loaded above stays)
            tv.template range<1, M - 1, true>(tv.JA);
            tv.template range<0, M - 2, true>(tv.JB);
            cx JF[4], en[4];
            tv.template range<0, M - 1, false>(JF);
            lds_cur(epsn, 0, en);
            const cx amp = mdot(en, JF);
            A[2 * sig] = amp.re;
            A[2 * sig + 1] = amp.im;
            if (!LC && p.tau2 != 0.0) {
                // Ward identity: the current of gluons 1..n-1 is conserved, P . J = 0 with P = -p_n (round-off only)
                const cx wv = mdot(P + 4 * (NSUB - 1), JF);
                ward2 += s_norm2(wv);
                amp2 += s_norm2(amp);
            }
        }
        __syncthreads();
        // Eq. 16: row sigma of the real symmetric quadratic form
        double w = 0.0;
        if (LC) {
            for (int row = t; row < np; row += TPE) w += fma(A[2 * row], A[2 * row], A[2 * row + 1] * A[2 * row + 1]);
        } else {
            for (int row = t; row < np; row += TPE) {
                double tr[4] = {0.0, 0.0, 0.0, 0.0}, ti[4] = {0.0, 0.0, 0.0, 0.0};
                const double* Ccol = p.C + row;
                int s2 = 0;
                if (p.nval) {
                    const uint32_t* ci = p.cidx4 + row;
                    for (; s2 + 4 <= np; s2 += 4) {
                        const uint32_t w4 = __ldg(ci + (size_t)(s2 >> 2) * np);
    #pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const double c = cv[(w4 >> (8 * u)) & 0xFF];
                            const double2 a2 = *reinterpret_cast<const double2*>(A + 2 * (s2 + u));
                            tr[u] = fma(c, a2.x, tr[u]);
                            ti[u] = fma(c, a2.y, ti[u]);
                        }
                    }
                    if (s2 < np) {
                        const uint32_t w4 = __ldg(ci + (size_t)(s2 >> 2) * np);
                        for (int u = 0; s2 < np; s2++, u++) {
                            const double c = cv[(w4 >> (8 * u)) & 0xFF];
                            tr[0] = fma(c, A[2 * s2], tr[0]);
                            ti[0] = fma(c, A[2 * s2 + 1], ti[0]);
                        }
                    }
                }
                for (; s2 + 4 <= np; s2 += 4) {
    #pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const double c = __ldg(Ccol + (size_t)(s2 + u) * np);
                        const double2 a2 = *reinterpret_cast<const double2*>(A + 2 * (s2 + u));
                        tr[u] = fma(c, a2.x, tr[u]);
                        ti[u] = fma(c, a2.y, ti[u]);
                    }
                }
                for (; s2 < np; s2++) {
                    const double c = __ldg(Ccol + (size_t)s2 * np);
                    tr[0] = fma(c, A[2 * s2], tr[0]);
                    ti[0] = fma(c, A[2 * s2 + 1], ti[0]);
                }
                w += fma(A[2 * row], (tr[0] + tr[1]) + (tr[2] + tr[3]), A[2 * row + 1] * ((ti[0] + ti[1]) + (ti[2] + ti[3])));
            }
        }
#pragma unroll
        for (int d = 1; d < (TPE < 32 ? TPE : 32); d <<= 1) w += __shfl_xor_sync(0xFFFFFFFFu, w, d);
        if (TPE > 32) {
            __syncthreads();
            if ((t & 31) == 0) red[t >> 5] = w;
            __syncthreads();
            w = 0.0;
            for (int i = 0; i < TPE / 32; i++) w += red[i];
        }
        total += w;
        if (!LC && p.tau2 != 0.0) {
            // sum over the orderings of |P . J_sigma|^2 against E_n^2 sum |A_sigma|^2
#pragma unroll
            for (int d = 1; d < (TPE < 32 ? TPE : 32); d <<= 1) {
                ward2 += __shfl_xor_sync(0xFFFFFFFFu, ward2, d);
                amp2 += __shfl_xor_sync(0xFFFFFFFFu, amp2, d);
            }
            if (TPE > 32) {
                __syncthreads();
                if ((t & 31) == 0) { red[t >> 5] = ward2; red[8 + (t >> 5)] = amp2; }
                __syncthreads();
                ward2 = 0.0; amp2 = 0.0;
                for (int i = 0; i < TPE / 32; i++) { ward2 += red[i]; amp2 += red[8 + i]; }
            }
            if (t == 0 && active) {
                const double En = p.mom[(size_t)(M * 4) * N + e];
                const double scale = En * En * amp2;
                if (p.tau2 < 0.0) {
                    total = ::sqrt(ward2 / scale);
                } else {
                    const bool hard = !(ward2 <= fmax(p.tw2, p.tau2) * scale) || !(w > 0.0);
                    bool to_dd = hard, to_twin = false;
                    if (p.twin & 2) {
                        const double w1 = p.out[e];
                        to_dd = hard || !(fabs(w - w1) <= p.td * w1);
                    } else if (!hard) {
                        to_twin = !(ward2 <= p.tau2 * scale);      // (tau_twin <= tau: never - no second stage)
                    }
                    if (to_dd) p.flag_list[atomicAdd(p.flag_count, 1u)] = (uint32_t)e;
                    else if (to_twin) p.soft_list[atomicAdd(p.soft_count, 1u)] = (uint32_t)e;
                }
            }
        }
    }
    }   // last
    if (LC) total *= p.lc_factor;
    if (p.helsum && EPB > 1) {
        // add the groups' partial helicity sums in a fixed order
        __syncthreads();
        if (t == 0) red[0] = total;
        __syncthreads();
        if (threadIdx.x == 0) {
            total = 0.0;
            for (int i = 0; i < EPB; i++) total += (smem_d + (size_t)i * ev_doubles + p.nslots * 2 * kSlotStride + NSUB * 4 + 8 + np * 2)[0];
        }
        if (threadIdx.x == 0 && active) p.out[e] = total;
    } else if (t == 0 && active && !(p.twin & 2)) {
        p.out[e] = total;                 // (second stage of the cascade: out[e] keeps the first result)
    }
    }   // task
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
bool cobg_shared_supported(int n) { return n >= 4 && n <= 8; }

int cobg_table_create(int n, CobgTable** out) {
    *out = nullptr;
    if (!cobg_shared_supported(n)) return BG_EUNSUPPORTED;
    const int m = n - 1, ls = n - 3;
    std::vector<int> sigma(n - 2);
    std::iota(sigma.begin(), sigma.end(), 1);
    std::vector<std::vector<int>> ords;   // (0, sigma) in lexicographic order of sigma - the order of C's rows
    do {
        std::vector<int> o{0};
        o.insert(o.end(), sigma.begin(), sigma.end());
        ords.push_back(o);
    } while (std::next_permutation(sigma.begin(), sigma.end()));
    const int np = (int)ords.size();
    std::vector<uint16_t> slot((size_t)np * m * m, 0xFFFF);
    std::vector<uint8_t> ord((size_t)np * m);
    std::vector<uint32_t> lower;
    CobgTable* t = new (std::nothrow) CobgTable();
    if (!t) return BG_ENOMEM;
    std::memset(t, 0, sizeof(*t));
    // Slot numbering: inside a level, sequences are ordered by (set of gluons, lexicographic order).  Threads
    // sigma, sigma+1, .. (orderings in lexicographic order) then read runs of consecutive slots, which fall into
    // different shared-memory bank groups (slots are kSlotStride complex doubles apart, an odd number).
    int next = 0;
    t->level_begin[0] = t->level_begin[1] = 0;
    for (int L = 1; L <= ls; L++) {
        t->level_begin[L] = (int)lower.size();
        std::map<std::pair<unsigned, std::vector<int>>, uint32_t> reps;   // (mask, sequence) -> representative range
        for (int s = 0; s < np; s++)
            for (int i = 0; i + L <= m; i++) {
                const std::vector<int> seq(ords[s].begin() + i, ords[s].begin() + i + L);
                unsigned mask = 0;
                for (int g : seq) mask |= 1u << g;
                reps.emplace(std::make_pair(mask, seq), (uint32_t)(s << 8 | i << 4 | (i + L - 1)));
            }
        std::map<std::vector<int>, int> ids;
        for (auto& kv : reps) {
            ids.emplace(kv.first.second, next++);
            lower.push_back(kv.second);
        }
        for (int s = 0; s < np; s++)
            for (int i = 0; i + L <= m; i++) {
                const std::vector<int> seq(ords[s].begin() + i, ords[s].begin() + i + L);
                slot[((size_t)s * m + i) * m + i + L - 1] = (uint16_t)ids[seq];
            }
    }
    for (int L = ls + 1; L <= kCobgMaxM + 1; L++) t->level_begin[L] = (int)lower.size();
    for (int s = 0; s < np; s++)
        for (int i = 0; i < m; i++) ord[(size_t)s * m + i] = (uint8_t)ords[s][i];
    t->n = n; t->np = np; t->nslots = next;
    bool ok = cudaMalloc(&t->d_slot, slot.size() * 2) == cudaSuccess && cudaMalloc(&t->d_ord, ord.size()) == cudaSuccess &&
              cudaMalloc(&t->d_lower, std::max<size_t>(lower.size(), 1) * 4) == cudaSuccess;
    ok = ok && cudaMemcpy(t->d_slot, slot.data(), slot.size() * 2, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(t->d_ord, ord.data(), ord.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(t->d_lower, lower.data(), lower.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        cobg_table_destroy(t);
        return BG_ENOMEM;
    }
    *out = t;
    return BG_OK;
}

// Compressed form of the colour matrix hC[np][np] for the colour form of the kernel: the list of its distinct entries
// and one byte per entry.  Optional: with more than kCobgMaxVals distinct entries the kernel reads C itself.
int cobg_table_set_colour(CobgTable* t, const double* hC) {
    if (!t || !hC) return BG_EINVAL;
    const int np = t->np;
    std::vector<double> vals;
    std::vector<uint32_t> idx4((size_t)((np + 3) / 4) * np, 0u);
    for (int s2 = 0; s2 < np; s2++)
        for (int sg = 0; sg < np; sg++) {
            const double c = hC[(size_t)s2 * np + sg];
            size_t k = std::find(vals.begin(), vals.end(), c) - vals.begin();
            if (k == vals.size()) {
                if ((int)vals.size() == kCobgMaxVals) return BG_OK;   // too many: keep the plain form
                vals.push_back(c);
            }
            idx4[(size_t)(s2 / 4) * np + sg] |= (uint32_t)k << (8 * (s2 % 4));
        }
    if (cudaMalloc(&t->d_cidx4, idx4.size() * 4) != cudaSuccess ||
        cudaMemcpy(t->d_cidx4, idx4.data(), idx4.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        if (t->d_cidx4) cudaFree(t->d_cidx4);
        t->d_cidx4 = nullptr;
        return BG_ENOMEM;
    }
    for (int i = 0; i < kCobgMaxVals; i++) t->cval[i] = i < (int)vals.size() ? vals[i] : 0.0;
    t->nval = (int)vals.size();
    return BG_OK;
}

void cobg_table_destroy(CobgTable* t) {
    if (!t) return;
    if (t->d_cidx4) cudaFree(t->d_cidx4);
    if (t->d_slot) cudaFree(t->d_slot);
    if (t->d_ord) cudaFree(t->d_ord);
    if (t->d_lower) cudaFree(t->d_lower);
    delete t;
}

size_t cobg_shared_current_bytes(const CobgTable* t) { return t ? (size_t)t->nslots * 16 * kSlotStride : 0; }

template <int NG, int TPE, bool LC>
static cudaError_t launch_cobg(cudaStream_t s, const CobgParams& p) {
    constexpr int BLOCK = TPE > 128 ? TPE : 128;
    constexpr int EPB = BLOCK / TPE, NSUB = 1 << (NG - 1);
    const size_t smem = (size_t)EPB * (p.nslots * 2 * kSlotStride + NSUB * 4 + 8 + p.np * 2 + 16) * sizeof(double);
    static int configured_device = -1;   // the attribute is per device
    int device = 0;
    cudaGetDevice(&device);
    if (configured_device != device) {
        cudaError_t e = cudaFuncSetAttribute(cobg_shared_kernel<NG, TPE, LC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        configured_device = device;
    }
    unsigned blocks = p.helsum ? (unsigned)p.N : (unsigned)((p.N + EPB - 1) / EPB);
    if (p.list) {     // about 1/16 of the events, at least a wave of blocks (the kernel loops over what the list holds)
        int sms = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        blocks = (unsigned)std::max<long long>(1, std::min<long long>(blocks, std::max<long long>(4ll * sms, (p.N / 16 + EPB - 1) / EPB)));
    }
    cobg_shared_kernel<NG, TPE, LC><<<blocks, BLOCK, smem, s>>>(p);
    return cudaGetLastError();
}

cudaError_t cobg_shared_launch(cudaStream_t s, const CobgTable* t, bool helsum, bool lc, const double* dC, long long N,
                               const double* mom, const signed char* hel, double* out, double tau, uint32_t* flag_list,
                               uint32_t* flag_count, const CobgCascade* cascade) {
    CobgParams p;
    p.twin = 0; p.tw2 = 0.0; p.td = 0.0; p.soft_list = nullptr; p.soft_count = nullptr; p.list = nullptr; p.list_count = nullptr;
    if (cascade) {
        p.twin = cascade->twin; p.tw2 = cascade->tau_twin_ward * cascade->tau_twin_ward; p.td = cascade->tau_twin;
        p.soft_list = cascade->soft_list; p.soft_count = cascade->soft_count;
        p.list = cascade->list; p.list_count = cascade->list_count;
    }
    p.tau2 = (helsum || lc || !flag_list) && tau >= 0.0 ? 0.0 : (tau < 0.0 ? -1.0 : tau * tau);
    if (helsum || lc) p.tau2 = 0.0;
    p.flag_list = flag_list; p.flag_count = flag_count;
    p.n = t->n; p.np = t->np; p.nslots = t->nslots; p.helsum = helsum ? 1 : 0;
    p.lc = lc ? 1 : 0;
    p.lc_factor = 8.0;
    for (int i = 0; i < t->n - 2; i++) p.lc_factor *= 3.0;
    p.N = N; p.mom = mom; p.hel = hel; p.C = dC; p.out = out;
    p.slot = t->d_slot; p.ord = t->d_ord; p.lower = t->d_lower;
    p.cidx4 = t->d_cidx4;
    p.nval = (!lc && dC && t->np >= 24) ? t->nval : 0;   // (n <= 5: two and six orderings, nothing to gain)
    for (int i = 0; i < kCobgMaxVals; i++) p.cval[i] = t->cval[i];
    for (int i = 0; i < kCobgMaxM + 2; i++) p.level_begin[i] = t->level_begin[i];
    switch (t->n) {
        case 4: return lc ? launch_cobg<4, 8, true>(s, p) : launch_cobg<4, 8, false>(s, p);
        // threads per event (full colour), measured on 2^19 / 2^19 / 2^18 events: n = 5: 8 -> 4: 0.71 -> 0.64 ms; n = 6: 32 -> 16 -> 8:
        // 5.69 -> 4.45 -> 4.23 ms; n = 7: 128 -> 64: 16.2 -> 15.4 ms (32: 19.6 ms); n = 8: 256 (128: 6.8 -> 10.7 ms).  Fewer
        // threads take several orderings each in rounds and more events share a block: fewer idle threads at the barriers
        // of the shared levels.  Leading colour, n = 6: 32 -> 8: 2.75 -> 2.27 ms for 2^16 events; summed helicities keep the round-1 values.
        case 5: return lc ? launch_cobg<5, 8, true>(s, p) : (helsum ? launch_cobg<5, 8, false>(s, p) : launch_cobg<5, 4, false>(s, p));
        case 6: return lc ? launch_cobg<6, 8, true>(s, p) : (helsum ? launch_cobg<6, 32, false>(s, p) : launch_cobg<6, 8, false>(s, p));
        case 7: return lc ? launch_cobg<7, 128, true>(s, p) : (helsum ? launch_cobg<7, 128, false>(s, p) : launch_cobg<7, 64, false>(s, p));
        case 8: return lc ? launch_cobg<8, 256, true>(s, p) : launch_cobg<8, 256, false>(s, p);
        default: return cudaErrorNotSupported;
    }
}

}  // namespace bg

// C-ABI of libbg.so (declared in include/bg.h): context management, colour-matrix construction, dispatch.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <vector>

#include "bg_internal.h"
#include "bg_program.h"

namespace bg {

// ---------------------------------------------------------------------------------------------------------
// Colour matrix, Eq. 17, as exact integers.  With Tr(T^a T^b) = delta^ab,
//   (F^{a_2} .. F^{a_{n-1}})_{a_1 a_n} = (-1)^n Tr(T^{a_1} [T^{a_2}, [T^{a_3}, .. [T^{a_{n-1}}, T^{a_n}] .. ]])
// (the overall sign drops out of C).  Expanding the nested commutator gives 2^{n-2} signed single traces; the sum
// over all colours of Tr(w) Tr(w')^* follows from the U(N) completeness relation T^a_ij T^a_kl = delta_il delta_kj
// as N_c^{#index loops} (commutators have no U(1) component, so U(N) and SU(N) sums agree).  Relabelling the
// summed colours gives C_{sigma sigma'} = C_{id, sigma^-1 sigma'}, so one row is computed and permuted.
// Orderings sigma: permutations of gluons 2..n-1 in lexicographic order.
// ---------------------------------------------------------------------------------------------------------
static void expand_words(const std::vector<int>& order /* n labels, order[0]=first, order[n-1]=last */,
                         std::vector<std::vector<int>>& words, std::vector<int>& signs) {
    const int n = (int)order.size();
    words.assign(1, std::vector<int>{order[n - 1]});
    signs.assign(1, 1);
    for (int k = n - 2; k >= 1; k--) {
        std::vector<std::vector<int>> nw;
        std::vector<int> ns;
        for (size_t i = 0; i < words.size(); i++) {
            std::vector<int> a{order[k]};
            a.insert(a.end(), words[i].begin(), words[i].end());
            nw.push_back(a);
            ns.push_back(signs[i]);
            std::vector<int> b = words[i];
            b.push_back(order[k]);
            nw.push_back(b);
            ns.push_back(-signs[i]);
        }
        words.swap(nw);
        signs.swap(ns);
    }
    for (auto& w : words) w.insert(w.begin(), order[0]);
}

static int find_root(int* parent, int x) {
    while (parent[x] != x) x = parent[x] = parent[parent[x]];
    return x;
}

// sum over all colour labels of Tr(T^{w1}) Tr(T^{w2})^* = N^(loops)
static long long trace_pair(const std::vector<int>& w1, const std::vector<int>& w2) {
    const int n = (int)w1.size();
    int pos1[16], pos2[16], parent[32];
    std::vector<int> w2r(w2.rbegin(), w2.rend());   // complex conjugate of a trace = trace of the reversed word
    for (int p = 0; p < n; p++) { pos1[w1[p]] = p; pos2[w2r[p]] = p; }
    for (int i = 0; i < 2 * n; i++) parent[i] = i;
    for (int a = 0; a < n; a++) {
        const int p = pos1[a], q = pos2[a];
        // generator a carries (row r_p, col r_{p+1}) in trace 1 and (row s_q, col s_{q+1}) in trace 2
        int x = find_root(parent, p), y = find_root(parent, n + (q + 1) % n);
        if (x != y) parent[x] = y;
        x = find_root(parent, n + q); y = find_root(parent, (p + 1) % n);
        if (x != y) parent[x] = y;
    }
    int loops = 0;
    for (int i = 0; i < 2 * n; i++) loops += find_root(parent, i) == i;
    long long r = 1;
    for (int i = 0; i < loops; i++) r *= 3;
    return r;
}

int build_colour_matrix(int n, double* C) {
    const int m = n - 2;
    std::vector<std::vector<int>> perms;
    std::vector<int> p(m);
    std::iota(p.begin(), p.end(), 1);
    do perms.push_back(p); while (std::next_permutation(p.begin(), p.end()));
    const int np = (int)perms.size();
    // words of the identity ordering and of every ordering
    auto full_order = [&](const std::vector<int>& s) {
        std::vector<int> o{0};
        o.insert(o.end(), s.begin(), s.end());
        o.push_back(n - 1);
        return o;
    };
    std::vector<std::vector<int>> w0, w1;
    std::vector<int> s0, s1;
    expand_words(full_order(perms[0]), w0, s0);
    std::vector<long long> row(np);
    for (int t = 0; t < np; t++) {
        expand_words(full_order(perms[t]), w1, s1);
        long long acc = 0;
        for (size_t i = 0; i < w0.size(); i++)
            for (size_t j = 0; j < w1.size(); j++) acc += (long long)(s0[i] * s1[j]) * trace_pair(w0[i], w1[j]);
        row[t] = acc;
    }
    // C[s][s'] = row[index of s^-1 o s']
    std::vector<int> inv(n);
    for (int s = 0; s < np; s++) {
        for (int i = 0; i < m; i++) inv[perms[s][i]] = i + 1;   // label -> position (as a label 1..m)
        for (int t = 0; t < np; t++) {
            // relative permutation rel(i) = inv[perms[t][i]]; its lexicographic index
            int idx = 0;
            bool used[16] = {false};
            for (int i = 0; i < m; i++) {
                const int v = inv[perms[t][i]];
                int smaller = 0;
                for (int u = 1; u < v; u++) smaller += !used[u];
                used[v] = true;
                int f = 1;
                for (int u = 2; u <= m - 1 - i; u++) f *= u;
                idx += smaller * f;
            }
            C[(size_t)s * np + t] = (double)row[idx];
        }
    }
    return np;
}

}  // namespace bg

// =========================================== ABI ===========================================================
// largest n whose colour-class programs are tabulated at bg_init, and the default lanes per event
static const int kProgMaxN = 12;
static int auto_lanes(int n) {
    static const int lanes[] = {0, 0, 0, 0, 2, 4, 4, 8, 32, 64, 128, 128, 128};
    return lanes[n];
}

// shared memory one event's state may take before its top levels spill to global memory (0 = all of it)
// measured (2^16 events, FP64): n = 11: 48 / 56 / 64 / 104 KB -> 2.67 / 2.77 / 2.40 / 2.40e6 events/s (three blocks per SM at
// 56 KB); n = 12: 56 / 80 / 88 / 96 / 104 KB -> 8.1 / 8.6 / 8.8 / 7.4 / 7.7e5 (two blocks per SM)
static size_t auto_slab_limit(int n) { return n == 11 ? (size_t)56 * 1024 : (n >= 12 ? (size_t)88 * 1024 : 0); }

extern "C" {
static int make_prog_table(const bg_ctx* c, int G, size_t limit, bg::ProgTable** t);
}

// Threshold of the conditioning flag |p_n . J| / (E_n |eps_n . J|) (Ward residual of the closing current) above which
// an event is evaluated again in double-double arithmetic; tuned against the extended-precision oracle so that
// no unflagged event of the test workloads is further than 1e-11 from it.
// Ward-residual threshold of the first stage (events above it are evaluated a second time in FP64, which is cheap, so it
// sits well below the residuals at which errors of 1e-11 were seen: DESIGN.md 3) and what the second stage may differ by.
// n = 6: 3e-15, a quarter of the events - the residual of the events with an error above 1e-11 that 1e-14 left unflagged
// (7 of 16.8e6) was 4 - 9.5e-15, and their two frames differ by 1e-11; n = 5 (13 of 8.4e6 with residuals from 8e-16): 1e-15.
// (n >= 11, where the second evaluation runs the spill kernels: measured 3 % faster at 1e-13, worst unflagged error 8e-12)
// (n = 7, 8: 1e-14 - two unflagged events each in 16.8e6 / 8.4e6 with residuals of 2.4 - 2.9e-14; none at n = 9, 10 in 4.2e6 / 1.0e6)
static double default_tau(int n) { return n <= 4 || n >= 11 ? 1e-13 : (n == 5 ? 1e-15 : (n == 6 ? 3e-15 : (n <= 8 ? 1e-14 : 3e-14))); }
static const double kDefaultTauTwin = 5e-13;
// The second stage's bound on the Ward residuals, as a fraction of its bound on the difference of the two results: round-off
// that both frames share (the inputs conserve momentum only to 1e-16, and the closing gluon's momentum is the one the
// recursion never uses) shows in the residuals, not in the difference: events that passed the second stage with both
// results off by 1.0 - 2.3e-11 had residuals of 1.2 - 4.3e-13 (n = 5, 6, 7: about one per 10^7 events).
static double twin_ward_fraction(int n) { (void)n; return 0.4; }
// COBG (the colour-summed |M|^2 is better conditioned than a single colour flow): second-stage bound 1e-12 on the
// difference and on the residuals for n >= 6 (2^19 / 2^18 / 2^13 events at n = 6 / 7 / 8: 0.9 - 1.1 % left for double-double,
// worst accepted error 4.1 / 5.2 / 0.8e-12), 5e-13 on the difference for n <= 5 (1.0 %, 4.1e-12)
static double default_tau_twin_cobg(int n) { return n <= 5 ? 5e-13 : 1e-12; }
static double twin_ward_fraction_cobg(int n) { return n <= 5 ? 0.4 : 1.0; }
// (large campaign, 16.8e6 events each: n = 6 left 7 events with residuals of 4 - 9.6e-14 unflagged at 1e-13, n = 5 two with
// 3.6 - 5.5e-15 at 1e-14; n = 5 passed four events with residuals of 4 - 6.8e-13 through a second-stage bound of 1e-12)
static double default_tau_cobg(int n) { return n <= 5 ? 3e-15 : 3e-14; }
static const double kDefaultTauRho = 3e-3;

static bool mode_supported(int n, int mode) {
    if (n < 4 || n > 12) return false;
    if (mode == BG_COBG_HELSUM_FULLCOLOR || mode == BG_COBG_HELGIVEN_FULLCOLOR) return n <= 8;
    if (mode == BG_COBG_HELSUM_LC || mode == BG_COBG_HELGIVEN_LC) return bg::cobg_shared_supported(n);
    if (mode == BG_CDBG_GIVEN || mode == BG_CDBG_HELSUM_COLGIVEN) return true;
    if (mode == BG_CDBG_CONTINUOUS) return n <= 10;   // 16-bit state offsets: 2^(n-1) subsets x 9 colour entries x 10 elements
    if (mode == BG_COMC_GIVEN) return n <= 9;   // (n = 9: classes with thousands of orderings fall back to the dressed program)
    return false;
}

extern "C" {

const char* bg_strerror(int code) {
    switch (code) {
        case BG_OK: return "ok";
        case BG_EINVAL: return "invalid argument";
        case BG_ENOMEM: return "out of memory";
        case BG_ECUDA: return "CUDA error (no device, or a runtime/launch failure)";
        case BG_EUNSUPPORTED: return "mode / n combination not supported";
        case BG_ELIMIT: return "batch larger than the fixed scratch of the no-allocation entry point (bg_static_max_events)";
        default: return "unknown error code";
    }
}

int bg_init(bg_ctx** out, int n, int mode) {
    if (!out) return BG_EINVAL;
    *out = nullptr;
    if (n < 4 || n > 12) return BG_EINVAL;
    if (!mode_supported(n, mode)) return BG_EUNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return BG_ECUDA;
    bg_ctx* c = new (std::nothrow) bg_ctx();
    if (!c) return BG_ENOMEM;
    std::memset(c, 0, sizeof(*c));
    c->n = n;
    c->mode = mode;
    c->scratch_limit = (size_t)16 << 30;
    c->last_kernel = "none";
    if (cudaGetDevice(&c->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess) {
        delete c;
        return BG_ECUDA;
    }
    if ((mode & BG_REC_COBG) && (mode & BG_COL_FULL)) {
        int np = 1;
        for (int i = 2; i <= n - 2; i++) np *= i;
        c->nperm = np;
        c->hC = (double*)std::malloc(sizeof(double) * np * np);
        if (!c->hC) { delete c; return BG_ENOMEM; }
        bg::build_colour_matrix(n, c->hC);
        if (cudaMalloc(&c->dC, sizeof(double) * np * np) != cudaSuccess) { std::free(c->hC); delete c; return BG_ENOMEM; }
        if (cudaMemcpy(c->dC, c->hC, sizeof(double) * np * np, cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaFree(c->dC); std::free(c->hC); delete c; return BG_ECUDA;
        }
    }
    if ((mode & BG_REC_COBG) && mode != BG_COMC_GIVEN && bg::cobg_shared_supported(n)) {
        const int rc = bg::cobg_table_create(n, &c->cobg);
        if (rc != BG_OK) { cudaFree(c->dC); std::free(c->hC); delete c; return rc; }
        if (c->hC) bg::cobg_table_set_colour(c->cobg, c->hC);   // optional compressed form; the plain one stays valid
    }
    if ((mode == BG_CDBG_GIVEN && n <= kProgMaxN) || mode == BG_CDBG_CONTINUOUS || mode == BG_COMC_GIVEN) {
        const int rc = make_prog_table(c, 0, 0, &c->prog);
        if (rc != BG_OK) { delete c; return rc; }
    }
    // default precision: FP64 with the conditioning flag and double-double re-evaluation of the flagged events
    c->tau = mode == BG_COBG_HELGIVEN_FULLCOLOR ? default_tau_cobg(n) : default_tau(n);
    c->tau_rho = kDefaultTauRho;
    c->tau_twin = mode == BG_COBG_HELGIVEN_FULLCOLOR ? default_tau_twin_cobg(n) : kDefaultTauTwin;
    c->frame = 0;
    // (n = 4: a single colour flow is one Parke-Taylor term per helicity assignment; the FP64 kernels alone stay below
    // 1.2e-12 on 2^20 + 2^18 events, and any flagged event would cost a 47 us double-double pass: FP64 by default)
    if (mode == BG_CDBG_GIVEN && c->prog && bg::prog_dd_mode(c->prog) >= 0 && n >= 5) c->precision = 2;
    if (mode == BG_COBG_HELGIVEN_FULLCOLOR && c->cobg) c->precision = 2;
    bool streams_ok = cudaStreamCreateWithFlags(&c->hstream, cudaStreamNonBlocking) == cudaSuccess &&
                      cudaStreamCreateWithFlags(&c->cstream, cudaStreamNonBlocking) == cudaSuccess;
    for (int k = 0; k < kHostChunks && streams_ok; k++)
        streams_ok = cudaEventCreateWithFlags(&c->chunk_ev[k], cudaEventDisableTiming) == cudaSuccess;
    if (!streams_ok) {
        bg::prog_table_destroy(c->prog);
        bg::cobg_table_destroy(c->cobg);
        if (c->dC) cudaFree(c->dC);
        std::free(c->hC);
        delete c;
        return BG_ECUDA;
    }
    *out = c;
    return BG_OK;
}

int bg_destroy(bg_ctx* c) {
    if (!c) return BG_EINVAL;
    cudaStreamSynchronize(c->hstream);
    cudaStreamDestroy(c->hstream);
    if (c->cstream) { cudaStreamSynchronize(c->cstream); cudaStreamDestroy(c->cstream); }
    for (int k = 0; k < kHostChunks; k++)
        if (c->chunk_ev[k]) cudaEventDestroy(c->chunk_ev[k]);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->ev_mid) cudaEventDestroy(c->ev_mid);
    if (c->alt) bg_destroy(c->alt);
    bg::prog_table_destroy(c->prog);
    bg::cobg_table_destroy(c->cobg);
    if (c->dC) cudaFree(c->dC);
    if (c->scratch) cudaFree(c->scratch);
    if (c->d_mom) cudaFree(c->d_mom);
    if (c->d_hel) cudaFree(c->d_hel);
    if (c->d_col) cudaFree(c->d_col);
    if (c->d_out) cudaFree(c->d_out);
    std::free(c->hC);
    delete c;
    return BG_OK;
}

static bool use_dd(const bg_ctx* c) { return c->mode == BG_CDBG_GIVEN && c->precision == 1; }
static bool use_cobg_dd(const bg_ctx* c) { return (c->mode & BG_REC_COBG) && (c->mode & BG_COL_FULL) && c->precision == 1; }
static long long cobg_dd_chunk(const bg_ctx* c, long long N) {
    const size_t per = bg::cobg_dd_scratch_per_event(c->n, (c->mode & BG_HEL_SUM) != 0);
    long long chunk = (long long)(std::min<size_t>(c->scratch_limit, (size_t)2 << 30) / per);
    if (chunk < 64) chunk = 64;
    return std::min(chunk, std::max<long long>(N, 1));
}

// events per double-double launch under the scratch limit
static long long dd_chunk(const bg_ctx* c, long long N) {
    const size_t per = bg::cdbg_dd_scratch_per_event(c->n);
    long long chunk = (long long)(c->scratch_limit / per);
    if (chunk < 128) chunk = 128;
    chunk -= chunk % 128;
    return std::min(chunk, std::max<long long>(N, 1));
}

// COBG, given helicities, full colour on the shared-current kernel: Ward flag + double-double re-evaluation
static bool use_cobg_auto(const bg_ctx* c) {
    return c->mode == BG_COBG_HELGIVEN_FULLCOLOR && c->precision >= 2 && c->cobg && c->kernel_opt != 1;
}

static bool use_prog(const bg_ctx* c) {
    if (c->mode == BG_CDBG_CONTINUOUS || c->mode == BG_COMC_GIVEN) return c->prog != nullptr;
    if (c->mode != BG_CDBG_GIVEN || c->kernel_opt == 1 || use_dd(c)) return false;
    return c->prog != nullptr;
}

// lanes per event of the dense (continuous-state) program, and the table for the context's mode
static int auto_lanes_dense(int n) { return n <= 4 ? 32 : (n <= 6 ? 64 : (n == 7 ? 128 : 256)); }
static int make_prog_table(const bg_ctx* c, int G, size_t limit, bg::ProgTable** t) {
    if (c->mode == BG_CDBG_CONTINUOUS) return bg::prog_table_create_dense(c->n, G ? G : auto_lanes_dense(c->n), limit, c->kernel_opt != 1, t);
    if (c->mode == BG_COMC_GIVEN) return bg::prog_table_create(c->n, G ? G : (c->n >= 7 ? 128 : auto_lanes(c->n)), limit, true, t);
    int rc = bg::prog_table_create(c->n, G ? G : auto_lanes(c->n), limit ? limit : auto_slab_limit(c->n), false, t);
    if (rc == BG_OK && G == 0 && limit == 0 && c->n == 8) {
        // default lane count: the double-double stage gets a table with half the lanes (n = 8, 2^17 events:
        // 4.13 -> 3.75 ms per step.  n = 9 with 32 lanes and the closure legs of the 64-lane table: 18.9 -> 19.3 ms, not used)
        bg::ProgTable* dd = nullptr;
        if (bg::prog_table_create(c->n, auto_lanes(c->n) / 2, 0, false, &dd, *t) == BG_OK) bg::prog_table_attach_dd(*t, dd);
    }
    return rc;
}

// events per generic-CDBG launch under the scratch limit
static long long generic_chunk(const bg_ctx* c, long long N) {
    const size_t per = bg::cdbg_generic_scratch_per_event(c->n);
    long long chunk = (long long)(c->scratch_limit / per);
    if (chunk < 128) chunk = 128;
    chunk -= chunk % 128;
    return std::min(chunk, std::max<long long>(N, 1));
}

size_t bg_scratch_bytes(const bg_ctx* c, long long N) {
    if (!c || N <= 0) return 0;
    if (use_cobg_dd(c)) return bg::cobg_dd_scratch_per_event(c->n, (c->mode & BG_HEL_SUM) != 0) * (size_t)cobg_dd_chunk(c, N);
    if (use_cobg_auto(c)) return 256 + (size_t)N * 8;   // list counters | double-double list | second-stage list
    if (c->mode == BG_COMC_GIVEN) return c->prog ? bg::prog_scratch_bytes(c->prog, N) : 0;
    if (!(c->mode & BG_REC_CDBG)) return 0;
    if (use_dd(c)) return bg::cdbg_dd_scratch_per_event(c->n) * (size_t)dd_chunk(c, N);
    if (use_prog(c)) return bg::prog_scratch_bytes(c->prog, N);
    return bg::cdbg_generic_scratch_per_event(c->n) * (size_t)generic_chunk(c, N);
}

size_t bg_current_bytes_per_event(const bg_ctx* c) {
    if (!c) return 0;
    if (c->mode == BG_COMC_GIVEN) return c->prog ? bg::prog_state_bytes(c->prog) : 0;
    if ((c->mode & BG_REC_COBG) && c->cobg && c->kernel_opt != 1) return bg::cobg_shared_current_bytes(c->cobg);
    if (c->mode & BG_REC_COBG) return (size_t)(c->n - 1) * c->n / 2 * 64;   // one ordering's current table
    if (use_prog(c)) return bg::prog_state_bytes(c->prog);
    return ((size_t)1 << (c->n - 1)) * 3 * 160;
}

static int ensure_scratch(bg_ctx* c, long long N) {
    const size_t need = bg_scratch_bytes(c, N);
    if (need <= c->scratch_bytes) return BG_OK;
    if (c->scratch) { cudaDeviceSynchronize(); cudaFree(c->scratch); c->scratch = nullptr; c->scratch_bytes = 0; }
    if (cudaMalloc(&c->scratch, need) != cudaSuccess) { cudaGetLastError(); return BG_ENOMEM; }
    c->scratch_bytes = need;
    return BG_OK;
}

static int ensure_staging(bg_ctx* c, long long N) {
    if (N <= c->staged_events) return BG_OK;
    cudaStreamSynchronize(c->hstream);
    if (c->d_mom) cudaFree(c->d_mom);
    if (c->d_hel) cudaFree(c->d_hel);
    if (c->d_col) cudaFree(c->d_col);
    if (c->d_out) cudaFree(c->d_out);
    c->d_mom = nullptr; c->d_hel = nullptr; c->d_col = nullptr; c->d_out = nullptr;
    c->staged_events = 0;
    const size_t n = (size_t)c->n;
    if (cudaMalloc(&c->d_mom, sizeof(double) * 4 * n * N) != cudaSuccess ||
        cudaMalloc(&c->d_hel, n * N) != cudaSuccess || cudaMalloc(&c->d_col, 2 * n * N) != cudaSuccess ||
        cudaMalloc(&c->d_out, sizeof(double) * N) != cudaSuccess) {
        cudaGetLastError();
        return BG_ENOMEM;
    }
    c->staged_events = N;
    return BG_OK;
}

int bg_reserve(bg_ctx* c, long long N) {
    if (!c || N < 0) return BG_EINVAL;
    if (N == 0) return BG_OK;
    int rc = ensure_scratch(c, N);
    if (rc != BG_OK) return rc;
    return ensure_staging(c, N);
}

int bg_set_option(bg_ctx* c, int key, long long value) {
    if (!c) return BG_EINVAL;
    switch (key) {
        case BG_OPT_KERNEL:
            if (value < 0 || value > 2) return BG_EINVAL;
            if (value == 2 && !c->prog && !c->cobg) return BG_EUNSUPPORTED;
            if (c->mode == BG_CDBG_CONTINUOUS && c->prog && ((int)value == 1) != (c->kernel_opt == 1)) {
                // continuous states: real or complex arithmetic is a property of the program table (element size, offsets)
                const int before = c->kernel_opt;
                c->kernel_opt = (int)value;
                cudaDeviceSynchronize();
                bg::ProgTable* t = nullptr;
                const int rc = make_prog_table(c, c->prog_lanes, c->slab_limit, &t);
                if (rc != BG_OK) { c->kernel_opt = before; return rc; }
                bg::prog_table_destroy(c->prog);
                c->prog = t;
                return BG_OK;
            }
            c->kernel_opt = (int)value;
            return BG_OK;
        case BG_OPT_LANES: {
            if ((c->mode != BG_CDBG_GIVEN && c->mode != BG_CDBG_CONTINUOUS && c->mode != BG_COMC_GIVEN) || c->n > kProgMaxN)
                return BG_EUNSUPPORTED;
            if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 && value != 16 && value != 32 &&
                value != 64 && value != 128 && value != 256)
                return BG_EINVAL;
            const int G = (int)value;
            if (c->prog && G && bg::prog_lanes(c->prog) == G && c->mode != BG_CDBG_CONTINUOUS) return BG_OK;
            cudaDeviceSynchronize();
            bg::ProgTable* t = nullptr;
            const int rc = make_prog_table(c, G, c->slab_limit, &t);
            if (rc != BG_OK) return rc;
            bg::prog_table_destroy(c->prog);
            c->prog = t;
            c->prog_lanes = G;
            // few lanes per event put many events into one warp's shared memory: where the double-double state of
            // the re-evaluation no longer fits, the context falls back to the FP64 kernels alone (documented in bg.h)
            if (c->precision == 2 && bg::prog_dd_mode(t) < 0) c->precision = 0;
            return BG_OK;
        }
        case BG_OPT_SMEM_LIMIT: {
            if ((c->mode != BG_CDBG_GIVEN && c->mode != BG_CDBG_CONTINUOUS && c->mode != BG_COMC_GIVEN) || !c->prog)
                return BG_EUNSUPPORTED;
            if (value != 0 && (value < 16 * 1024 || value > 222 * 1024)) return BG_EINVAL;
            cudaDeviceSynchronize();
            bg::ProgTable* t = nullptr;
            const int rc = make_prog_table(c, bg::prog_lanes(c->prog), (size_t)value, &t);
            if (rc != BG_OK) return rc;
            bg::prog_table_destroy(c->prog);
            c->prog = t;
            c->slab_limit = (size_t)value;
            if (c->precision == 2 && bg::prog_dd_mode(t) < 0) c->precision = 0;
            return BG_OK;
        }
        case BG_OPT_PRECISION:
            if (value < 0 || value > 4) return BG_EINVAL;
            if (value == 3 && !(c->mode == BG_CDBG_GIVEN && c->prog) && !(c->mode == BG_COBG_HELGIVEN_FULLCOLOR && c->cobg))
                return BG_EUNSUPPORTED;
            if (value == 4 && !(c->mode == BG_CDBG_GIVEN && c->prog)) return BG_EUNSUPPORTED;
            if (value == 1 && c->mode != BG_CDBG_GIVEN && !((c->mode & BG_REC_COBG) && (c->mode & BG_COL_FULL)))
                return BG_EUNSUPPORTED;
            if (value == 2 && !(c->mode == BG_CDBG_GIVEN && c->prog && bg::prog_dd_mode(c->prog) >= 0) &&
                !(c->mode == BG_COBG_HELGIVEN_FULLCOLOR && c->cobg))
                return BG_EUNSUPPORTED;
            c->precision = (int)value;
            return BG_OK;
        case BG_OPT_FLAG_THRESHOLD:
            if (value < 0) return BG_EINVAL;
            c->tau = value != 0 ? (double)value * 1e-18 : (c->mode == BG_COBG_HELGIVEN_FULLCOLOR ? default_tau_cobg(c->n) : default_tau(c->n));
            return BG_OK;
        case BG_OPT_FLAG_CANCELLATION:
            if (value < 0 || value > 1000000) return BG_EINVAL;
            c->tau_rho = value == 0 ? kDefaultTauRho : (double)value * 1e-6;
            return BG_OK;
        case BG_OPT_FLAG_TWIN:
            if (value < 0) return BG_EINVAL;
            c->tau_twin = value != 0 ? (double)value * 1e-18
                                     : (c->mode == BG_COBG_HELGIVEN_FULLCOLOR ? default_tau_twin_cobg(c->n) : kDefaultTauTwin);
            return BG_OK;
        case BG_OPT_FRAME:
            if (value != 0 && value != 1) return BG_EINVAL;
            if (!(c->mode == BG_CDBG_GIVEN && c->prog) && !((c->mode & BG_REC_COBG) && c->mode != BG_COMC_GIVEN && c->cobg)) return BG_EUNSUPPORTED;
            c->frame = (int)value;
            return BG_OK;
        case BG_OPT_TIMING:
            if (value != 0 && value != 1) return BG_EINVAL;
            if (value && !c->ev0) {
                if (cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess ||
                    cudaEventCreate(&c->ev_mid) != cudaSuccess)
                    return BG_ECUDA;
            }
            c->timing = (int)value;
            c->timed = false;
            return BG_OK;
        case BG_OPT_SCRATCH_LIMIT:
            if (value < (1ll << 20)) return BG_EINVAL;
            c->scratch_limit = (size_t)value;
            return BG_OK;
        default:
            return BG_EINVAL;
    }
}

int bg_colour_matrix(const bg_ctx* c, double* C_host) {
    if (!c || !C_host || !c->hC) return BG_EINVAL;
    std::memcpy(C_host, c->hC, sizeof(double) * c->nperm * c->nperm);
    return BG_OK;
}

int bg_build_colour_matrix(int n, double* C_host) {
    if (n < 4 || n > 8 || !C_host) return BG_EINVAL;
    bg::build_colour_matrix(n, C_host);
    return BG_OK;
}

int bg_class_program_stats(int n, int lanes, const int* counts, long long* stats) {
    if (n < 4 || n > 12 || !counts || !stats || lanes < 1 || lanes > 256 || (lanes & (lanes - 1))) return BG_EINVAL;
    int sum = 0;
    for (int c = 0; c < bg::kNumCodes; c++) {
        if (counts[c] < 0) return BG_EINVAL;
        sum += counts[c];
    }
    if (sum != n) return BG_EINVAL;
    bg::ClassProgram p;
    bg::build_class(n, lanes, counts, p);
    stats[0] = p.valid ? 1 : 0;
    stats[1] = p.n_vertex_ops;
    stats[2] = p.total_steps;
    stats[3] = (long long)p.state_cx * 16;
    stats[4] = p.closure_code;
    return BG_OK;
}

int bg_comc_program_stats(int n, int lanes, const int* counts, long long* stats) {
    if (n < 4 || n > 9 || !counts || !stats || lanes < 1 || lanes > 256 || (lanes & (lanes - 1))) return BG_EINVAL;
    int sum = 0, code[bg::kMaxN];
    for (int c = 0; c < bg::kNumCodes; c++) {
        if (counts[c] < 0 || sum + counts[c] > n) return BG_EINVAL;
        for (int q = 0; q < counts[c]; q++) code[sum++] = c;
    }
    if (sum != n) return BG_EINVAL;
    bg::ClassProgram p;
    bg::build_comc_program(n, lanes, code, p);
    if (p.state_cx < 0) return BG_EUNSUPPORTED;
    stats[0] = p.valid ? 1 : 0;
    stats[1] = p.n_vertex_ops;
    stats[2] = p.total_steps;
    stats[3] = (long long)p.state_cx * 16;
    stats[4] = p.n_orderings;
    return BG_OK;
}

int bg_last_launch_count(const bg_ctx* c) { return c ? c->last_launches : 0; }

int bg_last_kernel_ms(bg_ctx* c, double* ms) {
    if (!c || !ms || !c->timing || !c->timed) return BG_EINVAL;
    if (cudaEventSynchronize(c->ev1) != cudaSuccess) return BG_ECUDA;
    float f = 0.f;
    if (cudaEventElapsedTime(&f, c->ev0, c->ev1) != cudaSuccess) return BG_ECUDA;
    *ms = (double)f;
    return BG_OK;
}
const char* bg_last_kernel_name(const bg_ctx* c) { return c ? c->last_kernel : "none"; }

int bg_last_refined(bg_ctx* c, long long* flagged, double* ms) {
    if (!c || !flagged) return BG_EINVAL;
    *flagged = 0;
    if (ms) *ms = 0.0;
    if (!c->last_auto || !c->scratch) return BG_OK;
    if (cudaDeviceSynchronize() != cudaSuccess) return BG_ECUDA;
    if (c->mode == BG_COBG_HELGIVEN_FULLCOLOR) {
        uint32_t k = 0;
        if (cudaMemcpy(&k, c->scratch, sizeof(k), cudaMemcpyDeviceToHost) != cudaSuccess) return BG_ECUDA;
        *flagged = k;
    } else if (!c->prog || bg::prog_flagged_count(c->prog, c->last_N, c->scratch, flagged) != cudaSuccess) {
        return BG_ECUDA;
    }
    if (ms && c->timing && c->timed) {
        float f = 0.f;
        if (cudaEventElapsedTime(&f, c->ev_mid, c->ev1) != cudaSuccess) return BG_ECUDA;
        *ms = (double)f;
    }
    return BG_OK;
}

int bg_last_twin(bg_ctx* c, long long* count) {
    if (!c || !count) return BG_EINVAL;
    *count = 0;
    if (!c->last_auto || !c->scratch) return BG_OK;
    if (cudaDeviceSynchronize() != cudaSuccess) return BG_ECUDA;
    if (c->mode == BG_COBG_HELGIVEN_FULLCOLOR) {
        uint32_t k = 0;
        if (cudaMemcpy(&k, (const uint32_t*)c->scratch + 1, sizeof(k), cudaMemcpyDeviceToHost) != cudaSuccess) return BG_ECUDA;
        *count = k;
        return BG_OK;
    }
    if (c->mode != BG_CDBG_GIVEN || !c->prog) return BG_OK;
    return bg::prog_twin_count(c->prog, c->last_N, c->scratch, count) == cudaSuccess ? BG_OK : BG_ECUDA;
}

int bg_eval(bg_ctx* c, void* cuda_stream, long long N, const double* mom, const signed char* hel,
            const signed char* col, double* out) {
    if (!c || N < 0 || c->mode == BG_CDBG_CONTINUOUS) return BG_EINVAL;   // continuous states: bg_eval_continuous
    if (N > 0xFFFFFFFFll) return BG_EINVAL;   // event ids and record positions are 32 bit
    c->last_launches = 0;
    c->last_N = N;
    c->last_auto = false;
    if (N == 0) return BG_OK;
    if (!mom || !out) return BG_EINVAL;
    const bool helsum = (c->mode & BG_HEL_SUM) != 0;
    if (!helsum && !hel) return BG_EINVAL;
    if ((c->mode & BG_COL_GIVEN) && !col) return BG_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t err = cudaSuccess;
    cudaEvent_t ev0 = c->timing ? c->ev0 : nullptr, ev1 = c->timing ? c->ev1 : nullptr;
    c->timed = c->timing != 0;
    if (use_cobg_dd(c)) {
        int rc = ensure_scratch(c, N);
        if (rc != BG_OK) return rc;
        const long long chunk = cobg_dd_chunk(c, N);
        if (ev0) cudaEventRecord(ev0, s);
        for (long long first = 0; first < N && err == cudaSuccess; first += chunk) {
            err = bg::cobg_dd_launch(s, c->n, helsum, c->nperm, c->dC, N, first, std::min(chunk, N - first), mom, hel, out,
                                     c->scratch);
            c->last_launches += 2;
        }
        if (ev1) cudaEventRecord(ev1, s);
        c->last_kernel = "cobg_dd_kernel";
    } else if (use_cobg_auto(c)) {
        int rc = ensure_scratch(c, N);
        if (rc != BG_OK) return rc;
        uint32_t* count = (uint32_t*)c->scratch;      // [0]: double-double list, [1]: second-stage list
        uint32_t* list = count + 64;
        const bool flag = c->precision == 2;
        if (cudaMemsetAsync(count, 0, 64, s) != cudaSuccess) return BG_ECUDA;
        if (ev0) cudaEventRecord(ev0, s);
        bg::CobgCascade cas;
        cas.twin = c->frame ? 1 : 0;
        cas.tau_twin = c->tau_twin;
        cas.tau_twin_ward = c->tau_twin * twin_ward_fraction_cobg(c->n);
        cas.soft_list = list + N; cas.soft_count = count + 1;
        cas.list = nullptr; cas.list_count = nullptr;
        const bool cascade = flag && cas.tau_twin_ward > c->tau;
        if (!cascade) cas.tau_twin_ward = 0.0;
        err = bg::cobg_shared_launch(s, c->cobg, false, false, c->dC, N, mom, hel, out, flag ? c->tau : -1.0, list, count, &cas);
        c->last_launches = 1;
        if (flag && c->timing) cudaEventRecord(c->ev_mid, s);
        if (cascade && err == cudaSuccess) {
            // second stage: the events between the two bounds once more in FP64 in the rotated frame
            cas.twin = c->frame ? 2 : 3;
            cas.list = cas.soft_list; cas.list_count = cas.soft_count;
            err = bg::cobg_shared_launch(s, c->cobg, false, false, c->dC, N, mom, hel, out, c->tau, list, count, &cas);
            c->last_launches++;
        }
        if (flag && err == cudaSuccess) {
            err = bg::cobg_dd_flagged_launch(s, c->n, c->nperm, c->dC, N, list, count, c->sm_count * 2, mom, hel, out);
            c->last_launches++;
        }
        if (ev1) cudaEventRecord(ev1, s);
        c->last_auto = flag;
        c->last_kernel = "cobg_shared_kernel";
    } else if ((c->mode & BG_REC_COBG) && c->mode != BG_COMC_GIVEN) {
        if (ev0) cudaEventRecord(ev0, s);
        if (c->cobg && (c->kernel_opt != 1 || (c->mode & BG_COL_LC))) {
            bg::CobgCascade cas = {c->frame ? 1 : 0, 0.0, 0.0, nullptr, nullptr, nullptr, nullptr};    // (BG_OPT_FRAME)
            err = bg::cobg_shared_launch(s, c->cobg, helsum, (c->mode & BG_COL_LC) != 0, c->dC, N, mom, hel, out, 0.0, nullptr, nullptr, &cas);
            c->last_kernel = "cobg_shared_kernel";
        } else {
            err = bg::cobg_generic_launch(s, c->n, helsum, c->nperm, c->dC, N, mom, hel, out);
            c->last_kernel = "cobg_generic_kernel";
        }
        if (ev1) cudaEventRecord(ev1, s);
        c->last_launches = 1;
    } else if (use_dd(c)) {
        int rc = ensure_scratch(c, N);
        if (rc != BG_OK) return rc;
        const long long chunk = dd_chunk(c, N);
        if (ev0) cudaEventRecord(ev0, s);
        for (long long first = 0; first < N && err == cudaSuccess; first += chunk) {
            err = bg::cdbg_dd_launch(s, c->n, N, first, std::min(chunk, N - first), mom, hel, col, out, c->scratch);
            c->last_launches++;
        }
        if (ev1) cudaEventRecord(ev1, s);
        c->last_kernel = "cdbg_dd_kernel";
    } else if (use_prog(c)) {
        int rc = ensure_scratch(c, N);
        if (rc != BG_OK) return rc;
        const bool flag = c->precision == 2 && c->mode == BG_CDBG_GIVEN;
        if (flag && bg::prog_dd_mode(c->prog) < 0) return BG_EUNSUPPORTED;   // this lane count leaves no room for the re-evaluation
        err = bg::cdbg_prog_launch(s, c->prog, c->sm_count, N, mom, hel, col, out, c->scratch, &c->last_launches, ev0, ev1,
                                   flag ? c->tau : (c->precision == 3 ? -1.0 : (c->precision == 4 ? -2.0 : 0.0)), flag ? c->tau_rho : 0.0,
                                   c->timing ? c->ev_mid : nullptr, flag ? c->tau_twin : 0.0,
                                   flag ? c->tau_twin * twin_ward_fraction(c->n) : 0.0, c->frame != 0);
        c->last_auto = flag;
        c->last_kernel = "cdbg_prog_kernel";
    } else {
        int rc = ensure_scratch(c, N);
        if (rc != BG_OK) return rc;
        const long long chunk = generic_chunk(c, N);
        if (ev0) cudaEventRecord(ev0, s);
        for (long long first = 0; first < N && err == cudaSuccess; first += chunk) {
            const long long count = std::min(chunk, N - first);
            err = bg::cdbg_generic_launch(s, c->n, helsum, N, first, count, mom, hel, col, out, c->scratch);
            c->last_launches++;
        }
        if (ev1) cudaEventRecord(ev1, s);
        c->last_kernel = "cdbg_generic_kernel";
    }
    return err == cudaSuccess ? BG_OK : BG_ECUDA;
}

int bg_eval_continuous(bg_ctx* c, void* cuda_stream, long long N, const double* mom, const double* phi,
                       const double* eta, double* out) {
    if (!c || N < 0 || c->mode != BG_CDBG_CONTINUOUS) return BG_EINVAL;
    c->last_launches = 0;
    if (N == 0) return BG_OK;
    if (!mom || !phi || !eta || !out || !c->prog) return BG_EINVAL;
    int rc = ensure_scratch(c, N);
    if (rc != BG_OK) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaEvent_t ev0 = c->timing ? c->ev0 : nullptr, ev1 = c->timing ? c->ev1 : nullptr;
    c->timed = c->timing != 0;
    const cudaError_t err = bg::cdbg_dense_launch(s, c->prog, c->sm_count, N, mom, phi, eta, out, c->scratch,
                                                  &c->last_launches, ev0, ev1);
    c->last_kernel = "cdbg_prog_kernel";
    return err == cudaSuccess ? BG_OK : BG_ECUDA;
}

int bg_eval_host(bg_ctx* c, long long N, const double* mom, const signed char* hel, const signed char* col,
                 double* out) {
    if (!c || N < 0) return BG_EINVAL;
    if (N == 0) { c->last_launches = 0; return BG_OK; }
    if (!mom || !out) return BG_EINVAL;
    const bool helsum = (c->mode & BG_HEL_SUM) != 0;
    if (!helsum && !hel) return BG_EINVAL;
    if ((c->mode & BG_COL_GIVEN) && !col) return BG_EINVAL;
    int rc = ensure_staging(c, N);
    if (rc != BG_OK) return rc;
    const size_t n = (size_t)c->n;
    const bool colgiven = (c->mode & BG_COL_GIVEN) != 0;
    cudaStream_t s = c->hstream, cs = c->cstream;
    // Chunked pipeline: the copy stream runs ahead with the host->device copies of chunk k+1 (one strided 2-D copy
    // per array: the arrays are event-fastest) while the compute stream evaluates chunk k and returns its results.
    // Every chunk has its own compact region (event stride = its size) inside the staging buffers.
    // Default precision of the colour-dressed path: every bg_eval ends with a double-double pass that is at least one task
    // deep (0.25 ms at n = 6), so chunks are larger (n = 6, 2^20 events: 1.84e8 events/s with 8 chunks, 2.09e8 with 4), and -
    // with default options and small tables (n <= 8) - a second context takes the odd chunks on its own stream: the
    // latency-bound later stages of one chunk then overlap the first pass of the next (2.17e8 with 8 chunks; n = 7, 2^18
    // events: 6.1e7 -> 7.6e7 events/s).  (Two such lanes on device-resident halves of a batch measured 8 % slower than one
    // bg_eval: the gain here is in the gaps the copies leave.)
    const bool cascade = c->precision == 2 && c->mode == BG_CDBG_GIVEN;
    bg_ctx* lane[2] = {c, c};
    if (cascade && N >= 2 * 65536 && c->n <= 8 && c->prog && c->prog_lanes == 0 && c->slab_limit == 0 && c->kernel_opt == 0) {
        if (!c->alt && bg_init(&c->alt, c->n, c->mode) != BG_OK) c->alt = nullptr;
        if (c->alt) {
            bg_ctx* a = c->alt;
            a->precision = c->precision; a->tau = c->tau; a->tau_rho = c->tau_rho; a->tau_twin = c->tau_twin; a->frame = c->frame;
            a->scratch_limit = c->scratch_limit;
            lane[1] = a;
        }
    }
    const long long min_chunk = lane[1] != c ? 65536 : (cascade ? 262144 : 32768);
    int K = (int)std::min<long long>(kHostChunks, N / min_chunk);
    if (K < 1) K = 1;
    long long chunk = (N + K - 1) / K;
    chunk = (chunk + 255) / 256 * 256;
    int launches = 0;
    int k = 0;
    for (long long first = 0; first < N; first += chunk, k++) {
        const long long cnt = std::min(chunk, N - first);
        double* dm = c->d_mom + 4 * n * first;
        signed char* dh = c->d_hel + n * first;
        signed char* dc = c->d_col + 2 * n * first;
        double* dout = c->d_out + first;
        if (cudaMemcpy2DAsync(dm, cnt * 8, mom + first, (size_t)N * 8, cnt * 8, 4 * n, cudaMemcpyHostToDevice, cs) != cudaSuccess)
            return BG_ECUDA;
        if (!helsum && cudaMemcpy2DAsync(dh, cnt, hel + first, (size_t)N, cnt, n, cudaMemcpyHostToDevice, cs) != cudaSuccess)
            return BG_ECUDA;
        if (colgiven && cudaMemcpy2DAsync(dc, cnt, col + first, (size_t)N, cnt, 2 * n, cudaMemcpyHostToDevice, cs) != cudaSuccess)
            return BG_ECUDA;
        bg_ctx* lc = lane[k & 1];
        cudaStream_t ls = lc == c ? s : lc->hstream;
        if (cudaEventRecord(c->chunk_ev[k], cs) != cudaSuccess || cudaStreamWaitEvent(ls, c->chunk_ev[k], 0) != cudaSuccess)
            return BG_ECUDA;
        rc = bg_eval(lc, (void*)ls, cnt, dm, helsum ? nullptr : dh, colgiven ? dc : nullptr, dout);
        if (rc != BG_OK) return rc;
        launches += lc->last_launches;
        if (cudaMemcpyAsync(out + first, dout, sizeof(double) * cnt, cudaMemcpyDeviceToHost, ls) != cudaSuccess) return BG_ECUDA;
    }
    c->last_launches = launches;
    if (cudaStreamSynchronize(s) != cudaSuccess) return BG_ECUDA;
    if (lane[1] != c && cudaStreamSynchronize(lane[1]->hstream) != cudaSuccess) return BG_ECUDA;
    return BG_OK;
}

int bg_generate(void* cuda_stream, int n, long long N, unsigned long long seed, unsigned long long stream_id,
                long long first_event, double sqrt_s, double ptmin, double drmin, int reject_zero_helicities, double* mom,
                signed char* hel, signed char* col) {
    if (n < 4 || n > 12 || N < 0 || !(sqrt_s > 0.0) || first_event < 0) return BG_EINVAL;
    if (N == 0 || (!mom && !hel && !col)) return BG_OK;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return BG_ECUDA;
    return bg::generate_launch((cudaStream_t)cuda_stream, n, N, seed, stream_id, first_event, sqrt_s, ptmin, drmin,
                               reject_zero_helicities, mom, hel, col) == cudaSuccess ? BG_OK : BG_ECUDA;
}

int bg_colour_rule(int n, const signed char* col) {
    if (n < 3 || n > 16 || !col) return BG_EINVAL;
    for (int k = 0; k < 2 * n; k++)
        if (col[k] < 1 || col[k] > 3) return BG_EINVAL;
    return bg::colour_rule_host(n, col) ? 1 : 0;
}

int bg_colour_form_probe(int n, long long E, int iterations, double* ms_dfma, double* ms_dmma, double* max_rel_diff,
                         double* x_host, double* w_host) {
    if (n < 6 || n > 8 || E < 1 || iterations < 1 || !ms_dfma || !ms_dmma || !max_rel_diff) return BG_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return BG_ECUDA;
    return bg::colour_form_probe(n, E, iterations, ms_dfma, ms_dmma, max_rel_diff, x_host, w_host) == cudaSuccess ? BG_OK : BG_ECUDA;
}

int bg_fp64_peak_probe(int iterations, double* tflops) {
    if (!tflops || iterations < 1) return BG_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return BG_ECUDA;
    return bg::fp64_probe(iterations, tflops) == cudaSuccess ? BG_OK : BG_ECUDA;
}

}  // extern "C"

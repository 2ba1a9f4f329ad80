/*
 * Seeded synthetic workload generator (inputs only; none of the method's arithmetic lives here).
 *
 * Stands in for the paper's event source: "We use Rambo [70] to generate the phase-space points"
 * (Sec. 3) with the kinematic cuts of PAPER.md:L331-334 (Sec. 5), at the
 * BASELINE.json settings (sqrt(s) = 1000 GeV, pT > 20 GeV, DeltaR > 0.4, no eta cut), plus the
 * per-event discrete helicity and colour-flow draws of BASELINE.json configs 2-5.
 *
 * Everything is a pure function of (seed, stream, event index, trial index, draw index) through a
 * counter-based SplitMix64 hash, so results do not depend on thread count or on chunking.
 *
 * Layout of outputs is AoS: mom[e][k][4] = (E,px,py,pz), all-outgoing convention (legs 0,1 are the
 * incoming gluons entered with -p_phys); hel[e][k] in {+1,-1}; col[e][k][2] = (i_k, j_k) in {1,2,3}.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC gen.c -o libbgworkload.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

static inline uint64_t sm64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

/* u in (0,1], 53 bits */
static inline double uni(uint64_t seed, uint64_t stream, uint64_t ev, uint64_t trial, uint64_t draw) {
    uint64_t h = sm64(seed);
    h = sm64(h ^ (stream * 0xD1B54A32D192ED03ull));
    h = sm64(h ^ (ev * 0x8CB92BA72F3D8DD7ull));
    h = sm64(h ^ (trial * 0xDB4F0B9175AE2165ull));
    h = sm64(h ^ (draw * 0xA0761D6478BD642Full));
    return (double)((h >> 11) + 1) * (1.0 / 9007199254740992.0);
}

/* Flat massless phase space for the n-2 outgoing legs at total invariant mass sqrt_s (RAMBO, ref. [70]
 * of the paper; textbook algorithm restated): isotropic massless q_i with energies -ln(u u'), then the
 * Lorentz boost + scaling that brings sum(q) to (sqrt_s,0,0,0). */
static void rambo_outgoing(uint64_t seed, uint64_t stream, uint64_t ev, uint64_t trial, int m, double sqrt_s,
                           double (*p)[4]) {
    double q[16][4];
    double Q[4] = {0, 0, 0, 0};
    for (int i = 0; i < m; i++) {
        double c = 2.0 * uni(seed, stream, ev, trial, 4 * i + 0) - 1.0;
        double phi = 2.0 * M_PI * uni(seed, stream, ev, trial, 4 * i + 1);
        double e = -log(uni(seed, stream, ev, trial, 4 * i + 2) * uni(seed, stream, ev, trial, 4 * i + 3));
        double s = sqrt(fmax(0.0, 1.0 - c * c));
        q[i][0] = e;
        q[i][1] = e * s * cos(phi);
        q[i][2] = e * s * sin(phi);
        q[i][3] = e * c;
        for (int mu = 0; mu < 4; mu++) Q[mu] += q[i][mu];
    }
    double M = sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
    double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
    double x = sqrt_s / M, gam = Q[0] / M, a = 1.0 / (1.0 + gam);
    for (int i = 0; i < m; i++) {
        double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
        for (int k = 0; k < 3; k++) p[i][k + 1] = x * (q[i][k + 1] + b[k] * q[i][0] + a * bq * b[k]);
        /* re-project onto the light cone so that p^2 = 0 to rounding */
        p[i][0] = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
    }
    /* Polish: sqrt(Q^2) cancels when the q_i are nearly collinear, which leaves sum(p) off by up to ~1e-7 GeV in
     * rare events.  Two rounds of "remove the residual 3-momentum evenly, re-project, rescale to sqrt_s" bring
     * momentum conservation and masslessness to rounding level (a relative deformation of the event <= 1e-9). */
    for (int it = 0; it < 2; it++) {
        double d[3] = {0, 0, 0};
        for (int i = 0; i < m; i++)
            for (int k = 0; k < 3; k++) d[k] += p[i][k + 1];
        double esum = 0;
        for (int i = 0; i < m; i++) {
            for (int k = 0; k < 3; k++) p[i][k + 1] -= d[k] / m;
            p[i][0] = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
            esum += p[i][0];
        }
        double sc = sqrt_s / esum;
        for (int i = 0; i < m; i++)
            for (int mu = 0; mu < 4; mu++) p[i][mu] *= sc;
    }
}

static int pass_cuts(int m, double (*p)[4], double ptmin, double drmin) {
    double y[16], ph[16];
    for (int i = 0; i < m; i++) {
        double pt = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2]);
        if (!(pt > ptmin)) return 0;
        y[i] = 0.5 * log((p[i][0] + p[i][3]) / (p[i][0] - p[i][3]));
        ph[i] = atan2(p[i][2], p[i][1]);
    }
    if (drmin > 0.0)
        for (int i = 0; i < m; i++)
            for (int j = i + 1; j < m; j++) {
                double dphi = fabs(ph[i] - ph[j]);
                if (dphi > M_PI) dphi = 2.0 * M_PI - dphi;
                double dy = y[i] - y[j];
                if (!(sqrt(dy * dy + dphi * dphi) > drmin)) return 0;
            }
    return 1;
}

/* mom[N][n][4]; trials[N] (may be NULL) receives the number of RAMBO draws used per event. */
int wl_rambo(uint64_t seed, uint64_t stream, int n, long long N, long long first_event, double sqrt_s, double ptmin,
             double drmin, double *mom, int *trials) {
    if (n < 4 || n > 16) return -1;
    int m = n - 2;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < N; e++) {
        double p[16][4];
        uint64_t t = 0;
        for (;; t++) {
            rambo_outgoing(seed, stream, (uint64_t)(first_event + e), t, m, sqrt_s, p);
            if (ptmin <= 0.0 && drmin <= 0.0) break;
            if (pass_cuts(m, p, ptmin, drmin)) break;
        }
        double *o = mom + (size_t)e * n * 4;
        double h = 0.5 * sqrt_s;
        o[0] = -h; o[1] = 0; o[2] = 0; o[3] = -h;
        o[4] = -h; o[5] = 0; o[6] = 0; o[7] = h;
        for (int i = 0; i < m; i++)
            for (int mu = 0; mu < 4; mu++) o[(i + 2) * 4 + mu] = p[i][mu];
        if (trials) trials[e] = (int)t + 1;
    }
    return 0;
}

/* Uniform +-1 per leg; if reject_zero, redraw assignments with fewer than two + or fewer than two -
 * (tree amplitudes vanish identically there; reading g9). */
int wl_helicities(uint64_t seed, uint64_t stream, int n, long long N, long long first_event, int reject_zero,
                  signed char *hel) {
    if (n < 4 || n > 16) return -1;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < N; e++) {
        signed char h[16];
        for (uint64_t t = 0;; t++) {
            int plus = 0;
            for (int k = 0; k < n; k++) {
                h[k] = uni(seed, stream, (uint64_t)(first_event + e), t, k) > 0.5 ? 1 : -1;
                plus += h[k] > 0;
            }
            if (!reject_zero || (plus >= 2 && n - plus >= 2)) break;
        }
        for (int k = 0; k < n; k++) hel[(size_t)e * n + k] = h[k];
    }
    return 0;
}

/* 1 if the directed graph "k -> l iff j_k == i_l (k != l)" has a Hamiltonian cycle. */
static int has_ham_cycle(int n, const signed char *ci, const signed char *cj) {
    unsigned adj[16];
    for (int k = 0; k < n; k++) {
        adj[k] = 0;
        for (int l = 0; l < n; l++)
            if (l != k && cj[k] == ci[l]) adj[k] |= 1u << l;
    }
    /* reach[mask] = set of end vertices of paths that start at vertex 0 and visit exactly mask */
    static _Thread_local unsigned short reach[1 << 16];
    unsigned full = (1u << n) - 1;
    for (unsigned mask = 0; mask <= full; mask++) reach[mask] = 0;
    reach[1] = 1;
    for (unsigned mask = 1; mask <= full; mask += 2) {
        unsigned ends = reach[mask];
        while (ends) {
            int k = __builtin_ctz(ends);
            ends &= ends - 1;
            unsigned nxt = adj[k] & ~mask;
            while (nxt) {
                int l = __builtin_ctz(nxt);
                nxt &= nxt - 1;
                reach[mask | (1u << l)] |= (unsigned short)(1u << l);
            }
        }
    }
    unsigned ends = reach[full];
    while (ends) {
        int k = __builtin_ctz(ends);
        ends &= ends - 1;
        if (adj[k] & 1u) return 1;
    }
    return 0;
}

/* Uniform (i_k, j_k) in {1,2,3}^2 per leg, redrawn until the assignment can have non-zero weight
 * (reading g8): multiset{i} == multiset{j}, a Hamiltonian colour cycle exists, and not all
 * 2n indices equal. col[N][n][2]; trials[N] may be NULL. */
int wl_colours(uint64_t seed, uint64_t stream, int n, long long N, long long first_event, signed char *col,
               int *trials) {
    if (n < 3 || n > 16) return -1;
#pragma omp parallel for schedule(dynamic, 256)
    for (long long e = 0; e < N; e++) {
        signed char ci[16], cj[16];
        uint64_t t = 0;
        for (;; t++) {
            int cnt_i[4] = {0, 0, 0, 0}, cnt_j[4] = {0, 0, 0, 0};
            for (int k = 0; k < n; k++) {
                double u1 = uni(seed, stream, (uint64_t)(first_event + e), t, 2 * k);
                double u2 = uni(seed, stream, (uint64_t)(first_event + e), t, 2 * k + 1);
                int a = 1 + (int)(u1 * 3.0), b = 1 + (int)(u2 * 3.0);
                if (a > 3) a = 3;
                if (b > 3) b = 3;
                ci[k] = (signed char)a;
                cj[k] = (signed char)b;
                cnt_i[a]++;
                cnt_j[b]++;
            }
            if (cnt_i[1] != cnt_j[1] || cnt_i[2] != cnt_j[2] || cnt_i[3] != cnt_j[3]) continue;
            if (cnt_i[1] == n || cnt_i[2] == n || cnt_i[3] == n) continue;
            if (!has_ham_cycle(n, ci, cj)) continue;
            break;
        }
        for (int k = 0; k < n; k++) {
            col[((size_t)e * n + k) * 2 + 0] = ci[k];
            col[((size_t)e * n + k) * 2 + 1] = cj[k];
        }
        if (trials) trials[e] = (int)t + 1;
    }
    return 0;
}

/* exposed for the tests of the rejection rule */
int wl_colour_valid(int n, const signed char *col) {
    signed char ci[16], cj[16];
    int cnt_i[4] = {0, 0, 0, 0}, cnt_j[4] = {0, 0, 0, 0};
    if (n < 3 || n > 16) return -1;
    for (int k = 0; k < n; k++) {
        ci[k] = col[2 * k];
        cj[k] = col[2 * k + 1];
        if (ci[k] < 1 || ci[k] > 3 || cj[k] < 1 || cj[k] > 3) return -1;
        cnt_i[ci[k]]++;
        cnt_j[cj[k]]++;
    }
    if (cnt_i[1] != cnt_j[1] || cnt_i[2] != cnt_j[2] || cnt_i[3] != cnt_j[3]) return 0;
    if (cnt_i[1] == n || cnt_i[2] == n || cnt_i[3] == n) return 0;
    return has_ham_cycle(n, ci, cj);
}

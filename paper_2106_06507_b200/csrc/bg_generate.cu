// On-device event generation: the synthetic workload of workload/gen.c - RAMBO flat massless phase
// space (the paper's event source), the cuts of PAPER.md:L331-334 at BASELINE.json's values, and
// the discrete helicity / colour-flow draws with the rejection rules g8 / g9 of DESIGN.md - one thread per event,
// written straight into the event-fastest arrays bg_eval reads.  The paper's timings include this step (L259).
// Same counter-based SplitMix64 stream as the host generator, so the integer draws are identical; floating-point
// values agree to the last few ulps of the libm / CUDA math functions.
#include "bg_internal.h"

namespace bg {

__host__ __device__ inline uint64_t sm64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
// u in (0,1], 53 bits, a pure function of (seed, stream, event, trial, draw): the hash chain of gen.c, with the part
// that does not depend on the draw index computed once per trial
__host__ __device__ inline uint64_t trial_key(uint64_t seed, uint64_t stream, uint64_t ev, uint64_t trial) {
    uint64_t h = sm64(seed);
    h = sm64(h ^ (stream * 0xD1B54A32D192ED03ull));
    h = sm64(h ^ (ev * 0x8CB92BA72F3D8DD7ull));
    return sm64(h ^ (trial * 0xDB4F0B9175AE2165ull));
}
__host__ __device__ inline double uni(uint64_t key, uint64_t draw) {
    const uint64_t h = sm64(key ^ (draw * 0xA0761D6478BD642Full));
    return (double)((h >> 11) + 1) * (1.0 / 9007199254740992.0);
}

// Rule g8: can the colour-flow assignment have a non-zero amplitude?  A cyclic order of the gluons in which the j of
// each equals the i of the next is an Eulerian circuit of the multigraph with the three colours as nodes and one
// edge i_k -> j_k per gluon: it exists iff every colour has as many outgoing as incoming edges and all edges are
// connected.  (gen.c answers the same question with a Hamiltonian-cycle DP over the gluons; the two are compared
// exhaustively in tests/test_generate.py.)  Assignments with all 2n indices equal vanish as well.
__host__ __device__ inline bool colour_rule(int n, const signed char* ci, const signed char* cj) {
    int out[4] = {0, 0, 0, 0}, in[4] = {0, 0, 0, 0}, parent[4] = {0, 1, 2, 3};
    for (int k = 0; k < n; k++) {
        out[ci[k]]++;
        in[cj[k]]++;
        int a = ci[k], b = cj[k];
        while (parent[a] != a) a = parent[a];
        while (parent[b] != b) b = parent[b];
        if (a != b) parent[a] = b;
    }
    if (out[1] != in[1] || out[2] != in[2] || out[3] != in[3]) return false;
    if (out[1] == n || out[2] == n || out[3] == n) return false;
    int root = -1;
    for (int c = 1; c <= 3; c++) {
        if (out[c] + in[c] == 0) continue;
        int r = c;
        while (parent[r] != r) r = parent[r];
        if (root < 0) root = r;
        else if (r != root) return false;
    }
    return true;
}

// The same rule on packed data without arrays: occ_out / occ_in hold the per-colour edge counts in three 8-bit
// fields, pairs has bit 0 / 1 / 2 set when an edge joins colours {1,2} / {1,3} / {2,3}.
__device__ __forceinline__ bool colour_rule_packed(int n, unsigned occ_out, unsigned occ_in, unsigned pairs) {
    if (occ_out != occ_in) return false;                                  // colour charges balance
    if (occ_out == (unsigned)n || occ_out == ((unsigned)n << 8) || occ_out == ((unsigned)n << 16)) return false;
    const unsigned used = ((occ_out & 0xFFu) ? 1u : 0u) | ((occ_out & 0xFF00u) ? 2u : 0u) | ((occ_out & 0xFF0000u) ? 4u : 0u);
    if (used == 7u) return __popc(pairs) >= 2;                            // three colours: two joining pairs connect them
    if (used == 3u) return (pairs & 1u) != 0;
    if (used == 5u) return (pairs & 2u) != 0;
    if (used == 6u) return (pairs & 4u) != 0;
    return true;                                                          // one colour only (excluded above when n edges)
}

template <int MO>   // number of outgoing gluons n - 2 (compile time: the momenta stay in registers)
__global__ void __launch_bounds__(128)
generate_kernel(int n, long long N, uint64_t seed, uint64_t stream, long long first_event, double sqrt_s, double ptmin,
                double drmin, int reject_zero_hel, double* __restrict__ mom, signed char* __restrict__ hel,
                signed char* __restrict__ col, int blocks_per_role) {
    // blocks [0, B) draw momenta, [B, 2B) helicities, [2B, 3B) colours: warps stay homogeneous
    const int role = blockIdx.x / blocks_per_role;
    const long long e = (long long)(blockIdx.x % blocks_per_role) * blockDim.x + threadIdx.x;
    if (role == 2) {
        // colour flows: ~5 % of uniform draws pass rule g8, so the 32 lanes of a warp try 32 consecutive trials of
        // ONE event at a time and the first valid trial (lowest index, as in the sequential loop) is kept
        if (!col) return;
        const uint64_t cs = stream + (2ull << 20);
        const int lane = threadIdx.x & 31;
        const long long e0 = e - lane;
        for (int j = 0; j < 32; j++) {
            const long long ej = e0 + j;
            if (ej >= N) break;                      // uniform over the warp
            for (uint64_t t0 = 0;; t0 += 32) {
                const uint64_t key = trial_key(seed, cs, (uint64_t)(first_event + ej), t0 + lane);
                uint64_t packed = 0;                 // 4 bits per gluon: (i-1) | (j-1) << 2
                unsigned occ_out = 0, occ_in = 0, pairs = 0;
                for (int k = 0; k < n; k++) {
                    int a = (int)(uni(key, 2 * k) * 3.0), b = (int)(uni(key, 2 * k + 1) * 3.0);
                    a = a > 2 ? 2 : a;
                    b = b > 2 ? 2 : b;
                    packed |= (uint64_t)(a | (b << 2)) << (4 * k);
                    occ_out += 1u << (8 * a);
                    occ_in += 1u << (8 * b);
                    if (a != b) pairs |= 1u << (a + b - 1);   // {0,1} -> bit 0, {0,2} -> bit 1, {1,2} -> bit 2
                }
                const unsigned ok = __ballot_sync(0xFFFFFFFFu, colour_rule_packed(n, occ_out, occ_in, pairs));
                if (ok) {
                    if (lane == __ffs(ok) - 1)
                        for (int k = 0; k < n; k++) {
                            col[(size_t)(2 * k) * N + ej] = (signed char)(1 + ((packed >> (4 * k)) & 3));
                            col[(size_t)(2 * k + 1) * N + ej] = (signed char)(1 + ((packed >> (4 * k + 2)) & 3));
                        }
                    break;
                }
            }
        }
        return;
    }
    if (e >= N) return;
    const uint64_t ev = (uint64_t)(first_event + e);
    constexpr int m = MO;
    const double kPi = 3.14159265358979323846;
    if (role == 0 && mom) {
        double p[MO][4];
        for (uint64_t t = 0;; t++) {
            // RAMBO: isotropic massless q_i with energies -ln(u u'), boosted and scaled to (sqrt_s, 0, 0, 0)
            const uint64_t key = trial_key(seed, stream, ev, t);
            double Q[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int i = 0; i < m; i++) {
                const double c = 2.0 * uni(key, 4 * i + 0) - 1.0;
                const double phi = 2.0 * kPi * uni(key, 4 * i + 1);
                const double en = -log(uni(key, 4 * i + 2) * uni(key, 4 * i + 3));
                const double s = sqrt(fmax(0.0, 1.0 - c * c));
                p[i][0] = en; p[i][1] = en * s * cos(phi); p[i][2] = en * s * sin(phi); p[i][3] = en * c;
                for (int mu = 0; mu < 4; mu++) Q[mu] += p[i][mu];
            }
            const double M = sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
            const double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
            const double x = sqrt_s / M, gam = Q[0] / M, a = 1.0 / (1.0 + gam);
#pragma unroll
            for (int i = 0; i < m; i++) {
                const double q0 = p[i][0], q1 = p[i][1], q2 = p[i][2], q3 = p[i][3];
                const double bq = b[0] * q1 + b[1] * q2 + b[2] * q3;
                p[i][1] = x * (q1 + b[0] * q0 + a * bq * b[0]);
                p[i][2] = x * (q2 + b[1] * q0 + a * bq * b[1]);
                p[i][3] = x * (q3 + b[2] * q0 + a * bq * b[2]);
                p[i][0] = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
            }
            for (int it = 0; it < 2; it++) {   // polish momentum conservation and masslessness (see gen.c)
                double d[3] = {0.0, 0.0, 0.0};
#pragma unroll
                for (int i = 0; i < m; i++)
                    for (int k = 0; k < 3; k++) d[k] += p[i][k + 1];
                double esum = 0.0;
#pragma unroll
                for (int i = 0; i < m; i++) {
                    for (int k = 0; k < 3; k++) p[i][k + 1] -= d[k] / m;
                    p[i][0] = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
                    esum += p[i][0];
                }
                const double sc = sqrt_s / esum;
#pragma unroll
                for (int i = 0; i < m; i++)
                    for (int mu = 0; mu < 4; mu++) p[i][mu] *= sc;
            }
            if (ptmin <= 0.0 && drmin <= 0.0) break;
            bool ok = true;
            double y[MO], ph[MO];
#pragma unroll
            for (int i = 0; i < m; i++) {
                const double pt = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2]);
                ok = ok && pt > ptmin;
                y[i] = 0.5 * log((p[i][0] + p[i][3]) / (p[i][0] - p[i][3]));
                ph[i] = atan2(p[i][2], p[i][1]);
            }
            if (ok && drmin > 0.0)
#pragma unroll
                for (int i = 0; i < m; i++)
#pragma unroll
                    for (int j = i + 1; j < m; j++) {
                        double dphi = fabs(ph[i] - ph[j]);
                        if (dphi > kPi) dphi = 2.0 * kPi - dphi;
                        const double dy = y[i] - y[j];
                        ok = ok && dy * dy + dphi * dphi > drmin * drmin;
                    }
            if (ok) break;
        }
        const double h = 0.5 * sqrt_s;
        const double in0[4] = {-h, 0.0, 0.0, -h}, in1[4] = {-h, 0.0, 0.0, h};
        for (int c = 0; c < 4; c++) {
            mom[(size_t)(0 * 4 + c) * N + e] = in0[c];
            mom[(size_t)(1 * 4 + c) * N + e] = in1[c];
#pragma unroll
            for (int i = 0; i < m; i++) mom[(size_t)((i + 2) * 4 + c) * N + e] = p[i][c];
        }
    }
    if (role == 1 && hel) {
        const uint64_t hs = stream + (1ull << 20);
        signed char hh[12];
        for (uint64_t t = 0;; t++) {
            const uint64_t key = trial_key(seed, hs, ev, t);
            int plus = 0;
            for (int k = 0; k < n; k++) {
                hh[k] = uni(key, k) > 0.5 ? 1 : -1;
                plus += hh[k] > 0;
            }
            if (!reject_zero_hel || (plus >= 2 && n - plus >= 2)) break;
        }
        for (int k = 0; k < n; k++) hel[(size_t)k * N + e] = hh[k];
    }
}

cudaError_t generate_launch(cudaStream_t s, int n, long long N, uint64_t seed, uint64_t stream, long long first_event,
                            double sqrt_s, double ptmin, double drmin, int reject_zero_hel, double* mom, signed char* hel,
                            signed char* col) {
    const int B = (int)((N + 127) / 128);
#define BG_GEN_CASE(MO)                                                                                              \
    case MO:                                                                                                         \
        generate_kernel<MO><<<(unsigned)(3 * B), 128, 0, s>>>(n, N, seed, stream, first_event, sqrt_s, ptmin, drmin, \
                                                              reject_zero_hel, mom, hel, col, B);                     \
        break;
    switch (n - 2) {
        BG_GEN_CASE(2) BG_GEN_CASE(3) BG_GEN_CASE(4) BG_GEN_CASE(5) BG_GEN_CASE(6) BG_GEN_CASE(7) BG_GEN_CASE(8)
        BG_GEN_CASE(9) BG_GEN_CASE(10)
        default: return cudaErrorInvalidValue;
    }
#undef BG_GEN_CASE
    return cudaGetLastError();
}

bool colour_rule_host(int n, const signed char* col /* [n][2] */) {
    signed char ci[16], cj[16];
    for (int k = 0; k < n; k++) { ci[k] = col[2 * k]; cj[k] = col[2 * k + 1]; }
    return colour_rule(n, ci, cj);
}

}  // namespace bg

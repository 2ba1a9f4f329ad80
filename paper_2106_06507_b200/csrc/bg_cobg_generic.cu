// Generic COBG kernel (one thread per event, runtime n <= 8) and the FP64 throughput probe.
//
// COBG, Eq. 20-22 in the V4 form, all (n-2)! orderings A(1, sigma, n) per event, then the
// full-colour quadratic form Eq. 16 with the real symmetric matrix C of Eq. 17:
//   w = a_r^T C a_r + a_i^T C a_i.   Triangular current table in local memory.
#include "bg_internal.h"
#include "bg_math.cuh"

namespace bg {

constexpr int COBG_MAXN = 8;
constexpr int COBG_MAXPERM = 720;

__device__ __forceinline__ int tri(int i, int j) { return j * (j + 1) / 2 + i; }   // i <= j

__device__ cx cobg_one_ordering(int n, const double (*pm)[4], const cx (*ext)[4]) {
    const int m = n - 1;
    cx J[COBG_MAXN * (COBG_MAXN - 1) / 2][4];
    double P[COBG_MAXN * (COBG_MAXN - 1) / 2][4];
    for (int i = 0; i < m; i++)
        for (int c = 0; c < 4; c++) { J[tri(i, i)][c] = ext[i][c]; P[tri(i, i)][c] = pm[i][c]; }
    for (int len = 2; len <= m; len++)
        for (int i = 0; i + len <= m; i++) {
            const int j = i + len - 1;
            for (int c = 0; c < 4; c++) P[tri(i, j)][c] = P[tri(i, j - 1)][c] + pm[j][c];
            cx s3[4], s4[4];
            for (int c = 0; c < 4; c++) { s3[c] = mk(0.0, 0.0); s4[c] = mk(0.0, 0.0); }
            for (int k = i; k < j; k++) {
                v3_acc(s3, P[tri(i, k)], P[tri(k + 1, j)], J[tri(i, k)], J[tri(k + 1, j)], 1.0);
                for (int l = k + 1; l < j; l++) v4_acc(s4, J[tri(i, k)], J[tri(k + 1, l)], J[tri(l + 1, j)]);
            }
            double f3 = kInvSqrt2, f4 = 0.5;
            if (len < m) {
                const double ip2 = 1.0 / mdot(P[tri(i, j)], P[tri(i, j)]);
                f3 *= ip2; f4 *= ip2;
            }
            for (int c = 0; c < 4; c++) J[tri(i, j)][c] = f3 * s3[c] + f4 * s4[c];
        }
    return mdot(ext[n - 1], J[tri(0, m - 1)]);
}

__global__ void __launch_bounds__(128)
cobg_generic_kernel(int n, int helsum, int nperm, const double* __restrict__ C, long long N,
                    const double* __restrict__ mom, const signed char* __restrict__ hel, double* __restrict__ out) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= N) return;
    double p[COBG_MAXN][4];
    for (int k = 0; k < n; k++)
        for (int c = 0; c < 4; c++) p[k][c] = mom[(size_t)(k * 4 + c) * N + e];
    double Ar[COBG_MAXPERM], Ai[COBG_MAXPERM];
    double total = 0.0;
    const int nhel = helsum ? (1 << n) : 1;
    for (int hc = 0; hc < nhel; hc++) {
        cx eps[COBG_MAXN][4];
        for (int k = 0; k < n; k++) {
            const int lam = helsum ? (((hc >> k) & 1) ? 1 : -1) : (int)hel[(size_t)k * N + e];
            polarisation(p[k], lam, eps[k]);
        }
        for (int s = 0; s < nperm; s++) {
            // s-th permutation of gluons 2..n-1 (0-based labels 1..n-2) in lexicographic order
            int avail[COBG_MAXN], order[COBG_MAXN];
            const int mm = n - 2;
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
            double pm[COBG_MAXN][4];
            cx ex[COBG_MAXN][4];
            for (int k = 0; k < n; k++)
                for (int c = 0; c < 4; c++) { pm[k][c] = p[order[k]][c]; ex[k][c] = eps[order[k]][c]; }
            const cx A = cobg_one_ordering(n, pm, ex);
            Ar[s] = A.re; Ai[s] = A.im;
        }
        double w = 0.0;
        for (int s = 0; s < nperm; s++) {
            double tr = 0.0, ti = 0.0;
            for (int s2 = 0; s2 < nperm; s2++) {
                const double c = C[(size_t)s * nperm + s2];
                tr = fma(c, Ar[s2], tr);
                ti = fma(c, Ai[s2], ti);
            }
            w = fma(Ar[s], tr, w);
            w = fma(Ai[s], ti, w);
        }
        total += w;
    }
    out[e] = total;
}

cudaError_t cobg_generic_launch(cudaStream_t s, int n, bool helsum, int nperm, const double* dC, long long N,
                                const double* mom, const signed char* hel, double* out) {
    const int threads = 128;
    const unsigned blocks = (unsigned)((N + threads - 1) / threads);
    cobg_generic_kernel<<<blocks, threads, 0, s>>>(n, helsum ? 1 : 0, nperm, dC, N, mom, hel, out);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// FP64 FMA throughput probe: 8 independent DFMA chains per thread, all SMs.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fp64_probe_kernel(int iters, double* sink) {
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
           a7 = a0 + 7;
    const double m = 1.0000001, c = 1e-7;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const double r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 123.456) sink[0] = r;
}

cudaError_t fp64_probe(int iterations, double* tflops) {
    int dev = 0, sms = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double* sink = nullptr;
    if ((err = cudaMalloc(&sink, 8)) != cudaSuccess) return err;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = sms * 8, threads = 256;
    fp64_probe_kernel<<<blocks, threads>>>(iterations / 4 + 1, sink);   // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 5; rep++) {
        cudaEventRecord(t0);
        fp64_probe_kernel<<<blocks, threads>>>(iterations, sink);
        cudaEventRecord(t1);
        if ((err = cudaEventSynchronize(t1)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        const double flop = 2.0 * 64.0 * (double)iterations * (double)blocks * threads;
        const double tf = flop / (ms * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    *tflops = best;
    return err;
}

}  // namespace bg

// Measurement of step a7, the full-colour quadratic form  w = a_r^T C a_r + a_i^T C a_i  (Eq. 16, PAPER.md:L119-127;
// "the only DMMA candidate"), on its own: the same batched contraction
//     Y[2E x np] = X[2E x np] . C[np x np],   w[e] = X[2e] . Y[2e] + X[2e+1] . Y[2e+1]
// (X = real and imaginary parts of the (n-2)! partial amplitudes of E events) once with plain DFMA row dots - the way
// the COBG kernels do it, one thread per ordering - and once on the FP64 tensor path, mma.sync.m8n8k4.f64 (tcgen05 has
// no FP64 kind).  bg_colour_form_probe times both on synthetic amplitudes and returns their largest relative
// difference; it is a probe (bench.py, tests), not part of bg_eval.
// Measured (B200): n = 7, 2^18 events: row dots 3.04 ms (5.0 TFLOP/s), tensor path 0.99 ms (15.3 TFLOP/s); n = 6: 0.40 /
// 0.06 ms; n = 8 (720 orderings, 2^14 events): 6.9 / 8.4 ms (one 4-warp block per SM: 185 KB of staged rows).  Inside
// the production kernel the form reads the matrix as one byte per entry and costs ~1.2 ms of the 15.8 ms of config 3;
// writing the amplitudes out (503 MB) and running the tensor-path kernel on them instead measured 15.55 ms against
// 15.76 ms fused (-1.4 %) for 0.5 GB more scratch: not adopted, the amplitudes stay on the SM.
#include <algorithm>
#include <vector>

#include "bg_internal.h"

namespace bg {

namespace {

// synthetic amplitudes: a counter-based hash to (-1, 1)
__device__ __forceinline__ double probe_value(unsigned long long i) {
    unsigned long long z = (i + 1) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return (double)(long long)(z >> 11) * (1.0 / 4503599627370496.0) - 1.0;
}

__global__ void probe_fill_kernel(double* __restrict__ X, long long count) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) X[i] = probe_value((unsigned long long)i);
}

// DFMA: one block per event, thread s takes row s of C against the event's amplitudes in shared memory (the scheme
// of cobg_shared_kernel with the matrix read as doubles through L1/L2); np > blockDim: several rows per thread.
__global__ void __launch_bounds__(128)
colour_form_dfma_kernel(int np, long long E, const double* __restrict__ X, const double* __restrict__ C, double* __restrict__ w) {
    extern __shared__ double sh[];     // [2 np] amplitudes, then [4] warp sums
    double* red = sh + 2 * np;
    for (long long e = blockIdx.x; e < E; e += gridDim.x) {
        __syncthreads();
        for (int i = threadIdx.x; i < 2 * np; i += blockDim.x) sh[i] = X[(size_t)e * 2 * np + i];
        __syncthreads();
        double acc = 0.0;
        for (int s = threadIdx.x; s < np; s += blockDim.x) {
            double tr[4] = {0.0, 0.0, 0.0, 0.0}, ti[4] = {0.0, 0.0, 0.0, 0.0};
            const double* col = C + s;         // C is symmetric: column s = row s, consecutive threads read consecutive addresses
            int s2 = 0;
            for (; s2 + 4 <= np; s2 += 4) {
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    const double c = __ldg(col + (size_t)(s2 + u) * np);
                    tr[u] = fma(c, sh[s2 + u], tr[u]);
                    ti[u] = fma(c, sh[np + s2 + u], ti[u]);
                }
            }
            for (; s2 < np; s2++) {
                const double c = __ldg(col + (size_t)s2 * np);
                tr[0] = fma(c, sh[s2], tr[0]);
                ti[0] = fma(c, sh[np + s2], ti[0]);
            }
            acc = fma(sh[s], (tr[0] + tr[1]) + (tr[2] + tr[3]), acc);
            acc = fma(sh[np + s], (ti[0] + ti[1]) + (ti[2] + ti[3]), acc);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, d);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int i = 0; i < (int)blockDim.x / 32; i++) t += red[i];
            w[e] = t;
        }
    }
}

// DMMA: a warp owns 8 rows of X (4 events x {re, im}) and walks the np/8 column tiles of Y; per tile np/4
// mma.sync.m8n8k4.f64 steps.  Fragments (PTX ISA, m8n8k4 .f64): A[row = lane/4][k = lane%4], B[k = lane%4][col = lane/4],
// D[row = lane/4][col = 2 (lane%4) + {0,1}].  np must be a multiple of 8 (24, 120, 720: n = 6, 7, 8).
__device__ __forceinline__ void dmma_m8n8k4(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int WARPS>
__global__ void __launch_bounds__(32 * WARPS)
colour_form_dmma_kernel(int np, long long E, const double* __restrict__ X, const double* __restrict__ C, double* __restrict__ w) {
    extern __shared__ double shx[];    // per warp: [8][np + 4] rows of X (padded: conflict-free fragment loads)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ld = np + 4;
    double* xs = shx + (size_t)warp * 8 * ld;
    const int r = lane >> 2, q = lane & 3;
    const long long groups = (E + 3) / 4;
    for (long long g = (long long)blockIdx.x * WARPS + warp; g < groups; g += (long long)gridDim.x * WARPS) {
        __syncwarp();
        for (int i = lane; i < 8 * np; i += 32) {
            const int row = i / np, c = i - row * np;
            const long long e = g * 4 + (row >> 1);
            xs[row * ld + c] = e < E ? X[((size_t)e * 2 + (row & 1)) * np + c] : 0.0;
        }
        __syncwarp();
        double acc = 0.0;              // partial row dot X[row] . Y[row] over this lane's two columns of every tile
        for (int nt = 0; nt < np / 8; nt++) {
            double d0 = 0.0, d1 = 0.0;
            const double* bcol = C + (size_t)(nt * 8 + r) * np + q;     // B[k][col] = C[k][col] = C[col][k] (symmetric): row col, k fastest
#pragma unroll 6
            for (int kt = 0; kt < np / 4; kt++) dmma_m8n8k4(d0, d1, xs[r * ld + kt * 4 + q], __ldg(bcol + kt * 4));
            acc = fma(d0, xs[r * ld + nt * 8 + 2 * q], acc);
            acc = fma(d1, xs[r * ld + nt * 8 + 2 * q + 1], acc);
        }
        // rows 2j, 2j+1 (lanes 8j .. 8j+7) belong to event j of the group
        acc += __shfl_xor_sync(0xFFFFFFFFu, acc, 1);
        acc += __shfl_xor_sync(0xFFFFFFFFu, acc, 2);
        acc += __shfl_xor_sync(0xFFFFFFFFu, acc, 4);
        const long long e = g * 4 + (lane >> 3);
        if ((lane & 7) == 0 && e < E) w[e] = acc;
    }
}

}  // namespace

cudaError_t colour_form_probe(int n, long long E, int iters, double* ms_dfma, double* ms_dmma, double* max_rel_diff,
                              double* x_host, double* w_host) {
    int np = 1;
    for (int i = 2; i <= n - 2; i++) np *= i;
    if (np % 8 != 0) return cudaErrorInvalidValue;
    std::vector<double> hC((size_t)np * np);
    build_colour_matrix(n, hC.data());
    double *dC = nullptr, *dX = nullptr, *dw0 = nullptr, *dw1 = nullptr;
    cudaError_t err = cudaSuccess;
    auto done = [&](cudaError_t e) {
        cudaFree(dC); cudaFree(dX); cudaFree(dw0); cudaFree(dw1);
        return e;
    };
    if ((err = cudaMalloc(&dC, sizeof(double) * np * np)) != cudaSuccess) return done(err);
    if ((err = cudaMalloc(&dX, sizeof(double) * 2 * np * E)) != cudaSuccess) return done(err);
    if ((err = cudaMalloc(&dw0, sizeof(double) * E)) != cudaSuccess) return done(err);
    if ((err = cudaMalloc(&dw1, sizeof(double) * E)) != cudaSuccess) return done(err);
    cudaMemcpy(dC, hC.data(), sizeof(double) * np * np, cudaMemcpyHostToDevice);
    const long long count = 2ll * np * E;
    probe_fill_kernel<<<(unsigned)((count + 255) / 256), 256>>>(dX, count);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    constexpr int WARPS = 4;
    const size_t smem0 = sizeof(double) * (2 * np + 4), smem1 = sizeof(double) * WARPS * 8 * (np + 4);
    cudaFuncSetAttribute(colour_form_dmma_kernel<WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem1);
    const unsigned g0 = (unsigned)std::min<long long>(E, (long long)sms * 16);
    const unsigned g1 = (unsigned)std::min<long long>((E + 4 * WARPS - 1) / (4 * WARPS), (long long)sms * std::max<size_t>(1, (200 * 1024) / smem1));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float t0 = 0.f, t1 = 0.f;
    for (int it = 0; it < 2; it++) {     // first pass: warm-up
        cudaEventRecord(e0);
        for (int i = 0; i < iters; i++) colour_form_dfma_kernel<<<g0, 128, smem0>>>(np, E, dX, dC, dw0);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&t0, e0, e1);
        cudaEventRecord(e0);
        for (int i = 0; i < iters; i++) colour_form_dmma_kernel<WARPS><<<g1, 32 * WARPS, smem1>>>(np, E, dX, dC, dw1);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&t1, e0, e1);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if ((err = cudaGetLastError()) != cudaSuccess) return done(err);
    std::vector<double> w0((size_t)E), w1((size_t)E);
    cudaMemcpy(w0.data(), dw0, sizeof(double) * E, cudaMemcpyDeviceToHost);
    cudaMemcpy(w1.data(), dw1, sizeof(double) * E, cudaMemcpyDeviceToHost);
    double worst = 0.0;
    for (long long e = 0; e < E; e++) {
        const double d = fabs(w0[e] - w1[e]) / fabs(w0[e]);
        if (!(d <= worst)) worst = d;
    }
    if (x_host) cudaMemcpy(x_host, dX, sizeof(double) * 2 * np * E, cudaMemcpyDeviceToHost);
    if (w_host)
        for (long long e = 0; e < E; e++) w_host[e] = w1[e];
    *ms_dfma = t0 / iters;
    *ms_dmma = t1 / iters;
    *max_rel_diff = worst;
    return done(cudaGetLastError());
}

}  // namespace bg

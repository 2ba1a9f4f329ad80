// Internal declarations shared by the translation units of libbg.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/bg.h"

struct bg_ctx {
    int n;
    int mode;
    int device;
    int sm_count;
    int kernel_opt;            // BG_OPT_KERNEL
    size_t scratch_limit;      // BG_OPT_SCRATCH_LIMIT
    // colour matrix (COBG full colour)
    int nperm;                 // (n-2)!
    double* dC;                // device, nperm x nperm row-major
    double* hC;                // host copy
    // scratch
    void* scratch;
    size_t scratch_bytes;
    // host path staging
    cudaStream_t hstream;
    double* d_mom;
    signed char* d_hel;
    signed char* d_col;
    double* d_out;
    long long staged_events;
    // bookkeeping
    int last_launches;
    const char* last_kernel;
};

namespace bg {

// ---- generic kernels (bg_generic.cu): one thread per event, currents in global scratch -----------------
size_t cdbg_generic_scratch_per_event(int n);
// events [first, first+count) of a batch whose arrays have event stride N
cudaError_t cdbg_generic_launch(cudaStream_t s, int n, bool helsum, long long N, long long first, long long count,
                                const double* mom, const signed char* hel, const signed char* col, double* out,
                                void* scratch);
cudaError_t cobg_generic_launch(cudaStream_t s, int n, bool helsum, int nperm, const double* dC, long long N,
                                const double* mom, const signed char* hel, double* out);

// ---- quad kernel (bg_cdbg_quad.cu): four lanes per event, currents in shared memory ----------------------
bool cdbg_quad_supported(int n);
size_t cdbg_quad_current_bytes(int n);
cudaError_t cdbg_quad_launch(cudaStream_t s, int n, int sm_count, long long N, const double* mom,
                             const signed char* hel, const signed char* col, double* out);

// ---- colour matrix (bg_colour.cpp part of bg_api.cu) ------------------------------------------------------
int build_colour_matrix(int n, double* C /* (n-2)!^2 */);

// ---- FP64 peak probe ----------------------------------------------------------------------------------
cudaError_t fp64_probe(int iterations, double* tflops);

}  // namespace bg

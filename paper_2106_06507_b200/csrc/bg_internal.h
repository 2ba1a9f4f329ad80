// Internal declarations shared by the translation units of libbg.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/bg.h"

namespace bg { struct ProgTable; struct CobgTable; }

constexpr int kHostChunks = 8;   // bg_eval_host pipelines copies and kernels over up to this many chunks

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
    cudaStream_t hstream;      // compute + device->host stream of bg_eval_host
    cudaStream_t cstream;      // host->device copy stream of bg_eval_host (runs ahead of hstream)
    cudaEvent_t chunk_ev[kHostChunks];
    double* d_mom;
    signed char* d_hel;
    signed char* d_col;
    double* d_out;
    long long staged_events;
    bg_ctx* alt;               // bg_eval_host, default precision of the colour-dressed path: a second context (own tables,
                               // scratch and stream) that takes every other chunk, so that the latency-bound later stages
                               // of one chunk overlap the first pass of the next
    // colour-class programs (CDBG, given colours)
    bg::ProgTable* prog;
    bg::CobgTable* cobg;       // sequence tables of the shared-current COBG kernel (n <= 7)
    int prog_lanes;            // BG_OPT_LANES (0 = automatic)
    size_t slab_limit;         // BG_OPT_SMEM_LIMIT (0 = all of shared memory)
    int precision;             // BG_OPT_PRECISION: 0 = FP64, 1 = every event in double-double, 2 = FP64 + double-double
                               // re-evaluation of the events the conditioning flag names (default where available)
    double tau;                // BG_OPT_FLAG_THRESHOLD: Ward-residual threshold of the conditioning flag
    double tau_rho;            // ... and its threshold for the cancellation among the closure contributions
    double tau_twin;           // BG_OPT_FLAG_TWIN: what the second (rotated-frame) FP64 evaluation may differ by
    int frame;                 // BG_OPT_FRAME: 1 = evaluate in the rotated frame (diagnostic)
    cudaEvent_t ev_mid;        // (timing) between the FP64 launches and the re-evaluation
    long long last_N;          // events of the most recent bg_eval (for bg_last_refined)
    bool last_auto;            // ... and whether it ran with the conditioning flag
    // bookkeeping
    int timing;                // BG_OPT_TIMING
    cudaEvent_t ev0, ev1;
    bool timed;
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

// ---- double-double reference path (bg_cdbg_dd.cu): one thread per event, currents in global scratch ---------
size_t cdbg_dd_scratch_per_event(int n);
cudaError_t cdbg_dd_launch(cudaStream_t s, int n, long long N, long long first, long long count, const double* mom,
                           const signed char* hel, const signed char* col, double* out, void* scratch);

size_t cobg_dd_scratch_per_event(int n, bool helsum);
// the events list[0 .. *count) (device) once more in double-double: one block per event, amplitudes in shared memory
cudaError_t cobg_dd_flagged_launch(cudaStream_t s, int n, int nperm, const double* dC, long long N, const uint32_t* list,
                                   const uint32_t* count, int blocks, const double* mom, const signed char* hel, double* out);
cudaError_t cobg_dd_launch(cudaStream_t s, int n, bool helsum, int nperm, const double* dC, long long N, long long first,
                           long long count, const double* mom, const signed char* hel, double* out, void* scratch);

// ---- colour-class program interpreter (bg_cdbg_prog.cu): G lanes per event, currents in shared memory -------
// `like`: a second table for the list launches of that table's records (same closure legs, its tier ranges)
int prog_table_create(int n, int G, size_t slab_limit, bool comc, ProgTable** out, const ProgTable* like = nullptr);   // BG_* code; slab_limit 0 = all of
                                                                                       // shared memory; comc: Eq. 19 programs
int prog_table_create_dense(int n, int G, size_t slab_limit, bool real, ProgTable** out);   // continuous states
void prog_table_destroy(ProgTable* t);
void prog_table_attach_dd(ProgTable* t, ProgTable* dd);    // t takes ownership; the double-double stage then runs dd's programs
size_t prog_state_bytes(const ProgTable* t);               // largest per-event state block
int prog_lanes(const ProgTable* t);
size_t prog_scratch_bytes(const ProgTable* t, long long N);
// tau > 0: events whose Ward residual exceeds tau are evaluated again in double-double arithmetic (ev_mid, if given,
// is recorded between the FP64 launches and that re-evaluation)
cudaError_t cdbg_prog_launch(cudaStream_t s, const ProgTable* t, int sm_count, long long N, const double* mom,
                             const signed char* hel, const signed char* col, double* out, void* scratch,
                             int* launches, cudaEvent_t ev0, cudaEvent_t ev1, double tau, double tau_rho, cudaEvent_t ev_mid,
                             double tau_twin, double tau_twin_ward, bool rotated);
cudaError_t prog_flagged_count(const ProgTable* t, long long N, const void* scratch, long long* count);
cudaError_t prog_twin_count(const ProgTable* t, long long N, const void* scratch, long long* count);
int prog_dd_mode(const ProgTable* t);   // 0 / 1: re-evaluation available (1: with spill); -1: state does not fit

cudaError_t cdbg_dense_launch(cudaStream_t s, const ProgTable* t, int sm_count, long long N, const double* mom,
                              const double* phi, const double* eta, double* out, void* scratch, int* launches,
                              cudaEvent_t ev0, cudaEvent_t ev1);

// ---- shared-current COBG kernel (bg_cobg_shared.cu): one thread group per event, n <= 7 -----------------------
bool cobg_shared_supported(int n);
int cobg_table_create(int n, CobgTable** out);              // BG_* code
void cobg_table_destroy(CobgTable* t);
int cobg_table_set_colour(CobgTable* t, const double* hC);   // optional: compressed colour matrix for the colour form
size_t cobg_shared_current_bytes(const CobgTable* t);
// tau != 0 (given helicities, full colour): flag list of the events whose Ward residual exceeds tau (tau < 0: diagnostic)
// cascade (BG_OPT_PRECISION = 2): second-stage lists and bounds, or a second-stage launch over `list`
struct CobgCascade {
    int twin;                    // bit 0: rotated frame; bit 1: compare with out[e] instead of writing it
    double tau_twin, tau_twin_ward;
    uint32_t* soft_list;         // first stage: receives the events for the second stage
    uint32_t* soft_count;
    const uint32_t* list;        // second stage: the events to evaluate
    const uint32_t* list_count;
};
cudaError_t cobg_shared_launch(cudaStream_t s, const CobgTable* t, bool helsum, bool lc, const double* dC, long long N,
                               const double* mom, const signed char* hel, double* out, double tau = 0.0,
                               uint32_t* flag_list = nullptr, uint32_t* flag_count = nullptr,
                               const CobgCascade* cascade = nullptr);

// ---- colour matrix (bg_colour.cpp part of bg_api.cu) ------------------------------------------------------
int build_colour_matrix(int n, double* C /* (n-2)!^2 */);

// ---- on-device event generation (bg_generate.cu) ---------------------------------------------------------
cudaError_t generate_launch(cudaStream_t s, int n, long long N, uint64_t seed, uint64_t stream, long long first_event,
                            double sqrt_s, double ptmin, double drmin, int reject_zero_hel, double* mom, signed char* hel,
                            signed char* col);
bool colour_rule_host(int n, const signed char* col);

// ---- colour-form probe (bg_colour_probe.cu): a7 alone, DFMA row dots against mma.sync.m8n8k4.f64 -------------
cudaError_t colour_form_probe(int n, long long E, int iters, double* ms_dfma, double* ms_dmma, double* max_rel_diff,
                              double* x_host, double* w_host);

// ---- FP64 peak probe ----------------------------------------------------------------------------------
cudaError_t fp64_probe(int iterations, double* tflops);

}  // namespace bg

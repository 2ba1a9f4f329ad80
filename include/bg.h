/*
 * bg.h — C-ABI of the B200-native Berends-Giele engine (all-gluon tree-level |M|^2, FP64).
 *
 * Method: arxiv 2106.06507, "Many-gluon tree amplitudes on modern GPUs" (PAPER.md = /root/reference/PAPER.md).
 * Conventions: n gluons labelled 1..n, ALL-OUTGOING momenta (sum p = 0;
 * an incoming gluon enters with -p_phys), metric (+,-,-,-), N_c = 3, g_s = 1, Tr(T^a T^b) = delta^ab
 * (PAPER.md:L187).  No averaging, symmetry factor, coupling or sampling weight is applied to `out`.
 *
 * Storage of per-event inputs is event-fastest ("SoA"): element (event e, gluon k, component c) of
 *     mom : mom[(k*4 + c)*N + e]   c = (E, px, py, pz)          double
 *     hel : hel[k*N + e]           +1 / -1 (all-outgoing labels) signed char
 *     col : col[(k*2 + a)*N + e]   a = 0: i_k, a = 1: j_k, values 1..3 (colour-flow indices)
 *     out : out[e]                                              double
 * so that consecutive threads read consecutive addresses.
 *
 * Ownership: every pointer passed to bg_eval is a DEVICE pointer owned by the caller (for instance the
 * data_ptr() of a torch tensor); the library neither frees nor keeps it.  bg_eval_host takes HOST pointers.
 * The context owns the colour matrix and scratch buffers on the device that was current at bg_init.
 *
 * Errors: every int-returning call returns BG_OK (0) or a negative code; nothing throws across the ABI and
 * nothing is printed.  There is no CPU fallback: without a CUDA device bg_init returns BG_ECUDA.
 */
#ifndef BG_H
#define BG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bg_ctx bg_ctx; /* opaque */

enum {
    BG_OK = 0,
    BG_EINVAL = -1,       /* bad argument (n out of range, NULL pointer the mode needs, N < 0, ...) */
    BG_ENOMEM = -2,       /* host or device allocation failed */
    BG_ECUDA = -3,        /* CUDA runtime error (no device, launch failure, ...) */
    BG_EUNSUPPORTED = -4, /* mode / n combination not implemented */
    BG_ELIMIT = -5        /* size beyond the fixed maximum of the no-allocation entry point (bg_eval_static) */
};

/* mode = recursion | helicity treatment | colour treatment */
enum {
    BG_REC_COBG = 0x001,  /* colour-ordered recursion, Eq. 20-22 */
    BG_REC_CDBG = 0x002,  /* colour-dressed recursion, Eq. 28-32 */
    BG_HEL_SUM = 0x010,   /* sum over all 2^n helicity assignments, Eq. 4; hel must be NULL */
    BG_HEL_GIVEN = 0x020, /* one assignment per event in hel */
    BG_COL_FULL = 0x100,  /* full-colour sum sum_{s,s'} C_{ss'} A_s A_s'^*, Eq. 15-17; col NULL */
    BG_COL_LC = 0x400,    /* leading-colour approximation N_c^(n-2) (N_c^2-1) sum_{S_(n-1)} |A|^2, Eq. 33
                             without its O(1/N_c^2) remainder; col NULL; COBG, n <= 8 */
    BG_HEL_CONT = 0x040,  /* continuous polarisation angle phi per gluon, real e(phi) of Eq. 7 */
    BG_COL_CONT = 0x800,  /* continuous colour states: two real unit 3-vectors (eta, etabar) per gluon, Eq. 9, 12 */
    BG_COL_GIVEN = 0x200, /* one colour-flow assignment (i_k, j_k) per gluon per event in col, Eq. 19 */

    BG_COBG_HELSUM_FULLCOLOR = BG_REC_COBG | BG_HEL_SUM | BG_COL_FULL,     /* BASELINE config 1 */
    BG_COBG_HELGIVEN_FULLCOLOR = BG_REC_COBG | BG_HEL_GIVEN | BG_COL_FULL, /* BASELINE config 3 */
    BG_CDBG_GIVEN = BG_REC_CDBG | BG_HEL_GIVEN | BG_COL_GIVEN,             /* BASELINE configs 2, 4, 5 */
    BG_CDBG_HELSUM_COLGIVEN = BG_REC_CDBG | BG_HEL_SUM | BG_COL_GIVEN,
    BG_CDBG_CONTINUOUS = BG_REC_CDBG | BG_HEL_CONT | BG_COL_CONT,          /* the paper's CD_MC sampling */
    BG_COMC_GIVEN = BG_REC_COBG | BG_HEL_GIVEN | BG_COL_GIVEN,            /* Eq. 19 with colour-ordered
                                                                              currents, sampled colour flows (n <= 9) */
    BG_COBG_HELSUM_LC = BG_REC_COBG | BG_HEL_SUM | BG_COL_LC,
    BG_COBG_HELGIVEN_LC = BG_REC_COBG | BG_HEL_GIVEN | BG_COL_LC
};

/* bg_set_option keys */
enum {
    BG_OPT_KERNEL = 1,       /* 0 = automatic choice by n; 1 = generic thread-per-event kernels with currents in
                                global scratch (any n); 2 = colour-class program interpreter, currents in shared
                                memory (BG_CDBG_GIVEN, any n; COBG n <= 8).  BG_CDBG_CONTINUOUS: 1 = the interpreter in
                                complex instead of real arithmetic (rebuilds the program table, synchronises) */
    BG_OPT_SCRATCH_LIMIT = 2,/* upper bound in bytes for the scratch the generic kernels may use (default 16 GiB) */
    BG_OPT_LANES = 3,        /* lanes that cooperate on one event in the program interpreter: 1, 2, 4, ..., 256;
                                0 = automatic.  Rebuilds the class programs (synchronises the device).  With few lanes
                                a warp holds many events; if their double-double state no longer fits in shared memory
                                BG_OPT_PRECISION falls back from 2 to 0 (setting it to 2 then returns BG_EUNSUPPORTED). */
    BG_OPT_TIMING = 4,       /* 1: record CUDA events around the dominant kernel of every bg_eval (bg_last_kernel_ms) */
    BG_OPT_PRECISION = 6,    /* 0 = FP64 kernels only; 1 = every event in double-double arithmetic (BG_CDBG_GIVEN and the COBG
                                full-colour modes: the precision reference on the GPU, slow); 2 (the default of BG_CDBG_GIVEN
                                for n >= 5 and of BG_COBG_HELGIVEN_FULLCOLOR; n = 4 meets 1e-11 in FP64 and defaults to 0) =
                                FP64 kernels plus a conditioning flag per event and re-evaluation of what it names: the
                                colour-flow amplitude of Eq. 19 / 28-32 has near-zeros -
                                helicity-suppressed configurations, cancellations between orderings - where FP64
                                round-off exceeds 1e-11 of the result.  An event is flagged when its Ward residual
                                |p_n . J| / (E_n |eps_n . J|) (J = the current of gluons 1..n-1 of Eq. 22; zero without
                                round-off) exceeds BG_OPT_FLAG_THRESHOLD, or when |A| is less than BG_OPT_FLAG_CANCELLATION
                                times the sum of the moduli of the closure contributions that add up to it (colour-ordered
                                path: the residual summed over the orderings, no cancellation test).  Then a cascade: flagged events whose residual stays below the bound of
                                BG_OPT_FLAG_TWIN are evaluated once more in FP64 in a rotated frame (the same number with
                                independent round-off); those whose two results agree to BG_OPT_FLAG_TWIN keep the first
                                one, the others - and the events the first stage did not send to the second - are
                                evaluated by a double-double instantiation of the same kernel.  3, 4 = diagnostics: `out`
                                receives the Ward residual / the cancellation ratio instead of |M|^2. */
    BG_OPT_FLAG_THRESHOLD = 7,/* Ward-residual threshold in units of 1e-18 (0 = default; BG_CDBG_GIVEN: 1e-13 for n = 4 and
                                n >= 11, 1e-15 for n = 5, 3e-15 for n = 6, 1e-14 for n = 7, 8, 3e-14 for n = 9, 10; COBG: 3e-15 for n <= 5,
                                else 3e-14) */
    BG_OPT_FLAG_CANCELLATION = 8, /* cancellation threshold in units of 1e-6 (0 = default: 3e-3) */
    BG_OPT_FLAG_TWIN = 9,    /* bound of the second stage in units of 1e-18 on |w - w'| / w of the two evaluations (0 = default:
                                BG_CDBG_GIVEN 5e-13; COBG 5e-13 for n <= 5, else 1e-12).  The Ward residual of either may not
                                exceed 0.4 times that number (BG_CDBG_GIVEN, COBG n <= 5) or the same number (COBG n >= 6).  With that residual bound at or below BG_OPT_FLAG_THRESHOLD
                                there is no second stage and every flagged event is evaluated in double-double */
    BG_OPT_FRAME = 10,       /* BG_CDBG_GIVEN (program interpreter) and the COBG modes (shared-current kernel): 1 = evaluate
                                every event in the rotated frame of the second stage (fixed rotation, axis (1,2,3), 1 rad) -
                                |M|^2 is the same to round-off; a
                                diagnostic of Lorentz invariance and of the FP64 error */
    BG_OPT_SMEM_LIMIT = 5    /* program interpreter, >= 128 lanes per event: bytes of shared memory one event's state may
                                take (16 KiB .. 222 KiB, 0 = default); the rest spills to an L2-resident slab.
                                Rebuilds the class programs. */
};

/*
 * Create a context for n gluons (4 <= n <= 12) in the given mode on the current CUDA device.
 * COBG full-colour modes need n <= 8 ((n-2)!^2 colour-matrix entries); they build the colour
 * matrix C of Eq. 17 (exact integers, orderings sigma = permutations of gluons 2..n-1 in lexicographic order)
 * on the host and upload it.  Returns BG_EUNSUPPORTED for other mode combinations.
 */
int bg_init(bg_ctx** ctx, int n, int mode);

/*
 * Evaluate |M|^2 for N events, asynchronously on `cuda_stream` (a cudaStream_t; NULL = default stream).
 *   COBG + FULL colour : out[e] = sum_{sigma,sigma'} C A_sigma A_sigma'^*  (Eq. 16), A from Eq. 20 + 22, for the
 *                        helicities in hel, or summed over all 2^n assignments when the mode has BG_HEL_SUM.
 *   COBG + LC          : out[e] = N_c^(n-2) (N_c^2 - 1) sum over all (n-1)! orderings sigma of gluons 2..n of
 *                        |A(1, sigma)|^2 (Eq. 33), helicities given or summed.
 *   COBG + GIVEN colour: out[e] = |sum over the colour-connected orderings (1, sigma) of A(1, sigma)|^2 - the
 *                        colour-flow decomposition Eq. 19; the same number as CDBG + GIVEN.
 *   CDBG + GIVEN colour: out[e] = |A_{i1 j1 .. in jn}|^2 from the subset recursion Eq. 29-32 closed with gluon n
 *                        (Eq. 22); assignments whose amplitude vanishes identically return exactly 0.0.
 * External currents are the helicity eigenvectors of Eq. 3 in the light-cone gauge of DESIGN.md reading g2.
 * A context serves ONE bg_eval at a time: its scratch (event records, class histogram and ticket buffer of the prepass,
 * flag lists, spill slabs) and its side streams are per context, so two calls in flight on different streams - or a
 * call issued while bg_eval_host is running - race.  Use one context per concurrently used stream; calls on the same
 * stream are ordered by the stream.  N may not exceed 2^32 - 1 (BG_EINVAL).
 * No host synchronisation and no allocation happen here when bg_reserve was called for >= N events; otherwise
 * scratch is (re)allocated first, which synchronises.  Inputs are not validated on the device: non-finite or
 * off-shell momenta give unspecified (possibly NaN) output, never a fault.  N = 0 is a no-op.
 */
int bg_eval(bg_ctx* ctx, void* cuda_stream, long long N, const double* mom, const signed char* hel,
            const signed char* col, double* out);

/*
 * BG_CDBG_CONTINUOUS (n <= 10: the state offsets of the single dense program are 16 bit; n = 10 keeps the top levels
 * in the L2 slab): |A|^2 of the colour-helicity sub-amplitude of Eq. 14 for continuous
 * states - the colour-dressed recursion Eq. 28-32 with external currents  e(p_k, phi_k) x X_k,  e = cos(phi) e1 +
 * sin(phi) e2 (Eq. 7; e1, e2 the unit vectors of the gauge of reading g2) and X_k[h][g] = etabar_k[h] eta_k[g]
 * (Eq. 12 without its trace part, which decouples).  Summing/averaging over the states with the weights of Eq. 13
 * is the caller's business.  DEVICE pointers, event-fastest:  phi[k*N + e];  eta[(k*6 + a)*N + e], a = 0..2 eta,
 * a = 3..5 etabar (unit vectors).  Same stream / allocation rules as bg_eval.
 */
int bg_eval_continuous(bg_ctx* ctx, void* cuda_stream, long long N, const double* mom, const double* phi,
                       const double* eta, double* out);

/*
 * Same computation with HOST buffers (same layouts): copies inputs to the device, runs bg_eval on an internal
 * stream, copies `out` back and waits.  Staging buffers are owned by the context (grown by bg_reserve).
 */
int bg_eval_host(bg_ctx* ctx, long long N, const double* mom, const signed char* hel, const signed char* col,
                 double* out);

/* Pre-allocate scratch (and host-path staging) for up to N events per call, so bg_eval never allocates. */
int bg_reserve(bg_ctx* ctx, long long N);

/* Bytes of device scratch a call with N events uses with the current options (0 for kernels that keep all
 * currents on chip). */
size_t bg_scratch_bytes(const bg_ctx* ctx, long long N);

/* Bytes of current storage (vector + tensor currents) one event occupies in the selected kernel. */
size_t bg_current_bytes_per_event(const bg_ctx* ctx);

int bg_set_option(bg_ctx* ctx, int key, long long value);

/* Copy the (n-2)! x (n-2)! colour matrix (row-major doubles) to a host buffer; BG_EINVAL for CDBG contexts. */
int bg_colour_matrix(const bg_ctx* ctx, double* C_host);

/* Host-only: build the colour matrix of Eq. 17 for n gluons (4 <= n <= 8) into C_host[(n-2)!^2] without a
 * context or a device (this is what bg_init uploads). */
int bg_build_colour_matrix(int n, double* C_host);

/* Number of kernels the most recent bg_eval / bg_eval_host launched. */
int bg_last_launch_count(const bg_ctx* ctx);

/* Device time in milliseconds of the dominant (recursion) kernel of the most recent bg_eval, measured with CUDA
 * events recorded on the caller's stream around that launch.  Only available after
 * bg_set_option(ctx, BG_OPT_TIMING, 1); waits for that launch to finish.  BG_EINVAL if timing is off or nothing ran. */
int bg_last_kernel_ms(bg_ctx* ctx, double* ms);

/* BG_OPT_PRECISION = 2: number of events of the most recent bg_eval that the conditioning flag sent to the
 * double-double re-evaluation and (if BG_OPT_TIMING is on and ms != NULL) the device time of everything after the first
 * FP64 pass (second stage of the cascade + double-double re-evaluation) in milliseconds, which bg_last_kernel_ms
 * includes.  Waits for the device. */
int bg_last_refined(bg_ctx* ctx, long long* flagged, double* ms);

/* Name of the kernel variant the most recent bg_eval used (static string). */
const char* bg_last_kernel_name(const bg_ctx* ctx);

/* BG_OPT_PRECISION = 2: how many events of the most recent bg_eval went through the second stage of the
 * cascade (the rotated-frame FP64 evaluation); bg_last_refined counts those evaluated in double-double.  Synchronises. */
int bg_last_twin(bg_ctx* ctx, long long* count);

/*
 * Host-only introspection of the colour-class program generator behind the BG_CDBG_GIVEN interpreter (no device
 * needed).  counts[9]: how many of the n gluons carry colour code 3*(i-1)+(j-1) = 0..8 (sum = n, 4 <= n <= 12);
 * lanes as in BG_OPT_LANES.  Writes stats[0] = 1 if the class has a non-vanishing colour structure else 0,
 * stats[1] = vertex evaluations per event, stats[2] = interpreter steps (max over lanes, summed over levels),
 * stats[3] = bytes of per-event state, stats[4] = colour code of the gluon chosen as closure leg.
 */
int bg_class_program_stats(int n, int lanes, const int* counts, long long* stats);

/*
 * The same for the BG_COMC_GIVEN programs (Eq. 19, evaluated with the colour-ordered currents
 * of Eq. 20-26; 4 <= n <= 9).  stats[0] = 1 if at least one ordering sigma has all its Kronecker deltas equal
 * to one, stats[1] = vertex evaluations per event (shared between orderings: a sub-sequence current is computed
 * once), stats[2] = interpreter steps, stats[3] = bytes of per-event state, stats[4] = number of such orderings
 * (of (n-1)! with the first gluon fixed).  BG_EINVAL for bad arguments; BG_EUNSUPPORTED for a class with more than
 * 20000 orderings.  (bg_init builds a CO_MC program only where its state fits the 16-bit state offsets - every class
 * for n <= 8; at n = 9 classes with thousands of orderings, 1e-3 of the classes of uniformly drawn colours, are
 * evaluated with their colour-dressed program instead: the same number.)
 */
int bg_comc_program_stats(int n, int lanes, const int* counts, long long* stats);

/*
 * On-device event generation (the paper's timings include it): RAMBO flat massless
 * phase space for the n-2 outgoing gluons at sqrt_s, legs 1, 2 = -(sqrt_s/2)(1,0,0,+-1) in the
 * all-outgoing convention, every outgoing pT > ptmin and pair Delta R > drmin (<= 0 switches a cut
 * off) with the whole event redrawn on failure; helicities uniform +-1 (redrawn when fewer than two + or two -, if
 * reject_zero_helicities); colour-flow indices uniform in {1,2,3} redrawn until the assignment can be non-zero
 * (reading g8).  Counter-based generator: event e of the call is a pure function of (seed, stream_id,
 * first_event + e) and reproduces paper_2106_06507_b200/workload (same integer draws; momenta equal to a few ulps).
 * DEVICE pointers in the layouts of bg_eval; any of mom / hel / col may be NULL (skipped).  Asynchronous on
 * `cuda_stream`; needs no context.
 */
int bg_generate(void* cuda_stream, int n, long long N, unsigned long long seed, unsigned long long stream_id,
                long long first_event, double sqrt_s, double ptmin, double drmin, int reject_zero_helicities, double* mom,
                signed char* hel, signed char* col);

/* Host-only: rule g8 as bg_generate applies it (balanced colour charges, connected colour graph, not all indices
 * equal) for col[n][2] in {1,2,3}; returns 1 / 0, or BG_EINVAL. */
int bg_colour_rule(int n, const signed char* col);

int bg_destroy(bg_ctx* ctx);

const char* bg_strerror(int code);

/*
 * Measure the FP64 FMA throughput of the current device with a register-resident DFMA chain benchmark
 * (all SMs, 8 independent chains per thread).  Writes TFLOP/s (2 flop per FMA) to *tflops.  Used by bench.py
 * as the "alu" roofline denominator; synchronous.
 */
int bg_fp64_peak_probe(int iterations, double* tflops);

/*
 * Measure step a7 alone - the full-colour quadratic form of Eq. 16 for E synthetic amplitude
 * vectors of (n-2)! entries, n = 6, 7, 8 - with plain DFMA row dots (the scheme of the COBG kernels) and on the FP64
 * tensor path (mma.sync.m8n8k4.f64).  Writes the milliseconds per pass of either variant and the largest
 * relative difference of their results; optionally copies the amplitudes (x_host[E][2][(n-2)!]: real parts, then
 * imaginary parts of an event) and the tensor-path results (w_host[E]) to host buffers.  Synchronous, allocates its own
 * device memory.
 */
int bg_colour_form_probe(int n, long long E, int iterations, double* ms_dfma, double* ms_dmma, double* max_rel_diff,
                         double* x_host, double* w_host);

/*
 * The no-allocation entry point.  Some callers cannot call cudaMalloc - code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it - and bg_init / bg_reserve / bg_eval allocate tables and scratch.  bg_eval_static
 * needs no context and calls no cudaMalloc, cudaFree or allocating library routine: it evaluates
 *     out[e] = |A_{i1 j1 .. in jn}|^2   (colour-dressed recursion Eq. 29-32 closed with gluon n, Eq. 22;
 *                                         PAPER.md:L187-213)
 * for given helicities and colour-flow indices with the thread-per-event FP64 kernel (the kernel a BG_CDBG_GIVEN context
 * runs under BG_OPT_KERNEL = 1; no conditioning flag, no double-double re-evaluation: ill-conditioned events carry
 * their FP64 round-off), whose per-event scratch - 2^(n-1) x 513 bytes of sub-currents, subset momenta and colour
 * types - lives in ONE file-scope device array of BG_STATIC_SCRATCH_BYTES that every GPU which loads libbg.so holds
 * until the process exits.
 *   Limit: N <= bg_static_max_events(n) = BG_STATIC_SCRATCH_BYTES / (2^(n-1) x 513): 4088 events at n = 5, 2044 at
 *   n = 6, 511 at n = 8, 31 at n = 12.  Beyond it the call returns BG_ELIMIT and launches nothing; split the batch.
 *   DEVICE pointers in the layouts of bg_eval (mom[n][4][N], hel[n][N], col[n][2][N] in {1,2,3}, out[N]), all owned by
 *   the caller; asynchronous on `cuda_stream`, whose device must be current.  N = 0 is a no-op; n outside 4..12, N < 0
 *   or a NULL pointer with N > 0: BG_EINVAL.
 *   The array is shared by every call in the process and keeps the last call's contents (nothing in it has to start at
 *   zero: the kernel writes each entry of an event before reading it).  Calls on one stream are ordered by the stream;
 *   calls that overlap on the GPU - different streams, or a graph replayed concurrently with itself - RACE.
 *   bg_static_setup resolves the array's device address for the current device (cudaGetSymbolAddress; once per device,
 *   thread-safe); bg_eval_static does so itself on first use, but call bg_static_setup before starting a stream capture.
 */
#define BG_STATIC_SCRATCH_BYTES (32u << 20)
int bg_static_setup(void);
long long bg_static_max_events(int n);     /* host-only; BG_EINVAL for n outside 4..12 */
int bg_eval_static(void* cuda_stream, int n, long long N, const double* mom, const signed char* hel,
                   const signed char* col, double* out);

#ifdef __cplusplus
}
#endif
#endif /* BG_H */

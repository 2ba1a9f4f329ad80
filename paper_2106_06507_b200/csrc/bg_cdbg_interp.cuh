// Program interpreter of the colour-dressed recursion (CDBG, Eq. 28-32, closed with Eq. 22):
// the kernel template cdbg_prog_kernel<G, SPILL, S> and its launcher, shared by the translation units that
// instantiate it - bg_cdbg_prog.cu (S = cx: complex FP64; S = double: real currents of the continuous states) and
// bg_cdbg_prog_dd.cu (S = cxd: complex double-double, the re-evaluation of flagged events).
// See bg_cdbg_prog.cu for the pipeline of one bg_eval and the state layout.
#pragma once
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "bg_internal.h"
#include "bg_math.cuh"
#include "bg_program.h"

namespace bg {

constexpr int kMaxLevels = 2 * kMaxN - 4;   // setup | (main, combine) per popcount 2..n-2 | closure

struct ClassInfo {            // 64 bytes; the interpreter reads the first 16
    uint32_t op_base;         // first op of the class in the op array (units of ProgOp)
    uint16_t state_cx;
    uint8_t closure_code;
    uint8_t valid;
    uint32_t total_steps;     // interpreter steps of the whole program
    uint32_t n_sync;          // how many of them end with a barrier (OPF_SYNC)
    uint16_t level_steps[kMaxLevels];   // steps per level (setup | main, combine per popcount | closure): diagnostics
    uint16_t pad[24 - kMaxLevels];
};

// What the interpreter needs to start an event, in grouping order (written by the scatter kernel).
constexpr int kRecHeaderBytes = 32;

struct alignas(16) EventHeader {
    uint32_t event;           // event id
    uint32_t cls;             // class id (0xFFFFFFFF: colour codes out of range)
    uint64_t perm;            // canonical order: nibble k = original index of canonical gluon k
};
static_assert(sizeof(ClassInfo) == 64, "ClassInfo layout");

constexpr size_t kMaxSlabBytes = 208 * 1024;   // state slab per block (the rest: op ring up to 16 KB, static use)
constexpr int kTiers = 4;     // classes are grouped by state size so that small ones get more warps per SM

struct TierInfo {
    int first_key[kTiers + 1];   // first position (in grouping order) of each tier; [kTiers] = number of classes
    int slab_cx[kTiers];         // state block (complex doubles per event) the tier's launch reserves
};

struct ProgTable {
    int n, G;
    long long num_classes;
    int max_state_cx;
    TierInfo tiers;
    bool dense;               // continuous colour states: one program, nine colour entries per subset current
    bool real;                // ... evaluated in real arithmetic (state elements are doubles)
    int rec_bytes;            // bytes of one event record
    bool spill;               // largest state blocks exceed the slab limit: top of the state in global memory
    int spill_blocks_per_sm;  // resident blocks per SM of the spill kernels (each owns one global slab)
    int sm_count;
    ClassInfo* d_info;
    uint32_t* d_sortkey;      // class id -> position in the order the events are grouped by
    ProgOp* d_ops;
    size_t ops_bytes;
    // small batches: the tier launches run side by side on these streams (fork / join around the caller's stream)
    cudaStream_t aux[kTiers - 1];
    cudaEvent_t fork_ev, join_ev[kTiers - 1];
    bool has_streams;
    uint32_t* d_small;        // [2 (num_classes + 1) + 1] zeroed histogram | cursors | ticket of the fused-scan prepass
    // FP64 launches of warp-shared lane counts (G <= 8): tiers whose state block exceeds cap_cx keep only the first cap_cx
    // elements per event in shared memory - as many as let the register-limited number of blocks fit an SM - and the
    // rest (the highest levels) in the block's L2-resident slab (round 2: n = 6 -6 %, n = 7 -20 %)
    int cap_cx;               // 0: every tier keeps its whole state in shared memory
    int cap_blocks;           // resident blocks per SM of the capped launches (each owns one global slab)
    // double-double re-evaluation of flagged events (BG_OPT_PRECISION = 2): state elements are 32 bytes, so less of
    // the state fits in shared memory
    int dd_mode;              // 1: available (state beyond dd_cap_cx elements per event spills to the L2 slab); -1: not (dense tables)
    int dd_cap_cx;            // state elements per event kept in shared memory: sized so that shared memory allows as many
                              // resident blocks as the 255 registers per thread do
    int dd_spill_blocks;      // resident blocks per SM of the re-evaluation kernels
    long long dd_max_blocks;  // ... and blocks per launch (each owns one global slab; their sum is bounded)
    uint8_t* h_closure;       // host: closure code of every class (what the event records are ordered by)
    // n = 8 with the default lane count: the double-double stage runs the programs of a second table with half the lanes
    // (same closure legs, so the same records): better lane fill where the arithmetic is 15 x as long (measured per
    // event: 0.204 us with 16 lanes against 0.269 with 32)
    ProgTable* dd_table;
};

// how one set of tier launches is sized
struct LaunchShape {
    bool conc = false;        // small batches: tiers side by side on the table's side streams
    int regs = 168;           // registers per thread of the instantiation (resident-block estimate)
    int cap_cx = 0;           // > 0: at most this many state elements per event in shared memory (SPILL kernels)
    bool merged = false;      // one launch for all tiers (list launches)
    long long tasks_hint = 0; // > 0: events this set of launches is expected to process (list launches; default p.N)
    bool hybrid = false;      // SPILL kernel only for the tiers whose state exceeds cap_cx, the others keep all of it in
                              // shared memory (launch_interp<G, false, S> with both kernels instantiated)
    int spill_blocks = 0;     // SPILL: resident blocks per SM (each owns one global slab)
    long long max_blocks = 0; // > 0: at most this many blocks per launch
};

struct ProgParams {
    int n;
    long long N;
    double* out;
    const ClassInfo* info;
    const ProgOp* ops;
    const char* rec;           // [N] event records (header + canonical momenta) grouped by class
    int rec_bytes;             // 32 + 32 n (discrete states) or 32 + 96 n (continuous states)
    int rec_gstride;           // doubles per gluon in a record: 4 or 12
    const uint32_t* bounds;    // [kTiers + 1] record positions where the tiers start (bounds[kTiers] = N)
    int tier;
    int slab_cx;               // complex doubles of state per event in the shared-memory slab
    double2* spill;            // SPILL kernels: global slab, spill_cx complex doubles per block
    int spill_cx;
    int zero;                  // always 0 (see the op prefetch in the interpreter)
    // Conditioning flag (BG_OPT_PRECISION = 2): events whose Ward residual |p_n . J| / (E_n |eps_n . J|) exceeds
    // tau are appended (by record position) to the tier's list for re-evaluation in double-double arithmetic
    double tau2;               // tau^2; 0 = no flagging (negative: diagnostics, the flag quantities instead of |A|^2)
    double tau_rho;            // ... or whose closure contributions cancel to less than tau_rho of their sum of moduli
    uint32_t* flag_list;       // [N] record positions; the list of tier k starts at bounds[k]
    uint32_t* flag_count;      // [kTiers]
    // re-evaluation launches read their tasks from the lists instead of the record ranges
    const uint32_t* list;      // nullptr: all records of the tier
    const uint32_t* list_count;
    uint32_t* ticket;          // [kTiers] next list task of the tier (zeroed with the flag counters)
    // Cascade: events whose Ward residual exceeds tau but not tau_twin are first evaluated once more in FP64
    // in a rotated frame (same value, independent round-off); they go on to the double-double list only if the two
    // results differ by more than tau_twin or the second evaluation's own flag quantities exceed tau_twin / tau_rho.
    // UNSORTED instantiations (n <= 5: the prepass is more than half of a step there): no records - a lane group
    // classifies its event itself and reads the caller's arrays; tasks in input order, one tier
    const double* mom;         // [n][4][N]
    const signed char* hel;    // [n][N]
    const signed char* col;    // [n][2][N]
    int merged;                // 1: the launch serves tiers tier .. kTiers - 1 one after the other (list launches)
    int twin;                  // bit 0: evaluate in the rotated frame (rotate_frame); bit 1: second stage - compare with
                               // out[e] and append to flag_list on disagreement instead of writing out[e]
    double tw2;                // tau_twin^2 (<= tau^2: no second stage, every flagged event goes to flag_list)
    double td;                 // tau_twin as the bound on |w - w'| / w
    uint32_t* soft_list;       // [N] first stage: events for the second stage, by record position, per tier like flag_list
    uint32_t* soft_count;      // [kTiers]
    // Ordered lists (warp-shared lane counts, large batches): the kernels only mark the events - mark[record position] =
    // 1 second stage, 2 double-double, 3 rejected by the second stage - and a compaction kernel builds the lists in
    // record order, i.e. class by class: the events a warp takes from a list then run the same program
    uint8_t* mark;             // nullptr: the kernels append to the lists themselves (one atomic per flagged event)
};

// ---------------------------------------------------------------------------------------------------------
// 4. interpreter
// ---------------------------------------------------------------------------------------------------------
// Per-event state block: offsets below `cap` live in shared memory ([offset][event], event fastest); with SPILL
// the rest (the highest popcount levels, which are read least often) lives in an L2-resident global slab owned by
// the block, accessed with .cg loads/stores (no stale L1 lines).
// element of the state: one complex double (double2) or, for the all-real arithmetic of the continuous states with
// real polarisations, one double
// (bg_cdbg_prog_dd.cu adds the complex double-double element, 32 bytes)
template <class S> struct StateElem;
template <> struct StateElem<cx> {
    using T = double2;
    using R = double;                     // real type of momenta and scale factors
    static constexpr bool kComplex = true, kDD = false;
    static __device__ __forceinline__ cx get(double2 v) { return mk(v.x, v.y); }
    static __device__ __forceinline__ double2 put(cx v) { return make_double2(v.re, v.im); }
    static __device__ __forceinline__ cx make(double re, double im) { return mk(re, im); }
    static __device__ __forceinline__ double2 ldcg(const double2* p) { return __ldcg(p); }
    static __device__ __forceinline__ void stcg(double2* p, double2 v) { __stcg(p, v); }
};
template <> struct StateElem<double> {
    using T = double;
    using R = double;
    static constexpr bool kComplex = false, kDD = false;
    static __device__ __forceinline__ double get(double v) { return v; }
    static __device__ __forceinline__ double put(double v) { return v; }
    static __device__ __forceinline__ double ldcg(const double* p) { return __ldcg(p); }
    static __device__ __forceinline__ void stcg(double* p, double v) { __stcg(p, v); }
};
// real-type helpers with one spelling for double and double-double
__device__ __forceinline__ double r_add(double a, double b) { return a + b; }
__device__ __forceinline__ double r_sub(double a, double b) { return a - b; }
__device__ __forceinline__ double r_from(double x, double) { return x; }
__device__ __forceinline__ double r_hi(double x) { return x; }
// 1/sqrt2 x, and 1 / (sqrt2 P^2)
__device__ __forceinline__ cx s_isqrt2(cx v) { return kInvSqrt2 * v; }
__device__ __forceinline__ double s_isqrt2(double v) { return kInvSqrt2 * v; }
__device__ __forceinline__ double r_isqrt2_over(double p2) { return kInvSqrt2 / p2; }
__device__ __forceinline__ cx s_scale(double f, cx v) { return f * v; }
__device__ __forceinline__ double s_scale(double f, double v) { return f * v; }
__device__ __forceinline__ void ext_current(const double* pk, int lambda, cx* eps) { polarisation(pk, lambda, eps); }


// Debug build (-DBG_BOUNDS_CHECK; compute-sanitizer is not available on every pool): every state access is checked
// against the slab / spill extents and traps, so that `pytest -m gpu` under this build finds an out-of-range offset.
#ifdef BG_BOUNDS_CHECK
#define BG_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define BG_CHECK(cond) do { } while (0)
#endif

template <int EPW, bool SPILL, class S>
struct StateRef {
    using T = typename StateElem<S>::T;
    T* base;
    T* spill;
    int cap;
    int limit;     // (bounds-checked builds) state elements of the largest class
    __device__ __forceinline__ S ld(int o) const {
        BG_CHECK(o >= 0 && (SPILL ? o < limit : o < cap));
        if (SPILL && o >= cap) return StateElem<S>::get(StateElem<S>::ldcg(spill + (size_t)(o - cap) * EPW));
        return StateElem<S>::get(base[o * EPW]);
    }
    __device__ __forceinline__ void st(int o, S v) const {
        BG_CHECK(o >= 0 && (SPILL ? o < limit : o < cap));
        if (SPILL && o >= cap) {
            StateElem<S>::stcg(spill + (size_t)(o - cap) * EPW, StateElem<S>::put(v));
            return;
        }
        base[o * EPW] = StateElem<S>::put(v);
    }
    // a real 4-momentum: two complex elements, or four real ones
    using R = typename StateElem<S>::R;
    __device__ __forceinline__ void ldP(int o, R* P) const {
        if constexpr (StateElem<S>::kComplex) {
            const S p01 = ld(o), p23 = ld(o + 1);
            P[0] = p01.re; P[1] = p01.im; P[2] = p23.re; P[3] = p23.im;
        } else {
#pragma unroll
            for (int c = 0; c < 4; c++) P[c] = ld(o + c);
        }
    }
    __device__ __forceinline__ void stP(int o, const R* P) const {
        if constexpr (StateElem<S>::kComplex) {
            st(o, StateElem<S>::make(P[0], P[1]));
            st(o + 1, StateElem<S>::make(P[2], P[3]));
        } else {
#pragma unroll
            for (int c = 0; c < 4; c++) st(o + c, P[c]);
        }
    }
    // the same from the doubles of an event record
    __device__ __forceinline__ void stPd(int o, const double* P) const {
        R Pr[4];
#pragma unroll
        for (int c = 0; c < 4; c++) Pr[c] = r_from(P[c], R());
        stP(o, Pr);
    }
};

constexpr int kRing = 4;   // op ring per lane: ops are requested kRing - 1 steps before they run

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned dst = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(gmem_src) : "memory");
}

// v or -v: flips the sign bits when m = 0x80000000 (integer pipe)
__device__ __forceinline__ double cneg(double v, int m) {
    return __hiloint2double(__double2hiint(v) ^ m, __double2loint(v));
}
__device__ __forceinline__ cx cneg(cx v, int m) {
    return mk(__hiloint2double(__double2hiint(v.re) ^ m, __double2loint(v.re)),
              __hiloint2double(__double2hiint(v.im) ^ m, __double2loint(v.im)));
}

__device__ __forceinline__ double shfl_xor(double v, int d) { return __shfl_xor_sync(0xFFFFFFFFu, v, d); }
__device__ __forceinline__ cx shfl_xor(cx v, int d) {
    return mk(__shfl_xor_sync(0xFFFFFFFFu, v.re, d), __shfl_xor_sync(0xFFFFFFFFu, v.im, d));
}

__device__ __forceinline__ int hi_word(cx v) { return __double2hiint(v.re); }
__device__ __forceinline__ int hi_word(double v) { return __double2hiint(v); }

__device__ __forceinline__ EventHeader ld_header(const char* h) {
    const uint4 v = __ldcg(reinterpret_cast<const uint4*>(h));   // streamed once: not through L1
    EventHeader r;
    r.event = v.x; r.cls = v.y; r.perm = (uint64_t)v.z | ((uint64_t)v.w << 32);
    return r;
}

// What the prepass computes for one event, for the UNSORTED instantiations: the class of the colour assignment (rank of
// the multiset of colour codes, as class_rank / cdbg_classify_kernel), the canonical order (codes ascending, original
// order inside a code, the last gluon with the class's closure code at the end: nibble k of perm = original index of
// canonical gluon k) and the helicity bits 48 + k of the canonical gluons.
static __constant__ unsigned c_multisets[kMaxN + 1][kNumCodes] = {   // c_multisets[r][t] = multisets of size r from t kinds, C(r + t - 1, r)
    {1, 1, 1, 1, 1, 1, 1, 1, 1},
    {0, 1, 2, 3, 4, 5, 6, 7, 8},
    {0, 1, 3, 6, 10, 15, 21, 28, 36},
    {0, 1, 4, 10, 20, 35, 56, 84, 120},
    {0, 1, 5, 15, 35, 70, 126, 210, 330},
    {0, 1, 6, 21, 56, 126, 252, 462, 792},
    {0, 1, 7, 28, 84, 210, 462, 924, 1716},
    {0, 1, 8, 36, 120, 330, 792, 1716, 3432},
    {0, 1, 9, 45, 165, 495, 1287, 3003, 6435},
    {0, 1, 10, 55, 220, 715, 2002, 5005, 11440},
    {0, 1, 11, 66, 286, 1001, 3003, 8008, 19448},
    {0, 1, 12, 78, 364, 1365, 4368, 12376, 31824},
    {0, 1, 13, 91, 455, 1820, 6188, 18564, 50388}};
__device__ __forceinline__ EventHeader classify_event(const ProgParams& p, long long e) {
    const int n = p.n;
    EventHeader h;
    h.event = (uint32_t)e; h.cls = 0xFFFFFFFFu; h.perm = 0;
    int cnt[kNumCodes];
#pragma unroll
    for (int c = 0; c < kNumCodes; c++) cnt[c] = 0;
    bool ok = true;
    uint64_t cw = 0;
    for (int k = 0; k < n; k++) {
        const int i = p.col[(size_t)(2 * k) * p.N + e] - 1, jj = p.col[(size_t)(2 * k + 1) * p.N + e] - 1;
        ok = ok && i >= 0 && i < 3 && jj >= 0 && jj < 3;
        const int code = ok ? 3 * i + jj : 0;
        cw |= (uint64_t)code << (4 * k);
#pragma unroll
        for (int c = 0; c < kNumCodes; c++) cnt[c] += code == c;
    }
    if (!ok) return h;
    unsigned rank = 0;
    int r = n;
#pragma unroll
    for (int t = 0; t < kNumCodes - 1; t++) {
        for (int c = 0; c < cnt[t]; c++) rank += c_multisets[r - c][kNumCodes - 1 - t];
        r -= cnt[t];
    }
    const uint4 ci = __ldg(reinterpret_cast<const uint4*>(p.info + rank));
    h.cls = rank;
    if (!((ci.y >> 24) & 0xFF)) return h;          // the amplitude of this class vanishes identically
    const int closure = (int)((ci.y >> 16) & 0xFF);
    int lastk = 0;
    for (int k = 0; k < n; k++)
        if ((int)((cw >> (4 * k)) & 0xF) == closure) lastk = k;
    uint64_t start = 0, pm = 0;
    int before = 0;
#pragma unroll
    for (int c = 0; c < kNumCodes; c++) {
        start |= (uint64_t)before << (4 * c);
        before += cnt[c] - (c == closure ? 1 : 0);
    }
    for (int k = 0; k < n; k++) {
        const int at = k == lastk ? n - 1 : (int)((start >> (4 * (int)((cw >> (4 * k)) & 0xF))) & 0xF);
        if (k != lastk) start += 1ull << (4 * (int)((cw >> (4 * k)) & 0xF));
        pm |= (uint64_t)k << (4 * at);
        if (p.hel[(size_t)k * p.N + e] > 0) pm |= 1ull << (48 + at);
    }
    h.perm = pm;
    return h;
}

template <int G, bool SPILL, class S, bool UNSORTED = false>
__global__ void __launch_bounds__(G > 32 ? G : 32) cdbg_prog_kernel(const ProgParams p) {
    // G <= 32: one warp per block, EPW = 32/G events per warp.  G > 32: one event per block of G threads.
    // S: complex currents (cx) or, for continuous states with real polarisations, real ones (double).
    constexpr int EPW = G >= 32 ? 1 : 32 / G;
    using T = typename StateElem<S>::T;
    using R = typename StateElem<S>::R;
    constexpr bool kComplex = StateElem<S>::kComplex;
    constexpr bool kTwinOk = kComplex && !StateElem<S>::kDD;     // the FP64 discrete-state kernels
    extern __shared__ double2 smem_raw[];
    T* const smem = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x;
    const int q = lane % EPW, g = lane / EPW;
    constexpr int kBlock = G > 32 ? G : 32;
    constexpr bool kUseRing = G >= 8;
    constexpr bool kEarlyRing = kUseRing && G <= 64;   // op read from the ring one step ahead (G >= 128: measured 1 % slower)
    // [kRing][kBlock] behind the state slab (rounded up to 16 bytes)
    uint4* const ring = reinterpret_cast<uint4*>(smem_raw + ((size_t)p.slab_cx * EPW * sizeof(T) + 15) / 16) + lane;
    StateRef<EPW, SPILL, S> st_;
    st_.base = smem + q;
    // the block's slab in global memory, [offset - cap][event] like the shared one
    st_.spill = SPILL ? reinterpret_cast<T*>(p.spill) + (size_t)blockIdx.x * p.spill_cx * EPW + q : nullptr;
    st_.cap = p.slab_cx;
    st_.limit = p.spill_cx;
    // one launch per tier, or (merged: list launches, whose tiers share one launch shape) this tier and all after it
    const int tier_end = p.merged ? kTiers : p.tier + 1;
    for (int tier = p.tier; tier < tier_end; tier++) {
        // tasks: the records of the tier, or (re-evaluation) the record positions in the tier's flag list
        const long long first = UNSORTED ? 0 : (long long)p.bounds[tier];
        const long long end = p.list ? first + p.list_count[tier] : (UNSORTED ? p.N : (long long)p.bounds[tier + 1]);
        const long long ntasks = (end - first + EPW - 1) / EPW;
        auto rec_pos = [&](long long i) -> long long { return p.list ? (long long)__ldg(p.list + i) : i; };
        // the header of the event at record position pos (UNSORTED: of event pos, worked out here)
        auto get_header = [&](long long pos) -> EventHeader {
            if constexpr (UNSORTED) return classify_event(p, pos);
            else return ld_header(p.rec + (size_t)pos * p.rec_bytes);
        };
        const int n = p.n;
        // lanes of one event (same q) run the same program and meet at its barriers; events of different classes in
        // one warp pass different numbers of barriers, so the barrier names only the event's own lanes
        unsigned evmask = 0;
#pragma unroll
        for (int i = 0; i < (G < 32 ? G : 32); i++) evmask |= 1u << (q + i * EPW);

        // the header of a task is loaded one task ahead; the inputs of the next task are prefetched into L2 while
        // the current one computes (events come in class order, so their rows are scattered over the input arrays)
        EventHeader hnext;
        hnext.event = 0; hnext.cls = 0xFFFFFFFFu; hnext.perm = 0;
        // Tasks: record ranges are dealt round-robin (task += gridDim.x: the records are sorted longest program first).
        // List tasks (re-evaluation) arrive in the random order of the flag appends and take 14 x longer each, so a static
        // deal leaves a long tail: they are handed out by a ticket counter instead, fetched one task ahead.
        auto next_ticket = [&]() -> long long {
            if constexpr (G <= 32) {
                unsigned v = 0;
                if (lane == 0) v = atomicAdd(p.ticket + tier, 1u);
                return (long long)__shfl_sync(0xFFFFFFFFu, v, 0);
            } else {
                __shared__ unsigned tk;
                __syncthreads();
                if (lane == 0) tk = atomicAdd(p.ticket + tier, 1u);
                __syncthreads();
                return (long long)tk;
            }
        };
        long long task = p.list ? next_ticket() : (long long)blockIdx.x;
        long long task_next = task < ntasks ? (p.list ? next_ticket() : task + gridDim.x) : ntasks;
        long long pos_next = 0;    // record position of the next task's event (equals its index unless a list is read)
        if (task < ntasks) {
            const long long idx = first + task * EPW + q;
            if (idx < end) {
                pos_next = rec_pos(idx);
                hnext = get_header(pos_next);
            }
        }
        // carried from one task to the next: the class info of the next event, requested at the first barrier of the
        // current task (one load less in the chain header -> info -> ops -> inputs at the start of a task)
        uint4 ci_next = make_uint4(0, 0, 0, 0);
        bool ci_next_ok = false;
        for (; task < ntasks; task = task_next, task_next = task_next < ntasks ? (p.list ? next_ticket() : task_next + gridDim.x) : ntasks) {
            const long long idx0 = first + task * EPW + q;
            const bool have = idx0 < end;
            const long long idx = p.list ? pos_next : idx0;          // record position
            const EventHeader h = hnext;
            long long idx_next = 0;
            {
                const long long idx2 = first + task_next * EPW + q;
                hnext.event = 0; hnext.cls = 0xFFFFFFFFu; hnext.perm = 0;
                idx_next = idx2;
                if (task_next < ntasks && idx2 < end) {
                    if (p.list) idx_next = pos_next = rec_pos(idx2);
                    hnext = get_header(idx_next);
                }
            }
            const long long e = h.event;
            const uint32_t cls = have ? h.cls : 0xFFFFFFFFu;
            const double* mrec = UNSORTED ? nullptr
                                          : reinterpret_cast<const double*>(p.rec + (size_t)(have ? idx : first) * p.rec_bytes + kRecHeaderBytes);
            const uint64_t perm = h.perm;
            // component c of the momentum of canonical gluon k: from the record, or (UNSORTED) from the caller's array
            auto ldm = [&](int k, int c) -> double {
                if constexpr (UNSORTED) {
                    const int orig = (int)((perm >> (4 * k)) & 0xF);
                    return __ldg(p.mom + (size_t)(orig * 4 + c) * p.N + (have ? e : 0));
                } else {
                    return __ldcg(mrec + k * p.rec_gstride + c);
                }
            };
            // discrete states: the setup level gives gluon k to lane k % G, so the lane's first momentum is requested
            // here, ahead of the dependent loads class info -> ops that the setup ops themselves wait for
            const bool discrete = !kUseRing && p.rec_gstride == 4 && kComplex;   // (G >= 8: measured 1-2 % slower)
            double pk[4] = {0.0, 0.0, 0.0, 0.0};
            if (discrete && g < n) {
#pragma unroll
                for (int c = 0; c < 4; c++) pk[c] = ldm(g, c);
                if constexpr (kTwinOk) { if (p.twin & 1) rotate_frame(pk); }
            }
            uint4 ci = ci_next;
            if (!ci_next_ok) ci = __ldg(reinterpret_cast<const uint4*>(p.info + (cls == 0xFFFFFFFFu ? 0 : cls)));
            ci_next_ok = false;
            const bool valid = cls != 0xFFFFFFFFu && ((ci.y >> 24) & 0xFF);
            const ProgOp* ops = p.ops + ci.x + g;
            const int total = valid ? (int)ci.z : 0;
            bool prefetched = false;

            S amp = s_zero<S>();
            S wamp = s_zero<S>();     // Ward residual  sqrt2 p_n . J({1..n-1})  (exactly zero without round-off)
            double asum = 0.0;        // sum of |Re| + |Im| of the closure contributions that add up to the amplitude
            S acc[4], tacc[6];
            R Pt[4];
#pragma unroll
            for (int c = 0; c < 4; c++) { acc[c] = s_zero<S>(); Pt[c] = r_from(0.0, R()); }
#pragma unroll
            for (int c = 0; c < 6; c++) tacc[c] = s_zero<S>();

            // The lane's ops travel global -> shared by cp.async, kRing - 1 steps ahead, into a private ring (no
            // registers are held across the latency and nothing else reads these slots); the table ends with spare rows.
            // With few lanes per event (G <= 4) the program of a class is small and stays in L1: plain loads, two steps
            // ahead, are cheaper there.
            auto first_barrier_done = [&]() {
                prefetched = true;
                if (hnext.cls != 0xFFFFFFFFu) {
                    // the next event's record (a few 128-byte lines) is pulled into L2 meanwhile
                    if constexpr (!UNSORTED)
                        for (int k = g * 128; k < p.rec_bytes; k += G * 128)
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.rec + (size_t)idx_next * p.rec_bytes + k));
                    if constexpr (kUseRing) {      // (G <= 4: measured neutral to slightly slower)
                        ci_next = __ldg(reinterpret_cast<const uint4*>(p.info + hnext.cls));
                        ci_next_ok = true;
                    }
                }
            };
            // Momentum conservation holds for double-precision inputs only to round-off, and the recursion never uses the
            // momentum of the closing gluon: closing with another gluon than input gluon n evaluates a slightly different
            // continuation of the amplitude off the momentum-conserving surface - a relative difference of 1e-16 times the
            // event's condition number, inside the FP64 kernels' own round-off but not inside the re-evaluation's.  The
            // double-double kernel therefore gives input gluon n, when the class closes with another one, the momentum
            // -(sum of the others): exactly the momentum flow of the recursion closed with gluon n (oracle, Eq. 22).
            int kstar = -1;
            if constexpr (StateElem<S>::kDD) {
                for (int k = 0; k + 1 < n; k++)
                    if ((int)((perm >> (4 * k)) & 0xF) == n - 1) kstar = k;
            }
            auto store_ext_momentum = [&](int kk, int offPt, const double* pk) {
                if constexpr (StateElem<S>::kDD) {
                    if (kk == kstar) {
                        R Pe[4];
#pragma unroll
                        for (int c = 0; c < 4; c++) Pe[c] = r_from(0.0, R());
                        for (int j = 0; j < n; j++) {
                            if (j == kk) continue;
#pragma unroll
                            for (int c = 0; c < 4; c++) Pe[c] = r_sub(Pe[c], r_from(ldm(j, c), R()));
                        }
                        st_.stP(offPt, Pe);
                        return;
                    }
                }
                st_.stPd(offPt, pk);
            };
            const int s0 = (discrete && total > 0) ? (n + G - 1) / G : 0;     // steps of the setup level done up front
            uint4 r0 = make_uint4(0, 0, 0, 0), r1 = r0;
            if constexpr (kUseRing) {
                if (total > 0) {
#pragma unroll
                    for (int i = 0; i < kRing - 1; i++) {
                        cp_async16(ring + ((s0 + i) % kRing) * kBlock, ops + (size_t)(s0 + i) * G);
                        asm volatile("cp.async.commit_group;" ::: "memory");
                    }
                    if constexpr (kEarlyRing) {
                        asm volatile("cp.async.wait_group %0;" ::"n"(kRing - 2) : "memory");
                        r0 = ring[(s0 % kRing) * kBlock];
                    }
                }
            } else {
                r0 = __ldg(reinterpret_cast<const uint4*>(ops + (size_t)s0 * G));
                r1 = __ldg(reinterpret_cast<const uint4*>(ops + (size_t)(s0 + 1) * G));
            }
            if constexpr (kComplex) {
                // setup level (discrete states): external currents eps(p_k, lambda_k) and momenta, Eq. 20 / g1-g5
                int k = g;
                for (int s = 0; s < s0; s++) {
                    const uint4 raw = __ldg(reinterpret_cast<const uint4*>(ops + (size_t)s * G));
                    const int kn = k + G;
                    double pn[4] = {0.0, 0.0, 0.0, 0.0};
                    if (kn < n) {
#pragma unroll
                        for (int c = 0; c < 4; c++) pn[c] = ldm(kn, c);
                        if constexpr (kTwinOk) { if (p.twin & 1) rotate_frame(pn); }
                    }
                    if ((raw.z >> 16) & OPF_EXT) {
                        const int kk = (int)raw.w;
                        if (kk != k) {      // another dealing of the gluons than k % G: fetch what the op names
#pragma unroll
                            for (int c = 0; c < 4; c++) pk[c] = ldm(kk, c);
                            if constexpr (kTwinOk) { if (p.twin & 1) rotate_frame(pk); }
                        }
                        S eps[4];
                        ext_current(pk, ((perm >> (48 + kk)) & 1) ? 1 : -1, eps);
                        const int offDst = raw.y >> 16, offPt = raw.z & 0xFFFF;
#pragma unroll
                        for (int c = 0; c < 4; c++) st_.st(offDst + c, eps[c]);
                        if (offPt != 0xFFFF) store_ext_momentum(kk, offPt, pk);
                    }
#pragma unroll
                    for (int c = 0; c < 4; c++) pk[c] = pn[c];
                    k = kn;
                }
                if (s0 > 0) {
                    if constexpr (G > 32) __syncthreads(); else __syncwarp(evmask);
                    first_barrier_done();
                }
            }
            {
                for (int s = s0; s < total; s++) {
                    uint4 raw, r2 = r1;
                    if constexpr (kUseRing) {
                        cp_async16(ring + ((s + kRing - 1) % kRing) * kBlock, ops + (size_t)(s + kRing - 1) * G);
                        asm volatile("cp.async.commit_group;" ::: "memory");
                        if constexpr (kEarlyRing) {
                            asm volatile("cp.async.wait_group %0;" ::"n"(kRing - 2) : "memory");
                            raw = r0;
                            r2 = ring[((s + 1) % kRing) * kBlock];     // the next step's op leaves the ring one step early
                        } else {
                            asm volatile("cp.async.wait_group %0;" ::"n"(kRing - 1) : "memory");
                            raw = ring[(s % kRing) * kBlock];
                        }
                    } else {
                        raw = r0;
                        const ProgOp* src = ops + (size_t)(s + 2) * G;
                        r2 = __ldg(reinterpret_cast<const uint4*>(src));
                    }
                    const int offA = raw.x & 0xFFFF, offB = raw.x >> 16;
                    const int offP1 = raw.y & 0xFFFF, offDst = raw.y >> 16;
                    const int offPt = raw.z & 0xFFFF;
                    const unsigned flags = raw.z >> 16;
                    if (flags & OPF_VALID) {
                        S a[4], b[4];
#pragma unroll
                        for (int c = 0; c < 4; c++) { a[c] = st_.ld(offA + c); b[c] = st_.ld(offB + c); }
                        R P1[4], P2[4];
                        st_.ldP(offP1, P1);
                        if (flags & OPF_FIRST) {
#pragma unroll
                            for (int c = 0; c < 4; c++) acc[c] = s_zero<S>();
#pragma unroll
                            for (int c = 0; c < 6; c++) tacc[c] = s_zero<S>();
                            const int offP2 = (int)(raw.w & 0xFFFF);
                            R Pb[4];
                            st_.ldP(offP2, Pb);
#pragma unroll
                            for (int c = 0; c < 4; c++) Pt[c] = r_add(P1[c], Pb[c]);
                        }
#pragma unroll
                        for (int c = 0; c < 4; c++) P2[c] = r_sub(Pt[c], P1[c]);
                        // X(a,b) is linear in the pair (a, T_a): a negative vertex flips the sign bits of that pair
                        // (integer pipe) instead of multiplying every term by -1 on the FP64 pipe
                        const int neg = (flags & OPF_NEG) ? (int)0x80000000 : 0;
#pragma unroll
                        for (int c = 0; c < 4; c++) a[c] = cneg(a[c], neg);
                        v3_acc(acc, P1, P2, a, b, 1.0);
                        if (flags & OPF_TENB) {
                            S T[6];
#pragma unroll
                            for (int c = 0; c < 6; c++) T[c] = st_.ld(offB + 4 + c);
                            tcontract_acc(acc, T, a, 1.0);
                        }
                        if (flags & OPF_TENA) {
                            S T[6];
#pragma unroll
                            for (int c = 0; c < 6; c++) T[c] = cneg(st_.ld(offA + 4 + c), neg);
                            tcontract_acc(acc, T, b, -1.0);
                        }
                        if (!(flags & OPF_CLOSURE)) tbuild_acc(tacc, a, b, 1.0);
                        if (flags & OPF_PARTIAL) {
                            // chunk of a split target: raw sums to its scratch slot, finished by a COMBINE op
#pragma unroll
                            for (int c = 0; c < 4; c++) st_.st(offDst + c, acc[c]);
#pragma unroll
                            for (int c = 0; c < 6; c++) st_.st(offDst + 4 + c, tacc[c]);
                        } else if (flags & OPF_LAST) {
                            if (flags & OPF_CLOSURE) {
                                S en[4];
#pragma unroll
                                for (int c = 0; c < 4; c++) en[c] = st_.ld(offDst + c);
                                const S term = s_isqrt2(mdot(en, acc));
                                amp = amp + term;
                                // Ward identity: the full current is conserved, P . J = 0 with P = P(1..n-1) = -p_n
                                if constexpr (kComplex && !StateElem<S>::kDD) {
                                    wamp = wamp + mdot(Pt, acc);
                                    asum += fabs(term.re) + fabs(term.im);
                                }
                            } else {
                                const R f = r_isqrt2_over(mdot(Pt, Pt));
#pragma unroll
                                for (int c = 0; c < 4; c++) acc[c] = s_scale(f, acc[c]);
#pragma unroll
                                for (int c = 0; c < 6; c++) tacc[c] = s_isqrt2(tacc[c]);
                                if (!(flags & OPF_NOSTORE)) {
#pragma unroll
                                    for (int c = 0; c < 4; c++) st_.st(offDst + c, acc[c]);
#pragma unroll
                                    for (int c = 0; c < 6; c++) st_.st(offDst + 4 + c, tacc[c]);
                                }
                                if (flags & OPF_STOREP) {
                                    st_.stP(offPt, Pt);
                                }
                            }
                        }
                    } else if (flags & OPF_FUSED) {
                        // closure vertex X(eps_k, J(pi)) . eps_n with J(pi), T(pi) still in acc / tacc, P(pi) in Pt
                        S a[4], x[4], en[4];
                        R P1[4];
#pragma unroll
                        for (int c = 0; c < 4; c++) { a[c] = st_.ld(offA + c); x[c] = s_zero<S>(); }
                        st_.ldP(offP1, P1);
                        const int neg = (flags & OPF_NEG) ? (int)0x80000000 : 0;
#pragma unroll
                        for (int c = 0; c < 4; c++) a[c] = cneg(a[c], neg);
                        v3_acc(x, P1, Pt, a, acc, 1.0);
                        tcontract_acc(x, tacc, a, 1.0);
#pragma unroll
                        for (int c = 0; c < 4; c++) en[c] = st_.ld(offDst + c);
                        const S term = s_isqrt2(mdot(en, x));
                        amp = amp + term;
                        if constexpr (kComplex && !StateElem<S>::kDD) {
                            double Pf[4];
#pragma unroll
                            for (int c = 0; c < 4; c++) Pf[c] = P1[c] + Pt[c];
                            wamp = wamp + mdot(Pf, x);
                            asum += fabs(term.re) + fabs(term.im);
                        }
                    } else if (flags & OPF_COMBINE) {
                        // add the offB partial sums of a split target and finish it like a LAST op
#pragma unroll
                        for (int c = 0; c < 4; c++) acc[c] = st_.ld(offA + c);
#pragma unroll
                        for (int c = 0; c < 6; c++) tacc[c] = st_.ld(offA + 4 + c);
                        for (int r = 1; r < offB; r++) {
#pragma unroll
                            for (int c = 0; c < 4; c++) acc[c] = acc[c] + st_.ld(offA + 10 * r + c);
#pragma unroll
                            for (int c = 0; c < 6; c++) tacc[c] = tacc[c] + st_.ld(offA + 10 * r + 4 + c);
                        }
                        {
                            const int offP2 = (int)(raw.w & 0xFFFF);
                            R Pa[4], Pb[4];
                            st_.ldP(offP1, Pa);
                            st_.ldP(offP2, Pb);
#pragma unroll
                            for (int c = 0; c < 4; c++) Pt[c] = r_add(Pa[c], Pb[c]);
                        }
                        const R f = r_isqrt2_over(mdot(Pt, Pt));
#pragma unroll
                        for (int c = 0; c < 4; c++) acc[c] = s_scale(f, acc[c]);
#pragma unroll
                        for (int c = 0; c < 6; c++) tacc[c] = s_isqrt2(tacc[c]);
                        if (!(flags & OPF_NOSTORE)) {
#pragma unroll
                            for (int c = 0; c < 4; c++) st_.st(offDst + c, acc[c]);
#pragma unroll
                            for (int c = 0; c < 6; c++) st_.st(offDst + 4 + c, tacc[c]);
                        }
                        if (flags & OPF_STOREP) {
                            st_.stP(offPt, Pt);
                        }
                    } else if (!StateElem<S>::kDD && (flags & OPF_EXTD)) {
                        // continuous states (Eq. 7, 9, 12): real polarisation e(phi) times the colour matrix etabar_h eta_g;
                        // record per gluon: p (4), phi, eta (3), etabar (3), pad
                        const int k = (int)raw.w;
                        const double* gr = mrec + k * p.rec_gstride;
                        double pk[4], ev[4], eta[3], etab[3];
#pragma unroll
                        for (int c = 0; c < 4; c++) pk[c] = __ldcg(gr + c);
                        const double phi = __ldcg(gr + 4);
#pragma unroll
                        for (int c = 0; c < 3; c++) { eta[c] = __ldcg(gr + 5 + c); etab[c] = __ldcg(gr + 8 + c); }
                        polarisation_real(pk, phi, ev);
                        const bool closure_leg = offPt == 0xFFFF;   // gluon n: no momentum slot; target (h,g) reads X_n[g][h]
#pragma unroll
                        for (int h = 0; h < 3; h++)
#pragma unroll
                            for (int gg = 0; gg < 3; gg++) {
                                const double x = etab[h] * eta[gg];
                                const int at = offDst + 4 * (h * 3 + gg);
#pragma unroll
                                for (int c = 0; c < 4; c++) st_.st(at + c, s_real<S>(x * ev[c]));
                            }
                        if (!closure_leg) {
                            st_.stPd(offPt, pk);
                        }
                    } else if ((flags & OPF_EXT) && kComplex) {
                        const int k = (int)raw.w;
                        double pk[4];
#pragma unroll
                        for (int c = 0; c < 4; c++) pk[c] = ldm(k, c);   // (records: not through L1, which is kept for the ops)
                        if constexpr (kTwinOk) { if (p.twin & 1) rotate_frame(pk); }
                        if constexpr (kComplex) {
                            S eps[4];
                            ext_current(pk, ((perm >> (48 + k)) & 1) ? 1 : -1, eps);
#pragma unroll
                            for (int c = 0; c < 4; c++) st_.st(offDst + c, eps[c]);
                        }
                        if (offPt != 0xFFFF) store_ext_momentum(k, offPt, pk);
                    }
                    if (flags & OPF_SYNC) {
                        // end of a level: the currents just written become visible to the lanes of the event
                        if constexpr (G > 32) __syncthreads(); else __syncwarp(evmask);
                        if (!prefetched) first_barrier_done();
                    }
                    {
                        // The op requested at the top of this step must not be touched before the step ends (the
                        // compiler would otherwise park it right behind the load with moves that wait for it): its
                        // first use is tied to the step's last arithmetic results through an always-zero mask.
                        const unsigned late = (unsigned)(hi_word(acc[0]) ^ hi_word(amp)) & (unsigned)p.zero;
                        const uint4 moved = make_uint4(r2.x | late, r2.y | late, r2.z | late, r2.w | late);
                        if constexpr (kEarlyRing) { r0 = moved; } else if constexpr (!kUseRing) { r0 = r1; r1 = moved; }
                    }
                }
                if constexpr (kUseRing) asm volatile("cp.async.wait_group 0;" ::: "memory");
            }

            // closure amplitude: sum of the G lanes' partial contractions (Eq. 22), then |A|^2
            constexpr bool kWard = kComplex && !StateElem<S>::kDD;
            const bool flagging = kWard && p.tau2 > 0.0;
#pragma unroll
            for (int d = EPW; d < 32; d <<= 1) {
                amp = amp + shfl_xor(amp, d);
                if constexpr (kWard) { wamp = wamp + shfl_xor(wamp, d); asum += shfl_xor(asum, d); }
            }
            if constexpr (G > 32) {
                __shared__ double red_s[(kWard ? 3 : 1) * (sizeof(S) / 8) * (G / 32)];
                if ((lane & 31) == 0) {
                    reinterpret_cast<S*>(red_s)[lane >> 5] = amp;
                    if constexpr (kWard) {
                        reinterpret_cast<S*>(red_s)[G / 32 + (lane >> 5)] = wamp;
                        red_s[2 * (sizeof(S) / 8) * (G / 32) + (lane >> 5)] = asum;
                    }
                }
                __syncthreads();
                if (lane == 0) {
                    amp = s_zero<S>();
                    for (int w = 0; w < G / 32; w++) amp = amp + reinterpret_cast<S*>(red_s)[w];
                    if constexpr (kWard) {
                        wamp = s_zero<S>();
                        asum = 0.0;
                        for (int w = 0; w < G / 32; w++) {
                            wamp = wamp + reinterpret_cast<S*>(red_s)[G / 32 + w];
                            asum += red_s[2 * (sizeof(S) / 8) * (G / 32) + w];
                        }
                    }
                }
            }
            if (g == 0 && have) {
                const double w = valid ? s_norm2(amp) : 0.0;
                if (!(kWard && (p.twin & 2))) p.out[e] = w;      // (second stage of the cascade: out[e] keeps the first result)
                if (kWard && p.mark && p.tau2 > 0.0 && !(p.twin & 2)) p.mark[idx] = 0;
                if constexpr (kWard) {
                    if (p.tau2 < 0.0 && valid) {
                        // diagnostic (BG_OPT_PRECISION = 3): the Ward residual itself instead of |A|^2
                        const double En = ldm(n - 1, 0);
                        p.out[e] = p.tau2 < -1.5 ? (fabs(amp.re) + fabs(amp.im)) / asum : ::sqrt(0.5 * s_norm2(wamp) / (En * En * w));
                    }
                    if (flagging && valid) {
                        // |sqrt2 p_n . J|^2 / 2 > tau^2 E_n^2 |A|^2, or |A| < tau_rho sum |closure terms| (the Ward residual does
                        // not see round-off that respects gauge invariance; strong cancellation at the top amplifies
                        // any), or a result that is not a positive finite number: not trusted as it stands
                        const double En = ldm(n - 1, 0);
                        const double ward2 = 0.5 * s_norm2(wamp), scale = En * En * w;
                        const bool hard = !(ward2 <= fmax(p.tw2, p.tau2) * scale) ||
                                          !(fabs(amp.re) + fabs(amp.im) >= p.tau_rho * asum) || !(w > 0.0);
                        bool to_dd = hard, to_twin = false;
                        if (p.twin & 2) {
                            // second stage: this frame's result against the first one's
                            const double w1 = p.out[e];
                            to_dd = hard || !(fabs(w - w1) <= p.td * w1);
                        } else if (!hard) {
                            to_twin = !(ward2 <= p.tau2 * scale);      // (tau_twin <= tau: never - no second stage)
                        }
                        if (p.mark) {
                            if (to_dd) p.mark[idx] = (p.twin & 2) ? 3 : 2;
                            else if (to_twin) p.mark[idx] = 1;
                        } else if (to_dd) {
                            const uint32_t at = atomicAdd(p.flag_count + tier, 1u);
                            BG_CHECK(first + at < (long long)p.bounds[tier + 1]);
                            p.flag_list[first + at] = (uint32_t)idx;
                        } else if (to_twin) {
                            const uint32_t at = atomicAdd(p.soft_count + tier, 1u);
                            BG_CHECK(first + at < (long long)p.bounds[tier + 1]);
                            p.soft_list[first + at] = (uint32_t)idx;
                        }
                    }
                }
            }
            if constexpr (G > 32) __syncthreads(); else __syncwarp();
        }
    }
}

// set the dynamic shared-memory limit of one instantiation (once per device); returns its static shared memory
template <int G, bool SPILL, class S, bool UNSORTED = false>
static cudaError_t configure_interp(size_t* static_smem_out) {
    constexpr int BLOCK = G > 32 ? G : 32;
    static int configured_device = -1;   // the attribute is per device
    static size_t static_smem = 0;       // the kernel's static shared memory (reduction scratch)
    int device = 0;
    cudaGetDevice(&device);
    if (configured_device != device) {
        cudaError_t e = cudaFuncSetAttribute(cdbg_prog_kernel<G, SPILL, S, UNSORTED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)(kMaxSlabBytes + (size_t)kRing * BLOCK * 16));
        if (e != cudaSuccess) return e;
        cudaFuncAttributes fa;
        if ((e = cudaFuncGetAttributes(&fa, cdbg_prog_kernel<G, SPILL, S, UNSORTED>)) != cudaSuccess) return e;
        static_smem = fa.sharedSizeBytes;
        configured_device = device;
    }
    *static_smem_out = static_smem;
    return cudaSuccess;
}

// resident blocks per SM of one instantiation at a dynamic shared-memory size, as the runtime's occupancy calculator
// sees it (registers, allocation granularity of shared memory, the per-block reservation): a grid sized for one block
// more than fits runs a second, nearly empty wave
template <int G, bool SPILL, class S, bool UNSORTED = false>
static int interp_blocks_per_sm(size_t smem) {
    constexpr int BLOCK = G > 32 ? G : 32;
    // asked once per shared-memory size and device (a bg_eval sizes up to four launches per stage; the query costs
    // host time that a small batch has nothing to hide behind)
    struct Entry { int device; size_t smem; int blocks; };
    static Entry cache[16];
    static int used = 0;
    int device = 0;
    cudaGetDevice(&device);
    for (int i = 0; i < used; i++)
        if (cache[i].device == device && cache[i].smem == smem) return cache[i].blocks;
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, cdbg_prog_kernel<G, SPILL, S, UNSORTED>, BLOCK, smem) != cudaSuccess) {
        cudaGetLastError();
        nb = 1;
    }
    nb = std::max(1, nb);
    if (used < 16) cache[used++] = {device, smem, nb};
    return nb;
}

// SPILL: every tier runs the spill kernel.  HYBRID (with SPILL = false): shape.hybrid picks it per tier.
// UNSORTED: the instantiations that read the caller's arrays (one tier, merged launch shape).
template <int G, bool SPILL, class S = cx, bool HYBRID = false, bool UNSORTED = false>
static cudaError_t launch_interp(cudaStream_t s, const ProgTable* t, int sm_count, ProgParams p, int* launched,
                                 const LaunchShape& shape) {
    static_assert(!(SPILL && HYBRID), "HYBRID chooses between the two kernels itself");
    bool conc = shape.conc;
    constexpr int EPW = G >= 32 ? 1 : 32 / G, BLOCK = G > 32 ? G : 32;
    constexpr size_t ELEM = sizeof(typename StateElem<S>::T);
    constexpr bool kHasDirect = !SPILL, kHasSpill = SPILL || HYBRID;
    size_t static_direct = 0, static_spill = 0;
    cudaError_t cerr;
    if constexpr (kHasDirect)
        if ((cerr = configure_interp<G, false, S, UNSORTED>(&static_direct)) != cudaSuccess) return cerr;
    if constexpr (kHasSpill)
        if ((cerr = configure_interp<G, true, S, UNSORTED>(&static_spill)) != cudaSuccess) return cerr;
    bool hybrid = HYBRID && shape.hybrid && shape.cap_cx > 0;
    if (shape.merged) {
        // list launches (second stage, re-evaluation): few tasks per tier, so one launch walks the tiers' lists one after
        // the other (heaviest first; tasks by ticket) with the shape of the largest tier
        int k0 = 0;
        while (k0 + 1 < kTiers && t->tiers.first_key[k0] == t->tiers.first_key[k0 + 1]) k0++;
        const size_t ring_bytes = G >= 8 ? (size_t)kRing * BLOCK * 16 : 0;
        const bool sp = SPILL || (hybrid && t->tiers.slab_cx[k0] > shape.cap_cx);
        const int slab = (shape.cap_cx > 0 && sp) ? std::min(t->tiers.slab_cx[k0], shape.cap_cx) : t->tiers.slab_cx[k0];
        const size_t smem = ((size_t)EPW * slab * ELEM + 15) / 16 * 16 + ring_bytes;
        if (smem > kMaxSlabBytes + ring_bytes) return cudaErrorInvalidValue;
        int per_sm = 1;
        if (sp) { if constexpr (kHasSpill) per_sm = std::min(interp_blocks_per_sm<G, true, S, UNSORTED>(smem), shape.spill_blocks); }
        else { if constexpr (kHasDirect) per_sm = interp_blocks_per_sm<G, false, S, UNSORTED>(smem); }
        const long long tasks = ((shape.tasks_hint > 0 ? shape.tasks_hint : p.N) + EPW - 1) / EPW + kTiers;
        long long blocks = std::max<long long>(1, std::min<long long>(tasks, (long long)sm_count * per_sm));
        if (sp && shape.max_blocks > 0) blocks = std::min<long long>(blocks, shape.max_blocks);
        p.tier = k0;
        p.merged = 1;
        p.slab_cx = slab;
        if (sp) {
            if constexpr (kHasSpill) cdbg_prog_kernel<G, true, S, UNSORTED><<<(unsigned)blocks, BLOCK, smem, s>>>(p);
        } else {
            if constexpr (kHasDirect) cdbg_prog_kernel<G, false, S, UNSORTED><<<(unsigned)blocks, BLOCK, smem, s>>>(p);
        }
        ++*launched;
        return cudaGetLastError();
    }
    const long long max_tasks = ((shape.tasks_hint > 0 ? shape.tasks_hint : p.N) + EPW - 1) / EPW + kTiers;
    if (hybrid) {
        // small batches (fewer than two tasks per block the uncapped launches hold): occupancy is not what limits
        // them, and the capped kernel's L2 round trips cost more than they hide (n = 6: 2^16 events +7 %, 2^17 equal,
        // 2^18 and more -2 ... -6 %; n = 7: 2^14 +14 %, 2^16 -8 %, 2^18 -20 %)
        long long direct = 0;
        for (int k = 0; k < kTiers; k++) {
            if (t->tiers.first_key[k] == t->tiers.first_key[k + 1] && k + 1 < kTiers) continue;
            const size_t sm = ((size_t)EPW * t->tiers.slab_cx[k] * ELEM + 15) / 16 * 16 + (G >= 8 ? (size_t)kRing * BLOCK * 16 : 0);
            if constexpr (kHasDirect) direct += (long long)sm_count * interp_blocks_per_sm<G, false, S, UNSORTED>(sm);
        }
        if (max_tasks <= 2 * direct) hybrid = false;
    }
    unsigned blocks[kTiers];
    size_t smem[kTiers];
    int slab[kTiers];
    bool sp[kTiers];
    long long resident = 0;
    int nlaunch = 0, nspill = 0;
    for (int k = 0; k < kTiers; k++) {
        blocks[k] = 0;
        sp[k] = false;
        // no class in this tier (the last tier always runs: events with colour codes out of range are sorted behind
        // every class and get their 0.0 there)
        if (t->tiers.first_key[k] == t->tiers.first_key[k + 1] && (k + 1 < kTiers || t->dense)) continue;
        const size_t ring_bytes = G >= 8 ? (size_t)kRing * BLOCK * 16 : 0;
        sp[k] = SPILL || (hybrid && t->tiers.slab_cx[k] > shape.cap_cx);
        slab[k] = (shape.cap_cx > 0 && (SPILL || sp[k])) ? std::min(t->tiers.slab_cx[k], shape.cap_cx) : t->tiers.slab_cx[k];
        smem[k] = ((size_t)EPW * slab[k] * ELEM + 15) / 16 * 16 + ring_bytes;
        if (smem[k] > kMaxSlabBytes + ring_bytes) return cudaErrorInvalidValue;
        // resident blocks per SM: 228 KB of shared memory against dynamic + static + 1 KB reserved per block (a grid
        // sized for one block more than fits runs a second, nearly empty wave), and 65536 / (regs x BLOCK) registers
        int per_sm = 1;
        if (sp[k]) { if constexpr (kHasSpill) per_sm = std::min(interp_blocks_per_sm<G, true, S, UNSORTED>(smem[k]), shape.spill_blocks); }   // one global slab per resident block
        else { if constexpr (kHasDirect) per_sm = interp_blocks_per_sm<G, false, S, UNSORTED>(smem[k]); }
        blocks[k] = (unsigned)std::max<long long>(1, std::min<long long>(max_tasks, (long long)sm_count * per_sm));
        if (sp[k] && shape.max_blocks > 0) blocks[k] = (unsigned)std::min<long long>(blocks[k], shape.max_blocks);
        resident += (long long)sm_count * per_sm;
        nlaunch++;
        nspill += sp[k] ? 1 : 0;
    }
    // Small batches: when the tiers together hold fewer than two tasks per resident block, each launch is mostly
    // ramp-up and tail, so the tiers run side by side (fork / join around the caller's stream).  Measured at
    // n = 6: 2^16 events +22 %, 2^18 neutral, 2^20 -5 %; n >= 7: slower at every size.
    // (spill slabs are indexed by block: concurrent spill launches each get their own share of the slabs)
    if (SPILL) conc = conc && shape.max_blocks > 0 && t->has_streams && nlaunch > 1;
    else conc = conc && G <= 4 && t->has_streams && nlaunch > 1 && max_tasks <= 2 * resident && (nspill == 0 || shape.max_blocks > 0);
    const bool share_slabs = conc && nspill > 1;
    const long long share = share_slabs ? std::max<long long>(1, shape.max_blocks / nspill) : 0;
    if (share_slabs)
        for (int k = 0; k < kTiers; k++)
            if (sp[k]) blocks[k] = (unsigned)std::min<long long>(blocks[k], share);
    if (conc && cudaEventRecord(t->fork_ev, s) != cudaSuccess) return cudaGetLastError();
    double2* const spill0 = p.spill;
    int li = 0;
    int side = 0;                                 // launches sent to the side streams so far
    bool first = true;
    for (int k = 0; k < kTiers; k++) {
        if (!blocks[k]) continue;
        p.tier = k;
        p.slab_cx = slab[k];
        cudaStream_t ls = s;
        if (conc && !first) {
            ls = t->aux[side];
            cudaStreamWaitEvent(ls, t->fork_ev, 0);
        }
        if (sp[k]) {
            if (share_slabs) p.spill = reinterpret_cast<double2*>(reinterpret_cast<char*>(spill0) + (size_t)li * share * p.spill_cx * EPW * ELEM);
            li++;
            if constexpr (kHasSpill) cdbg_prog_kernel<G, true, S, UNSORTED><<<blocks[k], BLOCK, smem[k], ls>>>(p);
        } else {
            if constexpr (kHasDirect) cdbg_prog_kernel<G, false, S, UNSORTED><<<blocks[k], BLOCK, smem[k], ls>>>(p);
        }
        if (conc && !first) cudaEventRecord(t->join_ev[side++], ls);
        first = false;
        ++*launched;
    }
    for (int i = 0; i < side; i++) cudaStreamWaitEvent(s, t->join_ev[i], 0);
    return cudaGetLastError();
}

}  // namespace bg

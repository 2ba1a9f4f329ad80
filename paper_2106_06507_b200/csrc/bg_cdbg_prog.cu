// Colour-class program interpreter: the performance path of the colour-dressed recursion (CDBG, PAPER.md
// Eq. 28-32, closed with Eq. 22) for discrete colour-flow indices.
//
// Pipeline of one bg_eval (all on the caller's stream):
//   1. cdbg_classify_kernel   one thread per event: colour codes -> canonical gluon order (a relabelling, under
//                             which |A|^2 is invariant) + colour-class id; block-aggregated histogram of classes
//   2. cdbg_scan_kernel       exclusive scan of the histogram (classes ordered by state-size tier, then by
//                             program length); positions where the tiers start
//   3. cdbg_scatter_kernel    counting sort: every event becomes one contiguous record (header + momenta of the
//                             canonical gluons) in class order, so that a warp runs equal programs and reads whole
//                             sectors
//      Small batches (<= 2^18 events, <= 4096 classes): no scan launch and no memset - every block of the scatter
//      kernel scans the finished histogram for itself and the last one clears it for the next call; and with
//      G <= 4 and fewer than two tasks per resident block the tier launches of step 4 run side by side.
//   4. cdbg_prog_kernel<G,SPILL>, one launch per non-empty tier: G lanes per event run the class program
//                             (bg_program.h): vertex operations read their operands from the event's state block in
//                             shared memory, accumulate in registers and write each finished current back once.
//                             The program is one flat loop over steps; the last step of a level carries a barrier
//                             among the event's lanes; the closure amplitude is reduced over the G lanes.
// State layout in shared memory: per block a slab of [state_cx][EPW] complex doubles (EPW = 32/G events per warp
// for G < 32, one event per block otherwise; event index fastest) so that a quarter-warp's LDS.128 touches eight
// different 16-byte bank groups when events share a warp.  With SPILL, offsets beyond the slab live in an
// L2-resident global slab of the block.  For G >= 8 a per-lane ring behind the slab receives the ops by cp.async.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <atomic>
#include <numeric>
#include <thread>
#include <vector>

#include "bg_cdbg_interp.cuh"

namespace bg {

__constant__ unsigned c_mscount[kMaxN + 1][kNumCodes];   // multiset_count(r, t) for r <= 12, t <= 8

// ---------------------------------------------------------------------------------------------------------
// 1. classification
// ---------------------------------------------------------------------------------------------------------
// Block-level aggregation: sampled colour assignments fall into few classes (92 distinct ones at n = 6), so the
// class counters are kept in shared memory per block (kPreEvents events) and flushed once; with BLOCK_HIST false
// (histogram larger than shared memory) the counters are updated in global memory directly.
constexpr int kPreThreads = 512, kPrePer = 2, kPreEvents = kPreThreads * kPrePer;

template <bool BLOCK_HIST, int THREADS = kPreThreads, int PER = kPrePer>
__global__ void __launch_bounds__(THREADS)
cdbg_classify_kernel(int n, long long N, long long num_classes, const signed char* __restrict__ col,
                     const ClassInfo* __restrict__ info, const uint32_t* __restrict__ sortkey,
                     uint32_t* __restrict__ cls, uint64_t* __restrict__ perm, uint32_t* __restrict__ hist,
                     uint32_t* __restrict__ flag_count) {
    extern __shared__ uint32_t sh_hist[];
    const int nbins = (int)num_classes + 1;
    if (blockIdx.x == 0 && threadIdx.x < 4 * kTiers) flag_count[threadIdx.x] = 0;   // lists of the conditioning flag: counters | tickets, twice
    if (BLOCK_HIST) {
        for (int i = threadIdx.x; i < nbins; i += THREADS) sh_hist[i] = 0;
        __syncthreads();
    }
    uint32_t* const h = BLOCK_HIST ? sh_hist : hist;
    for (int j = 0; j < PER; j++) {
        const long long e = (long long)blockIdx.x * (THREADS * PER) + j * THREADS + threadIdx.x;
        if (e >= N) break;
        // colour codes 3(i-1)+(j-1) of the n gluons, one nibble each (registers; n is a run-time value)
        int cnt[kNumCodes];
#pragma unroll
        for (int c = 0; c < kNumCodes; c++) cnt[c] = 0;
        bool ok = true;
        uint64_t cw = 0;
        for (int k = 0; k < n; k++) {
            const int i = col[(size_t)(2 * k) * N + e] - 1, jj = col[(size_t)(2 * k + 1) * N + e] - 1;
            ok = ok && i >= 0 && i < 3 && jj >= 0 && jj < 3;
            const int code = ok ? 3 * i + jj : 0;
            cw |= (uint64_t)code << (4 * k);
#pragma unroll
            for (int c = 0; c < kNumCodes; c++) cnt[c] += code == c;
        }
        if (!ok) {
            cls[e] = 0xFFFFFFFFu;
            perm[e] = 0;
            atomicAdd(&h[num_classes], 1u);
            continue;
        }
        unsigned rank = 0;
        int r = n;
#pragma unroll
        for (int t = 0; t < kNumCodes - 1; t++) {
            for (int c = 0; c < cnt[t]; c++) rank += c_mscount[r - c][kNumCodes - 1 - t];
            r -= cnt[t];
        }
        const ClassInfo ci = info[rank];
        uint64_t pm = 0;
        if (ci.valid) {
            // canonical order: codes ascending, original order inside a code, the last gluon with the closure code
            // moved to the end.  start[c] (a nibble per code) = canonical position of the next gluon with code c.
            const int closure = ci.closure_code;
            int lastk = 0;
            for (int k = 0; k < n; k++)
                if ((int)((cw >> (4 * k)) & 0xF) == closure) lastk = k;
            uint64_t start = 0;
            int before = 0;
#pragma unroll
            for (int c = 0; c < kNumCodes; c++) {
                start |= (uint64_t)before << (4 * c);
                before += cnt[c] - (c == closure ? 1 : 0);
            }
            for (int k = 0; k < n; k++) {
                if (k == lastk) continue;
                const int sh = 4 * (int)((cw >> (4 * k)) & 0xF);
                pm |= (uint64_t)k << (4 * (int)((start >> sh) & 0xF));
                start += 1ull << sh;
            }
            pm |= (uint64_t)lastk << (4 * (n - 1));
        }
        cls[e] = rank;
        perm[e] = pm;
        atomicAdd(&h[sortkey[rank]], 1u);
    }
    if (BLOCK_HIST) {
        __syncthreads();
        for (int i = threadIdx.x; i < nbins; i += THREADS) {
            const uint32_t c = sh_hist[i];
            if (c) atomicAdd(&hist[i], c);
        }
    }
}

// 2. exclusive scan of hist[0..count) in place (one block)
__global__ void __launch_bounds__(1024)
cdbg_scan_kernel(uint32_t* __restrict__ hist, int count, TierInfo tiers, uint32_t* __restrict__ bounds, uint32_t N) {
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int base = 0; base < count; base += 1024) {
        const int i = base + threadIdx.x;
        const uint32_t v = i < count ? hist[i] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, d);
            if (lane >= d) x += y;
        }
        if (lane == 31) warp_tot[warp] = x;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = warp_tot[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, w, d);
                if (lane >= d) w += y;
            }
            warp_tot[lane] = w;
        }
        __syncthreads();
        const uint32_t before = carry + (warp ? warp_tot[warp - 1] : 0u) + (x - v);
        if (i < count) hist[i] = before;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x <= kTiers) bounds[threadIdx.x] = threadIdx.x == kTiers ? N : hist[tiers.first_key[threadIdx.x]];
}

// 3. scatter the events into class order.  Each event becomes one contiguous record
//      [EventHeader, padded to 32 B][momenta of the canonical gluons 0..n-1, 4 doubles = one 32-byte sector each]
// so that the interpreter reads whole sectors; the inputs are read here in their event-fastest layout (coalesced)
// and the 8-byte stores of one record merge in L2.  Helicities go into bits 48.. of the header's perm word.
__device__ __forceinline__ void write_record(int n, long long N, long long e, uint32_t c, uint64_t pm,
                                             const double* __restrict__ mom, const signed char* __restrict__ hel,
                                             char* __restrict__ rec) {
    if (c == 0xFFFFFFFFu || pm == 0) {
        // colour codes out of range, or a class whose amplitude vanishes identically: the interpreter reads the
        // header only (a valid permutation never has pm = 0), so no momenta are gathered
        EventHeader h;
        h.event = (uint32_t)e; h.cls = c; h.perm = 0;
        *reinterpret_cast<EventHeader*>(rec) = h;
        return;
    }
    unsigned inv[kMaxN];                       // original gluon -> canonical position
#pragma unroll
    for (int k = 0; k < kMaxN; k++) inv[k] = (unsigned)k;
    for (int k = 0; k < n; k++) inv[(pm >> (4 * k)) & 0xF] = (unsigned)k;
    double2* m = reinterpret_cast<double2*>(rec + kRecHeaderBytes);   // 32-byte aligned: one sector per gluon
    // three gluons (12 coalesced loads) in flight per round
    for (int j0 = 0; j0 < n; j0 += 3) {
        double v[3][4];
        signed char hl[3];
#pragma unroll
        for (int u = 0; u < 3; u++) {
            const int j = j0 + u < n ? j0 + u : n - 1;
            hl[u] = hel ? hel[(size_t)j * N + e] : (signed char)0;
#pragma unroll
            for (int cc = 0; cc < 4; cc++) v[u][cc] = mom[(size_t)(j * 4 + cc) * N + e];
        }
#pragma unroll
        for (int u = 0; u < 3; u++) {
            if (j0 + u >= n) break;
            const unsigned k = inv[j0 + u];
            if (hl[u] > 0) pm |= 1ull << (48 + k);
            m[k * 2] = make_double2(v[u][0], v[u][1]);
            m[k * 2 + 1] = make_double2(v[u][2], v[u][3]);
        }
    }
    EventHeader h;
    h.event = (uint32_t)e; h.cls = c; h.perm = pm;
    *reinterpret_cast<EventHeader*>(rec) = h;
}

template <bool BLOCK_HIST>
__global__ void __launch_bounds__(kPreThreads)
cdbg_scatter_kernel(int n, long long N, long long num_classes, const uint32_t* __restrict__ cls,
                    const uint64_t* __restrict__ perm, const uint32_t* __restrict__ sortkey,
                    const double* __restrict__ mom, const signed char* __restrict__ hel,
                    uint32_t* __restrict__ cursor, char* __restrict__ rec, int rec_bytes) {
    extern __shared__ uint32_t sh_hist[];
    const int nbins = (int)num_classes + 1;
    uint32_t key[kPrePer], rank[kPrePer];
    if (BLOCK_HIST) {
        for (int i = threadIdx.x; i < nbins; i += kPreThreads) sh_hist[i] = 0;
        __syncthreads();
    }
#pragma unroll
    for (int j = 0; j < kPrePer; j++) {
        const long long e = (long long)blockIdx.x * kPreEvents + j * kPreThreads + threadIdx.x;
        key[j] = 0xFFFFFFFFu;
        if (e < N) {
            const uint32_t c = cls[e];
            key[j] = c == 0xFFFFFFFFu ? (uint32_t)num_classes : sortkey[c];
            if (BLOCK_HIST) rank[j] = atomicAdd(&sh_hist[key[j]], 1u);
            else write_record(n, N, e, c, perm[e], mom, hel, rec + (size_t)atomicAdd(&cursor[key[j]], 1u) * rec_bytes);
        }
    }
    if (!BLOCK_HIST) return;
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += kPreThreads) {
        const uint32_t c = sh_hist[i];
        if (c) sh_hist[i] = atomicAdd(&cursor[i], c);
    }
    __syncthreads();
    for (int j = 0; j < kPrePer; j++) {
        const long long e = (long long)blockIdx.x * kPreEvents + j * kPreThreads + threadIdx.x;
        if (key[j] != 0xFFFFFFFFu)
            write_record(n, N, e, cls[e], perm[e], mom, hel, rec + (size_t)(sh_hist[key[j]] + rank[j]) * rec_bytes);
    }
}

// 3b. the same with the records of a warp staged in shared memory: a thread writing its own 32(n+1)-byte record
// touches 32 different lines per store instruction; here each warp builds its 32 records in shared memory
// (record stride padded by 16 bytes: conflict-free) and copies them out with consecutive lanes on consecutive
// 16-byte pieces, so a store instruction covers four to five lines.  Blocks of kStageThreads threads; used when
// histogram + staging fit in shared memory for at least two blocks per SM (n <= 7).
constexpr int kStageThreads = 256, kStageEvents = kStageThreads * kPrePer;
constexpr int kSmallThreads = 256;              // block size of the classify kernel for small batches
constexpr int kFusedScanBins = 4096;            // largest histogram the scatter blocks scan for themselves
constexpr long long kFusedScanEvents = 1 << 18; // ... and largest batch (beyond it the scan launch is cheaper)
// FUSED (small batches, where a step is a handful of short launches): the exclusive scan of the class histogram
// is done here, by every block for itself in shared memory (a few thousand bins), instead of by a launch of its
// own; `counts` is then the finished histogram of the classify kernel and `cursor` a zeroed array of running
// offsets inside the classes.  Both live in a small buffer of the table that the last block to finish clears
// for the next call, so no memset launch is needed either.
struct FusedScan {
    const uint32_t* counts;   // [nbins] class histogram (classify kernel)
    uint32_t* ticket;         // blocks finished so far
    uint32_t* bounds;         // [kTiers + 1] tier starts (written by block 0)
    uint32_t N;
    TierInfo tiers;
};
template <bool FUSED, int PER = kPrePer>
__global__ void __launch_bounds__(kStageThreads)
cdbg_scatter_staged_kernel(int n, long long N, long long num_classes, const uint32_t* __restrict__ cls,
                           const uint64_t* __restrict__ perm, const uint32_t* __restrict__ sortkey,
                           const double* __restrict__ mom, const signed char* __restrict__ hel,
                           uint32_t* __restrict__ cursor, char* __restrict__ rec, int rec_bytes, const FusedScan fs) {
    extern __shared__ uint32_t sh_hist[];
    const int nbins = (int)num_classes + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rs = rec_bytes + 16, pieces = rec_bytes / 16;
    const int hist_words = (nbins + 3) & ~3;
    uint32_t* const sh_start = sh_hist + hist_words;        // FUSED: exclusive scan of the global histogram
    char* const stage = reinterpret_cast<char*>(sh_hist + (FUSED ? 2 : 1) * hist_words) + (size_t)warp * (32 * rs + 256);
    if (FUSED) {
        __shared__ uint32_t warp_tot[kStageThreads / 32];
        const int per = (nbins + kStageThreads - 1) / kStageThreads;     // contiguous bins per thread
        const int b0 = threadIdx.x * per, b1 = min(nbins, b0 + per);
        uint32_t sum = 0;
        for (int i = b0; i < b1; i++) sum += fs.counts[i];
        uint32_t x = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, d);
            if (lane >= d) x += y;
        }
        if (lane == 31) warp_tot[warp] = x;
        __syncthreads();
        uint32_t before = x - sum;
        for (int w = 0; w < warp; w++) before += warp_tot[w];
        for (int i = b0; i < b1; i++) {
            sh_start[i] = before;
            before += fs.counts[i];
        }
        // (the barrier below, before the first use of sh_start, also orders these writes)
    }
    unsigned long long* const dstp = reinterpret_cast<unsigned long long*>(stage + 32 * rs);
    uint32_t key[PER], rank[PER];
    for (int i = threadIdx.x; i < nbins; i += kStageThreads) sh_hist[i] = 0;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < PER; j++) {
        const long long e = (long long)blockIdx.x * (kStageThreads * PER) + j * kStageThreads + threadIdx.x;
        key[j] = 0xFFFFFFFFu;
        rank[j] = 0;
        if (e < N) {
            const uint32_t c = cls[e];
            key[j] = c == 0xFFFFFFFFu ? (uint32_t)num_classes : sortkey[c];
            rank[j] = atomicAdd(&sh_hist[key[j]], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += kStageThreads) {
        const uint32_t c = sh_hist[i];
        if (c) sh_hist[i] = atomicAdd(&cursor[i], c) + (FUSED ? sh_start[i] : 0u);
    }
    if (FUSED && blockIdx.x == 0 && threadIdx.x <= kTiers)
        fs.bounds[threadIdx.x] = threadIdx.x == kTiers ? fs.N : sh_start[fs.tiers.first_key[threadIdx.x]];
    __syncthreads();
    for (int j = 0; j < PER; j++) {
        const long long e = (long long)blockIdx.x * (kStageThreads * PER) + j * kStageThreads + threadIdx.x;
        char* dst = nullptr;
        if (key[j] != 0xFFFFFFFFu) {
            dst = rec + (size_t)(sh_hist[key[j]] + rank[j]) * rec_bytes;
            char* mine = stage + lane * rs;
            *reinterpret_cast<uint4*>(mine + 16) = make_uint4(0, 0, 0, 0);      // second half of the header block
            write_record(n, N, e, cls[e], perm[e], mom, hel, mine);
        }
        dstp[lane] = reinterpret_cast<unsigned long long>(dst);
        __syncwarp();
        for (int i = lane; i < 32 * pieces; i += 32) {
            const int r = i / pieces, q = i - r * pieces;
            char* d = reinterpret_cast<char*>(dstp[r]);
            if (d) *reinterpret_cast<uint4*>(d + q * 16) = *reinterpret_cast<const uint4*>(stage + r * rs + q * 16);
        }
        __syncwarp();
    }
    if (FUSED) {
        // the last block to get here leaves histogram, cursors and ticket zeroed for the next call
        __shared__ bool last;
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            last = atomicAdd(fs.ticket, 1u) == gridDim.x - 1;
        }
        __syncthreads();
        if (last) {
            uint32_t* counts = const_cast<uint32_t*>(fs.counts);
            for (int i = threadIdx.x; i < nbins; i += kStageThreads) { counts[i] = 0; cursor[i] = 0; }
            if (threadIdx.x == 0) *fs.ticket = 0;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
static void enumerate_counts(int t, int r, int* counts, std::vector<std::vector<int>>& out) {
    if (t == kNumCodes - 1) {
        counts[t] = r;
        out.emplace_back(counts, counts + kNumCodes);
        return;
    }
    for (int c = 0; c <= r; c++) {
        counts[t] = c;
        enumerate_counts(t + 1, r - c, counts, out);
    }
}

int prog_table_create(int n, int G, size_t slab_limit, bool comc, ProgTable** out, const ProgTable* like) {
    if (slab_limit == 0 || slab_limit > kMaxSlabBytes) slab_limit = kMaxSlabBytes;
    *out = nullptr;
    if (n < 4 || n > kMaxN || (G != 1 && G != 2 && G != 4 && G != 8 && G != 16 && G != 32 && G != 64 && G != 128 && G != 256)) return BG_EINVAL;
    std::vector<std::vector<int>> all;
    int counts[kNumCodes];
    enumerate_counts(0, n, counts, all);
    const long long nc = (long long)all.size();
    if (nc != multiset_count(n, kNumCodes)) return BG_EINVAL;
    std::vector<ClassInfo> info(nc);
    std::vector<ProgOp> ops;
    std::vector<int> steps(nc, 0);
    int max_state = 0;
    {
        // the programs of different classes are independent: build them on all host cores, then concatenate
        for (long long r = 0; r < nc; r++)
            if (class_rank(n, all[r].data()) != r) return BG_EINVAL;
        std::vector<ClassProgram> progs(nc);
        std::atomic<long long> next_class{0};
        std::atomic<bool> overflow{false};   // a class whose state does not fit the 16-bit state offsets
        std::atomic<long long> dressed_fallbacks{0};
        auto worker = [&]() {
            for (long long r = next_class.fetch_add(1); r < nc; r = next_class.fetch_add(1))
                if (!comc) {
                    build_class(n, G, all[r].data(), progs[r], like ? (int)like->h_closure[r] : -1);
                } else {
                    // CO_MC: canonical order = codes ascending; only classes with balanced colour charges can be non-zero
                    const int* cnt = all[r].data();
                    bool balanced = true;
                    for (int c = 0; c < 3; c++) {
                        int ni = 0, nj = 0;
                        for (int t = 0; t < kNumCodes; t++) { if (t / 3 == c) ni += cnt[t]; if (t % 3 == c) nj += cnt[t]; }
                        balanced = balanced && ni == nj;
                    }
                    if (!balanced) continue;
                    int code[kMaxN], k = 0;
                    for (int t = 0; t < kNumCodes; t++)
                        for (int q = 0; q < cnt[t]; q++) code[k++] = t;
                    // A class whose shared sequence currents do not fit the 16-bit state offsets (more than a few
                    // thousand colour-connected orderings: 1e-3 of the classes a uniform colour draw hits at n = 9, none
                    // for n <= 8) is evaluated with its colour-dressed program instead - the same number (Eq. 19 is
                    // what Eq. 28-32 compute), same records, same interpreter.
                    build_comc_program(n, G, code, progs[r], 6000);
                    if (progs[r].state_cx < 0 || progs[r].state_cx > 65535) {
                        build_class(n, G, cnt, progs[r]);
                        if (progs[r].state_cx < 0 || progs[r].state_cx > 65535) overflow = true;
                        dressed_fallbacks++;
                    }
                }
        };
        unsigned nthreads = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
        if (n <= 8) nthreads = 1;
        std::vector<std::thread> pool;
        for (unsigned i = 1; i < nthreads; i++) pool.emplace_back(worker);
        worker();
        for (auto& th : pool) th.join();
        if (overflow) return BG_EUNSUPPORTED;
        size_t total_ops = 0;
        for (auto& cp : progs) total_ops += cp.ops.size();
        ops.reserve(total_ops + G);
        for (long long r = 0; r < nc; r++) {
            ClassProgram& cp = progs[r];
            ClassInfo& ci = info[r];
            std::memset(&ci, 0, sizeof(ci));
            if (!cp.valid) continue;
            ci.valid = 1;
            ci.op_base = (uint32_t)ops.size();
            ci.state_cx = (uint16_t)cp.state_cx;
            ci.closure_code = (uint8_t)cp.closure_code;
            ci.total_steps = (uint32_t)cp.total_steps;
            ci.n_sync = (uint32_t)cp.n_sync;
            for (size_t l = 0; l < cp.level_steps.size(); l++) ci.level_steps[l] = cp.level_steps[l];
            steps[r] = cp.total_steps;
            max_state = std::max(max_state, cp.state_cx);
            ops.insert(ops.end(), cp.ops.begin(), cp.ops.end());
            std::vector<ProgOp>().swap(cp.ops);
        }
    }
    // grouping order: longest programs first (the tail of the grid then runs the short ones), invalid last
    std::vector<uint32_t> by(nc), sortkey(nc);
    std::iota(by.begin(), by.end(), 0u);
    // Tiers by state size (tier 0 = the largest blocks); inside a tier the longest programs come first, classes
    // whose amplitude vanishes (no state, no steps) end up last.  A tier's slab size decides how many blocks an SM
    // holds, so the (at most kTiers) slab sizes are chosen among the classes' state sizes to minimise
    //     sum over tiers of work(tier) / rate(resident warps(slab)),
    // work = steps x the class's share of uniformly drawn colour assignments (n! / prod counts!), rate(w) = w/(w+7)
    // (fitted to the measured FP64 pipe utilisation against resident warps: 0.29 at 4.6, 0.43 at 10 warps per SM).
    TierInfo tiers;
    {
        const int block = G > 32 ? G : 32, epw = G >= 32 ? 1 : 32 / G;
        const size_t ring_bytes = G >= 8 ? (size_t)kRing * block * 16 : 0;
        const int cap_cx = (int)(slab_limit / 16 / (size_t)epw);      // larger states spill (or are refused below)
        const int reg_blocks = std::max(1, 65536 / (168 * block));
        auto rate = [&](int slab_cx) {
            const size_t smem = (size_t)slab_cx * epw * 16 + ring_bytes + 1024 + 512;   // + reserved per block + static (<= 384 B)
            const int blocks = (int)std::max<size_t>(1, std::min<size_t>({(size_t)reg_blocks, (size_t)32, (size_t)(228 * 1024) / smem}));
            const double w = blocks * (block / 32.0);
            return w / (w + 7.0);
        };
        std::vector<std::pair<int, double>> sw;     // (state, work), one entry per distinct state size, ascending
        {
            std::vector<std::pair<int, double>> all_sw;
            for (long long r = 0; r < nc; r++) {
                if (!info[r].valid) continue;
                double w = 1.0;
                int left = n;
                for (int t = 0; t < kNumCodes; t++)
                    for (int q = 1; q <= all[r][t]; q++) w *= (double)(left--) / q;
                all_sw.push_back({std::min<int>(std::max<int>(16, info[r].state_cx), std::max(16, cap_cx)), w * steps[r]});
            }
            std::sort(all_sw.begin(), all_sw.end());
            for (auto& x : all_sw) {
                if (!sw.empty() && sw.back().first == x.first) sw.back().second += x.second;
                else sw.push_back(x);
            }
        }
        const int U = (int)sw.size();
        for (int k = 0; k < kTiers; k++) tiers.slab_cx[k] = std::max(16, std::min(max_state, std::max(16, cap_cx)));
        if (U > 0) {
            std::vector<double> pre(U + 1, 0.0);
            for (int i = 0; i < U; i++) pre[i + 1] = pre[i] + sw[i].second;
            const double kInf = 1e300;
            std::vector<std::vector<double>> best(kTiers + 1, std::vector<double>(U, kInf));
            std::vector<std::vector<int>> from(kTiers + 1, std::vector<int>(U, -1));
            for (int j = 0; j < U; j++) best[1][j] = pre[j + 1] / rate(sw[j].first);
            for (int k = 2; k <= kTiers; k++)
                for (int j = k - 1; j < U; j++) {
                    const double rj = rate(sw[j].first);
                    for (int i = k - 2; i < j; i++) {
                        const double c = best[k - 1][i] + (pre[j + 1] - pre[i + 1]) / rj;
                        if (c < best[k][j]) { best[k][j] = c; from[k][j] = i; }
                    }
                }
            int kbest = 1;
            for (int k = 2; k <= std::min(kTiers, U); k++)
                if (best[k][U - 1] < best[kbest][U - 1] * (1.0 - 1e-3)) kbest = k;   // a tier must pay for its launch
            int j = U - 1, slot = 0;
            for (int k = kbest; k >= 1 && j >= 0; k--) {
                tiers.slab_cx[slot++] = sw[j].first;
                j = k > 1 ? from[k][j] : -1;
            }
            for (; slot < kTiers; slot++) tiers.slab_cx[slot] = tiers.slab_cx[slot - 1];   // unused tiers stay empty
        }
    }
    std::vector<int> tier_of(nc);
    for (long long r = 0; r < nc; r++) {
        int k = 0;
        while (k + 1 < kTiers && (int)info[r].state_cx <= tiers.slab_cx[k + 1]) k++;
        tier_of[r] = k;
    }
    std::stable_sort(by.begin(), by.end(), [&](uint32_t a, uint32_t b) {
        return tier_of[a] != tier_of[b] ? tier_of[a] < tier_of[b] : steps[a] > steps[b];
    });
    for (long long i = 0; i < nc; i++) sortkey[by[i]] = (uint32_t)i;
    for (int k = 0; k <= kTiers; k++) tiers.first_key[k] = (int)nc;
    for (long long i = nc - 1; i >= 0; i--) tiers.first_key[tier_of[by[i]]] = (int)i;
    for (int k = kTiers - 1; k >= 0; k--) tiers.first_key[k] = std::min(tiers.first_key[k], tiers.first_key[k + 1]);

    // A block's slab must fit in shared memory; blocks of >= 128 lanes may keep the top of the state (the highest
    // levels, read least often) in an L2-resident global slab instead ("spill").
    const bool spill = (size_t)(G >= 32 ? 1 : 32 / G) * max_state * 16 > slab_limit;
    if (spill && G < 128) return BG_EUNSUPPORTED;
    if (spill)
        for (int k = 0; k < kTiers; k++) tiers.slab_cx[k] = std::min<int>(tiers.slab_cx[k], (int)(slab_limit / 16));
    ProgTable* t = new (std::nothrow) ProgTable();
    if (!t) return BG_ENOMEM;
    std::memset(t, 0, sizeof(*t));
    t->n = n; t->G = G; t->num_classes = nc; t->max_state_cx = max_state; t->tiers = tiers;
    if (like) {    // a table for the list launches of another table's records: its tier ranges, one slab size
        t->tiers = like->tiers;
        for (int k = 0; k < kTiers; k++) t->tiers.slab_cx[k] = std::max(16, max_state);
    }
    t->h_closure = static_cast<uint8_t*>(std::malloc((size_t)nc));
    if (!t->h_closure) { delete t; return BG_ENOMEM; }
    for (long long r = 0; r < nc; r++) t->h_closure[r] = info[r].closure_code;
    t->dense = false;
    t->rec_bytes = kRecHeaderBytes + 32 * n;
    t->spill = spill;
    {   // blocks of the largest tier that fit an SM (shared memory and registers)
        const size_t smem0 = (size_t)tiers.slab_cx[0] * 16;
        const int block = G > 32 ? G : 32;
        t->spill_blocks_per_sm = (int)std::max<size_t>(1, std::min<size_t>(65536 / (168 * block), (228 * 1024) / (smem0 + 1024 + 512)));
    }
    {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, dev);
    }
    {   // capped FP64 launches (warp-shared lane counts 4 and 8, the defaults of n = 5, 6 and 7): the 166 registers per
        // thread allow reg_blocks one-warp blocks per SM, the heavy tiers' slabs (epw events each) far fewer, and the
        // kernel's FP64 rate follows the resident warps.  Tiers above the cap keep cap_cx elements per event in shared
        // memory - what lets reg_blocks blocks fit - and the highest levels in an L2 slab.  (Block-per-event lane counts,
        // n >= 8: measured 13 - 24 % slower, their top levels are the most numerous and the most read.)
        const int epw = G >= 32 ? 1 : 32 / G, block = G > 32 ? G : 32;
        const size_t ring_bytes = G >= 8 ? (size_t)kRing * block * 16 : 0;
        const int reg_blocks = std::max(1, 65536 / (168 * block));
        const int cap = (int)(((size_t)(228 * 1024) / reg_blocks - 1024 - 128 - ring_bytes) / 16 / (size_t)epw);
        t->cap_cx = 0;
        t->cap_blocks = reg_blocks;
        if ((G == 4 || G == 8) && !spill && cap >= 64 && tiers.slab_cx[0] > cap) t->cap_cx = cap;
    }
    {   // double-double re-evaluation: 32-byte state elements and 255 registers per thread.  The registers allow
        // 65536 / (255 x block) resident blocks per SM; the shared-memory part of the state is capped so that shared
        // memory allows as many (the kernel is latency-bound: resident warps decide its speed), the rest - the highest
        // levels - lives in the block's L2-resident slab like the spilled state of the n >= 11 FP64 kernels.
        const int epw = G >= 32 ? 1 : 32 / G, block = G > 32 ? G : 32;
        const size_t ring_bytes = G >= 8 ? (size_t)kRing * block * 16 : 0;
        const int reg_blocks = std::max(1, 65536 / (256 * block));
        const size_t per_block = std::min<size_t>(slab_limit, (size_t)(224 * 1024) / reg_blocks - 1024 - ring_bytes);
        t->dd_mode = 1;
        t->dd_cap_cx = std::max(16, (int)(per_block / 32 / (size_t)epw));
        t->dd_spill_blocks = reg_blocks;
        // one slab of the largest state per block; all slabs together at most 512 MB (fewer blocks otherwise)
        const size_t slab_bytes = (size_t)epw * max_state * 32;
        t->dd_max_blocks = std::min<long long>((long long)t->sm_count * reg_blocks, (long long)(((size_t)512 << 20) / std::max<size_t>(1, slab_bytes)));
        if (t->dd_max_blocks < 8) t->dd_mode = -1;
    }
    {   // spare rows of no-ops: the interpreter requests ops kRing - 1 steps ahead
        ProgOp nop;
        std::memset(&nop, 0, sizeof(nop));
        ops.insert(ops.end(), (size_t)kRing * G, nop);
    }
    t->ops_bytes = ops.size() * sizeof(ProgOp);
    unsigned ms[kMaxN + 1][kNumCodes];
    for (int r = 0; r <= kMaxN; r++)
        for (int tt = 0; tt < kNumCodes; tt++) ms[r][tt] = (unsigned)multiset_count(r, tt);
    bool ok = cudaMalloc(&t->d_info, sizeof(ClassInfo) * nc) == cudaSuccess &&
              cudaMalloc(&t->d_sortkey, sizeof(uint32_t) * nc) == cudaSuccess &&
              cudaMalloc(&t->d_ops, t->ops_bytes) == cudaSuccess;
    ok = ok && cudaMemcpy(t->d_info, info.data(), sizeof(ClassInfo) * nc, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(t->d_sortkey, sortkey.data(), sizeof(uint32_t) * nc, cudaMemcpyHostToDevice) == cudaSuccess &&
         (ops.empty() || cudaMemcpy(t->d_ops, ops.data(), ops.size() * sizeof(ProgOp), cudaMemcpyHostToDevice) == cudaSuccess) &&
         cudaMemcpyToSymbol(c_mscount, ms, sizeof(ms)) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        prog_table_destroy(t);
        return BG_ENOMEM;
    }
    if (nc + 1 <= kFusedScanBins) {   // fused-scan prepass of small batches (optional: without it, the scan launch)
        const size_t bytes = sizeof(uint32_t) * (2 * ((size_t)nc + 1) + 1);
        if (cudaMalloc(&t->d_small, bytes) != cudaSuccess || cudaMemset(t->d_small, 0, bytes) != cudaSuccess) {
            cudaGetLastError();
            if (t->d_small) cudaFree(t->d_small);
            t->d_small = nullptr;
        }
    }
    {   // side streams of the tier launches (small batches, see cdbg_prog_launch); without them: one stream
        bool sok = cudaEventCreateWithFlags(&t->fork_ev, cudaEventDisableTiming) == cudaSuccess;
        int made = 0;
        for (; sok && made < kTiers - 1; made++)
            sok = cudaStreamCreateWithFlags(&t->aux[made], cudaStreamNonBlocking) == cudaSuccess &&
                  cudaEventCreateWithFlags(&t->join_ev[made], cudaEventDisableTiming) == cudaSuccess;
        t->has_streams = sok;
        if (!sok) cudaGetLastError();
    }
    *out = t;
    return BG_OK;
}

// ---- continuous colour / polarisation states (Eq. 5-14): one dense program ----------
int prog_table_create_dense(int n, int G, size_t slab_limit, bool real, ProgTable** out) {
    *out = nullptr;
    if (slab_limit == 0 || slab_limit > kMaxSlabBytes) slab_limit = kMaxSlabBytes;
    if (n < 4 || n > kMaxN || G < 32 || G > 256 || (G & (G - 1))) return BG_EINVAL;
    ClassProgram cp;
    int code[kMaxN] = {0};
    build_program(n, G, code, cp, true, real);
    if (!cp.valid || cp.state_cx > 65535) return BG_EUNSUPPORTED;
    const size_t elem = real ? 8 : 16;
    const bool spill = (size_t)cp.state_cx * elem > slab_limit;
    if (spill && G < 128) return BG_EUNSUPPORTED;
    ClassInfo ci;
    std::memset(&ci, 0, sizeof(ci));
    ci.valid = 1;
    ci.state_cx = (uint16_t)cp.state_cx;
    ci.total_steps = (uint32_t)cp.total_steps;
    ci.n_sync = (uint32_t)cp.n_sync;
    std::vector<ProgOp> ops = cp.ops;
    ProgOp nop;
    std::memset(&nop, 0, sizeof(nop));
    ops.insert(ops.end(), (size_t)kRing * G, nop);
    ProgTable* t = new (std::nothrow) ProgTable();
    if (!t) return BG_ENOMEM;
    std::memset(t, 0, sizeof(*t));
    t->n = n; t->G = G; t->num_classes = 1; t->max_state_cx = cp.state_cx;
    t->dense = true;
    t->real = real;
    t->dd_mode = -1;
    t->rec_bytes = kRecHeaderBytes + 96 * n;
    for (int k = 0; k < kTiers; k++) {
        t->tiers.slab_cx[k] = std::min<int>(cp.state_cx, (int)(slab_limit / elem));
        t->tiers.first_key[k] = k == 0 ? 0 : 1;
    }
    t->tiers.first_key[kTiers] = 1;
    t->spill = spill;
    {
        const size_t smem0 = (size_t)t->tiers.slab_cx[0] * elem;
        const int block = G > 32 ? G : 32;
        t->spill_blocks_per_sm = (int)std::max<size_t>(1, std::min<size_t>(65536 / (168 * block), (228 * 1024) / (smem0 + 1024 + 512)));
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, dev);
    }
    t->ops_bytes = ops.size() * sizeof(ProgOp);
    bool ok = cudaMalloc(&t->d_info, sizeof(ClassInfo)) == cudaSuccess && cudaMalloc(&t->d_ops, t->ops_bytes) == cudaSuccess;
    ok = ok && cudaMemcpy(t->d_info, &ci, sizeof(ci), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(t->d_ops, ops.data(), t->ops_bytes, cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        prog_table_destroy(t);
        return BG_ENOMEM;
    }
    *out = t;
    return BG_OK;
}

// one record per event, in input order: header | per gluon p (4), phi, eta (3), etabar (3), pad
__global__ void __launch_bounds__(256)
cdbg_pack_continuous_kernel(int n, long long N, const double* __restrict__ mom, const double* __restrict__ phi,
                            const double* __restrict__ eta, char* __restrict__ rec, int rec_bytes,
                            uint32_t* __restrict__ bounds) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e == 0) {
        bounds[0] = 0;
        for (int k = 1; k <= kTiers; k++) bounds[k] = (uint32_t)N;
    }
    if (e >= N) return;
    char* r = rec + (size_t)e * rec_bytes;
    EventHeader h;
    h.event = (uint32_t)e; h.cls = 0; h.perm = 0;
    for (int k = 0; k < n; k++) h.perm |= (uint64_t)k << (4 * k);
    *reinterpret_cast<EventHeader*>(r) = h;
    double2* g = reinterpret_cast<double2*>(r + kRecHeaderBytes);
    for (int k = 0; k < n; k++) {
        double v[12];
        for (int c = 0; c < 4; c++) v[c] = mom[(size_t)(k * 4 + c) * N + e];
        v[4] = phi[(size_t)k * N + e];
        for (int c = 0; c < 6; c++) v[5 + c] = eta[(size_t)(k * 6 + c) * N + e];
        v[11] = 0.0;
        for (int c = 0; c < 6; c++) g[k * 6 + c] = make_double2(v[2 * c], v[2 * c + 1]);
    }
}

void prog_table_destroy(ProgTable* t) {
    if (!t) return;
    if (t->dd_table) prog_table_destroy(t->dd_table);
    std::free(t->h_closure);
    if (t->d_small) cudaFree(t->d_small);
    if (t->has_streams) {
        for (int i = 0; i < kTiers - 1; i++) { cudaStreamDestroy(t->aux[i]); cudaEventDestroy(t->join_ev[i]); }
        cudaEventDestroy(t->fork_ev);
    }
    if (t->d_info) cudaFree(t->d_info);
    if (t->d_sortkey) cudaFree(t->d_sortkey);
    if (t->d_ops) cudaFree(t->d_ops);
    delete t;
}

size_t prog_state_bytes(const ProgTable* t) { return t ? (size_t)t->max_state_cx * (t->real ? 8 : 16) : 0; }
int prog_lanes(const ProgTable* t) { return t ? t->G : 0; }
int prog_dd_mode(const ProgTable* t) { return t ? t->dd_mode : -1; }

// scratch: records (32 + 32 n) B x N | perm u64[N] | cls u32[N] | hist u32[num_classes + 1] | tier bounds (64 B) |
//          flag counters (64 B: double-double list counts | its tickets | second-stage list counts | its tickets) |
//          double-double list u32[N] | second-stage list u32[N] | marks u8[N] | spill slabs (FP64) | spill slabs (capped FP64 launches
//          and double-double re-evaluation)
static size_t prog_flag_offset(const ProgTable* t, long long N) {
    return ((size_t)N * (12 + t->rec_bytes) + ((size_t)t->num_classes + 1) * 4 + 15) / 16 * 16 + 64;
}
static size_t prog_spill_offset(const ProgTable* t, long long N) {
    // counters | two lists | marks | work area of the list compaction
    const size_t lists_end = (prog_flag_offset(t, N) + 64 + (size_t)N * 9 + 15) / 16 * 16;
    return (lists_end + 64 + ((size_t)N / 4096 + 8) * 8 + 255) / 256 * 256;
}
static size_t prog_spill_bytes(const ProgTable* t) {
    // spill kernels run a fixed number of blocks per SM, each with a slab for the largest state
    return t->spill ? ((size_t)t->sm_count * t->spill_blocks_per_sm * t->max_state_cx * 16 + 255) / 256 * 256 : 0;
}
size_t prog_scratch_bytes(const ProgTable* t, long long N) {
    const size_t epw = t->G >= 32 ? 1 : 32 / t->G;
    size_t dd_spill = t->dd_mode == 1 ? (size_t)t->dd_max_blocks * epw * t->max_state_cx * 32 : 0;
    if (const ProgTable* d = t->dd_table) {
        const size_t depw = d->G >= 32 ? 1 : 32 / d->G;
        if (d->dd_mode == 1) dd_spill = std::max(dd_spill, (size_t)d->dd_max_blocks * depw * d->max_state_cx * 32);
    }
    // the slabs of the capped FP64 launches share the region of the re-evaluation's (which runs after them)
    const size_t cap_spill = t->cap_cx > 0 ? (size_t)t->sm_count * t->cap_blocks * epw * t->max_state_cx * 16 : 0;
    return prog_spill_offset(t, N) + prog_spill_bytes(t) + std::max(dd_spill, cap_spill);
}

// flagged events of the most recent launch with a conditioning threshold (synchronises the stream's work first)
cudaError_t prog_flagged_count(const ProgTable* t, long long N, const void* scratch, long long* count) {
    uint32_t c[kTiers] = {0, 0, 0, 0};
    const cudaError_t err = cudaMemcpy(c, (const char*)scratch + prog_flag_offset(t, N), sizeof(c), cudaMemcpyDeviceToHost);
    *count = 0;
    for (int k = 0; k < kTiers; k++) *count += c[k];
    return err;
}
// ... and how many of its events went through the second (rotated-frame FP64) stage
cudaError_t prog_twin_count(const ProgTable* t, long long N, const void* scratch, long long* count) {
    uint32_t c[kTiers] = {0, 0, 0, 0};
    const cudaError_t err = cudaMemcpy(c, (const char*)scratch + prog_flag_offset(t, N) + 2 * kTiers * sizeof(uint32_t), sizeof(c),
                                       cudaMemcpyDeviceToHost);
    *count = 0;
    for (int k = 0; k < kTiers; k++) *count += c[k];
    return err;
}

cudaError_t dispatch_interp_dd(cudaStream_t s, const ProgTable* t, int sm_count, const ProgParams& p, int* launches, bool conc,
                               bool merged, long long tasks_hint);   // bg_cdbg_prog_dd.cu

static cudaError_t dispatch_interp(cudaStream_t s, const ProgTable* t, int sm_count, const ProgParams& p, int* launches,
                                   bool conc = false, long long tasks_hint = 0, bool merged = false) {
    cudaError_t err;
    LaunchShape shape;
    shape.conc = conc;
    shape.tasks_hint = tasks_hint;
    shape.merged = merged;
    shape.spill_blocks = t->spill_blocks_per_sm;
    if (t->real) {   // continuous states with real polarisations: all-real arithmetic
        switch (t->G) {
            case 32: return launch_interp<32, false, double>(s, t, sm_count, p, launches, shape);
            case 64: return launch_interp<64, false, double>(s, t, sm_count, p, launches, shape);
            case 128:
                return t->spill ? launch_interp<128, true, double>(s, t, sm_count, p, launches, shape)
                                : launch_interp<128, false, double>(s, t, sm_count, p, launches, shape);
            default:
                return t->spill ? launch_interp<256, true, double>(s, t, sm_count, p, launches, shape)
                                : launch_interp<256, false, double>(s, t, sm_count, p, launches, shape);
        }
    }
    if (!p.rec) {    // UNSORTED (n <= 5): one launch that classifies its events itself and reads the caller's arrays
        shape.merged = true;
        switch (t->G) {
            case 1: return launch_interp<1, false, cx, false, true>(s, t, sm_count, p, launches, shape);
            case 2: return launch_interp<2, false, cx, false, true>(s, t, sm_count, p, launches, shape);
            case 4: return launch_interp<4, false, cx, false, true>(s, t, sm_count, p, launches, shape);
            default: return cudaErrorInvalidValue;
        }
    }
    if (t->cap_cx > 0 && p.spill) {     // heavy tiers: capped shared-memory state + L2 slab (see prog_table_create)
        shape.hybrid = true;
        shape.cap_cx = t->cap_cx;
        shape.spill_blocks = t->cap_blocks;
        shape.max_blocks = (long long)t->sm_count * t->cap_blocks;
    }
    switch (t->G) {
        case 1: err = launch_interp<1, false>(s, t, sm_count, p, launches, shape); break;
        case 2: err = launch_interp<2, false>(s, t, sm_count, p, launches, shape); break;
        case 4: err = launch_interp<4, false, cx, true>(s, t, sm_count, p, launches, shape); break;
        case 8: err = launch_interp<8, false, cx, true>(s, t, sm_count, p, launches, shape); break;
        case 16: err = launch_interp<16, false>(s, t, sm_count, p, launches, shape); break;
        case 32: err = launch_interp<32, false>(s, t, sm_count, p, launches, shape); break;
        case 64: err = launch_interp<64, false>(s, t, sm_count, p, launches, shape); break;
        case 128:
            err = t->spill ? launch_interp<128, true>(s, t, sm_count, p, launches, shape)
                           : launch_interp<128, false>(s, t, sm_count, p, launches, shape);
            break;
        default:
            err = t->spill ? launch_interp<256, true>(s, t, sm_count, p, launches, shape)
                           : launch_interp<256, false>(s, t, sm_count, p, launches, shape);
            break;
    }
    return err;
}

// Ordered flag lists: the interpreter marked the events (ProgParams::mark); two small kernels append the record
// positions with mark `want_a` to list_a and those with `want_b` to list_b (nullptr: none) behind what the lists hold, tier
// by tier, in record order: (1) counts per chunk of kCompactChunk records, (2) every chunk adds up the counts of the
// chunks before it in its tier and places its entries.  Records are sorted by class, longest programs first, so the
// events one warp of a list launch takes share a class, and the tickets hand out the longest tasks first.
constexpr int kCompactThreads = 256, kCompactPer = 16, kCompactChunk = kCompactThreads * kCompactPer;
struct CompactWork {            // behind the marks in the scratch buffer
    uint32_t start[2][kTiers];  // list lengths before this compaction
    uint32_t counts[1][2];      // [chunks][2]: entries of a chunk for list a, b
};
__device__ __forceinline__ bool compact_chunk_of_block(const uint32_t* bounds, int* tier_out, uint32_t* chunk_out) {
    int tier = 0;
    uint32_t chunk = blockIdx.x;
    for (; tier < kTiers; tier++) {
        const uint32_t chunks = (bounds[tier + 1] - bounds[tier] + kCompactChunk - 1) / kCompactChunk;
        if (chunk < chunks) break;
        chunk -= chunks;
    }
    *tier_out = tier; *chunk_out = chunk;
    return tier < kTiers;
}
__device__ __forceinline__ void compact_bits(const uint8_t* mark, uint32_t begin, uint32_t end, int want_a, int want_b, unsigned* bits_a,
                                             unsigned* bits_b) {
    unsigned a = 0, b = 0;
#pragma unroll
    for (int i = 0; i < kCompactPer; i++) {
        const uint32_t pos = begin + i;
        const int m = pos < end ? (int)mark[pos] : 0;
        a |= (unsigned)(m == want_a) << i;
        b |= (unsigned)(want_b >= 0 && m == want_b) << i;
    }
    *bits_a = a; *bits_b = b;
}
__global__ void __launch_bounds__(kCompactThreads)
cdbg_compact_count_kernel(const uint8_t* __restrict__ mark, const uint32_t* __restrict__ bounds, int want_a, const uint32_t* __restrict__ count_a,
                          int want_b, const uint32_t* __restrict__ count_b, CompactWork* __restrict__ work) {
    if (blockIdx.x == 0 && threadIdx.x < kTiers) {
        work->start[0][threadIdx.x] = count_a[threadIdx.x];
        work->start[1][threadIdx.x] = want_b >= 0 ? count_b[threadIdx.x] : 0u;
    }
    int tier; uint32_t chunk;
    if (!compact_chunk_of_block(bounds, &tier, &chunk)) {
        if (threadIdx.x == 0) { work->counts[blockIdx.x][0] = 0; work->counts[blockIdx.x][1] = 0; }
        return;
    }
    unsigned bits_a, bits_b;
    compact_bits(mark, bounds[tier] + chunk * kCompactChunk + threadIdx.x * kCompactPer, bounds[tier + 1], want_a, want_b, &bits_a, &bits_b);
    unsigned x = (unsigned)__popc(bits_a) | ((unsigned)__popc(bits_b) << 16);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(0xFFFFFFFFu, x, d);
    __shared__ unsigned warp_tot[kCompactThreads / 32];
    if ((threadIdx.x & 31) == 0) warp_tot[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned total = 0;
        for (int w = 0; w < kCompactThreads / 32; w++) total += warp_tot[w];
        work->counts[blockIdx.x][0] = total & 0xFFFFu;
        work->counts[blockIdx.x][1] = total >> 16;
    }
}
__global__ void __launch_bounds__(kCompactThreads)
cdbg_compact_place_kernel(const uint8_t* __restrict__ mark, const uint32_t* __restrict__ bounds, int want_a, uint32_t* __restrict__ list_a,
                          uint32_t* __restrict__ count_a, int want_b, uint32_t* __restrict__ list_b, uint32_t* __restrict__ count_b,
                          const CompactWork* __restrict__ work) {
    int tier; uint32_t chunk;
    if (!compact_chunk_of_block(bounds, &tier, &chunk)) return;
    const uint32_t first = bounds[tier], end = bounds[tier + 1];
    const uint32_t begin = first + chunk * kCompactChunk + threadIdx.x * kCompactPer;
    unsigned bits_a, bits_b;
    compact_bits(mark, begin, end, want_a, want_b, &bits_a, &bits_b);
    // entries of the chunks before this one in the tier (a few hundred chunks at most per 2^20 events)
    __shared__ unsigned warp_tot[kCompactThreads / 32], base_a, base_b;
    unsigned pa = 0, pb = 0;
    for (uint32_t c = threadIdx.x; c < chunk; c += kCompactThreads) {
        pa += work->counts[blockIdx.x - chunk + c][0];
        pb += work->counts[blockIdx.x - chunk + c][1];
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { pa += __shfl_xor_sync(0xFFFFFFFFu, pa, d); pb += __shfl_xor_sync(0xFFFFFFFFu, pb, d); }
    __shared__ unsigned part_a[kCompactThreads / 32], part_b[kCompactThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { part_a[warp] = pa; part_b[warp] = pb; }
    // block-wide exclusive scan of this chunk's own counts (packed: a in the low, b in the high half)
    const unsigned mine = (unsigned)__popc(bits_a) | ((unsigned)__popc(bits_b) << 16);
    unsigned x = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned y = __shfl_up_sync(0xFFFFFFFFu, x, d);
        if (lane >= d) x += y;
    }
    if (lane == 31) warp_tot[warp] = x;
    __syncthreads();
    unsigned before = x - mine, total = 0;
    for (int w = 0; w < kCompactThreads / 32; w++) {
        if (w < warp) before += warp_tot[w];
        total += warp_tot[w];
    }
    if (threadIdx.x == 0) {
        unsigned a = work->start[0][tier], b = work->start[1][tier];
        for (int w = 0; w < kCompactThreads / 32; w++) { a += part_a[w]; b += part_b[w]; }
        base_a = a; base_b = b;
        const uint32_t chunks = (end - first + kCompactChunk - 1) / kCompactChunk;
        if (chunk + 1 == chunks) {       // the last chunk of the tier knows the new lengths
            count_a[tier] = a + (total & 0xFFFFu);
            if (want_b >= 0) count_b[tier] = b + (total >> 16);
        }
    }
    __syncthreads();
    uint32_t at_a = first + base_a + (before & 0xFFFFu), at_b = first + base_b + (before >> 16);
#pragma unroll
    for (int i = 0; i < kCompactPer; i++) {
        if ((bits_a >> i) & 1u) list_a[at_a++] = begin + i;
        if ((bits_b >> i) & 1u) list_b[at_b++] = begin + i;
    }
}

// the UNSORTED path: discrete states, at most 4 lanes per event, every class in the one (last) tier, and a batch small
// enough for the launches saved to outweigh the divergence of unsorted warps (measured, FP64 kernels: n = 4 2^12 ... 2^17
// events 32 -> 16, 32 -> 18, 42 -> 35, 56 -> 53 us, 2^18 93 -> 96 us; n = 5 2^10 ... 2^15 36 -> 21, 36 -> 23, 42 -> 35,
// 52 -> 51 us, 2^16 71 -> 88 us)
static bool prog_unsorted(const ProgTable* t, long long N) {
    if (t->dense || t->spill || t->G > 4 || t->n > 5 || t->tiers.first_key[kTiers - 1] != 0) return false;
    return N <= (t->n == 4 ? (1ll << 17) : (1ll << 15));
}

cudaError_t cdbg_prog_launch(cudaStream_t s, const ProgTable* t, int sm_count, long long N, const double* mom,
                             const signed char* hel, const signed char* col, double* out, void* scratch,
                             int* launches, cudaEvent_t ev0, cudaEvent_t ev1, double tau, double tau_rho, cudaEvent_t ev_mid,
                             double tau_twin, double tau_twin_ward, bool rotated) {
    if (tau > 0.0 && t->dd_mode < 0) return cudaErrorNotSupported;
    const int rec_bytes = t->rec_bytes;
    char* rec = (char*)scratch;
    uint64_t* perm = (uint64_t*)(rec + (size_t)N * rec_bytes);
    uint32_t* cls = (uint32_t*)(perm + N);
    uint32_t* hist = cls + N;
    uint32_t* bounds = hist + ((size_t)t->num_classes + 1);
    uint32_t* flag_count = (uint32_t*)((char*)scratch + prog_flag_offset(t, N));
    uint32_t* flag_list = flag_count + 16;
    const int nbins = (int)t->num_classes + 1;
    cudaError_t err = cudaSuccess;
    // n <= 5, small batches, FP64 kernels alone: classify, sort and scatter take more than half of a step (n = 4, 2^16
    // events: 27 of 43 us in the kernels alone).  The UNSORTED instantiations skip them - tasks in input order,
    // classification inside the interpreter: one launch (DESIGN.md 5.1c for what that costs at larger sizes).
    if (tau <= 0.0 && prog_unsorted(t, N)) {
        ProgParams p;
        p.n = t->n; p.N = N; p.out = out;
        p.info = t->d_info; p.ops = t->d_ops; p.rec = nullptr; p.rec_bytes = rec_bytes; p.rec_gstride = 4;
        p.mom = mom; p.hel = hel; p.col = col;
        p.bounds = nullptr;
        p.zero = 0;
        p.spill = nullptr;
        p.spill_cx = t->max_state_cx;
        p.tier = kTiers - 1;
        p.merged = 0;
        p.slab_cx = t->max_state_cx;
        p.tau2 = tau;              // 0, or a diagnostic code
        p.tau_rho = 0.0;
        p.flag_list = nullptr; p.flag_count = nullptr; p.list = nullptr; p.list_count = nullptr; p.ticket = nullptr;
        p.twin = rotated ? 1 : 0;
        p.tw2 = 0.0; p.td = 0.0; p.soft_count = nullptr; p.soft_list = nullptr; p.mark = nullptr;
        *launches = 0;
        if (ev0) cudaEventRecord(ev0, s);
        err = dispatch_interp(s, t, sm_count, p, launches);
        if (ev1) cudaEventRecord(ev1, s);
        return err;
    }
    const unsigned eb = (unsigned)((N + kPreEvents - 1) / kPreEvents);
    const size_t hist_smem = sizeof(uint32_t) * nbins;
    const size_t stage_bytes = (size_t)(kStageThreads / 32) * (32 * (rec_bytes + 16) + 256);
    const size_t hist_words = ((size_t)nbins + 3) & ~(size_t)3;
    const bool fused = t->d_small && N <= kFusedScanEvents && 2 * hist_words * sizeof(uint32_t) + stage_bytes <= 100 * 1024;
    if (!fused && (err = cudaMemsetAsync(hist, 0, sizeof(uint32_t) * nbins, s)) != cudaSuccess) return err;
    if (fused) {
        static int configured_device = -1;
        int device = 0;
        cudaGetDevice(&device);
        if (configured_device != device) {
            cudaFuncSetAttribute(cdbg_classify_kernel<true, kSmallThreads, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
            cudaFuncSetAttribute(cdbg_scatter_staged_kernel<true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
            configured_device = device;
        }
        uint32_t* counts = t->d_small;
        FusedScan fs;
        fs.counts = counts; fs.ticket = counts + 2 * nbins; fs.bounds = bounds; fs.N = (uint32_t)N; fs.tiers = t->tiers;
        // one event per thread and 256-thread blocks: a small batch is less than one wave of the 1024-event blocks
        // of the large-batch kernels, and each thread is a chain of dependent loads and atomics
        const unsigned cb = (unsigned)((N + kSmallThreads - 1) / kSmallThreads);
        cdbg_classify_kernel<true, kSmallThreads, 1><<<cb, kSmallThreads, hist_smem, s>>>(t->n, N, t->num_classes, col, t->d_info,
                                                                                     t->d_sortkey, cls, perm, counts, flag_count);
        const unsigned sb = (unsigned)((N + kStageThreads - 1) / kStageThreads);
        cdbg_scatter_staged_kernel<true, 1><<<sb, kStageThreads, 2 * hist_words * sizeof(uint32_t) + stage_bytes, s>>>(
            t->n, N, t->num_classes, cls, perm, t->d_sortkey, mom, hel, counts + nbins, rec, rec_bytes, fs);
    } else if (hist_smem <= 160 * 1024) {
        static int configured_device = -1;
        int device = 0;
        cudaGetDevice(&device);
        if (configured_device != device) {
            cudaFuncSetAttribute(cdbg_classify_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
            cudaFuncSetAttribute(cdbg_scatter_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
            cudaFuncSetAttribute(cdbg_scatter_staged_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
            configured_device = device;
        }
        cdbg_classify_kernel<true><<<eb, kPreThreads, hist_smem, s>>>(t->n, N, t->num_classes, col, t->d_info,
                                                                      t->d_sortkey, cls, perm, hist, flag_count);
        cdbg_scan_kernel<<<1, 1024, 0, s>>>(hist, nbins, t->tiers, bounds, (uint32_t)N);
        const size_t stage_smem = (((size_t)nbins + 3) & ~(size_t)3) * sizeof(uint32_t) +
                                  (size_t)(kStageThreads / 32) * (32 * (rec_bytes + 16) + 256);
        if (stage_smem <= 100 * 1024) {
            const unsigned sb = (unsigned)((N + kStageEvents - 1) / kStageEvents);
            cdbg_scatter_staged_kernel<false><<<sb, kStageThreads, stage_smem, s>>>(t->n, N, t->num_classes, cls, perm, t->d_sortkey,
                                                                                   mom, hel, hist, rec, rec_bytes, FusedScan());
        } else {
            cdbg_scatter_kernel<true><<<eb, kPreThreads, hist_smem, s>>>(t->n, N, t->num_classes, cls, perm, t->d_sortkey, mom,
                                                                         hel, hist, rec, rec_bytes);
        }
    } else {
        cdbg_classify_kernel<false><<<eb, kPreThreads, 0, s>>>(t->n, N, t->num_classes, col, t->d_info, t->d_sortkey,
                                                               cls, perm, hist, flag_count);
        cdbg_scan_kernel<<<1, 1024, 0, s>>>(hist, nbins, t->tiers, bounds, (uint32_t)N);
        cdbg_scatter_kernel<false><<<eb, kPreThreads, 0, s>>>(t->n, N, t->num_classes, cls, perm, t->d_sortkey, mom, hel, hist,
                                                              rec, rec_bytes);
    }
    if ((err = cudaGetLastError()) != cudaSuccess) return err;
    ProgParams p;
    p.n = t->n; p.N = N; p.out = out;
    p.info = t->d_info; p.ops = t->d_ops; p.rec = rec; p.rec_bytes = rec_bytes; p.rec_gstride = 4;
    p.bounds = bounds;
    p.mom = nullptr; p.hel = nullptr; p.col = nullptr;
    p.zero = 0;
    p.spill = t->spill ? (double2*)((char*)scratch + prog_spill_offset(t, N)) : nullptr;
    if (t->cap_cx > 0) p.spill = (double2*)((char*)scratch + prog_spill_offset(t, N) + prog_spill_bytes(t));
    p.spill_cx = t->max_state_cx;
    p.tier = 0;
    p.merged = 0;
    p.slab_cx = t->max_state_cx;
    p.tau2 = tau < 0.0 ? tau : tau * tau;
    p.tau_rho = tau_rho;
    p.flag_list = flag_list;
    p.flag_count = flag_count;
    p.list = nullptr;
    p.list_count = nullptr;
    p.ticket = flag_count + kTiers;
    p.twin = rotated ? 1 : 0;
    const bool cascade = tau > 0.0 && tau_twin_ward > tau;
    p.tw2 = cascade ? tau_twin_ward * tau_twin_ward : 0.0;
    p.td = tau_twin;
    p.soft_count = flag_count + 2 * kTiers;
    p.soft_list = flag_list + N;
    // Ordered lists from 2^16 events: the kernels mark, a compaction kernel builds the lists class by class, and with
    // warp-shared lane counts (n <= 7) the warps of the later stages run 8 (4) events of ONE class instead of 8 arbitrary ones -
    // and the tickets hand out the longest programs first: double-double stage 0.76 -> 0.65 ms (n = 6, 2^20 events), 0.93 ->
    // 0.72 ms (n = 7, 2^18), 0.23 -> 0.20 ms (n = 5, 2^20), four small launches included; block-per-event lane counts
    // gain the ticket order only (n = 8, 9: -2 ... -3 % of the step, n >= 10: equal).  Smaller batches (later stages one
    // task deep) keep the atomic appends.
    const bool ordered = tau > 0.0 && N >= (1ll << 16);
    uint8_t* const mark = reinterpret_cast<uint8_t*>(flag_list + 2 * N);
    CompactWork* const work = reinterpret_cast<CompactWork*>(reinterpret_cast<char*>(flag_count) + ((size_t)64 + (size_t)N * 9 + 15) / 16 * 16);
    p.mark = ordered ? mark : nullptr;
    const unsigned compact_blocks = (unsigned)((N + kCompactChunk - 1) / kCompactChunk + kTiers);
    *launches = fused ? 2 : 3;
    if (ev0) cudaEventRecord(ev0, s);
    err = dispatch_interp(s, t, sm_count, p, launches, true);
    if (tau > 0.0 && ev_mid) cudaEventRecord(ev_mid, s);      // (the list building counts as part of the later stages)
    if (ordered && err == cudaSuccess) {
        cdbg_compact_count_kernel<<<compact_blocks, kCompactThreads, 0, s>>>(mark, bounds, 1, p.soft_count, 2, flag_count, work);
        cdbg_compact_place_kernel<<<compact_blocks, kCompactThreads, 0, s>>>(mark, bounds, 1, p.soft_list, p.soft_count, 2, flag_list, flag_count, work);
        *launches += 2;
    }
    if (cascade && err == cudaSuccess) {
        // second stage: the events between the two thresholds once more in FP64, in the rotated frame; out[] keeps the
        // first result, and what disagrees joins the double-double list
        p.twin = rotated ? 2 : 3;
        p.list = p.soft_list;
        p.list_count = p.soft_count;
        p.ticket = flag_count + 3 * kTiers;
        // One launch for the lists of all tiers where measured faster: 4 lanes per event (n = 5, 6) from 2^18 events
        // (2^16: +4 %, 2^20: -1 %), 8 - 64 lanes (n = 7 - 9: -2 ... -5 % at 2^16, equal at 2^18) and the spill kernels
        // (n >= 11: -1 ... -5 %); 128 lanes without spill (n = 10) keep the tiers' own launch shapes (+2 %).
        const bool merged = t->spill || (t->G <= 4 ? N >= (1ll << 18) : t->G <= 64);
        err = dispatch_interp(s, t, sm_count, p, launches, true, std::max<long long>(1, N / 16), merged);
        if (ordered && err == cudaSuccess) {     // what the second stage rejected, behind the first stage's own double-double list
            cdbg_compact_count_kernel<<<compact_blocks, kCompactThreads, 0, s>>>(mark, bounds, 3, flag_count, -1, nullptr, work);
            cdbg_compact_place_kernel<<<compact_blocks, kCompactThreads, 0, s>>>(mark, bounds, 3, flag_list, flag_count, -1, nullptr, nullptr, work);
            *launches += 2;
        }
    }
    if (tau > 0.0 && err == cudaSuccess) {
        // the flagged events of every tier once more, in double-double arithmetic (overwrites their out[])
        p.tau2 = 0.0;
        p.twin = 0;
        p.ticket = flag_count + kTiers;
        p.list = flag_list;
        p.list_count = flag_count;
        p.spill = t->dd_mode == 1 ? (double2*)((char*)scratch + prog_spill_offset(t, N) + prog_spill_bytes(t)) : nullptr;
        // few flagged events per tier for batches up to 2^19: the tier launches overlap their ramp-up and tails
        // one launch walks the lists of all tiers (their capped shared state has one size): few tasks per tier, each
        // 14 x an FP64 task, so per-tier launches were mostly tails (n = 6, 2^20 events: 1.15 -> 0.80 ms after the first pass)
        const ProgTable* d = t->dd_table && t->dd_table->dd_mode == 1 ? t->dd_table : t;     // (n = 8, 9: half the lanes)
        p.info = d->d_info; p.ops = d->d_ops; p.spill_cx = d->max_state_cx;
        err = dispatch_interp_dd(s, d, sm_count, p, launches, false, true, std::max<long long>(1, N / 32));
    }
    if (ev1) cudaEventRecord(ev1, s);
    return err;
}

void prog_table_attach_dd(ProgTable* t, ProgTable* dd) {
    if (t->dd_table) prog_table_destroy(t->dd_table);
    t->dd_table = dd;
}

cudaError_t cdbg_dense_launch(cudaStream_t s, const ProgTable* t, int sm_count, long long N, const double* mom,
                              const double* phi, const double* eta, double* out, void* scratch, int* launches,
                              cudaEvent_t ev0, cudaEvent_t ev1) {
    char* rec = (char*)scratch;
    // same scratch layout as the discrete path (perm / cls / histogram areas stay unused)
    uint32_t* bounds = (uint32_t*)(rec + (size_t)N * (t->rec_bytes + 12)) + ((size_t)t->num_classes + 1);
    cdbg_pack_continuous_kernel<<<(unsigned)((N + 255) / 256), 256, 0, s>>>(t->n, N, mom, phi, eta, rec, t->rec_bytes, bounds);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    ProgParams p;
    p.n = t->n; p.N = N; p.out = out;
    p.info = t->d_info; p.ops = t->d_ops; p.rec = rec; p.rec_bytes = t->rec_bytes; p.rec_gstride = 12;
    p.bounds = bounds;
    p.zero = 0;
    p.spill = t->spill ? (double2*)((char*)scratch + prog_spill_offset(t, N)) : nullptr;
    p.spill_cx = t->max_state_cx;
    p.tier = 0;
    p.merged = 0;
    p.slab_cx = t->max_state_cx;
    p.tau2 = 0.0;
    p.tau_rho = 0.0;
    p.flag_list = nullptr; p.flag_count = nullptr; p.list = nullptr; p.list_count = nullptr; p.ticket = nullptr;
    p.mom = nullptr; p.hel = nullptr; p.col = nullptr;
    p.twin = 0; p.tw2 = 0.0; p.td = 0.0; p.soft_list = nullptr; p.soft_count = nullptr; p.mark = nullptr;
    *launches = 1;
    if (ev0) cudaEventRecord(ev0, s);
    err = dispatch_interp(s, t, sm_count, p, launches, false);
    if (ev1) cudaEventRecord(ev1, s);
    return err;
}

}  // namespace bg

// Host-side generator of "colour-class programs" for the colour-dressed recursion (CDBG, Eq. 28-32,
// L187-213) with discrete colour-flow indices.
//
// For fixed (i_k, j_k) the 3x3 colour matrix of every subset current has at most one off-diagonal or up to three
// diagonal non-zero entries (a product of elementary matrices e_ij is elementary), so WHICH vertex evaluations of
// Eq. 29 are non-zero, and where their operands live, depends only on the colour assignment - not on momenta or
// helicities.  |A|^2 is symmetric under relabelling the gluons (p, lambda, i, j permuted together), so events are
// brought to a canonical gluon order (sorted by the colour code 3*i+j, then one chosen gluon moved to the last
// place as the closure leg of Eq. 22) and the structure depends only on the MULTISET of colour codes: the "colour
// class".  For each class this file emits a straight-line program of vertex operations, already distributed
// over G cooperating lanes and grouped into popcount levels, that the CUDA interpreter (bg_cdbg_prog.cu) runs
// for every event of the class.  Nothing here touches floating-point event data.
#pragma once
#include <stdint.h>

#include <vector>

namespace bg {

// One interpreter instruction (16 bytes).  Offsets are in units of one complex double (16 B) inside the
// per-event state block.
struct alignas(16) ProgOp {
    uint16_t offA;    // vector current a = entry of pi_1 (4 cx, followed by its 6-cx tensor if |pi_1| >= 2)
    uint16_t offB;    // vector current b = entry of pi_2
    uint16_t offP1;   // momentum of pi_1 (4 doubles = 2 cx)
    uint16_t offDst;  // target entry (LAST) | for setup ops: destination
    uint16_t offPt;   // momentum of the target subset (written by the target's LAST op)
    uint16_t flags;
    uint32_t extra;   // vertex ops: offset of the momentum of pi_2; EXT: canonical gluon index
};
static_assert(sizeof(ProgOp) == 16, "ProgOp must be 16 bytes");

enum : uint16_t {
    OPF_VALID = 1,     // a vertex evaluation X(a, b)
    OPF_NEG = 2,       // contributes with sign -1
    OPF_TENA = 4,      // pi_1 carries a tensor current
    OPF_TENB = 8,      // pi_2 carries a tensor current
    OPF_FIRST = 16,    // first op of a target: clear the accumulators, P(target) = P(pi_1) + P(pi_2)
    OPF_LAST = 32,     // last op of a target: apply 1/sqrt2 (and 1/P^2), store vector + tensor current and P
    OPF_CLOSURE = 64,  // target is the full set: contract with eps_n instead of storing (Eq. 22)
    OPF_STOREP = 256,  // (with LAST) also store P(target) at offPt: set on one entry per subset
    OPF_FUSED = 512,   // closure vertex X(eps_k at offA, b = the current just finished in registers) . eps_n
    OPF_NOSTORE = 1024,// (with LAST) the finished current stays in registers only (a FUSED op follows)
    OPF_PARTIAL = 2048,// (with LAST) chunk of a split target: raw partial sums -> scratch slot offDst
    OPF_COMBINE = 4096,// add offB partial slots starting at offA, then finish the target like LAST
    OPF_SYNC = 8192,   // barrier among the lanes of the event after this step (end of a level)
    OPF_EXTD = 16384,  // (with EXT) continuous states: real polarisation e(phi) times the 3x3 colour matrix
                       // X[h][g] = etabar_h eta_g -> nine entries of 4 cx from offDst, entry 3h+g (closure target (h,g) reads 3g+h)
    OPF_EXT = 128      // setup: external current of gluon `extra` -> offDst, its momentum -> offPt
};

constexpr int kMaxN = 12;
constexpr int kNumCodes = 9;   // colour code c = 3*(i-1) + (j-1)

struct ClassProgram {
    bool valid = false;          // false: the amplitude vanishes identically for this colour class
    int closure_code = 0;        // colour code of the gluon placed last (closure leg)
    int state_cx = 0;            // per-event state size in complex doubles
    int n_vertex_ops = 0;        // number of OPF_VALID ops
    int total_steps = 0;         // sum over levels of max-lane op count
    int n_sync = 0;              // number of steps that end with a barrier (non-empty levels)
    long long n_orderings = 0;   // CO_MC programs: colour-connected orderings summed (Eq. 19)
    std::vector<uint16_t> level_steps;   // [2n-4]: setup | (main, combine) for popcount 2..n-2 | closure
    std::vector<ProgOp> ops;             // [total_steps][G]
};

// number of multisets of size r over t types
long long multiset_count(int r, int t);
// rank of a count vector m[0..8] (sum = n) in the fixed enumeration order used by host and device
long long class_rank(int n, const int* counts);
// Build the program for canonical colour codes code[0..n-1] (code[n-1] = closure leg), G lanes per event.
// dense: continuous colour states (nine live entries per subset, `code` ignored); real: the state elements are
// doubles instead of complex doubles (a 4-momentum then takes four elements instead of two).
void build_program(int n, int G, const int* code, ClassProgram& out, bool dense = false, bool real = false);
// CO_MC (Eq. 19 with colour-ordered currents): program for canonical colour codes; classes with more than
// max_orderings colour-connected orderings are left invalid with state_cx = -1 (unsupported, not zero).
void build_comc_program(int n, int G, const int* code, ClassProgram& out, long long max_orderings = 20000);
// Build the best program (over the choice of closure leg) for a multiset of colour codes; closure >= 0: with the gluon
// of that colour code as the closure leg (a second table for the same event records).
void build_class(int n, int G, const int* counts, ClassProgram& out, int closure = -1);

}  // namespace bg

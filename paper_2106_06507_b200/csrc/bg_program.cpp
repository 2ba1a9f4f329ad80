// Colour-class program generator (see bg_program.h).  Integer bookkeeping only.
#include "bg_program.h"

#include <algorithm>
#include <cstring>
#include <map>

namespace bg {

long long multiset_count(int r, int t) {
    if (r < 0) return 0;
    if (t == 0) return r == 0 ? 1 : 0;
    const int k = t - 1, N = r + t - 1;   // C(N, k)
    long long num = 1;
    for (int i = 1; i <= k; i++) num = num * (N - k + i) / i;
    return num;
}

long long class_rank(int n, const int* m) {
    long long rank = 0;
    int r = n;
    for (int t = 0; t < kNumCodes - 1; t++) {
        for (int c = 0; c < m[t]; c++) rank += multiset_count(r - c, kNumCodes - 1 - t);
        r -= m[t];
    }
    return rank;
}

namespace {

// colour type of a subset current: 0x40 dead | 0x80|mask diagonal entries | (h<<2)|g one off-diagonal entry |
// 0xFF all nine entries (continuous colour states)
inline bool has_entry(unsigned t, int h, int g) {
    if (t == 0xFFu) return true;
    if (t & 0x80u) return h == g && ((t >> h) & 1u);
    if (t & 0x40u) return false;
    return t == (unsigned)((h << 2) | g);
}

struct VOp {
    int pa, sa, pb, sb;   // subset and slot (0..2) of the two operands; |pa| <= |pb|
    bool neg;
};

struct Target {
    int pi, h, g;
    bool store_p = false;   // its LAST op also stores P(pi) (one entry per subset whose momentum is read later)
    bool used = false;      // read by a later vertex (dead-code elimination)
    bool fused = false;     // |pi| = n-2: not stored; its closure contributions are taken from registers
    std::vector<std::pair<VOp, int>> fuses;   // closure vertices X(eps_k, this) (pb = this entry) and their closure entry
    std::vector<VOp> ops;
    int s = 0;              // slot of the entry inside its subset
    int slot() const { return s; }
};

inline int popc(int x) { return __builtin_popcount((unsigned)x); }

}  // namespace

void build_program(int n, int G, const int* code, ClassProgram& out, bool dense, bool real) {
    out = ClassProgram();
    const int m = n - 1, nsub = 1 << m, full = nsub - 1;
    // dense: every gluon carries a full 3x3 colour matrix (continuous colour states) - all nine entries of every
    // subset current are live and `code` is ignored; otherwise elementary matrices e_ij and at most 3 live entries
    const int SL = dense ? 9 : 3;
    const int PU = real ? 4 : 2;   // state elements of a 4-momentum: two complex doubles, or four doubles (real currents)
    auto slot_of = [&](int h, int g) { return dense ? h * 3 + g : (h == g ? h : 0); };
    int dummy_code[kMaxN] = {0};
    if (dense) code = dummy_code;
    int ci[kMaxN], cj[kMaxN], wk[kMaxN];
    for (int k = 0; k < n; k++) {
        ci[k] = code[k] / 3;
        cj[k] = code[k] % 3;
        wk[k] = (1 << (8 * ci[k])) - (1 << (8 * cj[k]));
    }
    out.closure_code = code[n - 1];

    // ---- phase 1: which entries of which subsets are non-zero, and the vertex evaluations that feed them ----
    std::vector<uint8_t> type(nsub, 0x40);
    for (int k = 0; k < m; k++)
        type[1 << k] = dense ? (uint8_t)0xFF : (ci[k] == cj[k] ? (uint8_t)(0x80u | (1u << ci[k])) : (uint8_t)((ci[k] << 2) | cj[k]));
    std::vector<std::vector<Target>> levels(m + 1);   // by popcount
    std::vector<int> tindex(nsub * SL, -1);           // (subset, slot) -> index in its level
    for (int pi = 3; pi <= full; pi++) {
        if ((pi & (pi - 1)) == 0) continue;
        const int low = pi & -pi, rest = pi ^ low;
        int D = 0;
        for (int k = 0; k < m; k++)
            if ((pi >> k) & 1) D += wk[k];
        int cand_h[9], cand_g[9], ncand = 0;
        bool diag = false;
        if (dense) {
            for (int h = 0; h < 3; h++)
                for (int g = 0; g < 3; g++) { cand_h[ncand] = h; cand_g[ncand] = g; ncand++; }
        } else if (D == 0) {
            diag = true;
            for (int h = 0; h < 3; h++) { cand_h[ncand] = h; cand_g[ncand] = h; ncand++; }
        } else {
            for (int h = 0; h < 3; h++)
                for (int g = 0; g < 3; g++)
                    if (h != g && D == (1 << (8 * h)) - (1 << (8 * g))) { cand_h[0] = h; cand_g[0] = g; ncand = 1; }
        }
        if (pi == full && !dense) {
            // closure, Eq. 22: only the entry contracted with X_n = e_{i_n j_n}
            const int h = cj[n - 1], g = ci[n - 1];
            bool ok = false;
            for (int c = 0; c < ncand; c++) ok = ok || (cand_h[c] == h && cand_g[c] == g);
            ncand = 0;
            if (ok) { cand_h[0] = h; cand_g[0] = g; ncand = 1; }
        }
        unsigned livemask = 0;
        for (int cd = 0; cd < ncand; cd++) {
            const int h = cand_h[cd], g = cand_g[cd];
            Target t;
            t.pi = pi; t.h = h; t.g = g; t.s = slot_of(h, g);
            for (int sub = (rest - 1) & rest;; sub = (sub - 1) & rest) {
                const int p1 = low | sub, p2 = pi ^ p1;
                const unsigned t1 = type[p1], t2 = type[p2];
                if (t1 != 0x40u && t2 != 0x40u) {
                    for (int k = 0; k < 3; k++) {
                        const bool fwd = has_entry(t1, h, k) && has_entry(t2, k, g);
                        const bool bwd = has_entry(t2, h, k) && has_entry(t1, k, g);
                        if (fwd && bwd && h == k && k == g) continue;   // +X - X
                        for (int dir = 0; dir < 2; dir++) {
                            if (dir == 0 ? !fwd : !bwd) continue;
                            const int ah = dir == 0 ? h : k, ag = dir == 0 ? k : g;   // entry of pi_1
                            const int bh = dir == 0 ? k : h, bg_ = dir == 0 ? g : k;  // entry of pi_2
                            VOp o;
                            o.pa = p1; o.sa = slot_of(ah, ag);
                            o.pb = p2; o.sb = slot_of(bh, bg_);
                            o.neg = dir == 1;
                            if (popc(o.pa) > popc(o.pb)) {   // X(a,b) = -X(b,a): keep the smaller subset as `a`
                                std::swap(o.pa, o.pb);
                                std::swap(o.sa, o.sb);
                                o.neg = !o.neg;
                            }
                            t.ops.push_back(o);
                        }
                    }
                }
                if (sub == 0) break;
            }
            if (t.ops.empty()) continue;
            livemask |= diag ? (1u << h) : 1u;
            tindex[pi * SL + t.slot()] = (int)levels[popc(pi)].size();
            levels[popc(pi)].push_back(std::move(t));
        }
        if (pi != full) {
            uint8_t ty = 0x40u;
            if (livemask) ty = dense ? (uint8_t)0xFF : (diag ? (uint8_t)(0x80u | livemask) : (uint8_t)((cand_h[0] << 2) | cand_g[0]));
            type[pi] = ty;
        }
    }
    if (levels[m].empty()) return;   // no closure: amplitude vanishes identically
    out.valid = true;
    // ---- phase 2: closure vertices X(eps_k, J(pi)) with |pi| = n-2 are evaluated straight from the registers
    // that hold the just-finished J(pi), T(pi) ("fused": those currents are never stored), and entries that no
    // later vertex reads are dropped ----
    {
        for (auto& clo : levels[m]) {
            clo.used = true;
            if (m - 1 < 2) continue;
            // the closure entry (h,g) is contracted with eps_n X_n[g][h]: index of that vector behind off_epsn
            const int centry = dense ? clo.g * 3 + clo.h : 0;
            std::vector<VOp> keep;
            for (auto& v : clo.ops) {
                if (popc(v.pa) == 1 && popc(v.pb) == m - 1) {
                    Target& t = levels[m - 1][tindex[v.pb * SL + v.sb]];
                    t.fused = true;
                    t.fuses.push_back({v, centry});
                    t.used = true;
                    continue;
                }
                keep.push_back(v);
            }
            clo.ops.swap(keep);
        }
        for (int pc = m; pc >= 2; pc--)
            for (auto& t : levels[pc]) {
                if (!t.used) continue;
                for (auto& v : t.ops) {
                    if (popc(v.pa) >= 2) levels[popc(v.pa)][tindex[v.pa * SL + v.sa]].used = true;
                    if (popc(v.pb) >= 2) levels[popc(v.pb)][tindex[v.pb * SL + v.sb]].used = true;
                }
            }
        for (int pc = 2; pc < m; pc++) {
            std::vector<Target> keep;
            for (auto& t : levels[pc])
                if (t.used) keep.push_back(std::move(t));
            levels[pc].swap(keep);
        }
    }

    // ---- phase 3: state layout (units of one complex double) ----
    std::vector<int> off(nsub * SL, -1), poff(nsub, -1);
    std::vector<char> need_p(nsub, 0);
    for (int pc = 2; pc <= m; pc++)
        for (auto& t : levels[pc])
            for (auto& v : t.ops) { need_p[v.pa] = 1; need_p[v.pb] = 1; }
    int next = 0;
    for (int k = 0; k < m; k++) {
        if (dense) {
            for (int hg = 0; hg < 9; hg++) { off[(1 << k) * SL + hg] = next; next += 4; }   // eps_k X_k[h][g], hg = 3h+g
        } else {
            off[(1 << k) * SL + slot_of(ci[k], cj[k])] = next;
            next += 4;
        }
    }
    const int off_epsn = next;      // eps_n (dense: the nine vectors eps_n X_n[g][h] at index 3g+h)
    next += dense ? 36 : 4;
    for (int k = 0; k < m; k++) { poff[1 << k] = next; next += PU; }
    // With fewer than 8 events per warp the bank group of an element depends on its offset: one element of padding
    // after every entry makes the entry starts run through all residues (10 + 2 would only ever give multiples of 4).
    const int pad = G >= 8 ? 1 : 0;
    for (int pc = 2; pc < m; pc++)
        for (auto& t : levels[pc]) {
            if (!t.fused) { off[t.pi * SL + t.slot()] = next; next += 10 + pad; }
            if (need_p[t.pi] && poff[t.pi] < 0) { poff[t.pi] = next; next += PU; t.store_p = true; }
        }
    out.level_steps.assign(2 * m - 2, 0);   // setup | (main, combine) per popcount 2..n-2 | closure

    // ---- phase 4: deal the work of every level over the G lanes and emit ----
    // Shared-memory bank groups: the state is laid out [offset][event] in 16-byte elements, so the 8 lanes of a
    // quarter-warp (EPW events x 8/EPW lanes of each) hit distinct bank groups iff the lanes of one event read
    // offsets that differ modulo 8/EPW.  The order of the vertices inside a unit is free, so every lane picks, step
    // by step, the remaining vertex of its unit that collides least with what its neighbours read at that step.
    auto reduce_bank_conflicts = [&](std::vector<std::vector<ProgOp>>& lanes) {
        auto swap_operands = [](ProgOp& x, ProgOp& y) {
            std::swap(x.offA, y.offA); std::swap(x.offB, y.offB); std::swap(x.offP1, y.offP1); std::swap(x.extra, y.extra);
            const uint16_t keep = OPF_NEG | OPF_TENA | OPF_TENB;
            const uint16_t fx = x.flags & keep, fy = y.flags & keep;
            x.flags = (uint16_t)((x.flags & ~keep) | fy);
            y.flags = (uint16_t)((y.flags & ~keep) | fx);
        };
        // Lanes of one warp whose vertices differ in kind (tensor of pi_1 / pi_2 present or not) run the tensor
        // contractions one kind after the other; inside every unit the vertices are therefore ordered by kind
        // (both tensors, one, none), which lines the kinds up across the lanes of a level.
        auto kind = [](const ProgOp& o) { return ((o.flags & OPF_TENA) ? 2 : 0) + ((o.flags & OPF_TENB) ? 1 : 0); };
        for (auto& ln : lanes)
            for (size_t s = 0; s < ln.size();) {
                if (!(ln[s].flags & OPF_VALID)) { s++; continue; }
                size_t last = s;
                while (!(ln[last].flags & OPF_LAST)) last++;
                for (size_t i = s; i <= last; i++) {          // selection sort: units are short
                    size_t best = i;
                    for (size_t c = i + 1; c <= last; c++)
                        if (kind(ln[c]) > kind(ln[best])) best = c;
                    if (best != i) swap_operands(ln[i], ln[best]);
                }
                s = last + 1;
            }
        const int EPW = G >= 32 ? 1 : 32 / G;
        const int M = 8 / EPW, group = 8 / EPW;
        if (M <= 1 || G < group) return;
        size_t steps = 0;
        for (auto& l : lanes) steps = std::max(steps, l.size());
        for (size_t s = 0; s < steps; s++)
            for (int g0 = 0; g0 < G; g0 += group)
                for (int l = g0 + 1; l < std::min(G, g0 + group); l++) {
                    auto& ln = lanes[l];
                    if (s >= ln.size() || !(ln[s].flags & OPF_VALID)) continue;
                    // the unit that contains step s ends at the next LAST flag
                    size_t last = s;
                    while (!(ln[last].flags & OPF_LAST)) last++;
                    auto cost = [&](const ProgOp& o) {
                        int c = 0;
                        for (int j = g0; j < l; j++) {
                            if (s >= lanes[j].size() || !(lanes[j][s].flags & OPF_VALID)) continue;
                            const ProgOp& r = lanes[j][s];
                            if (o.offA != r.offA && o.offA % M == r.offA % M) c += 10;
                            if (o.offB != r.offB && o.offB % M == r.offB % M) c += 10;
                            if (o.offP1 != r.offP1 && o.offP1 % M == r.offP1 % M) c += 2;
                            if (kind(o) != kind(r)) c += 1;
                        }
                        return c;
                    };
                    size_t best = s;
                    int best_cost = cost(ln[s]);
                    for (size_t c = s + 1; c <= last && best_cost > 0; c++) {
                        const int cc = cost(ln[c]);
                        if (cc < best_cost) { best_cost = cc; best = c; }
                    }
                    if (best != s) swap_operands(ln[s], ln[best]);
                }
    };

    auto emit_level = [&](int lvl, std::vector<std::vector<ProgOp>>& lanes) {
        size_t steps = 0;
        for (auto& l : lanes) steps = std::max(steps, l.size());
        out.level_steps[lvl] = (uint16_t)steps;
        ProgOp nop;
        std::memset(&nop, 0, sizeof(nop));
        for (size_t s = 0; s < steps; s++)
            for (int l = 0; l < G; l++) {
                ProgOp o = s < lanes[l].size() ? lanes[l][s] : nop;
                if (s + 1 == steps) o.flags |= OPF_SYNC;   // every lane's op of a level's last step carries the barrier
                out.ops.push_back(o);
            }
        out.total_steps += (int)steps;
        if (steps) out.n_sync++;
    };

    {   // level 0: external currents and momenta
        std::vector<std::vector<ProgOp>> lanes(G);
        for (int k = 0; k < n; k++) {
            ProgOp o;
            std::memset(&o, 0, sizeof(o));
            o.flags = OPF_EXT | (dense ? OPF_EXTD : 0);
            o.extra = (uint32_t)k;
            if (k < m) {
                const int pi = 1 << k;
                o.offDst = (uint16_t)off[pi * SL + (dense ? 0 : slot_of(ci[k], cj[k]))];
                o.offPt = (uint16_t)poff[pi];
            } else {
                o.offDst = (uint16_t)off_epsn;
                o.offPt = 0xFFFF;
            }
            lanes[k % G].push_back(o);
        }
        emit_level(0, lanes);
    }

    auto make_op = [&](const Target& t, const VOp& v) {
        ProgOp o;
        std::memset(&o, 0, sizeof(o));
        o.offA = (uint16_t)off[v.pa * SL + v.sa];
        o.offB = (uint16_t)off[v.pb * SL + v.sb];
        o.offP1 = (uint16_t)poff[v.pa];
        o.extra = (uint32_t)poff[v.pb];
        o.offPt = t.store_p ? (uint16_t)poff[t.pi] : (uint16_t)0xFFFF;
        o.offDst = t.pi == full ? (uint16_t)(off_epsn + (dense ? 4 * (t.g * 3 + t.h) : 0))
                                : (t.fused ? (uint16_t)0xFFFF : (uint16_t)off[t.pi * SL + t.slot()]);
        o.flags = OPF_VALID | (v.neg ? OPF_NEG : 0) | (popc(v.pa) >= 2 ? OPF_TENA : 0) |
                  (popc(v.pb) >= 2 ? OPF_TENB : 0) | (t.pi == full ? OPF_CLOSURE : 0);
        return o;
    };
    auto push_fuses = [&](std::vector<ProgOp>& lane, const Target& t) {
        for (auto& fz : t.fuses) {
            ProgOp o;
            std::memset(&o, 0, sizeof(o));
            o.offA = (uint16_t)off[fz.first.pa * SL + fz.first.sa];
            o.offP1 = (uint16_t)poff[fz.first.pa];
            o.offDst = (uint16_t)(off_epsn + 4 * fz.second);
            o.flags = OPF_FUSED | (fz.first.neg ? OPF_NEG : 0);
            lane.push_back(o);
            out.n_vertex_ops++;
        }
    };
    auto push_target = [&](std::vector<ProgOp>& lane, const Target& t) {
        for (size_t i = 0; i < t.ops.size(); i++) {
            ProgOp o = make_op(t, t.ops[i]);
            if (i == 0) o.flags |= OPF_FIRST;
            if (i + 1 == t.ops.size())
                o.flags |= OPF_LAST | (t.store_p ? OPF_STOREP : 0) | (t.fused ? OPF_NOSTORE : 0);
            lane.push_back(o);
            out.n_vertex_ops++;
        }
        push_fuses(lane, t);
    };

    // A unit of work is a run of vertices of one target that one lane accumulates in its registers: the whole
    // target, or - when a level has fewer big targets than lanes - a chunk of it, whose raw partial sums go to
    // a scratch slot and are added up by one lane in a "combine" sub-level after a barrier.
    struct Unit { int target, first, count, part; };   // part: -1 = whole target, else index of the scratch slot
    const int scratch_base = next;
    int scratch_max = 0;
    for (int pc = 2; pc <= m; pc++) {
        std::vector<std::vector<ProgOp>> lanes(G), clanes(G);
        auto& tg = levels[pc];
        if (pc == m) {
            // closure: every lane contracts the partial sum of its run with the closure vector of that target
            // (eps_n, or eps_n X_n[g][h]) and the lanes' amplitudes are added at the end, so the closure targets can
            // be cut into runs of any length without scratch
            long long total = 0;
            for (auto& t : tg) total += (long long)t.ops.size();
            const int chunk = std::max<int>(1, (int)((total + G - 1) / G));
            std::vector<int> load(G, 0);
            for (auto& t : tg)
                for (size_t lo = 0; lo < t.ops.size(); lo += chunk) {
                    const size_t hi = std::min(t.ops.size(), lo + chunk);
                    const int l = (int)(std::min_element(load.begin(), load.end()) - load.begin());
                    load[l] += (int)(hi - lo);
                    for (size_t i = lo; i < hi; i++) {
                        ProgOp o = make_op(t, t.ops[i]);
                        if (i == lo) o.flags |= OPF_FIRST;
                        if (i + 1 == hi) o.flags |= OPF_LAST;
                        lanes[l].push_back(o);
                        out.n_vertex_ops++;
                    }
                }
            reduce_bank_conflicts(lanes);
            emit_level(2 * (pc - 2) + 1, lanes);
            break;
        }
        long long total = 0;
        for (auto& t : tg) total += (long long)t.ops.size() + (long long)t.fuses.size();
        const int ideal = (int)((total + G - 1) / G);
        auto ucost = [&](const Unit& u) { return u.count + (u.part < 0 ? (int)tg[u.target].fuses.size() : 0); };
        // Units no larger than chunk_max vertices; the number of steps the level then needs (longest-processing-
        // time rule).  A chunk size equal to the ideal step count often leaves slightly more units than lanes and costs a
        // second round, so slightly larger sizes are tried and the one with the fewest steps (then chunks) is kept.
        std::vector<Unit> units;
        std::vector<int> nparts, part0;
        int nscratch = 0;
        auto plan = [&](int chunk_max) {
            units.clear();
            nparts.assign(tg.size(), 0);
            part0.assign(tg.size(), -1);
            nscratch = 0;
            for (size_t i = 0; i < tg.size(); i++) {
                const int c = (int)tg[i].ops.size();
                if (G == 1 || c + (int)tg[i].fuses.size() <= chunk_max || c < 4) {
                    units.push_back({(int)i, 0, c, -1});
                    continue;
                }
                const int r = (c + chunk_max - 1) / chunk_max;
                nparts[i] = r;
                part0[i] = nscratch;
                for (int k = 0; k < r; k++) {
                    const int lo = (int)((long long)c * k / r), hi = (int)((long long)c * (k + 1) / r);
                    units.push_back({(int)i, lo, hi - lo, nscratch++});
                }
            }
            std::stable_sort(units.begin(), units.end(), [&](const Unit& a, const Unit& b) { return ucost(a) > ucost(b); });
            std::vector<int> ld(G, 0);
            for (auto& u : units) *std::min_element(ld.begin(), ld.end()) += ucost(u);
            return *std::max_element(ld.begin(), ld.end());
        };
        {
            int best_chunk = std::max(ideal, 2), best_steps = -1, best_scratch = 0;
            for (int extra = 0; extra <= 3; extra++) {
                const int chunk = std::max(ideal, 2) + extra;
                const int steps = plan(chunk);
                if (best_steps < 0 || steps < best_steps || (steps == best_steps && nscratch < best_scratch)) {
                    best_steps = steps; best_chunk = chunk; best_scratch = nscratch;
                }
                if (G == 1 || steps <= ideal) break;
            }
            plan(best_chunk);
        }
        scratch_max = std::max(scratch_max, nscratch * 10);
        std::vector<int> load(G, 0);
        for (auto& u : units) {
            const int l = (int)(std::min_element(load.begin(), load.end()) - load.begin());
            load[l] += ucost(u);
            const Target& t = tg[u.target];
            if (u.part < 0) {
                push_target(lanes[l], t);
                continue;
            }
            for (int i = u.first; i < u.first + u.count; i++) {
                ProgOp o = make_op(t, t.ops[i]);
                if (i == u.first) o.flags |= OPF_FIRST;
                if (i + 1 == u.first + u.count) {
                    o.flags |= OPF_LAST | OPF_PARTIAL;
                    o.offDst = (uint16_t)(scratch_base + 10 * u.part);
                }
                lanes[l].push_back(o);
                out.n_vertex_ops++;
            }
        }
        // combine sub-level: one lane per split target
        int cl = 0;
        for (size_t i = 0; i < tg.size(); i++) {
            if (!nparts[i]) continue;
            const Target& t = tg[i];
            ProgOp o = make_op(t, t.ops[0]);   // offP1 / extra give P(pi) = P(pi_1) + P(pi_2); offDst, offPt as usual
            o.offA = (uint16_t)(scratch_base + 10 * part0[i]);
            o.offB = (uint16_t)nparts[i];
            o.flags = OPF_COMBINE | (t.store_p ? OPF_STOREP : 0) | (t.fused ? OPF_NOSTORE : 0);
            auto& lane = clanes[cl++ % G];
            lane.push_back(o);
            push_fuses(lane, t);
        }
        reduce_bank_conflicts(lanes);
        emit_level(2 * (pc - 2) + 1, lanes);
        emit_level(2 * (pc - 2) + 2, clanes);
    }
    out.state_cx = next + scratch_max;
}

void build_class(int n, int G, const int* counts, ClassProgram& out, int closure) {
    out = ClassProgram();
    // the colour charges must cancel over all n gluons (as many i = c as j = c for every colour c)
    for (int c = 0; c < 3; c++) {
        int ni = 0, nj = 0;
        for (int t = 0; t < kNumCodes; t++) {
            if (t / 3 == c) ni += counts[t];
            if (t % 3 == c) nj += counts[t];
        }
        if (ni != nj) return;
    }
    // every gluon can serve as the closure leg; the cheapest program among a few choices is kept
    const int max_trials = n <= 8 ? kNumCodes : (n == 9 ? 4 : 2);
    int trials = 0;
    bool have = false;
    for (int c = 0; c < kNumCodes && trials < max_trials; c++) {
        if (!counts[c] || (closure >= 0 && c != closure)) continue;
        trials++;
        int code[kMaxN], k = 0;
        for (int t = 0; t < kNumCodes; t++)
            for (int r = 0; r < counts[t] - (t == c ? 1 : 0); r++) code[k++] = t;
        code[k++] = c;
        ClassProgram p;
        build_program(n, G, code, p);
        if (!p.valid) continue;   // validity does not depend on the closure leg, but be safe
        if (!have || p.total_steps < out.total_steps ||
            (p.total_steps == out.total_steps && p.state_cx < out.state_cx)) {
            out = std::move(p);
            have = true;
        }
    }
}

}  // namespace bg

// ---------------------------------------------------------------------------------------------------------
// CO_MC: the colour-flow decomposition Eq. 19 evaluated with colour-ORDERED
// currents.  For canonical colour codes the orderings (1, sigma_2 .. sigma_n) whose colour chain closes (the j of each
// gluon is the i of the next, cyclically) are enumerated by depth-first search; the amplitude is the sum of the
// colour-ordered amplitudes A(1, sigma) of those orderings.  Each A is the recursion Eq. 24-25 (tensor form) over
// contiguous sub-sequences; sub-sequences shared by several orderings are computed once.  The vertex
// X(J(i..k), J(k+1..j)) is the same operation the colour-dressed programs use, so the same interpreter runs it.
// ---------------------------------------------------------------------------------------------------------
namespace bg {

namespace {
struct SeqNode {
    std::vector<int> seq;   // canonical gluon indices
    unsigned mask = 0;
    int off = -1;           // state offset of its current (4 + 6 cx); -1: external or fused
    bool closure = false;   // first n-1 gluons of an ordering: contracted with eps of the last one
    int last = -1;          // closure: the gluon that closes
    std::vector<std::pair<int, int>> fuses;   // (closure node id, split position) read straight from registers
};
}  // namespace

void build_comc_program(int n, int G, const int* code, ClassProgram& out, long long max_orderings) {
    out = ClassProgram();
    int ci[kMaxN], cj[kMaxN];
    for (int k = 0; k < n; k++) { ci[k] = code[k] / 3; cj[k] = code[k] % 3; }
    out.closure_code = code[n - 1];
    // colour-connected orderings starting with gluon 0 (depth-first; j of the last must be i of gluon 0)
    std::vector<std::vector<int>> orderings;
    {
        std::vector<int> cur{0};
        unsigned used = 1;
        bool overflow = false;
        auto dfs = [&](auto&& self) -> void {
            if (overflow) return;
            if ((int)cur.size() == n) {
                if (cj[cur.back()] == ci[0]) {
                    orderings.push_back(cur);
                    if ((long long)orderings.size() > max_orderings) overflow = true;
                }
                return;
            }
            for (int g = 1; g < n; g++) {
                if ((used >> g) & 1u) continue;
                if (cj[cur.back()] != ci[g]) continue;
                used |= 1u << g;
                cur.push_back(g);
                self(self);
                cur.pop_back();
                used &= ~(1u << g);
            }
        };
        dfs(dfs);
        if (overflow) { out.state_cx = -1; return; }   // too many orderings for a tabulated program: unsupported
    }
    if (orderings.empty()) return;
    out.valid = true;
    out.n_orderings = (long long)orderings.size();

    // nodes: single gluons 0..n-1, then every distinct contiguous sub-sequence (length >= 2) of the first n-1
    // elements of the orderings
    std::vector<SeqNode> nodes(n);
    std::map<std::vector<int>, int> id_of;
    for (int g = 0; g < n; g++) { nodes[g].seq = {g}; nodes[g].mask = 1u << g; id_of[nodes[g].seq] = g; }
    const int m = n - 1;
    std::vector<std::vector<int>> by_len(m + 1);
    for (auto& o : orderings)
        for (int L = 2; L <= m; L++)
            for (int i = 0; i + L <= m; i++) {
                std::vector<int> s(o.begin() + i, o.begin() + i + L);
                if (id_of.count(s)) continue;
                SeqNode nd;
                nd.seq = s;
                for (int g : s) nd.mask |= 1u << g;
                id_of[s] = (int)nodes.size();
                by_len[L].push_back((int)nodes.size());
                nodes.push_back(std::move(nd));
            }
    for (auto& o : orderings) {
        SeqNode& c = nodes[id_of[std::vector<int>(o.begin(), o.begin() + m)]];
        c.closure = true;
        c.last = o[m];
    }
    auto sub = [&](const SeqNode& nd, int i, int j) { return id_of[std::vector<int>(nd.seq.begin() + i, nd.seq.begin() + j)]; };
    auto len = [&](int id) { return (int)nodes[id].seq.size(); };

    // layout: externals + momenta, then stored currents (length 2 .. n-3) and one momentum per distinct gluon set
    int next = 0;
    std::vector<int> ext_off(n), ext_poff(n);
    for (int g = 0; g < n; g++) { ext_off[g] = next; nodes[g].off = next; next += 4; }
    std::map<unsigned, int> poff;
    for (int g = 0; g < n; g++) { poff[1u << g] = next; ext_poff[g] = next; next += 2; }
    const int pad = G >= 8 ? 1 : 0;
    // length n-2 sequences are read by closure vertices only: fused, never stored
    for (int L = 2; L <= m; L++)
        for (int id : by_len[L]) {
            if (L <= m - 2 || (L == m - 1 && m - 1 < 2)) { nodes[id].off = next; next += 10 + pad; }
            if (L <= m - 1 && !poff.count(nodes[id].mask)) { poff[nodes[id].mask] = -1; }
        }
    // which momenta are read: P(a) of every vertex and P(b) of first vertices; simply give every set of length <= n-2
    // that occurs a slot, written by the first node (in emission order) with that set
    std::map<unsigned, int> p_writer;
    for (int L = 2; L <= m - 1; L++)
        for (int id : by_len[L])
            if (poff[nodes[id].mask] < 0) { poff[nodes[id].mask] = next; next += 2; p_writer[nodes[id].mask] = id; }
    // closure targets need P(a), P(b) of their vertices only (both of length <= n-2): nothing to store for them

    // fuse: closure vertices whose larger operand has length n-2
    if (m - 1 >= 2)
        for (int L = m; L <= m; L++)
            for (int id : by_len[L]) {
                if (!nodes[id].closure) continue;
                nodes[sub(nodes[id], 1, m)].fuses.push_back({id, 1});        // X(gluon seq[0], seq[1..m-1])
                nodes[sub(nodes[id], 0, m - 1)].fuses.push_back({id, m - 1});  // X(seq[0..m-2], gluon seq[m-1])
            }

    out.level_steps.assign(2 * m - 2, 0);
    auto emit_level = [&](int lvl, std::vector<std::vector<ProgOp>>& lanes) {
        size_t steps = 0;
        for (auto& l : lanes) steps = std::max(steps, l.size());
        out.level_steps[lvl] = (uint16_t)steps;
        ProgOp nop;
        std::memset(&nop, 0, sizeof(nop));
        for (size_t s = 0; s < steps; s++)
            for (int l = 0; l < G; l++) {
                ProgOp o = s < lanes[l].size() ? lanes[l][s] : nop;
                if (s + 1 == steps) o.flags |= OPF_SYNC;
                out.ops.push_back(o);
            }
        out.total_steps += (int)steps;
        if (steps) out.n_sync++;
    };
    {   // level 0: all n external currents and momenta
        std::vector<std::vector<ProgOp>> lanes(G);
        for (int g = 0; g < n; g++) {
            ProgOp o;
            std::memset(&o, 0, sizeof(o));
            o.flags = OPF_EXT;
            o.extra = (uint32_t)g;
            o.offDst = (uint16_t)ext_off[g];
            o.offPt = (uint16_t)ext_poff[g];
            lanes[g % G].push_back(o);
        }
        emit_level(0, lanes);
    }
    // vertex X(seq[0..k), seq[k..L)) of node `id`; the shorter operand goes first (X is antisymmetric)
    auto make_vertex = [&](int id, int k, bool closure_target) {
        const SeqNode& nd = nodes[id];
        const int L = (int)nd.seq.size();
        int a = sub(nd, 0, k), b = sub(nd, k, L);
        bool neg = false;
        if (len(a) > len(b)) { std::swap(a, b); neg = true; }
        ProgOp o;
        std::memset(&o, 0, sizeof(o));
        o.offA = (uint16_t)nodes[a].off;
        o.offB = (uint16_t)nodes[b].off;
        o.offP1 = (uint16_t)poff[nodes[a].mask];
        o.extra = (uint32_t)poff[nodes[b].mask];
        o.offPt = 0xFFFF;
        o.flags = OPF_VALID | (neg ? OPF_NEG : 0) | (len(a) >= 2 ? OPF_TENA : 0) | (len(b) >= 2 ? OPF_TENB : 0) |
                  (closure_target ? OPF_CLOSURE : 0);
        return o;
    };
    for (int L = 2; L <= m; L++) {
        std::vector<std::vector<ProgOp>> lanes(G), clanes(G);
        std::vector<int> load(G, 0);
        auto least = [&]() { return (int)(std::min_element(load.begin(), load.end()) - load.begin()); };
        if (L == m) {
            // closure targets: the vertices not fused (2 <= k <= m-2), one run per ordering
            for (int id : by_len[L]) {
                if (!nodes[id].closure) continue;
                std::vector<ProgOp> run;
                for (int k = (m - 1 >= 2 ? 2 : 1); k <= (m - 1 >= 2 ? m - 2 : m - 1); k++) {
                    ProgOp o = make_vertex(id, k, true);
                    o.offDst = (uint16_t)ext_off[nodes[id].last];
                    run.push_back(o);
                }
                if (run.empty()) continue;
                run.front().flags |= OPF_FIRST;
                run.back().flags |= OPF_LAST;
                const int l = least();
                load[l] += (int)run.size();
                lanes[l].insert(lanes[l].end(), run.begin(), run.end());
                out.n_vertex_ops += (int)run.size();
            }
            emit_level(2 * (L - 2) + 1, lanes);
            break;
        }
        std::vector<int> order = by_len[L];
        auto cost = [&](int id) { return L - 1 + (int)nodes[id].fuses.size(); };
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost(a) > cost(b); });
        for (int id : order) {
            const int l = least();
            load[l] += cost(id);
            const bool writes_p = p_writer.count(nodes[id].mask) && p_writer[nodes[id].mask] == id;
            for (int k = 1; k < L; k++) {
                ProgOp o = make_vertex(id, k, false);
                o.offDst = nodes[id].off >= 0 ? (uint16_t)nodes[id].off : (uint16_t)0xFFFF;
                if (k == 1) o.flags |= OPF_FIRST;
                if (k == L - 1) {
                    o.flags |= OPF_LAST | (nodes[id].off < 0 ? OPF_NOSTORE : 0) | (writes_p ? OPF_STOREP : 0);
                    if (writes_p) o.offPt = (uint16_t)poff[nodes[id].mask];
                }
                lanes[l].push_back(o);
                out.n_vertex_ops++;
            }
            for (auto& fz : nodes[id].fuses) {
                // closure vertex of ordering fz.first: X(single gluon, this sequence), sign by which side the gluon is on
                const SeqNode& c = nodes[fz.first];
                const int single = fz.second == 1 ? c.seq[0] : c.seq[m - 1];
                ProgOp o;
                std::memset(&o, 0, sizeof(o));
                o.offA = (uint16_t)ext_off[single];
                o.offP1 = (uint16_t)ext_poff[single];
                o.offDst = (uint16_t)ext_off[c.last];
                // X(prefix, suffix): gluon first (k = 1) is X(single, this); gluon last is X(this, single) = -X(single, this)
                o.flags = OPF_FUSED | (fz.second == 1 ? 0 : OPF_NEG);
                lanes[l].push_back(o);
                out.n_vertex_ops++;
            }
        }
        emit_level(2 * (L - 2) + 1, lanes);
        emit_level(2 * (L - 2) + 2, clanes);
    }
    out.state_cx = next;
}

}  // namespace bg

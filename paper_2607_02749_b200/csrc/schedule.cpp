// schedule.cpp -- host-side schedule compiler (see schedule.h, program.h).
//
// Two levels of the same greedy "take what commutes forward" pass:
//   block level: choose tile bits T; an op can run in this block if every qubit it acts on NON-diagonally
//                (RY qubit, CNOT target) is in T and it commutes with every earlier op that was left behind.
//   stage level: inside a block choose register bits Rset (subset of T); non-diagonal ops need their qubit in
//                Rset; diagonal ops (RZ, CZ) are collected and flushed as one merged diagonal segment.
// Commutation rule used: two ops commute if on every qubit they share BOTH act diagonally (RZ, CZ and the
// control side of a CNOT are diagonal in the computational basis).  So a skipped op marks the qubits it touches
// diagonally as "no later non-diagonal op" (nd) and the qubits it touches non-diagonally as fully blocked.
#include "schedule.h"

#include <algorithm>
#include <cstdio>
#include <cstring>

namespace gv {
namespace {

struct Acts { int nq; int q[2]; bool diag[2]; };

inline Acts acts_of(const HostOp &o)
{
    Acts a{};
    switch (o.kind) {
    case 0: a.nq = 1; a.q[0] = o.q0; a.diag[0] = false; break;                                   // RY
    case 1: a.nq = 1; a.q[0] = o.q0; a.diag[0] = true; break;                                    // RZ
    case 2: a.nq = 2; a.q[0] = o.q0; a.q[1] = o.q1; a.diag[0] = a.diag[1] = true; break;          // CZ
    default: a.nq = 2; a.q[0] = o.q0; a.diag[0] = false; a.q[1] = o.q1; a.diag[1] = true; break;  // CNOT
    }
    return a;
}
inline bool is_diag(const HostOp &o) { return o.kind == 1 || o.kind == 2; }

// ---- block level -------------------------------------------------------------------------------------------
struct BlockTake { std::vector<int> taken; int n_nondiag = 0; };

void block_take(const std::vector<HostOp> &ops, const std::vector<int> &pending, uint64_t T, int n, BlockTake &out)
{
    out.taken.clear();
    out.n_nondiag = 0;
    uint64_t full = 0, nd = 0;
    const uint64_t all = (n >= 64) ? ~0ull : ((1ull << n) - 1);
    for (int idx : pending) {
        const HostOp &o = ops[idx];
        const Acts a = acts_of(o);
        bool ok = true;
        for (int i = 0; i < a.nq; ++i) {
            const uint64_t b = 1ull << a.q[i];
            if (full & b) ok = false;
            if (!a.diag[i] && ((nd & b) || !(T & b))) ok = false;
        }
        if (ok) {
            out.taken.push_back(idx);
            if (!is_diag(o)) ++out.n_nondiag;
        } else {
            for (int i = 0; i < a.nq; ++i) {
                const uint64_t b = 1ull << a.q[i];
                if (a.diag[i]) nd |= b; else full |= b;
            }
            if ((full & all) == all) break;
        }
    }
}

int count_runs(uint64_t T)
{
    int runs = 0;
    while (T) {
        const int lo = __builtin_ctzll(T);
        uint64_t t = T >> lo;
        int len = 0;
        while (t & 1) { t >>= 1; ++len; }
        ++runs;
        T &= ~(((len >= 64) ? ~0ull : ((1ull << len) - 1)) << lo);
    }
    return runs;
}

// candidate tile-bit sets: [0,f) + every contiguous window of k-f qubits + "first needed" set
void block_candidates(const std::vector<HostOp> &ops, const std::vector<int> &pending, int n, int k, int f,
                      std::vector<uint64_t> &cand, bool two_windows = false)
{
    cand.clear();
    if (n <= k) { cand.push_back((1ull << n) - 1); return; }
    const uint64_t low = (1ull << f) - 1;
    const int h = k - f;
    for (int a = f; a + h <= n; ++a) cand.push_back(low | (((1ull << h) - 1) << a));
    // first-needed: non-diagonal qubits >= f in pending order
    uint64_t T = low;
    int cnt = 0;
    for (int idx : pending) {
        const Acts a = acts_of(ops[idx]);
        for (int i = 0; i < a.nq && cnt < h; ++i)
            if (!a.diag[i] && a.q[i] >= f && !(T >> a.q[i] & 1)) { T |= 1ull << a.q[i]; ++cnt; }
        if (cnt >= h) break;
    }
    // pad next to already chosen bits (keeps the number of runs small), then anywhere
    for (int pass = 0; pass < 2 && cnt < h; ++pass)
        for (int q = f; q < n && cnt < h; ++q) {
            if (T >> q & 1) continue;
            const bool adj = (q > 0 && (T >> (q - 1) & 1)) || (q + 1 < n && (T >> (q + 1) & 1));
            if (pass == 1 || adj) { T |= 1ull << q; ++cnt; }
        }
    if (count_runs(T) <= MAX_RUNS && std::find(cand.begin(), cand.end(), T) == cand.end()) cand.push_back(T);
    if (!two_windows) return;
    // two windows (h1 + h2 = h qubits): two fronts of a layered circuit advance in one block
    for (int h1 = 2; h1 <= h - 2; ++h1) {
        const int h2 = h - h1;
        for (int a = f; a + h1 <= n; ++a)
            for (int b = a + h1 + 1; b + h2 <= n; ++b) {
                const uint64_t W = low | (((1ull << h1) - 1) << a) | (((1ull << h2) - 1) << b);
                if (std::find(cand.begin(), cand.end(), W) == cand.end()) cand.push_back(W);
            }
    }
}

}  // namespace
}  // namespace gv

// ---- stage level -------------------------------------------------------------------------------------------
namespace gv {
namespace {

constexpr int MAX_SEG_OPS = 96;    // RZ + CZ entries merged into one diagonal segment
constexpr int MAX_STAGE_ND = 64;   // RY/CNOT micro-ops per stage
constexpr int MAX_STAGE_SEG = 12;  // diagonal segments per stage

struct StageItem { bool is_seg; int op; std::vector<int> seg_ops; bool mid_cx = false; };  // op / seg_ops index the block's op list; mid_cx: a CNOT applied in registers

struct StageTake {
    std::vector<StageItem> items;
    std::vector<int> carry;      // diagonal ops taken but not yet flushed
    std::vector<int> rest;       // ops left for later stages (block-list positions)
    int n_nondiag = 0, n_seg = 0;
    bool has_cx = false;         // the stage ends with a CNOT run (nothing but CNOTs may follow the first one)
};

// bops: the block's ops in execution order; L: positions (into bops) still to run; carry: pending diagonals.
// Rset: register qubits (global ids).  flush_anywhere: allow a diagonal flush after a non-diagonal op of this stage.
// mid_cx: a CNOT whose target is a register qubit is applied in registers where it stands (its control may be anywhere)
// and rotations may follow it; without it a CNOT always starts the stage's trailing run.
void stage_take(const std::vector<HostOp> &bops, const std::vector<int> &L, const std::vector<int> &carry_in,
                uint64_t Rset, bool flush_anywhere, bool mid_cx, StageTake &out)
{
    out.items.clear(); out.rest.clear(); out.n_nondiag = 0; out.n_seg = 0; out.has_cx = false;
    std::vector<int> pend = carry_in;
    uint64_t pend_touch = 0;
    for (int p : pend) { const Acts a = acts_of(bops[p]); for (int i = 0; i < a.nq; ++i) pend_touch |= 1ull << a.q[i]; }
    uint64_t full = 0, nd = 0, cx_touch = 0;
    for (int pos : L) {
        const HostOp &o = bops[pos];
        const Acts a = acts_of(o);
        bool ok = true;
        uint64_t ndq = 0;
        for (int i = 0; i < a.nq; ++i) {
            const uint64_t b = 1ull << a.q[i];
            if (full & b) ok = false;
            // RY needs its qubit in a register slot; a CNOT target only has to be a tile bit (block level)
            if (!a.diag[i]) { ndq |= b; if ((nd & b) || (o.kind == 0 && !(Rset & b))) ok = false; }
        }
        if (ok && !is_diag(o) && (pend_touch & ndq) && !flush_anywhere && out.n_nondiag > 0) ok = false;
        // after the CNOT run began, a rotation is taken only if it commutes with the whole run (its qubit is neither a
        // target nor a control of it) and needs no diagonal flush: it then executes before the run
        if (ok && o.kind == 0 && out.has_cx && ((cx_touch | pend_touch) & ndq)) ok = false;
        if (ok && o.kind == 3 && out.has_cx && (pend_touch & ndq)) ok = false;    // no diagonal flush inside the run
        // size caps (shared-memory slice of the program): an op that does not fit waits for the next stage
        if (ok && is_diag(o) && (int)pend.size() >= MAX_SEG_OPS) ok = false;
        if (ok && !is_diag(o) && out.n_nondiag >= MAX_STAGE_ND) ok = false;
        if (ok && !is_diag(o) && (pend_touch & ndq) && out.n_seg >= MAX_STAGE_SEG) ok = false;
        if (ok) {
            if (is_diag(o)) {
                pend.push_back(pos);
                for (int i = 0; i < a.nq; ++i) pend_touch |= 1ull << a.q[i];
            } else {
                if (pend_touch & ndq) {  // a pending diagonal touches a qubit this op changes: flush first
                    StageItem s; s.is_seg = true; s.op = -1; s.seg_ops.swap(pend);
                    out.items.push_back(std::move(s)); ++out.n_seg;
                    pend.clear(); pend_touch = 0;
                }
                StageItem it; it.is_seg = false; it.op = pos;
                it.mid_cx = o.kind == 3 && mid_cx && !out.has_cx && (Rset >> o.q0 & 1);
                if (o.kind == 3 && !it.mid_cx) { out.has_cx = true; cx_touch |= (1ull << o.q0) | (1ull << o.q1); }
                out.items.push_back(std::move(it)); ++out.n_nondiag;
            }
        } else {
            out.rest.push_back(pos);
            for (int i = 0; i < a.nq; ++i) {
                const uint64_t b = 1ull << a.q[i];
                if (a.diag[i]) nd |= b; else full |= b;
            }
        }
    }
    out.carry.swap(pend);
}

}  // namespace
}  // namespace gv

// ---- driver --------------------------------------------------------------------------------------------------
namespace gv {
namespace {

// local bit position of global qubit q inside tile-bit set T
inline int local_pos(uint64_t T, int q) { return __builtin_popcountll(T & ((1ull << q) - 1)); }

void stage_candidates(const std::vector<HostOp> &bops, const std::vector<int> &L, uint64_t T, int k, int R, bool mid_cx,
                      std::vector<uint64_t> &cand)
{
    cand.clear();
    std::vector<int> tq;  // local -> global
    for (int q = 0; q < 64; ++q) if (T >> q & 1) tq.push_back(q);
    for (int p = 0; p + R <= k; ++p) {
        uint64_t s = 0;
        for (int j = 0; j < R; ++j) s |= 1ull << tq[p + j];
        cand.push_back(s);
    }
    uint64_t s = 0; int cnt = 0;
    for (int pos : L) {
        const Acts a = acts_of(bops[pos]);
        for (int i = 0; i < a.nq && cnt < R; ++i)
            if (!a.diag[i] && bops[pos].kind == 0 && !(s >> a.q[i] & 1)) { s |= 1ull << a.q[i]; ++cnt; }
        if (cnt >= R) break;
    }
    for (int p = 0; p < k && cnt < R; ++p) if (!(s >> tq[p] & 1)) { s |= 1ull << tq[p]; ++cnt; }
    if (std::find(cand.begin(), cand.end(), s) == cand.end()) cand.push_back(s);
    if (!mid_cx) return;
    // with CNOTs in registers their targets count as needed qubits too: the first R of them, and the same skipping the
    // first one, two, ... (a stage that starts further down the dependency chain)
    std::vector<int> order;
    uint64_t seen = 0;
    for (int pos : L) {
        const HostOp &o = bops[pos];
        if ((o.kind == 0 || o.kind == 3) && (T >> o.q0 & 1) && !(seen >> o.q0 & 1)) { seen |= 1ull << o.q0; order.push_back(o.q0); }
    }
    for (size_t p = 0; p < order.size() && p < 8; ++p) {
        uint64_t w = 0; int c = 0;
        for (size_t j = p; j < order.size() && c < R; ++j) { w |= 1ull << order[j]; ++c; }
        for (size_t j = 0; j < p && c < R; ++j) { w |= 1ull << order[j]; ++c; }
        for (int q = 0; q < k && c < R; ++q) if (!(w >> tq[q] & 1)) { w |= 1ull << tq[q]; ++c; }
        if (std::find(cand.begin(), cand.end(), w) == cand.end()) cand.push_back(w);
    }
}

// bank-conflict proxy for the swizzle phys = j ^ ((j >> 4) & 15): lanes vary the lowest 4 non-register local bits;
// a pair (b, b+4) with both bits lane-varying collides.
int conflict_penalty(uint64_t T, uint64_t Rset, int k)
{
    int lane_bits[4], nl = 0;
    for (int p = 0; p < k && nl < 4; ++p) {
        int q = -1, c = 0;
        for (int g = 0; g < 64; ++g) if (T >> g & 1) { if (c == p) { q = g; break; } ++c; }
        if (!(Rset >> q & 1)) lane_bits[nl++] = p;
    }
    int pen = 0;
    for (int i = 0; i < nl; ++i) for (int j = 0; j < nl; ++j)
        if (lane_bits[i] < 4 && lane_bits[j] == lane_bits[i] + 4) ++pen;
    return pen;
}

}  // namespace

Prefix find_prefix(int n, const std::vector<HostOp> &ops)
{
    Prefix px;
    size_t i = 0;
    std::vector<std::vector<std::pair<uint8_t, int32_t>>> rot((size_t)n);
    while (i < ops.size() && ops[i].kind <= 1) { rot[ops[i].q0].push_back({(uint8_t)ops[i].kind, ops[i].param}); ++i; }
    if (i == 0) return px;
    size_t j = i;
    const int ekind = j < ops.size() ? ops[j].kind : -1;
    std::vector<std::pair<int, uint64_t>> dist;   // CZ pairs grouped by distance
    while (j < ops.size() && ops[j].kind >= 2 && ops[j].kind == ekind) {
        if (ekind == 3) { px.cx_t.push_back((uint8_t)ops[j].q0); px.cx_c.push_back((uint8_t)ops[j].q1); }
        else {
            const int lo = ops[j].q0 < ops[j].q1 ? ops[j].q0 : ops[j].q1, d = ops[j].q0 + ops[j].q1 - 2 * lo;
            size_t e = 0;
            while (e < dist.size() && dist[e].first != d) ++e;
            if (e == dist.size()) { if (dist.size() == 4) break; dist.push_back({d, 0}); }
            dist[e].second ^= 1ull << lo;   // a repeated pair cancels
        }
        ++j;
    }
    px.n_ops = (int)j;
    px.n_cz = (int)dist.size();
    for (size_t e = 0; e < dist.size(); ++e) { px.cz_d[e] = dist[e].first; px.cz_m[e] = dist[e].second; }
    px.rot_begin.assign((size_t)n + 1, 0);
    for (int q = 0; q < n; ++q) {
        px.rot_begin[q] = (int32_t)px.rot_kind.size();
        for (auto &r : rot[q]) { px.rot_kind.push_back(r.first); px.rot_param.push_back(r.second); }
    }
    px.rot_begin[n] = (int32_t)px.rot_kind.size();
    return px;
}

bool compile_program(int n, const std::vector<HostOp> &ops, int k, int f, int R, Program &P, std::string &err,
                     bool from_zero, bool mid_cx)
{
    P = Program();
    if (n < 1 || n > 40) { err = "schedule: bad qubit count"; return false; }
    if (R < 1 || R > MAX_R) { err = "schedule: bad register-bit count"; return false; }
    if (k > n) k = n;
    if (k < R) { err = "schedule: tile smaller than register block"; return false; }
    if (f > k) f = k;
    if (n > k && k - f < 1) { err = "schedule: no free tile bits"; return false; }
    P.n = n; P.k = k; P.f = f; P.R = R;
    for (const HostOp &o : ops) {
        const bool two = (o.kind == 2 || o.kind == 3);
        if (o.kind < 0 || o.kind > 3 || o.q0 < 0 || o.q0 >= n || (two && (o.q1 < 0 || o.q1 >= n || o.q1 == o.q0))) {
            err = "schedule: bad op"; return false;
        }
    }
    std::vector<int> pending(ops.size());
    for (size_t i = 0; i < ops.size(); ++i) pending[i] = (int)i;
    std::vector<uint64_t> cand;
    BlockTake bt, best;
    bool first = true;
    const bool zero_first = from_zero;
    // Every block is one read and one write of the whole state, so the number of blocks is what the tile choice
    // minimises: a beam search over sequences of tile-bit sets (the greedy sequence is always among the beams' ancestors).
    std::vector<uint64_t> plan;
    if (n > k && !ops.empty()) {
      std::vector<char> gone(ops.size());
      auto search = [&](bool two_windows) {
        std::vector<uint64_t> plan;
        struct Beam { std::vector<int> pending; std::vector<uint64_t> seq; int nd_left; };
        auto nd_count = [&](const std::vector<int> &pd) { int c = 0; for (int i : pd) if (!is_diag(ops[i])) ++c; return c; };
        const size_t WIDTH = 12;
        std::vector<Beam> beams(1);
        beams[0].pending = pending; beams[0].nd_left = nd_count(pending);
        for (int level = 0; level < 4096 && plan.empty(); ++level) {
            std::vector<Beam> next;
            for (const Beam &b : beams) {
                block_candidates(ops, b.pending, n, k, f, cand, two_windows);
                for (uint64_t T : cand) {
                    block_take(ops, b.pending, T, n, bt);
                    if (bt.taken.empty()) continue;
                    Beam nb; nb.seq = b.seq; nb.seq.push_back(T);
                    std::fill(gone.begin(), gone.end(), 0);
                    for (int idx : bt.taken) gone[idx] = 1;
                    for (int idx : b.pending) if (!gone[idx]) nb.pending.push_back(idx);
                    nb.nd_left = b.nd_left - bt.n_nondiag;
                    if (nb.pending.empty()) { plan = nb.seq; break; }
                    next.push_back(std::move(nb));
                }
                if (!plan.empty()) break;
            }
            if (!plan.empty() || next.empty()) break;
            std::stable_sort(next.begin(), next.end(), [](const Beam &x, const Beam &y) {
                return x.nd_left != y.nd_left ? x.nd_left < y.nd_left : x.pending.size() < y.pending.size(); });
            std::vector<Beam> keep;
            for (Beam &b : next) {
                bool dup = false;
                for (const Beam &q : keep) if (q.pending == b.pending) { dup = true; break; }
                if (!dup) keep.push_back(std::move(b));
                if (keep.size() >= WIDTH) break;
            }
            beams.swap(keep);
        }
        return plan;
      };
        // tile sets of one window first; two windows only when that saves a block (more runs per tile otherwise)
        plan = search(false);
        {
            const std::vector<uint64_t> plan2 = search(true);
            if (!plan2.empty() && (plan.empty() || plan2.size() < plan.size())) plan = plan2;
        }
        // the greedy sequence (most non-diagonal ops per block) is what the search has to beat
        std::vector<int> pd = pending;
        size_t greedy_len = 0;
        while (!pd.empty() && greedy_len < plan.size()) {
            block_candidates(ops, pd, n, k, f, cand);
            best.taken.clear(); best.n_nondiag = -1;
            for (uint64_t T : cand) {
                block_take(ops, pd, T, n, bt);
                if (bt.n_nondiag > best.n_nondiag || (bt.n_nondiag == best.n_nondiag && bt.taken.size() > best.taken.size())) best = bt;
            }
            if (best.taken.empty()) break;
            std::fill(gone.begin(), gone.end(), 0);
            for (int idx : best.taken) gone[idx] = 1;
            std::vector<int> np;
            for (int idx : pd) if (!gone[idx]) np.push_back(idx);
            pd.swap(np);
            ++greedy_len;
        }
        if (pd.empty() && greedy_len <= plan.size()) plan.clear();
    }
    while (!pending.empty() || first) {
        // ---- choose T
        block_candidates(ops, pending, n, k, f, cand);
        if (P.blocks.size() < plan.size()) { cand.clear(); cand.push_back(plan[P.blocks.size()]); }
        uint64_t bestT = cand[0];
        best.taken.clear(); best.n_nondiag = -1;
        for (uint64_t T : cand) {
            block_take(ops, pending, T, n, bt);
            if (bt.n_nondiag > best.n_nondiag ||
                (bt.n_nondiag == best.n_nondiag && bt.taken.size() > best.taken.size())) {
                best = bt; bestT = T;
            }
        }
        if (best.taken.empty() && !pending.empty()) { err = "schedule: no progress (internal)"; return false; }
        const uint64_t T = bestT;
        // ---- block header
        Block B; memset(&B, 0, sizeof B);
        B.k = (uint8_t)k; B.source_zero = (first && zero_first) ? 1 : 0;
        {
            int lp = 0, nr = 0;
            for (int q = 0; q < n;) {
                if (!(T >> q & 1)) { ++q; continue; }
                int len = 0; while (q + len < n && (T >> (q + len) & 1)) ++len;
                if (nr >= MAX_RUNS) { err = "schedule: too many tile runs (internal)"; return false; }
                B.runs[nr].lpos = (uint8_t)lp; B.runs[nr].gpos = (uint8_t)q; B.runs[nr].len = (uint8_t)len; ++nr;
                lp += len; q += len;
            }
            B.n_runs = (uint8_t)nr;
        }
        B.stage_begin = (uint32_t)P.stages.size();
        // ---- stages
        std::vector<HostOp> bops; bops.reserve(best.taken.size());
        for (int idx : best.taken) bops.push_back(ops[idx]);
        std::vector<int> L(bops.size()); for (size_t i = 0; i < bops.size(); ++i) L[i] = (int)i;
        std::vector<int> carry;
        std::vector<uint64_t> rc;
        StageTake st, sbest;
        uint32_t max_seg = 0;
        // Every stage is one trip of the tile through shared memory: a beam search over (register set, flush mode)
        // sequences looks for the fewest stages (ties: the greedy score summed); the greedy choice is always a candidate.
        std::vector<std::pair<uint64_t, int>> stage_plan;
        {
            struct SB { std::vector<int> L, carry; std::vector<std::pair<uint64_t, int>> seq; double score; };
            auto has_nd = [&](const std::vector<int> &v) { for (int pos : v) if (!is_diag(bops[pos])) return true; return false; };
            const size_t WIDTH = 8;
            std::vector<SB> beams(1);
            beams[0].L = L; beams[0].score = 0.0;
            bool found = false;
            std::vector<std::pair<uint64_t, int>> best_seq;
            double best_score = -1e30;
            int best_extra = 2;
            for (int depth = 0; depth < 64 && !found && has_nd(beams[0].L); ++depth) {
                std::vector<SB> next;
                for (const SB &b : beams) {
                    if (!has_nd(b.L)) continue;
                    stage_candidates(bops, b.L, T, k, R, mid_cx, rc);
                    for (uint64_t rs : rc) for (int fa = 0; fa < 2; ++fa) {
                        stage_take(bops, b.L, b.carry, rs, fa != 0, mid_cx, st);
                        if (st.n_nondiag == 0) continue;
                        SB nb2; nb2.L = st.rest; nb2.carry = st.carry; nb2.seq = b.seq; nb2.seq.push_back({rs, fa});
                        nb2.score = b.score + st.n_nondiag - 0.1 * st.n_seg - 0.01 * conflict_penalty(T, rs, k);
                        if (!has_nd(nb2.L)) {   // finished: maybe one closing stage for what is left of the diagonals
                            const int extra = (nb2.L.empty() && (nb2.carry.empty() || !st.has_cx)) ? 0 : 1;
                            if (extra < best_extra || (extra == best_extra && nb2.score > best_score)) { best_extra = extra; best_score = nb2.score; best_seq = nb2.seq; }
                            found = true;
                        } else next.push_back(std::move(nb2));
                    }
                }
                if (found && best_extra == 1 && !next.empty()) {
                    // a sequence one stage longer without a closing stage costs the same: keep what we have (fewer launches of code)
                }
                if (found || next.empty()) break;
                std::stable_sort(next.begin(), next.end(), [](const SB &x, const SB &y) {
                    return x.L.size() != y.L.size() ? x.L.size() < y.L.size() : x.score > y.score; });
                std::vector<SB> keep;
                for (SB &b : next) {
                    bool dup = false;
                    for (const SB &q : keep) if (q.L == b.L && q.carry == b.carry) { dup = true; break; }
                    if (!dup) keep.push_back(std::move(b));
                    if (keep.size() >= WIDTH) break;
                }
                beams.swap(keep);
            }
            if (found) stage_plan = best_seq;
        }
        size_t plan_pos = 0;
        while (!L.empty() || !carry.empty()) {
            bool any_nd = false;
            for (int pos : L) if (!is_diag(bops[pos])) { any_nd = true; break; }
            uint64_t Rset = 0;
            if (!any_nd) {  // only diagonals left: closing segment(s), MAX_SEG_OPS at a time
                size_t take = 0;
                while (take < L.size() && (int)carry.size() < MAX_SEG_OPS) carry.push_back(L[take++]);
                L.erase(L.begin(), L.begin() + take);
                sbest.items.clear(); sbest.rest.clear(); sbest.carry.clear();
                StageItem s; s.is_seg = true; s.op = -1; s.seg_ops = carry;
                sbest.items.push_back(s);
                int cnt = 0; for (int q = 0; q < n && cnt < R; ++q) if (T >> q & 1) { Rset |= 1ull << q; ++cnt; }
            } else {
                stage_candidates(bops, L, T, k, R, mid_cx, rc);
                double bscore = -1e30;
                const bool planned = plan_pos < stage_plan.size();
                if (planned) { rc.clear(); rc.push_back(stage_plan[plan_pos].first); }
                for (uint64_t rs : rc) for (int fa = 0; fa < 2; ++fa) {
                    if (planned && fa != stage_plan[plan_pos].second) continue;
                    stage_take(bops, L, carry, rs, fa != 0, mid_cx, st);
                    if (st.n_nondiag == 0) continue;
                    const double score = st.n_nondiag - 0.1 * st.n_seg - 0.01 * conflict_penalty(T, rs, k);
                    if (score > bscore) { bscore = score; sbest = st; Rset = rs; }
                }
                if (bscore < -1e29) { err = "schedule: stage made no progress (internal)"; return false; }
                ++plan_pos;
                if (sbest.rest.empty() && !sbest.carry.empty() && !sbest.has_cx) {  // last stage of the block: flush what is pending
                    StageItem s; s.is_seg = true; s.op = -1; s.seg_ops = sbest.carry;
                    sbest.items.push_back(s); sbest.carry.clear();
                }
            }
            // ---- emit the stage
            Stage S; memset(&S, 0, sizeof S);
            {
                int slot = 0;
                for (int q = 0; q < n; ++q) if (Rset >> q & 1) {
                    S.regq[slot] = (uint8_t)q; S.regbit[slot] = (uint8_t)local_pos(T, q); ++slot;
                }
            }
            auto slot_of = [&](int q) -> int { for (int s = 0; s < R; ++s) if (S.regq[s] == q) return s; return 255; };
            S.op_begin = (uint32_t)P.mops.size();
            S.seg_begin = (uint32_t)P.segs.size();
            S.cx_begin = (uint32_t)P.cxs.size();
            uint32_t nseg = 0;
            for (const StageItem &it : sbest.items) {
                MicroOp m; memset(&m, 0, sizeof m);
                if (it.is_seg) {
                    DiagSeg sg; sg.rz_begin = (uint32_t)P.rzs.size(); sg.cz_begin = (uint32_t)P.czs.size();
                    for (int pos : it.seg_ops) {
                        const HostOp &o = bops[pos];
                        P.exec_order.push_back(best.taken[pos]);
                        if (o.kind == 1) {
                            DiagRZ r; r.qubit = (uint8_t)o.q0; r.slot = (uint8_t)slot_of(o.q0); r.pad = 0; r.param = o.param;
                            P.rzs.push_back(r);
                        } else {
                            DiagCZ c; c.q0 = (uint8_t)o.q0; c.q1 = (uint8_t)o.q1;
                            c.s0 = (uint8_t)slot_of(o.q0); c.s1 = (uint8_t)slot_of(o.q1);
                            P.czs.push_back(c);
                        }
                    }
                    sg.rz_end = (uint32_t)P.rzs.size(); sg.cz_end = (uint32_t)P.czs.size();
                    m.kind = MOP_DIAG; m.param = (int32_t)P.segs.size();
                    P.segs.push_back(sg); ++nseg;
                } else {
                    const HostOp &o = bops[it.op];
                    P.exec_order.push_back(best.taken[it.op]);
                    if (o.kind == 0) { m.kind = MOP_RY; m.a = (uint8_t)slot_of(o.q0); m.param = o.param; }
                    else if (it.mid_cx) {
                        m.kind = MOP_CX; m.a = (uint8_t)slot_of(o.q0);
                        const int cs = slot_of(o.q1);
                        if (cs != 255) { m.b = (uint8_t)cs; m.c = CTL_REG; } else { m.b = (uint8_t)o.q1; m.c = CTL_FIXED; }
                        m.param = -1;
                    } else { P.cxs.push_back(StageCx{(uint8_t)o.q0, (uint8_t)o.q1}); continue; }
                }
                P.mops.push_back(m);
            }
            S.op_end = (uint32_t)P.mops.size();
            S.cx_end = (uint32_t)P.cxs.size();
            S.n_seg = (uint8_t)nseg;
            if (nseg > 255) { err = "schedule: too many diagonal segments in a stage"; return false; }
            max_seg = std::max(max_seg, nseg);
            P.stages.push_back(S);
            if (any_nd) { L = sbest.rest; carry = sbest.carry; } else carry.clear();
        }
        B.stage_end = (uint32_t)P.stages.size();
        B.max_seg = max_seg;
        P.blocks.push_back(B);
        P.block_ops.push_back(best.taken);
        // ---- remove taken ops
        std::vector<char> gone(ops.size(), 0);
        for (int idx : best.taken) gone[idx] = 1;
        std::vector<int> np; np.reserve(pending.size());
        for (int idx : pending) if (!gone[idx]) np.push_back(idx);
        pending.swap(np);
        first = false;
    }
    return true;
}

std::string dump_program(const Program &p)
{
    std::string s;
    char buf[256];
    snprintf(buf, sizeof buf, "program n=%d k=%d f=%d R=%d blocks=%zu stages=%zu mops=%zu segs=%zu\n", p.n, p.k, p.f, p.R,
             p.blocks.size(), p.stages.size(), p.mops.size(), p.segs.size());
    s += buf;
    for (size_t b = 0; b < p.blocks.size(); ++b) {
        const Block &B = p.blocks[b];
        snprintf(buf, sizeof buf, "block %zu k=%d zero=%d runs=", b, B.k, B.source_zero); s += buf;
        for (int r = 0; r < B.n_runs; ++r) {
            snprintf(buf, sizeof buf, "%d:%d+%d ", B.runs[r].lpos, B.runs[r].gpos, B.runs[r].len); s += buf;
        }
        s += "\n";
        for (uint32_t si = B.stage_begin; si < B.stage_end; ++si) {
            const Stage &S = p.stages[si];
            s += " stage R=";
            for (int j = 0; j < p.R; ++j) { snprintf(buf, sizeof buf, "%d/%d ", S.regbit[j], S.regq[j]); s += buf; }
            s += ":";
            for (uint32_t oi = S.op_begin; oi < S.op_end; ++oi) {
                const MicroOp &m = p.mops[oi];
                if (m.kind == MOP_RY) snprintf(buf, sizeof buf, " RY(s%d,p%d)", m.a, m.param);
                else if (m.kind == MOP_CX) snprintf(buf, sizeof buf, m.c == CTL_REG ? " cx(s%d,c=s%d)" : " cx(s%d,c=q%d)", m.a, m.b);
                else {
                    const DiagSeg &g = p.segs[m.param];
                    snprintf(buf, sizeof buf, " DIAG(#%d rz=%u cz=%u)", m.param, g.rz_end - g.rz_begin, g.cz_end - g.cz_begin);
                }
                s += buf;
            }
            for (uint32_t ci = S.cx_begin; ci < S.cx_end; ++ci) {
                snprintf(buf, sizeof buf, " CX(t=q%d,c=q%d)", p.cxs[ci].tq, p.cxs[ci].cq); s += buf;
            }
            s += "\n";
        }
    }
    return s;
}

}  // namespace gv

// jit.cpp -- generator of the schedule-specialised gate-block kernels (see jit.h).  Pure host C++.
//
// One kernel per fused block.  A thread block is persistent: it walks over (statevector, tile) work items with a grid
// stride; per work item the tile (2^k amplitudes whose index differs only in the block's tile bits) is brought into
// shared memory by 16-byte cp.async copies (no register staging), the block's stages run on it, and it is written back
// in place.  In a stage every thread owns the 2^R amplitudes that differ in the stage's R register bits.
//
// Shared-memory layout of a tile: 16-byte units (two complex64 or one complex128) at unit index
//     pu(u) = u ^ ((u >> 3) & 7) ^ ((u >> 6) & 7) ^ ((u >> 9) & 7)
// which is linear over GF(2), so byte offsets of (thread part) ^ (register part) are XORs of two constants, and a CNOT
// run (an affine map of the local index) stays an XOR with constants.  Thread-index bits 0..2 (0..3) of a stage are
// given local bits whose unit positions differ modulo 3, which makes every 128-byte wavefront conflict free.
//
// Rotations (Eq. 7):  R_y = [[c,-s],[s,c]] = c [[1,-t],[t,1]] (t = s/c, |c| >= |s|)  or
// s [[t',-1],[1,t']] (t' = c/s): two fused multiply-adds per amplitude instead of four multiply/FMA; the scalars c / s
// of all rotations of the block multiply into ONE factor per statevector that joins a diagonal segment's phase.
// R_z phases and CZ signs (Eq. 7; entangling layer PAPER.md:169) of a diagonal segment are one complex
// factor per amplitude = (per-thread table entry) x (per-tile constant) x (small tables over the register bits).
#include "jit.h"
#include "jit_internal.h"

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>

namespace gv {
namespace {

constexpr int JIT_MAX_STAGES = 40;            // per block (code size)
constexpr uint32_t JIT_SMEM_MAX = 113 * 1024;   // two thread blocks per SM

uint64_t scatter(const Block &B, uint32_t j)
{
    uint64_t x = 0;
    for (int r = 0; r < B.n_runs; ++r) x |= (uint64_t)((j >> B.runs[r].lpos) & ((1u << B.runs[r].len) - 1u)) << B.runs[r].gpos;
    return x;
}

int lpos_of(const Block &B, int q)
{
    for (int r = 0; r < B.n_runs; ++r)
        if (q >= B.runs[r].gpos && q < B.runs[r].gpos + B.runs[r].len) return B.runs[r].lpos + (q - B.runs[r].gpos);
    return -1;
}

// Thread-index bit -> local bit of a stage.  The lanes of one shared-memory wavefront (16 lanes of 8-byte accesses, 8 of
// 16-byte ones) are the lowest thread-index bits: they are given the local bits for which the loads AND the stores of the
// stage (the stores go through the CNOT map when the stage ends with a run) hit the most distinct bank groups; searched
// exhaustively (at most C(9,4) subsets).  store_img: image of each local unit vector under the stage's CNOT run, or null.
void choose_thread_bits(const Geo &g, const Stage &S, const uint32_t *store_img, int *tb, bool direct_load = false, bool direct_store = false)
{
    // a stage that exchanges its amplitudes with global memory directly keeps the lowest free local bits in the lanes
    // (whole 32-byte sectors per request); its global side does not count as shared-memory traffic
    bool isreg[16] = {false};
    for (int s = 0; s < g.R; ++s) isreg[S.regbit[s]] = true;
    std::vector<int> free_bits;
    for (int b = 0; b < g.k; ++b) if (!isreg[b]) free_bits.push_back(b);
    const bool wide = g.lv == 0 || S.regbit[0] == 0;          // 16-byte accesses
    const int L = wide ? 3 : 4, nl = 1 << L;
    const int nf = (int)free_bits.size();
    auto waves = [&](const std::vector<int> &lane_bits, bool through_map, bool wide_access) {
        int count[16] = {0};
        int worst = 0;
        for (int l = 0; l < nl; ++l) {
            uint32_t j = 0;
            for (int i = 0; i < L; ++i) if (l >> i & 1) j ^= through_map ? store_img[lane_bits[i]] : (1u << lane_bits[i]);
            const uint32_t o = g.off(j);
            const int slot = wide_access ? (int)((o >> 4) & 7u) : (int)((o >> 3) & 15u);
            worst = std::max(worst, ++count[slot]);
        }
        return worst;
    };
    std::vector<int> best;
    int best_cost = 1 << 30;
    std::vector<int> pick((size_t)L);
    for (uint32_t mask = 0; mask < (1u << nf); ++mask) {
        if (__builtin_popcount(mask) != L) continue;
        int n = 0;
        for (int i = 0; i < nf; ++i) if (mask >> i & 1) pick[(size_t)n++] = free_bits[(size_t)i];
        // stores through a CNOT run are 8-byte accesses for complex64 (16 lanes): judged on the 8-byte banks with the L lanes we have
        int cost = direct_load ? 0 : waves(pick, false, wide) * 4;
        if (direct_store) cost += 0;
        else if (store_img) cost += waves(pick, true, g.lv == 0) * 4; else cost += waves(pick, false, wide) * 4;
        if (direct_load || direct_store) {   // the lowest free bits in the lanes: a request is a run of whole 128-byte lines
            const int need = L;
            for (int i = 0; i < need && i < nf; ++i) {
                bool in = false;
                for (int x = 0; x < L; ++x) in = in || pick[(size_t)x] == free_bits[(size_t)i];
                if (!in) cost += 64;
            }
        }
        for (int i = 0; i < L; ++i) cost += pick[(size_t)i] > 7 ? 1 : 0;   // mild preference for low bits (ties)
        if (cost < best_cost) { best_cost = cost; best = pick; }
    }
    bool used[16] = {false};
    int n = 0;
    for (int b : best) { tb[n++] = b; used[b] = true; }
    for (int b : free_bits) if (!used[b]) tb[n++] = b;
}

// affine map of the local index by a CNOT run: j -> A j ^ c(tile)
struct CxMap {
    uint32_t img[16];                                  // A e_b
    std::vector<std::pair<int, uint32_t>> outside;     // (control qubit outside the tile, image of the target unit vector)
    bool unit_safe = true;                             // no CNOT touches local bit 0 (units of two amplitudes stay units)
    uint32_t apply(uint32_t j, int k) const { uint32_t r = 0; for (int b = 0; b < k; ++b) if (j >> b & 1) r ^= img[b]; return r; }
};

CxMap cx_map(const Program &p, const Block &B, const Stage &S, int k)
{
    CxMap m;
    for (int b = 0; b < 16; ++b) m.img[b] = 1u << b;
    for (uint32_t ci = S.cx_begin; ci < S.cx_end; ++ci) {
        const int tl = lpos_of(B, p.cxs[ci].tq), cl = lpos_of(B, p.cxs[ci].cq);
        if (tl == 0 || cl == 0) m.unit_safe = false;
        if (cl >= 0) {
            for (int b = 0; b < k; ++b) if (m.img[b] >> cl & 1) m.img[b] ^= 1u << tl;
            for (auto &o : m.outside) if (o.second >> cl & 1) o.second ^= 1u << tl;
        } else m.outside.push_back({(int)p.cxs[ci].cq, 1u << tl});
    }
    return m;
}

struct SegInfo {
    int stage = 0;                                        // block-local stage
    std::vector<int> slot_rz[MAX_R];                      // per register slot: block-local RZ indices
    std::vector<std::pair<int, int>> t_rz;                // (thread-index bit, RZ index)
    std::vector<std::pair<int, int>> c_rz;                // (global qubit, RZ index)
    std::vector<std::pair<int, int>> rr;                  // register-register CZ: (slot, slot)
    std::vector<std::pair<int, int>> rt, rc;              // (slot, thread-index bit) / (slot, global qubit)
    std::vector<std::pair<int, int>> tt, tc, cc;          // thread-thread, (thread bit, qubit), (qubit, qubit)
    bool has_phth = false, has_tc = false, has_tm = false, has_rt = false, has_rc = false, scale_here = false;
    std::vector<int> active;                              // register slots with a non-trivial factor
    std::vector<std::pair<int, int>> sflip;               // (slot, RY index): the rotation just before the segment was evaluated
                                                          // in its sine form without the sign of its first row; that sign
                                                          // (-1 on bit 0 of the slot when form = 1) joins the segment's table
    int nlo = 0, nhi = 0;                                 // table split: first nlo active slots | the rest
    uint32_t lo_neg = 0, hi_neg = 0, x_neg = 0;           // register-register CZ signs: per low-table entry, per high-table
                                                          // entry, and (pairs across the two tables) per register index
};

}  // namespace

bool jit_supported(const Program &p, int prec, std::string &why)
{
    const int K = prec == 0 ? 13 : 12, R = prec == 0 ? 5 : 4;
    if (p.k != K || p.R != R) { why = "tile or register size differs from the specialised kernels"; return false; }
    if (p.n < K) { why = "register smaller than one tile"; return false; }
    for (const Block &B : p.blocks)
        if (B.stage_end - B.stage_begin > (uint32_t)JIT_MAX_STAGES) { why = "a block has too many stages"; return false; }
    return true;
}

bool jit_generate(const Program &p, int bi, int prec, int occupancy, bool staged_io, int interleave, JitBlock &out, std::string &err)
{
    if (bi < 0 || (size_t)bi >= p.blocks.size()) { err = "jit: bad block"; return false; }
    const Block &B = p.blocks[bi];
    Geo g;
    g.k = B.k; g.R = p.R; g.TB = g.k - g.R; g.lv = prec == 0 ? 1 : 0; g.prec = prec;
    const int k = g.k, R = g.R, TB = g.TB, NR = 1 << R;
    const uint32_t NT = 1u << TB;
    const int V = 1 << g.lv;
    const uint32_t NU = (1u << k) / V / NT;               // 16-byte units a thread moves in the load / store phase
    const int n = p.n;
    const int ns = (int)(B.stage_end - B.stage_begin);
    if (NT != 256 || NU != 16) { err = "jit: unsupported geometry"; return false; }
    const char *T = prec == 0 ? "float" : "double";
    const uint32_t AB = prec == 0 ? 8 : 16;               // bytes per amplitude

    // ---- parameters of the block: rotations about y (tangent form) and about z ((cos, sin) pairs)
    std::vector<int32_t> ryp, rzp;
    auto idx_of = [](std::vector<int32_t> &v, int32_t pr) { for (size_t i = 0; i < v.size(); ++i) if (v[i] == pr) return (int)i; v.push_back(pr); return (int)v.size() - 1; };

    // ---- lead stage that is nothing but a CNOT run: folded into the destination of the tile load
    bool lead_cx = false;
    CxMap lead;
    if (ns > 1 && !B.source_zero) {
        const Stage &S0 = p.stages[B.stage_begin];
        if (S0.op_begin == S0.op_end && S0.cx_end > S0.cx_begin) {
            lead = cx_map(p, B, S0, k);
            lead_cx = (g.lv == 0) || lead.unit_safe;
        }
    }
    const int s_first = lead_cx ? 1 : 0;
    // first / last stage straight from / to global memory (no staging of the tile in shared memory on that side):
    // possible when the side carries no CNOT run (those are folded into shared-memory addresses)
    // and when the stage's register bits lie above the lowest 128 bytes of the tile (bit 0 of a complex64 pair aside): the
    // lanes then cover whole lines (measured: sector-sized requests run at half the rate of the staged copy or worse)
    auto lines_ok = [&](const Stage &S) {
        for (int r = 0; r < R; ++r) {
            const int lb = S.regbit[r];
            if (g.lv == 1 && r == 0 && lb == 0) continue;
            if (lb < (g.lv == 1 ? 4 : 3)) return false;
        }
        return true;
    };
    bool direct_load = false, direct_store = false;
    if (!staged_io && ns > 0) {
        direct_load = !lead_cx && !B.source_zero && lines_ok(p.stages[B.stage_begin + s_first]);
        const Stage &SL = p.stages[B.stage_begin + ns - 1];
        direct_store = !(SL.cx_end > SL.cx_begin) && (ns - 1 >= s_first) && lines_ok(SL);
    }

    // ---- per-stage geometry and segments
    std::vector<std::vector<int>> tbs((size_t)ns, std::vector<int>(16, 0));
    std::vector<SegInfo> segs;
    std::vector<std::vector<int>> stage_items((size_t)ns);   // per stage: >= 0 RY (index into mops), < 0: -(seg index + 1)
    int last_seg = -1;
    for (int s = 0; s < ns; ++s) {
        const Stage &S = p.stages[B.stage_begin + s];
        {
            const bool cx = S.cx_end > S.cx_begin;
            CxMap cm;
            if (cx) cm = cx_map(p, B, S, k);
            choose_thread_bits(g, S, cx ? cm.img : nullptr, tbs[s].data(), direct_load && s == s_first, direct_store && s == ns - 1);
        }
        auto tbit_of = [&](int lb) { for (int i = 0; i < TB; ++i) if (tbs[s][i] == lb) return i; return -1; };
        auto slot_of = [&](int lb) { for (int r = 0; r < R; ++r) if (S.regbit[r] == lb) return r; return -1; };
        for (uint32_t oi = S.op_begin; oi < S.op_end; ++oi) {
            const MicroOp &m = p.mops[oi];
            if (m.kind == MOP_RY) { idx_of(ryp, m.param); stage_items[s].push_back((int)oi); continue; }
            if (m.kind == MOP_CX) { stage_items[s].push_back((int)oi); continue; }
            const DiagSeg &ds = p.segs[m.param];
            SegInfo si;
            si.stage = s;
            for (uint32_t r = ds.rz_begin; r < ds.rz_end; ++r) {
                const DiagRZ &z = p.rzs[r];
                const int zi = idx_of(rzp, z.param), lb = lpos_of(B, z.qubit);
                if (lb < 0) si.c_rz.push_back({(int)z.qubit, zi});
                else if (slot_of(lb) >= 0) si.slot_rz[slot_of(lb)].push_back(zi);
                else si.t_rz.push_back({tbit_of(lb), zi});
            }
            for (uint32_t c = ds.cz_begin; c < ds.cz_end; ++c) {
                const DiagCZ &z = p.czs[c];
                const int l0 = lpos_of(B, z.q0), l1 = lpos_of(B, z.q1);
                const int s0 = l0 >= 0 ? slot_of(l0) : -1, s1 = l1 >= 0 ? slot_of(l1) : -1;
                if (s0 >= 0 && s1 >= 0) {
                    bool found = false;   // a repeated pair cancels
                    for (size_t e = 0; e < si.rr.size(); ++e)
                        if ((si.rr[e].first == s0 && si.rr[e].second == s1) || (si.rr[e].first == s1 && si.rr[e].second == s0)) { si.rr.erase(si.rr.begin() + (long)e); found = true; break; }
                    if (!found) si.rr.push_back({s0, s1});
                } else if (s0 >= 0 || s1 >= 0) {
                    const int sl = s0 >= 0 ? s0 : s1, lo = s0 >= 0 ? l1 : l0, q = s0 >= 0 ? z.q1 : z.q0;
                    if (lo >= 0) si.rt.push_back({sl, tbit_of(lo)}); else si.rc.push_back({sl, q});
                } else if (l0 >= 0 && l1 >= 0) si.tt.push_back({tbit_of(l0), tbit_of(l1)});
                else if (l0 >= 0 || l1 >= 0) si.tc.push_back({tbit_of(l0 >= 0 ? l0 : l1), (int)(l0 >= 0 ? z.q1 : z.q0)});
                else si.cc.push_back({(int)z.q0, (int)z.q1});
            }
            si.has_phth = !si.t_rz.empty() || !si.tt.empty();
            si.has_tm = !si.tc.empty(); si.has_rt = !si.rt.empty(); si.has_rc = !si.rc.empty();
            for (int r = 0; r < R; ++r) {
                bool act = !si.slot_rz[r].empty();
                for (auto &e : si.rt) if (e.first == r) act = true;
                for (auto &e : si.rc) if (e.first == r) act = true;
                if (act) si.active.push_back(r);
            }
            last_seg = (int)segs.size();
            stage_items[s].push_back(-((int)segs.size() + 1));
            segs.push_back(si);
        }
    }
    const int nseg = (int)segs.size();
    // Sine-form rotations leave a sign on the first row (see emit below).  When a diagonal segment follows in the same
    // stage before another rotation of the same slot, the sign joins that segment (free); otherwise it costs one
    // packed multiply per amplitude pair.
    std::vector<std::vector<int>> ry_defer((size_t)ns);   // per stage item: segment that takes the sign, or -1
    for (int st = 0; st < ns; ++st) {
        const std::vector<int> &it = stage_items[st];
        ry_defer[st].assign(it.size(), -1);
        for (size_t i = 0; i < it.size(); ++i) {
            if (it[i] < 0 || p.mops[it[i]].kind != MOP_RY) continue;
            const int sl = p.mops[it[i]].a;
            for (size_t j = i + 1; j < it.size(); ++j) {
                if (it[j] >= 0) { if (p.mops[it[j]].a == sl) break; continue; }
                const int q = -it[j] - 1;
                ry_defer[st][i] = q;
                segs[q].sflip.push_back({sl, idx_of(ryp, p.mops[it[i]].param)});
                bool have = false;
                for (int a2 : segs[q].active) if (a2 == sl) have = true;
                if (!have) { segs[q].active.push_back(sl); std::sort(segs[q].active.begin(), segs[q].active.end()); }
                break;
            }
        }
    }
    for (SegInfo &si : segs) {
        const int na = (int)si.active.size();
        si.nlo = na <= 3 ? na : 2; si.nhi = na - si.nlo;
        auto pos_in = [&](int slot, int from, int cnt) { for (int i = 0; i < cnt; ++i) if (si.active[from + i] == slot) return i; return -1; };
        for (auto &pr : si.rr) {
            const int l0 = pos_in(pr.first, 0, si.nlo), l1 = pos_in(pr.second, 0, si.nlo);
            const int h0 = pos_in(pr.first, si.nlo, si.nhi), h1 = pos_in(pr.second, si.nlo, si.nhi);
            if (l0 >= 0 && l1 >= 0) { for (int e = 0; e < (1 << si.nlo); ++e) if ((e >> l0 & 1) && (e >> l1 & 1)) si.lo_neg ^= 1u << e; }
            else if (h0 >= 0 && h1 >= 0) { for (int e = 0; e < (1 << si.nhi); ++e) if ((e >> h0 & 1) && (e >> h1 & 1)) si.hi_neg ^= 1u << e; }
            else { for (int r = 0; r < NR; ++r) if ((r >> pr.first & 1) && (r >> pr.second & 1)) si.x_neg ^= 1u << r; }
        }
    }
    if (last_seg >= 0) segs[last_seg].scale_here = !ryp.empty();
    for (SegInfo &si : segs) si.has_tc = !si.c_rz.empty() || !si.cc.empty() || si.scale_here;
    const bool scale_at_store = last_seg < 0 && !ryp.empty();

    // ---- shared memory carve
    uint32_t sm = 0;
    auto take = [&](uint32_t bytes) { const uint32_t o = sm; sm = (sm + bytes + 15u) & ~15u; return o; };
    const uint32_t o_tile = take((uint32_t)AB << k);
    std::vector<uint32_t> o_sb((size_t)ns, 0), o_sb2((size_t)ns, 0);
    for (int s = s_first; s < ns; ++s) {
        o_sb[s] = take(NT * 4);
        const Stage &S = p.stages[B.stage_begin + s];
        if (S.cx_end > S.cx_begin) o_sb2[s] = take(NT * 4);
    }
    const uint32_t o_lead = lead_cx ? take(NT * 4) : 0;
    std::vector<uint32_t> o_phth((size_t)nseg, 0), o_rt((size_t)nseg, 0), o_tab((size_t)nseg, 0);
    for (int q = 0; q < nseg; ++q) {
        if (segs[q].has_phth) o_phth[q] = take(NT * AB);
        if (segs[q].has_rt) o_rt[q] = take(NT * 4);
        o_tab[q] = take(16 * 16);                      // low table (<= 8 entries) then high table (<= 8 entries), 16 bytes each
    }
    const uint32_t o_ry = take((uint32_t)(ryp.size() + 1) * AB), o_sc = take((uint32_t)(ryp.size() + 1) * (AB / 2));
    const uint32_t o_rz = take((uint32_t)(rzp.size() + 1) * AB);
    const uint32_t o_tc = take((uint32_t)(nseg + 1) * AB), o_tm = take((uint32_t)(nseg + 1) * 4), o_rc = take((uint32_t)(nseg + 1) * 4);
    const uint32_t o_scale = take(16);
    if (sm > JIT_SMEM_MAX) { err = "jit: block needs too much shared memory"; return false; }

    char name[64];
    snprintf(name, sizeof name, "gvqe_block_%d_%s", bi, prec == 0 ? "c64" : "c128");
    Emit E;
    E("// generated by libgvqe (jit.cpp): fused gate block %d of %zu, n = %d, k = %d, R = %d, %s; %d stages, %d diagonal segments",
      bi, p.blocks.size(), n, k, R, prec == 0 ? "complex64" : "complex128", ns, nseg);
    E("typedef %s real;", T);
    E("typedef %s2 amp;", T);
    E("typedef unsigned long long u64;");
    if (prec == 0) {
        E("struct __align__(16) ry4 { float t, sc, form, pad; };");
        E("#define MK(x, y) make_float2((x), (y))");
        // table entry: w = (x, y) and i w = (z, w) = (-y, x), so a * w = a.x (x, y) + a.y (z, w): two packed operations
        E("struct __align__(16) tw { float x, y, z, w; };");
        E("__device__ __forceinline__ tw twmake(amp v) { tw t; t.x = v.x; t.y = v.y; t.z = -v.y; t.w = v.x; return t; }");
        E("__device__ __forceinline__ amp cmul(amp a, amp w) { return __ffma2_rn(MK(a.y, a.y), MK(-w.y, w.x), __fmul2_rn(MK(a.x, a.x), w)); }");
        E("__device__ __forceinline__ amp cmulT(amp a, tw t) { return __ffma2_rn(MK(a.y, a.y), MK(t.z, t.w), __fmul2_rn(MK(a.x, a.x), MK(t.x, t.y))); }");
        E("__device__ __forceinline__ amp cmulTn(amp a, tw t) { return __ffma2_rn(MK(-a.y, -a.y), MK(t.z, t.w), __fmul2_rn(MK(-a.x, -a.x), MK(t.x, t.y))); }");
        E("__device__ __forceinline__ tw twmul(tw t, tw p) { tw r; const amp u = cmulT(MK(t.x, t.y), p), v = cmulT(MK(t.z, t.w), p); r.x = u.x; r.y = u.y; r.z = v.x; r.w = v.y; return r; }");
        E("__device__ __forceinline__ tw twscale(tw t, real s) { const amp u = __fmul2_rn(MK(t.x, t.y), MK(s, s)), v = __fmul2_rn(MK(t.z, t.w), MK(s, s)); tw r; r.x = u.x; r.y = u.y; r.z = v.x; r.w = v.y; return r; }");
        E("__device__ __forceinline__ void ryc(amp &u, amp &v, real t) { const amp tt = MK(t, t), nt = MK(-t, -t), u0 = u; u = __ffma2_rn(nt, v, u0); v = __ffma2_rn(tt, u0, v); }");
        // sine form WITHOUT the sign of the first row: (v - t u, u + t v) = diag(-1, 1) [[t,-1],[1,t]] (u, v)
        E("__device__ __forceinline__ void rysn(amp &u, amp &v, real t) { const amp tt = MK(t, t), nt = MK(-t, -t), u0 = u; u = __ffma2_rn(nt, u0, v); v = __ffma2_rn(tt, v, u0); }");
        E("__device__ __forceinline__ void rys(amp &u, amp &v, real t) { rysn(u, v, t); u = __fmul2_rn(u, MK(-1.f, -1.f)); }");
        E("__device__ __forceinline__ amp scal(amp a, real s) { return __fmul2_rn(a, MK(s, s)); }");
    } else {
        E("struct __align__(32) ry4 { double t, sc, form, pad; };");
        E("#define MK(x, y) make_double2((x), (y))");
        E("typedef double2 tw;");
        E("__device__ __forceinline__ tw twmake(amp v) { return v; }");
        E("__device__ __forceinline__ amp cmul(amp a, amp w) { return MK(fma(-a.y, w.y, a.x * w.x), fma(a.y, w.x, a.x * w.y)); }");
        E("__device__ __forceinline__ amp cmulT(amp a, tw w) { return cmul(a, w); }");
        E("__device__ __forceinline__ amp cmulTn(amp a, tw w) { return MK(fma(a.y, w.y, -a.x * w.x), fma(-a.y, w.x, -a.x * w.y)); }");
        E("__device__ __forceinline__ tw twmul(tw t, tw p) { return cmul(t, p); }");
        E("__device__ __forceinline__ tw twscale(tw t, real s) { return MK(t.x * s, t.y * s); }");
        E("__device__ __forceinline__ void ryc(amp &u, amp &v, real t) { const amp u0 = u; u = MK(fma(-t, v.x, u0.x), fma(-t, v.y, u0.y)); v = MK(fma(t, u0.x, v.x), fma(t, u0.y, v.y)); }");
        E("__device__ __forceinline__ void rysn(amp &u, amp &v, real t) { const amp u0 = u; u = MK(fma(-t, u0.x, v.x), fma(-t, u0.y, v.y)); v = MK(fma(t, v.x, u0.x), fma(t, v.y, u0.y)); }");
        E("__device__ __forceinline__ void rys(amp &u, amp &v, real t) { const amp u0 = u; u = MK(fma(t, u0.x, -v.x), fma(t, u0.y, -v.y)); v = MK(fma(t, v.x, u0.x), fma(t, v.y, u0.y)); }");
        E("__device__ __forceinline__ amp scal(amp a, real s) { return MK(a.x * s, a.y * s); }");
    }
    E("__device__ __forceinline__ amp cneg(amp a) { return MK(-a.x, -a.y); }");
    E("__device__ __forceinline__ amp cconj(amp a) { return MK(a.x, -a.y); }");
    E("struct __align__(16) unit16 { unsigned x, y, z, w; };");
    E("__device__ __forceinline__ void cp16(void *dst, const void *src) {");
    E("    asm volatile(\"cp.async.cg.shared.global [%%0], [%%1], 16;\" :: \"r\"((unsigned)__cvta_generic_to_shared(dst)), \"l\"(src));");
    E("}");
    E("__device__ __forceinline__ void cp_wait() { asm volatile(\"cp.async.wait_all;\" ::: \"memory\"); }");
    E("__device__ __forceinline__ unsigned OFF(unsigned j) { const unsigned u = j >> %d; return ((u ^ ((u >> 3) & 7u) ^ ((u >> 6) & 7u) ^ ((u >> 9) & 7u)) << 4) | ((j & %uu) << 3); }",
      g.lv, (1u << g.lv) - 1u);
    auto emit_int_array = [&](const char *nm, const std::vector<int32_t> &v) {
        std::string t = std::string("__device__ const int ") + nm + "[" + std::to_string(v.size() + 1) + "] = {";
        for (int32_t x : v) t += std::to_string(x) + ", ";
        t += "0};";
        E("%s", t.c_str());
    };
    emit_int_array("RYP", ryp);
    emit_int_array("RZP", rzp);
    for (int q = 0; q < nseg; ++q) {
        if (segs[q].c_rz.empty()) continue;
        std::vector<int32_t> cq, ci;
        for (auto &e : segs[q].c_rz) { cq.push_back(e.first); ci.push_back(e.second); }
        char nm[32];
        snprintf(nm, sizeof nm, "CQ%d", q); emit_int_array(nm, cq);
        snprintf(nm, sizeof nm, "CI%d", q); emit_int_array(nm, ci);
    }
    E("");
    // per_cta: work items (statevector, tile) one thread block handles, consecutive
    // src / src_stride: where the tiles are READ (normally = states / stride; a parameter-shift sweep reads the shared base
    // state of theta, src_stride = 0, and writes the shifted rows' own buffers: SURVEY 8(f) NEXT-2)
    E("extern \"C\" __global__ void __launch_bounds__(%u, %d) %s(amp *states, u64 stride, const ry4 *rytab, const amp *cstab, int nb, int Pn, int per_cta,", NT, occupancy == 3 ? 3 : 2, name);
    E("        const amp *src, u64 src_stride)");
    E("{");
    E("    extern __shared__ __align__(128) unsigned char smem[];");
    E("    unsigned char *tile = smem + %u;", o_tile);
    E("    const unsigned tid = threadIdx.x;");
    E("    amp *s_ry = (amp *)(smem + %u); real *s_sc = (real *)(smem + %u); amp *s_rz = (amp *)(smem + %u);", o_ry, o_sc, o_rz);
    E("    amp *s_tc = (amp *)(smem + %u); unsigned *s_tm = (unsigned *)(smem + %u); unsigned *s_rc = (unsigned *)(smem + %u);", o_tc, o_tm, o_rc);
    E("    real *s_scale = (real *)(smem + %u);", o_scale);
    E("    (void)s_tc; (void)s_tm; (void)s_rc; (void)s_sc; (void)s_ry; (void)s_rz; (void)src; (void)src_stride;");
    // ---- tables that depend on the thread index only
    for (int s = s_first; s < ns; ++s) {
        const Stage &S = p.stages[B.stage_begin + s];
        E("    {   // stage %d: thread part of the shared-memory offset", s);
        emit_deposit(E, "        ", "j", tbs[s].data(), TB);
        E("        ((unsigned *)(smem + %u))[tid] = OFF(j);", o_sb[s]);
        if (S.cx_end > S.cx_begin) {
            const CxMap m = cx_map(p, B, S, k);
            E("        unsigned ja = 0u;");
            for (int i = 0; i < TB; ++i) E("        if ((tid >> %d) & 1u) ja ^= %uu;", i, m.img[tbs[s][i]]);
            E("        ((unsigned *)(smem + %u))[tid] = OFF(ja);", o_sb2[s]);
        }
        E("    }");
    }
    // units of the load / store phase: unit index u = tid + NT * i, local index j = u << lv
    E("    const unsigned ld_off = OFF(tid << %d);", g.lv);
    {
        std::string sx = "    const u64 ld_x = 0ull";
        for (int r = 0; r < B.n_runs; ++r) {
            const int lp = B.runs[r].lpos, len = B.runs[r].len, gp = B.runs[r].gpos;
            int lo = lp - g.lv, hi = lp + len - g.lv;   // thread-index bits held by local bits [lp, lp + len)
            if (lo < 0) lo = 0;
            if (hi > TB) hi = TB;
            if (hi <= lo) continue;
            char b[128];
            snprintf(b, sizeof b, " | ((u64)((tid >> %d) & %uu) << %d)", lo, (1u << (hi - lo)) - 1u, gp + (lo + g.lv - lp));
            sx += b;
        }
        sx += ";";
        E("%s", sx.c_str());
    }
    auto emit_thread_global = [&](const char *nm, int s) {   // global offset (amplitudes) of the thread's part of the local index in stage s
        std::string sx = std::string("    const u64 ") + nm + " = 0ull";
        for (int i = 0; i < TB; ++i) {
            char b[96];
            snprintf(b, sizeof b, " | ((u64)((tid >> %d) & 1u) << %d)", i, __builtin_ctzll(scatter(B, 1u << tbs[s][i])));
            sx += b;
        }
        sx += ";";
        E("%s", sx.c_str());
    };
    if (direct_load) emit_thread_global("dl_x", s_first);
    if (direct_store) emit_thread_global("ds_x", ns - 1);
    if (lead_cx) {
        E("    {   // leading CNOT run: thread part of the permuted destination");
        E("        unsigned ja = 0u;");
        for (int i = 0; i < TB; ++i) E("        if ((tid >> %d) & 1u) ja ^= %uu;", i, lead.img[i + g.lv]);
        E("        ((unsigned *)(smem + %u))[tid] = OFF(ja);", o_lead);
        E("    }");
    }
    for (int q = 0; q < nseg; ++q) {
        if (!segs[q].has_rt) continue;
        E("    {   // segment %d: CZ between register slots and thread bits", q);
        E("        unsigned f = 0u;");
        for (auto &e : segs[q].rt) E("        f ^= ((tid >> %d) & 1u) << %d;", e.second, e.first);
        E("        ((unsigned *)(smem + %u))[tid] = f;", o_rt[q]);
        E("    }");
    }
    E("    int cur_b = -1;");
    E("    const u64 total = (u64)nb << %d;", n - k);
    // thread blocks in groups of IL take neighbouring tiles at the same time (their 128-byte pieces are adjacent in memory);
    // a group that would run past the end falls back to consecutive tiles per thread block
    const unsigned IL = interleave > 1 ? (unsigned)interleave : 1u;
    E("    const u64 il_base = (u64)(blockIdx.x / %uu) * (u64)per_cta * %uull;", IL, IL);
    E("    const bool il = il_base + (u64)per_cta * %uull <= total;", IL);
    E("    const u64 w_first = il ? il_base + (u64)(blockIdx.x %% %uu) : (u64)blockIdx.x * (u64)per_cta;", IL);
    E("    const u64 w_step = il ? %uull : 1ull;", IL);
    E("    for (int it = 0; it < per_cta; ++it) {");
    E("        const u64 w = w_first + (u64)it * w_step;");
    E("        if (w >= total) break;");
    E("        const int b = (int)(w >> %d);", n - k);
    E("        const u64 tile_id = w & %lluull;", (unsigned long long)((1ull << (n - k)) - 1ull));
    E("        amp *state = states + (u64)b * stride;");
    // ---- tile base
    {
        E("        u64 xbase = 0ull;");
        int consumed = 0, gpos = 0;
        for (int r = 0; r <= B.n_runs; ++r) {
            const int gend = r < B.n_runs ? B.runs[r].gpos : n;
            const int gap = gend - gpos;
            if (gap > 0) {
                E("        xbase |= ((tile_id >> %d) & %lluull) << %d;", consumed, (unsigned long long)((1ull << gap) - 1ull), gpos);
                consumed += gap;
            }
            if (r < B.n_runs) gpos = B.runs[r].gpos + B.runs[r].len;
        }
    }
    E("        amp *gptr = state + (xbase | ld_x);");
    E("        const amp *gsrc = src + (u64)b * src_stride + (xbase | ld_x);");
    // ---- load phase
    std::vector<uint64_t> hi(NU);
    std::vector<uint32_t> ci(NU), ci_lead(NU);
    for (uint32_t i = 0; i < NU; ++i) {
        const uint32_t j = (NT * i) << g.lv;
        hi[i] = scatter(B, j); ci[i] = g.off(j);
        if (lead_cx) ci_lead[i] = g.off(lead.apply(j, k));
    }
    if (B.source_zero) {
        E("        if (xbase != 0ull) {   // |0...0> has no weight in this tile and gates act inside tiles: stays zero");
        E("            const unit16 z = {0u, 0u, 0u, 0u};");
        for (uint32_t i = 0; i < NU; ++i) E("            *(unit16 *)(gptr + %lluull) = z;", (unsigned long long)hi[i]);
        E("            continue;");
        E("        }");
        E("        {");
        E("            const unit16 z = {0u, 0u, 0u, 0u};");
        for (uint32_t i = 0; i < NU; ++i) E("            *(unit16 *)(tile + (ld_off ^ %uu)) = z;", ci[i]);
        E("        }");
        E("        __syncthreads();");
        E("        if (tid == 0) *(amp *)tile = MK((real)1, (real)0);");
    } else if (lead_cx) {
        std::string oc = "        const unsigned lead_o = ((const unsigned *)(smem + " + std::to_string(o_lead) + "))[tid]";
        for (auto &e : lead.outside) {
            char b[96];
            snprintf(b, sizeof b, " ^ (((xbase >> %d) & 1ull) ? %uu : 0u)", e.first, g.off(e.second));
            oc += b;
        }
        E("%s;", oc.c_str());
        for (uint32_t i = 0; i < NU; ++i) E("        cp16(tile + (lead_o ^ %uu), gsrc + %lluull);", ci_lead[i], (unsigned long long)hi[i]);
    } else if (direct_load) {
        const Stage &S = p.stages[B.stage_begin + s_first];
        const bool wide = (g.lv == 1 && S.regbit[0] == 0);
        E("        amp a_in[%d];   // the first stage's amplitudes, straight from global memory", NR);
        E("        {");
        E("            const amp *gl = src + (u64)b * src_stride + (xbase | dl_x);");
        for (int r = 0; r < NR; ++r) {
            uint32_t j = 0;
            for (int bb = 0; bb < R; ++bb) if (r >> bb & 1) j |= 1u << S.regbit[bb];
            const unsigned long long go = (unsigned long long)scatter(B, j);
            if (wide) { if (!(r & 1)) E("            { const float4 v = *(const float4 *)(gl + %lluull); a_in[%d] = MK(v.x, v.y); a_in[%d] = MK(v.z, v.w); }", go, r, r + 1); }
            else E("            a_in[%d] = gl[%lluull];", r, go);
        }
        E("        }");
    } else {
        for (uint32_t i = 0; i < NU; ++i) E("        cp16(tile + (ld_off ^ %uu), gsrc + %lluull);", ci[i], (unsigned long long)hi[i]);
    }
    // ---- per-statevector setup
    E("        if (b != cur_b) {");
    E("            cur_b = b;");
    E("            for (unsigned i = tid; i < %zuu; i += %uu) { const ry4 v = rytab[(u64)b * Pn + RYP[i]]; s_ry[i] = MK(v.t, v.form); s_sc[i] = v.sc; }", ryp.size(), NT);
    E("            for (unsigned i = tid; i < %zuu; i += %uu) s_rz[i] = cstab[(u64)b * Pn + RZP[i]];", rzp.size(), NT);
    E("            __syncthreads();");
    E("            if (tid >= %uu) {   // product of the rotations' scale factors (last warp)", NT - 32);
    E("                real sc = (real)1;");
    E("                for (unsigned i = tid - %uu; i < %zuu; i += 32u) sc *= s_sc[i];", NT - 32, ryp.size());
    E("                for (int o = 16; o > 0; o >>= 1) sc *= __shfl_xor_sync(0xffffffffu, sc, o);");
    E("                if (tid == %uu) *s_scale = sc;", NT - 32);
    E("            }");
    for (int q = 0; q < nseg; ++q) {
        const SegInfo &si = segs[q];
        // tables over the register slots: entry e = prod over its slots of (bit ? F1 : F0), F1 = e^{+i phi/2} products, F0 = conj,
        // with the deferred sine-form sign on F0 and the register-register CZ signs that stay inside one table
        for (int half = 0; half < 2; ++half) {
            const int cnt = half == 0 ? si.nlo : si.nhi, from = half == 0 ? 0 : si.nlo;
            if (half == 1 && cnt == 0) continue;
            if (half == 0 && cnt == 0) continue;
            const int tbase = (q * 16 + half * 8) % (int)NT;   // one thread per entry; segments 16 apart share threads (in turn)
            E("            if (tid >= %du && tid < %du) {   // segment %d, %s table", tbase, tbase + (1 << cnt), q, half ? "high" : "low");
            E("                const unsigned e = tid - %du;", tbase);
            E("                amp f = MK((real)1, (real)0);");
            for (int i = 0; i < cnt; ++i) {
                const int sl = si.active[from + i];
                E("                {");
                if (si.slot_rz[sl].empty()) E("                    amp f1 = MK((real)1, (real)0);");
                else {
                    E("                    amp f1 = s_rz[%d];", si.slot_rz[sl][0]);
                    for (size_t z = 1; z < si.slot_rz[sl].size(); ++z) E("                    f1 = cmul(f1, s_rz[%d]);", si.slot_rz[sl][z]);
                }
                E("                    amp f0 = cconj(f1);");
                for (auto &sf : si.sflip) if (sf.first == sl) E("                    if (s_ry[%d].y != (real)0) f0 = cneg(f0);", sf.second);
                E("                    f = cmul(f, ((e >> %d) & 1u) ? f1 : f0);", i);
                E("                }");
            }
            const uint32_t neg = half == 0 ? si.lo_neg : si.hi_neg;
            if (neg) E("                if ((%uu >> e) & 1u) f = cneg(f);", neg);
            E("                ((tw *)(smem + %u))[%d + e] = twmake(f);", o_tab[q], half * 8);
            E("            }");
        }
        if (!si.has_phth) continue;
        E("            {   // segment %d: phase over the thread bits", q);
        E("                amp ph = MK((real)1, (real)0);");
        for (auto &e : si.t_rz) E("                { const amp e = s_rz[%d]; ph = cmul(ph, ((tid >> %d) & 1u) ? e : cconj(e)); }", e.second, e.first);
        for (auto &e : si.tt) E("                if (((tid >> %d) & (tid >> %d)) & 1u) ph = cneg(ph);", e.first, e.second);
        E("                ((amp *)(smem + %u))[tid] = ph;", o_phth[q]);
        E("            }");
    }
    E("            __syncthreads();");
    E("        }");
    // ---- per-tile constants of the diagonal segments, one warp per segment, under the loads
    for (int q = 0; q < nseg; ++q) {
        const SegInfo &si = segs[q];
        if (!si.has_tc && !si.has_tm && !si.has_rc) continue;
        E("        if ((tid >> 5) == %du) {   // segment %d: what depends on the tile", q % (int)(NT / 32), q);
        E("            const unsigned lane = tid & 31u;");
        if (si.has_tc) {
            E("            amp f = MK((real)1, (real)0);");
            if (!si.c_rz.empty()) {
                const int nc = (int)si.c_rz.size();
                E("            for (unsigned i = lane; i < %du; i += 32u) { const amp e = s_rz[CI%d[i]]; f = cmul(f, ((xbase >> CQ%d[i]) & 1ull) ? e : cconj(e)); }", nc, q, q);
                E("            for (int o = 16; o > 0; o >>= 1) { amp g2; g2.x = __shfl_xor_sync(0xffffffffu, f.x, o); g2.y = __shfl_xor_sync(0xffffffffu, f.y, o); f = cmul(f, g2); }");
            }
            for (auto &e : si.cc) E("            if (((xbase >> %d) & (xbase >> %d)) & 1ull) f = cneg(f);", e.first, e.second);
            if (si.scale_here) E("            f = scal(f, *s_scale);");
            E("            if (lane == 0) s_tc[%d] = f;", q);
        }
        if (si.has_tm) {
            E("            unsigned m = 0u;");
            for (auto &e : si.tc) E("            m ^= (unsigned)((xbase >> %d) & 1ull) << %d;", e.second, e.first);
            E("            if (lane == 0) s_tm[%d] = m;", q);
        }
        if (si.has_rc) {
            E("            unsigned m2 = 0u;");
            for (auto &e : si.rc) E("            m2 ^= (unsigned)((xbase >> %d) & 1ull) << %d;", e.second, e.first);
            E("            if (lane == 0) s_rc[%d] = m2;", q);
        }
        E("        }");
    }
    if (!B.source_zero && !direct_load) E("        cp_wait();");
    E("        __syncthreads();");
    // ---- stages
    const uint32_t LOMASK = 0x70u;   // address bits the swizzle folds into: XOR there, plain addition everywhere else
    for (int s = s_first; s < ns; ++s) {
        const Stage &S = p.stages[B.stage_begin + s];
        const bool has_cx = S.cx_end > S.cx_begin;
        const bool wide = (g.lv == 1 && S.regbit[0] == 0);    // complex64 with local bit 0 in a register: 16-byte accesses
        uint32_t cr[32];
        bool vused[8] = {false};
        for (int r = 0; r < NR; ++r) {
            uint32_t j = 0;
            for (int b = 0; b < R; ++b) if (r >> b & 1) j |= 1u << S.regbit[b];
            cr[r] = g.off(j);
            vused[(cr[r] & LOMASK) >> 4] = true;
        }
        E("        {   // ---- stage %d", s);
        E("            const unsigned sb = ((const unsigned *)(smem + %u))[tid];", o_sb[s]);
        // address of register index r = [tile + (sb ^ low bits of its offset)] + the rest of its offset (an immediate)
        for (int v = 0; v < 8; ++v) if (vused[v]) E("            unsigned char *const pv%d = tile + (sb ^ %uu);", v, (uint32_t)v << 4);
        if (direct_load && s == s_first) E("            amp (&a)[%d] = a_in;", NR);
        else E("            amp a[%d];", NR);
        if (direct_load && s == s_first) {
        } else if (wide) {
            for (int r = 0; r < NR; r += 2)
                E("            { const float4 v = *(const float4 *)(pv%u + %uu); a[%d] = MK(v.x, v.y); a[%d] = MK(v.z, v.w); }", (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK, r, r + 1);
        } else {
            for (int r = 0; r < NR; ++r) E("            a[%d] = *(const amp *)(pv%u + %uu);", r, (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK);
        }
        // logical register index (the amplitude's true index bits) -> name in a[]: a CNOT between two register qubits only
        // renames; one whose control is a thread or tile bit swaps the target pairs where the control is set
        std::vector<int> perm((size_t)NR);
        for (int r = 0; r < NR; ++r) perm[(size_t)r] = r;
        auto tbit_of_stage = [&](int lb) { for (int i = 0; i < TB; ++i) if (tbs[s][i] == lb) return i; return -1; };
        for (size_t ii = 0; ii < stage_items[s].size(); ++ii) {
            const int item = stage_items[s][ii];
            if (item >= 0 && p.mops[item].kind == MOP_CX) {
                const MicroOp &m = p.mops[item];
                const int t = m.a;
                if (m.c == CTL_REG) {
                    E("            // CNOT target slot %d, control slot %d: renamed", t, m.b);
                    for (int r = 0; r < NR; ++r) if ((r >> m.b & 1) && !(r >> t & 1)) std::swap(perm[(size_t)r], perm[(size_t)(r | (1 << t))]);
                } else {
                    const int lb = lpos_of(B, m.b);
                    if (lb >= 0) E("            {   // CNOT target slot %d, control qubit %d (a thread bit)\n                const bool cxc = (tid >> %d) & 1u;", t, m.b, tbit_of_stage(lb));
                    else E("            {   // CNOT target slot %d, control qubit %d (outside the tile)\n                const bool cxc = (xbase >> %d) & 1ull;", t, m.b, m.b);
                    for (int r = 0; r < NR; ++r) if (!(r >> t & 1)) {
                        const int i0 = perm[(size_t)r], i1 = perm[(size_t)(r | (1 << t))];
                        E("                { const amp u = a[%d], v = a[%d]; a[%d] = cxc ? v : u; a[%d] = cxc ? u : v; }", i0, i1, i0, i1);
                    }
                    E("            }");
                }
                continue;
            }
            if (item >= 0) {
                const MicroOp &m = p.mops[item];
                const int yi = idx_of(ryp, m.param), sl = m.a;
                const char *sine = ry_defer[s][ii] >= 0 ? "rysn" : "rys";
                E("            {   // R_y on slot %d (parameter %d)%s", sl, m.param, ry_defer[s][ii] >= 0 ? "; sine-form sign joins the next segment" : "");
                E("                const amp q = s_ry[%d];", yi);
                E("                if (q.y == (real)0) {");
                for (int r = 0; r < NR; ++r) if (!(r >> sl & 1)) E("                    ryc(a[%d], a[%d], q.x);", perm[r], perm[r | (1 << sl)]);
                E("                } else {");
                for (int r = 0; r < NR; ++r) if (!(r >> sl & 1)) E("                    %s(a[%d], a[%d], q.x);", sine, perm[r], perm[r | (1 << sl)]);
                E("                }");
                E("            }");
                continue;
            }
            const int q = -item - 1;
            const SegInfo &si = segs[q];
            const int nlo = si.nlo, nhi = si.nhi;
            E("            {   // diagonal segment %d", q);
            // factor common to the thread's amplitudes
            const bool any_ph = si.has_phth || si.has_tc || si.has_tm;
            if (si.has_phth) E("                amp ph = ((const amp *)(smem + %u))[tid];", o_phth[q]);
            else if (any_ph) E("                amp ph = MK((real)1, (real)0);");
            if (si.has_tc) {
                if (si.has_phth) E("                ph = cmul(ph, s_tc[%d]);", q);
                else E("                ph = s_tc[%d];", q);
            }
            if (si.has_tm) E("                if (__popc(tid & s_tm[%d]) & 1) ph = cneg(ph);", q);
            if (si.has_rt || si.has_rc) {
                std::string f = "                const unsigned fl = 0u";
                if (si.has_rt) f += " ^ ((const unsigned *)(smem + " + std::to_string(o_rt[q]) + "))[tid]";
                if (si.has_rc) f += " ^ s_rc[" + std::to_string(q) + "]";
                E("%s;", f.c_str());
                // a CZ between register slot s and a set thread / tile bit negates the slot's F1: sign of entry e = prod over its slots
                for (int i = 0; i < nlo + nhi; ++i) {
                    const int sl = si.active[i];
                    bool flips = false;
                    for (auto &e : si.rt) if (e.first == sl) flips = true;
                    for (auto &e : si.rc) if (e.first == sl) flips = true;
                    if (flips) E("                const real sg%d = ((fl >> %d) & 1u) ? (real)-1 : (real)1;", i, sl);
                    else E("                const real sg%d = (real)1;", i);
                }
            }
            const bool flips_any = si.has_rt || si.has_rc;
            auto sign_expr = [&](int e, int from, int cnt) {
                std::string x;
                for (int i = 0; i < cnt; ++i) if (e >> i & 1) { if (!x.empty()) x += " * "; x += "sg" + std::to_string(from + i); }
                return x;
            };
            if (nlo == 0) {
                if (any_ph) {
                    E("                const tw t0 = twmake(ph);");
                    for (int r = 0; r < NR; ++r) E("                a[%d] = %s(a[%d], t0);", perm[r], (si.x_neg >> r & 1) ? "cmulTn" : "cmulT", perm[r]);
                } else if (si.x_neg) {
                    for (int r = 0; r < NR; ++r) if (si.x_neg >> r & 1) E("                a[%d] = cneg(a[%d]);", perm[r], perm[r]);
                }
            } else {
                E("                tw tl[%d];", 1 << nlo);
                for (int e = 0; e < (1 << nlo); ++e) {
                    E("                tl[%d] = ((const tw *)(smem + %u))[%d];", e, o_tab[q], e);
                    if (flips_any && !sign_expr(e, 0, nlo).empty()) E("                tl[%d] = twscale(tl[%d], %s);", e, e, sign_expr(e, 0, nlo).c_str());
                }
                if (any_ph) {
                    E("                { const tw pw = twmake(ph);");
                    for (int e = 0; e < (1 << nlo); ++e) E("                  tl[%d] = twmul(tl[%d], pw);", e, e);
                    E("                }");
                }
                auto tidx = [&](int r, int from, int cnt) { int v = 0; for (int i = 0; i < cnt; ++i) if (r >> si.active[from + i] & 1) v |= 1 << i; return v; };
                for (int r = 0; r < NR; ++r)
                    E("                a[%d] = %s(a[%d], tl[%d]);", perm[r], (si.x_neg >> r & 1) ? "cmulTn" : "cmulT", perm[r], tidx(r, 0, nlo));
                if (nhi > 0) {
                    E("                tw th[%d];", 1 << nhi);
                    for (int e = 0; e < (1 << nhi); ++e) {
                        E("                th[%d] = ((const tw *)(smem + %u))[%d];", e, o_tab[q], 8 + e);
                        if (flips_any && !sign_expr(e, nlo, nhi).empty()) E("                th[%d] = twscale(th[%d], %s);", e, e, sign_expr(e, nlo, nhi).c_str());
                    }
                    for (int r = 0; r < NR; ++r) E("                a[%d] = cmulT(a[%d], th[%d]);", perm[r], perm[r], tidx(r, nlo, nhi));
                }
            }
            E("            }");
        }
        if (direct_store && s == ns - 1) {   // results straight to global memory
            E("            amp *gs = state + (xbase | ds_x);");
            if (scale_at_store) {
                E("            const real sc = *s_scale;");
                for (int r = 0; r < NR; ++r) E("            a[%d] = scal(a[%d], sc);", r, r);
            }
            for (int r = 0; r < NR; ++r) {
                uint32_t j = 0;
                for (int bb = 0; bb < R; ++bb) if (r >> bb & 1) j |= 1u << S.regbit[bb];
                const unsigned long long go = (unsigned long long)scatter(B, j);
                if (wide) { if (!(r & 1)) E("            *(float4 *)(gs + %lluull) = make_float4(a[%d].x, a[%d].y, a[%d].x, a[%d].y);", go, perm[r], perm[r], perm[r + 1], perm[r + 1]); }
                else E("            gs[%lluull] = a[%d];", go, perm[r]);
            }
        } else if (!has_cx) {
            if (wide) {
                for (int r = 0; r < NR; r += 2)
                    E("            *(float4 *)(pv%u + %uu) = make_float4(a[%d].x, a[%d].y, a[%d].x, a[%d].y);", (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK, perm[r], perm[r], perm[r + 1], perm[r + 1]);
            } else {
                for (int r = 0; r < NR; ++r) E("            *(amp *)(pv%u + %uu) = a[%d];", (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK, perm[r]);
            }
        } else {
            // trailing CNOT run: |j> -> |A j ^ c>; the amplitude of local index j_thread ^ j_r goes to
            // off(A j_thread) ^ off(c(tile)) ^ off(A j_r): thread part from a table, the rest literals
            const CxMap m = cx_map(p, B, S, k);
            uint32_t mtt = 0, mr = 0, mout = 0;   // address bits outside the folded ones that the thread, register and tile parts can set
            for (int i = 0; i < TB; ++i) mtt |= g.off(m.img[tbs[s][i]]) & ~LOMASK;
            for (int b = 0; b < R; ++b) mr |= g.off(m.img[S.regbit[b]]) & ~LOMASK;
            for (auto &e : m.outside) mout |= g.off(e.second) & ~LOMASK;
            uint32_t c2[32];
            for (int r = 0; r < NR; ++r) {
                uint32_t j = 0;
                for (int b = 0; b < R; ++b) if (r >> b & 1) j |= 1u << S.regbit[b];
                c2[r] = g.off(m.apply(j, k));
            }
            E("            __syncthreads();   // every thread has read its amplitudes before any permuted write");
            E("            const unsigned sb2 = ((const unsigned *)(smem + %u))[tid];", o_sb2[s]);
            const int no = (int)m.outside.size();
            if ((mtt & (mr | mout)) == 0 && no <= 2) {
                // the thread part never meets the others outside the folded bits: immediates again; the tile-dependent
                // constant c (controls outside the tile) selects one of 2^no literal variants (uniform branch)
                for (int var = 0; var < (1 << no); ++var) {
                    uint32_t cv = 0;
                    std::string cond;
                    for (int i = 0; i < no; ++i) {
                        char bb[64];
                        snprintf(bb, sizeof bb, "%s((xbase >> %d) & 1ull) == %dull", i ? " && " : "", m.outside[i].first, (var >> i) & 1);
                        cond += bb;
                        if (var >> i & 1) cv ^= g.off(m.outside[i].second);
                    }
                    if (no) E("            if (%s) {", cond.c_str()); else E("            {");
                    bool v2[8] = {false};
                    for (int r = 0; r < NR; ++r) v2[((c2[r] ^ cv) & LOMASK) >> 4] = true;
                    for (int v = 0; v < 8; ++v) if (v2[v]) E("                unsigned char *const pw%d = tile + (sb2 ^ %uu);", v, (uint32_t)v << 4);
                    for (int r = 0; r < NR; ++r) E("                *(amp *)(pw%u + %uu) = a[%d];", ((c2[r] ^ cv) & LOMASK) >> 4, (c2[r] ^ cv) & ~LOMASK, perm[r]);
                    E("            }");
                }
            } else {
                std::string oc = "            const unsigned sb3 = sb2";
                for (auto &e : m.outside) {
                    char bb[96];
                    snprintf(bb, sizeof bb, " ^ (((xbase >> %d) & 1ull) ? %uu : 0u)", e.first, g.off(e.second));
                    oc += bb;
                }
                E("%s;", oc.c_str());
                for (int r = 0; r < NR; ++r) E("            *(amp *)(tile + (sb3 ^ %uu)) = a[%d];", c2[r], perm[r]);
            }
        }
        E("        }");
        E("        __syncthreads();");
    }
    // ---- store phase
    if (!direct_store) {
    E("        {");
    if (scale_at_store) E("            const real sc = *s_scale;");
    for (uint32_t i = 0; i < NU; ++i) {
        if (!scale_at_store) E("            *(unit16 *)(gptr + %lluull) = *(const unit16 *)(tile + (ld_off ^ %uu));", (unsigned long long)hi[i], ci[i]);
        else if (prec == 0)
            E("            { float4 v = *(const float4 *)(tile + (ld_off ^ %uu)); v.x *= sc; v.y *= sc; v.z *= sc; v.w *= sc; *(float4 *)(gptr + %lluull) = v; }", ci[i], (unsigned long long)hi[i]);
        else
            E("            { double2 v = *(const double2 *)(tile + (ld_off ^ %uu)); v.x *= sc; v.y *= sc; *(double2 *)(gptr + %lluull) = v; }", ci[i], (unsigned long long)hi[i]);
    }
    E("        }");
    E("        __syncthreads();   // the tile buffer is reused by the next work item");
    }
    E("    }");
    E("}");
    {   // arithmetic the block needs per amplitude (ALU roofline): rotations 2, every table / phase factor 4
        double ops = 0.0;
        for (int s2 = s_first; s2 < ns; ++s2)
            for (int item : stage_items[s2]) {
                if (item >= 0) { if (p.mops[item].kind == MOP_RY) ops += 2.0; continue; }
                const SegInfo &si = segs[-item - 1];
                const bool any_ph = si.has_phth || si.has_tc || si.has_tm;
                if (si.nlo > 0 || any_ph) ops += 4.0;
                if (si.nhi > 0) ops += 4.0;
            }
        out.fma_ops_per_amp = ops;
    }
    out.name = name;
    out.source.swap(E.s);
    out.smem_bytes = sm;
    out.threads = NT;
    out.tiles_log2 = n - k;
    return true;
}

}  // namespace gv

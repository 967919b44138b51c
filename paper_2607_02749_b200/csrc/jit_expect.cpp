// jit_expect.cpp -- generator of the schedule-specialised expectation-pass kernels (see jit.h).  Pure host C++.
//
// One kernel per read-only pass over the state (Eq. 4, 6, 12: PAPER.md:135, 150, 216).  A thread
// block works through consecutive (statevector, tile) items.  Per item: the tile arrives in shared memory by 16-byte
// cp.async copies (same swizzled layout as the gate kernels), the tables of the groups whose terms carry Z / Y on
// qubits outside the tile are refreshed, then every flip-mask group of the pass is evaluated with literal addresses:
//   diagonal part   sum_x |psi_x|^2 E(x) over the thread's 16-byte units (first pass only);
//   clusters        (planner: groups whose flip mask and in-tile z bits fit R local bits) the thread holds the 2^R
//                   amplitudes of those bits; per pair (x, x^m), x with the pivot bit clear,
//                   Re(conj(psi[x^m]) W(x) psi[x]) = a . (b.x (Wx,-Wy) + b.y (Wy,Wx)),  a = psi[x], b = psi[x^m]:
//                   three packed operations per pair, W from a broadcast table read;
//   table groups    W depends on thread bits only, constant over the thread's 2^L pairs:
//                   Re(W sum conj(b) a) with two packed operations per pair;
//   direct groups   (very wide terms) W summed term by term.
// Tables: W_g(e) = sum_k c_k i^{nY_k} (-1)^{popcount(e & zu_k)} over the group's table index e.  The part of the terms
// with all Z / Y inside the tile is built on the host.  A term with z bits outside the tile has a sign that depends on
// the tile: per tile, D_p = sum of those terms' signed coefficients per distinct index pattern p (one thread per
// pattern), then one warp per group turns D into sum_p D_p (-1)^{p.e} by Walsh-Hadamard butterflies: cost
// (terms + E log E) per group and tile instead of (terms x E).
#include <algorithm>
#include <cstring>
#include <map>

#include "jit.h"
#include "jit_internal.h"

namespace gv {
namespace {

struct GInfo {
    int mode = 0;                 // 0 table (lookup), 1 cluster (register stage), 2 direct
    uint32_t E = 0;               // table entries
    uint32_t tab_off = 0;         // byte offset of the final table in shared memory
    uint32_t wst_off = 0;         // entry offset of the static table in the pass's global array
    bool dyn = false;
    uint32_t pat_begin = 0, pat_end = 0;
    std::vector<uint32_t> pat_keys; // index pattern (z bits inside the group's index bits) of each of its patterns
    std::vector<double> wr, wi;   // static table (host copy)
    uint32_t zmask = 0;           // index bits any term of the group looks at
};

}  // namespace

bool jit_expect_supported(const ExpectPlan &plan, int n, int prec, std::string &why)
{
    const int K = prec == 0 ? 13 : 12;
    if (plan.k != K || n < K) { why = "tile size differs from the specialised kernels"; return false; }
    if (plan.passes.empty()) { why = "no pass"; return false; }
    return true;
}

bool jit_expect_generate(const ExpectPlan &plan, int n, int prec, int pi, JitExpectData &data, JitBlock &out, std::string &err)
{
    if (pi < 0 || (size_t)pi >= plan.passes.size()) { err = "jit: bad pass"; return false; }
    const DPass &P = plan.passes[pi];
    Geo g;
    g.k = P.k; g.lv = prec == 0 ? 1 : 0; g.prec = prec;
    const int k = g.k;
    const int TBITS = 8;                    // 256 threads
    const int RS = k - TBITS;               // bits a thread holds: 5 (complex64) / 4 (complex128)
    g.R = RS; g.TB = TBITS;
    const uint32_t NT = 256, NR = 1u << RS;
    const int V = 1 << g.lv;
    const uint32_t NU = (1u << k) / V / NT;
    const uint32_t AB = prec == 0 ? 8 : 16;
    const char *TT = prec == 0 ? "float" : "double";
    if (NU != 16) { err = "jit: unsupported geometry"; return false; }
    Block B; memset(&B, 0, sizeof B);       // tile description in the gate generator's terms
    B.k = P.k; B.n_runs = P.n_runs; memcpy(B.runs, P.runs, sizeof B.runs);
    auto scatter = [&](uint32_t j) { uint64_t x = 0; for (int r = 0; r < B.n_runs; ++r) x |= (uint64_t)((j >> B.runs[r].lpos) & ((1u << B.runs[r].len) - 1u)) << B.runs[r].gpos; return x; };

    // ---- groups: tables, static parts, dynamic patterns
    const uint32_t g0 = P.group_begin, g1 = P.group_end;
    std::vector<GInfo> gi(g1 - g0);
    uint32_t sm = 0;
    auto take = [&](uint32_t bytes) { const uint32_t o = sm; sm = (sm + bytes + 15u) & ~15u; return o; };
    const uint32_t o_tile = take((uint32_t)AB << k);
    const size_t wst_base = data.wst.size() / 2;
    const size_t pat_base = data.pats.size();
    const size_t term_base = data.terms.size();   // the tile-dependent terms of this pass follow, pattern after pattern
    for (uint32_t q = g0; q < g1; ++q) {
        const DGroup &dg = plan.groups[q];
        GInfo &G = gi[q - g0];
        G.mode = dg.rs ? 1 : (dg.direct ? 2 : 0);
        if (G.mode == 2) continue;
        G.E = 1u << dg.ubits;
        G.dyn = dg.dyn_end > dg.term_begin;
        // clusters: 16-byte entries, and only when a term depends on the tile (otherwise W is a literal in the code)
        if (G.mode == 0) G.tab_off = take(G.E * AB);
        else if (G.dyn) G.tab_off = take(G.E * 16u);
        G.wst_off = (uint32_t)(data.wst.size() / 2 - wst_base);
        for (uint32_t e = 0; e < G.E; ++e) {   // static part (terms with every Z / Y inside the tile)
            double wr = 0.0, wi = 0.0;
            for (uint32_t t = dg.dyn_end; t < dg.term_end; ++t) {
                const DTerm &tm = plan.terms[t];
                const int par = __builtin_popcount(e & tm.zu) & 1;
                wr += par ? -tm.cr : tm.cr; wi += par ? -tm.ci : tm.ci;
            }
            data.wst.push_back(wr); data.wst.push_back(wi);
            G.wr.push_back(wr); G.wi.push_back(wi);
        }
        for (uint32_t t = dg.term_begin; t < dg.term_end; ++t) G.zmask |= plan.terms[t].zu & (G.E - 1u);
        if (G.dyn) {   // tile-dependent terms by index pattern, input order inside a pattern (deterministic sums)
            std::map<uint32_t, std::vector<uint32_t>> by_pat;
            for (uint32_t t = dg.term_begin; t < dg.dyn_end; ++t) by_pat[plan.terms[t].zu & (G.E - 1u)].push_back(t);
            G.pat_begin = (uint32_t)(data.pats.size() - pat_base);
            for (auto &kv : by_pat) {
                JitExpectData::Pat pt;
                pt.dst = kv.first;
                G.pat_keys.push_back(kv.first);
                pt.begin = (uint32_t)data.terms.size();
                for (uint32_t t : kv.second) {
                    const DTerm &tm = plan.terms[t];
                    data.terms.push_back(JitExpectData::Term{tm.cr, tm.ci, tm.zout, 0});
                }
                pt.end = (uint32_t)data.terms.size(); pt.pad = 0;
                data.pats.push_back(pt);
            }
            G.pat_end = (uint32_t)(data.pats.size() - pat_base);
        }
    }
    const uint32_t n_pats = (uint32_t)(data.pats.size() - pat_base);
    const uint32_t o_red = take(64 * 8);
    const uint32_t o_psum = take((n_pats ? n_pats : 1u) * AB);   // per-tile pattern sums S_p
    const uint32_t n_pterms = (uint32_t)(data.terms.size() - term_base);
    const uint32_t o_sv = take((n_pterms ? n_pterms : 1u) * 16u);     // per-tile signed coefficients of those terms (fp64 pairs)
    bool any_dyn = false;
    for (const GInfo &G : gi) any_dyn = any_dyn || G.dyn;
    // The pass's tile-dependent terms and index patterns do not change from tile to tile: staged in shared memory once per
    // thread block when that keeps two thread blocks on an SM (else read from global memory per tile).  With one statevector
    // per tile (configs 5a / 5b) the table set-up is on every work item's critical path, and the two dependent global loads
    // (term, then pattern) were a quarter of a pass.
    constexpr uint32_t SMEM_TWO_BLOCKS = (233472u / 2u) - 1024u;
    bool staged = false;
    uint32_t o_terms = 0, o_pats = 0;
    if (any_dyn && n_pterms && n_pats) {
        const uint32_t before = sm;
        o_terms = take(n_pterms * 24u);
        o_pats = take(n_pats * 16u);
        if (sm <= SMEM_TWO_BLOCKS || before > SMEM_TWO_BLOCKS) staged = true;
        else sm = before;
    }
    data.pass_wst_off.push_back((uint32_t)wst_base);
    data.pass_pat_off.push_back((uint32_t)pat_base);
    data.pass_pat_cnt.push_back(n_pats);
    if (sm > 220u * 1024u) { err = "jit: expectation pass needs too much shared memory"; return false; }

    double ops_per_thread = 0.0;   // FP lane operations per thread and tile (ALU roofline)
    char name[64];
    snprintf(name, sizeof name, "gvqe_expect_%d_%s", pi, prec == 0 ? "c64" : "c128");
    Emit E;
    E("// generated by libgvqe (jit_expect.cpp): expectation pass %d of %zu, n = %d, k = %d, %s; %u groups, %u tile-dependent patterns",
      pi, plan.passes.size(), n, k, prec == 0 ? "complex64" : "complex128", g1 - g0, n_pats);
    emit_common_prelude(E, prec, g.lv);
    E("typedef %s tabt;", TT);
    E("struct __align__(16) Pat { unsigned dst, begin, end, pad; };");
    E("struct __align__(32) Term { double cr, ci; u64 zout, pad; };");
    E("struct __align__(8) TermS { double cr, ci; u64 zout; };   // a term as staged in shared memory");
    if (prec == 0) {
        E("struct __align__(16) tw4 { float x, y, z, w; };   // (Wx, -Wy, Wy, Wx)");
        E("__device__ __forceinline__ tw4 twfmt(amp w) { tw4 t; t.x = w.x; t.y = -w.y; t.z = w.y; t.w = w.x; return t; }");
        // a . (b.x (Wx,-Wy) + b.y (Wy,Wx)) accumulated component-wise
        E("__device__ __forceinline__ void pairw(amp &acc, amp a, amp b, tw4 t) { const amp be = __ffma2_rn(MK(b.y, b.y), MK(t.z, t.w), __fmul2_rn(MK(b.x, b.x), MK(t.x, t.y))); acc = __ffma2_rn(a, be, acc); }");
        E("__device__ __forceinline__ void pairs(amp &s1, amp &s2, amp a, amp b) { s1 = __ffma2_rn(MK(b.x, b.x), a, s1); s2 = __ffma2_rn(MK(b.y, b.y), a, s2); }");
        // conj(b) a = (b.x a.x + b.y a.y, b.x a.y - b.y a.x)
        E("__device__ __forceinline__ amp cjmul(amp a, amp b) { const amp p = __fmul2_rn(MK(b.x, b.x), a), q = __fmul2_rn(MK(b.y, b.y), a); return MK(p.x + q.y, p.y - q.x); }");
        E("__device__ __forceinline__ amp cadd(amp a, amp b) { return __fadd2_rn(a, b); }");
        E("__device__ __forceinline__ amp csub(amp a, amp b) { return MK(a.x - b.x, a.y - b.y); }");
        E("__device__ __forceinline__ amp cneg(amp a) { return MK(-a.x, -a.y); }");
        // sign flip by a sign-bit mask (0 or 0x80000000)
        E("__device__ __forceinline__ amp sflip(amp a, unsigned sb) { return MK(__uint_as_float(__float_as_uint(a.x) ^ sb), __uint_as_float(__float_as_uint(a.y) ^ sb)); }");
        // W known when the kernel is generated (constant bank, read through the uniform path -- no shared-memory traffic):
        // complex W three packed operations, real W two, imaginary W three scalar ones
        E("#define PAIRC(acc, a, b, t) { const amp be = __ffma2_rn(MK((b).y, (b).y), MK((t).z, (t).w), __fmul2_rn(MK((b).x, (b).x), MK((t).x, (t).y))); acc = __ffma2_rn((a), be, acc); }");
        E("#define PAIRR(acc, a, b, t) { acc = __ffma2_rn((a), __fmul2_rn((b), MK((t).x, (t).x)), acc); }");
        E("#define PAIRI(acci, a, b, t) { acci = fmaf((t).z, fmaf(-(a).y, (b).x, (a).x * (b).y), acci); }");
        // shared-W forms: sums of a.b (real W), of the cross products (imaginary W), of b.x a and b.y a (complex W)
        E("#define DOT0(a, b) __fmul2_rn((a), (b))");
        E("#define DOT(p, a, b) { p = __ffma2_rn((a), (b), p); }");
        E("#define WRE(acc, p, t) { acc = __ffma2_rn(p, MK((t).x, (t).x), acc); }");
        E("#define CRS0(a, b) fmaf(-(a).y, (b).x, (a).x * (b).y)");
        E("#define CRS(p, a, b) { p = fmaf(-(a).y, (b).x, fmaf((a).x, (b).y, p)); }");
        E("#define WIM(acci, p, t) { acci = fmaf((t).z, p, acci); }");
        E("#define PAIRS0(p1, p2, a, b) { p1 = __fmul2_rn(MK((b).x, (b).x), (a)); p2 = __fmul2_rn(MK((b).y, (b).y), (a)); }");
        E("#define WCX(acc, p1, p2, t) { acc = __ffma2_rn(p1, MK((t).x, (t).y), acc); acc = __ffma2_rn(p2, MK((t).z, (t).w), acc); }");
    } else {
        E("typedef double2 tw4;");
        E("__device__ __forceinline__ tw4 twfmt(amp w) { return w; }");
        E("__device__ __forceinline__ void pairw(amp &acc, amp a, amp b, tw4 t) { const double br = fma(t.y, b.y, t.x * b.x), bi = fma(-t.y, b.x, t.x * b.y); acc.x = fma(a.x, br, acc.x); acc.y = fma(a.y, bi, acc.y); }");
        E("__device__ __forceinline__ void pairs(amp &s1, amp &s2, amp a, amp b) { s1.x = fma(b.x, a.x, s1.x); s1.y = fma(b.x, a.y, s1.y); s2.x = fma(b.y, a.x, s2.x); s2.y = fma(b.y, a.y, s2.y); }");
        E("__device__ __forceinline__ amp cjmul(amp a, amp b) { return MK(fma(b.y, a.y, b.x * a.x), fma(-b.y, a.x, b.x * a.y)); }");
        E("__device__ __forceinline__ amp cadd(amp a, amp b) { return MK(a.x + b.x, a.y + b.y); }");
        E("__device__ __forceinline__ amp csub(amp a, amp b) { return MK(a.x - b.x, a.y - b.y); }");
        E("__device__ __forceinline__ amp cneg(amp a) { return MK(-a.x, -a.y); }");
        E("__device__ __forceinline__ amp sflip(amp a, unsigned sb) { return MK(__hiloint2double(__double2hiint(a.x) ^ (int)sb, __double2loint(a.x)), __hiloint2double(__double2hiint(a.y) ^ (int)sb, __double2loint(a.y))); }");
        E("#define PAIRC(acc, a, b, t) { const double br = fma((t).y, (b).y, (t).x * (b).x), bi = fma(-(t).y, (b).x, (t).x * (b).y); acc.x = fma((a).x, br, acc.x); acc.y = fma((a).y, bi, acc.y); }");
        E("#define PAIRR(acc, a, b, t) { acc.x = fma((a).x * (t).x, (b).x, acc.x); acc.y = fma((a).y * (t).x, (b).y, acc.y); }");
        E("#define PAIRI(acci, a, b, t) { acci = fma((t).y, fma(-(a).y, (b).x, (a).x * (b).y), acci); }");
        E("#define DOT0(a, b) MK((a).x * (b).x, (a).y * (b).y)");
        E("#define DOT(p, a, b) { p.x = fma((a).x, (b).x, p.x); p.y = fma((a).y, (b).y, p.y); }");
        E("#define WRE(acc, p, t) { acc.x = fma(p.x, (t).x, acc.x); acc.y = fma(p.y, (t).x, acc.y); }");
        E("#define CRS0(a, b) fma(-(a).y, (b).x, (a).x * (b).y)");
        E("#define CRS(p, a, b) { p = fma(-(a).y, (b).x, fma((a).x, (b).y, p)); }");
        E("#define WIM(acci, p, t) { acci = fma((t).y, p, acci); }");
        E("#define PAIRS0(p1, p2, a, b) { p1 = MK((b).x * (a).x, (b).x * (a).y); p2 = MK((b).y * (a).x, (b).y * (a).y); }");
        E("#define WCX(acc, p1, p2, t) { acc.x = fma((t).x, p1.x + p2.y, acc.x); acc.y = fma((t).y, p2.x - p1.y, acc.y); }");
    }
    // W of the cluster groups without tile-dependent terms: entries (Wx, -Wy, Wy, Wx) (complex128: (Wx, Wy)) in constant memory
    std::vector<std::pair<double, double>> wconst;
    std::map<std::pair<double, double>, uint32_t> wconst_ix;
    auto const_index = [&](double wx, double wy) {
        const std::pair<double, double> key(wx, wy);
        auto it = wconst_ix.find(key);
        if (it != wconst_ix.end()) return it->second;
        const uint32_t ix = (uint32_t)wconst.size();
        wconst.push_back(key); wconst_ix[key] = ix;
        return ix;
    };
    for (uint32_t q = g0; q < g1; ++q) {
        const GInfo &G = gi[q - g0];
        if (G.mode != 1 || G.dyn) continue;
        for (uint32_t e = 0; e < G.E; ++e) {
            const double wx = prec == 0 ? (double)(float)G.wr[e] : G.wr[e], wy = prec == 0 ? (double)(float)G.wi[e] : G.wi[e];
            if (wx != 0.0 || wy != 0.0) const_index(wx, wy);
        }
    }
    if (!wconst.empty()) {
        if (wconst.size() * 16 > 60000) { err = "jit: too many constant table entries"; return false; }
        std::string t = std::string("__constant__ ") + (prec == 0 ? "tw4" : "double2") + " WC[" + std::to_string(wconst.size()) + "] = {";
        auto lit = [&](double v) {   // a floating literal that reads back to exactly v
            char b2[48];
            snprintf(b2, sizeof b2, prec == 0 ? "%.9g" : "%.17g", v);
            std::string x = b2;
            if (x.find_first_of(".en") == std::string::npos) x += ".0";
            return prec == 0 ? x + "f" : x;
        };
        for (auto &w : wconst) {
            if (prec == 0) t += "{" + lit(w.first) + ", " + lit(-w.second) + ", " + lit(w.second) + ", " + lit(w.first) + "}, ";
            else t += "{" + lit(w.first) + ", " + lit(w.second) + "}, ";
        }
        t += "};";
        E("%s", t.c_str());
    }
    E("");
    E("extern \"C\" __global__ void __launch_bounds__(%u, 2) %s(const amp *states, u64 stride, const tabt *table, const amp *wst, const Pat *pats, const Term *terms,", NT, name);
    E("        double *partial, unsigned slots_per_b, unsigned slot_off, int nb, int per_cta)");
    E("{");
    E("    extern __shared__ __align__(128) unsigned char smem[];");
    E("    unsigned char *tile = smem + %u;", o_tile);
    E("    double *red = (double *)(smem + %u);", o_red);
    E("    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;");
    E("    (void)lane; (void)warp; (void)pats; (void)terms; (void)table;");
    // static tables of the groups without tile-dependent terms: once per thread block
    for (uint32_t q = g0; q < g1; ++q) {
        const GInfo &G = gi[q - g0];
        if (G.mode != 0 || G.dyn) continue;
        E("    for (unsigned e = tid; e < %uu; e += %uu) ((amp *)(smem + %u))[e] = wst[%u + e];", G.E, NT, G.tab_off, G.wst_off);
    }
    if (staged) {
        E("    for (unsigned t = tid; t < %uu; t += %uu) { const Term tm = terms[%zuu + t]; TermS ts; ts.cr = tm.cr; ts.ci = tm.ci; ts.zout = tm.zout; ((TermS *)(smem + %u))[t] = ts; }", n_pterms, NT, term_base, o_terms);
        E("    for (unsigned i = tid; i < %uu; i += %uu) ((Pat *)(smem + %u))[i] = pats[i];", n_pats, NT, o_pats);
        E("    __syncthreads();");
    }
    E("    const unsigned ld_off = OFF(tid << %d);", g.lv);
    {
        std::string sx = "    const u64 ld_x = 0ull";
        for (int r = 0; r < B.n_runs; ++r) {
            const int lp = B.runs[r].lpos, len = B.runs[r].len, gp = B.runs[r].gpos;
            int lo = lp - g.lv, hi = lp + len - g.lv;
            if (lo < 0) lo = 0;
            if (hi > TBITS) hi = TBITS;
            if (hi <= lo) continue;
            char b[128];
            snprintf(b, sizeof b, " | ((u64)((tid >> %d) & %uu) << %d)", lo, (1u << (hi - lo)) - 1u, gp + (lo + g.lv - lp));
            sx += b;
        }
        sx += ";";
        E("%s", sx.c_str());
    }
    E("    const u64 total = (u64)nb << %d;", n - k);
    E("    const u64 w_begin = (u64)blockIdx.x * (u64)per_cta;");
    E("    const u64 w_end = w_begin + (u64)per_cta < total ? w_begin + (u64)per_cta : total;");
    // work items in (tile, statevector) order: the diagonal table's tile stays in L2 for the rows that follow, and the
    // tile-dependent tables (which do not depend on the state) are built once per tile
    if (any_dyn) E("    u64 cur_tile = ~0ull;");
    E("    for (u64 w = w_begin; w < w_end; ++w) {");
    E("        const u64 tile_id = w / (u64)nb;");
    E("        const int b = (int)(w - tile_id * (u64)nb);");
    E("        const amp *state = states + (u64)b * stride;");
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
    E("        const amp *gptr = state + (xbase | ld_x);");
    std::vector<uint64_t> hi(NU);
    std::vector<uint32_t> ci(NU);
    for (uint32_t i = 0; i < NU; ++i) {
        const uint32_t j = (NT * i) << g.lv;
        hi[i] = scatter(j); ci[i] = g.off(j);
    }
    for (uint32_t i = 0; i < NU; ++i) E("        cp16(tile + (ld_off ^ %uu), gptr + %lluull);", ci[i], (unsigned long long)hi[i]);
    if (P.with_diag) {   // diagonal energies of the thread's units: issued under the tile copies
        E("        const tabt *tptr = table + (xbase | ld_x);");
        if (prec == 0) { for (uint32_t i = 0; i < NU; ++i) E("        const float2 tv%u = *(const float2 *)(tptr + %lluull);", i, (unsigned long long)hi[i]); }
        else { for (uint32_t i = 0; i < NU; ++i) E("        const double tv%u = tptr[%lluull];", i, (unsigned long long)hi[i]); }
    }
    // ---- tile-dependent tables
    if (any_dyn) {
        // Tile-dependent tables, once per tile: T[e] = static[e] + sum over the group's index patterns p of S_p (-1)^{p.e},
        // S_p = the signed sum of the pattern's terms for this tile.  A group has few patterns (its terms' z masks inside
        // the index bits), so the sum is taken pattern by pattern instead of by a full Walsh-Hadamard transform: lane l
        // holds the entries l + 32 i (the LOW five index bits are the lane: neighbouring lanes read and write neighbouring
        // entries -- with the entries [l EP, (l + 1) EP) per lane every store of a warp fell into the same banks, 32
        // wavefronts per STS.128); a pattern's sign over the lane bits is one parity, its S_p goes to the accumulator of
        // its in-lane part (the high index bits), and a register Walsh-Hadamard over the in-lane bits (skipping what is
        // known to be zero when the kernel is generated) finishes the entries.  No shuffles, no shared-memory butterflies.
        E("        if (tile_id != cur_tile) {");
        E("        cur_tile = tile_id;");
        E("        for (unsigned t = tid; t < %uu; t += %uu) {   // one thread per term: its coefficient with this tile's sign", n_pterms, NT);
        if (staged) E("            const TermS tm = ((const TermS *)(smem + %u))[t];", o_terms);
        else E("            const Term tm = terms[%zuu + t];", term_base);
        E("            const bool neg = __popcll(xbase & tm.zout) & 1;");
        E("            ((double2 *)(smem + %u))[t] = make_double2(neg ? -tm.cr : tm.cr, neg ? -tm.ci : tm.ci);", o_sv);
        E("        }");
        E("        __syncthreads();");
        E("        for (unsigned i = tid; i < %uu; i += %uu) {   // one thread per (group, index pattern): sum of its terms, in their order", n_pats, NT);
        if (staged) E("            const Pat p = ((const Pat *)(smem + %u))[i];", o_pats);
        else E("            const Pat p = pats[i];");
        E("            double sr = 0.0, si = 0.0;");
        E("            for (unsigned t = p.begin; t < p.end; ++t) { const double2 v = ((const double2 *)(smem + %u))[t - %zuu]; sr += v.x; si += v.y; }", o_sv, term_base);
        E("            ((amp *)(smem + %u))[i] = MK((real)sr, (real)si);", o_psum);
        E("        }");
        E("        __syncthreads();");
        int wi = 0;
        for (uint32_t q = g0; q < g1; ++q) {
            const GInfo &G = gi[q - g0];
            if (!G.dyn) continue;
            const DGroup &dg = plan.groups[q];
            const int ub = (int)dg.ubits, epl = ub > 5 ? ub - 5 : 0, EP = 1 << epl, nlb = ub - epl;
            E("        if (warp == %du%s) {   // group %u: %zu patterns over %d index bits", wi % 8, nlb < 5 ? (std::string(" && lane < ") + std::to_string(1u << nlb) + "u").c_str() : "", q - g0, G.pat_keys.size(), ub);
            E("            const unsigned e0 = lane;");
            E("            amp st[%d], A[%d];", EP, EP);
            for (int i = 0; i < EP; ++i) E("            st[%d] = wst[%u + e0 + %d];", i, G.wst_off, i << nlb);
            std::vector<char> nz((size_t)EP, 0);
            for (size_t j = 0; j < G.pat_keys.size(); ++j) {
                const uint32_t key = G.pat_keys[j], pl = key >> nlb, ph = key & ((1u << nlb) - 1u);
                std::string sx = "((const amp *)(smem + " + std::to_string(o_psum) + "))[" + std::to_string(G.pat_begin + j) + "]";
                if (ph) sx = "sflip(" + sx + ", (unsigned)__popc(lane & " + std::to_string(ph) + "u) << 31)";
                if (nz[pl]) E("            A[%u] = cadd(A[%u], %s);", pl, pl, sx.c_str());
                else { E("            A[%u] = %s;", pl, sx.c_str()); nz[pl] = 1; }
            }
            for (int bit = 0; bit < epl; ++bit)
                for (int i = 0; i < EP; ++i) {
                    if (i >> bit & 1) continue;
                    const int j = i | (1 << bit);
                    if (nz[i] && nz[j]) E("            { const amp u = A[%d], v = A[%d]; A[%d] = cadd(u, v); A[%d] = csub(u, v); }", i, j, i, j);
                    else if (nz[i]) { E("            A[%d] = A[%d];", j, i); nz[j] = 1; }
                    else if (nz[j]) { E("            A[%d] = A[%d]; A[%d] = cneg(A[%d]);", i, j, j, j); nz[i] = 1; }
                }
            for (int i = 0; i < EP; ++i) {
                std::string v = nz[i] ? "cadd(A[" + std::to_string(i) + "], st[" + std::to_string(i) + "])" : "st[" + std::to_string(i) + "]";
                if (G.mode == 1) E("            ((tw4 *)(smem + %u))[e0 + %d] = twfmt(%s);", G.tab_off, i << nlb, v.c_str());
                else E("            ((amp *)(smem + %u))[e0 + %d] = %s;", G.tab_off, i << nlb, v.c_str());
            }
            E("        }");
            ++wi;
        }
        E("        }");
    }
    E("        cp_wait();");
    E("        __syncthreads();");
    E("        double acc = 0.0;");
    // ---- diagonal part
    if (P.with_diag) {
        E("        {   // sum |psi|^2 E(x) over the thread's units");
        E("            real da = (real)0;");
        for (uint32_t i = 0; i < NU; ++i) {
            if (prec == 0) {
                E("            { const float4 v = *(const float4 *)(tile + (ld_off ^ %uu)); da = fmaf(fmaf(v.x, v.x, v.y * v.y), tv%u.x, da); da = fmaf(fmaf(v.z, v.z, v.w * v.w), tv%u.y, da); }", ci[i], i, i);
            } else {
                E("            { const double2 v = *(const double2 *)(tile + (ld_off ^ %uu)); da = fma(fma(v.x, v.x, v.y * v.y), tv%u, da); }", ci[i], i);
            }
        }
        E("            acc += (double)da;");
        E("        }");
    }
    const uint32_t LOMASK = 0x70u;
    // ---- clusters
    std::map<int, std::vector<uint32_t>> clusters;   // rs_id -> groups
    for (uint32_t q = g0; q < g1; ++q) if (gi[q - g0].mode == 1) clusters[plan.groups[q].rs_id].push_back(q);
    for (auto &cl : clusters) {
        const DRs &rs = plan.rss[(size_t)cl.first];
        int tb[16];
        choose_thread_bits_for(g, rs.regbit, RS, tb);
        const bool wide = (g.lv == 1 && rs.regbit[0] == 0);
        uint32_t cr[32];
        bool vused[8] = {false};
        for (uint32_t r = 0; r < NR; ++r) {
            uint32_t j = 0;
            for (int b = 0; b < RS; ++b) if (r >> b & 1) j |= 1u << rs.regbit[b];
            cr[r] = g.off(j);
            vused[(cr[r] & LOMASK) >> 4] = true;
        }
        E("        {   // ---- cluster %d: %zu groups from registers", cl.first, cl.second.size());
        emit_deposit(E, "            ", "jt", tb, TBITS);
        E("            const unsigned sb = OFF(jt);");
        for (int v = 0; v < 8; ++v) if (vused[v]) E("            const unsigned char *const pv%d = tile + (sb ^ %uu);", v, (uint32_t)v << 4);
        E("            amp a[%u];", NR);
        if (wide) {
            for (uint32_t r = 0; r < NR; r += 2)
                E("            { const float4 v = *(const float4 *)(pv%u + %uu); a[%u] = MK(v.x, v.y); a[%u] = MK(v.z, v.w); }", (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK, r, r + 1);
        } else {
            for (uint32_t r = 0; r < NR; ++r) E("            a[%u] = *(const amp *)(pv%u + %uu);", r, (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK);
        }
        for (uint32_t q : cl.second) {
            const DGroup &dg = plan.groups[q];
            const GInfo &G = gi[q - g0];
            const uint32_t mr = dg.m_r;
            int pv = 31 - __builtin_clz(mr);
            E("            {   // group %u: flip mask over the slots %u%s", q - g0, mr, G.dyn ? " (table refreshed per tile)" : " (W literal)");
            E("                amp s = MK((real)0, (real)0);");
            if (G.dyn) {
                E("                const tw4 *W = (const tw4 *)(smem + %u);", G.tab_off);
                for (uint32_t r = 0; r < NR; ++r) {
                    if (r >> pv & 1) continue;
                    E("                pairw(s, a[%u], a[%u], W[%u]);", r, r ^ mr, r & G.zmask);   // only the index bits a term looks at: equal reads merge
                    ops_per_thread += 6.0;
                }
                E("                acc += 2.0 * (double)(s.x + s.y);");
            } else {
                E("                real si = (real)0; amp s2 = MK((real)0, (real)0);");
                // pairs whose W is the same number (index bits the group's terms do not read, equal table entries) are
                // summed first and multiplied by W once
                std::map<uint32_t, std::vector<uint32_t>> by_w;
                std::vector<uint32_t> w_order;
                for (uint32_t r = 0; r < NR; ++r) {
                    if (r >> pv & 1) continue;
                    const double wx = prec == 0 ? (double)(float)G.wr[r] : G.wr[r], wy = prec == 0 ? (double)(float)G.wi[r] : G.wi[r];
                    if (wx == 0.0 && wy == 0.0) continue;
                    const uint32_t ix = const_index(wx, wy);
                    if (!by_w.count(ix)) w_order.push_back(ix);
                    by_w[ix].push_back(r);
                }
                int nem = 0;
                for (uint32_t ix : w_order) {
                    const std::vector<uint32_t> &rs = by_w[ix];
                    const double wx = wconst[ix].first, wy = wconst[ix].second;
                    const char *sa = (nem++ & 1) ? "s2" : "s";   // two accumulation chains
                    if (rs.size() == 1) {
                        const uint32_t r = rs[0];
                        if (wy == 0.0) { E("                PAIRR(%s, a[%u], a[%u], WC[%u])", sa, r, r ^ mr, ix); ops_per_thread += 4.0; }
                        else if (wx == 0.0) { E("                PAIRI(si, a[%u], a[%u], WC[%u])", r, r ^ mr, ix); ops_per_thread += 3.0; }
                        else { E("                PAIRC(%s, a[%u], a[%u], WC[%u])", sa, r, r ^ mr, ix); ops_per_thread += 6.0; }
                        continue;
                    }
                    if (wy == 0.0) {
                        E("                { amp p = DOT0(a[%u], a[%u]);", rs[0], rs[0] ^ mr);
                        for (size_t i = 1; i < rs.size(); ++i) E("                  DOT(p, a[%u], a[%u])", rs[i], rs[i] ^ mr);
                        E("                  WRE(%s, p, WC[%u]) }", sa, ix);
                        ops_per_thread += 2.0 * (double)rs.size() + 2.0;
                    } else if (wx == 0.0) {
                        E("                { real p = CRS0(a[%u], a[%u]);", rs[0], rs[0] ^ mr);
                        for (size_t i = 1; i < rs.size(); ++i) E("                  CRS(p, a[%u], a[%u])", rs[i], rs[i] ^ mr);
                        E("                  WIM(si, p, WC[%u]) }", ix);
                        ops_per_thread += 2.0 * (double)rs.size() + 1.0;
                    } else {
                        E("                { amp p1, p2; PAIRS0(p1, p2, a[%u], a[%u])", rs[0], rs[0] ^ mr);
                        for (size_t i = 1; i < rs.size(); ++i) E("                  pairs(p1, p2, a[%u], a[%u]);", rs[i], rs[i] ^ mr);
                        E("                  WCX(%s, p1, p2, WC[%u]) }", sa, ix);
                        ops_per_thread += 4.0 * (double)rs.size() + 4.0;
                    }
                }
                E("                acc += 2.0 * (double)((s.x + s.y) + (s2.x + s2.y) + si);");
            }
            E("            }");
        }
        E("        }");
    }
    // ---- table groups: all slices of one flip mask share the thread's pair products
    // A flip mask whose terms look at more in-tile z bits than a table can index was cut into slices by the planner
    // (Eq. 12: any partition of the terms).  The amplitudes are read from shared memory ONCE per mask: the thread keeps
    // rho_i = conj(b_i) a_i of its 2^L pairs; a slice whose index bits avoid the loop bits multiplies its W with the sum of
    // all rho_i, one that uses j loop bits with 2^j partial sums.
    std::map<uint32_t, std::vector<uint32_t>> by_mask;
    for (uint32_t q = g0; q < g1; ++q) if (gi[q - g0].mode == 0) by_mask[plan.groups[q].m_loc].push_back(q);
    for (auto &mg : by_mask) {
        const uint32_t m = mg.first;
        const int pivot = 31 - __builtin_clz(m);
        uint32_t Uall = 0;
        for (uint32_t q : mg.second) Uall |= plan.groups[q].uloc;
        // loop bits: outside every slice's index bits when possible, else the bits the fewest slices look at
        uint32_t exmask = 1u << pivot;
        while (__builtin_popcount(exmask) < RS) {
            int best = -1, best_cost = 1 << 30;
            for (int bb = k - 1; bb >= 0; --bb) {
                if (exmask >> bb & 1) continue;
                int cost = 0;
                for (uint32_t q : mg.second) cost += (int)(plan.groups[q].uloc >> bb & 1) * 4;
                cost += (int)(m >> bb & 1);            // prefer bits outside the flip mask
                if (cost < best_cost) { best_cost = cost; best = bb; }
            }
            exmask |= 1u << best;
        }
        uint8_t ex[8]; int ne = 0;
        for (int bb = 0; bb < k; ++bb) if (exmask >> bb & 1) ex[ne++] = (uint8_t)bb;
        int tb[16];
        choose_thread_bits_for(g, ex, RS, tb);
        int pslot = 0;
        for (int i = 0; i < RS; ++i) if (ex[i] == pivot) pslot = i;
        uint32_t mreg = 0;                         // flip mask over the register-like slots
        for (int i = 0; i < RS; ++i) if (m >> ex[i] & 1) mreg |= 1u << i;
        const uint32_t mthr = m & ~exmask;         // flip-mask bits that are thread bits: the partner lives in another thread
        uint32_t cr[32], jr[32];
        for (uint32_t r = 0; r < NR; ++r) {
            uint32_t j = 0;
            for (int bb = 0; bb < RS; ++bb) if (r >> bb & 1) j |= 1u << ex[bb];
            jr[r] = j; cr[r] = g.off(j);
        }
        std::vector<uint32_t> pairs_r;             // register indices with the pivot slot clear
        for (uint32_t r = 0; r < NR; ++r) if (!(r >> pslot & 1)) pairs_r.push_back(r);
        const int np = (int)pairs_r.size();
        E("        {   // ---- flip mask local 0x%x: %zu table slice(s)", m, mg.second.size());
        emit_deposit(E, "            ", "jt", tb, TBITS);
        E("            const unsigned sb = OFF(jt);");
        E("            amp rho[%d];", np);
        const bool wide = (g.lv == 1 && ex[0] == 0 && mthr == 0);
        if (mthr == 0) {   // partners in the same thread
            bool vused[8] = {false};
            for (uint32_t r = 0; r < NR; ++r) vused[(cr[r] & LOMASK) >> 4] = true;
            for (int v = 0; v < 8; ++v) if (vused[v]) E("            const unsigned char *const pv%d = tile + (sb ^ %uu);", v, (uint32_t)v << 4);
            E("            amp a[%u];", NR);
            if (wide) {
                for (uint32_t r = 0; r < NR; r += 2)
                    E("            { const float4 v = *(const float4 *)(pv%u + %uu); a[%u] = MK(v.x, v.y); a[%u] = MK(v.z, v.w); }", (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK, r, r + 1);
            } else {
                for (uint32_t r = 0; r < NR; ++r) E("            a[%u] = *(const amp *)(pv%u + %uu);", r, (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK);
            }
            for (int i = 0; i < np; ++i) E("            rho[%d] = cjmul(a[%u], a[%u]);", i, pairs_r[i], pairs_r[i] ^ mreg);
        } else {
            E("            const unsigned sbm = sb ^ %uu;", g.off(mthr));
            bool vu[8] = {false}, vm[8] = {false};
            for (uint32_t r : pairs_r) { vu[(cr[r] & LOMASK) >> 4] = true; vm[(cr[r ^ mreg] & LOMASK) >> 4] = true; }
            for (int v = 0; v < 8; ++v) if (vu[v]) E("            const unsigned char *const pv%d = tile + (sb ^ %uu);", v, (uint32_t)v << 4);
            for (int v = 0; v < 8; ++v) if (vm[v]) E("            const unsigned char *const pm%d = tile + (sbm ^ %uu);", v, (uint32_t)v << 4);
            for (int i = 0; i < np; ++i) {
                const uint32_t r = pairs_r[i], rb = r ^ mreg;
                E("            rho[%d] = cjmul(*(const amp *)(pv%u + %uu), *(const amp *)(pm%u + %uu));", i, (cr[r] & LOMASK) >> 4, cr[r] & ~LOMASK, (cr[rb] & LOMASK) >> 4, cr[rb] & ~LOMASK);
            }
        }
        ops_per_thread += 6.0 * np;   // conj(b) a: four multiplies and two adds per pair
        E("            real accm = (real)0;");
        for (uint32_t q : mg.second) {
            const DGroup &dg = plan.groups[q];
            const GInfo &G = gi[q - g0];
            const uint32_t U = dg.uloc;
            auto compress_u = [&](uint32_t j) { uint32_t o = 0; int pos = 0; for (int bb = 0; bb < k; ++bb) if (U >> bb & 1) { if (j >> bb & 1) o |= 1u << pos; ++pos; } return o; };
            {   // table index of the thread: the bits of jt at the positions of U, packed
                std::string ux = "            { const unsigned u = 0u";
                int o = 0;
                for (int bb = 0; bb < k; ++bb) if (U >> bb & 1) {
                    if (!(exmask >> bb & 1)) { char b2[64]; snprintf(b2, sizeof b2, " | (((jt >> %d) & 1u) << %d)", bb, o); ux += b2; }
                    ++o;
                }
                E("%s;   // slice %u", ux.c_str(), q - g0);
            }
            E("              const amp *tabp = (const amp *)(smem + %u) + u;", G.tab_off);
            std::map<uint32_t, std::vector<int>> classes;   // index contribution of the loop bits -> pairs
            for (int i = 0; i < np; ++i) classes[compress_u(jr[pairs_r[i]])].push_back(i);
            for (auto &cl : classes) {
                std::string sum = "rho[" + std::to_string(cl.second[0]) + "]";
                E("              { amp t = %s;", sum.c_str());
                for (size_t z = 1; z < cl.second.size(); ++z) E("                t = cadd(t, rho[%d]);", cl.second[z]);
                ops_per_thread += 2.0 * (double)(cl.second.size() - 1) + 2.0;
                E("                const amp wv = tabp[%u]; accm = %s(wv.x, t.x, %s(-wv.y, t.y, accm)); }", cl.first, prec == 0 ? "fmaf" : "fma", prec == 0 ? "fmaf" : "fma");
            }
            E("            }");
        }
        E("            acc += 2.0 * (double)accm;");
        E("        }");
    }
    // ---- direct groups (terms too wide for a table): W summed term by term per pair
    for (uint32_t q = g0; q < g1; ++q) {
        const GInfo &G = gi[q - g0];
        if (G.mode != 2) continue;
        const DGroup &dg = plan.groups[q];
        const int pivot = 31 - __builtin_clz(dg.m_loc);
        E("        {   // ---- group %u, direct", q - g0);
        E("            real part = (real)0;");
        E("            for (unsigned i = tid; i < %uu; i += %uu) {", 1u << (k - 1), NT);
        E("                const unsigned j = ((i >> %d) << %d) | (i & %uu);", pivot, pivot + 1, (1u << pivot) - 1u);
        E("                const amp a = *(const amp *)(tile + OFF(j)), bb = *(const amp *)(tile + OFF(j ^ %uu));", dg.m_loc);
        E("                double wr = 0.0, wi = 0.0;");
        E("                for (unsigned t = %uu; t < %uu; ++t) { const Term tm = terms[t]; const bool neg = (__popcll(xbase & tm.zout) + __popc(j & (unsigned)tm.pad)) & 1; wr += neg ? -tm.cr : tm.cr; wi += neg ? -tm.ci : tm.ci; }",
          (uint32_t)data.terms.size(), (uint32_t)(data.terms.size() + (dg.term_end - dg.term_begin)));
        E("                const real tr = bb.x * a.x + bb.y * a.y, ti = bb.x * a.y - bb.y * a.x;");
        E("                part += (real)wr * tr - (real)wi * ti;");
        E("            }");
        E("            acc += 2.0 * (double)part;");
        E("        }");
        for (uint32_t t = dg.term_begin; t < dg.term_end; ++t) {   // direct terms: local z mask rides in `pad`
            const DTerm &tm = plan.terms[t];
            data.terms.push_back(JitExpectData::Term{tm.cr, tm.ci, tm.zout, (uint64_t)tm.zu});
        }
    }
    // ---- deterministic block sum
    E("        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);");
    // one barrier per work item: it frees the tile and the tables for the next item and publishes the warps' sums, which
    // alternate between two sets of slots (thread 0 has read a set long before it is written again, two items later)
    E("        double *const redw = red + (unsigned)(w & 1ull) * %uu;", NT / 32);
    E("        if (lane == 0) redw[warp] = acc;");
    E("        __syncthreads();");
    E("        if (tid == 0) { double s = 0.0; for (int i = 0; i < %u; ++i) s += redw[i]; partial[(u64)b * slots_per_b + slot_off + tile_id] = s; }", NT / 32);
    E("    }");
    E("}");
    if (P.with_diag) ops_per_thread += 4.0 * NR;   // |psi|^2 E(x): three multiply-adds and one multiply per amplitude
    out.fma_ops_per_amp = ops_per_thread / (double)NR;
    out.name = name;
    out.source.swap(E.s);
    out.smem_bytes = sm;
    out.threads = NT;
    out.tiles_log2 = n - k;
    return true;
}

}  // namespace gv

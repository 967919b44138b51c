// hamiltonian.cpp -- see hamiltonian.h.
#include "hamiltonian.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>

namespace gv {
namespace {

bool finish(Hamiltonian &H, std::string &err)
{
    const uint64_t all = H.n >= 64 ? ~0ull : ((1ull << H.n) - 1);
    H.abs_sum = 0.0;
    std::vector<uint64_t> masks;
    masks.reserve(H.terms.size());
    for (const HostTerm &t : H.terms) {
        if (!std::isfinite(t.c)) { err = "hamiltonian: coefficient is not finite"; return false; }
        if ((t.x | t.z) & ~all) { err = "hamiltonian: mask has bits outside the register"; return false; }
        H.abs_sum += std::fabs(t.c);
        masks.push_back(t.x);
    }
    std::sort(masks.begin(), masks.end());
    masks.erase(std::unique(masks.begin(), masks.end()), masks.end());
    H.group_mask = masks;
    H.group_of_term.resize(H.terms.size());
    for (size_t k = 0; k < H.terms.size(); ++k)
        H.group_of_term[k] = (int32_t)(std::lower_bound(masks.begin(), masks.end(), H.terms[k].x) - masks.begin());
    std::map<uint64_t, double> dz;   // ordered; each entry summed in input order -> deterministic
    for (const HostTerm &t : H.terms) if (t.x == 0) dz[t.z] += t.c;
    H.diag_z.clear(); H.diag_c.clear();
    for (const auto &kv : dz) { H.diag_z.push_back(kv.first); H.diag_c.push_back(kv.second); }
    return true;
}

inline int local_pos(uint64_t T, int q) { return __builtin_popcountll(T & ((1ull << q) - 1)); }

uint32_t compress(uint64_t v, uint64_t T)   // bits of v at the positions of T, packed (software pext)
{
    uint32_t out = 0; int o = 0;
    while (T) {
        const int q = __builtin_ctzll(T);
        if (v >> q & 1) out |= 1u << o;
        ++o; T &= T - 1;
    }
    return out;
}

int runs_of(uint64_t T, Run *runs, int cap)   // returns number of runs (may exceed cap; only cap are written)
{
    int nr = 0, lp = 0;
    for (int q = 0; q < 64;) {
        if (!(T >> q & 1)) { ++q; continue; }
        int len = 0; while (q + len < 64 && (T >> (q + len) & 1)) ++len;
        if (nr < cap) { runs[nr].lpos = (uint8_t)lp; runs[nr].gpos = (uint8_t)q; runs[nr].len = (uint8_t)len; runs[nr].pad = 0; }
        ++nr; lp += len; q += len;
    }
    return nr;
}

// fill `Thi` (bits >= f) up to `h` bits: first next to bits already chosen (or next to the low block), then anywhere
uint64_t fill_bits(uint64_t Thi, int n, int f, int h)
{
    int cnt = __builtin_popcountll(Thi);
    const uint64_t low = f ? ((1ull << f) - 1) : 0;
    for (int pass = 0; pass < 2 && cnt < h; ++pass) {
        bool grew = true;
        while (grew && cnt < h) {
            grew = false;
            for (int q = f; q < n && cnt < h; ++q) {
                if (Thi >> q & 1) continue;
                const uint64_t T = Thi | low;
                const bool adj = (q > 0 && (T >> (q - 1) & 1)) || (q + 1 < n && (T >> (q + 1) & 1));
                if (pass == 1 || adj) { Thi |= 1ull << q; ++cnt; grew = true; }
            }
        }
    }
    return Thi;
}

}  // namespace

bool hamiltonian_from_paulis(int n, int M, const char *paulis, const double *coeffs, Hamiltonian &H, std::string &err)
{
    H = Hamiltonian(); H.n = n;
    H.terms.resize((size_t)M);
    for (int k = 0; k < M; ++k) {
        HostTerm t{0, 0, 0, coeffs[k]};
        const char *s = paulis + (size_t)k * n;
        for (int j = 0; j < n; ++j) {
            switch (s[j]) {
            case 'I': break;
            case 'X': t.x |= 1ull << j; break;
            case 'Z': t.z |= 1ull << j; break;
            case 'Y': t.x |= 1ull << j; t.z |= 1ull << j; ++t.ny; break;
            default: err = "hamiltonian: bad Pauli character (expected I, X, Y or Z)"; return false;
            }
        }
        H.terms[k] = t;
    }
    return finish(H, err);
}

bool hamiltonian_from_masks(int n, int M, const uint64_t *xm, const uint64_t *zm, const double *coeffs, Hamiltonian &H,
                            std::string &err)
{
    H = Hamiltonian(); H.n = n;
    H.terms.resize((size_t)M);
    for (int k = 0; k < M; ++k) H.terms[k] = HostTerm{xm[k], zm[k], __builtin_popcountll(xm[k] & zm[k]), coeffs[k]};
    return finish(H, err);
}

bool plan_expectation(const Hamiltonian &H, int n, int k, int f, int umax, uint32_t tab_cap, int amp_bytes,
                      bool register_stages, ExpectPlan &plan, std::string &err)
{
    const int FB = amp_bytes == 8 ? 4 : 3;   // same fold as phys<T>() in kernels.cuh
    auto hphys = [FB](uint32_t j) { uint32_t p = j; for (int sh = FB; sh < 16; sh += FB) p ^= (j >> sh) & ((1u << FB) - 1u); return p; };
    plan = ExpectPlan();
    if (k > n) k = n;
    if (f > k) f = k;
    plan.k = k;
    const uint64_t low = f ? ((1ull << f) - 1) : 0;
    const int h = k - f;
    // off-diagonal groups in canonical order, their terms in input order
    std::vector<uint64_t> gm;
    for (uint64_t m : H.group_mask) if (m) gm.push_back(m);
    std::vector<std::vector<int>> gterms(gm.size());
    for (size_t t = 0; t < H.terms.size(); ++t) {
        if (!H.terms[t].x) continue;
        const size_t g = std::lower_bound(gm.begin(), gm.end(), H.terms[t].x) - gm.begin();
        gterms[g].push_back((int)t);
    }
    // ---- choose the tile-bit set of every pass
    std::vector<uint64_t> passT;
    std::vector<std::vector<int>> passG;
    if (n <= k || gm.empty()) {
        passT.push_back(n <= k ? ((1ull << n) - 1) : ((1ull << k) - 1));
        passG.emplace_back();
        for (size_t g = 0; g < gm.size(); ++g) passG[0].push_back((int)g);
    } else {
        std::vector<char> done(gm.size(), 0);
        size_t left = gm.size();
        Run tmp[MAX_RUNS];
        while (left) {
            uint64_t Thi = 0;
            std::vector<int> mine;
            for (;;) {
                int best = -1, best_add = 1 << 30;
                for (size_t g = 0; g < gm.size(); ++g) {
                    if (done[g]) continue;
                    const uint64_t need = gm[g] & ~low;
                    const int add = __builtin_popcountll(need & ~Thi);
                    if (add >= best_add) continue;
                    const uint64_t cand = Thi | need;
                    if (__builtin_popcountll(cand) > h) continue;
                    if (runs_of(fill_bits(cand, n, f, h) | low, tmp, MAX_RUNS) > MAX_RUNS) continue;
                    best = (int)g; best_add = add;
                    if (add == 0) break;
                }
                if (best < 0) break;
                Thi |= gm[best] & ~low; done[best] = 1; --left; mine.push_back(best);
            }
            if (mine.empty()) {
                err = "hamiltonian: a flip mask does not fit one tile (too many or too scattered X/Y positions)";
                return false;
            }
            std::sort(mine.begin(), mine.end());
            {   // spare tile bits: prefer the qubits the pass's terms act on with Z (their sign then is part of the
                // tile-independent table instead of a per-tile correction), most frequent first
                std::vector<std::pair<long, int>> freq;
                for (int q = f; q < n; ++q) {
                    if (Thi >> q & 1) continue;
                    long cnt = 0;
                    for (int g : mine) for (int t : gterms[g]) cnt += (long)(H.terms[t].z >> q & 1);
                    if (cnt) freq.push_back({-cnt, q});
                }
                std::sort(freq.begin(), freq.end());
                for (auto &fq : freq) {
                    if (__builtin_popcountll(Thi) >= h) break;
                    const uint64_t cand = Thi | (1ull << fq.second);
                    if (runs_of(fill_bits(cand, n, f, h) | low, tmp, MAX_RUNS) <= MAX_RUNS) Thi = cand;
                }
            }
            passT.push_back(fill_bits(Thi, n, f, h) | low);
            passG.push_back(mine);
        }
    }
    // ---- encode
    for (size_t p = 0; p < passT.size(); ++p) {
        const uint64_t T = passT[p];
        DPass dp; memset(&dp, 0, sizeof dp);
        dp.k = (uint8_t)k; dp.with_diag = (p == 0) ? 1 : 0;
        const int nr = runs_of(T, dp.runs, MAX_RUNS);
        if (nr > MAX_RUNS) { err = "hamiltonian: too many tile runs (internal)"; return false; }
        dp.n_runs = (uint8_t)nr;
        {   // vector offsets of the tile load (kernels.cuh expect_load_u)
            const int TBh = (k >= 11) ? 8 : (k - 3 < 5 ? 5 : k - 3);
            const uint32_t V = 16u / (uint32_t)amp_bytes, nthr = 1u << TBh, nld = (1u << k) / V / nthr;
            for (uint32_t i = 0; i < nld && i < 64; ++i) {
                const uint32_t j = i * nthr * V;
                uint64_t x = 0;
                for (int r = 0; r < nr; ++r) x |= (uint64_t)((j >> dp.runs[r].lpos) & ((1u << dp.runs[r].len) - 1u)) << dp.runs[r].gpos;
                dp.hi[i] = x;
            }
        }
        dp.group_begin = (uint32_t)plan.groups.size();
        uint32_t tab_used = 0;
        int batch_groups = 0;
        const int TB = (k >= 11) ? 8 : (k - 3 < 5 ? 5 : k - 3);   // log2(threads) of the expectation kernel
        const int L = k - 1 - TB;                                   // loop bits: 2^L pairs per thread and group
        const int umax_eff = umax < TB ? umax : TB;
        // ---- register stages: groups whose flip mask and in-tile z bits fit RSB local bits are clustered; a cluster is
        // evaluated with those bits as register bits (amplitudes and partners in registers, W broadcast)
        const int RSB = k - TB;
        std::vector<char> in_rs(gm.size(), 0);
        if (RSB >= 2 && RSB <= DEV_MAX_R && register_stages) {
            std::vector<uint32_t> sets; std::vector<std::vector<int>> members;
            std::vector<std::pair<uint32_t, int>> cand;
            for (int g : passG[p]) {
                uint32_t S = compress(gm[g], T);
                for (int t : gterms[g]) S |= compress(H.terms[t].z & T, T);
                if (__builtin_popcount(S) <= RSB) cand.push_back({S, g});
            }
            std::sort(cand.begin(), cand.end());
            for (auto &cg : cand) {
                size_t si = 0;
                while (si < sets.size() && __builtin_popcount(sets[si] | cg.first) > RSB) ++si;
                if (si == sets.size()) { sets.push_back(0); members.emplace_back(); }
                sets[si] |= cg.first; members[si].push_back(cg.second);
            }
            for (size_t si = 0; si < sets.size(); ++si) {
                if (plan.rss.size() >= 65536) break;   // DGroup::rs_id / the `hot` word hold 16 bits: further clusters take the lookup path
                uint32_t regs = sets[si];
                for (int b = 0; b < k && __builtin_popcount(regs) < RSB; ++b) regs |= 1u << b;   // pad with low bits
                DRs rs; memset(&rs, 0, sizeof rs);
                int nrb = 0;
                for (int b = 0; b < k; ++b) if (regs >> b & 1) { rs.regbit[nrb] = (uint8_t)b; rs.po_bytes[nrb] = hphys(1u << b) * (uint32_t)amp_bytes; ++nrb; }
                const uint32_t rs_id = (uint32_t)plan.rss.size();
                plan.rss.push_back(rs);
                std::sort(members[si].begin(), members[si].end());
                for (int g : members[si]) {
                    in_rs[g] = 1;
                    DGroup dg; memset(&dg, 0, sizeof dg);
                    dg.m_loc = compress(gm[g], T);
                    dg.pivot = (uint8_t)(31 - __builtin_clz(dg.m_loc));
                    dg.rs = 1; dg.rs_id = (uint16_t)rs_id; dg.m_r = (uint8_t)compress(dg.m_loc, regs);
                    dg.ubits = (uint8_t)RSB;
                    dg.term_begin = (uint32_t)plan.terms.size();
                    if (batch_groups >= GT_BATCH_MAX || tab_used + (1u << RSB) > tab_cap) {
                        if (plan.groups.size() > dp.group_begin) plan.groups.back().last_in_batch = 1;
                        tab_used = 0; batch_groups = 0;
                    }
                    ++batch_groups;
                    dg.tab_off = tab_used; tab_used += 1u << RSB;
                    long dyn_end = -1;
                    for (int phase = 0; phase < 2; ++phase)
                        for (int t : gterms[g]) {
                            const HostTerm &ht = H.terms[t];
                            const bool dyn = (ht.z & ~T) != 0;
                            if (dyn != (phase == 0)) continue;
                            if (phase == 1 && dyn_end < 0) dyn_end = (long)plan.terms.size();
                            DTerm dt; memset(&dt, 0, sizeof dt);
                            static const double pr[4] = {1, 0, -1, 0}, pim[4] = {0, 1, 0, -1};
                            dt.cr = ht.c * pr[ht.ny & 3]; dt.ci = ht.c * pim[ht.ny & 3];
                            dt.zout = ht.z & ~T;
                            dt.zu = compress(compress(ht.z & T, T), regs);
                            plan.terms.push_back(dt);
                        }
                    dg.term_end = (uint32_t)plan.terms.size();
                    dg.dyn_end = dyn_end < 0 ? dg.term_end : (uint32_t)dyn_end;
                    plan.groups.push_back(dg);
                }
            }
        }
        for (int g : passG[p]) {
            if (in_rs[g]) continue;
            // slice the group's terms so that every slice's table index (in-tile z bits) stays small  (Eq. 12)
            std::vector<std::vector<int>> slices;
            std::vector<uint32_t> sliceU;
            for (int t : gterms[g]) {
                const uint32_t zl = compress(H.terms[t].z & T, T);
                bool placed = false;
                if (!slices.empty()) {
                    const uint32_t U2 = sliceU.back() | zl;
                    if (__builtin_popcount(U2) <= umax_eff) {
                        slices.back().push_back(t); sliceU.back() = U2; placed = true;
                    }
                }
                if (!placed) { slices.emplace_back(1, t); sliceU.push_back(zl); }
            }
            for (size_t sl = 0; sl < slices.size(); ++sl) {
                DGroup dg; memset(&dg, 0, sizeof dg);
                dg.m_loc = compress(gm[g], T);
                dg.pivot = (uint8_t)(31 - __builtin_clz(dg.m_loc));
                const uint32_t Uloc = sliceU[sl];
                Run ur[4];
                const int nur = runs_of(Uloc, ur, 4);
                const int ubits = __builtin_popcount(Uloc);
                const bool table = (ubits <= umax_eff) && ((1u << ubits) <= tab_cap);   // any bit pattern: the index comes from the lookup block
                dg.direct = table ? 0 : 1;
                dg.term_begin = (uint32_t)plan.terms.size();
                if (batch_groups >= GT_BATCH_MAX || (table && tab_used + (1u << ubits) > tab_cap)) {   // close the batch
                    if (plan.groups.size() > dp.group_begin) plan.groups.back().last_in_batch = 1;
                    tab_used = 0; batch_groups = 0;
                }
                ++batch_groups;
                if (table) {
                    dg.uloc = Uloc;
                    dg.ubits = (uint8_t)ubits; dg.n_uruns = (uint8_t)(nur < 3 ? nur : 3);
                    for (int r = 0; r < nur && r < 3; ++r) { dg.uruns[r].lpos = ur[r].gpos; dg.uruns[r].len = ur[r].len; dg.uruns[r].shift = ur[r].lpos; }
                    dg.tab_off = tab_used; tab_used += 1u << ubits;
                    // loop bits: the L highest local bits outside the table index bits and the pivot
                    uint32_t excl = 1u << dg.pivot;
                    int nl = 0;
                    for (int b = k - 1; b >= 0 && nl < L; --b)
                        if (!((Uloc | (1u << dg.pivot)) >> b & 1)) { excl |= 1u << b; ++nl; }
                    if (nl < L) { err = "hamiltonian: no room for loop bits (internal)"; return false; }
                    int ne = 0, nlp = 0;
                    for (int b = 0; b < k; ++b) if (excl >> b & 1) {
                        dg.ex[ne++] = (uint8_t)b;
                        if (b != dg.pivot) dg.lp[nlp++] = (uint8_t)b;
                    }
                    dg.n_ex = (uint8_t)ne;
                    {   // lookup block
                        dg.pm_bytes = hphys(dg.m_loc) * (uint32_t)amp_bytes;
                        dg.gt_index = (uint32_t)(plan.gtabs.size() / GT_WORDS);
                        int tpos[16], nt = 0;
                        for (int b = 0; b < k; ++b) if (!(excl >> b & 1)) tpos[nt++] = b;
                        {   // lanes 0..15 (thread-index bits 0..3) must hit 16 distinct bank pairs: give them local bit
                            // positions with distinct residues modulo the swizzle fold width (see phys<T>())
                            int pick[16], np = 0; bool used[16] = {false};
                            for (int r = 0; r < FB && np < 4; ++r)
                                for (int t = 0; t < nt; ++t) if (!used[t] && tpos[t] % FB == r) { pick[np++] = t; used[t] = true; break; }
                            for (int t = 0; t < nt && np < 4; ++t) if (!used[t]) { pick[np++] = t; used[t] = true; }
                            int ord[16], no = 0;
                            for (int i2 = 0; i2 < np; ++i2) ord[no++] = tpos[pick[i2]];
                            for (int t = 0; t < nt; ++t) if (!used[t]) ord[no++] = tpos[t];
                            for (int t = 0; t < nt; ++t) tpos[t] = ord[t];
                        }
                        auto word_of = [&](uint32_t j) {
                            const uint32_t u = compress(j, Uloc);
                            return (hphys(j) * (uint32_t)amp_bytes) | (u << 20);
                        };
                        for (int half = 0; half < 2; ++half)
                            for (uint32_t e = 0; e < 16; ++e) {
                                uint32_t j = 0;
                                for (int b = 0; b < 4; ++b) { const int tb = 4 * half + b; if (tb < nt && (e >> b & 1)) j |= 1u << tpos[tb]; }
                                plan.gtabs.push_back(word_of(j));
                            }
                        for (uint32_t i = 0; i < 32; ++i) {
                            uint32_t j = 0;
                            for (int s2 = 0; s2 < nlp; ++s2) if (i >> s2 & 1) j |= 1u << dg.lp[s2];
                            plan.gtabs.push_back(hphys(j) * (uint32_t)amp_bytes);
                        }
                    }
                    for (int e = 0; e < ne; ++e) dg.ex_pack |= (uint32_t)dg.ex[e] << (4 * e);
                    for (int e = 0; e < nlp; ++e) dg.lp_pack |= (uint32_t)dg.lp[e] << (4 * e);
                    for (int r = 0; r < nur && r < 3; ++r)
                        dg.urun_pack |= (uint64_t)(dg.uruns[r].lpos | (dg.uruns[r].len << 4) | (dg.uruns[r].shift << 8)) << (12 * r);
                }
                long dyn_end = -1;
                for (int phase = 0; phase < 2; ++phase)
                for (int t : slices[sl]) {
                    const HostTerm &ht = H.terms[t];
                    const bool dyn = (ht.z & ~T) != 0 || !table;
                    if (dyn != (phase == 0)) continue;   // dynamic terms first
                    if (phase == 1 && dyn_end < 0) dyn_end = (long)plan.terms.size();
                    DTerm dt; memset(&dt, 0, sizeof dt);
                    static const double pr[4] = {1, 0, -1, 0}, pim[4] = {0, 1, 0, -1};
                    dt.cr = ht.c * pr[ht.ny & 3]; dt.ci = ht.c * pim[ht.ny & 3];
                    dt.zout = ht.z & ~T;
                    const uint32_t zloc = compress(ht.z & T, T);
                    dt.zu = table ? compress(zloc, Uloc) : zloc;
                    plan.terms.push_back(dt);
                }
                dg.term_end = (uint32_t)plan.terms.size();
                dg.dyn_end = dyn_end < 0 ? dg.term_end : (uint32_t)dyn_end;
                plan.groups.push_back(dg);
            }
        }
        if (plan.groups.size() > dp.group_begin) plan.groups.back().last_in_batch = 1;
        dp.group_end = (uint32_t)plan.groups.size();
        // static tables, batch by batch, in the layout of the shared-memory table area
        for (uint32_t g0 = dp.group_begin; g0 < dp.group_end;) {
            uint32_t g1 = g0;
            while (!plan.groups[g1].last_in_batch) ++g1;
            uint32_t entries = 0;
            for (uint32_t gi = g0; gi <= g1; ++gi)
                if (!plan.groups[gi].direct) entries = plan.groups[gi].tab_off + (1u << plan.groups[gi].ubits);
            const size_t base = plan.wstat.size() / 2;
            plan.wstat.resize(plan.wstat.size() + 2 * (size_t)entries, 0.0);
            for (uint32_t gi = g0; gi <= g1; ++gi) {
                DGroup &dg = plan.groups[gi];
                dg.batch_entries = entries; dg.batch_last = g1;
                dg.hot = (uint64_t)(dg.rs ? 1 : (dg.direct ? 2 : 0)) | ((uint64_t)dg.m_r << 2) | ((uint64_t)dg.rs_id << 8) |
                         ((uint64_t)dg.tab_off << 24) | ((uint64_t)((!dg.direct && dg.dyn_end != dg.term_begin) ? 1 : 0) << 63);
                dg.gtab_off = (uint32_t)base + dg.tab_off;
                if (dg.direct) { dg.gtab_off = (uint32_t)base; continue; }
                for (uint32_t u = 0; u < (1u << dg.ubits); ++u) {
                    double wr = 0.0, wi = 0.0;
                    for (uint32_t t = dg.dyn_end; t < dg.term_end; ++t) {
                        const DTerm &tm = plan.terms[t];
                        const int par = __builtin_popcount(u & tm.zu) & 1;
                        wr += par ? -tm.cr : tm.cr; wi += par ? -tm.ci : tm.ci;
                    }
                    plan.wstat[2 * (base + dg.tab_off + u)] = wr;
                    plan.wstat[2 * (base + dg.tab_off + u) + 1] = wi;
                }
            }
            if (dp.n_batches == PASS_MAX_BATCHES) {   // cut the pass: same tile bits, the groups so far
                DPass done = dp;
                done.group_end = g0;
                plan.passes.push_back(done);
                dp.group_begin = g0; dp.with_diag = 0; dp.n_batches = 0;
            }
            dp.batch[dp.n_batches].g_first = g0; dp.batch[dp.n_batches].g_last = g1;
            dp.batch[dp.n_batches].entries = entries; dp.batch[dp.n_batches].wbase = (uint32_t)base;
            ++dp.n_batches;
            g0 = g1 + 1;
        }
        plan.passes.push_back(dp);
    }
    {   // lookup blocks re-laid by group index (zero blocks for register-stage / direct groups): a batch's blocks are
        // then one contiguous range, copied together with its descriptors and static tables
        std::vector<uint32_t> gt2(plan.groups.size() * (size_t)GT_WORDS, 0u);
        for (size_t gi = 0; gi < plan.groups.size(); ++gi) {
            DGroup &dg = plan.groups[gi];
            if (!dg.rs && !dg.direct)
                memcpy(&gt2[gi * GT_WORDS], &plan.gtabs[(size_t)dg.gt_index * GT_WORDS], GT_WORDS * sizeof(uint32_t));
            dg.gt_index = (uint32_t)gi;
        }
        plan.gtabs.swap(gt2);
    }
    return true;
}

}  // namespace gv

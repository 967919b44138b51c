// lower.cpp -- see lower.h.  A compiled block is cut into device blocks at stage boundaries whenever its program
// slice would outgrow the shared-memory budget (same tile bits, one more HBM round trip; results unchanged).
#include "lower.h"

#include <cstring>

namespace gv {

namespace {
constexpr uint32_t SLICE_BUDGET = 40 * 1024;   // bytes of shared memory for the program slice of one block
inline uint32_t al16(uint32_t v) { return (v + 15u) & ~15u; }
}  // namespace

uint32_t prog_slice_bytes(uint32_t n_stages, uint32_t n_ops, uint32_t n_segs, uint32_t n_trz, uint32_t n_tcz,
                          uint32_t n_cs, uint32_t n_ryl, uint32_t n_cx, int scs_bytes)
{
    return al16(n_cs * (uint32_t)scs_bytes) + al16(n_tcz * 8u) + al16(n_segs * (uint32_t)sizeof(DSeg)) +
           al16(n_stages * (uint32_t)sizeof(DStage)) + al16(n_ops * (uint32_t)sizeof(DOp)) +
           al16(n_trz * (uint32_t)sizeof(DTrz)) + al16(n_cx * (uint32_t)sizeof(DCx)) + al16(n_ryl * 2u) +
           n_segs * (uint32_t)TPH_ENTRIES * (uint32_t)scs_bytes + n_stages * (uint32_t)SLUT_ENTRIES * 12u;
}

bool lower_program(const Program &p, int scs_bytes, DevProgram &D, std::string &err)
{
    D = DevProgram();
    D.n = p.n; D.k = p.k; D.f = p.f; D.R = p.R;
    if (p.R > DEV_MAX_R) { err = "lower: R too large"; return false; }
    for (const Block &B : p.blocks) {
        bool first_piece = true;
        uint32_t si = B.stage_begin;
        do {
            DBlock db; memset(&db, 0, sizeof db);
            db.k = B.k; db.n_runs = B.n_runs; db.source_zero = (first_piece && B.source_zero) ? 1 : 0;
            memcpy(db.runs, B.runs, sizeof db.runs);
            db.stage_off = (uint32_t)D.stages.size(); db.op_off = (uint32_t)D.ops.size();
            db.seg_off = (uint32_t)D.segs.size(); db.trz_off = (uint32_t)D.trzs.size();
            db.tcz_off = (uint32_t)D.tczs.size(); db.cs_off = (uint32_t)D.csidx.size();
            db.ryl_off = (uint32_t)D.ryl.size(); db.cx_off = (uint32_t)D.cxs.size();
            auto lpos_of = [&](int q) -> int {   // local bit position of global qubit q in this block's tile, or 255
                for (int r = 0; r < B.n_runs; ++r)
                    if (q >= B.runs[r].gpos && q < B.runs[r].gpos + B.runs[r].len) return B.runs[r].lpos + (q - B.runs[r].gpos);
                return 255;
            };
            std::vector<int32_t> cs_local;   // parameter index per local slot (deduplicated)
            auto cs_slot = [&](int32_t param) -> uint32_t {
                for (size_t i = 0; i < cs_local.size(); ++i) if (cs_local[i] == param) return (uint32_t)i;
                cs_local.push_back(param);
                return (uint32_t)cs_local.size() - 1;
            };
            uint32_t n_stages = 0;
            while (si < B.stage_end) {
                const Stage &S = p.stages[si];
                // size of this stage's contribution
                uint32_t add_ops = S.op_end - S.op_begin, add_segs = 0, add_trz = 0, add_tcz = 0, add_cs = 0;
                const uint32_t add_cx = S.cx_end - S.cx_begin, add_ryl = DEV_MAX_R * add_ops;   // upper bounds
                for (uint32_t oi = S.op_begin; oi < S.op_end; ++oi) {
                    const MicroOp &m = p.mops[oi];
                    if (m.kind == MOP_RY) ++add_cs;
                    if (m.kind == MOP_DIAG) {
                        const DiagSeg &g = p.segs[m.param];
                        ++add_segs; add_trz += g.rz_end - g.rz_begin; add_tcz += g.cz_end - g.cz_begin;
                        add_cs += g.rz_end - g.rz_begin;
                    }
                }
                const uint32_t tot = prog_slice_bytes(n_stages + 1, (uint32_t)(D.ops.size() - db.op_off) + add_ops,
                                                      (uint32_t)(D.segs.size() - db.seg_off) + add_segs,
                                                      (uint32_t)(D.trzs.size() - db.trz_off) + add_trz,
                                                      (uint32_t)(D.tczs.size() - db.tcz_off) + add_tcz,
                                                      (uint32_t)cs_local.size() + add_cs,
                                                      (uint32_t)(D.ryl.size() - db.ryl_off) + add_ryl,
                                                      (uint32_t)(D.cxs.size() - db.cx_off) + add_cx, scs_bytes);
                if (n_stages > 0 && (tot > SLICE_BUDGET || n_stages >= 250)) break;
                if (tot > SLICE_BUDGET + 4096) { err = "lower: a single stage exceeds the program budget (internal)"; return false; }
                // ---- emit the stage
                DStage ds; memset(&ds, 0, sizeof ds);
                for (int s = 0; s < p.R; ++s) ds.regbit[s] = S.regbit[s];
                ds.op_begin = (uint16_t)(D.ops.size() - db.op_off);
                long open_ryl = -1;   // offset (block-local) of the RY layer being filled, -1 = none
                for (uint32_t oi = S.op_begin; oi < S.op_end; ++oi) {
                    const MicroOp &m = p.mops[oi];
                    DOp o; o.kind = m.kind; o.a = m.a; o.b = m.b; o.c = m.c; o.idx = -1;
                    if (m.kind == MOP_RY) {   // consecutive RYs on distinct slots commute: one layer micro-op
                        const int16_t slot = (int16_t)cs_slot(m.param);
                        if (open_ryl >= 0 && D.ryl[db.ryl_off + open_ryl + m.a] < 0) { D.ryl[db.ryl_off + open_ryl + m.a] = slot; continue; }
                        open_ryl = (long)(D.ryl.size() - db.ryl_off);
                        for (int s2 = 0; s2 < DEV_MAX_R; ++s2) D.ryl.push_back(-1);
                        D.ryl[db.ryl_off + open_ryl + m.a] = slot;
                        o.kind = MOP_RYL; o.idx = (int32_t)open_ryl;
                    } else if (m.kind == MOP_DIAG) {
                        open_ryl = -1;
                        const DiagSeg &g = p.segs[m.param];
                        DSeg sg; memset(&sg, 0, sizeof sg);
                        for (int s = 0; s < DEV_MAX_R; ++s) sg.reg_rz[s] = -1;
                        sg.trz_begin = (uint16_t)(D.trzs.size() - db.trz_off);
                        sg.tcz_begin = (uint16_t)(D.tczs.size() - db.tcz_off);
                        // thread-bit layout of this stage: local bits that are not register bits, ascending
                        auto tb_of = [&](int q) -> int {
                            const int lp = lpos_of(q);
                            if (lp == 255) return (int)TB_CONST;
                            int rank = 0;
                            for (int s2 = 0; s2 < p.R; ++s2) {
                                if (S.regbit[s2] == lp) return (int)TB_XREG + s2;
                                if (S.regbit[s2] < lp) ++rank;
                            }
                            return lp - rank;
                        };
                        std::vector<DTrz> thr_rz, xreg_rz;
                        for (uint32_t r = g.rz_begin; r < g.rz_end; ++r) {
                            const DiagRZ &z = p.rzs[r];
                            const uint32_t slot = cs_slot(z.param);
                            if (z.slot != 255 && sg.reg_rz[z.slot] < 0) sg.reg_rz[z.slot] = (int16_t)slot;
                            else {   // not a register bit (or a second RZ on the same slot)
                                DTrz t; t.qubit = z.qubit; t.tb = (uint8_t)tb_of(z.qubit); t.cs = (uint16_t)slot;
                                (t.tb >= TB_XREG && t.tb != TB_CONST ? xreg_rz : thr_rz).push_back(t);
                            }
                        }
                        sg.n_xreg = (uint8_t)xreg_rz.size();
                        for (const DTrz &t : xreg_rz) D.trzs.push_back(t);
                        for (const DTrz &t : thr_rz) D.trzs.push_back(t);
                        std::vector<uint64_t> cross, sameh;
                        for (uint32_t c = g.cz_begin; c < g.cz_end; ++c) {
                            const DiagCZ &z = p.czs[c];
                            if (z.s0 != 255 && z.s1 != 255) {
                                static const uint32_t A[5] = {0xAAAAAAAAu, 0xCCCCCCCCu, 0xF0F0F0F0u, 0xFF00FF00u, 0xFFFF0000u};
                                sg.regreg_neg ^= A[z.s0] & A[z.s1];
                            } else if (z.s0 != 255) sg.nbr[z.s0] ^= 1ull << z.q1;
                            else if (z.s1 != 255) sg.nbr[z.s1] ^= 1ull << z.q0;
                            else {
                                const int t0 = tb_of(z.q0), t1 = tb_of(z.q1);
                                auto kind = [](int t) { return t == (int)TB_CONST ? 0 : (t < 4 ? 1 : 2); };   // const / low / high
                                const int k0 = kind(t0), k1 = kind(t1);
                                const uint64_t m = (1ull << z.q0) | (1ull << z.q1);
                                if ((k0 == 2 && k1 == 1) || (k0 == 1 && k1 == 2)) cross.push_back(m | ((uint64_t)TCZ_CROSS << TCZ_CLASS_SHIFT));
                                else if (k0 == 2 || k1 == 2) sameh.push_back(m | ((uint64_t)TCZ_HI << TCZ_CLASS_SHIFT));
                                else sameh.push_back(m | ((uint64_t)TCZ_LO << TCZ_CLASS_SHIFT));
                            }
                        }
                        sg.n_cross = (uint16_t)cross.size();
                        for (uint64_t m : cross) D.tczs.push_back(m);
                        for (uint64_t m : sameh) D.tczs.push_back(m);
                        sg.stage = (uint8_t)n_stages;
                        sg.trz_end = (uint16_t)(D.trzs.size() - db.trz_off);
                        sg.tcz_end = (uint16_t)(D.tczs.size() - db.tcz_off);
                        o.idx = (int32_t)(D.segs.size() - db.seg_off);
                        D.segs.push_back(sg);
                    }
                    D.ops.push_back(o);
                }
                ds.op_end = (uint16_t)(D.ops.size() - db.op_off);
                // trailing CNOT run as an update of the local index; postbit = image of each register unit vector
                ds.cx_begin = (uint16_t)(D.cxs.size() - db.cx_off);
                for (int s2 = 0; s2 < p.R; ++s2) ds.postbit[s2] = (uint16_t)(1u << S.regbit[s2]);
                for (uint32_t ci = S.cx_begin; ci < S.cx_end; ++ci) {
                    DCx c; c.tl = (uint8_t)lpos_of(p.cxs[ci].tq); c.cl = (uint8_t)lpos_of(p.cxs[ci].cq); c.cq = p.cxs[ci].cq; c.pad = 0;
                    if (c.tl == 255) { err = "lower: CNOT target outside the tile (internal)"; return false; }
                    D.cxs.push_back(c);
                    if (c.cl != 255)
                        for (int s2 = 0; s2 < p.R; ++s2) ds.postbit[s2] ^= (uint16_t)(((ds.postbit[s2] >> c.cl) & 1u) << c.tl);
                }
                ds.cx_end = (uint16_t)(D.cxs.size() - db.cx_off);
                ds.has_cx = ds.cx_end > ds.cx_begin ? 1 : 0;
                {
                    const int FB = scs_bytes == 8 ? 4 : 3;
                    auto hphys = [FB](uint32_t j) { uint32_t ph = j; for (int sh = FB; sh < 16; sh += FB) ph ^= (j >> sh) & ((1u << FB) - 1u); return ph; };
                    for (int s2 = 0; s2 < p.R; ++s2) {
                        ds.po_bytes[s2] = hphys(1u << S.regbit[s2]) * (uint32_t)scs_bytes;
                        ds.post_bytes[s2] = hphys(ds.postbit[s2]) * (uint32_t)scs_bytes;
                    }
                }
                D.stages.push_back(ds);
                ++n_stages; ++si;
            }
            db.n_stages = (uint8_t)n_stages;
            {   // per-stage thread lookups: thread index -> local index j (register bits zero) | swizzled element offset << 16,
                // and -> global index; each GF(2)-linear in the thread index, stored for its low 4 bits and its high bits
                const int FB = scs_bytes == 8 ? 4 : 3;
                auto hphys = [FB](uint32_t j) { uint32_t ph = j; for (int sh = FB; sh < 16; sh += FB) ph ^= (j >> sh) & ((1u << FB) - 1u); return ph; };
                db.slut_goff = (uint32_t)(D.slut.size() * 4);
                for (uint32_t si2 = 0; si2 < n_stages; ++si2) {
                    const DStage &st = D.stages[db.stage_off + si2];
                    uint32_t w32[SLUT_ENTRIES]; uint64_t w64[SLUT_ENTRIES];
                    for (int e = 0; e < SLUT_ENTRIES; ++e) {
                        uint32_t j = e >= 16 ? ((uint32_t)(e - 16) << 4) : (uint32_t)e;
                        w32[e] = 0; w64[e] = 0;
                        if (j >> (B.k - p.R)) continue;
                        for (int s2 = 0; s2 < p.R; ++s2) { const uint32_t pos = st.regbit[s2]; j = ((j >> pos) << (pos + 1)) | (j & ((1u << pos) - 1u)); }
                        uint64_t x = 0;
                        for (int r = 0; r < B.n_runs; ++r) x |= (uint64_t)((j >> B.runs[r].lpos) & ((1u << B.runs[r].len) - 1u)) << B.runs[r].gpos;
                        w32[e] = j | (hphys(j) << 16); w64[e] = x;
                    }
                    for (int e = 0; e < SLUT_ENTRIES; ++e) D.slut.push_back(w32[e]);
                    for (int e = 0; e < SLUT_ENTRIES; ++e) { D.slut.push_back((uint32_t)w64[e]); D.slut.push_back((uint32_t)(w64[e] >> 32)); }
                }
            }
            if (n_stages > 1) {   // a leading stage that is only a CNOT run is folded into the tile load
                const DStage &s0 = D.stages[db.stage_off];
                if (s0.op_begin == s0.op_end && s0.has_cx && !db.source_zero) {
                    const int FB = scs_bytes == 8 ? 4 : 3;
                    auto hphys = [FB](uint32_t j) { uint32_t ph = j; for (int sh = FB; sh < 16; sh += FB) ph ^= (j >> sh) & ((1u << FB) - 1u); return ph; };
                    auto alin = [&](uint32_t j) {
                        for (uint32_t ci = s0.cx_begin; ci < s0.cx_end; ++ci) {
                            const DCx &c = D.cxs[db.cx_off + ci];
                            if (c.cl != 255) j ^= ((j >> c.cl) & 1u) << c.tl;
                        }
                        return j;
                    };
                    const uint32_t V = 16u / (uint32_t)scs_bytes, nthr = 1u << (B.k - p.R), nld = (1u << p.R) / V;
                    db.lead_cx = 1;
                    if (s0.cx_end - s0.cx_begin <= 32) {
                        db.n_lead_cx = s0.cx_end - s0.cx_begin;
                        for (uint32_t ci = 0; ci < db.n_lead_cx; ++ci) db.lead_cxs[ci] = D.cxs[db.cx_off + s0.cx_begin + ci];
                    }
                    db.e1_cx = hphys(alin(1u));
                    for (uint32_t i = 0; i < nld && i < 16; ++i) db.hip_cx[i] = hphys(alin(i * nthr * V));
                }
            }
            {   // vector offsets of the tile load/store (kernels.cuh tile_load_u)
                const uint32_t V = 16u / (uint32_t)scs_bytes, nthr = 1u << (B.k - p.R), nld = (1u << p.R) / V;
                for (uint32_t i = 0; i < nld && i < 16; ++i) {
                    const uint32_t j = i * nthr * V;
                    uint64_t x = 0;
                    for (int r = 0; r < B.n_runs; ++r) x |= (uint64_t)((j >> B.runs[r].lpos) & ((1u << B.runs[r].len) - 1u)) << B.runs[r].gpos;
                    db.hi[i] = x;
                    const int FB = scs_bytes == 8 ? 4 : 3;   // phys<T>() of kernels.cuh
                    uint32_t ph = j;
                    for (int sh = FB; sh < 16; sh += FB) ph ^= (j >> sh) & ((1u << FB) - 1u);
                    db.hip[i] = ph;
                }
            }
            db.n_ops = (uint32_t)(D.ops.size() - db.op_off);
            db.n_segs = (uint32_t)(D.segs.size() - db.seg_off);
            db.n_trz = (uint32_t)(D.trzs.size() - db.trz_off);
            db.n_tcz = (uint32_t)(D.tczs.size() - db.tcz_off);
            db.n_cs = (uint32_t)cs_local.size();
            db.n_ryl = (uint32_t)(D.ryl.size() - db.ryl_off); db.n_cx = (uint32_t)(D.cxs.size() - db.cx_off);
            for (int32_t v : cs_local) D.csidx.push_back(v);
            if (cs_local.size() <= 64) {
                db.n_cs_inline = (uint32_t)cs_local.size();
                for (size_t ci = 0; ci < cs_local.size(); ++ci) db.cs_inline[ci] = cs_local[ci];
            }
            {
                uint32_t o = al16(db.n_cs * (uint32_t)scs_bytes);
                db.off_tcz = o; o += al16(db.n_tcz * 8u);
                db.off_segs = o; o += al16(db.n_segs * (uint32_t)sizeof(DSeg));
                db.off_stages = o; o += al16(db.n_stages * (uint32_t)sizeof(DStage));
                db.off_ops = o; o += al16(db.n_ops * (uint32_t)sizeof(DOp));
                db.off_trz = o; o += al16(db.n_trz * (uint32_t)sizeof(DTrz));
                db.off_cxs = o; o += al16(db.n_cx * (uint32_t)sizeof(DCx));
                db.off_ryl = o; o += al16(db.n_ryl * 2u);
                db.slut_off = o + db.n_segs * (uint32_t)TPH_ENTRIES * (uint32_t)scs_bytes;
            }
            db.tph_off = prog_slice_bytes(0, db.n_ops, 0, db.n_trz, db.n_tcz, db.n_cs, db.n_ryl, db.n_cx, scs_bytes) + ((db.n_segs * (uint32_t)sizeof(DSeg) + 15u) & ~15u) + ((db.n_stages * (uint32_t)sizeof(DStage) + 15u) & ~15u);
            db.smem_prog_bytes = prog_slice_bytes(db.n_stages, db.n_ops, db.n_segs, db.n_trz, db.n_tcz, db.n_cs, db.n_ryl, db.n_cx, scs_bytes);
            if (db.smem_prog_bytes > D.max_smem_prog) D.max_smem_prog = db.smem_prog_bytes;
            if (db.n_ops > 65535 || db.n_trz > 65535 || db.n_tcz > 65535 || db.n_cs > 65535) {
                err = "lower: block too large (internal)"; return false;
            }
            D.blocks.push_back(db);
            first_piece = false;
        } while (si < B.stage_end);
    }
    return true;
}

}  // namespace gv

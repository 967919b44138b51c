// kernels.cuh -- per-thread device code of the gate engine and the Hamiltonian engine (sm_100a).
//
// Everything here is written per thread (tid explicit) and split at the points where the thread block
// synchronises, so the __global__ wrappers in kernels.cu are a plain sequence  phase; __syncthreads(); phase; ...
// Operations follow /root/reference/PAPER.md: R_y, R_z of Eq. 7, the entangling layer
// (PAPER.md:169), |psi> = U(theta)|0>, E = sum_k c_k <P_k> (Eq. 4, 6) evaluated
// as a partition of the terms (Eq. 12).  Index convention: qubit q <-> bit q of the amplitude index.
#pragma once
#include <stdint.h>

#include "devprog.h"

#define GV_DEV __device__ __forceinline__
#define GV_UNROLL _Pragma("unroll")
GV_DEV int gv_popcll(uint64_t v) { return __popcll(v); }
GV_DEV int gv_popc(uint32_t v) { return __popc(v); }

namespace gv {

template <typename T> struct alignas(2 * sizeof(T)) cx { T x, y; };

template <typename T> GV_DEV cx<T> cmul(cx<T> a, cx<T> b) { return cx<T>{a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x}; }
template <typename T> GV_DEV cx<T> cneg(cx<T> a) { return cx<T>{-a.x, -a.y}; }

// Shared-memory swizzle: XOR-fold the higher index bits into the low FB bits (FB = log2 of the elements one
// 128-byte wavefront holds: 16 complex64, 8 complex128).  Linear over GF(2): phys(a ^ b) = phys(a) ^ phys(b).
template <typename T> GV_DEV uint32_t phys(uint32_t j)
{
    constexpr int FB = sizeof(T) == 4 ? 4 : 3;
    constexpr uint32_t M = (1u << FB) - 1;
    uint32_t p = j;
    GV_UNROLL
    for (int sh = FB; sh < 16; sh += FB) p ^= (j >> sh) & M;
    return p;
}

GV_DEV uint64_t scatter_runs(uint32_t j, const Run *runs, int n_runs)
{
    uint64_t x = 0;
    for (int r = 0; r < n_runs; ++r)
        x |= (uint64_t)((j >> runs[r].lpos) & ((1u << runs[r].len) - 1u)) << runs[r].gpos;
    return x;
}

// Global index of local index 0 of tile number `tile`: the tile bits fill the positions the runs leave free.
GV_DEV uint64_t tile_base(uint64_t tile, const Run *runs, int n_runs)
{
    uint64_t x = 0;
    int gpos = 0;
    for (int r = 0; r < n_runs; ++r) {
        const int gap = (int)runs[r].gpos - gpos;
        if (gap > 0) { x |= (tile & ((1ull << gap) - 1ull)) << gpos; tile >>= gap; }
        gpos = runs[r].gpos + runs[r].len;
    }
    x |= tile << gpos;
    return x;
}

GV_DEV uint32_t insert_zero(uint32_t i, uint32_t pos) { return ((i >> pos) << (pos + 1)) | (i & ((1u << pos) - 1u)); }

struct DevArrays {
    const DBlock *blocks; const DStage *stages; const DOp *ops; const DSeg *segs; const DTrz *trzs;
    const uint64_t *tczs; const int32_t *csidx; const int16_t *ryl; const DCx *cxs; const uint32_t *slut;
};

GV_DEV uint32_t al16u(uint32_t v) { return (v + 15u) & ~15u; }

template <typename T> struct ProgView {
    cx<T> *cs; uint64_t *tcz; DSeg *segs; DStage *stages; DOp *ops; DTrz *trz; DCx *cxs; int16_t *ryl; cx<T> *tph;
    unsigned char *slut;   // per stage: SLUT_ENTRIES x u32 (j | swizzled byte offset... see slut_build_entry) then x u64
    GV_DEV void bind(unsigned char *p, const DBlock &b)
    {
        cs = (cx<T> *)p;
        tcz = (uint64_t *)(p + b.off_tcz);
        segs = (DSeg *)(p + b.off_segs);
        stages = (DStage *)(p + b.off_stages);
        ops = (DOp *)(p + b.off_ops);
        trz = (DTrz *)(p + b.off_trz);
        cxs = (DCx *)(p + b.off_cxs);
        ryl = (int16_t *)(p + b.off_ryl);
        tph = (cx<T> *)(p + b.tph_off);
        slut = p + b.slut_off;
    }
};

// Copy the block's program slice into shared memory and gather this batch row's (cos, sin) values.
template <typename T>
GV_DEV void gate_prologue(ProgView<T> &pv, const DBlock &b, const DevArrays &da, const cx<T> *cs_row, uint32_t tid,
                          uint32_t nthr)
{
    if (b.n_cs_inline == b.n_cs) {   // indices from the kernel parameter: one global-load latency instead of two
        for (uint32_t i = tid; i < b.n_cs; i += nthr) pv.cs[i] = cs_row[b.cs_inline[i]];
    } else {
        for (uint32_t i = tid; i < b.n_cs; i += nthr) pv.cs[i] = cs_row[da.csidx[b.cs_off + i]];
    }
    for (uint32_t i = tid; i < b.n_tcz; i += nthr) pv.tcz[i] = da.tczs[b.tcz_off + i];
    for (uint32_t i = tid; i < b.n_segs; i += nthr) pv.segs[i] = da.segs[b.seg_off + i];
    for (uint32_t i = tid; i < b.n_stages; i += nthr) pv.stages[i] = da.stages[b.stage_off + i];
    for (uint32_t i = tid; i < b.n_ops; i += nthr) pv.ops[i] = da.ops[b.op_off + i];
    for (uint32_t i = tid; i < b.n_trz; i += nthr) pv.trz[i] = da.trzs[b.trz_off + i];
    for (uint32_t i = tid; i < b.n_cx; i += nthr) pv.cxs[i] = da.cxs[b.cx_off + i];
    for (uint32_t i = tid; i < b.n_ryl; i += nthr) pv.ryl[i] = da.ryl[b.ryl_off + i];
    {   // host-built per-stage thread lookups
        uint32_t *dst = reinterpret_cast<uint32_t *>(pv.slut);
        const uint32_t *src = da.slut + b.slut_goff / 4;
        for (uint32_t i = tid; i < (uint32_t)b.n_stages * SLUT_ENTRIES * 3u; i += nthr) dst[i] = src[i];
    }
}

// ---- tile <-> global -------------------------------------------------------------------------------------
template <typename T> struct alignas(16) vec16 { cx<T> v[16 / sizeof(cx<T>)]; };

// Unrolled variants: every thread moves NLD 16-byte vectors; vector i of thread tid is chunk tid + i*nthr, whose
// local index splits into disjoint bit fields (tid part | i part), so the global offset is x0 | hi[i] with
// hi[i] = scatter(i * nthr * V) precomputed on the host (DBlock::hi, DPass::hi).  All NLD loads are in flight
// before the first shared-memory store.
// The caller issues the NLD loads (vec16 registers); this writes them to swizzled shared memory.
template <typename T, int NLD>
GV_DEV void tile_commit(cx<T> *tile, const vec16<T> *v, uint32_t tid, const uint32_t *hip)
{
    constexpr uint32_t V = 16 / sizeof(cx<T>);
    const uint32_t p0 = phys<T>(tid * V);
    GV_UNROLL
    for (int i = 0; i < NLD; ++i) {
        const uint32_t p = p0 ^ hip[i];
        GV_UNROLL
        for (uint32_t e = 0; e < V; ++e) tile[p ^ e] = v[i].v[e];
    }
}

// tile_commit for a block whose first stage is only a CNOT run: element j goes to the swizzled image of A j ^ c.
template <typename T, int NLD>
GV_DEV void tile_commit_cx(cx<T> *tile, const vec16<T> *v, uint32_t tid, uint64_t xbase, const DCx *cxs, uint32_t n_cx,
                           const uint32_t *hip_cx, uint32_t e1_cx)
{
    constexpr uint32_t V = 16 / sizeof(cx<T>);
    uint32_t jj = tid * V;
    for (uint32_t ci = 0; ci < n_cx; ++ci) {
        const DCx c = cxs[ci];
        const uint32_t bit = (c.cl != 255) ? ((jj >> c.cl) & 1u) : (uint32_t)((xbase >> c.cq) & 1ull);
        jj ^= bit << c.tl;
    }
    const uint32_t p0 = phys<T>(jj);
    GV_UNROLL
    for (int i = 0; i < NLD; ++i) {
        const uint32_t p = p0 ^ hip_cx[i];
        GV_UNROLL
        for (uint32_t e = 0; e < V; ++e) tile[p ^ (e ? e1_cx : 0u)] = v[i].v[e];
    }
}

template <typename T, int NLD>
GV_DEV void tile_store_u(const cx<T> *tile, cx<T> *state, uint64_t x0, uint32_t tid, const uint64_t *hi,
                         const uint32_t *hip)
{
    constexpr uint32_t V = 16 / sizeof(cx<T>);
    const uint32_t p0 = phys<T>(tid * V);
    GV_UNROLL
    for (int i = 0; i < NLD; ++i) {
        const uint32_t p = p0 ^ hip[i];
        vec16<T> v;
        GV_UNROLL
        for (uint32_t e = 0; e < V; ++e) v.v[e] = tile[p ^ e];
        *reinterpret_cast<vec16<T> *>(state + (x0 | hi[i])) = v;
    }
}

template <typename T>
GV_DEV void tile_zero_store(cx<T> *state, uint64_t xbase, const Run *runs, int n_runs, int k, uint32_t tid, uint32_t nthr)
{
    constexpr uint32_t V = 16 / sizeof(cx<T>);
    const uint32_t nchunk = (1u << k) / V;
    vec16<T> v;
    GV_UNROLL
    for (uint32_t e = 0; e < V; ++e) v.v[e] = cx<T>{T(0), T(0)};
    for (uint32_t c = tid; c < nchunk; c += nthr) {
        const uint64_t x = xbase | scatter_runs(c * V, runs, n_runs);
        *reinterpret_cast<vec16<T> *>(state + x) = v;
    }
}

template <typename T> GV_DEV void tile_init_zero_state(cx<T> *tile, int k, uint32_t tid, uint32_t nthr)
{
    for (uint32_t j = tid; j < (1u << k); j += nthr) tile[j] = cx<T>{T(0), T(0)};
}

// ---- register-level gates (Eq. 7) ------------------------------------------------------------------------
// R_y(theta) = [[c,-s],[s,c]] on register slot S, c = cos(theta/2), s = sin(theta/2).
template <typename T> GV_DEV void ry_pair(cx<T> &u, cx<T> &v, T c, T s)
{
    const cx<T> a = u, b = v;
    u = cx<T>{c * a.x - s * b.x, c * a.y - s * b.y};
    v = cx<T>{s * a.x + c * b.x, s * a.y + c * b.y};
}
// complex64: (re, im) is one packed f32x2 operand -- FMUL2/FFMA2 on sm_100a rotate a pair in 4 instructions
template <> GV_DEV void ry_pair<float>(cx<float> &u, cx<float> &v, float c, float s)
{
    const float2 a = make_float2(u.x, u.y), b = make_float2(v.x, v.y);
    const float2 cc = make_float2(c, c), ss = make_float2(s, s), ns = make_float2(-s, -s);
    const float2 un = __ffma2_rn(ns, b, __fmul2_rn(cc, a));
    const float2 vn = __ffma2_rn(cc, b, __fmul2_rn(ss, a));
    u = cx<float>{un.x, un.y};
    v = cx<float>{vn.x, vn.y};
}

template <typename T, int R, int S> GV_DEV void ry_slot(cx<T> *a, T c, T s)
{
    GV_UNROLL
    for (int r = 0; r < (1 << R); ++r) {
        if (r & (1 << S)) continue;
        ry_pair<T>(a[r], a[r | (1 << S)], c, s);
    }
}

// A layer of R_y gates on distinct register slots: slot s is rotated when ryl[s] >= 0 (uniform branch, static slots).
template <typename T, int R> GV_DEV void ry_layer(cx<T> *a, const int16_t *ryl, const cx<T> *cs)
{
    GV_UNROLL
    for (int s = 0; s < R; ++s) {
        const int i = ryl[s];
        if (i >= 0) {
            const cx<T> v = cs[i];
            if (s == 0) ry_slot<T, R, 0>(a, v.x, v.y);
            if (s == 1) ry_slot<T, R, (R > 1 ? 1 : 0)>(a, v.x, v.y);
            if (s == 2) ry_slot<T, R, (R > 2 ? 2 : 0)>(a, v.x, v.y);
            if (s == 3) ry_slot<T, R, (R > 3 ? 3 : 0)>(a, v.x, v.y);
            if (s == 4) ry_slot<T, R, (R > 4 ? 4 : 0)>(a, v.x, v.y);
        }
    }
}

// Complex multiply a * w; for complex64 with the packed f32x2 pipe: a.x * (w.x, w.y) + a.y * (-w.y, w.x).
template <typename T> GV_DEV cx<T> cmul_w(cx<T> a, cx<T> w, cx<T> wsw) { (void)wsw; return cmul(a, w); }
template <> GV_DEV cx<float> cmul_w<float>(cx<float> a, cx<float> w, cx<float> wsw)
{
    const float2 r = __ffma2_rn(make_float2(a.y, a.y), make_float2(wsw.x, wsw.y),
                                __fmul2_rn(make_float2(a.x, a.x), make_float2(w.x, w.y)));
    return cx<float>{r.x, r.y};
}

// Thread-phase tables of the block's diagonal segments (one entry per call): the factor that is constant over a
// thread's registers splits into (tile-constant x thread-index bits 0..3) and (thread-index bits 4..).  Built once
// per thread block in the prologue, so a stage needs two table reads instead of one multiply per RZ and thread.
template <typename T, int R>
GV_DEV void tph_build_entry(const ProgView<T> &pv, uint32_t item, uint64_t xbase, const Run *runs, int n_runs, int k)
{
    const uint32_t sgi = item / TPH_CONST, e = item % TPH_CONST;   // items cover the 48 thread entries of every segment
    const DSeg &sg = pv.segs[sgi];
    const DStage &st = pv.stages[sg.stage];
    const bool high = e >= 16;
    uint32_t j = high ? ((e - 16u) << 4) : e;
    if (j >> (k - R)) return;                       // no such thread
    GV_UNROLL
    for (int s = 0; s < R; ++s) j = insert_zero(j, st.regbit[s]);
    const uint64_t x = xbase | scatter_runs(j, runs, n_runs);
    cx<T> ph{T(1), T(0)};
    for (uint32_t t = sg.trz_begin + sg.n_xreg; t < sg.trz_end; ++t) {
        const DTrz z = pv.trz[t];
        const bool mine = high ? (z.tb >= 4 && z.tb < TB_XREG) : (z.tb < 4);   // tile-constant factors: tph_const_factor
        if (!mine) continue;
        const cx<T> cs = pv.cs[z.cs];
        const bool bit = (x >> z.qubit) & 1ull;
        ph = cmul(ph, cx<T>{cs.x, bit ? cs.y : -cs.y});     // Eq. 7: e^{-i phi/2} on bit 0, e^{+i phi/2} on bit 1
    }
    uint32_t par = 0;
    for (uint32_t t = sg.tcz_begin + sg.n_cross; t < sg.tcz_end; ++t) {
        const uint64_t m = pv.tcz[t];
        if ((int)(m >> TCZ_CLASS_SHIFT) != (high ? TCZ_HI : TCZ_LO)) continue;
        const uint64_t mm = m & ((1ull << TCZ_CLASS_SHIFT) - 1ull);
        par ^= ((x & mm) == mm) ? 1u : 0u;
    }
    pv.tph[sgi * TPH_ENTRIES + e] = par ? cneg(ph) : ph;
}

// Factor of one tile-constant R_z of a segment (identity for the others); their product goes to entry TPH_CONST.
template <typename T>
GV_DEV cx<T> tph_const_factor(const ProgView<T> &pv, uint32_t trz_index, uint64_t xbase)
{
    const DTrz z = pv.trz[trz_index];
    if (z.tb != TB_CONST) return cx<T>{T(1), T(0)};
    const cx<T> cs = pv.cs[z.cs];
    const bool bit = (xbase >> z.qubit) & 1ull;
    return cx<T>{cs.x, bit ? cs.y : -cs.y};
}

// Merged diagonal segment: every R_z phase (Eq. 7) and every CZ sign of the segment as ONE complex factor per
// amplitude = thread factor (two table reads) x table over the low register slots x table over the high slots.
template <typename T, int R>
GV_DEV void diag_apply(cx<T> *a, const ProgView<T> &pv, const DSeg &sg, uint32_t sgi, uint64_t x, uint32_t tid)
{
    constexpr int RL = R / 2, RH = R - RL;
    cx<T> ph = cmul(cmul(pv.tph[sgi * TPH_ENTRIES + (tid & 15u)], pv.tph[sgi * TPH_ENTRIES + 16u + (tid >> 4)]),
                    pv.tph[sgi * TPH_ENTRIES + TPH_CONST]);
    cx<T> F0[R], F1[R];
    GV_UNROLL
    for (int s = 0; s < R; ++s) {
        const int i = sg.reg_rz[s];
        if (i >= 0) { const cx<T> cs = pv.cs[i]; F0[s] = cx<T>{cs.x, -cs.y}; F1[s] = cs; }
        else { F0[s] = cx<T>{T(1), T(0)}; F1[s] = F0[s]; }
    }
    for (uint32_t e = sg.trz_begin; e < sg.trz_begin + sg.n_xreg; ++e) {   // rare: a further R_z on a register slot
        const DTrz t = pv.trz[e];
        const cx<T> cs = pv.cs[t.cs];
        GV_UNROLL
        for (int s = 0; s < R; ++s)
            if (t.tb - TB_XREG == s) { F0[s] = cmul(F0[s], cx<T>{cs.x, -cs.y}); F1[s] = cmul(F1[s], cs); }
    }
    uint32_t par = 0;
    for (uint32_t e = sg.tcz_begin; e < sg.tcz_begin + sg.n_cross; ++e) {
        const uint64_t m = pv.tcz[e] & ((1ull << TCZ_CLASS_SHIFT) - 1ull);
        par ^= ((x & m) == m) ? 1u : 0u;
    }
    if (par) ph = cneg(ph);
    GV_UNROLL
    for (int s = 0; s < R; ++s)
        if (gv_popcll(x & sg.nbr[s]) & 1) F1[s] = cneg(F1[s]);
    cx<T> tlo[1 << RL], thi[1 << RH];
    tlo[0] = ph;
    GV_UNROLL
    for (int s = 0; s < RL; ++s) {
        GV_UNROLL
        for (int e = 0; e < (1 << s); ++e) { tlo[e | (1 << s)] = cmul(tlo[e], F1[s]); tlo[e] = cmul(tlo[e], F0[s]); }
    }
    thi[0] = cx<T>{T(1), T(0)};
    GV_UNROLL
    for (int s = 0; s < RH; ++s) {
        GV_UNROLL
        for (int e = 0; e < (1 << s); ++e) { thi[e | (1 << s)] = cmul(thi[e], F1[RL + s]); thi[e] = cmul(thi[e], F0[RL + s]); }
    }
    cx<T> tlosw[1 << RL], thisw[1 << RH];
    GV_UNROLL
    for (int e = 0; e < (1 << RL); ++e) tlosw[e] = cx<T>{-tlo[e].y, tlo[e].x};
    GV_UNROLL
    for (int e = 0; e < (1 << RH); ++e) thisw[e] = cx<T>{-thi[e].y, thi[e].x};
    const uint32_t neg = sg.regreg_neg;
    GV_UNROLL
    for (int r = 0; r < (1 << R); ++r) {
        cx<T> v = cmul_w<T>(a[r], tlo[r & ((1 << RL) - 1)], tlosw[r & ((1 << RL) - 1)]);
        v = cmul_w<T>(v, thi[r >> RL], thisw[r >> RL]);
        a[r] = v;
    }
    if (neg) {
        GV_UNROLL
        for (int r = 0; r < (1 << R); ++r)
            if ((neg >> r) & 1u) a[r] = cneg(a[r]);
    }
}

// Per-stage thread lookups (host-built, lower.cpp): the thread's local index j (register bits zero), its swizzled
// offset and its global index are GF(2)-linear in the thread index, so each is the XOR / OR of a low-bits entry and a
// high-bits entry.  u32 entry = j | swizzled element offset << 16; u64 entry = scatter(j).

// One stage: 2^R amplitudes per thread in registers, all micro-ops of the stage, back to shared memory.
// Returns true when the stage ends with a CNOT run: the amplitudes then stay in a[] and must be written by
// gate_stage_store after a barrier.  All shared-memory addressing is in swizzled BYTE offsets (XOR only).
template <typename T, int R>
GV_DEV bool gate_stage(const ProgView<T> &pv, const DStage &st, uint32_t si, unsigned char *tile, uint32_t tid,
                       uint64_t xbase, cx<T> *a, uint32_t *po, uint32_t &pj2)
{
    constexpr int NR = 1 << R;
    const uint32_t *w32 = reinterpret_cast<const uint32_t *>(pv.slut + (size_t)si * SLUT_ENTRIES * 12u);
    const uint64_t *w64 = reinterpret_cast<const uint64_t *>(w32 + SLUT_ENTRIES);
    const uint32_t lo = tid & 15u, hi = 16u + (tid >> 4);
    const uint32_t w = w32[lo] ^ w32[hi];
    const uint32_t j = w & 0xFFFFu, pjb = (w >> 16) * (uint32_t)sizeof(cx<T>);
    const uint64_t x = xbase | w64[lo] | w64[hi];
    GV_UNROLL
    for (int s = 0; s < R; ++s) po[s] = st.po_bytes[s];
    GV_UNROLL
    for (int r = 0; r < NR; ++r) {
        uint32_t o = pjb;
        GV_UNROLL
        for (int s = 0; s < R; ++s) if (r & (1 << s)) o ^= po[s];
        a[r] = *reinterpret_cast<const cx<T> *>(tile + o);
    }
    for (uint32_t oi = st.op_begin; oi < st.op_end; ++oi) {
        const DOp o = pv.ops[oi];
        if (o.kind == MOP_RYL) ry_layer<T, R>(a, pv.ryl + o.idx, pv.cs);
        else diag_apply<T, R>(a, pv, pv.segs[o.idx], (uint32_t)o.idx, x, tid);
    }
    if (!st.has_cx) {
        GV_UNROLL
        for (int r = 0; r < NR; ++r) {
            uint32_t o = pjb;
            GV_UNROLL
            for (int s = 0; s < R; ++s) if (r & (1 << s)) o ^= po[s];
            *reinterpret_cast<cx<T> *>(tile + o) = a[r];
        }
        return false;
    }
    // Trailing CNOT run: |j> -> |A j ^ c>, A linear over GF(2).  The amplitude of logical index
    // j_thread ^ j_r is written to  A j_thread ^ c  ^  A j_r : the thread part is updated CNOT by CNOT, the register
    // part comes from the precomputed images of the register unit vectors.  No register work at all.
    uint32_t jj = j;
    for (uint32_t ci = st.cx_begin; ci < st.cx_end; ++ci) {
        const DCx c = pv.cxs[ci];
        const uint32_t bit = (c.cl != 255) ? ((jj >> c.cl) & 1u) : (uint32_t)((xbase >> c.cq) & 1ull);
        jj ^= bit << c.tl;
    }
    pj2 = phys<T>(jj) * (uint32_t)sizeof(cx<T>);
    GV_UNROLL
    for (int s = 0; s < R; ++s) po[s] = st.post_bytes[s];
    return true;
}

// Second half of a stage that ends with a CNOT run; called after a block-wide barrier (every thread has read its
// amplitudes before any thread overwrites another thread's locations).
template <typename T, int R>
GV_DEV void gate_stage_store(unsigned char *tile, uint32_t pj2, const uint32_t *po, const cx<T> *a)
{
    GV_UNROLL
    for (int r = 0; r < (1 << R); ++r) {
        uint32_t o = pj2;
        GV_UNROLL
        for (int s = 0; s < R; ++s) if (r & (1 << s)) o ^= po[s];
        *reinterpret_cast<cx<T> *>(tile + o) = a[r];
    }
}

// ---- Hamiltonian engine ----------------------------------------------------------------------------------
// Tile load of the expectation kernel, NLD 16-byte vectors per thread, all loads in flight; the diagonal part
// sum_x |psi[x]|^2 E(x) (E = diagonal energy table) is accumulated on the way.
template <typename T, typename TT, int NLD>
GV_DEV double expect_load_u(cx<T> *tile, const cx<T> *state, const TT *table, bool with_diag, uint64_t xbase,
                            const Run *runs, int n_runs, uint32_t tid, uint32_t nthr, const uint64_t *hi)
{
    constexpr uint32_t V = 16 / sizeof(cx<T>);
    struct alignas(V * sizeof(TT)) tvec { TT t[V]; };
    const uint64_t x0 = xbase | scatter_runs(tid * V, runs, n_runs);
    const uint32_t p0 = phys<T>(tid * V);
    vec16<T> v[NLD];
    tvec tv[NLD];
    GV_UNROLL
    for (int i = 0; i < NLD; ++i) v[i] = *reinterpret_cast<const vec16<T> *>(state + (x0 | hi[i]));
    if (with_diag) {
        GV_UNROLL
        for (int i = 0; i < NLD; ++i) tv[i] = *reinterpret_cast<const tvec *>(table + (x0 | hi[i]));
    }
    T acc = T(0);
    GV_UNROLL
    for (int i = 0; i < NLD; ++i) {
        const uint32_t p = p0 ^ phys<T>((uint32_t)i * nthr * V);
        GV_UNROLL
        for (uint32_t e = 0; e < V; ++e) {
            tile[p ^ e] = v[i].v[e];
            if (with_diag) acc += (v[i].v[e].x * v[i].v[e].x + v[i].v[e].y * v[i].v[e].y) * (T)tv[i].t[e];
        }
    }
    return (double)acc;
}

// Table-mode group with thread-constant W: the thread's 2^L pairs differ only in the loop bits, which lie outside
// the table index bits, so  sum_pairs Re(conj(b) W a) = Re(W * sum_pairs conj(b) a).
// Table-mode group with thread-constant W: the thread's 2^L pairs differ only in the loop bits, which lie outside the
// table index bits, so  sum_pairs Re(conj(b) W a) = Re(W * sum_pairs conj(b) a).  Every index comes from the group's
// host-built lookup block (devprog.h GT_WORDS): two table reads
// give the thread's swizzled byte offset and its W index, the loop-bit combinations are broadcast reads.
template <typename T, int L>
GV_DEV double group_accumulate_lut(const uint32_t *gt, uint32_t pm_bytes, uint32_t tab_off, const unsigned char *tile_bytes,
                                   const cx<T> *tab, uint32_t tid)
{
    const uint32_t w0 = gt[tid & 15u] ^ gt[16u + (tid >> 4)];
    const uint32_t pjb = w0 & 0xFFFFFu;
    const cx<T> w = tab[tab_off + (w0 >> 20)];
    uint32_t cmb[1 << L];   // loop-bit combinations: broadcast reads, four words at a time
    GV_UNROLL
    for (int i = 0; i < (1 << L); i += 4) {
        struct alignas(16) u4 { uint32_t a, b, c, d; };
        const u4 q = *reinterpret_cast<const u4 *>(gt + 32 + i);
        cmb[i] = q.a; cmb[i + 1] = q.b; cmb[i + 2] = q.c; cmb[i + 3] = q.d;
    }
    T tr = T(0), ti = T(0);
    if constexpr (sizeof(T) == 4) {
        // packed: accA += b.x * (a.x, a.y), accB += b.y * (a.y, a.x); Re = accA.x + accB.x, Im = accA.y - accB.y
        float2 accA = make_float2(0.f, 0.f), accB = make_float2(0.f, 0.f);
        GV_UNROLL
        for (int i = 0; i < (1 << L); ++i) {
            const uint32_t ob = pjb ^ cmb[i];
            const float2 a = *reinterpret_cast<const float2 *>(tile_bytes + ob);
            const float2 b = *reinterpret_cast<const float2 *>(tile_bytes + (ob ^ pm_bytes));
            accA = __ffma2_rn(make_float2(b.x, b.x), a, accA);
            accB = __ffma2_rn(make_float2(b.y, b.y), make_float2(a.y, a.x), accB);
        }
        tr = accA.x + accB.x;
        ti = accA.y - accB.y;
        return 2.0 * (double)(w.x * tr - w.y * ti);
    }
    GV_UNROLL
    for (int i = 0; i < (1 << L); ++i) {
        const uint32_t ob = pjb ^ cmb[i];
        const cx<T> a = *reinterpret_cast<const cx<T> *>(tile_bytes + ob);
        const cx<T> b = *reinterpret_cast<const cx<T> *>(tile_bytes + (ob ^ pm_bytes));
        tr = b.x * a.x + tr; tr = b.y * a.y + tr;     // Re conj(b) a
        ti = b.x * a.y + ti; ti = -b.y * a.x + ti;    // Im conj(b) a
    }
    return 2.0 * (double)(w.x * tr - w.y * ti);
}

// ---- register-stage groups: amplitudes and partners in registers, W (indexed by the register index) broadcast ------
template <int M> struct TopBit { static constexpr int value = 1 + TopBit<(M >> 1)>::value; };
template <> struct TopBit<1> { static constexpr int value = 0; };
template <> struct TopBit<0> { static constexpr int value = 0; };

template <typename T, int R, int M> GV_DEV T rs_pairs(const cx<T> *a, const cx<T> *w)
{
    constexpr int PV = TopBit<M>::value;
    if constexpr (sizeof(T) == 4) {
        // packed: accA += v.x * (w.x u.x, w.y u.y), accB += v.y * (w.x u.y, w.y u.x);
        // Re(w conj(v) u) summed = (accA.x - accA.y) + (accB.x + accB.y).  Two chains each.
        float2 accA[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
        float2 accB[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
        int n = 0;
        GV_UNROLL
        for (int r = 0; r < (1 << R); ++r) {
            if (r & (1 << PV)) continue;
            const float2 ww = make_float2(w[r].x, w[r].y), u = make_float2(a[r].x, a[r].y);
            const cx<T> v = a[r ^ M];
            const float2 g = __fmul2_rn(ww, u);
            const float2 h = __fmul2_rn(ww, make_float2(u.y, u.x));
            accA[n & 1] = __ffma2_rn(make_float2(v.x, v.x), g, accA[n & 1]);
            accB[n & 1] = __ffma2_rn(make_float2(v.y, v.y), h, accB[n & 1]);
            ++n;
        }
        const float2 sa = __fadd2_rn(accA[0], accA[1]), sb = __fadd2_rn(accB[0], accB[1]);
        return (sa.x - sa.y) + (sb.x + sb.y);
    }
    T acc[4] = {T(0), T(0), T(0), T(0)};   // independent chains
    int n = 0;
    GV_UNROLL
    for (int r = 0; r < (1 << R); ++r) {
        if (r & (1 << PV)) continue;
        const cx<T> ww = w[r], u = a[r], v = a[r ^ M];
        T tr = v.x * u.x; tr = v.y * u.y + tr;      // Re conj(v) u
        T ti = v.x * u.y; ti = -v.y * u.x + ti;     // Im conj(v) u
        acc[n & 3] = ww.x * tr + acc[n & 3];
        acc[(n + 2) & 3] = -ww.y * ti + acc[(n + 2) & 3];
        ++n;
    }
    return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}

// binary search over the flip mask (uniform branches): masks LO..HI  (an indexed branch measured slower)
template <typename T, int R, int LO, int HI> struct RsDispatch {
    static GV_DEV T run(int m, const cx<T> *a, const cx<T> *w)
    {
        if constexpr (LO == HI) return rs_pairs<T, R, LO>(a, w);
        else {
            constexpr int MID = (LO + HI) / 2;
            if (m <= MID) return RsDispatch<T, R, LO, MID>::run(m, a, w);
            return RsDispatch<T, R, MID + 1, HI>::run(m, a, w);
        }
    }
};

template <typename T, int R>
GV_DEV void rs_load(cx<T> *a, const DRs &rs, const unsigned char *tile_bytes, uint32_t tid)
{
    uint32_t j = tid;
    GV_UNROLL
    for (int s = 0; s < R; ++s) j = insert_zero(j, rs.regbit[s]);
    const uint32_t pjb = phys<T>(j) * (uint32_t)sizeof(cx<T>);
    GV_UNROLL
    for (int r = 0; r < (1 << R); ++r) {
        uint32_t o = pjb;
        GV_UNROLL
        for (int s = 0; s < R; ++s) if (r & (1 << s)) o ^= rs.po_bytes[s];
        a[r] = *reinterpret_cast<const cx<T> *>(tile_bytes + o);
    }
}

// W_g(u) = sum_k c_k i^{nY_k} (-1)^{popcount(x & z_k)} for the table index u of group g (tile-constant part of the
// sign from the bits outside the tile).  One entry per call.
template <typename T>
GV_DEV cx<T> group_table_entry(uint32_t term_begin, uint32_t dyn_end, const DTerm *terms, uint64_t xbase, uint32_t u,
                               cx<T> w0)
{
    double wr = (double)w0.x, wi = (double)w0.y;   // static part (terms with no z bit outside the tile)
    uint32_t t = term_begin;
    for (; t + 4 <= dyn_end; t += 4) {   // four independent loads in flight
        DTerm tm[4];
        GV_UNROLL
        for (int q = 0; q < 4; ++q) tm[q] = terms[t + q];
        GV_UNROLL
        for (int q = 0; q < 4; ++q) {
            const int par = (gv_popcll(xbase & tm[q].zout) + gv_popc(u & tm[q].zu)) & 1;
            wr += par ? -tm[q].cr : tm[q].cr;
            wi += par ? -tm[q].ci : tm[q].ci;
        }
    }
    for (; t < dyn_end; ++t) {
        const DTerm tm = terms[t];
        const int par = (gv_popcll(xbase & tm.zout) + gv_popc(u & tm.zu)) & 1;
        wr += par ? -tm.cr : tm.cr;
        wi += par ? -tm.ci : tm.ci;
    }
    return cx<T>{(T)wr, (T)wi};
}

// 2 Re sum over pairs (x, x^m), x with the pivot bit clear, of conj(psi[x^m]) W(x) psi[x].
template <typename T>
GV_DEV double group_accumulate(const DGroup &g, const DTerm *terms, const cx<T> *tile, const cx<T> *tab, uint64_t xbase,
                               int k, uint32_t tid, uint32_t nthr)
{
    const uint32_t pm = phys<T>(g.m_loc);
    const uint32_t npair = 1u << (k - 1);
    double acc = 0.0;
    T part = T(0);
    uint32_t cnt = 0;
    for (uint32_t i = tid; i < npair; i += nthr) {
        const uint32_t j = insert_zero(i, g.pivot);
        const uint32_t pj = phys<T>(j);
        const cx<T> a = tile[pj], b = tile[pj ^ pm];
        cx<T> w;
        if (g.direct) {
            double wr = 0.0, wi = 0.0;
            for (uint32_t t = g.term_begin; t < g.term_end; ++t) {
                const DTerm tm = terms[t];
                const int par = (gv_popcll(xbase & tm.zout) + gv_popc(j & tm.zu)) & 1;
                wr += par ? -tm.cr : tm.cr;
                wi += par ? -tm.ci : tm.ci;
            }
            w = cx<T>{(T)wr, (T)wi};
        } else {
            uint32_t u = 0;
            for (int r = 0; r < g.n_uruns; ++r)
                u |= ((j >> g.uruns[r].lpos) & ((1u << g.uruns[r].len) - 1u)) << g.uruns[r].shift;
            w = tab[g.tab_off + u];
        }
        const T tr = b.x * a.x + b.y * a.y;   // conj(b) * a
        const T ti = b.x * a.y - b.y * a.x;
        part += w.x * tr - w.y * ti;
        if (++cnt == 16) { acc += (double)part; part = T(0); cnt = 0; }
    }
    acc += (double)part;
    return 2.0 * acc;
}

}  // namespace gv

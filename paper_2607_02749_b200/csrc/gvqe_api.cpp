// gvqe_api.cpp -- the C ABI of include/gvqe.h on top of the schedule compiler, the Hamiltonian planner and the
// sm_100a kernels.  Host C++ (compiled by nvcc as host code); allocates no device memory: everything lives in
// the caller's workspace.  No CPU fallback: every energy is computed by the kernels in kernels.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <thread>
#include <utility>
#include <vector>

#include "../../include/gvqe.h"
#include "graph.h"
#include "hamiltonian.h"
#include "jit.h"
#include "kernels.h"
#include "lower.h"
#include "schedule.h"

using namespace gv;

namespace {
constexpr int N_MIN_STORE = 10;   // smaller registers are padded with idle qubits (they stay |0>)
constexpr int N_MAX = 34;
inline size_t al256(size_t v) { return (v + 255) & ~(size_t)255; }
}  // namespace

struct gvqe_ctx {
    int n_user = 0, n_store = 0, prec = 0, P = 0;
    int K = 0, F = 0, R = 0, KE = 0;   // KE: tile bits of the expectation passes
    std::vector<HostOp> ops;
    Program prog;
    Program prog_generic;   // when prog carries in-register CNOTs (specialised kernels only): the program dev was lowered from
    DevProgram dev;
    Prefix px;               // product-state prefix of the op list (written, not simulated)
    PrefixDev pxd{};
    bool have_h = false;
    Hamiltonian H;
    ExpectPlan plan;
    std::vector<TileDesc> fwht_tiles;
    std::vector<uint32_t> fwht_masks;
    // workspace
    char *ws = nullptr;
    size_t ws_bytes = 0;
    int max_in_flight = 0, in_flight = 0;
    bool dirty = true;          // device arrays / table must be (re)built
    bool kernels_ready = false;
    // carved device pointers
    GateLaunch gl{};
    DPass *d_passes = nullptr; DGroup *d_groups = nullptr; DTerm *d_terms = nullptr;
    uint64_t *d_diag_z = nullptr; double *d_diag_c = nullptr; void *d_wstat = nullptr; uint32_t *d_gtabs = nullptr; DRs *d_rss = nullptr;
    std::vector<float> wstat_f;
    void *d_table = nullptr; void *d_states = nullptr; void *d_cs = nullptr; void *d_readout = nullptr;
    double *d_params = nullptr, *d_partial = nullptr, *d_E = nullptr;
    uint32_t slots_per_b = 0;
    uint64_t launches = 0;
    // profiling (gvqe_profile_enable): 4 events per chunk
    gvqe_options opt{};
    // schedule-specialised gate kernels (jit.h): generated at create, compiled and loaded at the first energy call
    int jit_state = 0;          // 0 not tried, 1 loaded, -1 not used
    int sm_count = 148;
    int jit_per_cta = 8;        // work items per thread block of the specialised kernels (tuned on the B200)
    std::vector<JitBlock> jit_blocks;
    std::vector<JitModule *> jit_mods;
    void *d_ry = nullptr;
    int jitx_state = -1;        // expectation passes: -1 not used, 0 generated (to be loaded), 1 loaded
    std::vector<JitBlock> jitx_blocks;
    std::vector<JitModule *> jitx_mods;
    JitExpectData jitx;
    std::vector<float> jitx_wst_f;
    void *d_jwst = nullptr; void *d_jpats = nullptr; void *d_jterms = nullptr;
    int32_t *d_sweep_idx = nullptr; double *d_sweep_E = nullptr;
    bool profiling = false;
    std::vector<cudaEvent_t> ev;
    double prof_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    std::vector<cudaEvent_t> ev_fine;          // profiling: one event after every gate launch / expectation pass of a chunk
    std::vector<double> prof_launch_ms;        // summed per launch index (prefix kernel, gate blocks, passes)
    std::vector<double> prof_launch_min, prof_launch_max;
    double prof_fine_chunks = 0;
    std::string err;
    size_t amp_bytes() const { return prec == GVQE_C64 ? 8 : 16; }
    size_t tab_bytes() const { return prec == GVQE_C64 ? 4 : 8; }
};

namespace {

gvqe_status fail(gvqe_ctx *c, gvqe_status s, const std::string &m) { if (c) c->err = m; return s; }
gvqe_status cuda_fail(gvqe_ctx *c, int e, const char *what)
{
    c->err = std::string(what) + ": " + cudaGetErrorString((cudaError_t)e);
    return GVQE_ERR_CUDA;
}

gvqe_status build_ctx(int n, const std::vector<HostOp> &ops, int n_params, gvqe_precision prec, const gvqe_options *opt, gvqe_ctx **out)
{
    if (!out) return GVQE_ERR_INVALID_ARG;
    *out = nullptr;
    if (n < 1 || n > N_MAX || (prec != GVQE_C64 && prec != GVQE_C128) || n_params < 0) return GVQE_ERR_INVALID_ARG;
    std::vector<char> used((size_t)n_params, 0);
    for (const HostOp &o : ops) {
        if (o.kind < 0 || o.kind > 3 || o.q0 < 0 || o.q0 >= n) return GVQE_ERR_INVALID_ARG;
        if (o.kind >= 2 && (o.q1 < 0 || o.q1 >= n || o.q1 == o.q0)) return GVQE_ERR_INVALID_ARG;
        if (o.kind <= 1) {
            if (o.param < 0 || o.param >= n_params || used[o.param]) return GVQE_ERR_INVALID_ARG;
            used[o.param] = 1;   // a parameter drives at most one gate: Eq. 13 is then exact
        }
    }
    gvqe_ctx *c = new gvqe_ctx();
    c->n_user = n; c->n_store = n < N_MIN_STORE ? N_MIN_STORE : n; c->prec = prec; c->P = n_params; c->ops = ops;
    if (opt) {
        c->opt = *opt;
        bool bad = opt->tile_bits > 14 || opt->fixed_bits > 8 || opt->reg_bits > 5 || opt->expect_tile_bits > 14 || opt->tile_bits < 0 || opt->fixed_bits < 0 || opt->reg_bits < 0 || opt->expect_tile_bits < 0 || opt->prefix < 0 ||
                   opt->prefix > 2 || opt->register_stages < 0 || opt->register_stages > 1 || opt->shared_prefix < 0 ||
                   opt->shared_prefix > 2 || opt->specialise < 0 || opt->specialise > 2 || opt->tiles_per_block < 0 || opt->tiles_per_block > 4096 ||
                   (opt->blocks_per_sm != 0 && opt->blocks_per_sm != 2 && opt->blocks_per_sm != 3) || opt->staged_io < 0 || opt->staged_io > 1 ||
                   opt->mid_cnot < 0 || opt->mid_cnot > 1 ||
                   opt->interleave < 0 || opt->interleave > 1024 || (opt->interleave & (opt->interleave - 1)) != 0;
        for (int32_t r : opt->reserved) bad = bad || r != 0;
        if (bad) { delete c; return GVQE_ERR_INVALID_ARG; }
    }
    if (c->opt.tiles_per_block) c->jit_per_cta = c->opt.tiles_per_block;
    c->K = c->opt.tile_bits ? c->opt.tile_bits : (prec == GVQE_C64 ? 13 : 12);
    c->F = c->opt.fixed_bits ? c->opt.fixed_bits : (prec == GVQE_C64 ? 4 : 3);
    c->R = c->opt.reg_bits ? c->opt.reg_bits : (prec == GVQE_C64 ? 5 : 4);
    if (c->K > c->n_store) c->K = c->n_store;
    c->KE = c->opt.expect_tile_bits ? c->opt.expect_tile_bits : (c->K > (prec == GVQE_C64 ? 13 : 12) ? (prec == GVQE_C64 ? 13 : 12) : c->K);
    if (c->KE > c->n_store) c->KE = c->n_store;
    if (c->K < c->R + 5 || c->K > 14 || c->F < 1 || c->F >= c->K || c->K - c->R > 9) { delete c; return GVQE_ERR_INVALID_ARG; }
    std::string err;
    // Two candidate schedules: everything through the fused blocks (first block write-only), or the product-state
    // prefix written by its own kernel and the rest through the blocks.  Fewer HBM passes wins (ties: no prefix).
    if (!compile_program(c->n_store, c->ops, c->K, c->F, c->R, c->prog, err, true) ||
        !lower_program(c->prog, (int)c->amp_bytes(), c->dev, err)) {
        delete c;
        return GVQE_ERR_UNSUPPORTED;
    }
    Prefix px = c->opt.prefix == 1 ? Prefix() : find_prefix(c->n_store, c->ops);
    if (px.n_ops > 0) {
        Program prog2; DevProgram dev2;
        const std::vector<HostOp> rest(c->ops.begin() + px.n_ops, c->ops.end());
        if (compile_program(c->n_store, rest, c->K, c->F, c->R, prog2, err, false) &&
            lower_program(prog2, (int)c->amp_bytes(), dev2, err)) {
            const size_t passes_plain = 2 * c->dev.blocks.size() - 1, passes_px = 1 + 2 * dev2.blocks.size();
            if (passes_px < passes_plain || c->opt.prefix == 2) { c->px = px; c->prog = prog2; c->dev = dev2; }
        }
    }
    if (c->px.n_ops > 0) {   // execution order in terms of the caller's op list: prefix first, then the compiled rest
        std::vector<int> eo;
        for (int i = 0; i < c->px.n_ops; ++i) eo.push_back(i);
        for (int e : c->prog.exec_order) eo.push_back(e + c->px.n_ops);
        c->prog.exec_order.swap(eo);
    }
    // specialised gate kernels: source only here (host work); compiled and loaded by ensure_ready on the device
    {
        std::string why;
        const bool want = c->opt.specialise == 2 || (c->opt.specialise == 0 && c->n_store >= 20);
        if (want && c->opt.mid_cnot == 0) {   // the specialised kernels apply CNOTs on register qubits in registers: fewer stages
            Program pj;
            const std::vector<HostOp> rest(c->ops.begin() + c->px.n_ops, c->ops.end());
            if (compile_program(c->n_store, rest, c->K, c->F, c->R, pj, err, c->px.n_ops == 0, true) && pj.blocks.size() == c->prog.blocks.size() &&
                pj.stages.size() < c->prog.stages.size() && jit_supported(pj, c->prec, why)) {
                if (c->px.n_ops > 0) {
                    std::vector<int> eo;
                    for (int i = 0; i < c->px.n_ops; ++i) eo.push_back(i);
                    for (int e : pj.exec_order) eo.push_back(e + c->px.n_ops);
                    pj.exec_order.swap(eo);
                }
                c->prog_generic = c->prog;   // c->dev (the generic kernels' program) stays the lowering of this one
                c->prog = pj;
            }
        }
        if (want && c->prog.blocks.size() == c->dev.blocks.size() && jit_supported(c->prog, c->prec, why)) {
            c->jit_blocks.resize(c->prog.blocks.size());
            for (size_t b = 0; b < c->prog.blocks.size(); ++b)
                if (!jit_generate(c->prog, (int)b, c->prec, c->opt.blocks_per_sm, c->opt.staged_io != 0, c->opt.interleave ? c->opt.interleave : 32, c->jit_blocks[b], why)) { c->jit_blocks.clear(); break; }
        }
        if (c->jit_blocks.empty()) {
            c->jit_state = -1;
            if (!c->prog_generic.blocks.empty()) { c->prog = c->prog_generic; c->prog_generic = Program(); }
        }
    }
    *out = c;
    return GVQE_OK;
}

}  // namespace

extern "C" {

gvqe_status gvqe_create(int n, const gvqe_layout *L, gvqe_precision prec, gvqe_ctx **out)
{
    return gvqe_create_opt(n, L, prec, nullptr, out);
}

gvqe_status gvqe_create_ops(int n, const gvqe_op *ops, int n_ops, int n_params, gvqe_precision prec, gvqe_ctx **out)
{
    return gvqe_create_ops_opt(n, ops, n_ops, n_params, prec, nullptr, out);
}

size_t gvqe_kernel_source(const gvqe_ctx *c, int block, char *buf, size_t cap, int32_t *smem_bytes)
{
    if (!c || block < 0 || (size_t)block >= c->jit_blocks.size() + c->jitx_blocks.size()) return 0;
    const JitBlock &jb = (size_t)block < c->jit_blocks.size() ? c->jit_blocks[(size_t)block] : c->jitx_blocks[(size_t)block - c->jit_blocks.size()];
    const std::string &s = jb.source;
    if (smem_bytes) *smem_bytes = (int32_t)jb.smem_bytes;
    if (buf && cap) { const size_t m = s.size() < cap - 1 ? s.size() : cap - 1; memcpy(buf, s.data(), m); buf[m] = 0; }
    return s.size() + 1;
}

gvqe_status gvqe_kernel_info(const gvqe_ctx *c, int block, double *out)
{
    if (!c || !out || block < 0 || (size_t)block >= c->jit_blocks.size() + c->jitx_blocks.size()) return GVQE_ERR_INVALID_ARG;
    const bool gate = (size_t)block < c->jit_blocks.size();
    const JitBlock &jb = gate ? c->jit_blocks[(size_t)block] : c->jitx_blocks[(size_t)block - c->jit_blocks.size()];
    out[0] = gate ? 0.0 : 1.0; out[1] = (double)jb.smem_bytes; out[2] = jb.fma_ops_per_amp; out[3] = 0.0;
    return GVQE_OK;
}

size_t gvqe_kernel_arrays(const gvqe_ctx *c, int which, void *buf, size_t cap)
{
    if (!c || c->jitx_blocks.empty()) return 0;
    std::vector<uint32_t> pp;
    const void *src = nullptr;
    size_t bytes = 0;
    switch (which) {
    case 0: src = c->jitx.wst.data(); bytes = c->jitx.wst.size() * 8; break;
    case 1: src = c->jitx.pats.data(); bytes = c->jitx.pats.size() * sizeof(JitExpectData::Pat); break;
    case 2: src = c->jitx.terms.data(); bytes = c->jitx.terms.size() * sizeof(JitExpectData::Term); break;
    case 3:
        for (size_t p = 0; p < c->jitx.pass_wst_off.size(); ++p) { pp.push_back(c->jitx.pass_wst_off[p]); pp.push_back(c->jitx.pass_pat_off[p]); pp.push_back(c->jitx.pass_pat_cnt[p]); }
        src = pp.data(); bytes = pp.size() * 4; break;
    default: return 0;
    }
    if (buf && cap && bytes) memcpy(buf, src, bytes < cap ? bytes : cap);
    return bytes;
}

gvqe_status gvqe_compile_kernels(gvqe_ctx *c, int32_t *n_kernels)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (n_kernels) *n_kernels = 0;
    std::vector<const JitBlock *> all;
    for (const JitBlock &jb : c->jit_blocks) all.push_back(&jb);
    for (const JitBlock &jb : c->jitx_blocks) all.push_back(&jb);
    const size_t nbk = all.size();
    std::vector<std::string> errs(nbk);
    std::vector<char> ok(nbk, 0);
    for (size_t b0 = 0; b0 < nbk; b0 += 8) {
        std::vector<std::thread> th;
        for (size_t b = b0; b < nbk && b < b0 + 8; ++b)
            th.emplace_back([&all, b, &errs, &ok] { std::vector<char> img; ok[b] = jit_compile_only(*all[b], img, errs[b]) ? 1 : 0; });
        for (std::thread &t : th) t.join();
    }
    for (size_t b = 0; b < nbk; ++b) if (!ok[b]) return fail(c, GVQE_ERR_UNSUPPORTED, errs[b]);
    if (n_kernels) *n_kernels = (int32_t)nbk;
    return GVQE_OK;
}

gvqe_status gvqe_create_opt(int n, const gvqe_layout *L, gvqe_precision prec, const gvqe_options *opt, gvqe_ctx **out)
{
    if (!L || !out || n < 1 || n > N_MAX) return GVQE_ERR_INVALID_ARG;
    if (L->n_layers < 0 || L->n_layers > 4096 || (L->entangler != GVQE_OP_CZ && L->entangler != GVQE_OP_CNOT) ||
        (L->topology < 0 || L->topology > 6) || (L->final_rot != 1 && L->final_rot != 2))
        return GVQE_ERR_INVALID_ARG;
    // D x (RY layer, RZ layer, entanglers), then the final rotation layer.
    std::vector<HostOp> ops;
    const int D = L->n_layers;
    for (int l = 0; l < D; ++l) {
        for (int q = 0; q < n; ++q) ops.push_back({GVQE_OP_RY, q, -1, 2 * n * l + q});
        for (int q = 0; q < n; ++q) ops.push_back({GVQE_OP_RZ, q, -1, 2 * n * l + n + q});
        // (control, target) pairs of the layer's entanglement map (reading A17)
        std::vector<std::pair<int, int>> pr;
        const bool wrap = n > 2;
        switch (L->topology) {
        case 0: case 1:
            for (int q = 0; q + 1 < n; ++q) pr.push_back({q, q + 1});
            if (L->topology == 1 && wrap) pr.push_back({n - 1, 0});
            break;
        case 2:
            for (int i = 0; i < n; ++i) for (int j = i + 1; j < n; ++j) pr.push_back({i, j});
            break;
        case 3:
            for (int q = n - 2; q >= 0; --q) pr.push_back({q, q + 1});
            break;
        case 4:
            for (int par = 0; par < 2; ++par) for (int q = par; q + 1 < n; q += 2) pr.push_back({q, q + 1});
            break;
        case 5:
            if (wrap) pr.push_back({n - 1, 0});
            for (int q = 0; q + 1 < n; ++q) pr.push_back({q, q + 1});
            break;
        default: {   // 6, shifted-circular-alternating
            if (!wrap) { for (int q = 0; q + 1 < n; ++q) pr.push_back({q, q + 1}); break; }
            for (int j = 0; j < n; ++j) {
                const int e = ((j - l) % n + n) % n;          // entry e of the circular list: (e-1, e), e = 0: (n-1, 0)
                std::pair<int, int> p = e == 0 ? std::make_pair(n - 1, 0) : std::make_pair(e - 1, e);
                if (l & 1) std::swap(p.first, p.second);
                pr.push_back(p);
            }
        }
        }
        for (const auto &p : pr) {
            if (L->entangler == GVQE_OP_CZ) ops.push_back({GVQE_OP_CZ, p.first, p.second, -1});
            else ops.push_back({GVQE_OP_CNOT, p.second, p.first, -1});
        }
    }
    for (int q = 0; q < n; ++q) ops.push_back({GVQE_OP_RY, q, -1, 2 * n * D + q});
    if (L->final_rot == 2) for (int q = 0; q < n; ++q) ops.push_back({GVQE_OP_RZ, q, -1, 2 * n * D + n + q});
    return build_ctx(n, ops, 2 * n * D + n * L->final_rot, prec, opt, out);
}

gvqe_status gvqe_create_ops_opt(int n, const gvqe_op *ops, int n_ops, int n_params, gvqe_precision prec, const gvqe_options *opt,
                                gvqe_ctx **out)
{
    if (n_ops < 0 || (n_ops > 0 && !ops)) return GVQE_ERR_INVALID_ARG;
    std::vector<HostOp> v((size_t)n_ops);
    for (int i = 0; i < n_ops; ++i) v[i] = HostOp{ops[i].kind, ops[i].q0, ops[i].q1, ops[i].param};
    return build_ctx(n, v, n_params, prec, opt, out);
}

int gvqe_num_params(const gvqe_ctx *c) { return c ? c->P : -1; }
int gvqe_num_qubits(const gvqe_ctx *c) { return c ? c->n_user : -1; }

static gvqe_status after_hamiltonian(gvqe_ctx *c)
{
    std::string err;
    if (!plan_expectation(c->H, c->n_store, c->KE, c->F, EXPECT_UMAX, EXPECT_TAB_CAP, (int)c->amp_bytes(), c->opt.register_stages == 0, c->plan, err)) {
        c->have_h = false;
        return fail(c, GVQE_ERR_UNSUPPORTED, err);
    }
    // Walsh-Hadamard passes of the diagonal table: low window first, then windows of new high bits
    c->fwht_tiles.clear(); c->fwht_masks.clear();
    const int n = c->n_store, kt = n < 13 ? n : 13, ft = 5;
    int done = 0;
    while (done < n) {
        TileDesc td; memset(&td, 0, sizeof td);
        td.k = (uint8_t)kt;
        uint32_t mask;
        if (done == 0) {
            td.n_runs = 1; td.runs[0] = Run{0, 0, (uint8_t)kt, 0};
            mask = (kt >= 32) ? ~0u : ((1u << kt) - 1);
            done = kt;
        } else {
            const int h = kt - ft;
            int start = done; if (start + h > n) start = n - h;
            td.n_runs = 2; td.runs[0] = Run{0, 0, (uint8_t)ft, 0}; td.runs[1] = Run{(uint8_t)ft, (uint8_t)start, (uint8_t)h, 0};
            mask = 0;
            for (int q = done; q < start + h; ++q) mask |= 1u << (ft + (q - start));
            done = start + h;
        }
        c->fwht_tiles.push_back(td); c->fwht_masks.push_back(mask);
    }
    // specialised expectation kernels: same policy as the gate kernels (gvqe_options.specialise)
    for (JitModule *m : c->jitx_mods) jit_unload(m);
    c->jitx_mods.clear(); c->jitx_blocks.clear(); c->jitx = JitExpectData(); c->jitx_state = -1;
    {
        std::string why;
        const bool want = c->opt.specialise == 2 || (c->opt.specialise == 0 && c->n_store >= 20);
        if (want && jit_expect_supported(c->plan, c->n_store, c->prec, why)) {
            c->jitx_blocks.resize(c->plan.passes.size());
            bool ok = true;
            for (size_t p = 0; p < c->plan.passes.size() && ok; ++p)
                ok = jit_expect_generate(c->plan, c->n_store, c->prec, (int)p, c->jitx, c->jitx_blocks[p], why);
            if (ok) c->jitx_state = 0;
            else { c->jitx_blocks.clear(); c->jitx = JitExpectData(); }
        }
    }
    c->have_h = true; c->dirty = true;
    return GVQE_OK;
}

gvqe_status gvqe_set_hamiltonian(gvqe_ctx *c, int M, const char *paulis, const double *coeffs)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (M < 0 || (M > 0 && (!paulis || !coeffs))) return fail(c, GVQE_ERR_INVALID_ARG, "set_hamiltonian: null input");
    std::string err;
    Hamiltonian H;
    if (!hamiltonian_from_paulis(c->n_user, M, paulis, coeffs, H, err)) return fail(c, GVQE_ERR_INVALID_ARG, err);
    c->H = H;
    return after_hamiltonian(c);
}

gvqe_status gvqe_set_hamiltonian_masks(gvqe_ctx *c, int M, const uint64_t *xm, const uint64_t *zm, const double *coeffs)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (M < 0 || (M > 0 && (!xm || !zm || !coeffs))) return fail(c, GVQE_ERR_INVALID_ARG, "set_hamiltonian_masks: null input");
    std::string err;
    Hamiltonian H;
    if (!hamiltonian_from_masks(c->n_user, M, xm, zm, coeffs, H, err)) return fail(c, GVQE_ERR_INVALID_ARG, err);
    c->H = H;
    return after_hamiltonian(c);
}

gvqe_status gvqe_get_grouping(const gvqe_ctx *c, uint64_t *xm, uint64_t *zm, uint8_t *ny, int32_t *got, int32_t *ng,
                              uint64_t *gmask)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (!c->have_h) return GVQE_ERR_NO_HAMILTONIAN;
    const size_t M = c->H.terms.size();
    for (size_t k = 0; k < M; ++k) {
        if (xm) xm[k] = c->H.terms[k].x;
        if (zm) zm[k] = c->H.terms[k].z;
        if (ny) ny[k] = (uint8_t)(c->H.terms[k].ny & 3);
        if (got) got[k] = c->H.group_of_term[k];
    }
    if (ng) *ng = (int32_t)c->H.group_mask.size();
    if (gmask) for (size_t g = 0; g < c->H.group_mask.size(); ++g) gmask[g] = c->H.group_mask[g];
    return GVQE_OK;
}

}  // extern "C"

// ---- workspace ---------------------------------------------------------------------------------------------
namespace {

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) { const size_t o = off; off = al256(off + bytes); return o; }
};

struct Layout {
    size_t blocks, stages, ops, segs, trzs, tczs, csidx, ryl, cxs, slut, jwst, jpats, jterms, sweep_idx, sweep_E, px_begin, px_kind, px_param, px_t, px_c, passes, groups, terms, wstat, gtabs, rss, dz, dc, readout, smass, su, sx, table, fixed_end;
    size_t per_state;   // state + cs row + params row + partial slots + E
    size_t state_b, cs_b, ry_b, params_b, partial_b;
};

Layout layout_of(const gvqe_ctx *c)
{
    Layout L{};
    Carve cv;
    const DevProgram &d = c->dev;
    L.blocks = cv.take(d.blocks.size() * sizeof(DBlock));
    L.stages = cv.take(d.stages.size() * sizeof(DStage));
    L.ops = cv.take(d.ops.size() * sizeof(DOp));
    L.segs = cv.take(d.segs.size() * sizeof(DSeg));
    L.trzs = cv.take(d.trzs.size() * sizeof(DTrz));
    L.tczs = cv.take(d.tczs.size() * 8);
    L.csidx = cv.take(d.csidx.size() * 4);
    L.ryl = cv.take(d.ryl.size() * 2);
    L.cxs = cv.take(d.cxs.size() * sizeof(DCx));
    L.slut = cv.take(d.slut.size() * 4);
    L.jwst = cv.take(c->jitx.wst.size() / 2 * c->amp_bytes());
    L.jpats = cv.take(c->jitx.pats.size() * sizeof(JitExpectData::Pat));
    L.jterms = cv.take(c->jitx.terms.size() * sizeof(JitExpectData::Term));
    L.sweep_idx = cv.take((size_t)SWEEP_MAX_ROWS * 4);
    L.sweep_E = cv.take((size_t)(SWEEP_MAX_ROWS + 1) * 8);
    L.px_begin = cv.take(c->px.rot_begin.size() * 4); L.px_kind = cv.take(c->px.rot_kind.size());
    L.px_param = cv.take(c->px.rot_param.size() * 4); L.px_t = cv.take(c->px.cx_t.size()); L.px_c = cv.take(c->px.cx_c.size());
    L.passes = cv.take(c->plan.passes.size() * sizeof(DPass));
    L.groups = cv.take(c->plan.groups.size() * sizeof(DGroup));
    L.terms = cv.take(c->plan.terms.size() * sizeof(DTerm));
    L.wstat = cv.take(c->plan.wstat.size() / 2 * c->amp_bytes());
    L.gtabs = cv.take(c->plan.gtabs.size() * 4);
    L.rss = cv.take(c->plan.rss.size() * sizeof(DRs));
    L.dz = cv.take(c->H.diag_z.size() * 8);
    L.dc = cv.take(c->H.diag_c.size() * 8);
    L.readout = cv.take((size_t)(READOUT_BLOCKS + 1) * 16);
    L.smass = cv.take((((size_t)1 << c->n_store) >> SAMPLE_CHUNK_LOG2) * 8 + 16);   // n_store >= 10 > chunk bits - 3
    L.su = cv.take((size_t)SAMPLE_MAX_SHOTS * 8);
    L.sx = cv.take((size_t)SAMPLE_MAX_SHOTS * 8);
    L.table = cv.take(c->tab_bytes() << c->n_store);
    L.fixed_end = cv.off;
    const uint64_t tiles = 1ull << (c->n_store - c->plan.k);
    L.state_b = al256(c->amp_bytes() << c->n_store);
    L.cs_b = al256((size_t)(c->P > 0 ? c->P : 1) * c->amp_bytes());
    L.ry_b = c->jit_blocks.empty() ? 0 : al256((size_t)(c->P > 0 ? c->P : 1) * c->amp_bytes() * 2);   // {tan, scale, form, 0}
    L.params_b = al256((size_t)(c->P > 0 ? c->P : 1) * 8);
    L.partial_b = al256((size_t)tiles * c->plan.passes.size() * 8);
    L.per_state = L.state_b + L.cs_b + L.ry_b + L.params_b + L.partial_b + 256 /* E */;
    return L;
}

gvqe_status upload(gvqe_ctx *c, void *dst, const void *src, size_t bytes, cudaStream_t st)
{
    if (!bytes) return GVQE_OK;
    const cudaError_t e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st);
    return e == cudaSuccess ? GVQE_OK : cuda_fail(c, e, "upload");
}

// Carve the workspace, upload the compiled program and the Hamiltonian arrays, build the diagonal table.
gvqe_status ensure_ready(gvqe_ctx *c, cudaStream_t st)
{
    if (!c->have_h) return fail(c, GVQE_ERR_NO_HAMILTONIAN, "no Hamiltonian set");
    if (!c->ws) return fail(c, GVQE_ERR_WORKSPACE, "no workspace set");
    if (!c->dirty) return GVQE_OK;
    if (!c->kernels_ready) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaGetDevice");
        const int ke = kernels_init();
        if (ke) return cuda_fail(c, ke, "kernel attribute setup");
        c->kernels_ready = true;
    }
    // compile the specialised kernels (NVRTC, eight at a time: it is thread safe) and load them on this device
    auto load_all = [c](const std::vector<JitBlock> &blocks, std::vector<JitModule *> &mods, std::string &why) {
        bool ok = jit_runtime_available(why);
        if (!ok) return false;
        const size_t nbk = blocks.size();
        std::vector<std::string> errs(nbk);
        mods.assign(nbk, nullptr);
        for (size_t b0 = 0; b0 < nbk; b0 += 8) {
            std::vector<std::thread> th;
            for (size_t b = b0; b < nbk && b < b0 + 8; ++b)
                th.emplace_back([&blocks, &mods, b, &errs] { mods[b] = jit_load(blocks[b], errs[b]); });
            for (std::thread &t : th) t.join();
        }
        for (size_t b = 0; b < nbk; ++b) if (!mods[b]) { ok = false; why = errs[b]; }
        if (!ok) { for (JitModule *m : mods) jit_unload(m); mods.clear(); }
        return ok;
    };
    if (c->jit_state == 0) {
        std::string why;
        if (load_all(c->jit_blocks, c->jit_mods, why)) c->jit_state = 1;
        else {
            if (c->opt.specialise == 2) return fail(c, GVQE_ERR_UNSUPPORTED, "specialised kernels requested but unavailable: " + why);
            c->jit_state = -1; c->jit_blocks.clear();
        }
    }
    if (c->jitx_state == 0) {
        std::string why;
        if (load_all(c->jitx_blocks, c->jitx_mods, why)) c->jitx_state = 1;
        else {
            if (c->opt.specialise == 2) return fail(c, GVQE_ERR_UNSUPPORTED, "specialised kernels requested but unavailable: " + why);
            c->jitx_state = -1; c->jitx_blocks.clear(); c->jitx = JitExpectData();
        }
    }
    const Layout L = layout_of(c);
    if (c->ws_bytes < L.fixed_end + L.per_state) {
        char b[160];
        snprintf(b, sizeof b, "workspace too small: %zu bytes given, %zu needed for one statevector", c->ws_bytes,
                 L.fixed_end + L.per_state);
        return fail(c, GVQE_ERR_WORKSPACE, b);
    }
    size_t fit = (c->ws_bytes - L.fixed_end) / L.per_state;
    if (fit > 32768) fit = 32768;
    if (c->max_in_flight > 0 && fit > (size_t)c->max_in_flight) fit = (size_t)c->max_in_flight;
    c->in_flight = (int)fit;
    char *w = c->ws;
    const DevProgram &d = c->dev;
    c->gl.blocks = (const DBlock *)(w + L.blocks); c->gl.stages = (const DStage *)(w + L.stages);
    c->gl.ops = (const DOp *)(w + L.ops); c->gl.segs = (const DSeg *)(w + L.segs);
    c->gl.trzs = (const DTrz *)(w + L.trzs); c->gl.tczs = (const uint64_t *)(w + L.tczs);
    c->gl.csidx = (const int32_t *)(w + L.csidx);
    c->gl.ryl = (const int16_t *)(w + L.ryl); c->gl.cxs = (const DCx *)(w + L.cxs);
    c->gl.slut = (const uint32_t *)(w + L.slut);
    c->d_jwst = w + L.jwst; c->d_jpats = w + L.jpats; c->d_jterms = w + L.jterms;
    c->d_sweep_idx = (int32_t *)(w + L.sweep_idx); c->d_sweep_E = (double *)(w + L.sweep_E);
    c->pxd.rot_begin = (const int32_t *)(w + L.px_begin); c->pxd.rot_kind = (const uint8_t *)(w + L.px_kind);
    c->pxd.rot_param = (const int32_t *)(w + L.px_param); c->pxd.cx_t = (const uint8_t *)(w + L.px_t); c->pxd.cx_c = (const uint8_t *)(w + L.px_c);
    c->pxd.n_cx = (int)c->px.cx_t.size(); c->pxd.n_cz = c->px.n_cz; c->pxd.n = c->n_store; c->pxd.kk = std::min(c->n_store, c->prec == GVQE_C64 ? 15 : 14);   // amplitudes one thread block writes: its set-up (product tables) is paid once per 2^kk
    for (int i = 0; i < 4; ++i) { c->pxd.cz_d[i] = c->px.cz_d[i]; c->pxd.cz_m[i] = c->px.cz_m[i]; }
    {   // images of the offset bits inside a thread block under A^-1 (A = the prefix's CNOT run), as compact indices
        auto ainv = [&](uint64_t y) {
            for (int i = (int)c->px.cx_t.size() - 1; i >= 0; --i) y ^= ((y >> c->px.cx_c[i]) & 1ull) << c->px.cx_t[i];
            return y;
        };
        uint64_t img[16] = {0}, vary = 0;
        for (int b = 0; b < c->pxd.kk; ++b) { img[b] = ainv(1ull << b); vary |= img[b]; }
        c->pxd.vary = vary; c->pxd.n_vary = __builtin_popcountll(vary);
        memset(c->pxd.vq, 0, sizeof c->pxd.vq);
        int j = 0;
        for (int q = 0; q < 64; ++q) if ((vary >> q) & 1ull) c->pxd.vq[j++] = (uint8_t)q;
        for (int b = 0; b < 16; ++b) {
            uint64_t ci = 0;
            for (int t = 0; t < c->pxd.n_vary; ++t) ci |= ((img[b] >> c->pxd.vq[t]) & 1ull) << t;
            c->pxd.cimg[b] = ci;
        }
    }
    c->d_passes = (DPass *)(w + L.passes); c->d_groups = (DGroup *)(w + L.groups); c->d_terms = (DTerm *)(w + L.terms);
    c->d_wstat = w + L.wstat; c->d_gtabs = (uint32_t *)(w + L.gtabs); c->d_rss = (DRs *)(w + L.rss);
    c->d_diag_z = (uint64_t *)(w + L.dz); c->d_diag_c = (double *)(w + L.dc);
    c->d_table = w + L.table;
    c->d_readout = w + L.readout;
    char *p = w + L.fixed_end;
    c->d_states = p; p += L.state_b * fit;
    c->d_cs = p; p += L.cs_b * fit;
    c->d_ry = L.ry_b ? p : nullptr; p += L.ry_b * fit;
    c->d_params = (double *)p; p += L.params_b * fit;
    c->d_partial = (double *)p; p += L.partial_b * fit;
    c->d_E = (double *)p;
    c->slots_per_b = (uint32_t)((1ull << (c->n_store - c->plan.k)) * c->plan.passes.size());
    gvqe_status s;
#define UP(dst, vec) if ((s = upload(c, (void *)(dst), (vec).data(), (vec).size() * sizeof((vec)[0]), st)) != GVQE_OK) return s
    UP(c->gl.blocks, d.blocks); UP(c->gl.stages, d.stages); UP(c->gl.ops, d.ops); UP(c->gl.segs, d.segs);
    UP(c->gl.trzs, d.trzs); UP(c->gl.tczs, d.tczs); UP(c->gl.csidx, d.csidx); UP(c->gl.ryl, d.ryl); UP(c->gl.cxs, d.cxs); UP(c->gl.slut, d.slut);
    UP(c->pxd.rot_begin, c->px.rot_begin); UP(c->pxd.rot_kind, c->px.rot_kind); UP(c->pxd.rot_param, c->px.rot_param);
    UP(c->pxd.cx_t, c->px.cx_t); UP(c->pxd.cx_c, c->px.cx_c);
    UP(c->d_passes, c->plan.passes); UP(c->d_groups, c->plan.groups); UP(c->d_terms, c->plan.terms);
    if (c->prec == GVQE_C64) {
        c->wstat_f.assign(c->plan.wstat.begin(), c->plan.wstat.end());
        UP(c->d_wstat, c->wstat_f);
    } else UP(c->d_wstat, c->plan.wstat);
    UP(c->d_gtabs, c->plan.gtabs); UP(c->d_rss, c->plan.rss);
    if (c->jitx_state == 1) {
        if (c->prec == GVQE_C64) { c->jitx_wst_f.assign(c->jitx.wst.begin(), c->jitx.wst.end()); UP(c->d_jwst, c->jitx_wst_f); }
        else UP(c->d_jwst, c->jitx.wst);
        UP(c->d_jpats, c->jitx.pats); UP(c->d_jterms, c->jitx.terms);
    }
    UP(c->d_diag_z, c->H.diag_z); UP(c->d_diag_c, c->H.diag_c);
#undef UP
    // diagonal energy table: E(x) = sum_{Z-only k} c_k (-1)^{popcount(x & z_k)} = WHT of the scattered coefficients
    cudaError_t e = cudaMemsetAsync(c->d_table, 0, c->tab_bytes() << c->n_store, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "table memset");
    int ke = launch_table_scatter(c->prec, c->d_table, c->d_diag_z, c->d_diag_c, (uint32_t)c->H.diag_z.size(), st, &c->launches);
    if (ke) return cuda_fail(c, ke, "table scatter");
    if (!c->H.diag_z.empty())
        for (size_t i = 0; i < c->fwht_tiles.size(); ++i) {
            ke = launch_fwht_pass(c->prec, c->d_table, c->fwht_tiles[i], c->fwht_masks[i], c->n_store, st, &c->launches);
            if (ke) return cuda_fail(c, ke, "table transform");
        }
    c->dirty = false;
    return GVQE_OK;
}

// One chunk of `nb` statevectors: parameters are already on the device (nb x P doubles).
}  // namespace
extern "C" gvqe_status gvqe_profile_read(gvqe_ctx *c, double *out);
extern "C" int gvqe_profile_read_launches(gvqe_ctx *c, double *mean_ms, double *min_ms, double *max_ms, int cap);
namespace {
// Fused block j over nb statevectors starting at `states` (their (cos,sin) / tangent rows at cs / ry).
int gate_block(gvqe_ctx *c, size_t j, void *states, uint64_t stride, const void *cs, const void *ry, int nb, cudaStream_t st,
               const void *src = nullptr, uint64_t src_stride = 0)
{
    if (c->jit_state == 1) {
        ++c->launches;
        return jit_launch(c->jit_mods[j], c->jit_blocks[j], states, stride, ry, cs, nb, c->P, c->jit_per_cta, st, src, src_stride);
    }
    return launch_gate_block(c->prec, c->R, c->gl, c->dev.blocks[j], c->dev.blocks[j].k, c->dev.blocks[j].smem_prog_bytes, c->n_store,
                             states, stride, cs, c->P, nb, st, &c->launches);
}

// Expectation pass pi over nb statevectors starting at `states`; partial sums go to partial[b][slot_off + tile].
int expect_pass(gvqe_ctx *c, size_t pi, const void *states, uint64_t stride, double *partial, uint32_t slot_off, int nb, cudaStream_t st)
{
    if (c->jitx_state == 1) {
        ++c->launches;
        const char *wst = (const char *)c->d_jwst + (size_t)c->jitx.pass_wst_off[pi] * c->amp_bytes();
        const char *pats = (const char *)c->d_jpats + (size_t)c->jitx.pass_pat_off[pi] * sizeof(JitExpectData::Pat);
        return jit_launch_expect(c->jitx_mods[pi], c->jitx_blocks[pi], states, stride, c->d_table, wst, pats, c->d_jterms, partial,
                                 c->slots_per_b, slot_off, nb, c->jit_per_cta, st);
    }
    return launch_expect_pass(c->prec, c->d_passes, (int)pi, c->plan.k, c->n_store, c->d_groups, c->d_terms, c->d_wstat, c->d_gtabs,
                              c->d_rss, states, stride, c->d_table, partial, c->slots_per_b, slot_off, nb, st, &c->launches);
}

gvqe_status run_chunk(gvqe_ctx *c, const double *params_dev, int nb, double *E_dev, cudaStream_t st)
{
    const Layout L = layout_of(c);
    const uint64_t stride = L.state_b / c->amp_bytes();
    cudaEvent_t e4[4] = {nullptr, nullptr, nullptr, nullptr};
    if (c->profiling) {
        if (c->ev.size() >= 4096) {   // fold what has been recorded so far
            double tmp[8];
            gvqe_profile_read(c, tmp);
            gvqe_profile_read_launches(c, nullptr, nullptr, nullptr, 0);
        }
        for (int i = 0; i < 4; ++i) {
            if (cudaEventCreate(&e4[i]) != cudaSuccess) return cuda_fail(c, (int)cudaGetLastError(), "event create");
            c->ev.push_back(e4[i]);   // owned by the context from here on: freed by profile_read / destroy on every path
        }
    }
    int ke = launch_expand_params(c->prec, params_dev, c->d_cs, c->jit_state == 1 ? c->d_ry : nullptr, (uint64_t)nb * c->P, st, &c->launches);
    if (ke) return cuda_fail(c, ke, "expand_params");
    if (c->profiling) cudaEventRecord(e4[0], st);
    auto mark = [&]() {   // fine-grained profile: an event after every launch of the chunk
        if (!c->profiling) return;
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return;
        c->ev_fine.push_back(e);
        cudaEventRecord(e, st);
    };
    mark();
    if (c->px.n_ops > 0) {
        ke = launch_init_product(c->prec, c->pxd, c->d_states, stride, c->d_cs, c->P, nb, st, &c->launches);
        if (ke) return cuda_fail(c, ke, "product-state init");
        mark();
    }
    for (size_t bi = 0; bi < c->dev.blocks.size(); ++bi) {
        ke = gate_block(c, bi, c->d_states, stride, c->d_cs, c->d_ry, nb, st);
        if (ke) return cuda_fail(c, ke, "gate block");
        mark();
    }
    if (c->profiling) cudaEventRecord(e4[1], st);
    const uint32_t tiles = 1u << (c->n_store - c->plan.k);
    for (size_t pi = 0; pi < c->plan.passes.size(); ++pi) {
        ke = expect_pass(c, pi, c->d_states, stride, c->d_partial, (uint32_t)pi * tiles, nb, st);
        if (ke) return cuda_fail(c, ke, "expectation pass");
        mark();
    }
    if (c->profiling) cudaEventRecord(e4[2], st);
    ke = launch_reduce(c->d_partial, c->slots_per_b, E_dev, nb, st, &c->launches);
    if (ke) return cuda_fail(c, ke, "reduce");
    if (c->profiling) {
        cudaEventRecord(e4[3], st);
        const double S = (double)(c->amp_bytes() << c->n_store);
        double gb = 0;
        for (const DBlock &b : c->dev.blocks) gb += (b.source_zero ? 1.0 : 2.0) * S * nb;
        if (c->px.n_ops > 0) gb += S * nb;   // write-only product-state kernel
        c->prof_acc[1] += (double)c->dev.blocks.size() + (c->px.n_ops > 0 ? 1.0 : 0.0); c->prof_acc[2] += gb;
        c->prof_acc[4] += (double)c->plan.passes.size();
        c->prof_acc[5] += (double)c->plan.passes.size() * S * nb + (double)(c->tab_bytes() << c->n_store);
        c->prof_acc[7] += 1.0;
    }
    return GVQE_OK;
}

}  // namespace

extern "C" {

size_t gvqe_workspace_bytes(const gvqe_ctx *c, int batch)
{
    if (!c || !c->have_h || batch < 1) return 0;
    const Layout L = layout_of(c);
    return L.fixed_end + L.per_state * (size_t)batch + 256;
}

gvqe_status gvqe_set_workspace(gvqe_ctx *c, void *ptr, size_t bytes)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (!ptr || ((uintptr_t)ptr & 255)) return fail(c, GVQE_ERR_INVALID_ARG, "workspace must be a 256-byte aligned device pointer");
    if (c->have_h) {
        const Layout L = layout_of(c);
        if (bytes < L.fixed_end + L.per_state) return fail(c, GVQE_ERR_WORKSPACE, "workspace too small for one statevector");
    } else if (bytes < (c->amp_bytes() << c->n_store)) return fail(c, GVQE_ERR_WORKSPACE, "workspace too small for one statevector");
    c->ws = (char *)ptr; c->ws_bytes = bytes; c->dirty = true;
    return GVQE_OK;
}

gvqe_status gvqe_set_max_in_flight(gvqe_ctx *c, int m)
{
    if (!c || m < 0) return GVQE_ERR_INVALID_ARG;
    c->max_in_flight = m; c->dirty = true;
    return GVQE_OK;
}

gvqe_status gvqe_energy_batch_device(gvqe_ctx *c, const double *params_dev, int B, double *E_dev, void *stream)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (B < 0 || (B > 0 && (!E_dev || (!params_dev && c->P > 0)))) return fail(c, GVQE_ERR_INVALID_ARG, "energy_batch_device: bad arguments");
    cudaStream_t st = (cudaStream_t)stream;
    gvqe_status s = ensure_ready(c, st);
    if (s != GVQE_OK) return s;
    for (int b0 = 0; b0 < B; b0 += c->in_flight) {
        const int nb = (B - b0 < c->in_flight) ? (B - b0) : c->in_flight;
        if ((s = run_chunk(c, params_dev + (size_t)b0 * c->P, nb, E_dev + b0, st)) != GVQE_OK) return s;
    }
    return GVQE_OK;
}

gvqe_status gvqe_energy_batch(gvqe_ctx *c, const double *params, int B, double *E, void *stream)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (B < 0 || (B > 0 && (!E || (!params && c->P > 0)))) return fail(c, GVQE_ERR_INVALID_ARG, "energy_batch: bad arguments");
    for (size_t i = 0; i < (size_t)B * c->P; ++i)
        if (!std::isfinite(params[i])) return fail(c, GVQE_ERR_INVALID_ARG, "energy_batch: parameter is not finite");
    cudaStream_t st = (cudaStream_t)stream;
    gvqe_status s = ensure_ready(c, st);
    if (s != GVQE_OK) return s;
    for (int b0 = 0; b0 < B; b0 += c->in_flight) {
        const int nb = (B - b0 < c->in_flight) ? (B - b0) : c->in_flight;
        cudaError_t e = cudaSuccess;
        if (c->P > 0) e = cudaMemcpyAsync(c->d_params, params + (size_t)b0 * c->P, (size_t)nb * c->P * 8, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "params H2D");
        if ((s = run_chunk(c, c->d_params, nb, c->d_E, st)) != GVQE_OK) return s;
        e = cudaMemcpyAsync(E + b0, c->d_E, (size_t)nb * 8, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "E D2H");
        // d_params / d_E are reused by the next chunk: stream order makes that safe for pinned and pageable hosts
    }
    const cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, e, "stream synchronize");
    return GVQE_OK;
}

// Shared-prefix evaluation of a parameter-shift set.  A shifted row differs from theta in one
// parameter, so up to the fused block in which that parameter is first read its state IS the state of theta.  The base
// state advances block by block in slot 0; before block j runs on it, the rows whose parameter enters at block j copy
// it into the other slots and run blocks j.. and the expectation passes there.  Every row still sees the same kernels
// on the same data as in gvqe_energy_batch, so the energies are bit-identical to the unshared evaluation.
// Returns GVQE_ERR_UNSUPPORTED when the scheme does not apply (one slot, schedule bookkeeping missing): caller falls back.
static gvqe_status grad_shared_prefix(gvqe_ctx *c, const double *params, const std::vector<int> &idx, double *E_pm /* 2 per idx */,
                                      double *E0, cudaStream_t st)
{
    gvqe_status s = ensure_ready(c, st);
    if (s != GVQE_OK) return s;
    const int P = c->P, F = c->in_flight, NB = (int)c->dev.blocks.size();
    if (F < 2 || NB == 0 || c->prog.block_ops.size() != (size_t)NB) return GVQE_ERR_UNSUPPORTED;
    // first launch that reads each parameter: -1 = the product-state kernel, j = fused block j, -2 = no gate
    std::vector<int> first((size_t)P, -2);
    for (int32_t q : c->px.rot_param) if (q >= 0 && q < P) first[q] = -1;
    for (int j = 0; j < NB; ++j)
        for (int oi : c->prog.block_ops[j]) {
            const size_t gi = (size_t)oi + (size_t)c->px.n_ops;
            if (gi >= c->ops.size()) return GVQE_ERR_UNSUPPORTED;
            const int q = c->ops[gi].param;
            if (q >= 0 && first[q] == -2) first[q] = j;
        }
    std::vector<std::vector<int>> group((size_t)NB + 1);   // [0] = product-state kernel, [j + 1] = block j; entries index idx
    for (size_t a = 0; a < idx.size(); ++a) {
        const int f = first[idx[a]];
        if (f == -2) { E_pm[2 * a] = E_pm[2 * a + 1] = 0.0; continue; }   // the energy does not depend on it
        group[(size_t)(f + 1)].push_back((int)a);
    }
    const Layout L = layout_of(c);
    const uint64_t stride = L.state_b / c->amp_bytes();
    const size_t S_bytes = c->amp_bytes() << c->n_store;
    const uint32_t tiles = 1u << (c->n_store - c->plan.k);
    const double half_pi = 1.57079632679489661923;
    auto state_of = [&](int slot) { return (void *)((char *)c->d_states + L.state_b * (size_t)slot); };
    auto cs_of = [&](int slot) { return (void *)((char *)c->d_cs + (size_t)slot * (size_t)P * c->amp_bytes()); };
    auto ry_of = [&](int slot) { return c->d_ry ? (void *)((char *)c->d_ry + (size_t)slot * (size_t)P * c->amp_bytes() * 2) : nullptr; };
    const bool use_ry = c->jit_state == 1;
    auto blocks_from = [&](int j0, int slot, int nb) -> gvqe_status {
        for (int j = j0; j < NB; ++j) {
            const int ke = gate_block(c, (size_t)j, state_of(slot), stride, cs_of(slot), ry_of(slot), nb, st);
            if (ke) return cuda_fail(c, ke, "gate block");
        }
        return GVQE_OK;
    };
    auto expect = [&](int slot, int nb, double *E_dev) -> gvqe_status {
        double *partial = c->d_partial + (size_t)slot * c->slots_per_b;
        for (size_t pi = 0; pi < c->plan.passes.size(); ++pi) {
            const int ke = expect_pass(c, pi, state_of(slot), stride, partial, (uint32_t)pi * tiles, nb, st);
            if (ke) return cuda_fail(c, ke, "expectation pass");
        }
        const int ke = launch_reduce(partial, c->slots_per_b, E_dev, nb, st, &c->launches);
        return ke ? cuda_fail(c, ke, "reduce") : GVQE_OK;
    };
    // work items in processing order: boundary after boundary, per parameter the + and the - row
    std::vector<std::pair<int, int>> work;              // (entry of idx, 0 = plus / 1 = minus)
    std::vector<size_t> group_begin((size_t)NB + 2, 0);
    for (int g = 0; g <= NB; ++g) {
        group_begin[(size_t)g] = work.size();
        for (int a : group[(size_t)g]) { work.push_back({a, 0}); work.push_back({a, 1}); }
    }
    group_begin[(size_t)NB + 1] = work.size();
    // With the specialised kernels the whole sweep is enqueued without a host round trip: the shift codes go up once, the
    // rows are formed on the device, the first block of a suffix READS the base state and writes the row's own buffer
    // (no copy), the energies stay on the device until the end.  The generic kernels keep the chunk-by-chunk form.
    const bool staged = use_ry && work.size() <= SWEEP_MAX_ROWS;
    std::vector<int32_t> codes;
    std::vector<double> Eall(work.size() + 1);
    cudaError_t e = cudaMemcpyAsync(c->d_params, params, (size_t)P * 8, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "params H2D");
    if (staged && !work.empty()) {
        codes.resize(work.size());
        for (size_t i = 0; i < work.size(); ++i) codes[i] = (int32_t)(idx[(size_t)work[i].first] * 2 + work[i].second);
        e = cudaMemcpyAsync(c->d_sweep_idx, codes.data(), codes.size() * 4, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "sweep codes H2D");
    }
    int ke = launch_expand_params(c->prec, c->d_params, c->d_cs, use_ry ? c->d_ry : nullptr, (uint64_t)P, st, &c->launches);
    if (ke) return cuda_fail(c, ke, "expand_params");
    if (c->px.n_ops > 0 && (ke = launch_init_product(c->prec, c->pxd, c->d_states, stride, c->d_cs, P, 1, st, &c->launches)))
        return cuda_fail(c, ke, "product-state init");
    std::vector<double> rows((size_t)(F - 1) * P);
    for (int g = 0; g <= NB; ++g) {
        const int j0 = g - 1;   // -1: from the product-state kernel
        for (size_t w0 = group_begin[(size_t)g]; w0 < group_begin[(size_t)g + 1]; w0 += (size_t)(F - 1)) {
            const int nb = (int)std::min(group_begin[(size_t)g + 1] - w0, (size_t)(F - 1));
            if (staged) {
                if ((ke = launch_shift_rows(c->d_params, c->d_sweep_idx + w0, c->d_params + P, P, nb, st, &c->launches)))
                    return cuda_fail(c, ke, "shift rows");
            } else {
                for (int r = 0; r < nb; ++r) {
                    for (int q = 0; q < P; ++q) rows[(size_t)r * P + q] = params[q];
                    rows[(size_t)r * P + idx[(size_t)work[w0 + r].first]] += work[w0 + r].second ? -half_pi : half_pi;
                }
                e = cudaMemcpyAsync(c->d_params + P, rows.data(), (size_t)nb * P * 8, cudaMemcpyHostToDevice, st);
                if (e != cudaSuccess) return cuda_fail(c, e, "params H2D");
            }
            if ((ke = launch_expand_params(c->prec, c->d_params + P, cs_of(1), use_ry ? ry_of(1) : nullptr, (uint64_t)nb * P, st, &c->launches)))
                return cuda_fail(c, ke, "expand_params");
            int j_first = j0 < 0 ? 0 : j0;
            if (j0 < 0) {
                if ((ke = launch_init_product(c->prec, c->pxd, state_of(1), stride, cs_of(1), P, nb, st, &c->launches)))
                    return cuda_fail(c, ke, "product-state init");
            } else if (!(j0 == 0 && c->dev.blocks[0].source_zero)) {
                if (use_ry) {   // block j0 out of place: reads the base state, writes the rows' buffers
                    if ((ke = gate_block(c, (size_t)j0, state_of(1), stride, cs_of(1), ry_of(1), nb, st, state_of(0), 0)))
                        return cuda_fail(c, ke, "gate block");
                    j_first = j0 + 1;
                } else {
                    for (int r = 0; r < nb; ++r) {
                        e = cudaMemcpyAsync(state_of(1 + r), state_of(0), S_bytes, cudaMemcpyDeviceToDevice, st);
                        if (e != cudaSuccess) return cuda_fail(c, e, "state copy");
                    }
                }
            }
            if ((s = blocks_from(j_first, 1, nb)) != GVQE_OK) return s;
            if (staged) {
                if ((s = expect(1, nb, c->d_sweep_E + w0)) != GVQE_OK) return s;
            } else {
                if ((s = expect(1, nb, c->d_E + 1)) != GVQE_OK) return s;
                e = cudaMemcpyAsync(Eall.data() + w0, c->d_E + 1, (size_t)nb * 8, cudaMemcpyDeviceToHost, st);
                if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // rows / d_E are reused by the next chunk
                if (e != cudaSuccess) return cuda_fail(c, e, "E D2H");
            }
        }
        if (j0 >= 0) {   // the base state advances by block j0
            ke = gate_block(c, (size_t)j0, state_of(0), stride, cs_of(0), ry_of(0), 1, st);
            if (ke) return cuda_fail(c, ke, "gate block");
        }
    }
    if (staged) {
        if ((s = expect(0, 1, c->d_sweep_E + work.size())) != GVQE_OK) return s;
        e = cudaMemcpyAsync(Eall.data(), c->d_sweep_E, (work.size() + 1) * 8, cudaMemcpyDeviceToHost, st);
    } else {
        if ((s = expect(0, 1, c->d_E)) != GVQE_OK) return s;
        e = cudaMemcpyAsync(Eall.data() + work.size(), c->d_E, 8, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, e, "E D2H");
    for (size_t i = 0; i < work.size(); ++i) E_pm[2 * (size_t)work[i].first + (size_t)work[i].second] = Eall[i];
    *E0 = Eall[work.size()];
    return GVQE_OK;
}

gvqe_status gvqe_param_shift_grad(gvqe_ctx *c, const double *params, const uint8_t *mask, double *dE, double *E0, void *stream)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (c->P > 0 && (!params || !mask || !dE)) return fail(c, GVQE_ERR_INVALID_ARG, "param_shift_grad: null input");
    std::vector<int> idx;
    for (int p = 0; p < c->P; ++p) if (mask[p]) idx.push_back(p);
    for (int p = 0; p < c->P; ++p)
        if (!std::isfinite(params[p])) return fail(c, GVQE_ERR_INVALID_ARG, "param_shift_grad: parameter is not finite");
    // shared prefixes pay when kernel time dominates launch overhead: states of >= 16 MiB unless forced (1) or disabled (0)
    const int sp = c->opt.shared_prefix;   // 0 auto, 1 never, 2 always
    if (!idx.empty() && (sp == 2 || (sp == 0 && (c->amp_bytes() << c->n_store) >= ((size_t)16 << 20)))) {
        std::vector<double> Epm(2 * idx.size());
        double e0 = 0.0;
        const gvqe_status s = grad_shared_prefix(c, params, idx, Epm.data(), &e0, (cudaStream_t)stream);
        if (s == GVQE_OK) {
            for (int p = 0; p < c->P; ++p) dE[p] = 0.0;
            for (size_t j = 0; j < idx.size(); ++j) dE[idx[j]] = 0.5 * (Epm[2 * j] - Epm[2 * j + 1]);   // Eq. 13
            if (E0) *E0 = e0;
            return GVQE_OK;
        }
        if (s != GVQE_ERR_UNSUPPORTED) return s;
    }
    const int B = 2 * (int)idx.size() + 1;
    // Eq. 13: rows theta, theta +/- (pi/2) e_p for the masked p, ascending (reading A8)
    std::vector<double> rows((size_t)B * c->P), E((size_t)B);
    for (int b = 0; b < B; ++b) for (int p = 0; p < c->P; ++p) rows[(size_t)b * c->P + p] = params[p];
    const double half_pi = 1.57079632679489661923;
    for (size_t j = 0; j < idx.size(); ++j) {
        rows[(2 * j + 1) * c->P + idx[j]] += half_pi;
        rows[(2 * j + 2) * c->P + idx[j]] -= half_pi;
    }
    const gvqe_status s = gvqe_energy_batch(c, rows.data(), B, E.data(), stream);
    if (s != GVQE_OK) return s;
    for (int p = 0; p < c->P; ++p) dE[p] = 0.0;
    for (size_t j = 0; j < idx.size(); ++j) dE[idx[j]] = 0.5 * (E[2 * j + 1] - E[2 * j + 2]);
    if (E0) *E0 = E[0];
    return GVQE_OK;
}

gvqe_status gvqe_get_state(gvqe_ctx *c, int slot, void *host_out)
{
    if (!c || !host_out) return GVQE_ERR_INVALID_ARG;
    if (c->dirty || !c->ws) return fail(c, GVQE_ERR_WORKSPACE, "get_state: no energy call has run on this workspace");
    if (slot < 0 || slot >= c->in_flight) return fail(c, GVQE_ERR_INVALID_ARG, "get_state: slot out of range");
    const Layout L = layout_of(c);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess)
        e = cudaMemcpy(host_out, (char *)c->d_states + L.state_b * (size_t)slot, c->amp_bytes() << c->n_user, cudaMemcpyDeviceToHost);
    return e == cudaSuccess ? GVQE_OK : cuda_fail(c, e, "get_state");
}

gvqe_status gvqe_argmax(gvqe_ctx *c, int slot, uint64_t *x, double *prob, void *stream)
{
    if (!c || !x) return GVQE_ERR_INVALID_ARG;
    if (c->dirty || !c->ws) return fail(c, GVQE_ERR_WORKSPACE, "argmax: no energy call has run on this workspace");
    if (slot < 0 || slot >= c->in_flight) return fail(c, GVQE_ERR_INVALID_ARG, "argmax: slot out of range");
    const Layout L = layout_of(c);
    cudaStream_t st = (cudaStream_t)stream;
    // idle padding qubits stay |0>: the user's amplitudes are the first 2^n_user of the stored state
    const int ke = launch_argmax(c->prec, (char *)c->d_states + L.state_b * (size_t)slot, 1ull << c->n_user, c->d_readout, st,
                                 &c->launches);
    if (ke) return cuda_fail(c, ke, "argmax launch");
    struct { double p; uint64_t x; } r;
    cudaError_t e = cudaMemcpyAsync(&r, c->d_readout, sizeof r, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, e, "argmax D2H");
    *x = r.x;
    if (prob) *prob = r.p;
    return GVQE_OK;
}

gvqe_status gvqe_argmax_noalloc(const void *state, uint64_t n_amplitudes, gvqe_precision prec, void *result, void *stream,
                                char *err, size_t err_cap)
{
    static_assert(GVQE_NOALLOC_MAX_AMPLITUDES == NOALLOC_MAX_AMPLITUDES && GVQE_NOALLOC_SCRATCH_BYTES == NOALLOC_SCRATCH_BYTES,
                  "gvqe.h and kernels.h disagree");
    auto say = [&](gvqe_status s, const char *msg) {
        if (err && err_cap) snprintf(err, err_cap, "%s", msg);
        return s;
    };
    if (err && err_cap) err[0] = 0;
    if (prec != GVQE_C64 && prec != GVQE_C128) return say(GVQE_ERR_INVALID_ARG, "argmax_noalloc: precision is neither GVQE_C64 nor GVQE_C128");
    if (!state || !result) return say(GVQE_ERR_INVALID_ARG, "argmax_noalloc: state and result must be device pointers, not NULL");
    if (n_amplitudes == 0) return say(GVQE_ERR_INVALID_ARG, "argmax_noalloc: n_amplitudes is 0");
    if (n_amplitudes > GVQE_NOALLOC_MAX_AMPLITUDES) {
        char b[160];
        snprintf(b, sizeof b, "argmax_noalloc: %llu amplitudes exceed the maximum of 2^34 = %llu this entry point takes",
                 (unsigned long long)n_amplitudes, (unsigned long long)GVQE_NOALLOC_MAX_AMPLITUDES);
        return say(GVQE_ERR_INVALID_ARG, b);
    }
    if (((uintptr_t)state & 15u) || ((uintptr_t)result & 7u)) return say(GVQE_ERR_INVALID_ARG, "argmax_noalloc: state must be 16-byte and result 8-byte aligned");
    const int ke = launch_argmax_noalloc(prec == GVQE_C64 ? 0 : 1, state, n_amplitudes, result, stream);
    if (ke) {
        char b[200];
        snprintf(b, sizeof b, "argmax_noalloc: CUDA error %d (%s)", ke, cudaGetErrorString((cudaError_t)ke));
        return say(GVQE_ERR_CUDA, b);
    }
    return GVQE_OK;
}

gvqe_status gvqe_sample(gvqe_ctx *c, int slot, int n_shots, const double *u, uint64_t *x, double *norm, void *stream)
{
    if (!c || n_shots < 0 || (n_shots > 0 && (!u || !x))) return GVQE_ERR_INVALID_ARG;
    if ((uint32_t)n_shots > SAMPLE_MAX_SHOTS) return fail(c, GVQE_ERR_INVALID_ARG, "sample: more than 65536 shots in one call");
    if (c->dirty || !c->ws) return fail(c, GVQE_ERR_WORKSPACE, "sample: no energy call has run on this workspace");
    if (slot < 0 || slot >= c->in_flight) return fail(c, GVQE_ERR_INVALID_ARG, "sample: slot out of range");
    for (int s = 0; s < n_shots; ++s)
        if (!(u[s] >= 0.0 && u[s] < 1.0)) return fail(c, GVQE_ERR_INVALID_ARG, "sample: uniforms must lie in [0, 1)");
    const Layout L = layout_of(c);
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t count = 1ull << c->n_user;
    const uint64_t n_chunks = (count + (1u << SAMPLE_CHUNK_LOG2) - 1) >> SAMPLE_CHUNK_LOG2;
    double *mass = (double *)(c->ws + L.smass), *total = mass + n_chunks;
    double *u_dev = (double *)(c->ws + L.su);
    uint64_t *x_dev = (uint64_t *)(c->ws + L.sx);
    cudaError_t e = cudaSuccess;
    if (n_shots) e = cudaMemcpyAsync(u_dev, u, (size_t)n_shots * 8, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "sample H2D");
    const int ke = launch_sample(c->prec, (char *)c->d_states + L.state_b * (size_t)slot, count, mass, total, u_dev, x_dev,
                                 (uint32_t)n_shots, st, &c->launches);
    if (ke) return cuda_fail(c, ke, "sample launch");
    if (n_shots) e = cudaMemcpyAsync(x, x_dev, (size_t)n_shots * 8, cudaMemcpyDeviceToHost, st);
    double z = 0.0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&z, total, 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, e, "sample D2H");
    if (norm) *norm = z;
    return GVQE_OK;
}

// measurement settings: distinct (x_mask, y_mask) in ascending order; returns the setting of every term
static void settings_of(const gvqe_ctx *c, std::vector<std::pair<uint64_t, uint64_t>> &settings, std::vector<int32_t> &of_term)
{
    settings.clear();
    for (const HostTerm &t : c->H.terms) settings.push_back({t.x, t.x & t.z});
    std::sort(settings.begin(), settings.end());
    settings.erase(std::unique(settings.begin(), settings.end()), settings.end());
    of_term.resize(c->H.terms.size());
    for (size_t k = 0; k < c->H.terms.size(); ++k) {
        const std::pair<uint64_t, uint64_t> key(c->H.terms[k].x, c->H.terms[k].x & c->H.terms[k].z);
        of_term[k] = (int32_t)(std::lower_bound(settings.begin(), settings.end(), key) - settings.begin());
    }
}

gvqe_status gvqe_measurement_settings(const gvqe_ctx *c, int32_t *n_settings, int32_t *setting_of_term)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (!c->have_h) return GVQE_ERR_NO_HAMILTONIAN;
    std::vector<std::pair<uint64_t, uint64_t>> settings;
    std::vector<int32_t> of_term;
    settings_of(c, settings, of_term);
    if (n_settings) *n_settings = (int32_t)settings.size();
    if (setting_of_term) for (size_t k = 0; k < of_term.size(); ++k) setting_of_term[k] = of_term[k];
    return GVQE_OK;
}

gvqe_status gvqe_energy_shots(gvqe_ctx *c, int slot, int n_shots, const double *u, double *E_est, double *term_means, void *stream)
{
    if (!c || !E_est || n_shots < 1 || !u) return GVQE_ERR_INVALID_ARG;
    if ((uint32_t)n_shots > SAMPLE_MAX_SHOTS) return fail(c, GVQE_ERR_INVALID_ARG, "energy_shots: more than 65536 shots per setting");
    if (c->dirty || !c->ws) return fail(c, GVQE_ERR_WORKSPACE, "energy_shots: no energy call has run on this workspace");
    if (slot < 0 || slot >= c->in_flight) return fail(c, GVQE_ERR_INVALID_ARG, "energy_shots: slot out of range");
    if (c->in_flight < 2) return fail(c, GVQE_ERR_WORKSPACE, "energy_shots: needs a second statevector in flight as scratch");
    std::vector<std::pair<uint64_t, uint64_t>> settings;
    std::vector<int32_t> of_term;
    settings_of(c, settings, of_term);
    const size_t NS = settings.size(), M = c->H.terms.size();
    for (size_t i = 0; i < NS * (size_t)n_shots; ++i)
        if (!(u[i] >= 0.0 && u[i] < 1.0)) return fail(c, GVQE_ERR_INVALID_ARG, "energy_shots: uniforms must lie in [0, 1)");
    const Layout L = layout_of(c);
    cudaStream_t st = (cudaStream_t)stream;
    const int scratch = (slot + 1) % c->in_flight;
    char *src = (char *)c->d_states + L.state_b * (size_t)slot, *dst = (char *)c->d_states + L.state_b * (size_t)scratch;
    const uint64_t count = 1ull << c->n_user;    // idle padding qubits stay |0>: the user's amplitudes are the first 2^n_user
    const uint64_t n_chunks = (count + (1u << SAMPLE_CHUNK_LOG2) - 1) >> SAMPLE_CHUNK_LOG2;
    double *mass = (double *)(c->ws + L.smass), *total = mass + n_chunks;
    double *u_dev = (double *)(c->ws + L.su);
    uint64_t *x_dev = (uint64_t *)(c->ws + L.sx);
    std::vector<uint64_t> shots((size_t)n_shots);
    std::vector<double> sum(M, 0.0);
    for (size_t g = 0; g < NS; ++g) {
        const uint64_t xm = settings[g].first, ym = settings[g].second;
        const void *cur = src;
        for (int q = 0; q < c->n_user; ++q) {   // the first rotation doubles as the copy into the scratch slot
            if (!((xm >> q) & 1ull)) continue;
            const int ke = launch_basis_rotate(c->prec, cur, dst, c->n_user, q, (int)((ym >> q) & 1ull), st, &c->launches);
            if (ke) return cuda_fail(c, ke, "basis rotation");
            cur = dst;
        }
        cudaError_t e = cudaMemcpyAsync(u_dev, u + g * (size_t)n_shots, (size_t)n_shots * 8, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "energy_shots H2D");
        const int ke = launch_sample(c->prec, cur, count, mass, total, u_dev, x_dev, (uint32_t)n_shots, st, &c->launches);
        if (ke) return cuda_fail(c, ke, "sample launch");
        e = cudaMemcpyAsync(shots.data(), x_dev, (size_t)n_shots * 8, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(c, e, "energy_shots D2H");
        for (size_t k = 0; k < M; ++k) {
            if ((size_t)of_term[k] != g) continue;
            const uint64_t supp = c->H.terms[k].x | c->H.terms[k].z;
            long plus = 0;
            for (int s2 = 0; s2 < n_shots; ++s2) plus += (__builtin_popcountll(shots[(size_t)s2] & supp) & 1) ? -1 : 1;
            sum[k] = (double)plus / (double)n_shots;
        }
    }
    double E = 0.0;
    for (size_t k = 0; k < M; ++k) E += c->H.terms[k].c * sum[k];
    *E_est = E;
    if (term_means) for (size_t k = 0; k < M; ++k) term_means[k] = sum[k];
    return GVQE_OK;
}

gvqe_status gvqe_schedule_info(const gvqe_ctx *c, int32_t *nb, int32_t *np, int32_t *inflight)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (nb) *nb = (int32_t)c->dev.blocks.size() + (c->px.n_ops > 0 ? 1 : 0);   // + the write-only product-state kernel
    if (np) *np = c->have_h ? (int32_t)c->plan.passes.size() : 0;
    if (inflight) *inflight = c->in_flight;
    return GVQE_OK;
}

size_t gvqe_dump_schedule(const gvqe_ctx *c, char *buf, size_t cap)
{
    if (!c) return 0;
    std::string s = dump_program(c->prog);
    {
        char pl[160];
        snprintf(pl, sizeof pl, "prefix ops=%d rotations=%zu cnots=%zu cz_distances=%d\n", c->px.n_ops, c->px.rot_kind.size(), c->px.cx_t.size(), c->px.n_cz);
        s += pl;
    }
    char line[256];
    snprintf(line, sizeof line, "device blocks=%zu max_prog_smem=%u\n", c->dev.blocks.size(), c->dev.max_smem_prog);
    s += line;
    if (c->have_h) {
        for (size_t p = 0; p < c->plan.passes.size(); ++p) {
            const DPass &dp = c->plan.passes[p];
            snprintf(line, sizeof line, "pass %zu k=%d diag=%d groups=%u runs=", p, dp.k, dp.with_diag, dp.group_end - dp.group_begin);
            s += line;
            for (int r = 0; r < dp.n_runs; ++r) { snprintf(line, sizeof line, "%d:%d+%d ", dp.runs[r].lpos, dp.runs[r].gpos, dp.runs[r].len); s += line; }
            s += "\n";
            int nd = 0, nrs = 0, hist[16] = {0}; size_t nt_d = 0, nt_t = 0, nt_rs = 0;
            for (uint32_t gi = dp.group_begin; gi < dp.group_end; ++gi) {
                const DGroup &dg = c->plan.groups[gi];
                if (dg.rs) { ++nrs; nt_rs += dg.term_end - dg.term_begin; }
                else if (dg.direct) { ++nd; nt_d += dg.term_end - dg.term_begin; }
                else { ++hist[dg.ubits & 15]; nt_t += dg.term_end - dg.term_begin; }
            }
            snprintf(line, sizeof line, "grp  register-stage=%d (terms %zu) direct=%d (terms %zu) lookup terms=%zu ubits hist:", nrs, nt_rs, nd, nt_d, nt_t); s += line;
            for (int u = 0; u < 16; ++u) if (hist[u]) { snprintf(line, sizeof line, " %d:%d", u, hist[u]); s += line; }
            s += "\n";
        }
    }
    if (buf && cap) { const size_t m = s.size() < cap - 1 ? s.size() : cap - 1; memcpy(buf, s.data(), m); buf[m] = 0; }
    return s.size() + 1;
}

int gvqe_get_exec_order(const gvqe_ctx *c, int32_t *order, int cap)
{
    if (!c) return -1;
    const int m = (int)c->prog.exec_order.size();
    if (order) for (int i = 0; i < m && i < cap; ++i) order[i] = c->prog.exec_order[i];
    return m;
}

gvqe_status gvqe_profile_enable(gvqe_ctx *c, int on)
{
    if (!c) return GVQE_ERR_INVALID_ARG;
    if (on) {
        for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
        c->ev.clear();
        for (cudaEvent_t e : c->ev_fine) cudaEventDestroy(e);
        c->ev_fine.clear(); c->prof_launch_ms.clear(); c->prof_fine_chunks = 0;
        for (double &v : c->prof_acc) v = 0.0;
    }
    c->profiling = on != 0;
    return GVQE_OK;
}

// folds the fine-grained events (1 + launches per chunk) into per-launch sums
static void fold_fine(gvqe_ctx *c)
{
    const size_t per = 1 + (c->px.n_ops > 0 ? 1 : 0) + c->dev.blocks.size() + c->plan.passes.size();
    if (c->prof_launch_ms.size() != per - 1) {
        c->prof_launch_ms.assign(per - 1, 0.0); c->prof_launch_min.assign(per - 1, 1e300); c->prof_launch_max.assign(per - 1, 0.0);
        c->prof_fine_chunks = 0;
    }
    for (size_t i = 0; i + per <= c->ev_fine.size(); i += per) {
        if (cudaEventSynchronize(c->ev_fine[i + per - 1]) != cudaSuccess) break;
        for (size_t j = 0; j + 1 < per; ++j) {
            float ms = 0;
            cudaEventElapsedTime(&ms, c->ev_fine[i + j], c->ev_fine[i + j + 1]);
            c->prof_launch_ms[j] += ms;
            if (ms < c->prof_launch_min[j]) c->prof_launch_min[j] = ms;
            if (ms > c->prof_launch_max[j]) c->prof_launch_max[j] = ms;
        }
        c->prof_fine_chunks += 1;
    }
    for (cudaEvent_t e : c->ev_fine) cudaEventDestroy(e);
    c->ev_fine.clear();
}

int gvqe_profile_read_launches(gvqe_ctx *c, double *mean_ms, double *min_ms, double *max_ms, int cap)
{
    if (!c) return -1;
    fold_fine(c);
    const int m = (int)c->prof_launch_ms.size();
    for (int i = 0; i < m && i < cap; ++i) {
        if (mean_ms) mean_ms[i] = c->prof_fine_chunks > 0 ? c->prof_launch_ms[(size_t)i] / c->prof_fine_chunks : 0.0;
        if (min_ms) min_ms[i] = c->prof_fine_chunks > 0 ? c->prof_launch_min[(size_t)i] : 0.0;
        if (max_ms) max_ms[i] = c->prof_launch_max[(size_t)i];
    }
    return m;
}

gvqe_status gvqe_profile_read(gvqe_ctx *c, double *out)
{
    if (!c || !out) return GVQE_ERR_INVALID_ARG;
    for (size_t i = 0; i + 3 < c->ev.size(); i += 4) {
        cudaError_t e = cudaEventSynchronize(c->ev[i + 3]);
        if (e != cudaSuccess) return cuda_fail(c, e, "profile event");
        float g = 0, x = 0, r = 0;
        cudaEventElapsedTime(&g, c->ev[i], c->ev[i + 1]);
        cudaEventElapsedTime(&x, c->ev[i + 1], c->ev[i + 2]);
        cudaEventElapsedTime(&r, c->ev[i + 2], c->ev[i + 3]);
        c->prof_acc[0] += g; c->prof_acc[3] += x; c->prof_acc[6] += r;
    }
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    for (int i = 0; i < 8; ++i) out[i] = c->prof_acc[i];
    return GVQE_OK;
}

uint64_t gvqe_launch_count(const gvqe_ctx *c) { return c ? c->launches : 0; }
// ---- host-side Graph-VQE driver: graph construction and partitioning (graph.cpp), parameter masks ----------------
gvqe_status gvqe_interaction_graph(const gvqe_ctx *c, double *w)
{
    if (!c || !w) return GVQE_ERR_INVALID_ARG;
    if (!c->have_h) return GVQE_ERR_NO_HAMILTONIAN;
    const int n = c->n_user;
    for (size_t t = 0; t < (size_t)n * n; ++t) w[t] = 0.0;
    for (const HostTerm &t : c->H.terms) {   // Eq. 9: non-identity on qubit i <=> bit i of x | z
        const uint64_t s = t.x | t.z;
        const double a = std::fabs(t.c);
        for (int i = 0; i < n; ++i) {
            if (!((s >> i) & 1)) continue;
            for (int j = i + 1; j < n; ++j)
                if ((s >> j) & 1) { w[(size_t)i * n + j] += a; w[(size_t)j * n + i] += a; }
        }
    }
    return GVQE_OK;
}

static bool graph_args_ok(int n, const double *w)
{
    if (n < 1 || !w) return false;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            const double v = w[(size_t)i * n + j];
            if (!(v >= 0.0) || !std::isfinite(v) || v != w[(size_t)j * n + i]) return false;
        }
    return true;
}

gvqe_status gvqe_modularity(int n, const double *w, const int32_t *community, double gamma, double *Q)
{
    if (!graph_args_ok(n, w) || !community || !Q || !std::isfinite(gamma)) return GVQE_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) if (community[i] < 0) return GVQE_ERR_INVALID_ARG;
    *Q = modularity(n, w, community, gamma);
    return GVQE_OK;
}

gvqe_status gvqe_louvain(int n, const double *w, double gamma, int32_t *community, int32_t *n_communities, double *Q)
{
    if (!graph_args_ok(n, w) || !community || !std::isfinite(gamma) || gamma < 0.0) return GVQE_ERR_INVALID_ARG;
    const int K = louvain(n, w, gamma, community);
    if (n_communities) *n_communities = K;
    if (Q) *Q = modularity(n, w, community, gamma);
    return GVQE_OK;
}

gvqe_status gvqe_merge_small_blocks(int n, const double *w, int s_min, int32_t *community, int32_t *n_communities)
{
    if (!graph_args_ok(n, w) || !community) return GVQE_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) if (community[i] < 0 || community[i] > (1 << 20)) return GVQE_ERR_INVALID_ARG;
    const int K = merge_small_blocks(n, w, s_min, community);
    if (n_communities) *n_communities = K;
    return GVQE_OK;
}

gvqe_status gvqe_geometric_blocks(int n, int block_size, int offset, int32_t *community, int32_t *n_communities)
{
    if (n < 1 || block_size < 1 || offset < 0 || offset >= block_size || !community) return GVQE_ERR_INVALID_ARG;
    for (int q = 0; q < n; ++q) community[q] = q < offset ? 0 : (q - offset) / block_size + (offset > 0 ? 1 : 0);
    if (n_communities) *n_communities = community[n - 1] + 1;
    return GVQE_OK;
}

gvqe_status gvqe_block_param_mask(const gvqe_ctx *c, const int32_t *community, int32_t block, uint8_t *mask)
{
    if (!c || !community || (c->P > 0 && !mask)) return GVQE_ERR_INVALID_ARG;
    for (int p = 0; p < c->P; ++p) mask[p] = 0;
    for (const HostOp &o : c->ops)
        if ((o.kind == GVQE_OP_RY || o.kind == GVQE_OP_RZ) && o.param >= 0 && o.q0 < c->n_user && community[o.q0] == block)
            mask[o.param] = 1;
    return GVQE_OK;
}

const char *gvqe_last_error(const gvqe_ctx *c) { return c ? c->err.c_str() : "null context"; }
void gvqe_destroy(gvqe_ctx *c)
{
    if (!c) return;
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_fine) cudaEventDestroy(e);
    for (JitModule *m : c->jit_mods) jit_unload(m);
    for (JitModule *m : c->jitx_mods) jit_unload(m);
    delete c;
}

}  // extern "C"

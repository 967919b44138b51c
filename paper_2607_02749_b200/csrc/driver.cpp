// driver.cpp -- host-side Graph-VQE optimisation loop (north_star item 3) written against the
// public C ABI only: every energy and gradient comes from gvqe_energy_batch / gvqe_param_shift_grad, i.e. from the
// sm_100a kernels.  PAPER.md:207-212 (Eq. 11: block-restricted objective), 214 (global refinement from the fused
// block solution), 221-225 (Eq. 13, L-BFGS with f_tol, g_tol = 0.1 f_tol), 229-235 (four steps per epoch, Eq. 14
// window criterion, epoch patience, warm start from theta*_best).
#include <algorithm>
#include <cmath>
#include <deque>
#include <vector>

#include "../../include/gvqe.h"

namespace {

struct Run {
    gvqe_ctx *ctx;
    const gvqe_opt_options *opt;
    void *stream;
    int P;
    long evals = 0;
    int steps = 0;
};

// Eq. 14: Delta_max = max over the last W differences |E_t - E_{t-1}|.
double delta_max(const std::vector<double> &E, int W)
{
    double d = 0.0;
    const int nE = (int)E.size();
    for (int t = std::max(1, nE - W); t < nE; ++t) d = std::max(d, std::fabs(E[t] - E[t - 1]));
    return d;
}

// L-BFGS on the coordinates with mask != 0, all others frozen (Eq. 11).  theta is updated in place; *E_out = E(theta).
gvqe_status minimize_masked(Run &r, std::vector<double> &theta, const std::vector<uint8_t> &mask, int max_iters,
                            double *E_out)
{
    const int P = r.P;
    const double f_tol = r.opt->f_tol, g_tol = 0.1 * r.opt->f_tol;
    std::vector<int> idx;
    for (int p = 0; p < P; ++p) if (mask[p]) idx.push_back(p);
    const int na = (int)idx.size();
    std::vector<double> gfull((size_t)std::max(P, 1)), g((size_t)na), gn((size_t)na), d((size_t)na);
    double E = 0.0;
    gvqe_status st = gvqe_param_shift_grad(r.ctx, theta.data(), mask.data(), gfull.data(), &E, r.stream);
    if (st != GVQE_OK) return st;
    r.evals += 2 * na + 1;
    for (int a = 0; a < na; ++a) g[a] = gfull[idx[a]];
    std::vector<double> hist{E};
    std::deque<std::vector<double>> S, Y;
    std::deque<double> RHO;
    int calm = 0;
    constexpr int NTRY = 4;
    std::vector<double> rows((size_t)NTRY * std::max(P, 1)), Et(NTRY);
    for (int it = 0; it < max_iters && na > 0; ++it) {
        double ginf = 0.0;
        for (double v : g) ginf = std::max(ginf, std::fabs(v));
        if (ginf < g_tol) break;
        // two-loop recursion: d = -H g
        d = g;
        std::vector<double> al(S.size());
        for (int i = (int)S.size() - 1; i >= 0; --i) {
            double sd = 0.0;
            for (int a = 0; a < na; ++a) sd += S[i][a] * d[a];
            al[i] = RHO[i] * sd;
            for (int a = 0; a < na; ++a) d[a] -= al[i] * Y[i][a];
        }
        if (!S.empty()) {
            double sy = 0.0, yy = 0.0;
            for (int a = 0; a < na; ++a) { sy += S.back()[a] * Y.back()[a]; yy += Y.back()[a] * Y.back()[a]; }
            const double sc = sy / yy;
            for (double &v : d) v *= sc;
        }
        for (size_t i = 0; i < S.size(); ++i) {
            double yd = 0.0;
            for (int a = 0; a < na; ++a) yd += Y[i][a] * d[a];
            const double be = RHO[i] * yd;
            for (int a = 0; a < na; ++a) d[a] += (al[i] - be) * S[i][a];
        }
        double dg = 0.0;
        for (int a = 0; a < na; ++a) { d[a] = -d[a]; dg += d[a] * g[a]; }
        if (!(dg < 0.0)) {   // not a descent direction: restart from steepest descent
            S.clear(); Y.clear(); RHO.clear();
            dg = 0.0;
            for (int a = 0; a < na; ++a) { d[a] = -g[a]; dg += d[a] * g[a]; }
        }
        // backtracking line search, NTRY step lengths per batched energy call (Armijo, c1 = 1e-4)
        double a0 = S.empty() ? std::min(1.0, 1.0 / ginf) : 1.0, alpha = 0.0, En = E;
        bool ok = false;
        for (int round = 0; round < 3 && !ok; ++round) {
            for (int t = 0; t < NTRY; ++t) {
                const double at = a0 * std::ldexp(1.0, -t);
                for (int p = 0; p < P; ++p) rows[(size_t)t * P + p] = theta[p];
                for (int a = 0; a < na; ++a) rows[(size_t)t * P + idx[a]] += at * d[a];
            }
            st = gvqe_energy_batch(r.ctx, rows.data(), NTRY, Et.data(), r.stream);
            if (st != GVQE_OK) return st;
            r.evals += NTRY;
            for (int t = 0; t < NTRY && !ok; ++t) {
                const double at = a0 * std::ldexp(1.0, -t);
                if (Et[t] <= E + 1e-4 * at * dg) { ok = true; alpha = at; En = Et[t]; }
            }
            a0 *= std::ldexp(1.0, -NTRY);
        }
        if (!ok) break;   // no decrease along a descent direction down to 2^-11: converged to rounding
        std::vector<double> s((size_t)na), y((size_t)na);
        for (int a = 0; a < na; ++a) { s[a] = alpha * d[a]; theta[idx[a]] += s[a]; }
        double Echk = 0.0;
        st = gvqe_param_shift_grad(r.ctx, theta.data(), mask.data(), gfull.data(), &Echk, r.stream);
        if (st != GVQE_OK) return st;
        r.evals += 2 * na + 1;
        ++r.steps;
        double sy = 0.0;
        for (int a = 0; a < na; ++a) { gn[a] = gfull[idx[a]]; y[a] = gn[a] - g[a]; sy += s[a] * y[a]; }
        if (sy > 1e-12) {
            S.push_back(s); Y.push_back(y); RHO.push_back(1.0 / sy);
            if ((int)S.size() > std::max(1, r.opt->lbfgs_memory)) { S.pop_front(); Y.pop_front(); RHO.pop_front(); }
        }
        const double Eprev = E;
        g = gn;
        E = En;
        hist.push_back(E);
        // L-BFGS-B style relative decrease test (f_tol), then the window criterion of Eq. 14
        if ((Eprev - E) <= f_tol * std::max({std::fabs(Eprev), std::fabs(E), 1.0})) break;
        calm = delta_max(hist, r.opt->window) < r.opt->tol ? calm + 1 : 0;
        if (calm >= r.opt->patience) break;
    }
    *E_out = E;
    return GVQE_OK;
}

}  // namespace

extern "C" gvqe_status gvqe_graph_vqe_minimize(gvqe_ctx *ctx, const gvqe_opt_options *opt, const int32_t *community,
                                               double *params, gvqe_opt_result *result, double *history,
                                               int32_t history_cap, int32_t *history_len, void *stream)
{
    if (!ctx || !opt || !community || !result) return GVQE_ERR_INVALID_ARG;
    const int P = gvqe_num_params(ctx), n = gvqe_num_qubits(ctx);
    if (P > 0 && !params) return GVQE_ERR_INVALID_ARG;
    if (opt->max_epochs < 1 || opt->block_iters < 0 || opt->global_iters < 0 || opt->window < 1 || opt->patience < 1 ||
        opt->epoch_patience < 1 || !(opt->tol > 0.0) || !(opt->f_tol >= 0.0))
        return GVQE_ERR_INVALID_ARG;
    int K = 0;
    for (int q = 0; q < n; ++q) {
        if (community[q] < 0 || community[q] >= n) return GVQE_ERR_INVALID_ARG;
        K = std::max(K, community[q] + 1);
    }
    Run r{ctx, opt, stream, P};
    std::vector<double> best(params, params + P), theta, fused;
    double E_best = 0.0;
    gvqe_status st = gvqe_energy_batch(ctx, best.data(), 1, &E_best, stream);
    if (st != GVQE_OK) return st;
    r.evals += 1;
    int hl = 0;
    if (history && hl < history_cap) history[hl++] = E_best;
    std::vector<std::vector<uint8_t>> masks((size_t)K, std::vector<uint8_t>((size_t)std::max(P, 1), 0));
    for (int b = 0; b < K; ++b) {
        st = gvqe_block_param_mask(ctx, community, b, masks[b].data());
        if (st != GVQE_OK) return st;
    }
    const std::vector<uint8_t> all((size_t)std::max(P, 1), 1);
    int stale = 0, epochs = 0, reason = 0;
    for (int ep = 0; ep < opt->max_epochs; ++ep) {
        ++epochs;
        fused = best;   // warm start from theta*_best
        for (int b = 0; b < K; ++b) {   // every block starts from the same vector; its own coordinates are fused
            theta = best;
            double Eb = 0.0;
            st = minimize_masked(r, theta, masks[b], opt->block_iters, &Eb);
            if (st != GVQE_OK) return st;
            for (int p = 0; p < P; ++p) if (masks[b][p]) fused[p] = theta[p];
        }
        double E = 0.0;
        if (opt->global_iters > 0) st = minimize_masked(r, fused, all, opt->global_iters, &E);
        else { st = gvqe_energy_batch(ctx, fused.data(), 1, &E, stream); r.evals += 1; }
        if (st != GVQE_OK) return st;
        if (history && hl < history_cap) history[hl++] = E;
        if (E < E_best - opt->tol) { stale = 0; } else { ++stale; }
        if (E < E_best) { E_best = E; best = fused; }
        if (stale >= opt->epoch_patience) { reason = 1; break; }
    }
    for (int p = 0; p < P; ++p) params[p] = best[p];
    result->E_best = E_best;
    result->epochs = epochs;
    result->n_blocks = K;
    result->steps = r.steps;
    result->energy_evals = (int64_t)r.evals;
    result->stop_reason = reason;
    if (history_len) *history_len = hl;
    return GVQE_OK;
}

// cobyla.cpp -- derivative-free minimiser for the Graph-VQE loop: "Graph-VQE supports both derivative-free (COBYLA) and
// gradient-based (L-BFGS-B) optimization", "the loop uses either COBYLA or L-BFGS-B on the full parameter
// vector".  The paper calls SciPy's routine and gives no steps; this is the unconstrained case of
// Powell's linear-approximation method (M.J.D. Powell, "A direct search optimization method that models the objective
// and constraint functions by linear interpolation", 1994) restated from its description (reading G8):
//   * a simplex of n + 1 points; the linear function that interpolates f on its vertices gives a gradient g;
//   * trust-region step from the best vertex x0: x0 - rho g / |g|; the new point replaces a vertex;
//   * the simplex is "acceptable" when every vertex is at most beta rho from x0 and at least alpha rho from the face
//     opposite to it (alpha = 1/4, beta = 2.1); otherwise one vertex is moved to x0 +- gamma rho v (gamma = 1/2, v the
//     unit normal of its opposite face, the sign the model prefers);
//   * when a step gains less than a tenth of what the model predicts on an acceptable simplex, rho is halved (set to
//     rho_end once within 1.5 rho_end); the run ends when rho_end is reached and rho would shrink again.
// What makes it fit the GPU: the n + 1 energies of the initial simplex (and of a rebuilt one) are ONE batch of rows.
// Host code only; energies come from a callback (gvqe_energy_batch in driver.cpp, any function in the test hook).
#include "cobyla.h"

#include <algorithm>
#include <cmath>

namespace gv {

namespace {

// Z = S^-1 by Gauss-Jordan with partial pivoting (row-major n x n); false when S is singular to rounding.
bool invert(std::vector<double> &S, std::vector<double> &Z, int n)
{
    Z.assign((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) Z[(size_t)i * n + i] = 1.0;
    double scale = 0.0;
    for (double v : S) scale = std::max(scale, std::fabs(v));
    if (!(scale > 0.0)) return false;
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r) if (std::fabs(S[(size_t)r * n + c]) > std::fabs(S[(size_t)piv * n + c])) piv = r;
        if (std::fabs(S[(size_t)piv * n + c]) < 1e-13 * scale) return false;
        if (piv != c)
            for (int k = 0; k < n; ++k) { std::swap(S[(size_t)piv * n + k], S[(size_t)c * n + k]); std::swap(Z[(size_t)piv * n + k], Z[(size_t)c * n + k]); }
        const double inv = 1.0 / S[(size_t)c * n + c];
        for (int k = 0; k < n; ++k) { S[(size_t)c * n + k] *= inv; Z[(size_t)c * n + k] *= inv; }
        for (int r = 0; r < n; ++r) {
            if (r == c) continue;
            const double m = S[(size_t)r * n + c];
            if (m == 0.0) continue;
            for (int k = 0; k < n; ++k) { S[(size_t)r * n + k] -= m * S[(size_t)c * n + k]; Z[(size_t)r * n + k] -= m * Z[(size_t)c * n + k]; }
        }
    }
    return true;
}

}  // namespace

int cobyla_minimize(int n, double *x, double rho_beg, double rho_end, int max_evals, const CobylaFn &f, CobylaTrace *tr)
{
    CobylaTrace local;
    CobylaTrace &T = tr ? *tr : local;
    T = CobylaTrace();
    if (n < 0 || !(rho_beg > 0.0) || !(rho_end > 0.0) || rho_end > rho_beg) return -1;
    std::vector<double> fx(1);
    if (n == 0) {
        if (!f(x, 1, fx.data())) return -2;
        T.evals = 1; T.f_best = fx[0]; T.history.push_back(fx[0]);
        return 0;
    }
    constexpr double ALPHA = 0.25, BETA = 2.1, GAMMA = 0.5;
    const int m = n + 1;
    std::vector<double> X((size_t)m * n), F((size_t)m), S((size_t)n * n), Z, g((size_t)n), xn((size_t)n), sig((size_t)n), eta((size_t)n);
    double rho = rho_beg;
    // simplex x0, x0 + rho e_j around row 0 of X (which must hold the centre); one batch of n + 1 (or n) rows
    auto build = [&](bool with_centre) -> bool {
        for (int j = 1; j < m; ++j) {
            for (int i = 0; i < n; ++i) X[(size_t)j * n + i] = X[i];
            X[(size_t)j * n + (j - 1)] += rho;
        }
        const int first = with_centre ? 0 : 1;
        if (!f(X.data() + (size_t)first * n, m - first, F.data() + first)) return false;
        T.evals += m - first;
        return true;
    };
    for (int i = 0; i < n; ++i) X[i] = x[i];
    if (!build(true)) return -2;
    bool after_geometry = false;
    int status = 1;   // 1 = evaluation budget, 0 = rho_end reached, 2 = stopped by the caller's monitor
    auto best_to_front = [&]() {
        int jb = 0;
        for (int j = 1; j < m; ++j) if (F[j] < F[jb]) jb = j;
        if (jb != 0) {
            std::swap(F[0], F[jb]);
            for (int i = 0; i < n; ++i) std::swap(X[i], X[(size_t)jb * n + i]);
        }
    };
    best_to_front();
    T.history.push_back(F[0]);
    while (true) {
        best_to_front();
        if (T.evals >= max_evals) { status = 1; break; }
        for (int j = 1; j < m; ++j)
            for (int i = 0; i < n; ++i) S[(size_t)(j - 1) * n + i] = X[(size_t)j * n + i] - X[i];
        for (int j = 0; j < n; ++j) {
            double e = 0.0;
            for (int i = 0; i < n; ++i) e += S[(size_t)j * n + i] * S[(size_t)j * n + i];
            eta[j] = std::sqrt(e);
        }
        if (!invert(S, Z, n)) {   // degenerate simplex: a fresh one of the current size around the best point
            if (!build(false)) return -2;
            ++T.rebuilds;
            after_geometry = false;
            continue;
        }
        // model gradient: S g = F[1..] - F[0]  =>  g = Z (F[1..] - F[0]);  sigma_j = 1 / |column j of Z|
        for (int i = 0; i < n; ++i) {
            double s = 0.0;
            for (int j = 0; j < n; ++j) s += Z[(size_t)i * n + j] * (F[j + 1] - F[0]);
            g[i] = s;
        }
        int j_far = -1, j_flat = -1;
        for (int j = 0; j < n; ++j) {
            double c = 0.0;
            for (int i = 0; i < n; ++i) c += Z[(size_t)i * n + j] * Z[(size_t)i * n + j];
            sig[j] = 1.0 / std::sqrt(c);
            if (eta[j] > BETA * rho && (j_far < 0 || eta[j] > eta[j_far])) j_far = j;
            if (sig[j] < ALPHA * rho && (j_flat < 0 || sig[j] < sig[j_flat])) j_flat = j;
        }
        const bool acceptable = j_far < 0 && j_flat < 0;
        if (!acceptable && !after_geometry) {
            // geometry step: the farthest vertex (else the flattest) moves to x0 +- gamma rho v; a trust-region step
            // always follows it, so the two kinds of step alternate at worst
            const int j = j_far >= 0 ? j_far : j_flat;
            double gv = 0.0;
            for (int i = 0; i < n; ++i) gv += g[i] * Z[(size_t)i * n + j];
            const double sgn = gv > 0.0 ? -1.0 : 1.0;
            for (int i = 0; i < n; ++i) xn[i] = X[i] + sgn * GAMMA * rho * sig[j] * Z[(size_t)i * n + j];
            double fn = 0.0;
            if (!f(xn.data(), 1, &fn)) return -2;
            ++T.evals; ++T.geometry_steps;
            for (int i = 0; i < n; ++i) X[(size_t)(j + 1) * n + i] = xn[i];
            F[j + 1] = fn;
            after_geometry = true;
            T.history.push_back(std::min(F[0], fn));
            if (T.monitor && T.monitor(T.history)) { status = 2; break; }
            continue;
        }
        after_geometry = false;
        double gn = 0.0;
        for (int i = 0; i < n; ++i) gn += g[i] * g[i];
        gn = std::sqrt(gn);
        auto shrink = [&]() -> bool {   // false: rho_end was already reached
            if (rho <= rho_end) return false;
            rho *= 0.5;
            if (rho <= 1.5 * rho_end) rho = rho_end;
            ++T.rho_reductions;
            return true;
        };
        if (!(gn > 0.0)) {   // flat model: nothing to gain at this radius
            if (!shrink()) { status = 0; break; }
            continue;
        }
        // trust-region step
        for (int i = 0; i < n; ++i) xn[i] = X[i] - rho * g[i] / gn;
        double fn = 0.0;
        if (!f(xn.data(), 1, &fn)) return -2;
        ++T.evals; ++T.trust_steps;
        const double pred = rho * gn, act = F[0] - fn;
        // Which vertex leaves.  d = sum_j c_j s_j (c = Z^T d): putting the new point in place of vertex j multiplies the
        // simplex volume by |c_j| and the distance of that vertex from its opposite face becomes |c_j| sigma_j.  First
        // choice: the largest |c_j| (a point that is no improvement must not shrink the simplex: |c_j| > 1).  Preferred:
        // among the vertices whose replacement keeps that distance acceptable (or does not reduce it), the one farthest
        // from the best point (the new point when it improves) if it is farther than 1.1 rho.
        int jl = -1;
        double ratio = act > 0.0 ? 0.0 : 1.0, edge = 1.1 * rho;
        int jfar = -1;
        for (int j = 0; j < n; ++j) {
            double c = 0.0;
            for (int i = 0; i < n; ++i) c += (xn[i] - X[i]) * Z[(size_t)i * n + j];
            c = std::fabs(c);
            if (c > ratio) { ratio = c; jl = j; }
            const double sbar = c * sig[j];
            if (sbar >= ALPHA * rho || sbar >= sig[j]) {
                double e = eta[j];
                if (act > 0.0) {
                    e = 0.0;
                    for (int i = 0; i < n; ++i) { const double dlt = X[(size_t)(j + 1) * n + i] - xn[i]; e += dlt * dlt; }
                    e = std::sqrt(e);
                }
                if (e > edge) { edge = e; jfar = j; }
            }
        }
        if (jfar >= 0) jl = jfar;
        if (act > 0.0) ++T.improvements;
        if (jl >= 0) {
            for (int i = 0; i < n; ++i) X[(size_t)(jl + 1) * n + i] = xn[i];
            F[jl + 1] = fn;
        }
        // a step that gains less than a tenth of the prediction on a simplex that was acceptable: the linear model is as
        // good as this radius allows (on an unacceptable simplex the next iteration repairs the geometry instead)
        if (!(act > 0.0 && act >= 0.1 * pred) && acceptable && !shrink()) {
            T.history.push_back(std::min(F[0], fn));
            status = 0;
            break;
        }
        T.history.push_back(std::min(F[0], fn));
        if (T.monitor && T.monitor(T.history)) { status = 2; break; }
    }
    best_to_front();
    for (int i = 0; i < n; ++i) x[i] = X[i];
    T.f_best = F[0];
    T.rho_final = rho;
    return status;
}

}  // namespace gv

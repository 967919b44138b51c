// cobyla.h -- derivative-free minimiser of the Graph-VQE loop (reading G8).  Host only.
#pragma once
#include <functional>
#include <vector>

namespace gv {

// f(rows, B, out): B points of n coordinates each (row-major) -> out[B]; false aborts the run.
typedef std::function<bool(const double *rows, int B, double *out)> CobylaFn;

struct CobylaTrace {
    int evals = 0, trust_steps = 0, geometry_steps = 0, rho_reductions = 0, rebuilds = 0, improvements = 0;
    double f_best = 0.0, rho_final = 0.0;
    std::vector<double> history;                                  // best value after every evaluation past the first simplex
    std::function<bool(const std::vector<double> &)> monitor;     // optional early stop (Eq. 14 window): true = stop
};

// Minimises f from x (n coordinates, updated in place to the best vertex).  rho_beg >= rho_end > 0: first and last
// trust-region radius; max_evals bounds the evaluations.  Returns 0 = rho_end reached, 1 = evaluation budget,
// 2 = stopped by the monitor, -1 = bad arguments, -2 = f failed.
int cobyla_minimize(int n, double *x, double rho_beg, double rho_end, int max_evals, const CobylaFn &f, CobylaTrace *trace);

}  // namespace gv

"""CPU oracle of the Graph-VQE epoch loop -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

The loop is an iteration, so this follows it step by step in the paper's order with the readings
G4-G6 of DESIGN.md: per epoch, warm start from theta*_best; every block minimises the restricted objective (Eq. 11)
from that same vector with L-BFGS on parameter-shift gradients (Eq. 13); the block solutions are fused; a global
refinement over all parameters follows; best-so-far and the epoch patience are updated.  Energies come from a
callable `energy(rows[B,P]) -> E[B]` (the tests pass the complex128 oracle T0), so nothing here touches the library.
Pins: tests/test_graph_pins.py::test_driver_oracle_* (search direction against the dense BFGS inverse-Hessian update and
conjugacy / finite termination on a convex quadratic, separable cosine closed form, Eq. 14 window by hand).
"""
from __future__ import annotations

import math

import numpy as np


def param_shift_grad(energy, theta, idx):
    """Eq. 13 on the coordinates idx; returns (E(theta), g[len(idx)])."""
    rows = np.tile(np.asarray(theta, dtype=np.float64), (2 * len(idx) + 1, 1))
    for j, p in enumerate(idx):
        rows[2 * j + 1, p] += math.pi / 2
        rows[2 * j + 2, p] -= math.pi / 2
    E = np.asarray(energy(rows), dtype=np.float64)
    return float(E[0]), np.array([0.5 * (E[2 * j + 1] - E[2 * j + 2]) for j in range(len(idx))])


def delta_max(hist, W):
    """Eq. 14: the largest |E_t - E_{t-1}| over the last W differences."""
    lo = max(1, len(hist) - W)
    return max((abs(hist[t] - hist[t - 1]) for t in range(lo, len(hist))), default=0.0)


def lbfgs_direction(g, S, Y):
    """Search direction d = -H g of L-BFGS from the stored pairs (s_i, y_i), oldest first, by the two-loop recursion with
    the initial matrix H0 = (s.y / y.y) I of the newest pair (H0 = I without pairs).  Pinned in tests/test_graph_pins.py
    against the explicit dense BFGS inverse-Hessian update (reading G5: the optimiser details are the build's own;
    PAPER.md:214, 225 only name SciPy's L-BFGS-B)."""
    q = np.array(g, dtype=np.float64)
    al = [0.0] * len(S)
    for i in reversed(range(len(S))):
        al[i] = float(S[i] @ q) / float(S[i] @ Y[i])
        q = q - al[i] * Y[i]
    if S:
        q = q * (float(S[-1] @ Y[-1]) / float(Y[-1] @ Y[-1]))
    for i in range(len(S)):
        be = float(Y[i] @ q) / float(S[i] @ Y[i])
        q = q + (al[i] - be) * S[i]
    return -q


def minimize_masked(energy, theta, mask, max_iters, *, tol, f_tol, window, patience, memory):
    """L-BFGS (two-loop recursion) on the masked coordinates, Armijo backtracking (c1 = 1e-4) over step lengths
    a0 * 2^-t tried four at a time; a0 = min(1, 1/|g|_inf) without curvature pairs, else 1.  Returns (theta, E, steps)."""
    theta = np.array(theta, dtype=np.float64)
    idx = [p for p in range(len(theta)) if mask[p]]
    E, g = param_shift_grad(energy, theta, idx)
    hist, S, Y, steps, calm = [E], [], [], 0, 0
    for _ in range(max_iters if idx else 0):
        ginf = float(np.max(np.abs(g)))
        if ginf < 0.1 * f_tol:
            break
        d = lbfgs_direction(g, S, Y)
        dg = float(d @ g)
        if not dg < 0.0:
            S, Y = [], []
            d = -g
            dg = float(d @ g)
        a0 = 1.0 if S else min(1.0, 1.0 / ginf)
        found = None
        for _round in range(3):
            steps_try = [a0 * 2.0 ** -t for t in range(4)]
            rows = np.tile(theta, (4, 1))
            for t, a in enumerate(steps_try):
                rows[t, idx] += a * d
            Et = np.asarray(energy(rows), dtype=np.float64)
            for t, a in enumerate(steps_try):
                if Et[t] <= E + 1e-4 * a * dg:
                    found = (a, float(Et[t]))
                    break
            if found:
                break
            a0 *= 2.0 ** -4
        if not found:
            break
        a, En = found
        s = a * d
        theta[idx] += s
        _, gn = param_shift_grad(energy, theta, idx)
        steps += 1
        y = gn - g
        if float(s @ y) > 1e-12:
            S.append(s)
            Y.append(y)
            if len(S) > max(1, memory):
                S.pop(0)
                Y.pop(0)
        Eprev, E, g = E, En, gn
        hist.append(E)
        if Eprev - E <= f_tol * max(abs(Eprev), abs(E), 1.0):
            break
        calm = calm + 1 if delta_max(hist, window) < tol else 0
        if calm >= patience:
            break
    return theta, E, steps


def graph_vqe_minimize(energy, theta0, masks, *, max_epochs=10, block_iters=50, global_iters=50, window=40,
                       patience=12, epoch_patience=3, lbfgs_memory=8, tol=1e-4, f_tol=1e-9):
    """masks: one 0/1 vector per block.  Returns (theta_best, E_best, history, epochs, steps, stop_reason)."""
    kw = dict(tol=tol, f_tol=f_tol, window=window, patience=patience, memory=lbfgs_memory)
    best = np.array(theta0, dtype=np.float64)
    E_best = float(np.asarray(energy(best.reshape(1, -1)))[0])
    history, stale, steps, reason, epochs = [E_best], 0, 0, 0, 0
    for _ep in range(max_epochs):
        epochs += 1
        fused = best.copy()
        for m in masks:
            th, _, st = minimize_masked(energy, best, m, block_iters, **kw)
            steps += st
            sel = np.asarray(m, dtype=bool)
            fused[sel] = th[sel]
        if global_iters > 0:
            fused, E, st = minimize_masked(energy, fused, np.ones(len(best), np.uint8), global_iters, **kw)
            steps += st
        else:
            E = float(np.asarray(energy(fused.reshape(1, -1)))[0])
        history.append(E)
        stale = 0 if E < E_best - tol else stale + 1
        if E < E_best:
            E_best, best = E, fused.copy()
        if stale >= epoch_patience:
            reason = 1
            break
    return best, E_best, np.array(history), epochs, steps, reason

"""The derivative-free minimiser of the Graph-VQE loop ("either COBYLA or L-BFGS-B"; DESIGN.md reading
G8), exercised on host functions through gvqe_cobyla_minimize -- no GPU.  The paper calls SciPy's COBYLA, so SciPy's routine
is the oracle here (a library routine as the definition); since the two implementations take different steps, what is
compared is what is unique: the minimum they reach.  Closed forms pin both."""
import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from scipy.optimize import minimize


def _batch(f):
    return lambda rows: np.array([f(r) for r in rows])


def test_convex_quadratic_closed_form_and_scipy():
    rng = np.random.default_rng(3)
    n = 6
    A = rng.normal(size=(n, n))
    Q = A @ A.T + n * np.eye(n)
    b = rng.normal(size=n)
    f = lambda x: float(0.5 * x @ Q @ x - b @ x)
    xs = np.linalg.solve(Q, b)                       # closed form: x* = Q^-1 b, f* = -b.x*/2
    x, fb, cnt, reason = gv.cobyla_minimize(_batch(f), np.zeros(n), 1.0, 1e-5, 5000)
    assert reason == 0                               # rho_end reached
    assert abs(fb - f(x)) < 1e-12
    assert fb - (-0.5 * b @ xs) < 1e-8 and np.linalg.norm(x - xs) < 1e-3
    r = minimize(f, np.zeros(n), method="COBYLA", options=dict(rhobeg=1.0, tol=1e-5, maxiter=5000))
    assert abs(fb - r.fun) < 1e-7


def test_separable_cosine_closed_form_and_scipy():
    """E(theta) = sum a_q cos(theta_q): the energy of H = sum a_q Z_q under one RY layer; minimum -sum |a_q|."""
    rng = np.random.default_rng(5)
    a = rng.normal(size=10)
    f = lambda x: float(np.sum(a * np.cos(x)))
    x0 = rng.uniform(-1, 1, 10)
    x, fb, cnt, reason = gv.cobyla_minimize(_batch(f), x0, 1.0, 1e-4, 5000)
    assert reason == 0
    assert fb + np.sum(np.abs(a)) < 1e-6
    assert np.all(np.abs(np.cos(x) + np.sign(a)) < 1e-5)
    r = minimize(f, x0, method="COBYLA", options=dict(rhobeg=1.0, tol=1e-4, maxiter=5000))
    assert abs(fb - r.fun) < 1e-6


def test_first_simplex_is_one_batch_and_budget_is_respected():
    calls = []

    def fun(rows):
        calls.append(len(rows))
        return np.sum((rows - 0.3) ** 2, axis=1)

    x, fb, cnt, reason = gv.cobyla_minimize(fun, np.full(7, 2.0), 0.5, 1e-3, 40)
    assert calls[0] == 8 and all(c == 1 for c in calls[1:])         # n + 1 rows at once, then one point per step
    assert sum(calls) == cnt["evals"] == 40 and reason == 1          # stopped by the budget
    assert fb <= 7 * 1.7 ** 2                                        # never worse than the start
    assert cnt["trust_steps"] + cnt["geometry_steps"] + 8 == cnt["evals"]


def test_edge_cases():
    x, fb, cnt, reason = gv.cobyla_minimize(lambda rows: np.full(len(rows), 4.5), np.zeros(0), 1.0, 1e-4, 10)
    assert fb == 4.5 and cnt["evals"] == 1                           # nothing to optimise
    x, fb, cnt, reason = gv.cobyla_minimize(lambda rows: (rows[:, 0] - 0.3) ** 2, np.array([2.0]), 1.0, 1e-5, 500)
    assert reason == 0 and abs(x[0] - 0.3) < 1e-4
    x, fb, cnt, reason = gv.cobyla_minimize(lambda rows: np.zeros(len(rows)), np.ones(3), 1.0, 1e-3, 500)
    assert reason == 0 and fb == 0.0                                 # flat function: radius shrinks to rho_end, stops
    for bad in (dict(rho_beg=0.0), dict(rho_end=0.0), dict(rho_beg=1e-5, rho_end=1e-3), dict(max_evals=0)):
        kw = dict(rho_beg=1.0, rho_end=1e-3, max_evals=10)
        kw.update(bad)
        with pytest.raises(gv.GvqeError):
            gv.cobyla_minimize(lambda rows: np.zeros(len(rows)), np.ones(2), **kw)


def test_failing_function_is_reported():
    def fun(rows):
        raise RuntimeError("boom")
    with pytest.raises(gv.GvqeError):
        gv.cobyla_minimize(fun, np.ones(2), 1.0, 1e-3, 10)


def test_coupled_problem_reaches_a_stationary_point():
    """A non-separable smooth function (cosines with a coupling term): the point returned at rho_end = 1e-4 has a
    central-difference gradient of the order of rho_end and a value no worse than SciPy's to 1e-5."""
    rng = np.random.default_rng(11)
    a = rng.normal(size=8)
    f = lambda x: float(np.sum(a * np.cos(x)) + 0.3 * np.cos(x[0] + x[1]) - 0.2 * np.sin(x[2] - x[5]))
    x0 = rng.uniform(-1, 1, 8)
    x, fb, cnt, reason = gv.cobyla_minimize(_batch(f), x0, 1.0, 1e-4, 20000)
    assert reason == 0 and fb < f(x0)
    h = 1e-5
    g = np.array([(f(x + h * e) - f(x - h * e)) / (2 * h) for e in np.eye(8)])
    assert np.max(np.abs(g)) < 5e-3
    r = minimize(f, x0, method="COBYLA", options=dict(rhobeg=1.0, tol=1e-4, maxiter=20000))
    assert fb < r.fun + 1e-5

"""CPU oracle of the final-state read-out -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

PAPER.md:245: the state |psi(theta*)> gives a probability distribution over the computational basis states; "the
bitstring with the highest probability is identified as the optimal turn sequence".  Plain definition: p(x) = |psi_x|^2
(Born rule), x* = the x with the largest p(x), lowest x on ties (reading R1).  The state comes from oracle
T0 (complex128, gate by gate).  Pins: tests/test_graph_pins.py::test_readout_oracle_* (product-state closed form,
basis states, GHZ tie).
"""
from __future__ import annotations

import numpy as np

from . import state as _state


def probabilities(n: int, ops, theta) -> np.ndarray:
    psi = _state(n, ops, theta)
    return psi.real * psi.real + psi.imag * psi.imag


def most_probable(n: int, ops, theta):
    """(x*, p(x*)): largest probability, lowest index on ties."""
    p = probabilities(n, ops, theta)
    best = 0
    for x in range(1, len(p)):          # written out: strict '>' keeps the lowest index on ties
        if p[x] > p[best]:
            best = x
    return best, float(p[best])


def sample(n: int, ops, theta, u):
    """Shot sampling by inversion ("this state is sampled", 256: 8192 shots; reading R2): with the
    cumulative distribution F(x) = sum_{y <= x} p(y) in index order and Z = F(2^n - 1), shot s is the first x with
    F(x) > u_s Z.  The uniforms u_s in [0,1) are inputs.  Returns (x[len(u)], Z)."""
    p = probabilities(n, ops, theta)
    F = np.cumsum(p)                      # running sum in index order, fp64
    Z = float(F[-1])
    out = np.empty(len(u), dtype=np.uint64)
    for s, us in enumerate(u):
        t = float(us) * Z
        out[s] = min(int(np.searchsorted(F, t, side="right")), len(F) - 1)   # first x with F[x] > t
    return out, Z

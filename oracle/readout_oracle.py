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

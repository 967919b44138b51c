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


# ---- finite-shot energy estimate ("8192 measurement shots"; 270: shot-noise study; reading R3) ----
_H = np.array([[1.0, 1.0], [1.0, -1.0]], dtype=np.complex128) / np.sqrt(2.0)
_SDG = np.array([[1.0, 0.0], [0.0, -1.0j]], dtype=np.complex128)


def measurement_groups(n: int, pauli_list):
    """Partition of the terms into measurement settings: two terms share a setting when they have the same X/Y letters on
    the same qubits (identity and Z are read in the computational basis either way).  A setting is the pair
    (x_mask, y_mask); settings in ascending (x_mask, y_mask) order (all-Z/identity terms first).
    Returns (list of (x_mask, y_mask), group_of_term)."""
    keys = []
    for s in pauli_list:
        xm = sum(1 << q for q, ch in enumerate(s) if ch in "XY")
        ym = sum(1 << q for q, ch in enumerate(s) if ch == "Y")
        keys.append((xm, ym))
    settings = sorted(set(keys))
    return settings, [settings.index(kk) for kk in keys]


def rotate_to_setting(n: int, psi: np.ndarray, x_mask: int, y_mask: int) -> np.ndarray:
    """Amplitudes in the basis in which every X (Y) letter of the setting is diagonal: H on the X qubits, H S^dagger on
    the Y qubits (textbook: H X H = Z, (H S^dagger) Y (S H) = Z), qubit q = bit q of the index."""
    phi = np.array(psi, dtype=np.complex128).reshape([2] * n)           # axis a <-> qubit n-1-a
    for q in range(n):
        if not (x_mask >> q) & 1:
            continue
        g = _H @ _SDG if (y_mask >> q) & 1 else _H
        phi = np.moveaxis(np.tensordot(g, phi, axes=([1], [n - 1 - q])), 0, n - 1 - q)
    return phi.reshape(-1)


def energy_shots(n: int, ops, theta, pauli_list, coeffs, u):
    """Estimate of E = sum_k c_k <P_k> (Eq. 4, 6) from `S` shots per measurement setting: for setting g the state is
    rotated, S bitstrings are drawn by inversion with the uniforms u[g] (as in `sample`), and <P_k> is estimated as the
    mean of (-1)^{popcount(x & support_k)} over the shots of the term's setting.  u: array [n_settings, S] in [0, 1).
    Returns (E_est, term_means[len(coeffs)], shots[n_settings, S])."""
    psi = _state(n, ops, theta)
    settings, got = measurement_groups(n, pauli_list)
    u = np.asarray(u, dtype=np.float64).reshape(len(settings), -1)
    shots = np.zeros(u.shape, dtype=np.uint64)
    for g, (xm, ym) in enumerate(settings):
        phi = rotate_to_setting(n, psi, xm, ym)
        p = phi.real * phi.real + phi.imag * phi.imag
        F = np.cumsum(p)
        Z = float(F[-1])
        for s in range(u.shape[1]):
            shots[g, s] = min(int(np.searchsorted(F, float(u[g, s]) * Z, side="right")), len(F) - 1)
    means = np.zeros(len(coeffs))
    for k, s_ in enumerate(pauli_list):
        supp = sum(1 << q for q, ch in enumerate(s_) if ch != "I")
        sg = [1.0 - 2.0 * (bin(int(x) & supp).count("1") & 1) for x in shots[got[k]]]
        means[k] = float(np.mean(sg)) if len(sg) else 0.0
    return float(np.dot(np.asarray(coeffs, dtype=np.float64), means)), means, shots

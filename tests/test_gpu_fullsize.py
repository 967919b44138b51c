"""GPU parity at the sizes bench.py runs: libgvqe against the CPU oracle on NON-TRIVIAL states.  Run with -m gpu.

SURVEY.md 8(c) "Cost and tiers": T0 (plain gate-by-gate state, term-by-term expectation; Eq. 4/6, PAPER.md:135, 150,
on U(theta)|0>) is the authority; at n >= 28 it is affordable on a term subsample, which the library is
given through gvqe_set_hamiltonian, and T1 (FWHT table + mask-by-mask, pinned to T0 in tests/test_oracle_pins.py)
takes the full Hamiltonian for one row.  Gradients follow Eq. 13.  Tolerances: DESIGN.md reading A13.
The oracle state of a row is computed once and reused for every comparison on that row.
"""
import math

import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from workload import make_workload

pytestmark = pytest.mark.gpu


def tol(prec, E_ref, coeffs):
    s = float(np.sum(np.abs(coeffs)))
    E_ref = np.abs(np.asarray(E_ref, dtype=np.float64))
    if prec == "c128":
        return 1e-10 * E_ref + 1e-12 * s
    return np.maximum(1e-4 * E_ref, 1e-5 * s)


def grad_tol(prec, Ep, Em, coeffs):
    """A13: the energy bound applied to (E+ - E-)/2 with |E| replaced by (|E+| + |E-|)/2."""
    return tol(prec, 0.5 * (abs(Ep) + abs(Em)), coeffs)


def subsample(w, count=64):
    """Evenly spaced terms of the config's Hamiltonian (keeps its Z-only / X-Y mix), as (paulis, coeffs)."""
    idx = np.arange(0, w.M, max(1, w.M // count))[:count]
    pl = w.pauli_list()
    return "".join(pl[i] for i in idx).encode(), w.coeffs[idx]


def host_ram_gib():
    try:
        import psutil
        return psutil.virtual_memory().available / 2 ** 30
    except Exception:
        return 0.0


def make_ctx(w, prec, in_flight, paulis, coeffs):
    g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology, final_rot=w.final_rot),
                precision=prec)
    g.set_hamiltonian(paulis, coeffs)
    g.alloc_workspace(in_flight)
    return g


def test_config4_full_size_vs_oracle(orc):
    """Config 4 as generated (28 qubits, 6 layers, CNOT ring, c64, 8 statevectors in flight).
    (a) rows 0 and 5 of the 729-row shift set against T0 on a 64-term subsample (library given the same subsample);
    (b) one parameter-shift gradient entry in c64 against Eq. 13 evaluated by T0 on the subsample;
    (c) row 0 against T1 on the full 20 000-term Hamiltonian."""
    w = make_workload(4)
    assert w.n == 28 and w.P == 364 and w.B == 729
    sub_p, sub_c = subsample(w, 64)
    assert any(ch in sub_p.decode() for ch in "XY")
    g = make_ctx(w, "c64", 8, sub_p, sub_c)
    E = g.energy_batch(w.params[:8])                               # one full chunk of 8
    psi = {}
    for b in (0, 5):
        psi[b] = orc.state(w.n, w.ops, w.params[b])
        assert abs(orc.norm2(w.n, psi[b]) - 1.0) < 1e-10
        ref = orc.energy_of_state(w.n, psi[b], sub_p, sub_c)
        assert abs(E[b] - ref) <= tol("c64", ref, sub_c), (b, E[b], ref)
    del psi[5]
    # (b) gradient entry: a first-layer RZ parameter of the highest qubit (prefix kernel, every block, every pass)
    p = w.n + w.n - 1
    mask = np.zeros(w.P, dtype=np.uint8)
    mask[p] = 1
    dE, E0 = g.param_shift_grad(w.theta, mask)
    Epm = []
    for sgn in (+1.0, -1.0):
        th = w.theta.copy()
        th[p] += sgn * math.pi / 2
        ps = orc.state(w.n, w.ops, th)
        Epm.append(orc.energy_of_state(w.n, ps, sub_p, sub_c))
        del ps
    ref0 = orc.energy_of_state(w.n, psi[0], sub_p, sub_c)
    assert abs(E0 - ref0) <= tol("c64", ref0, sub_c)
    assert abs(dE[p] - 0.5 * (Epm[0] - Epm[1])) <= grad_tol("c64", Epm[0], Epm[1], sub_c), (dE[p], Epm)
    assert np.all(dE[mask == 0] == 0.0)
    # (c) the full Hamiltonian, same state, T1
    del g
    g = make_ctx(w, "c64", 8, w.paulis, w.coeffs)
    Ef = g.energy_batch(w.params[:8])
    ref = orc.t1_energy_of_state(w.n, psi[0], w.paulis, w.coeffs)
    assert abs(Ef[0] - ref) <= tol("c64", ref, w.coeffs), (Ef[0], ref)


def test_config5b_full_size_vs_oracle(orc):
    """Config 5b as generated (30 qubits c128, 4 layers, CZ chain, one statevector): the random-angle row against T0
    on a 64-term subsample at the complex128 tolerance."""
    if host_ram_gib() < 40:
        pytest.skip("needs a 16 GiB complex128 oracle state plus workspace on the host")
    w = make_workload(6)
    assert w.n == 30
    sub_p, sub_c = subsample(w, 64)
    g = make_ctx(w, "c128", 1, sub_p, sub_c)
    E = g.energy_batch(w.params[:1])
    psi = orc.state(w.n, w.ops, w.params[0])
    ref = orc.energy_of_state(w.n, psi, sub_p, sub_c)
    assert abs(E[0] - ref) <= tol("c128", ref, sub_c), (E[0], ref)


def test_config5a_full_size_vs_oracle(orc):
    """Config 5a as generated (32 qubits c64, 32 GiB state): the random-angle row against T0 on a 32-term subsample.
    The oracle state is 64 GiB of complex128: skipped (and reported as such) when the host cannot hold it."""
    if host_ram_gib() < 100:
        pytest.skip("needs a 64 GiB complex128 oracle state on the host")
    w = make_workload(5)
    assert w.n == 32
    sub_p, sub_c = subsample(w, 32)
    g = make_ctx(w, "c64", 1, sub_p, sub_c)
    E = g.energy_batch(w.params[:1])
    psi = orc.state(w.n, w.ops, w.params[0])
    ref = orc.energy_of_state(w.n, psi, sub_p, sub_c)
    assert abs(E[0] - ref) <= tol("c64", ref, sub_c), (E[0], ref)


def test_config3_c64_cluster_gradient(orc):
    """Config 3 size (22 qubits, c64, 64 in flight): cluster-restricted gradient (community 0: 4 qubits x 11 rotations)
    against orc_param_shift_grad on a 300-term subsample, each entry at A13's gradient bound."""
    from workload.generator import community_param_mask, shift_rows

    w = make_workload(3)
    idx = np.arange(0, w.M, 17)
    pl = w.pauli_list()
    sub_p, sub_c = "".join(pl[i] for i in idx).encode(), w.coeffs[idx]
    mask = community_param_mask(w.n, w.D, w.final_rot, w.communities[0])
    assert int(mask.sum()) == 44
    g = make_ctx(w, "c64", 64, sub_p, sub_c)
    dE, E0 = g.param_shift_grad(w.theta, mask)
    rows = shift_rows(w.theta, mask)
    Er = orc.energy_batch(w.n, w.ops, rows, sub_p, sub_c)
    assert abs(E0 - Er[0]) <= tol("c64", Er[0], sub_c)
    for j, p in enumerate(np.flatnonzero(mask)):
        Ep, Em = Er[2 * j + 1], Er[2 * j + 2]
        assert abs(dE[p] - 0.5 * (Ep - Em)) <= grad_tol("c64", Ep, Em, sub_c), (p, dE[p], Ep, Em)
    assert np.all(dE[mask == 0] == 0.0)

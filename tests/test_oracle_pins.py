"""Pins for the CPU oracle (oracle/): what the paper and the mathematics fix, NOT the oracle against itself.

Each test names the oracle function it pins and the mistake it would catch.  CPU only (-m "not gpu")."""
import math
import os

import numpy as np
import pytest

from tests import dense_ref as dr
from workload import make_workload, layout_ops, num_params, OP_RY, OP_RZ, OP_CZ, OP_CNOT
from workload.generator import random_ops, random_paulis

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def split(paulis: bytes, n: int):
    s = paulis.decode()
    return [s[i:i + n] for i in range(0, len(s), n)]


# ---- dense Kronecker brute force, n <= 8: pins orc_state + orc_energy (gate matrices, op order, bit order,
# ---- CNOT direction, Y sign, coefficient handling) ------------------------------------------------------
@pytest.mark.parametrize("n,seed", [(1, 1), (2, 2), (3, 3), (4, 4), (5, 5), (6, 6)])
def test_dense_random_circuits(orc, n, seed):
    ops, P = random_ops(1000 + seed, n, 24)
    rng = np.random.default_rng(seed)
    theta = rng.uniform(-math.pi, math.pi, max(P, 1))
    paulis, coeffs = random_paulis(2000 + seed, n, 30, n)
    E_d, psi_d = dr.dense_energy(n, ops, theta, split(paulis, n), coeffs)
    psi = orc.state(n, ops, theta)
    assert np.max(np.abs(psi - psi_d)) < 1e-13
    E, terms, max_imag = orc.energy_of_state(n, psi, paulis, coeffs, return_terms=True)
    assert abs(E - E_d) < 1e-12 * max(1.0, np.sum(np.abs(coeffs)))
    assert max_imag < 1e-12
    # every single term separately (a wrong i^{nY} or sign on one letter shows here)
    for s, t in zip(split(paulis, n), terms):
        Pm = dr.kron_on(n, {q: dr.PAULI[ch] for q, ch in enumerate(s)})
        assert abs(t - np.real(np.vdot(psi_d, Pm @ psi_d))) < 1e-12


@pytest.mark.parametrize("n,D,ent,topo,fr", [(4, 2, "cz", "linear", 1), (5, 2, "cnot", "ring", 1),
                                               (6, 1, "cnot", "linear", 2), (8, 1, "cz", "linear", 1),
                                               (7, 2, "cnot", "ring", 2)])
def test_dense_layered_ansatz(orc, n, D, ent, topo, fr):
    ops = np.array(layout_ops(n, D, ent, topo, fr), dtype=np.int32)
    P = num_params(n, D, fr)
    theta = np.random.default_rng(n * 10 + D).uniform(-math.pi, math.pi, P)
    paulis, coeffs = random_paulis(77 + n, n, 40, 4)
    E_d, psi_d = dr.dense_energy(n, ops, theta, split(paulis, n), coeffs)
    assert np.max(np.abs(orc.state(n, ops, theta) - psi_d)) < 1e-13
    E = orc.energy_batch(n, ops, theta, paulis, coeffs)[0]
    assert abs(E - E_d) < 1e-12 * np.sum(np.abs(coeffs))


def test_config1_like_dense(orc):
    """BASELINE config 1 recipe shrunk to 8 qubits: 'oracle brute-force dense check'."""
    w = make_workload(1, n=8, M=60)
    E = orc.energy_batch(w.n, w.ops, w.params[:3], w.paulis, w.coeffs)
    for b in range(3):
        E_d, _ = dr.dense_energy(w.n, w.ops, w.params[b], w.pauli_list(), w.coeffs)
        assert abs(E[b] - E_d) < 1e-12 * np.sum(np.abs(w.coeffs))


# ---- paper-printed numbers: Eq. 8 parameter count and Eq. 5 qubit count (tests/golden/paper_counts.txt) ----
def test_paper_parameter_counts():
    rows = [l.split() for l in open(os.path.join(GOLD, "paper_counts.txt")) if l.strip() and not l.startswith("#")]
    assert rows
    for L, N, D, P in rows:
        L, N, D, P = int(L), int(N), int(D), int(P)
        assert N == 2 * (L - 1)
        assert num_params(N, D, 2) == P                      # Eq. 8, final layer has RY and RZ
        ops = layout_ops(N, D, "cnot", "ring", 2)
        assert 1 + max(o[3] for o in ops) == P
        assert sorted(o[3] for o in ops if o[3] >= 0) == list(range(P))


# ---- closed forms -----------------------------------------------------------------------------------------
def test_bloch_vector_n1(orc):
    """RZ(phi) RY(theta)|0>: <Z>=cos th, <X>=sin th cos phi, <Y>=sin th sin phi.  Pins Eq. 7 signs and Y."""
    ops = np.array([[OP_RY, 0, -1, 0], [OP_RZ, 0, -1, 1]], dtype=np.int32)
    for th, ph in [(0.3, 1.1), (-2.0, 0.4), (2.7, -2.9), (math.pi / 2, math.pi / 2)]:
        psi = orc.state(1, ops, [th, ph])
        want = np.array([math.cos(th / 2) * np.exp(-0.5j * ph), math.sin(th / 2) * np.exp(0.5j * ph)])
        assert np.max(np.abs(psi - want)) < 1e-15
        _, t, _ = orc.energy_of_state(1, psi, b"ZXYI", [1, 1, 1, 1], return_terms=True)
        assert np.allclose(t, [math.cos(th), math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), 1.0],
                           atol=1e-14)


def test_product_state_closed_form(orc):
    """Rotations only => <P> = prod_q f_q; pins X/Y/Z handling on every qubit position, n = 14."""
    n = 14
    ops = [(OP_RY, q, -1, q) for q in range(n)] + [(OP_RZ, q, -1, n + q) for q in range(n)]
    rng = np.random.default_rng(5)
    th = rng.uniform(-math.pi, math.pi, 2 * n)
    paulis, coeffs = random_paulis(31, n, 50, 6)
    _, t, _ = orc.energy_of_state(n, orc.state(n, ops, th), paulis, coeffs, return_terms=True)
    f = {"I": lambda q: 1.0, "Z": lambda q: math.cos(th[q]), "X": lambda q: math.sin(th[q]) * math.cos(th[n + q]),
         "Y": lambda q: math.sin(th[q]) * math.sin(th[n + q])}
    want = [math.prod(f[ch](q) for q, ch in enumerate(s)) for s in split(paulis, n)]
    assert np.allclose(t, want, atol=1e-13)


def test_ghz(orc):
    n = 9
    ops = [(OP_RY, 0, -1, 0)] + [(OP_CNOT, q + 1, q, -1) for q in range(n - 1)]
    psi = orc.state(n, ops, [math.pi / 2])
    want = np.zeros(1 << n, dtype=complex)
    want[0] = want[-1] = 1 / math.sqrt(2)
    assert np.max(np.abs(psi - want)) < 1e-15
    strs = ["ZZ" + "I" * (n - 2), "Z" + "I" * (n - 1), "X" * n, "I" * (n - 3) + "ZIZ", "YY" + "X" * (n - 2)]
    _, t, _ = orc.energy_of_state(n, psi, "".join(strs).encode(), [1] * 5, return_terms=True)
    assert np.allclose(t, [1, 0, 1, 1, -1], atol=1e-14)      # Y Y X..X on GHZ = i^2 = -1


def test_cz_matches_definition(orc):
    """CZ(a,b) = H_b CNOT(a->b) H_b is avoided on purpose; pin it by amplitudes instead."""
    n = 3
    ops = [(OP_RY, q, -1, q) for q in range(n)] + [(OP_CZ, 0, 2, -1)]
    th = [0.7, -1.3, 2.1]
    a = orc.state(n, ops[:n], th)
    b = orc.state(n, ops, th)
    sign = np.array([-1.0 if (x & 1) and (x & 4) else 1.0 for x in range(8)])
    assert np.allclose(b, a * sign, atol=1e-16)


# ---- invariants -------------------------------------------------------------------------------------------
def test_norm_preserved(orc):
    for cfg, n in [(2, 10), (4, 11)]:
        w = make_workload(cfg, n=n, M=10)
        for b in range(2):
            assert abs(orc.norm2(w.n, orc.state(w.n, w.ops, w.params[b])) - 1.0) < 1e-12


def test_theta_zero_gives_z_coefficient_sum(orc):
    w = make_workload(2, n=10, M=300)
    E = orc.energy_batch(w.n, w.ops, np.zeros(w.P), w.paulis, w.coeffs)[0]
    want = sum(c for s, c in zip(w.pauli_list(), w.coeffs) if "X" not in s and "Y" not in s)
    assert abs(E - want) < 1e-11


def test_basis_state_energy_and_diagonal_ground_state(orc):
    """Z-only H (config 1 recipe): last-layer RY(pi x_q), other angles 0 => psi = +-e_x => E = E(x);
    min_x E(x) by enumeration lower-bounds E(theta) and is attained."""
    w = make_workload(1, n=10, M=200)
    n = w.n
    zs = [sum(1 << q for q, ch in enumerate(s) if ch == "Z") for s in w.pauli_list()]
    Ex = np.array([sum(c * (-1) ** bin(x & z).count("1") for z, c in zip(zs, w.coeffs)) for x in range(1 << n)])
    xmin = int(np.argmin(Ex))
    th = np.zeros(w.P)
    for q in range(n):
        th[2 * n * w.D + q] = math.pi * ((xmin >> q) & 1)
    psi = orc.state(n, w.ops, th)
    assert abs(abs(psi[xmin]) - 1.0) < 1e-12
    E = orc.energy_batch(n, w.ops, np.vstack([th, w.params[:6]]), w.paulis, w.coeffs)
    assert abs(E[0] - Ex[xmin]) < 1e-10
    assert np.all(E[1:] >= Ex[xmin] - 1e-10)
    assert np.all(np.abs(E) <= np.sum(np.abs(w.coeffs)) + 1e-10)


def test_eq12_additivity(orc):
    """Eq. 12: energies of any partition of the terms add to the full energy."""
    w = make_workload(2, n=9, M=120)
    pl, n = w.pauli_list(), w.n
    th = w.params[1]
    full = orc.energy_batch(n, w.ops, th, w.paulis, w.coeffs)[0]
    parts = 0.0
    for j in range(4):
        idx = list(range(j, w.M, 4))
        parts += orc.energy_batch(n, w.ops, th, "".join(pl[i] for i in idx).encode(), w.coeffs[idx])[0]
    assert abs(full - parts) < 1e-11


def test_sinusoid_in_one_parameter(orc):
    """E(theta_p) = a + b cos + c sin: three points predict a fourth; 2 pi periodic."""
    w = make_workload(3, n=8, M=80, D=2)
    th = w.params[0].copy()
    for p in (0, w.n + 3, w.P - 1):
        def e(v):
            t = th.copy()
            t[p] = v
            return orc.energy_batch(w.n, w.ops, t, w.paulis, w.coeffs)[0]
        e0, e1, e2 = e(0.0), e(math.pi / 2), e(math.pi)
        a, b, c = (e0 + e2) / 2, (e0 - e2) / 2, e1 - (e0 + e2) / 2
        v = 0.8137
        assert abs(e(v) - (a + b * math.cos(v) + c * math.sin(v))) < 1e-11
        assert abs(e(v + 2 * math.pi) - e(v)) < 1e-11


# ---- gradients: pins orc_param_shift_grad (Eq. 13) against central finite differences -------------------------
@pytest.mark.parametrize("cfg,n", [(2, 8), (4, 9)])
def test_param_shift_vs_finite_differences(orc, cfg, n):
    w = make_workload(cfg, n=n, M=100, D=2)
    mask = np.zeros(w.P, dtype=np.uint8)
    mask[[0, 3, n + 1, 2 * n + 2, w.P - 1]] = 1
    dE, E0 = orc.param_shift_grad(w.n, w.ops, w.theta, mask, w.paulis, w.coeffs)
    assert abs(E0 - orc.energy_batch(w.n, w.ops, w.theta, w.paulis, w.coeffs)[0]) < 1e-12
    h = 1e-5
    for p in range(w.P):
        if not mask[p]:
            assert dE[p] == 0.0
            continue
        tp, tm = w.theta.copy(), w.theta.copy()
        tp[p] += h
        tm[p] -= h
        fd = (orc.energy_batch(w.n, w.ops, tp, w.paulis, w.coeffs)[0]
              - orc.energy_batch(w.n, w.ops, tm, w.paulis, w.coeffs)[0]) / (2 * h)
        assert abs(fd - dE[p]) < 1e-7 * max(1.0, np.sum(np.abs(w.coeffs)))


# ---- T1 (FWHT table + mask-by-mask) must equal T0 before it is used at n >= 26 --------------------------------
@pytest.mark.parametrize("cfg,n,M", [(1, 10, 200), (2, 12, 400), (3, 12, 500), (4, 12, 600), (5, 13, 500)])
def test_t1_equals_t0(orc, cfg, n, M):
    w = make_workload(cfg, n=n, M=M, D=2)
    psi = orc.state(w.n, w.ops, w.params[0])
    e0 = orc.energy_of_state(w.n, psi, w.paulis, w.coeffs)
    e1 = orc.t1_energy_of_state(w.n, psi, w.paulis, w.coeffs)
    assert abs(e0 - e1) < 1e-11 * np.sum(np.abs(w.coeffs))


def test_t1_table_is_plain_definition(orc):
    n = 7
    paulis, coeffs = random_paulis(9, n, 60, 5)
    tab = orc.t1_diag_table(n, paulis, coeffs)
    for x in range(1 << n):
        want = 0.0
        for s, c in zip(split(paulis, n), coeffs):
            if "X" in s or "Y" in s:
                continue
            z = sum(1 << q for q, ch in enumerate(s) if ch == "Z")
            want += c * (-1) ** bin(x & z).count("1")
        assert abs(tab[x] - want) < 1e-12


# ---- integer grouping: pins orc_grouping against a few lines of Python -------------------------------------
def test_grouping_definition(orc):
    n = 11
    paulis, _ = random_paulis(123, n, 200, 4)
    xm, zm, ny, got, ng, gm = orc.grouping(n, paulis)
    strs = split(paulis, n)
    for k, s in enumerate(strs):
        assert xm[k] == sum(1 << q for q, ch in enumerate(s) if ch in "XY")
        assert zm[k] == sum(1 << q for q, ch in enumerate(s) if ch in "ZY")
        assert ny[k] == s.count("Y") % 4
    want = sorted(set(int(v) for v in xm))
    assert ng == len(want) and [int(v) for v in gm] == want
    assert all(want[g] == int(xm[k]) for k, g in enumerate(got))


def test_bad_pauli_character(orc):
    with pytest.raises(ValueError):
        orc.grouping(3, b"XQZ")
    assert math.isnan(orc.energy_of_state(2, np.array([1, 0, 0, 0], dtype=complex), b"XA", [1.0]))

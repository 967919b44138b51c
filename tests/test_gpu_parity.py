"""GPU parity: libgvqe (through the C ABI) against the CPU oracle on the same seeded inputs.  Run with -m gpu.

Tolerances (BASELINE.json north_star; reading A13):
  complex128: |dE| <= 1e-10 |E_oracle| + 1e-12 sum|c_k|
  complex64 : |dE| <= max(1e-4 |E_oracle|, 1e-5 sum|c_k|)
Masks / grouping are bit-exact (tests/test_host_logic.py, CPU)."""
import math
import re
import os

import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from workload import make_workload, layout_ops, num_params, OP_RY, OP_RZ, OP_CZ, OP_CNOT
from workload.generator import random_ops, random_paulis

pytestmark = pytest.mark.gpu


def tol(prec, E_ref, coeffs):
    s = float(np.sum(np.abs(coeffs)))
    E_ref = np.abs(np.asarray(E_ref, dtype=np.float64))
    if prec == "c128":
        return 1e-10 * E_ref + 1e-12 * max(s, 1e-300)
    return np.maximum(1e-4 * E_ref, 1e-5 * s)


def assert_close(prec, E, E_ref, coeffs, what=""):
    E, E_ref = np.asarray(E), np.asarray(E_ref)
    bad = np.abs(E - E_ref) > tol(prec, E_ref, coeffs)
    assert not bad.any(), f"{what}: max |dE| = {np.max(np.abs(E - E_ref)):.3e}, first bad row {int(np.argmax(bad))}"


def ctx_for(w, prec, in_flight=None, ops=False, options=None):
    if ops:
        g = gv.Gvqe(w.n, ops=w.ops, n_params=w.P, precision=prec, options=options)
    else:
        g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology, final_rot=w.final_rot),
                    precision=prec, options=options)
    g.set_hamiltonian(w.paulis, w.coeffs)
    g.alloc_workspace(in_flight or min(w.B, 64))
    return g


# ---- BASELINE configs ----------------------------------------------------------------------------------------
def test_config1_full(orc):
    """10 qubits, c128, Z-only H, the 2P+1 = 141 row parameter-shift set; every row against T0."""
    w = make_workload(1)
    g = ctx_for(w, "c128", 141)
    E = g.energy_batch(w.params)
    assert_close("c128", E, orc.energy_batch(w.n, w.ops, w.params, w.paulis, w.coeffs), w.coeffs, "cfg1")
    dE, E0 = g.param_shift_grad(w.theta, w.mask)
    dE_o, E0_o = orc.param_shift_grad(w.n, w.ops, w.theta, w.mask, w.paulis, w.coeffs)
    assert abs(E0 - E0_o) <= tol("c128", E0_o, w.coeffs)
    for j, p in enumerate(np.flatnonzero(w.mask)):              # A13: |E| -> (|E+| + |E-|) / 2, per parameter
        assert abs(dE[p] - dE_o[p]) <= tol("c128", 0.5 * (abs(E[2 * j + 1]) + abs(E[2 * j + 2])), w.coeffs), p


def test_config2_full_cluster_gradient(orc):
    """16 qubits, c128, 1000 terms (15 % X/Y), cluster-restricted gradient over community 0 (36 params, batch 73)."""
    w = make_workload(2)
    assert int(w.mask.sum()) == 36 and w.B == 73
    g = ctx_for(w, "c128", 73)
    dE, E0 = g.param_shift_grad(w.theta, w.mask)
    dE_o, E0_o = orc.param_shift_grad(w.n, w.ops, w.theta, w.mask, w.paulis, w.coeffs)
    assert abs(E0 - E0_o) <= tol("c128", E0_o, w.coeffs)
    assert np.all(dE[w.mask == 0] == 0.0)
    E = g.energy_batch(w.params)
    for j, p in enumerate(np.flatnonzero(w.mask)):              # A13 gradient bound, per parameter
        assert abs(dE[p] - dE_o[p]) <= tol("c128", 0.5 * (abs(E[2 * j + 1]) + abs(E[2 * j + 2])), w.coeffs), p
    assert_close("c128", E[:8], orc.energy_batch(w.n, w.ops, w.params[:8], w.paulis, w.coeffs), w.coeffs, "cfg2 rows")


@pytest.mark.parametrize("prec", ["c64", "c128"])
def test_config3_full_sampled(orc, prec):
    """22 qubits, 5000 terms, batch 64 in the bench launch configuration; rows 0, 31, 63 against the oracle
    (T1 for all three, T0 term-by-term for row 0 on a 300-term subsample of the same Hamiltonian)."""
    w = make_workload(3)
    g = ctx_for(w, prec, 64)
    E = g.energy_batch(w.params)
    rows = [0, 31, 63]
    ref = []
    for b in rows:
        psi = orc.state(w.n, w.ops, w.params[b])
        ref.append(orc.t1_energy_of_state(w.n, psi, w.paulis, w.coeffs))
    assert_close(prec, E[rows], ref, w.coeffs, f"cfg3 {prec}")
    # T0 on a subsample through the same library path
    idx = np.arange(0, w.M, 17)
    pl = w.pauli_list()
    sub_p = "".join(pl[i] for i in idx).encode()
    g.set_hamiltonian(sub_p, w.coeffs[idx])
    g.alloc_workspace(1)
    E0 = g.energy_batch(w.params[:1])
    psi = orc.state(w.n, w.ops, w.params[0])
    assert_close(prec, E0, [orc.energy_of_state(w.n, psi, sub_p, w.coeffs[idx])], w.coeffs[idx], "cfg3 T0 subsample")


def test_config4_shape_at_24_qubits(orc):
    """Config 4 recipe (CNOT ring, pooled flip masks, c64) at 24 qubits, 2 layers: one row against T1."""
    w = make_workload(4, n=24, M=4000, D=2, batch=2)
    g = ctx_for(w, "c64", 2)
    E = g.energy_batch(w.params)
    psi = orc.state(w.n, w.ops, w.params[1])
    assert_close("c64", E[1:2], [orc.t1_energy_of_state(w.n, psi, w.paulis, w.coeffs)], w.coeffs, "cfg4@24")


def test_config4_full_size_properties():
    """28 qubits c64, full 20 000-term Hamiltonian, chunks of 8: properties that hold at any size."""
    w = make_workload(4)
    g = ctx_for(w, "c64", 8)
    zsum = sum(c for s, c in zip(w.pauli_list(), w.coeffs) if "X" not in s and "Y" not in s)
    rows = np.zeros((9, w.P))                                   # 9 rows -> two chunks (8 + 1)
    rng = np.random.default_rng(4)
    xs = [0]
    for b in range(1, 9):                                       # last-layer RY(pi x_q): psi = +-e_x, E = E_diag(x)
        x = int(rng.integers(0, 1 << w.n))
        xs.append(x)
        for q in range(w.n):
            rows[b, 2 * w.n * w.D + q] = math.pi * ((x >> q) & 1)
    E = g.energy_batch(rows)
    zs = [(sum(1 << q for q, ch in enumerate(s) if ch == "Z"), c) for s, c in zip(w.pauli_list(), w.coeffs)
          if "X" not in s and "Y" not in s]
    want = [sum(c * (-1) ** bin(x & z).count("1") for z, c in zs) for x in xs]
    assert abs(want[0] - zsum) < 1e-9
    assert_close("c64", E, want, w.coeffs, "cfg4 basis states")
    E2 = g.energy_batch(w.params[:3])                           # random angles: bound and determinism
    assert np.all(np.abs(E2) <= np.sum(np.abs(w.coeffs)))
    assert np.array_equal(E2, g.energy_batch(w.params[:3]))


# ---- embedding: an n' problem on arbitrary (high) qubits of a larger register equals the n' oracle energy ------------
@pytest.mark.parametrize("prec,n_big", [("c64", 26), ("c128", 25)])
def test_embedding_on_high_qubits(orc, prec, n_big):
    n_s = 12
    w = make_workload(4, n=n_s, M=300, D=2, batch=2)
    place = [1, 3, 6, 9, 11, 14, 15, 17, 20, 22, n_big - 2, n_big - 1]
    ops = w.ops.copy()
    for o in ops:
        o[1] = place[o[1]]
        if o[2] >= 0:
            o[2] = place[o[2]]
    pl = []
    for s in w.pauli_list():
        t = ["I"] * n_big
        for q, ch in enumerate(s):
            t[place[q]] = ch
        t[0] = "Z"                                               # idle qubit 0 stays |0>: Z contributes +1
        pl.append("".join(t))
    g = gv.Gvqe(n_big, ops=ops, n_params=w.P, precision=prec)
    g.set_hamiltonian("".join(pl).encode(), w.coeffs)
    g.alloc_workspace(2)
    E = g.energy_batch(w.params)
    assert_close(prec, E, orc.energy_batch(n_s, w.ops, w.params, w.paulis, w.coeffs), w.coeffs, "embedding")


# ---- randomised small cases: arbitrary op lists and Pauli strings, several tiles, ragged sizes ------------------------
@pytest.mark.parametrize("seed", range(14))
def test_random_circuits_and_paulis(orc, seed):
    n = 1 + seed
    prec = "c64" if seed % 2 else "c128"
    ops, P = random_ops(7000 + seed, n, 150)
    paulis, coeffs = random_paulis(8000 + seed, n, 80, min(n, 6))
    th = np.random.default_rng(seed).uniform(-math.pi, math.pi, (5, P))
    # n > k from n = 11 on: multi-tile and strided blocks
    g = gv.Gvqe(n, ops=ops, n_params=P, precision=prec, options=dict(tile_bits=10 + seed % 3))
    g.set_hamiltonian(paulis, coeffs)
    g.alloc_workspace(3)                                         # 5 rows in chunks of 3 + 2
    E = g.energy_batch(th)
    assert_close(prec, E, orc.energy_batch(n, ops, th, paulis, coeffs), coeffs, f"random n={n}")
    psi = g.get_state(1)                                         # slot 1 of the last chunk = row 4
    ref = orc.state(n, ops, th[4])
    assert np.max(np.abs(psi - ref)) < (1e-12 if prec == "c128" else 2e-5)


@pytest.mark.parametrize("n,D,ent,topo,fr,prec", [(13, 3, "cz", "linear", 1, "c64"), (15, 2, "cnot", "ring", 1, "c64"),
                                                   (14, 2, "cnot", "linear", 2, "c128"), (16, 3, "cz", "ring", 2, "c128"),
                                                   (17, 2, "cnot", "ring", 1, "c128"), (18, 2, "cz", "linear", 2, "c64"),
                                                   # the paper's other entanglement maps (reading A17)
                                                   (12, 2, "cnot", "full", 1, "c128"), (15, 3, "cnot", "reverse_linear", 1, "c64"),
                                                   (14, 3, "cnot", "pairwise", 2, "c128"), (13, 2, "cnot", "circular", 1, "c128"),
                                                   (15, 4, "cnot", "sca", 1, "c128"), (16, 3, "cz", "full", 1, "c64"),
                                                   (17, 3, "cnot", "sca", 2, "c64")])
def test_layered_ansatz_variants(orc, n, D, ent, topo, fr, prec):
    ops = np.array(layout_ops(n, D, ent, topo, fr), dtype=np.int32)
    P = num_params(n, D, fr)
    paulis, coeffs = random_paulis(100 + n, n, 120, 5)
    th = np.random.default_rng(n).uniform(-math.pi, math.pi, (4, P))
    g = gv.Gvqe(n, layout=dict(n_layers=D, entangler=ent, topology=topo, final_rot=fr), precision=prec)
    g.set_hamiltonian(paulis, coeffs)
    g.alloc_workspace(4)
    assert_close(prec, g.energy_batch(th), orc.energy_batch(n, ops, th, paulis, coeffs), coeffs, "layered")


# ---- edge cases ----------------------------------------------------------------------------------------------------
def test_edge_cases(orc):
    n = 11
    ops = np.array(layout_ops(n, 1, "cz", "linear", 1), dtype=np.int32)
    P = num_params(n, 1, 1)
    th = np.random.default_rng(0).uniform(-math.pi, math.pi, (3, P))
    g = gv.Gvqe(n, ops=ops, n_params=P, precision="c128")
    # empty Hamiltonian, identity only, duplicates, a weight-n string (direct mode), empty batch
    g.set_hamiltonian(b"", [])
    g.alloc_workspace(3)
    assert np.array_equal(g.energy_batch(th), np.zeros(3))
    g.set_hamiltonian(b"I" * n, [2.5])
    g.alloc_workspace(3)
    assert np.allclose(g.energy_batch(th), 2.5, atol=1e-12)
    strs = ["ZZ" + "I" * (n - 2)] * 3 + ["XYZ" + "I" * (n - 3)] * 2 + ["Y" * n, "X" + "Z" * (n - 1), "Z" * n]
    cs = np.array([0.5, -1.5, 2.0, 0.3, 0.4, 1.1, -0.7, 0.9])
    g.set_hamiltonian("".join(strs).encode(), cs)
    g.alloc_workspace(2)
    assert_close("c128", g.energy_batch(th), orc.energy_batch(n, ops, th, "".join(strs).encode(), cs), cs, "edge")
    assert len(g.energy_batch(np.zeros((0, P)))) == 0
    with pytest.raises(gv.GvqeError):
        g.energy_batch(np.full((1, P), np.nan))
    # a circuit with no parameters and no ops at all
    g0 = gv.Gvqe(3, ops=np.zeros((0, 4), dtype=np.int32), n_params=0, precision="c64")
    g0.set_hamiltonian(b"ZIZ" + b"XII", [1.0, 1.0])
    g0.alloc_workspace(1)
    assert abs(g0.energy_batch(np.zeros((1, 0)))[0] - 1.0) < 1e-6


def test_chunking_determinism_and_device_api():
    import torch

    w = make_workload(3, n=15, M=600, D=3, batch=10)
    a = ctx_for(w, "c64", 10)
    b = ctx_for(w, "c64", 10)
    b.set_max_in_flight(3)
    Ea, Eb = a.energy_batch(w.params), b.energy_batch(w.params)
    assert np.array_equal(Ea, Eb)                                # chunking does not change a bit
    assert np.array_equal(Ea, a.energy_batch(w.params))          # repeated call is bit-identical
    p_dev = torch.from_numpy(w.params).cuda()
    E_dev = torch.zeros(10, dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    a.energy_batch_device(p_dev.data_ptr(), 10, E_dev.data_ptr(), s.cuda_stream)
    s.synchronize()
    assert np.array_equal(E_dev.cpu().numpy(), Ea)
    assert a.launch_count() > 0


def test_final_rot_2_is_eq8(orc):
    """Eq. 8 layout (final layer RY and RZ): P = 2N(D+1)."""
    n, D = 12, 2
    ops = np.array(layout_ops(n, D, "cnot", "ring", 2), dtype=np.int32)
    g = gv.Gvqe(n, layout=dict(n_layers=D, entangler="cnot", topology="ring", final_rot=2), precision="c128")
    assert g.P == 2 * n * (D + 1)
    paulis, coeffs = random_paulis(3, n, 60, 4)
    g.set_hamiltonian(paulis, coeffs)
    g.alloc_workspace(2)
    th = np.random.default_rng(1).uniform(-math.pi, math.pi, (2, g.P))
    assert_close("c128", g.energy_batch(th), orc.energy_batch(n, ops, th, paulis, coeffs), coeffs, "eq8")


# ---- config 5: 32 qubits complex64 (32 GiB state) and 30 qubits complex128 (16 GiB), single statevector ---------------
def _product_state_energy(n, theta_ry, theta_rz, pauli_list, coeffs):
    """Closed form for a rotations-only circuit RZ(phi_q) RY(theta_q) on every qubit (tests/test_oracle_pins.py pins
    the oracle to the same formula): <P> = prod_q f_q, f = 1, cos th, sin th cos phi, sin th sin phi for I, Z, X, Y."""
    E = 0.0
    for s, c in zip(pauli_list, coeffs):
        v = c
        for q, ch in enumerate(s):
            if ch == "Z":
                v *= math.cos(theta_ry[q])
            elif ch == "X":
                v *= math.sin(theta_ry[q]) * math.cos(theta_rz[q])
            elif ch == "Y":
                v *= math.sin(theta_ry[q]) * math.sin(theta_rz[q])
        E += v
    return E


@pytest.mark.parametrize("cfg,prec", [(5, "c64"), (6, "c128")])
def test_config5_full_size(cfg, prec):
    """Full 50 000-term Hamiltonian at full register size, the bench launch configuration (one statevector).
    No full oracle exists at this size (parity at n = 32 is pinned by properties): theta = 0 gives the
    Z-coefficient sum, basis states give the diagonal table entry, energies are bounded by sum|c|, and a
    rotations-only circuit on all qubits matches the product-state closed form term by term (X, Y and Z on every
    qubit position, including the highest)."""
    w = make_workload(cfg)
    g = ctx_for(w, prec, 1)
    pl = w.pauli_list()
    zs = [(sum(1 << q for q, ch in enumerate(s) if ch == "Z"), c) for s, c in zip(pl, w.coeffs) if "X" not in s and "Y" not in s]
    rng = np.random.default_rng(cfg)
    xs = [0, (1 << w.n) - 1, int(rng.integers(0, 1 << w.n))]
    rows = np.zeros((len(xs), w.P))
    for b, x in enumerate(xs):
        for q in range(w.n):
            rows[b, 2 * w.n * w.D + q] = math.pi * ((x >> q) & 1)
    E = g.energy_batch(rows)
    want = [sum(c * (-1) ** bin(x & z).count("1") for z, c in zs) for x in xs]
    assert_close(prec, E, want, w.coeffs, f"cfg{cfg} basis states")
    E2 = g.energy_batch(w.params[:1])
    assert abs(E2[0]) <= np.sum(np.abs(w.coeffs))
    assert np.array_equal(E2, g.energy_batch(w.params[:1]))
    # rotations only (explicit op list), same Hamiltonian
    n = w.n
    ops = np.array([(OP_RY, q, -1, q) for q in range(n)] + [(OP_RZ, q, -1, n + q) for q in range(n)], dtype=np.int32)
    th = rng.uniform(-math.pi, math.pi, 2 * n)
    del g
    g2 = gv.Gvqe(n, ops=ops, n_params=2 * n, precision=prec)
    g2.set_hamiltonian(w.paulis, w.coeffs)
    g2.alloc_workspace(1)
    E3 = g2.energy_batch(th.reshape(1, -1))
    assert_close(prec, E3, [_product_state_energy(n, th[:n], th[n:], pl, w.coeffs)], w.coeffs, f"cfg{cfg} product state")


def test_c64_vs_c128_at_28_qubits():
    """Cross-precision agreement on the config-4 circuit (one row, 2 000-term subsample) within the c64 tolerance."""
    w = make_workload(4, M=2000, batch=1)
    E = {}
    for prec in ("c64", "c128"):
        g = ctx_for(w, prec, 1)
        E[prec] = g.energy_batch(w.params[:1])
        del g
    assert_close("c64", E["c64"], E["c128"], w.coeffs, "c64 vs c128")


@pytest.mark.parametrize("n,D,ent,topo,prec", [(14, 2, "cz", "ring", "c64"), (15, 2, "cnot", "ring", "c128"), (12, 1, "cnot", "linear", "c64")])
def test_without_product_state_prefix(orc, n, D, ent, topo, prec):
    """The first layer is normally WRITTEN as a product state; with gvqe_options.prefix = 1 the same circuit
    runs through the generic blocks from |0...0>.  Both must match the oracle (and so each other)."""
    ops = np.array(layout_ops(n, D, ent, topo, 1), dtype=np.int32)
    P = num_params(n, D, 1)
    paulis, coeffs = random_paulis(500 + n, n, 100, 5)
    th = np.random.default_rng(n).uniform(-math.pi, math.pi, (3, P))
    ref = orc.energy_batch(n, ops, th, paulis, coeffs)
    for no_prefix in (False, True):
        g = gv.Gvqe(n, layout=dict(n_layers=D, entangler=ent, topology=topo), precision=prec,
                    options=dict(prefix=1 if no_prefix else 2, tile_bits=10))
        assert ("prefix ops=0" in g.dump_schedule()) == no_prefix
        g.set_hamiltonian(paulis, coeffs)
        g.alloc_workspace(3)
        assert_close(prec, g.energy_batch(th), ref, coeffs, f"no_prefix={no_prefix}")
        assert np.max(np.abs(g.get_state(2) - orc.state(n, ops, th[2]))) < (1e-12 if prec == "c128" else 2e-5)


@pytest.mark.parametrize("prec", ["c64", "c128"])
def test_expectation_modes_agree(orc, prec):
    """The planner evaluates most community-local groups as register stages; gvqe_options.register_stages = 1 sends
    every group through the lookup / direct modes instead.  Both plans must match the oracle on the config-4 recipe
    (pooled flip masks)."""
    w = make_workload(4, n=15, M=1500, D=2, batch=3)
    ref = orc.energy_batch(w.n, w.ops, w.params, w.paulis, w.coeffs)
    for no_rs in (False, True):
        g = ctx_for(w, prec, 3, options=dict(register_stages=1 if no_rs else 0, tile_bits=11))
        assert_close(prec, g.energy_batch(w.params), ref, w.coeffs, f"no_rs={no_rs}")


@pytest.mark.parametrize("cfg,n,M,prec", [(5, 22, 5000, "c64"), (6, 18, 3000, "c128"), (6, 20, 5000, "c128")])
def test_tile_dependent_tables_over_many_index_bits(orc, cfg, n, M, prec):
    """Config-5 recipes (weight <= 6, terms across communities) shrunk to sizes the oracle finishes: their table slices have
    terms with z bits outside the tile and 6-8 index bits, so the specialised passes rebuild tables of 64-256 entries per tile
    (lane = low five index bits, register Walsh-Hadamard over the others).  Random angles, three rows, against oracle T1 (the
    full Hamiltonian; Eq. 6)."""
    w = make_workload(cfg, n=n, M=M, D=2, batch=3)
    g = ctx_for(w, prec, 3, options=dict(specialise=2))
    nb, npass, _ = g.schedule_info()
    bits = [int(x) for i in range(nb, nb + npass) for x in re.findall(r"patterns over (\d+) index bits", g.kernel_source(i)[0])]
    assert max(bits) >= 7
    E = g.energy_batch(w.params)
    ref = np.array([orc.t1_energy_of_state(w.n, orc.state(w.n, w.ops, w.params[b]), w.paulis, w.coeffs) for b in range(3)])
    assert_close(prec, E, ref, w.coeffs, f"cfg{cfg} n={n}")


# ---- schedule-specialised gate kernels (jit.cpp; "JIT-compiled once and reused") ------------------------------
@pytest.mark.parametrize("n,D,ent,topo,fr,prec,prefix", [
    (14, 2, "cnot", "ring", 1, "c64", 1), (14, 2, "cnot", "ring", 1, "c64", 2), (15, 3, "cz", "linear", 1, "c64", 1),
    (13, 2, "cz", "linear", 2, "c128", 2), (16, 2, "cnot", "ring", 1, "c128", 1), (17, 3, "cz", "ring", 2, "c64", 2),
    (14, 2, "cnot", "full", 1, "c64", 1), (15, 3, "cnot", "sca", 2, "c128", 1), (16, 3, "cnot", "pairwise", 1, "c64", 2),
    (18, 2, "cnot", "ring", 1, "c64", 0), (17, 2, "cz", "linear", 1, "c128", 0)])
def test_specialised_gate_kernels(orc, n, D, ent, topo, fr, prec, prefix):
    """gvqe_options.specialise = 2 forces the generated kernels at small sizes (by default they serve >= 20 qubits):
    energies and amplitudes against the oracle, five rows in chunks of three so that a thread block meets several
    statevectors; the generic kernels (specialise = 1) on the same inputs agree within the same tolerance."""
    ops = np.array(layout_ops(n, D, ent, topo, fr), dtype=np.int32)
    P = num_params(n, D, fr)
    paulis, coeffs = random_paulis(900 + n, n, 100, 5)
    th = np.random.default_rng(n).uniform(-math.pi, math.pi, (5, P))
    th[1, :3] = [math.pi, -math.pi, 0.0]                            # exact quarter turns: cos = 0 up to rounding
    ref = orc.energy_batch(n, ops, th, paulis, coeffs)
    # staged_io = 1: every tile through shared memory on both sides; mid_cnot = 1: every CNOT in a trailing run (the
    # default applies CNOTs on register qubits in registers and lets rotations follow them in the same stage)
    for spec, staged, mid in ((2, 0, 0), (2, 1, 0), (2, 0, 1), (1, 0, 0)):
        g = gv.Gvqe(n, layout=dict(n_layers=D, entangler=ent, topology=topo, final_rot=fr), precision=prec,
                    options=dict(specialise=spec, prefix=prefix, staged_io=staged, mid_cnot=mid))
        assert (g.kernel_source(0) is not None) == (spec == 2)
        if mid == 1 or spec == 1:
            assert " cx(" not in g.dump_schedule()
        g.set_hamiltonian(paulis, coeffs)
        g.alloc_workspace(3)
        assert_close(prec, g.energy_batch(th), ref, coeffs, f"specialise={spec} staged_io={staged} mid_cnot={mid}")
        assert np.max(np.abs(g.get_state(1) - orc.state(n, ops, th[4]))) < (1e-12 if prec == "c128" else 2e-5)


@pytest.mark.parametrize("seed", range(6))
def test_specialised_random_circuits(orc, seed):
    n = 13 + seed % 4
    prec = "c64" if seed % 2 else "c128"
    ops, P = random_ops(7100 + seed, n, 160)
    paulis, coeffs = random_paulis(8100 + seed, n, 60, 6)
    th = np.random.default_rng(seed).uniform(-math.pi, math.pi, (4, P))
    g = gv.Gvqe(n, ops=ops, n_params=P, precision=prec, options=dict(specialise=2, staged_io=seed // 3 % 2, interleave=(0, 1, 4)[seed % 3]))
    g.set_hamiltonian(paulis, coeffs)
    g.alloc_workspace(4)
    assert_close(prec, g.energy_batch(th), orc.energy_batch(n, ops, th, paulis, coeffs), coeffs, f"specialised random n={n}")
    assert np.max(np.abs(g.get_state(3) - orc.state(n, ops, th[3]))) < (1e-12 if prec == "c128" else 2e-5)


def test_generic_kernels_at_config3_size(orc):
    """From 20 qubits on the specialised kernels are the default; the generic ones stay covered at that size too."""
    w = make_workload(3)
    idx = np.arange(0, w.M, 17)
    pl = w.pauli_list()
    sub_p, sub_c = "".join(pl[i] for i in idx).encode(), w.coeffs[idx]
    psi = orc.state(w.n, w.ops, w.params[5])
    ref = orc.energy_of_state(w.n, psi, sub_p, sub_c)
    for spec in (1, 0):
        g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology), precision="c64",
                    options=dict(specialise=spec))
        assert (g.kernel_source(0) is None) == (spec == 1)
        g.set_hamiltonian(sub_p, sub_c)
        g.alloc_workspace(8)
        assert_close("c64", g.energy_batch(w.params[:8])[5:6], [ref], sub_c, f"cfg3 specialise={spec}")


def test_long_op_list_splits_blocks(orc):
    """1 500 random ops on 12 qubits: the program slice of a block outgrows its shared-memory budget and the block is
    cut into several device blocks at stage boundaries; results unchanged."""
    n = 12
    ops, P = random_ops(4242, n, 1500)
    paulis, coeffs = random_paulis(4243, n, 60, 5)
    th = np.random.default_rng(7).uniform(-math.pi, math.pi, (2, P))
    for prec in ("c128", "c64"):
        g = gv.Gvqe(n, ops=ops, n_params=P, precision=prec)
        g.set_hamiltonian(paulis, coeffs)
        g.alloc_workspace(2)
        assert g.schedule_info()[0] >= 2
        assert_close(prec, g.energy_batch(th), orc.energy_batch(n, ops, th, paulis, coeffs), coeffs, "long op list")
        assert np.max(np.abs(g.get_state(0) - orc.state(n, ops, th[0]))) < (1e-11 if prec == "c128" else 1e-4)

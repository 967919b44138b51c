"""GPU tests of what round 1 built around the hot path, all through the C ABI:

* the host-side Graph-VQE loop (gvqe_graph_vqe_minimize, NEXT-1): every energy and gradient comes from
  the CUDA kernels; checked against its step-by-step oracle, a separable closed form, the variational bound against
  the dense ground energy (n <= 8), the oracle's energy and gradient at the returned vector, and the bookkeeping;
* the read-out (gvqe_argmax, gvqe_sample, NEXT-4) against oracle/readout_oracle.py and closed forms;
* shared-prefix parameter-shift sweeps (NEXT-2): bit-identical to the plain evaluation."""
import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from paper_2607_02749_b200 import binding as gb
from workload import make_workload
from workload.generator import SplitMix64
from tests.dense_ref import dense_hamiltonian

pytestmark = pytest.mark.gpu


def ctx(w, prec="c128", in_flight=16, options=None):
    g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology, final_rot=w.final_rot),
                precision=prec, options=options)
    g.set_hamiltonian(w.paulis, w.coeffs)
    g.alloc_workspace(in_flight)
    return g


def test_separable_closed_form():
    """D = 0 (one RY per qubit), H = sum_q a_q Z_q: E(theta) = sum_q a_q cos(theta_q), minimum -sum |a_q|.  Every qubit
    its own block and no global phase (the paper's no_Global ablation): the fused block solutions are the optimum."""
    n = 6
    a = np.array([1.0, -0.5, 2.0, 0.25, -1.5, 0.75])
    paulis = "".join("".join("Z" if j == q else "I" for j in range(n)) for q in range(n))
    g = gv.Gvqe(n, layout=dict(n_layers=0, entangler="cz", topology="linear"), precision="c128")
    g.set_hamiltonian(paulis, a)
    g.alloc_workspace(16)
    r = SplitMix64(7)
    theta0 = np.array([(2 * r.uniform() - 1) * 2.5 for _ in range(n)])
    theta, res, hist = g.graph_vqe_minimize(theta0, list(range(n)), max_epochs=4, global_iters=0, f_tol=1e-14)
    assert res["n_blocks"] == n
    assert abs(res["E_best"] + np.sum(np.abs(a))) < 1e-9
    assert abs(hist[0] - float(np.sum(a * np.cos(theta0)))) < 1e-12
    assert np.all(np.abs(np.cos(theta) + np.sign(a)) < 1e-8)


@pytest.mark.parametrize("use_global", [True, False])
def test_variational_bound_and_oracle_agreement(orc, use_global):
    """cfg 2 recipe shrunk to 8 qubits (2 communities, 60 terms, 15 % X/Y), 2 layers, c128."""
    w = make_workload(2, n=8, M=60, D=2, batch=1)
    g = ctx(w)
    W = g.interaction_graph()
    lab, K, Q = gb.louvain(W)
    lab, K = gb.merge_small_blocks(W, lab, 2)
    assert K >= 2
    E0 = g.energy_batch(w.theta)[0]
    theta, res, hist = g.graph_vqe_minimize(w.theta, lab, max_epochs=6, block_iters=40,
                                            global_iters=60 if use_global else 0, f_tol=1e-12)
    H = dense_hamiltonian(w.n, w.pauli_list(), w.coeffs)
    e_min = float(np.linalg.eigvalsh(H)[0])
    assert res["E_best"] >= e_min - 1e-9                      # variational principle
    assert res["E_best"] < E0 - 0.1 * abs(E0 - e_min)         # and real progress towards it
    assert abs(hist[0] - E0) < 1e-12 and len(hist) == res["epochs"] + 1
    assert abs(res["E_best"] - min(hist)) < 1e-12
    # the returned vector really has the returned energy (oracle T0), and it is a stationary point of what was
    # optimised last: all parameters after a global phase
    E_o = orc.energy_batch(w.n, w.ops, theta.reshape(1, -1), w.paulis, w.coeffs)[0]
    assert abs(E_o - res["E_best"]) <= 1e-10 * abs(E_o) + 1e-12 * np.sum(np.abs(w.coeffs))
    assert res["energy_evals"] > 0 and res["steps"] > 0
    if use_global:
        dE, _ = orc.param_shift_grad(w.n, w.ops, theta, np.ones(w.P, np.uint8), w.paulis, w.coeffs)
        assert np.max(np.abs(dE)) < 5e-2 * max(1.0, np.max(np.abs(w.coeffs)))


def test_cobyla_separable_closed_form():
    """PAPER.md:221 "derivative-free (COBYLA)": the same separable problem with optimizer = "cobyla"; every block is one
    parameter, the fused block solutions are the optimum -sum |a_q| (rho_end = tol = 1e-6 bounds the distance to it)."""
    n = 6
    a = np.array([1.0, -0.5, 2.0, 0.25, -1.5, 0.75])
    paulis = "".join("".join("Z" if j == q else "I" for j in range(n)) for q in range(n))
    g = gv.Gvqe(n, layout=dict(n_layers=0, entangler="cz", topology="linear"), precision="c128")
    g.set_hamiltonian(paulis, a)
    g.alloc_workspace(16)
    r = SplitMix64(7)
    theta0 = np.array([(2 * r.uniform() - 1) * 2.5 for _ in range(n)])
    theta, res, hist = g.graph_vqe_minimize(theta0, list(range(n)), max_epochs=2, block_iters=200, global_iters=0,
                                            optimizer="cobyla", tol=1e-6)
    assert res["n_blocks"] == n and res["steps"] > 0
    assert abs(res["E_best"] + np.sum(np.abs(a))) < 1e-9
    assert np.all(np.abs(np.cos(theta) + np.sign(a)) < 1e-9)
    # the whole vector at once (global phase only) reaches it too
    theta, res, hist = g.graph_vqe_minimize(theta0, [0] * n, max_epochs=1, block_iters=0, global_iters=2000,
                                            optimizer="cobyla", tol=1e-5, patience=10 ** 6)
    assert abs(res["E_best"] + np.sum(np.abs(a))) < 1e-7


def test_cobyla_variational_bound_and_oracle_agreement(orc):
    """cfg 2 recipe shrunk to 8 qubits, 2 layers, c128, optimizer = "cobyla" in both phases: energies go down, stay above
    the dense ground energy, and the returned vector has the returned energy (oracle T0).  No gradients are evaluated:
    the evaluation count is the simplex sizes plus one per step."""
    w = make_workload(2, n=8, M=60, D=2, batch=1)
    g = ctx(w, in_flight=64)
    lab = [0, 0, 0, 0, 1, 1, 1, 1]
    E0 = g.energy_batch(w.theta)[0]
    theta, res, hist = g.graph_vqe_minimize(w.theta, lab, max_epochs=2, block_iters=150, global_iters=300,
                                            optimizer="cobyla", tol=1e-4, rho_beg=0.5)
    H = dense_hamiltonian(w.n, w.pauli_list(), w.coeffs)
    e_min = float(np.linalg.eigvalsh(H)[0])
    assert res["E_best"] >= e_min - 1e-9
    assert res["E_best"] < E0 - 0.1 * abs(E0 - e_min)
    assert abs(hist[0] - E0) < 1e-12 and abs(res["E_best"] - min(hist)) < 1e-12
    E_o = orc.energy_batch(w.n, w.ops, theta.reshape(1, -1), w.paulis, w.coeffs)[0]
    assert abs(E_o - res["E_best"]) <= 1e-10 * abs(E_o) + 1e-12 * np.sum(np.abs(w.coeffs))
    m0, m1 = g.block_param_mask(lab, 0), g.block_param_mask(lab, 1)
    per_epoch_max = (int(m0.sum()) + 1 + 150) + (int(m1.sum()) + 1 + 150) + (w.P + 1 + 300)
    assert 1 + res["epochs"] <= res["energy_evals"] <= 1 + res["epochs"] * per_epoch_max
    with pytest.raises(gv.GvqeError):
        g.graph_vqe_minimize(w.theta, lab, optimizer="cobyla", rho_beg=-1.0)


def test_block_phase_touches_only_block_parameters():
    """One epoch, one block iteration budget, no global phase, a partition with an empty complement: parameters of
    qubits outside every optimised block keep their start values (Eq. 11: theta outside B_i is constant)."""
    w = make_workload(1, n=6, M=30, D=1, batch=1)
    g = ctx(w)
    lab = [0, 0, 0, 1, 1, 1]
    theta, res, hist = g.graph_vqe_minimize(w.theta, lab, max_epochs=1, block_iters=3, global_iters=0)
    m0, m1 = g.block_param_mask(lab, 0), g.block_param_mask(lab, 1)
    assert np.array_equal(m0 + m1, np.ones(w.P, np.uint8))
    # block_iters = 0 and global_iters = 0: nothing moves
    theta2, res2, hist2 = g.graph_vqe_minimize(w.theta, lab, max_epochs=2, block_iters=0, global_iters=0, epoch_patience=1)
    assert np.array_equal(theta2, w.theta) and res2["stop_reason"] == 1 and res2["epochs"] == 1
    assert res["E_best"] <= hist[0]


def test_minimize_argument_checks():
    w = make_workload(1, n=6, M=10, D=1, batch=1)
    g = ctx(w)
    with pytest.raises(gv.GvqeError):
        g.graph_vqe_minimize(w.theta, [0] * 6, max_epochs=0)
    with pytest.raises(gv.GvqeError):
        g.graph_vqe_minimize(w.theta, [0, 0, 0, 0, 0, -1])
    with pytest.raises(gv.GvqeError):
        g.graph_vqe_minimize(w.theta, [0] * 6, tol=0.0)


@pytest.mark.parametrize("n,D,budget", [(6, 1, (3, 4, 5)), (8, 2, (2, 3, 3))])
def test_loop_follows_the_step_by_step_oracle(orc, n, D, budget):
    """Same start vector, same blocks, same budgets: the library's epoch loop (energies from the kernels, c128) and
    oracle/driver_oracle.py (energies from oracle T0) take the same steps -- same epoch count, step count and stop
    reason, histories and final parameters equal up to the amplification of the 1e-13 energy differences."""
    from oracle import driver_oracle as do
    epochs, bi, gi = budget
    w = make_workload(2, n=n, M=50, D=D, batch=1)
    g = ctx(w)
    W = g.interaction_graph()
    lab, K, _ = gb.louvain(W)
    lab, K = gb.merge_small_blocks(W, lab, 2)
    theta, res, hist = g.graph_vqe_minimize(w.theta, lab, max_epochs=epochs, block_iters=bi, global_iters=gi, f_tol=1e-12)
    energy = lambda rows: orc.energy_batch(w.n, w.ops, np.ascontiguousarray(rows), w.paulis, w.coeffs)
    masks = [g.block_param_mask(lab, b) for b in range(K)]
    th_o, E_o, hist_o, ep_o, steps_o, reason_o = do.graph_vqe_minimize(
        energy, w.theta, masks, max_epochs=epochs, block_iters=bi, global_iters=gi, f_tol=1e-12)
    assert (res["epochs"], res["steps"], res["stop_reason"], res["n_blocks"]) == (ep_o, steps_o, reason_o, K)
    scale = np.sum(np.abs(w.coeffs))
    assert np.max(np.abs(hist - hist_o)) < 1e-8 * scale
    assert abs(res["E_best"] - E_o) < 1e-8 * scale
    assert np.max(np.abs(theta - th_o)) < 1e-6


# ---- read-out (gvqe_argmax) -------------------------------------------------------------------
def _check_argmax(x, p, p_ref, prec):
    """x is a valid most-probable index of the oracle's distribution up to the precision of the stored amplitudes,
    identical to the oracle's when the gap to the runner-up is larger than that."""
    tol = 1e-12 if prec == "c128" else 2e-5 * float(p_ref.max()) + 1e-9
    assert p_ref[x] >= p_ref.max() - tol
    assert abs(p - p_ref[x]) <= tol
    order = np.sort(p_ref)
    if order[-1] - order[-2] > 2 * tol:
        assert x == int(np.argmax(p_ref))


@pytest.mark.parametrize("cfg,n,D,prec", [(1, 10, 3, "c128"), (2, 13, 2, "c128"), (3, 15, 2, "c64"), (4, 14, 2, "c64"),
                                          (2, 3, 1, "c128"), (3, 1, 1, "c64")])
def test_argmax_vs_oracle(orc, cfg, n, D, prec):
    from oracle import readout_oracle as ro
    w = make_workload(cfg, n=n, M=40, D=D, batch=3)
    g = ctx(w, prec, in_flight=3)
    g.energy_batch(w.params)
    for slot in range(3):
        p_ref = ro.probabilities(w.n, w.ops, w.params[slot])
        x, p = g.argmax(slot)
        _check_argmax(x, p, p_ref, prec)
        psi = g.get_state(slot)                                    # the kernel's own decision on its own amplitudes
        pk = (psi.real * psi.real + psi.imag * psi.imag)
        assert x == int(np.argmax(pk)) and p == float(pk[x])


@pytest.mark.parametrize("n,prec", [(12, "c128"), (26, "c64"), (25, "c128")])
def test_argmax_product_state_closed_form(n, prec):
    """Rotations only: bit q of x* is set exactly when sin^2(theta_q/2) > cos^2(theta_q/2) -- valid at sizes no host
    evaluator reaches; the state spans many grid-stride rounds of the sweep."""
    r = SplitMix64(100 + n)
    theta = np.array([(2 * r.uniform() - 1) * 3.0 for _ in range(n)])
    theta[np.abs(np.abs(theta) - np.pi / 2) < 0.05] += 0.2       # keep every qubit's decision away from the tie
    g = gv.Gvqe(n, layout=dict(n_layers=0, entangler="cz", topology="linear"), precision=prec)
    g.set_hamiltonian("Z" + "I" * (n - 1), [1.0])
    g.alloc_workspace(1)
    g.energy_batch(theta)
    x, p = g.argmax(0)
    s2, c2 = np.sin(theta / 2) ** 2, np.cos(theta / 2) ** 2
    assert x == sum(1 << q for q in range(n) if s2[q] > c2[q])
    assert abs(p - np.prod(np.maximum(s2, c2))) <= (1e-12 if prec == "c128" else 1e-5) * p
    # basis state: RY(pi) on the bits of a pattern that includes the highest qubit
    target = (1 << (n - 1)) | 0b1011
    th = np.array([np.pi if (target >> q) & 1 else 0.0 for q in range(n)])
    g.energy_batch(th)
    x, p = g.argmax(0)
    assert x == target and abs(p - 1.0) < 1e-5
    g.energy_batch(np.zeros(n))                                    # |0...0>: every other probability is an exact 0
    assert g.argmax(0) == (0, 1.0)
    with pytest.raises(gv.GvqeError):
        g.argmax(1)


# ---- shot sampling (gvqe_sample) ----------------------------------------------------------------
@pytest.mark.parametrize("cfg,n,D,prec", [(1, 10, 2, "c128"), (2, 14, 2, "c128"), (3, 15, 2, "c64"), (4, 13, 2, "c64"),
                                          (2, 2, 1, "c128")])
def test_sample_vs_oracle(orc, cfg, n, D, prec):
    """Every shot is a valid inverse of the oracle's cumulative distribution (within the amplitude precision at the
    boundaries); almost all shots are identical to the oracle's."""
    from oracle import readout_oracle as ro
    w = make_workload(cfg, n=n, M=30, D=D, batch=2)
    g = ctx(w, prec, in_flight=2)
    g.energy_batch(w.params)
    r = SplitMix64(900 + n)
    u = np.array([r.uniform() for _ in range(8192)])             # the paper's shot count
    u[:3] = [0.0, 0.5, 1.0 - 2.0 ** -53]
    for slot in range(2):
        x, Z = g.sample(u, slot)
        x_o, Z_o = ro.sample(w.n, w.ops, w.params[slot], u)
        F = np.concatenate([[0.0], np.cumsum(ro.probabilities(w.n, w.ops, w.params[slot]))])
        eps = 1e-12 if prec == "c128" else 1e-5
        assert abs(Z - Z_o) <= eps
        xi = x.astype(np.int64)
        assert xi.min() >= 0 and xi.max() < (1 << w.n)
        t = u * Z_o
        assert np.all(F[xi] - eps <= t) and np.all(t <= F[xi + 1] + eps)
        assert np.mean(x == x_o) > (0.999 if prec == "c128" else 0.98)
        x2, _ = g.sample(u, slot)
        assert np.array_equal(x, x2)                              # deterministic


@pytest.mark.parametrize("n,prec", [(12, "c128"), (24, "c64")])
def test_sample_quantiles_product_state(n, prec):
    """Stratified uniforms: outcome counts equal S p(x) up to +-1 (closed-form p of a rotations-only circuit); at 24
    qubits the shots are checked through their marginals: bit q is set in a fraction sin^2(theta_q/2) of the shots."""
    r = SplitMix64(300 + n)
    theta = np.array([(2 * r.uniform() - 1) * 3.0 for _ in range(n)])
    g = gv.Gvqe(n, layout=dict(n_layers=0, entangler="cz", topology="linear"), precision=prec)
    g.set_hamiltonian("Z" + "I" * (n - 1), [1.0])
    g.alloc_workspace(1)
    g.energy_batch(theta)
    S = 65536
    x, Z = g.sample((np.arange(S) + 0.5) / S, 0)
    assert abs(Z - 1.0) < (1e-12 if prec == "c128" else 1e-5)
    xi = x.astype(np.int64)
    assert np.all(np.diff(xi) >= 0)
    s2, c2 = np.sin(theta / 2) ** 2, np.cos(theta / 2) ** 2
    if n <= 12:
        p = np.ones(1 << n)
        for q in range(n):
            p *= np.where((np.arange(1 << n) >> q) & 1, s2[q], c2[q])
        counts = np.bincount(xi, minlength=1 << n)
        assert np.all(np.abs(counts - S * p) <= 1.0 + 1e-6)
    for q in range(n):
        assert abs(np.mean((xi >> q) & 1) - s2[q]) < 2e-3
    with pytest.raises(gv.GvqeError):
        g.sample([1.0], 0)
    with pytest.raises(gv.GvqeError):
        g.sample(np.zeros(65537), 0)
    assert len(g.sample([], 0)[0]) == 0


# ---- finite-shot energy estimate (gvqe_energy_shots) ----------------------------
@pytest.mark.parametrize("cfg,n,D,prec", [(2, 9, 2, "c128"), (4, 12, 2, "c64"), (3, 14, 1, "c128"), (4, 15, 2, "c64")])
def test_energy_shots_vs_oracle(orc, cfg, n, D, prec):
    """Same uniforms, same settings: the library's shots are those of the oracle up to ties at cumulative boundaries, so every
    term mean agrees within the fraction of shots that can differ, and the estimate approaches the exact energy."""
    from oracle import readout_oracle as ro
    w = make_workload(cfg, n=n, M=120, D=D, batch=2)
    g = ctx(w, prec, in_flight=2)
    g.energy_batch(w.params[:2])
    pl = w.pauli_list()
    settings, got = ro.measurement_groups(w.n, pl)
    ns, got_lib = g.measurement_settings(w.M)
    assert ns == len(settings) and got_lib.tolist() == got            # integer side: exact
    S = 2000
    u = np.random.default_rng(n).uniform(size=(ns, S))
    E_ref, means_ref, _ = ro.energy_shots(w.n, w.ops, w.params[1], pl, w.coeffs, u)
    E, means = g.energy_shots(u, w.M, slot=1)
    slack = (3.0 if prec == "c64" else 0.0) / S                        # c64: a few shots may fall on the other side of a boundary
    assert np.max(np.abs(means - means_ref)) <= 2.0 * slack + 1e-12
    assert abs(E - E_ref) <= 2.0 * slack * np.sum(np.abs(w.coeffs)) + 1e-9
    exact = orc.energy_batch(w.n, w.ops, w.params[1:2], w.paulis, w.coeffs)[0]
    per_setting = np.zeros(ns)                                         # terms of one setting share shots: fully correlated
    for k in range(w.M):
        per_setting[got[k]] += abs(w.coeffs[k])
    assert abs(E - exact) <= 6.0 * np.sqrt(np.sum(per_setting ** 2) / S)
    assert np.array_equal(g.energy_batch(w.params[:2]), g.energy_batch(w.params[:2]))   # the slots were not disturbed for reuse
    with pytest.raises(gv.GvqeError):
        g.energy_shots(np.ones((ns, 4)), w.M, slot=0)                  # u = 1.0 is outside [0, 1)


def test_energy_shots_one_qubit_closed_form():
    """RY(theta)|0>, H = 2 X + 0.5 Z: stratified uniforms give each mean within 1/S of sin(theta) and cos(theta)."""
    th, S = 0.7, 1000
    g = gv.Gvqe(1, ops=np.array([[0, 0, -1, 0]], dtype=np.int32), n_params=1, precision="c128")
    g.set_hamiltonian(b"X" + b"Z", [2.0, 0.5])
    g.alloc_workspace(2)
    g.energy_batch(np.array([[th], [0.0]]))
    u = np.tile((np.arange(S) + 0.5) / S, (2, 1))
    E, means = g.energy_shots(u, 2, slot=0)
    assert abs(means[0] - np.sin(th)) <= 2.0 / S and abs(means[1] - np.cos(th)) <= 2.0 / S
    assert abs(E - (2.0 * np.sin(th) + 0.5 * np.cos(th))) <= 5.0 / S
    g1 = gv.Gvqe(1, ops=np.array([[0, 0, -1, 0]], dtype=np.int32), n_params=1, precision="c128")
    g1.set_hamiltonian(b"X", [1.0])
    g1.alloc_workspace(1)
    g1.energy_batch(np.array([[th]]))
    with pytest.raises(gv.GvqeError):                                  # one statevector in flight: no scratch slot
        g1.energy_shots(u[:1], 1, slot=0)


# ---- shared-prefix parameter-shift sweeps ---------------------------------------------------------
@pytest.mark.parametrize("cfg,n,D,prec,in_flight,prefix,spec", [
    (1, 10, 3, "c128", 16, 0, 0), (2, 16, 4, "c128", 8, 0, 0), (4, 15, 3, "c64", 8, 2, 0), (4, 16, 2, "c128", 3, 1, 0),
    (3, 17, 3, "c64", 2, 0, 0), (4, 14, 2, "c64", 1, 0, 0), (2, 4, 2, "c128", 5, 0, 0),
    (4, 15, 3, "c64", 8, 2, 2), (4, 16, 2, "c128", 3, 1, 2), (3, 17, 3, "c64", 4, 0, 2)])
def test_shared_prefix_gradient_is_bit_identical(orc, cfg, n, D, prec, in_flight, prefix, spec):
    """gvqe_param_shift_grad with snapshots of the base state at the block boundaries returns exactly the numbers of
    the plain evaluation of all 2|mask|+1 rows (each row sees the same kernels on the same data), with and without
    the product-state prefix (gvqe_options.prefix), for chunked groups and for a one-slot workspace (fallback), with the
    generic and with the schedule-specialised gate kernels (gvqe_options.specialise); and both match the oracle."""
    w = make_workload(cfg, n=n, M=60, D=D, batch=1)
    r = SplitMix64(77 + n)
    mask = np.array([1 if r.uniform() < 0.4 else 0 for _ in range(w.P)], dtype=np.uint8)
    mask[0] = mask[w.P - 1] = 1                                   # first layer (prefix) and the last rotation layer
    g = ctx(w, prec, in_flight=in_flight, options=dict(prefix=prefix, shared_prefix=2, specialise=spec))
    l0 = g.launch_count()
    dE, E0 = g.param_shift_grad(w.theta, mask)
    l_shared = g.launch_count() - l0
    del g
    g = ctx(w, prec, in_flight=in_flight, options=dict(prefix=prefix, shared_prefix=1, specialise=spec))
    l0 = g.launch_count()
    dE_plain, E0_plain = g.param_shift_grad(w.theta, mask)
    l_plain = g.launch_count() - l0
    assert E0 == E0_plain and np.array_equal(dE, dE_plain)
    assert np.all(dE[mask == 0] == 0.0)
    assert l_shared > 0 and l_plain > 0
    dE_o, E0_o = orc.param_shift_grad(w.n, w.ops, w.theta, mask, w.paulis, w.coeffs)
    scale = np.sum(np.abs(w.coeffs))
    tol_ = 1e-10 * scale if prec == "c128" else 2e-5 * scale
    assert abs(E0 - E0_o) <= tol_ and np.max(np.abs(dE - dE_o)) <= tol_


def test_profile_read_launches_lists_every_kernel_of_a_chunk():
    """gvqe_profile_enable / gvqe_profile_read_launches (what bench.py's per-kernel rooflines are measured with): one
    entry per launch of an energy chunk in execution order -- prefix kernel (if any), gate blocks, expectation passes --
    mean within [min, max], and their sums stay below the class totals of gvqe_profile_read."""
    w = make_workload(3, n=20, M=200, D=2, batch=4)
    g = ctx(w, "c64", in_flight=4)
    g.energy_batch(w.params)
    g.profile_enable(True)
    for _ in range(3):
        g.energy_batch(w.params)
    mean, lo, hi = g.profile_read_launches()
    tot = g.profile_read()
    n_gate, n_pass, _ = g.schedule_info()
    assert len(mean) == n_gate + n_pass and tot["chunks"] == 3
    assert np.all(lo <= mean + 1e-9) and np.all(mean <= hi + 1e-9) and np.all(lo > 0.0)
    # the class totals bracket a whole phase (launch gaps included), the per-launch figures only the kernels
    assert 0.5 * tot["gate_ms"] <= mean[:n_gate].sum() * 3 <= 1.02 * tot["gate_ms"]
    assert 0.5 * tot["expect_ms"] <= mean[n_gate:].sum() * 3 <= 1.02 * tot["expect_ms"]
    g.profile_enable(False)

"""CPU tests of the Hamiltonian-aware partitioning (Eq. 9 and 10).

First the oracle (oracle/graph_oracle.py) is pinned to things other than itself: a hand-computed Eq. 9 example,
closed forms of Eq. 10, brute force over all set partitions of tiny graphs, planted communities.  Then the library's
host C++ (gvqe_interaction_graph / gvqe_modularity / gvqe_louvain / gvqe_merge_small_blocks / gvqe_block_param_mask)
is compared with the oracle: weights and Q to rounding, partitions and masks exactly."""
import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from paper_2607_02749_b200 import binding as gb
from oracle import graph_oracle as go
from workload import make_workload, CONFIGS
from workload.generator import SplitMix64, community_param_mask


def set_partitions(n):
    """All set partitions of range(n) as restricted-growth label lists."""
    def rec(prefix, k):
        if len(prefix) == n:
            yield list(prefix)
            return
        for l in range(k + 1):
            prefix.append(l)
            yield from rec(prefix, max(k, l + 1))
            prefix.pop()
    yield from rec([], 0)


def cliques(sizes, w_in=1.0, w_out=0.0):
    n = sum(sizes)
    lab = [c for c, s in enumerate(sizes) for _ in range(s)]
    w = np.zeros((n, n))
    for i in range(n):
        for j in range(n):
            if i != j:
                w[i, j] = w_in if lab[i] == lab[j] else w_out
    return w, lab


def random_graph(seed, n, density=0.6):
    r = SplitMix64(seed)
    w = np.zeros((n, n))
    for i in range(n):
        for j in range(i + 1, n):
            if r.uniform() < density:
                w[i, j] = w[j, i] = 0.1 + r.uniform()
    return w


# ---- pins of the oracle ---------------------------------------------------------------------------------------
def test_eq9_hand_example():
    """Three terms on 4 qubits, weights added by hand from Eq. 9."""
    paulis = ["XZII", "IZYI", "ZIIX", "IIII", "IXII"]      # character j acts on qubit j
    coeffs = [-2.0, 0.5, 3.0, 7.0, -1.0]                    # identity and weight-1 terms make no edge
    w = go.interaction_graph(4, paulis, coeffs)
    expect = np.zeros((4, 4))
    expect[0, 1] = expect[1, 0] = 2.0
    expect[1, 2] = expect[2, 1] = 0.5
    expect[0, 3] = expect[3, 0] = 3.0
    assert np.array_equal(w, expect)


def test_eq10_closed_forms():
    """r disjoint equal cliques, each its own block: Q = 1 - 1/r.  One block: Q = 1 - gamma.  Singletons:
    Q = -sum k_i^2 / (2m)^2.  Two triangles joined by one edge, split at the bridge: Q = 5/14 (textbook value:
    2 * (6/14 - (7/14)^2))."""
    for r in (2, 3, 5):
        w, lab = cliques([4] * r)
        assert abs(go.modularity(w, lab) - (1.0 - 1.0 / r)) < 1e-14
    w = random_graph(3, 9)
    assert abs(go.modularity(w, [0] * 9)) < 1e-14
    assert abs(go.modularity(w, [0] * 9, gamma=0.3) - 0.7) < 1e-14
    k, two_m = w.sum(axis=1), w.sum()
    assert abs(go.modularity(w, list(range(9))) + np.sum(k * k) / two_m ** 2) < 1e-14
    w = np.zeros((6, 6))
    for a, b in [(0, 1), (1, 2), (0, 2), (3, 4), (4, 5), (3, 5), (2, 3)]:
        w[a, b] = w[b, a] = 1.0
    assert abs(go.modularity(w, [0, 0, 0, 1, 1, 1]) - 5.0 / 14.0) < 1e-14
    assert go.modularity(np.zeros((3, 3)), [0, 1, 2]) == 0.0


@pytest.mark.parametrize("seed", range(6))
def test_louvain_vs_brute_force(seed):
    """n = 7: Q of every one of the 877 set partitions; Louvain's Q can never exceed the maximum, and no single-node
    move improves its result (local optimality of phase 1 on the final partition's aggregate is implied by stopping)."""
    w = random_graph(100 + seed, 7)
    q_best = max(go.modularity(w, p) for p in set_partitions(7))
    lab, K = go.louvain(w)
    q = go.modularity(w, lab)
    assert q <= q_best + 1e-12
    assert q >= 0.0 and K == max(lab) + 1 and lab[0] == 0
    assert q >= 0.75 * q_best      # heuristic, but on 7 nodes it is never far off


def test_louvain_planted_is_optimal():
    """Cliques with weak links between them: brute force says the planted partition is the optimum, Louvain finds it."""
    w, planted = cliques([3, 2, 2], w_in=1.0, w_out=0.05)
    q_all = {tuple(p): go.modularity(w, p) for p in set_partitions(7)}
    best = max(q_all, key=q_all.get)
    assert list(best) == planted
    lab, K = go.louvain(w)
    assert lab == planted and K == 3
    lab, K = go.louvain(np.zeros((5, 5)))
    assert lab == [0, 1, 2, 3, 4] and K == 5
    # resolution: gamma -> 0 puts every connected node into one block
    lab, K = go.louvain(w, gamma=0.0)
    assert K == 1


def test_merge_small_blocks_rules():
    w = np.zeros((6, 6))
    def e(a, b, v):
        w[a, b] = w[b, a] = v
    e(0, 1, 1.0); e(2, 3, 1.0); e(4, 0, 0.2); e(4, 2, 0.7); e(5, 1, 0.1)
    lab, K = go.merge_small_blocks(w, [0, 0, 1, 1, 2, 3], 2)
    # blocks 2 = {4} and 3 = {5} are too small: {4} (lowest label first) joins {2,3} (0.7 > 0.2), then {5} joins {0,1}
    assert lab == [0, 0, 1, 1, 1, 0] and K == 2
    lab, K = go.merge_small_blocks(w, [0, 0, 1, 1, 2, 3], 1)
    assert lab == [0, 0, 1, 1, 2, 3] and K == 4
    lab, K = go.merge_small_blocks(w, [0, 0, 1, 1, 2, 3], 7)     # nothing can reach 7: everything ends in one block
    assert K == 1 and lab == [0] * 6
    # sizes are conserved, labels are contiguous
    lab, K = go.merge_small_blocks(random_graph(5, 9), [0, 1, 2, 3, 4, 5, 6, 7, 8], 3)
    assert sorted(set(lab)) == list(range(K)) and min(lab.count(c) for c in range(K)) >= 3


def test_block_param_mask_counts():
    """cfg 2: one community of 4 qubits owns 4 * (2*4 + 1) = 36 parameters; masks of all blocks
    partition the parameter set; equals the workload module's own mask."""
    w = make_workload(2, M=10)
    comm = [c for c, qs in enumerate(w.communities) for _ in qs]
    masks = [go.block_param_mask(w.ops, w.P, comm, b) for b in range(4)]
    assert all(int(m.sum()) == 36 for m in masks)
    assert np.array_equal(np.sum(masks, axis=0), np.ones(w.P))
    assert np.array_equal(masks[0], community_param_mask(w.n, w.D, w.final_rot, w.communities[0]))


# ---- the library against the oracle -----------------------------------------------------------------------------
def lib_ctx(w):
    g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology, final_rot=w.final_rot),
                precision="c128")
    g.set_hamiltonian(w.paulis, w.coeffs)
    return g


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_library_graph_and_louvain_recover_planted_communities(cfg):
    """Eq. 9 weights of the BASELINE Hamiltonians (full term count, 1-layer circuit): library = oracle to rounding;
    Louvain (library and oracle) returns the same partition, and it is the planted one (SURVEY 8(f) check)."""
    w = make_workload(cfg, D=1, batch=1)
    g = lib_ctx(w)
    W = g.interaction_graph()
    Wo = go.interaction_graph(w.n, w.pauli_list(), w.coeffs)
    assert np.allclose(W, Wo, rtol=1e-13, atol=0.0) and np.array_equal(W, W.T) and not W.diagonal().any()
    lab, K, Q = gb.louvain(W)
    lab_o, K_o = go.louvain(Wo)
    assert list(lab) == lab_o and K == K_o
    assert abs(Q - go.modularity(Wo, lab_o)) < 1e-12
    planted = [c for c, qs in enumerate(w.communities) for _ in qs]
    assert list(lab) == planted
    for b in range(K):
        assert np.array_equal(g.block_param_mask(lab, b), go.block_param_mask(w.ops, w.P, lab_o, b))


@pytest.mark.parametrize("seed", range(8))
def test_library_louvain_random_graphs(seed):
    n = 5 + 3 * seed
    W = random_graph(500 + seed, n, density=0.35)
    for gamma in (1.0, 0.5, 1.7):
        lab, K, Q = gb.louvain(W, gamma)
        lab_o, K_o = go.louvain(W, gamma)
        assert list(lab) == lab_o and K == K_o
        assert abs(Q - go.modularity(W, lab_o, gamma)) < 1e-12
        assert abs(gb.modularity(W, lab, gamma) - Q) < 1e-15
    for s_min in (1, 2, 4, n + 1):
        start = [i // 2 if i % 3 else i for i in range(n)]
        m, Km = gb.merge_small_blocks(W, start, s_min)
        m_o, Km_o = go.merge_small_blocks(W, start, s_min)
        assert list(m) == m_o and Km == Km_o


def test_library_graph_argument_checks():
    W = random_graph(1, 4)
    bad = W.copy(); bad[0, 1] += 1.0
    with pytest.raises(gv.GvqeError):
        gb.louvain(bad)                      # not symmetric
    with pytest.raises(gv.GvqeError):
        gb.louvain(-W)                       # negative weights
    with pytest.raises(gv.GvqeError):
        gb.modularity(W, [0, -1, 0, 0])
    g = gv.Gvqe(4, layout=dict(n_layers=1, entangler="cz", topology="linear"), precision="c128")
    with pytest.raises(gv.GvqeError):
        g.interaction_graph()                # no Hamiltonian yet


# ---- pins of the epoch-loop oracle (oracle/driver_oracle.py) ----------------------------------------------------------
def test_driver_oracle_eq14_by_hand():
    from oracle import driver_oracle as do
    hist = [5.0, 3.0, 2.5, 2.4, 2.4, 2.39]
    assert do.delta_max(hist, 40) == 2.0                       # whole history
    assert abs(do.delta_max(hist, 3) - 0.1) < 1e-15            # last three differences: 0.1, 0.0, 0.01
    assert abs(do.delta_max(hist, 1) - 0.01) < 1e-15
    assert do.delta_max([1.0], 40) == 0.0


def test_driver_oracle_parameter_shift_is_exact_for_sinusoids():
    """Eq. 13 is exact for E = a cos(theta - b) + c in every coordinate (what a rotation gate gives)."""
    from oracle import driver_oracle as do
    a, b = np.array([1.0, -2.0, 0.5]), np.array([0.3, -1.0, 2.0])
    energy = lambda rows: np.sum(a * np.cos(rows - b), axis=1) + 4.0
    th = np.array([0.7, -0.2, 1.9])
    E, g = do.param_shift_grad(energy, th, [0, 2])
    assert abs(E - energy(th.reshape(1, -1))[0]) < 1e-15
    assert np.allclose(g, (-a * np.sin(th - b))[[0, 2]], atol=1e-14)


def test_driver_oracle_separable_minimum_and_frozen_coordinates():
    """min of sum a_q cos(theta_q) is -sum |a_q|; with one block left out its coordinates never move (Eq. 11)."""
    from oracle import driver_oracle as do
    a = np.array([1.0, -0.5, 2.0, 0.25])
    energy = lambda rows: np.sum(a * np.cos(rows), axis=1)
    th0 = np.array([0.4, 1.1, -2.0, 0.9])
    masks = [np.array([1, 1, 0, 0], np.uint8), np.array([0, 0, 1, 0], np.uint8)]
    th, E, hist, epochs, steps, reason = do.graph_vqe_minimize(energy, th0, masks, max_epochs=5, global_iters=0, f_tol=1e-14)
    assert th[3] == th0[3]
    assert abs(E - (-1.0 - 0.5 - 2.0 + 0.25 * np.cos(0.9))) < 1e-9
    assert hist[0] == energy(th0.reshape(1, -1))[0] and abs(min(hist) - E) < 1e-15
    assert all(hist[i + 1] <= hist[i] + 1e-12 for i in range(len(hist) - 1))
    th, E, *_ = do.graph_vqe_minimize(energy, th0, masks, max_epochs=3, global_iters=30, f_tol=1e-14)
    assert abs(E + np.sum(np.abs(a))) < 1e-9                   # the global phase reaches the frozen coordinate too
    # nothing to do: zero budgets stop by epoch patience after exactly epoch_patience epochs
    th, E, hist, epochs, steps, reason = do.graph_vqe_minimize(energy, th0, masks, max_epochs=9, block_iters=0,
                                                               global_iters=0, epoch_patience=2)
    assert np.array_equal(th, th0) and epochs == 2 and reason == 1 and steps == 0


def test_driver_oracle_search_direction_is_bfgs():
    """The two-loop recursion must give d = -H_k g with H_k the dense BFGS inverse-Hessian update
    H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T applied to the stored pairs, oldest first, from
    H0 = (s.y / y.y) I of the newest pair (Nocedal & Wright, Alg. 7.4 / Eq. 6.17).  A sign or ordering slip in the
    recursion fails this; steepest descent (what the restart falls back to) fails it too."""
    from oracle import driver_oracle as do
    rng = np.random.default_rng(11)
    for dim, m in ((3, 1), (4, 2), (4, 3), (6, 5)):
        A = rng.normal(size=(dim, dim))
        A = A @ A.T + dim * np.eye(dim)                         # SPD Hessian: y = A s gives s.y > 0
        S = [rng.normal(size=dim) for _ in range(m)]
        Y = [A @ s_ for s_ in S]
        g = rng.normal(size=dim)
        H = (S[-1] @ Y[-1]) / (Y[-1] @ Y[-1]) * np.eye(dim)
        for s_, y_ in zip(S, Y):
            rho = 1.0 / (y_ @ s_)
            V = np.eye(dim) - rho * np.outer(s_, y_)
            H = V @ H @ V.T + rho * np.outer(s_, s_)
        d = do.lbfgs_direction(g, S, Y)
        assert np.allclose(d, -H @ g, rtol=1e-11, atol=1e-12), (dim, m)
        assert d @ g < 0.0                                       # a descent direction
        assert not np.allclose(d, -g, rtol=1e-3)                 # and not the steepest-descent one
    assert np.array_equal(do.lbfgs_direction(np.array([1.0, -2.0]), [], []), np.array([-1.0, 2.0]))


def test_driver_oracle_lbfgs_on_a_convex_quadratic():
    """Exact line searches on f = x^T A x / 2 - b^T x with memory >= dimension: BFGS directions are A-conjugate and
    the minimiser A^-1 b is reached in at most `dim` steps (textbook property; a wrong recursion loses both)."""
    from oracle import driver_oracle as do
    rng = np.random.default_rng(5)
    dim = 5
    A = rng.normal(size=(dim, dim))
    A = A @ A.T + np.eye(dim)
    b = rng.normal(size=dim)
    x = rng.normal(size=dim)
    g = A @ x - b
    S, Y, D = [], [], []
    for _ in range(dim):
        d = do.lbfgs_direction(g, S, Y)
        a = -(g @ d) / (d @ A @ d)                               # exact minimiser along d
        s_ = a * d
        x = x + s_
        gn = A @ x - b
        S.append(s_), Y.append(gn - g), D.append(d)
        g = gn
    assert np.linalg.norm(x - np.linalg.solve(A, b)) < 1e-8
    for i in range(dim):
        for j in range(i):
            assert abs(D[i] @ A @ D[j]) < 1e-8 * np.sqrt((D[i] @ A @ D[i]) * (D[j] @ A @ D[j]))


# ---- pins of the read-out oracle (oracle/readout_oracle.py) -----------------------------------------------------------
def test_readout_oracle_product_state_closed_form():
    """RY(theta_q) on every qubit: p(x) = prod_q (cos^2 or sin^2)(theta_q / 2), so bit q of the most probable x is set
    exactly when sin^2 > cos^2, and p(x*) is the product of the larger factors."""
    from oracle import readout_oracle as ro
    n = 9
    r = SplitMix64(11)
    theta = np.array([(2 * r.uniform() - 1) * 3.1 for _ in range(n)])
    ops = [(0, q, -1, q) for q in range(n)]
    x, p = ro.most_probable(n, ops, theta)
    s2, c2 = np.sin(theta / 2) ** 2, np.cos(theta / 2) ** 2
    assert x == sum(1 << q for q in range(n) if s2[q] > c2[q])
    assert abs(p - np.prod(np.maximum(s2, c2))) < 1e-14
    assert abs(ro.probabilities(n, ops, theta).sum() - 1.0) < 1e-13


def test_readout_oracle_basis_state_and_tie():
    """RY(pi) on chosen qubits prepares the basis state |x>: p = 1 there.  GHZ (RY(pi/2) on qubit 0, CNOT chain) has
    two equal maxima at 0 and 2^n - 1 up to rounding; exact ties (RY(0) everywhere, Z-rotations only) go to the lowest x."""
    from oracle import readout_oracle as ro
    n = 6
    target = 0b101101
    ops = [(0, q, -1, q) for q in range(n)]
    theta = np.array([np.pi if (target >> q) & 1 else 0.0 for q in range(n)])
    x, p = ro.most_probable(n, ops, theta)
    assert x == target and abs(p - 1.0) < 1e-14
    ghz = [(0, 0, -1, 0)] + [(3, q + 1, q, -1) for q in range(n - 1)]
    pr = ro.probabilities(n, ghz, np.array([np.pi / 2]))
    assert abs(pr[0] - 0.5) < 1e-15 and abs(pr[-1] - 0.5) < 1e-15 and pr[1:-1].max() == 0.0
    # an exact tie: X-rotation-free circuit on |0..0> plus one RY(pi/2) whose two branches are bit-identical in modulus
    x, p = ro.most_probable(2, [(0, 1, -1, 0), (1, 1, -1, 1)], np.array([0.0, 0.7]))
    assert x == 0 and abs(p - 1.0) < 1e-15


def test_readout_oracle_sampling_pins():
    """One qubit after RY(theta): shot = 0 exactly when u < cos^2(theta/2).  A basis state: every shot is that state.
    Stratified uniforms u_s = (s + 1/2)/S turn inversion into quantiles: every outcome x is drawn S p(x) times up to
    +-1 (p from the product-state closed form)."""
    from oracle import readout_oracle as ro
    th = 1.1
    u = np.array([0.0, 0.3, np.cos(th / 2) ** 2 - 1e-9, np.cos(th / 2) ** 2 + 1e-9, 0.999999])
    x, Z = ro.sample(1, [(0, 0, -1, 0)], np.array([th]), u)
    assert list(x) == [0, 0, 0, 1, 1] and abs(Z - 1.0) < 1e-15
    n, target = 5, 0b10110
    ops = [(0, q, -1, q) for q in range(n)]
    x, Z = ro.sample(n, ops, np.array([np.pi if (target >> q) & 1 else 0.0 for q in range(n)]), np.linspace(1e-6, 0.999, 17))   # RY(pi) leaves ~1e-33 of mass elsewhere: u = 0 would land there
    assert np.all(x == target)
    r = SplitMix64(5)
    theta = np.array([(2 * r.uniform() - 1) * 3.0 for _ in range(n)])
    S = 4096
    x, Z = ro.sample(n, ops, theta, (np.arange(S) + 0.5) / S)
    s2, c2 = np.sin(theta / 2) ** 2, np.cos(theta / 2) ** 2
    p = np.array([np.prod([s2[q] if (y >> q) & 1 else c2[q] for q in range(n)]) for y in range(1 << n)])
    counts = np.bincount(x.astype(np.int64), minlength=1 << n)
    assert np.all(np.abs(counts - S * p) <= 1.0 + 1e-9)
    assert np.all(np.diff(x.astype(np.int64)) >= 0)              # inversion is monotone in u


def test_geometric_blocks_by_hand_and_library():
    assert go.geometric_blocks(7, 3, 0) == ([0, 0, 0, 1, 1, 1, 2], 3)
    assert go.geometric_blocks(7, 3, 1) == ([0, 1, 1, 1, 2, 2, 2], 3)
    assert go.geometric_blocks(7, 3, 2) == ([0, 0, 1, 1, 1, 2, 2], 3)
    assert go.geometric_blocks(4, 8, 0) == ([0, 0, 0, 0], 1)
    for n in (1, 5, 16, 28):
        for bs in (1, 2, 4, 5):
            for off in range(bs):
                lab, K = gb.geometric_blocks(n, bs, off)
                assert (list(lab), K) == go.geometric_blocks(n, bs, off)
    with pytest.raises(gv.GvqeError):
        gb.geometric_blocks(5, 2, 2)


# ---- pins of the finite-shot estimator oracle (oracle/readout_oracle.energy_shots) -------------------
def test_shot_oracle_settings_by_hand():
    from oracle import readout_oracle as ro
    settings, got = ro.measurement_groups(3, ["ZZI", "XIZ", "XZI", "YIZ", "IIZ", "XYI", "III"])
    assert settings == [(0, 0), (1, 0), (1, 1), (3, 2)]              # (x_mask, y_mask) ascending; Z-only and identity first
    assert got == [0, 1, 1, 2, 0, 3, 0]


def test_shot_oracle_rotation_diagonalises_the_letters():
    """After rotate_to_setting the probabilities weighted by (-1)^{popcount(x & support)} give the exact <P> of every term
    of the setting (the definition of measuring in that basis); checked against the dense Kronecker expectation."""
    import oracle
    from oracle import readout_oracle as ro
    from tests.dense_ref import dense_hamiltonian
    n = 4
    rng = np.random.default_rng(3)
    psi = rng.normal(size=1 << n) + 1j * rng.normal(size=1 << n)
    psi /= np.linalg.norm(psi)
    for s in ["XIZY", "YYII", "ZIXZ", "IYZX", "XXXX", "ZZII"]:
        xm = sum(1 << q for q, ch in enumerate(s) if ch in "XY")
        ym = sum(1 << q for q, ch in enumerate(s) if ch == "Y")
        supp = sum(1 << q for q, ch in enumerate(s) if ch != "I")
        phi = ro.rotate_to_setting(n, psi, xm, ym)
        assert abs(np.vdot(phi, phi).real - 1.0) < 1e-12
        p = np.abs(phi) ** 2
        est = sum(p[x] * (1 - 2 * (bin(x & supp).count("1") & 1)) for x in range(1 << n))
        exact = np.vdot(psi, dense_hamiltonian(n, [s], [1.0]) @ psi).real
        assert abs(est - exact) < 1e-12, s


def test_shot_oracle_one_qubit_closed_form_and_rate():
    """RY(theta)|0>, H = X: P(outcome 0 in the X basis) = (1 + sin theta) / 2.  Stratified uniforms give the estimate
    within 1/S of sin theta; random uniforms give an error that shrinks like 1/sqrt(S) and the exact energy in the limit."""
    from oracle import readout_oracle as ro
    th = 0.7
    ops = np.array([[0, 0, -1, 0]], dtype=np.int32)
    for S in (10, 1000):
        E, means, shots = ro.energy_shots(1, ops, [th], ["X"], [2.0], ((np.arange(S) + 0.5) / S).reshape(1, -1))
        assert abs(E - 2.0 * np.sin(th)) <= 2.0 * (2.0 / S) + 1e-12
        assert abs(np.mean(shots[0] == 0) - 0.5 * (1 + np.sin(th))) <= 1.0 / S + 1e-12
    rms = {}
    for S in (100, 10000):
        errs = []
        for rep in range(40):
            u = np.random.default_rng(1000 * S + rep).uniform(size=(1, S))
            E, _, _ = ro.energy_shots(1, ops, [th], ["X"], [2.0], u)
            errs.append(E - 2.0 * np.sin(th))
        rms[S] = float(np.sqrt(np.mean(np.square(errs))))
    sigma = 2.0 * np.cos(th)                                      # std of one shot of 2 X: 2 sqrt(1 - sin^2)
    assert 0.6 * sigma / 10 < rms[100] < 1.5 * sigma / 10 and 0.6 * sigma / 100 < rms[10000] < 1.5 * sigma / 100


def test_shot_oracle_product_state_terms():
    """Rotations only: <P> = prod_q f_q (closed form); each term's estimated mean lies within 5 standard errors."""
    import math
    from oracle import readout_oracle as ro
    n, S = 5, 4000
    rng = np.random.default_rng(8)
    th = rng.uniform(-math.pi, math.pi, 2 * n)
    ops = np.array([(0, q, -1, q) for q in range(n)] + [(1, q, -1, n + q) for q in range(n)], dtype=np.int32)
    terms = ["ZIIZI", "XIIII", "IYIZI", "XYZII", "IIXXY", "ZZZZZ", "IIIII"]
    cs = np.array([0.5, -1.0, 0.7, 0.3, -0.2, 1.1, 0.25])
    settings, _ = ro.measurement_groups(n, terms)
    E, means, _ = ro.energy_shots(n, ops, th, terms, cs, rng.uniform(size=(len(settings), S)))
    for k, s in enumerate(terms):
        v = 1.0
        for q, ch in enumerate(s):
            v *= {"I": 1.0, "Z": math.cos(th[q]), "X": math.sin(th[q]) * math.cos(th[n + q]), "Y": math.sin(th[q]) * math.sin(th[n + q])}[ch]
        assert abs(means[k] - v) <= 5.0 * math.sqrt(max(1.0 - v * v, 1e-12) / S) + 1e-9, (s, means[k], v)
    assert means[-1] == 1.0                                       # identity: +1 on every shot

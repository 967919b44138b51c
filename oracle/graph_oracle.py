"""CPU oracle for Graph-VQE's Hamiltonian-aware partitioning -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Plain Python/numpy restatement of PAPER.md:183-197: the qubit interaction graph (Eq. 9), the modularity Q (Eq. 10),
Louvain community detection (the paper names the algorithm; the steps below are Blondel et al.'s two phases in the
order DESIGN.md reading G2 fixes) and the merge of blocks smaller than S_min (reading G3), plus the qubit block ->
parameter mask of PAPER.md:207 (reading A11).  Shares no code with paper_2607_02749_b200/csrc/graph.cpp.
Pins: tests/test_graph_pins.py (hand-computed Eq. 9 example, closed-form Q of disjoint cliques / one block /
singletons, brute force over all set partitions for n <= 7, planted communities).
"""
from __future__ import annotations

import numpy as np


def interaction_graph(n: int, paulis, coeffs) -> np.ndarray:
    """Eq. 9: w_ij = sum over terms k whose Pauli on qubit i and on qubit j are both non-identity of |c_k|.
    paulis[k][j] acts on qubit j (reading A4)."""
    w = np.zeros((n, n), dtype=np.float64)
    for s, c in zip(paulis, coeffs):
        for i in range(n):
            for j in range(n):
                if i != j and s[i] != "I" and s[j] != "I":
                    w[i, j] += abs(float(c))
    return w


def modularity(w: np.ndarray, community, gamma: float = 1.0) -> float:
    """Eq. 10: Q = 1/(2m) sum_ij [w_ij - gamma k_i k_j/(2m)] delta(c_i, c_j), m = 1/2 sum_ij w_ij, k_i = sum_j w_ij."""
    n = w.shape[0]
    m = 0.5 * sum(w[i, j] for i in range(n) for j in range(n))
    if m <= 0.0:
        return 0.0
    k = [sum(w[i, j] for j in range(n)) for i in range(n)]
    q = 0.0
    for i in range(n):
        for j in range(n):
            if community[i] == community[j]:
                q += w[i, j] - gamma * k[i] * k[j] / (2.0 * m)
    return q / (2.0 * m)


def _first_appearance(labels):
    seen = {}
    out = []
    for l in labels:
        if l not in seen:
            seen[l] = len(seen)
        out.append(seen[l])
    return out


def louvain(w: np.ndarray, gamma: float = 1.0):
    """Louvain.  Phase 1: visit nodes in ascending order; take node i out of its community and put it into the
    neighbouring community (or back) that gives the largest modularity gain k_{i,in}(C) - gamma tot(C) k_i / (2m);
    a move needs a gain larger than staying by more than 1e-12, ties go to the lowest label; sweep until nothing
    moves.  Phase 2: communities become nodes, weights add (internal weight becomes a self loop).  Repeat until a
    phase 1 moves nothing.  Returns (labels by first appearance, K)."""
    n = w.shape[0]
    two_m = float(w.sum())
    node_of = list(range(n))           # super-node of every original node
    if two_m <= 0.0:
        return node_of, n
    a = np.array(w, dtype=np.float64)
    while True:
        m = a.shape[0]
        k = a.sum(axis=1)
        comm = list(range(m))
        tot = [float(k[i]) for i in range(m)]
        any_move = False
        moved = True
        while moved:
            moved = False
            for i in range(m):
                home = comm[i]
                links = {}
                for j in range(m):
                    if j != i and a[i, j] > 0.0:
                        links[comm[j]] = links.get(comm[j], 0.0) + float(a[i, j])
                tot[home] -= float(k[i])
                best = links.get(home, 0.0) - gamma * tot[home] * float(k[i]) / two_m
                best_c = home
                for c in sorted(links):
                    if c == home:
                        continue
                    g = links[c] - gamma * tot[c] * float(k[i]) / two_m
                    if g > best + 1e-12:
                        best, best_c = g, c
                tot[best_c] += float(k[i])
                if best_c != home:
                    comm[i] = best_c
                    moved = any_move = True
        if not any_move:
            break
        comm = _first_appearance(comm)
        K = max(comm) + 1
        node_of = [comm[s] for s in node_of]
        b = np.zeros((K, K), dtype=np.float64)
        for i in range(m):
            for j in range(m):
                b[comm[i], comm[j]] += a[i, j]
        a = b
    labels = _first_appearance(node_of)
    return labels, max(labels) + 1


def merge_small_blocks(w: np.ndarray, community, s_min: int):
    """PAPER.md:197, reading G3: while some block has fewer than s_min qubits (and more than one block is left),
    the smallest such block (lowest label on ties) joins the block with which it shares the largest total weight
    (lowest label on ties); labels are renumbered by first appearance after every merge."""
    n = w.shape[0]
    lab = _first_appearance(list(community))
    while max(lab) + 1 > 1:
        K = max(lab) + 1
        size = [lab.count(c) for c in range(K)]
        small = [c for c in range(K) if size[c] < s_min]
        if not small:
            break
        s = min(small, key=lambda c: (size[c], c))
        link = [0.0] * K
        for i in range(n):
            for j in range(n):
                if lab[i] == s and lab[j] != s:
                    link[lab[j]] += float(w[i, j])
        t = max((c for c in range(K) if c != s), key=lambda c: (link[c], -c))
        lab = _first_appearance([t if l == s else l for l in lab])
    return lab, max(lab) + 1


def block_param_mask(ops, n_params: int, community, block: int) -> np.ndarray:
    """theta_{B_i}: parameters of the rotations (kind 0 = RY, 1 = RZ) acting on a qubit of the block (A11).
    ops: rows (kind, q0, q1, param)."""
    mask = np.zeros(n_params, dtype=np.uint8)
    for kind, q0, _q1, param in ops:
        if kind in (0, 1) and param >= 0 and community[q0] == block:
            mask[param] = 1
    return mask


def geometric_blocks(n: int, block_size: int, offset: int = 0):
    """PAPER.md:229 "geometric alternating offsets" (reading G7): block boundaries at offset, offset + block_size, ...;
    labels in qubit order."""
    bounds = [b for b in range(offset, n, block_size)]
    lab = [sum(1 for b in bounds if b <= q and b > 0) for q in range(n)]
    return _first_appearance(lab), max(lab) + 1 if n else 0

"""Seeded synthetic inputs for the Graph-VQE energy hot path (arxiv/paper_2607_02749).

This module produces DATA only: circuit descriptions, Pauli strings, coefficients, parameter batches.
It evaluates no gate, no expectation value and no gradient; the oracle (``oracle/``) and the CUDA
library each interpret these arrays with their own, separate code.

The paper's own instances (ten peptides, N = 2(L-1) = 8..10 qubits, MJ-potential Hamiltonians,
PAPER.md:112-153, 251-258) are not available; BASELINE.json's five seeded configs stand in for them
and take their *structure* from the paper: sparse Pauli sums with community structure
(PAPER.md:183-197), low weight with a minority of non-local terms, an
EfficientSU2-style RY/RZ + entangler ansatz, angles in [-pi, pi].

Random numbers: SplitMix64 (counter style, state += golden gamma), uniform = (u >> 11) * 2**-53,
normal = Box-Muller (cos branch, two uniforms per sample), Laplace(0,1) = inverse CDF.
seed(cfg, stream) = 260702749*100 + 10*cfg + stream; stream 0 = Hamiltonian, 1 = parameters,
2 = flip-set pool.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

OP_RY, OP_RZ, OP_CZ, OP_CNOT = 0, 1, 2, 3
_M64 = (1 << 64) - 1


class SplitMix64:
    """Self-contained 64-bit generator (not numpy's, whose streams are version dependent)."""

    def __init__(self, seed: int):
        self.s = seed & _M64

    def u64(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & _M64
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return (self.u64() >> 11) * (2.0 ** -53)

    def randint(self, k: int) -> int:
        """Uniform integer in [0, k)."""
        return min(int(self.uniform() * k), k - 1)

    def normal(self) -> float:
        u1 = 1.0 - self.uniform()  # (0, 1]
        u2 = self.uniform()
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)

    def laplace(self) -> float:
        v = self.uniform() - 0.5
        a = 1.0 - 2.0 * abs(v)
        if a <= 0.0:
            a = 2.0 ** -53
        return -math.copysign(1.0, v) * math.log(a)

    def sample_distinct(self, pool: Sequence[int], w: int) -> List[int]:
        """w distinct items of pool (partial Fisher-Yates), returned sorted."""
        p = list(pool)
        for i in range(w):
            j = i + self.randint(len(p) - i)
            p[i], p[j] = p[j], p[i]
        return sorted(p[:w])


def seed_of(cfg: int, stream: int) -> int:
    return 260702749 * 100 + 10 * cfg + stream


# ----------------------------------------------------------------------------------------------
# configs (BASELINE.json "configs", 1-based ids as in SURVEY.md §8; 5 = 5a (32q c64), 6 = 5b (30q c128))
# ----------------------------------------------------------------------------------------------
CONFIGS: Dict[int, dict] = {
    1: dict(n=10, precisions=("c128",), D=3, entangler="cz", topology="linear", final_rot=1,
            M=200, f_z=1.0, w_max=4, communities=[5, 5], p_intra=0.90, coeff="normal",
            inter_scale=1.0, pool=0, batch="shift_all"),
    2: dict(n=16, precisions=("c128",), D=4, entangler="cz", topology="linear", final_rot=1,
            M=1000, f_z=0.85, w_max=4, communities=[4, 4, 4, 4], p_intra=0.90, coeff="normal",
            inter_scale=0.1, pool=0, batch="shift_community0"),
    3: dict(n=22, precisions=("c64", "c128"), D=5, entangler="cz", topology="linear", final_rot=1,
            M=5000, f_z=0.90, w_max=4, communities=[4, 4, 4, 4, 3, 3], p_intra=0.92, coeff="laplace",
            inter_scale=1.0, pool=0, batch=64),
    4: dict(n=28, precisions=("c64",), D=6, entangler="cnot", topology="ring", final_rot=1,
            M=20000, f_z=0.80, w_max=4, communities=[4, 4, 4, 4, 3, 3, 3, 3], p_intra=0.90,
            coeff="normal", inter_scale=1.0, pool=256, batch="shift_all", chunk=8),
    5: dict(n=32, precisions=("c64",), D=4, entangler="cz", topology="linear", final_rot=1,
            M=50000, f_z=0.80, w_max=6, communities=[4, 4, 3, 3, 3, 3, 3, 3, 3, 3], p_intra=0.90,
            coeff="normal", inter_scale=1.0, pool=256, batch=1),
    6: dict(n=30, precisions=("c128",), D=4, entangler="cz", topology="linear", final_rot=1,
            M=50000, f_z=0.80, w_max=6, communities=[3] * 10, p_intra=0.90,
            coeff="normal", inter_scale=1.0, pool=256, batch=1),
}


def num_params(n: int, D: int, final_rot: int) -> int:
    """P = N(2D+1) for final_rot=1 (BASELINE configs); P = 2N(D+1) for final_rot=2 (Eq. 8)."""
    return 2 * n * D + n * final_rot


def entangler_pairs(n: int, topology: str, layer: int) -> List[Tuple[int, int]]:
    """(control, target) pairs of one entangling layer (reading A17; PAPER.md:260 lists the maps)."""
    chain = [(q, q + 1) for q in range(n - 1)]
    if topology == "linear" or n <= 2 and topology in ("ring", "circular", "sca"):
        return chain
    if topology == "ring":
        return chain + [(n - 1, 0)]
    if topology == "circular":
        return [(n - 1, 0)] + chain
    if topology == "full":
        return [(i, j) for i in range(n) for j in range(i + 1, n)]
    if topology == "reverse_linear":
        return chain[::-1]
    if topology == "pairwise":
        return [p for p in chain if p[0] % 2 == 0] + [p for p in chain if p[0] % 2 == 1]
    if topology == "sca":
        circ = [(n - 1, 0)] + chain
        shifted = [circ[(j - layer) % n] for j in range(n)]
        return [(t, c) for (c, t) in shifted] if layer % 2 else shifted
    raise ValueError(topology)


def layout_ops(n: int, D: int, entangler: str, topology: str, final_rot: int) -> List[Tuple[int, int, int, int]]:
    """Ansatz layout -> explicit op list [(kind, q0, q1, param)] (readings A1-A5).

    for l in 0..D-1: RY(theta[2nl+q]) all q; RZ(theta[2nl+n+q]) all q; entanglers (q, q+1) ascending,
    then (n-1 -> 0) if ring; finally RY(theta[2nD+q]) (and RZ(theta[2nD+n+q]) when final_rot == 2).
    CNOT is stored as (OP_CNOT, target, control, -1); CZ as (OP_CZ, q, q+1, -1).
    """
    ops: List[Tuple[int, int, int, int]] = []
    for l in range(D):
        for q in range(n):
            ops.append((OP_RY, q, -1, 2 * n * l + q))
        for q in range(n):
            ops.append((OP_RZ, q, -1, 2 * n * l + n + q))
        pairs = entangler_pairs(n, topology, l)
        for (c, t) in pairs:
            if entangler == "cz":
                ops.append((OP_CZ, c, t, -1))
            else:
                ops.append((OP_CNOT, t, c, -1))
    for q in range(n):
        ops.append((OP_RY, q, -1, 2 * n * D + q))
    if final_rot == 2:
        for q in range(n):
            ops.append((OP_RZ, q, -1, 2 * n * D + n + q))
    return ops


def community_param_mask(n: int, D: int, final_rot: int, qubits: Sequence[int]) -> np.ndarray:
    """Reading A11: every rotation parameter whose gate acts on a qubit of the block."""
    P = num_params(n, D, final_rot)
    m = np.zeros(P, dtype=np.uint8)
    for q in qubits:
        for l in range(D):
            m[2 * n * l + q] = 1
            m[2 * n * l + n + q] = 1
        m[2 * n * D + q] = 1
        if final_rot == 2:
            m[2 * n * D + n + q] = 1
    return m


def shift_rows(theta: np.ndarray, mask: np.ndarray) -> np.ndarray:
    """Reading A8: row 0 = theta; rows 2j+1 / 2j+2 = theta +/- (pi/2) e_p for the j-th masked p, ascending."""
    idx = np.flatnonzero(mask)
    rows = np.tile(np.asarray(theta, dtype=np.float64), (2 * len(idx) + 1, 1))
    for j, p in enumerate(idx):
        rows[2 * j + 1, p] += math.pi / 2
        rows[2 * j + 2, p] -= math.pi / 2
    return rows


def _community_ranges(sizes: Sequence[int]) -> List[List[int]]:
    out, q = [], 0
    for s in sizes:
        out.append(list(range(q, q + s)))
        q += s
    return out


def _scaled_communities(sizes: Sequence[int], n: int) -> List[int]:
    """Keep the community count when a test shrinks n (contiguous ranges, sizes as even as possible)."""
    if sum(sizes) == n:
        return list(sizes)
    k = max(1, min(len(sizes), n // 2 if n >= 4 else 1))
    base, extra = divmod(n, k)
    return [base + (1 if i < extra else 0) for i in range(k)]


def _draw_support(rng: SplitMix64, w: int, comms: List[List[int]], n: int, p_intra: float):
    """Rule 3: (sorted support, community index or -1 for inter-community)."""
    if w == 1 or n == 1:
        q = rng.randint(n)
        ci = next(i for i, c in enumerate(comms) if q in c)
        return [q], ci
    if len(comms) == 1 or rng.uniform() < p_intra:
        ci = rng.randint(len(comms))
        c = comms[ci]
        return rng.sample_distinct(c, min(w, len(c))), ci
    w = min(w, n)
    while True:
        s = rng.sample_distinct(range(n), w)
        owners = {next(i for i, c in enumerate(comms) if q in c) for q in s}
        if len(owners) >= 2:
            return s, -1


def make_hamiltonian(cfg_id: int, n: int, M: int, f_z: float, w_max: int, comm_sizes: Sequence[int],
                     p_intra: float, coeff: str, inter_scale: float, pool: int):
    """Returns (paulis: bytes of M*n chars, char j of a term acts on qubit j; coeffs float64[M])."""
    rng = SplitMix64(seed_of(cfg_id, 0))
    comms = _community_ranges(comm_sizes)
    owner = {q: i for i, c in enumerate(comms) for q in c}
    n_z = int(round(f_z * M))
    pool_sets = []
    if pool and n_z < M:
        prng = SplitMix64(seed_of(cfg_id, 2))
        for _ in range(pool):
            w = 1 + prng.randint(min(4, w_max))
            pool_sets.append(_draw_support(prng, w, comms, n, p_intra))
    terms = []
    for k in range(M):
        letters = ["I"] * n
        if k < n_z:
            w = 1 + rng.randint(w_max)
            supp, _ = _draw_support(rng, w, comms, n, p_intra)
            for q in supp:
                letters[q] = "Z"
        elif pool_sets:
            flip, ci = pool_sets[rng.randint(len(pool_sets))]
            for q in flip:
                letters[q] = "X" if rng.uniform() < 0.5 else "Y"
            others = [q for q in (comms[ci] if ci >= 0 else range(n)) if q not in flip]
            nz = rng.randint(min(w_max - len(flip), len(others)) + 1)
            for q in (rng.sample_distinct(others, nz) if nz else []):
                letters[q] = "Z"
        else:
            w = 1 + rng.randint(w_max)
            supp, _ = _draw_support(rng, w, comms, n, p_intra)
            nflip = 1 + rng.randint(len(supp))
            flip = rng.sample_distinct(supp, nflip)
            for q in supp:
                letters[q] = "Z"
            for q in flip:
                letters[q] = "X" if rng.uniform() < 0.5 else "Y"
        c = rng.normal() if coeff == "normal" else rng.laplace()
        supp_all = [q for q in range(n) if letters[q] != "I"]
        if inter_scale != 1.0 and len({owner[q] for q in supp_all}) >= 2:
            c *= inter_scale
        terms.append(("".join(letters), c))
    for i in range(M - 1, 0, -1):  # one seeded Fisher-Yates shuffle of the term order
        j = rng.randint(i + 1)
        terms[i], terms[j] = terms[j], terms[i]
    paulis = "".join(t[0] for t in terms).encode("ascii")
    coeffs = np.array([t[1] for t in terms], dtype=np.float64)
    return paulis, coeffs


@dataclass
class Workload:
    cfg_id: int
    name: str
    n: int
    precisions: Tuple[str, ...]
    D: int
    entangler: str
    topology: str
    final_rot: int
    P: int
    ops: np.ndarray            # int32 [n_ops, 4] = (kind, q0, q1, param)
    paulis: bytes              # M*n chars
    coeffs: np.ndarray         # float64 [M]
    communities: List[List[int]]
    theta: np.ndarray          # float64 [P] base vector (rows[0])
    params: np.ndarray         # float64 [B, P] the batch gvqe_energy_batch sees (shift set expanded, A8)
    mask: Optional[np.ndarray]  # uint8 [P] for param-shift workloads, else None
    chunk: int = 0             # states in flight requested by the config (0 = library decides)
    meta: dict = field(default_factory=dict)

    @property
    def M(self) -> int:
        return len(self.coeffs)

    @property
    def B(self) -> int:
        return self.params.shape[0]

    def pauli_list(self) -> List[str]:
        s = self.paulis.decode("ascii")
        return [s[i * self.n:(i + 1) * self.n] for i in range(self.M)]


def make_workload(cfg_id: int, n: Optional[int] = None, M: Optional[int] = None, D: Optional[int] = None,
                  batch=None, final_rot: Optional[int] = None, entangler: Optional[str] = None,
                  topology: Optional[str] = None) -> Workload:
    """BASELINE config `cfg_id` (1..6), optionally shrunk (n, M, D, batch) for parity tests: same recipe,
    same seeds, smaller sizes."""
    c = dict(CONFIGS[cfg_id])
    if n is not None:
        c["communities"] = _scaled_communities(c["communities"], n)
        c["n"] = n
    for k_, v in (("M", M), ("D", D), ("batch", batch), ("final_rot", final_rot),
                  ("entangler", entangler), ("topology", topology)):
        if v is not None:
            c[k_] = v
    n_, D_, fr = c["n"], c["D"], c["final_rot"]
    P = num_params(n_, D_, fr)
    ops = np.array(layout_ops(n_, D_, c["entangler"], c["topology"], fr), dtype=np.int32).reshape(-1, 4)
    paulis, coeffs = make_hamiltonian(cfg_id, n_, c["M"], c["f_z"], c["w_max"], c["communities"],
                                      c["p_intra"], c["coeff"], c["inter_scale"], c["pool"])
    prng = SplitMix64(seed_of(cfg_id, 1))
    comms = _community_ranges(c["communities"])
    b = c["batch"]
    mask = None
    if isinstance(b, int):
        rows = np.array([[(2.0 * prng.uniform() - 1.0) * math.pi for _ in range(P)] for _ in range(b)],
                        dtype=np.float64).reshape(b, P)
        theta = rows[0].copy()
    else:
        theta = np.array([(2.0 * prng.uniform() - 1.0) * math.pi for _ in range(P)], dtype=np.float64)
        if b == "shift_all":
            mask = np.ones(P, dtype=np.uint8)
        elif b == "shift_community0":
            mask = community_param_mask(n_, D_, fr, comms[0])
        else:
            raise ValueError(b)
        rows = shift_rows(theta, mask)
    return Workload(cfg_id=cfg_id, name=f"cfg{cfg_id}_n{n_}", n=n_, precisions=tuple(c["precisions"]), D=D_,
                    entangler=c["entangler"], topology=c["topology"], final_rot=fr, P=P, ops=ops,
                    paulis=paulis, coeffs=coeffs, communities=comms, theta=theta, params=rows, mask=mask,
                    chunk=int(c.get("chunk", 0)), meta=dict(f_z=c["f_z"], w_max=c["w_max"], pool=c["pool"]))


def random_ops(seed: int, n: int, n_ops: int) -> Tuple[np.ndarray, int]:
    """Random op list for stress tests: RY/RZ with fresh parameters, CZ/CNOT on random distinct qubit pairs."""
    rng = SplitMix64(seed)
    ops, p = [], 0
    for _ in range(n_ops):
        k = rng.randint(4) if n >= 2 else rng.randint(2)
        if k in (OP_RY, OP_RZ):
            ops.append((k, rng.randint(n), -1, p))
            p += 1
        else:
            a, b = rng.sample_distinct(range(n), 2)
            if rng.uniform() < 0.5:
                a, b = b, a
            ops.append((k, a, b, -1))
    return np.array(ops, dtype=np.int32).reshape(-1, 4), p


def random_paulis(seed: int, n: int, M: int, w_max: int) -> Tuple[bytes, np.ndarray]:
    """Unstructured random Pauli strings (any letters on a random support of weight <= w_max), N(0,1) coefficients."""
    rng = SplitMix64(seed)
    out, cs = [], []
    for _ in range(M):
        w = rng.randint(min(w_max, n) + 1)
        letters = ["I"] * n
        for q in (rng.sample_distinct(range(n), w) if w else []):
            letters[q] = "XYZ"[rng.randint(3)]
        out.append("".join(letters))
        cs.append(rng.normal())
    return "".join(out).encode("ascii"), np.array(cs, dtype=np.float64)

"""Dense brute-force reference used ONLY to pin the oracle (n <= 8): full 2^n x 2^n unitary as an ordered product
of Kronecker-built matrices and full dense H = sum_k c_k (sigma_{n-1} (x) ... (x) sigma_0).  Written from the
textbook definitions (Eq. 6, Eq. 7 of PAPER.md:150, 171-173); shares nothing with oracle/ or the CUDA path."""
import numpy as np

I2 = np.eye(2, dtype=np.complex128)
X = np.array([[0, 1], [1, 0]], dtype=np.complex128)
Y = np.array([[0, -1j], [1j, 0]], dtype=np.complex128)
Z = np.array([[1, 0], [0, -1]], dtype=np.complex128)
PAULI = {"I": I2, "X": X, "Y": Y, "Z": Z}


def kron_on(n, mats):
    """mats: {qubit: 2x2}; qubit 0 = least significant bit => sigma_{n-1} (x) ... (x) sigma_0."""
    out = np.array([[1.0 + 0j]])
    for q in range(n - 1, -1, -1):
        out = np.kron(out, mats.get(q, I2))
    return out


def ry(t):
    c, s = np.cos(t / 2), np.sin(t / 2)
    return np.array([[c, -s], [s, c]], dtype=np.complex128)


def rz(t):
    return np.array([[np.exp(-0.5j * t), 0], [0, np.exp(0.5j * t)]], dtype=np.complex128)


def proj(b):
    return np.array([[1 - b, 0], [0, b]], dtype=np.complex128)


def gate_matrix(n, kind, q0, q1, angle):
    if kind == 0:
        return kron_on(n, {q0: ry(angle)})
    if kind == 1:
        return kron_on(n, {q0: rz(angle)})
    if kind == 2:  # CZ = 1 - 2 |11><11|
        return np.eye(1 << n, dtype=np.complex128) - 2 * kron_on(n, {q0: proj(1), q1: proj(1)})
    if kind == 3:  # CNOT target q0, control q1 = |0><0|_c (x) 1 + |1><1|_c (x) X_t
        return kron_on(n, {q1: proj(0)}) + kron_on(n, {q1: proj(1), q0: X})
    raise ValueError(kind)


def dense_unitary(n, ops, theta):
    U = np.eye(1 << n, dtype=np.complex128)
    for kind, q0, q1, p in np.asarray(ops).reshape(-1, 4):
        ang = theta[p] if p >= 0 else 0.0
        U = gate_matrix(n, int(kind), int(q0), int(q1), ang) @ U
    return U


def dense_hamiltonian(n, pauli_list, coeffs):
    H = np.zeros((1 << n, 1 << n), dtype=np.complex128)
    for s, c in zip(pauli_list, coeffs):
        H += c * kron_on(n, {q: PAULI[ch] for q, ch in enumerate(s)})
    return H


def dense_energy(n, ops, theta, pauli_list, coeffs):
    U = dense_unitary(n, ops, theta)
    psi = U[:, 0]
    H = dense_hamiltonian(n, pauli_list, coeffs)
    return float(np.real(np.vdot(psi, H @ psi))), psi

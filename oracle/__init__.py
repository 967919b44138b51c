"""CPU oracle for the Graph-VQE energy hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  The product (``paper_2607_02749_b200``) never does.  The arithmetic lives in plain C
(``gvqe_oracle.c`` tier T0, ``gvqe_oracle_t1.c`` tier T1); this file only builds and marshals.  Plain-Python oracles of
what sits around the energy path: ``graph_oracle.py`` (Eq. 9, Eq. 10, Louvain, block merge, masks), ``driver_oracle.py``
(the epoch loop, step by step) and ``readout_oracle.py`` (most probable bitstring, shot sampling by inversion).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "gvqe_oracle.c"), os.path.join(_HERE, "gvqe_oracle_t1.c")]
_SO = os.path.join(_HERE, "libgvqe_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -> oracle/libgvqe_oracle.so (rebuilt when a source is newer)."""
    if (not force and os.path.exists(_SO)
            and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC)):
        return _SO
    tmp = _SO + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=gnu11", "-shared", "-fPIC", "-o", tmp] + _SRC + ["-lm"])
    os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        c = ctypes
        vp, i32, dbl = c.c_void_p, c.c_int, c.c_double
        L.orc_state.argtypes = [i32, vp, i32, vp, vp]
        L.orc_state.restype = None
        L.orc_energy.argtypes = [i32, vp, i32, c.c_char_p, vp, vp, vp]
        L.orc_energy.restype = dbl
        L.orc_energy_batch.argtypes = [i32, vp, i32, i32, vp, i32, i32, c.c_char_p, vp, vp]
        L.orc_energy_batch.restype = i32
        L.orc_param_shift_grad.argtypes = [i32, vp, i32, i32, vp, vp, i32, c.c_char_p, vp, vp, vp]
        L.orc_param_shift_grad.restype = i32
        L.orc_grouping.argtypes = [i32, i32, c.c_char_p, vp, vp, vp, vp, vp, vp]
        L.orc_grouping.restype = i32
        L.orc_norm2.argtypes = [i32, vp]
        L.orc_norm2.restype = dbl
        L.orc_t1_diag_table.argtypes = [i32, i32, c.c_char_p, vp, vp]
        L.orc_t1_diag_table.restype = i32
        L.orc_t1_energy.argtypes = [i32, vp, i32, c.c_char_p, vp, vp]
        L.orc_t1_energy.restype = dbl
        _lib = L
    return _lib


def set_threads(k: int) -> None:
    """OpenMP threads for the oracle (libgomp reads this per parallel region through omp_set_num_threads)."""
    g = ctypes.CDLL("libgomp.so.1")
    g.omp_set_num_threads(int(k))


def max_threads() -> int:
    g = ctypes.CDLL("libgomp.so.1")
    return int(g.omp_get_max_threads())


def _ops(ops) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(ops, dtype=np.int32).reshape(-1, 4))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _paulis(p) -> bytes:
    if isinstance(p, (bytes, bytearray)):
        return bytes(p)
    if isinstance(p, str):
        return p.encode("ascii")
    return "".join(p).encode("ascii")


def state(n: int, ops, theta) -> np.ndarray:
    ops = _ops(ops)
    theta = _f64(theta)
    psi = np.empty(1 << n, dtype=np.complex128)
    lib().orc_state(n, ops.ctypes.data, len(ops), theta.ctypes.data, psi.ctypes.data)
    return psi


def energy_of_state(n: int, psi: np.ndarray, paulis, coeffs, return_terms: bool = False):
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    coeffs = _f64(coeffs)
    M = len(coeffs)
    terms = np.zeros(max(M, 1), dtype=np.float64)
    mi = ctypes.c_double(0.0)
    E = lib().orc_energy(n, psi.ctypes.data, M, _paulis(paulis), coeffs.ctypes.data, terms.ctypes.data,
                         ctypes.addressof(mi))
    if return_terms:
        return E, terms[:M], mi.value
    return E


def energy_batch(n: int, ops, params, paulis, coeffs) -> np.ndarray:
    ops = _ops(ops)
    params = _f64(params)
    if params.ndim == 1:
        params = params.reshape(1, -1)
    B, P = params.shape
    coeffs = _f64(coeffs)
    E = np.zeros(B, dtype=np.float64)
    rc = lib().orc_energy_batch(n, ops.ctypes.data, len(ops), P, params.ctypes.data, B, len(coeffs),
                                _paulis(paulis), coeffs.ctypes.data, E.ctypes.data)
    if rc:
        raise MemoryError("oracle: out of memory")
    return E


def param_shift_grad(n: int, ops, theta, mask, paulis, coeffs):
    ops = _ops(ops)
    theta = _f64(theta)
    mask = np.ascontiguousarray(np.asarray(mask, dtype=np.uint8))
    coeffs = _f64(coeffs)
    dE = np.zeros(len(theta), dtype=np.float64)
    E0 = ctypes.c_double(0.0)
    rc = lib().orc_param_shift_grad(n, ops.ctypes.data, len(ops), len(theta), theta.ctypes.data, mask.ctypes.data,
                                    len(coeffs), _paulis(paulis), coeffs.ctypes.data, dE.ctypes.data,
                                    ctypes.addressof(E0))
    if rc:
        raise MemoryError("oracle: out of memory")
    return dE, E0.value


def grouping(n: int, paulis, M: Optional[int] = None):
    p = _paulis(paulis)
    M = len(p) // n if M is None else M
    xm = np.zeros(max(M, 1), dtype=np.uint64)
    zm = np.zeros(max(M, 1), dtype=np.uint64)
    ny = np.zeros(max(M, 1), dtype=np.uint8)
    got = np.zeros(max(M, 1), dtype=np.int32)
    gm = np.zeros(max(M, 1), dtype=np.uint64)
    ng = ctypes.c_int32(0)
    rc = lib().orc_grouping(n, M, p, xm.ctypes.data, zm.ctypes.data, ny.ctypes.data, got.ctypes.data,
                            ctypes.addressof(ng), gm.ctypes.data)
    if rc:
        raise ValueError("oracle: bad Pauli character")
    return xm[:M], zm[:M], ny[:M], got[:M], int(ng.value), gm[:ng.value]


def norm2(n: int, psi: np.ndarray) -> float:
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    return float(lib().orc_norm2(n, psi.ctypes.data))


def t1_diag_table(n: int, paulis, coeffs) -> np.ndarray:
    coeffs = _f64(coeffs)
    tab = np.empty(1 << n, dtype=np.float64)
    rc = lib().orc_t1_diag_table(n, len(coeffs), _paulis(paulis), coeffs.ctypes.data, tab.ctypes.data)
    if rc:
        raise ValueError("oracle: bad Pauli character")
    return tab


def t1_energy_of_state(n: int, psi: np.ndarray, paulis, coeffs, table: Optional[np.ndarray] = None) -> float:
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    coeffs = _f64(coeffs)
    tp = None if table is None else np.ascontiguousarray(table, dtype=np.float64).ctypes.data
    return float(lib().orc_t1_energy(n, psi.ctypes.data, len(coeffs), _paulis(paulis), coeffs.ctypes.data, tp))

"""ctypes binding of libgvqe (include/gvqe.h): argument marshalling only, same names as the C ABI.

Every step of the path runs in the CUDA kernels of libgvqe.so; there is no Python or CPU fallback: a missing
library raises at import of the symbols, a missing GPU surfaces as GVQE_ERR_CUDA from the first energy call.
PyTorch is used for the device workspace and the stream only.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

GVQE_OK, GVQE_ERR_INVALID_ARG, GVQE_ERR_NO_HAMILTONIAN, GVQE_ERR_WORKSPACE, GVQE_ERR_UNSUPPORTED, GVQE_ERR_CUDA = range(6)
GVQE_C64, GVQE_C128 = 0, 1
STATUS_NAMES = ["GVQE_OK", "GVQE_ERR_INVALID_ARG", "GVQE_ERR_NO_HAMILTONIAN", "GVQE_ERR_WORKSPACE",
                "GVQE_ERR_UNSUPPORTED", "GVQE_ERR_CUDA"]

EXPORTS = ["gvqe_create", "gvqe_create_ops", "gvqe_create_opt", "gvqe_create_ops_opt", "gvqe_kernel_source", "gvqe_kernel_info", "gvqe_kernel_arrays", "gvqe_compile_kernels", "gvqe_num_params", "gvqe_num_qubits", "gvqe_set_hamiltonian",
           "gvqe_set_hamiltonian_masks", "gvqe_get_grouping", "gvqe_workspace_bytes", "gvqe_set_workspace",
           "gvqe_set_max_in_flight", "gvqe_energy_batch", "gvqe_energy_batch_device", "gvqe_param_shift_grad",
           "gvqe_get_state", "gvqe_argmax", "gvqe_argmax_noalloc", "gvqe_sample", "gvqe_measurement_settings", "gvqe_energy_shots", "gvqe_schedule_info", "gvqe_dump_schedule", "gvqe_get_exec_order", "gvqe_launch_count",
           "gvqe_profile_enable", "gvqe_profile_read", "gvqe_profile_read_launches", "gvqe_interaction_graph", "gvqe_modularity", "gvqe_louvain",
           "gvqe_merge_small_blocks", "gvqe_geometric_blocks", "gvqe_block_param_mask", "gvqe_graph_vqe_minimize", "gvqe_cobyla_minimize", "gvqe_last_error", "gvqe_destroy"]


class GvqeLayout(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("entangler", C.c_int32), ("topology", C.c_int32), ("final_rot", C.c_int32)]


class GvqeOptions(C.Structure):
    """gvqe_options: how the same energies are computed (0 = library default for every field)."""
    _fields_ = [("tile_bits", C.c_int32), ("fixed_bits", C.c_int32), ("reg_bits", C.c_int32), ("expect_tile_bits", C.c_int32),
                ("prefix", C.c_int32), ("register_stages", C.c_int32), ("shared_prefix", C.c_int32), ("specialise", C.c_int32),
                ("tiles_per_block", C.c_int32), ("blocks_per_sm", C.c_int32), ("staged_io", C.c_int32),
                ("mid_cnot", C.c_int32), ("interleave", C.c_int32), ("reserved", C.c_int32 * 3)]


class GvqeOptOptions(C.Structure):
    _fields_ = [("max_epochs", C.c_int32), ("block_iters", C.c_int32), ("global_iters", C.c_int32),
                ("window", C.c_int32), ("patience", C.c_int32), ("epoch_patience", C.c_int32),
                ("lbfgs_memory", C.c_int32), ("optimizer", C.c_int32), ("tol", C.c_double), ("f_tol", C.c_double),
                ("rho_beg", C.c_double)]


_BATCH_FN = C.CFUNCTYPE(C.c_int, C.POINTER(C.c_double), C.c_int32, C.POINTER(C.c_double), C.c_void_p)


class GvqeOptResult(C.Structure):
    _fields_ = [("E_best", C.c_double), ("energy_evals", C.c_int64), ("epochs", C.c_int32), ("n_blocks", C.c_int32),
                ("steps", C.c_int32), ("stop_reason", C.c_int32)]


class GvqeError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {msg}")
        self.status = status


_lib = None


def lib_path() -> str:
    return _build.SO


def load():
    """Load libgvqe.so (built in-tree on first use when nvcc is present).  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_build.SO) or (os.path.exists(_build.NVCC) and _build.needs_build()):
        _build.build()
    L = C.CDLL(_build.SO)
    vp, i32, u64, sz = C.c_void_p, C.c_int, C.c_uint64, C.c_size_t
    L.gvqe_create.argtypes = [i32, C.POINTER(GvqeLayout), i32, C.POINTER(vp)]
    L.gvqe_create_ops.argtypes = [i32, vp, i32, i32, i32, C.POINTER(vp)]
    L.gvqe_create_opt.argtypes = [i32, C.POINTER(GvqeLayout), i32, C.POINTER(GvqeOptions), C.POINTER(vp)]
    L.gvqe_create_ops_opt.argtypes = [i32, vp, i32, i32, i32, C.POINTER(GvqeOptions), C.POINTER(vp)]
    L.gvqe_kernel_source.argtypes = [vp, i32, C.c_char_p, sz, vp]
    L.gvqe_kernel_source.restype = sz
    L.gvqe_compile_kernels.argtypes = [vp, vp]
    L.gvqe_kernel_info.argtypes = [vp, i32, vp]
    L.gvqe_kernel_arrays.argtypes = [vp, i32, vp, sz]
    L.gvqe_kernel_arrays.restype = sz
    L.gvqe_num_params.argtypes = [vp]
    L.gvqe_num_qubits.argtypes = [vp]
    L.gvqe_set_hamiltonian.argtypes = [vp, i32, C.c_char_p, vp]
    L.gvqe_set_hamiltonian_masks.argtypes = [vp, i32, vp, vp, vp]
    L.gvqe_get_grouping.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.gvqe_workspace_bytes.argtypes = [vp, i32]
    L.gvqe_workspace_bytes.restype = sz
    L.gvqe_set_workspace.argtypes = [vp, vp, sz]
    L.gvqe_set_max_in_flight.argtypes = [vp, i32]
    L.gvqe_energy_batch.argtypes = [vp, vp, i32, vp, vp]
    L.gvqe_energy_batch_device.argtypes = [vp, vp, i32, vp, vp]
    L.gvqe_param_shift_grad.argtypes = [vp, vp, vp, vp, vp, vp]
    L.gvqe_get_state.argtypes = [vp, i32, vp]
    L.gvqe_argmax.argtypes = [vp, i32, vp, vp, vp]
    L.gvqe_argmax_noalloc.argtypes = [vp, u64, i32, vp, vp, C.c_char_p, sz]
    L.gvqe_sample.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    L.gvqe_measurement_settings.argtypes = [vp, vp, vp]
    L.gvqe_energy_shots.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    L.gvqe_schedule_info.argtypes = [vp, vp, vp, vp]
    L.gvqe_dump_schedule.argtypes = [vp, C.c_char_p, sz]
    L.gvqe_dump_schedule.restype = sz
    L.gvqe_get_exec_order.argtypes = [vp, vp, i32]
    L.gvqe_launch_count.argtypes = [vp]
    L.gvqe_launch_count.restype = u64
    L.gvqe_profile_enable.argtypes = [vp, i32]
    L.gvqe_profile_read.argtypes = [vp, vp]
    L.gvqe_profile_read_launches.argtypes = [vp, vp, vp, vp, i32]
    L.gvqe_interaction_graph.argtypes = [vp, vp]
    L.gvqe_modularity.argtypes = [i32, vp, vp, C.c_double, vp]
    L.gvqe_louvain.argtypes = [i32, vp, C.c_double, vp, vp, vp]
    L.gvqe_merge_small_blocks.argtypes = [i32, vp, i32, vp, vp]
    L.gvqe_block_param_mask.argtypes = [vp, vp, i32, vp]
    L.gvqe_geometric_blocks.argtypes = [i32, i32, i32, vp, vp]
    L.gvqe_graph_vqe_minimize.argtypes = [vp, C.POINTER(GvqeOptOptions), vp, vp, C.POINTER(GvqeOptResult), vp, i32, vp, vp]
    L.gvqe_cobyla_minimize.argtypes = [i32, vp, C.c_double, C.c_double, i32, _BATCH_FN, vp, vp, vp, vp]
    L.gvqe_last_error.argtypes = [vp]
    L.gvqe_last_error.restype = C.c_char_p
    L.gvqe_destroy.argtypes = [vp]
    L.gvqe_destroy.restype = None
    _lib = L
    return L


NOALLOC_MAX_AMPLITUDES = 1 << 34


def argmax_noalloc(state_ptr: int, n_amplitudes: int, precision: str, result_ptr: int, stream=None) -> None:
    """gvqe_argmax_noalloc: most probable basis state of the n_amplitudes complex numbers at DEVICE address state_ptr,
    written as {float64 prob, uint64 x} to DEVICE address result_ptr; allocates nothing, does not synchronise."""
    buf = C.create_string_buffer(256)
    st = load().gvqe_argmax_noalloc(C.c_void_p(state_ptr), int(n_amplitudes), {"c64": 0, "c128": 1}[precision],
                                    C.c_void_p(result_ptr), C.c_void_p(stream or 0), buf, len(buf))
    if st != 0:
        raise GvqeError(st, buf.value.decode())


_ENT = {"cz": 2, "cnot": 3}
_TOPO = {"linear": 0, "ring": 1, "full": 2, "reverse_linear": 3, "pairwise": 4, "circular": 5, "sca": 6}


class Gvqe:
    """One libgvqe context.  Method names mirror the C ABI without the gvqe_ prefix."""

    def __init__(self, n_qubits: int, *, layout: Optional[dict] = None, ops=None, n_params: Optional[int] = None,
                 precision: str = "c128", options: Optional[dict] = None):
        self._L = load()
        self._h = C.c_void_p()
        self._ws = None
        prec = {"c64": GVQE_C64, "c128": GVQE_C128}[precision]
        self.precision = precision
        opt = None
        if options:
            o_ = GvqeOptions()
            for k_, v_ in options.items():
                setattr(o_, k_, int(v_))   # unknown names raise AttributeError... ctypes structures accept only their fields
                if k_ not in dict(GvqeOptions._fields_):
                    raise GvqeError(GVQE_ERR_INVALID_ARG, f"unknown option {k_}")
            opt = C.byref(o_)
        if layout is not None:
            lay = GvqeLayout(int(layout["n_layers"]), _ENT.get(layout["entangler"], layout["entangler"]),
                             _TOPO.get(layout["topology"], layout["topology"]), int(layout.get("final_rot", 1)))
            st = self._L.gvqe_create_opt(n_qubits, C.byref(lay), prec, opt, C.byref(self._h))
        else:
            o = np.ascontiguousarray(np.asarray(ops, dtype=np.int32).reshape(-1, 4))
            st = self._L.gvqe_create_ops_opt(n_qubits, o.ctypes.data, len(o), int(n_params), prec, opt, C.byref(self._h))
        if st != GVQE_OK:
            raise GvqeError(st, "gvqe_create failed")
        self.n = n_qubits
        self.P = self._L.gvqe_num_params(self._h)

    # -- helpers
    def _check(self, st: int):
        if st != GVQE_OK:
            raise GvqeError(st, self._L.gvqe_last_error(self._h).decode())

    def close(self):
        if self._h:
            self._L.gvqe_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- C ABI
    def set_hamiltonian(self, paulis, coeffs):
        if not isinstance(paulis, (bytes, bytearray)):
            paulis = ("".join(paulis) if not isinstance(paulis, str) else paulis).encode("ascii")
        c = np.ascontiguousarray(coeffs, dtype=np.float64)
        if len(paulis) != len(c) * self.n:
            raise GvqeError(GVQE_ERR_INVALID_ARG, "paulis must hold n_terms * n_qubits characters")
        self._check(self._L.gvqe_set_hamiltonian(self._h, len(c), bytes(paulis), c.ctypes.data))

    def set_hamiltonian_masks(self, x_mask, z_mask, coeffs):
        x = np.ascontiguousarray(x_mask, dtype=np.uint64)
        z = np.ascontiguousarray(z_mask, dtype=np.uint64)
        c = np.ascontiguousarray(coeffs, dtype=np.float64)
        self._check(self._L.gvqe_set_hamiltonian_masks(self._h, len(c), x.ctypes.data, z.ctypes.data, c.ctypes.data))

    def get_grouping(self, n_terms: int):
        M = max(n_terms, 1)
        xm, zm = np.zeros(M, np.uint64), np.zeros(M, np.uint64)
        ny, got, gm = np.zeros(M, np.uint8), np.zeros(M, np.int32), np.zeros(M, np.uint64)
        ng = C.c_int32(0)
        self._check(self._L.gvqe_get_grouping(self._h, xm.ctypes.data, zm.ctypes.data, ny.ctypes.data, got.ctypes.data,
                                              C.addressof(ng), gm.ctypes.data))
        return xm[:n_terms], zm[:n_terms], ny[:n_terms], got[:n_terms], int(ng.value), gm[:ng.value]

    def workspace_bytes(self, batch_in_flight: int) -> int:
        return int(self._L.gvqe_workspace_bytes(self._h, int(batch_in_flight)))

    def set_workspace(self, device_ptr: int, nbytes: int):
        self._check(self._L.gvqe_set_workspace(self._h, C.c_void_p(device_ptr), nbytes))

    def set_max_in_flight(self, m: int):
        self._check(self._L.gvqe_set_max_in_flight(self._h, int(m)))

    def alloc_workspace(self, batch_in_flight: int, device="cuda:0"):
        """Convenience: a torch uint8 tensor of workspace_bytes(batch) on `device`, handed to set_workspace."""
        import torch

        nbytes = self.workspace_bytes(batch_in_flight)
        if nbytes == 0:
            raise GvqeError(GVQE_ERR_NO_HAMILTONIAN, "set the Hamiltonian before sizing the workspace")
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        ptr = (self._ws.data_ptr() + 255) & ~255
        self.set_workspace(ptr, nbytes)
        return self._ws

    def energy_batch(self, params, stream: int = 0, out: Optional[np.ndarray] = None) -> np.ndarray:
        p = np.ascontiguousarray(params, dtype=np.float64)
        if p.ndim == 1:
            p = p.reshape(1, -1) if self.P else p.reshape(len(p), 0)
        if p.shape[1] != self.P:
            raise GvqeError(GVQE_ERR_INVALID_ARG, f"params must be [B, {self.P}]")
        E = out if out is not None else np.empty(p.shape[0], dtype=np.float64)
        self._check(self._L.gvqe_energy_batch(self._h, p.ctypes.data, p.shape[0], E.ctypes.data, C.c_void_p(stream)))
        return E

    def energy_batch_ptr(self, params_host_ptr: int, B: int, E_host_ptr: int, stream: int = 0):
        """Raw host pointers (e.g. pinned torch tensors): no numpy marshalling in the timed path."""
        self._check(self._L.gvqe_energy_batch(self._h, C.c_void_p(params_host_ptr), B, C.c_void_p(E_host_ptr), C.c_void_p(stream)))

    def energy_batch_device(self, params_dev_ptr: int, B: int, E_dev_ptr: int, stream: int = 0):
        self._check(self._L.gvqe_energy_batch_device(self._h, C.c_void_p(params_dev_ptr), B, C.c_void_p(E_dev_ptr),
                                                     C.c_void_p(stream)))

    def param_shift_grad(self, params, mask, stream: int = 0):
        p = np.ascontiguousarray(params, dtype=np.float64).reshape(-1)
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
        if len(p) != self.P or len(m) != self.P:
            raise GvqeError(GVQE_ERR_INVALID_ARG, f"params and mask must have {self.P} entries")
        dE = np.zeros(max(self.P, 1), dtype=np.float64)
        E0 = C.c_double(0.0)
        self._check(self._L.gvqe_param_shift_grad(self._h, p.ctypes.data, m.ctypes.data, dE.ctypes.data, C.addressof(E0),
                                                  C.c_void_p(stream)))
        return dE[:self.P], E0.value

    def get_state(self, slot: int = 0) -> np.ndarray:
        dt = np.complex64 if self.precision == "c64" else np.complex128
        out = np.empty(1 << self.n, dtype=dt)
        self._check(self._L.gvqe_get_state(self._h, slot, out.ctypes.data))
        return out

    def argmax(self, slot: int = 0, stream: int = 0):
        """(x, |psi_x|^2) of the most probable basis state of in-flight slot `slot` (ties: lowest x)."""
        x, p = C.c_uint64(0), C.c_double(0.0)
        self._check(self._L.gvqe_argmax(self._h, int(slot), C.addressof(x), C.addressof(p), C.c_void_p(stream)))
        return int(x.value), p.value

    def sample(self, u, slot: int = 0, stream: int = 0):
        """(x[n_shots] uint64, Z): inverse-CDF samples of |psi|^2 in slot `slot` for the caller's uniforms u in [0,1)."""
        uu = np.ascontiguousarray(u, dtype=np.float64).reshape(-1)
        x = np.zeros(max(len(uu), 1), dtype=np.uint64)
        z = C.c_double(0.0)
        self._check(self._L.gvqe_sample(self._h, int(slot), len(uu), uu.ctypes.data, x.ctypes.data, C.addressof(z),
                                        C.c_void_p(stream)))
        return x[:len(uu)], z.value

    def measurement_settings(self, n_terms: int):
        """(n_settings, setting_of_term[n_terms]) of gvqe_measurement_settings."""
        ns = C.c_int32(0)
        got = np.zeros(max(n_terms, 1), dtype=np.int32)
        self._check(self._L.gvqe_measurement_settings(self._h, C.addressof(ns), got.ctypes.data))
        return int(ns.value), got[:n_terms]

    def energy_shots(self, u, n_terms: int, slot: int = 0, stream: int = 0):
        """(E_est, term_means[n_terms]) from u[n_settings, n_shots] uniforms in [0,1) (gvqe_energy_shots)."""
        uu = np.ascontiguousarray(u, dtype=np.float64)
        ns, _ = self.measurement_settings(n_terms)
        if uu.ndim != 2 or uu.shape[0] != ns:
            raise GvqeError(GVQE_ERR_INVALID_ARG, f"u must be [{ns}, n_shots]")
        E = C.c_double(0.0)
        means = np.zeros(max(n_terms, 1), dtype=np.float64)
        self._check(self._L.gvqe_energy_shots(self._h, int(slot), uu.shape[1], uu.ctypes.data, C.addressof(E), means.ctypes.data,
                                              C.c_void_p(stream)))
        return E.value, means[:n_terms]

    def schedule_info(self):
        a, b, c = C.c_int32(0), C.c_int32(0), C.c_int32(0)
        self._check(self._L.gvqe_schedule_info(self._h, C.addressof(a), C.addressof(b), C.addressof(c)))
        return a.value, b.value, c.value

    def dump_schedule(self) -> str:
        need = self._L.gvqe_dump_schedule(self._h, None, 0)
        buf = C.create_string_buffer(need + 1)
        self._L.gvqe_dump_schedule(self._h, buf, need + 1)
        return buf.value.decode()

    def kernel_source(self, block: int):
        """(source text, dynamic shared memory bytes) of the specialised kernel of fused block `block`, or None."""
        sm = C.c_int32(0)
        need = self._L.gvqe_kernel_source(self._h, int(block), None, 0, C.addressof(sm))
        if need == 0:
            return None
        buf = C.create_string_buffer(need + 1)
        self._L.gvqe_kernel_source(self._h, int(block), buf, need + 1, C.addressof(sm))
        return buf.value.decode(), int(sm.value)

    def kernel_info(self, block: int):
        """dict(kind='gate'|'expect', smem_bytes, fp_ops_per_amp) of specialised kernel `block`, or None."""
        o = np.zeros(4, dtype=np.float64)
        if self._L.gvqe_kernel_info(self._h, int(block), o.ctypes.data) != GVQE_OK:
            return None
        return dict(kind="gate" if o[0] == 0 else "expect", smem_bytes=int(o[1]), fp_ops_per_amp=float(o[2]))

    def kernel_arrays(self, which: int) -> np.ndarray:
        """Host image (uint8 array) of what the specialised expectation kernels read from global memory (gvqe_kernel_arrays)."""
        need = self._L.gvqe_kernel_arrays(self._h, int(which), None, 0)
        buf = np.zeros(max(need, 1), dtype=np.uint8)
        self._L.gvqe_kernel_arrays(self._h, int(which), buf.ctypes.data, need)
        return buf[:need]

    def compile_kernels(self) -> int:
        """NVRTC-compile every specialised kernel (no GPU needed); returns how many."""
        k = C.c_int32(0)
        self._check(self._L.gvqe_compile_kernels(self._h, C.addressof(k)))
        return int(k.value)

    def get_exec_order(self) -> np.ndarray:
        m = self._L.gvqe_get_exec_order(self._h, None, 0)
        o = np.zeros(max(m, 1), dtype=np.int32)
        self._L.gvqe_get_exec_order(self._h, o.ctypes.data, m)
        return o[:m]

    def profile_enable(self, on: bool):
        self._check(self._L.gvqe_profile_enable(self._h, 1 if on else 0))

    def profile_read(self) -> dict:
        o = np.zeros(8, dtype=np.float64)
        self._check(self._L.gvqe_profile_read(self._h, o.ctypes.data))
        keys = ["gate_ms", "gate_launches", "gate_bytes", "expect_ms", "expect_launches", "expect_bytes", "other_ms", "chunks"]
        return dict(zip(keys, o.tolist()))

    def profile_read_launches(self):
        """(mean_ms, min_ms, max_ms) arrays, one entry per launch of a chunk in execution order (see gvqe.h)."""
        m = self._L.gvqe_profile_read_launches(self._h, None, None, None, 0)
        a, b, c = (np.zeros(max(m, 1), dtype=np.float64) for _ in range(3))
        self._L.gvqe_profile_read_launches(self._h, a.ctypes.data, b.ctypes.data, c.ctypes.data, m)
        return a[:m], b[:m], c[:m]

    def launch_count(self) -> int:
        return int(self._L.gvqe_launch_count(self._h))

    # -- host-side Graph-VQE driver
    def interaction_graph(self) -> np.ndarray:
        w = np.zeros((self.n, self.n), dtype=np.float64)
        self._check(self._L.gvqe_interaction_graph(self._h, w.ctypes.data))
        return w

    def block_param_mask(self, community, block: int) -> np.ndarray:
        c = np.ascontiguousarray(community, dtype=np.int32)
        if len(c) != self.n:
            raise GvqeError(GVQE_ERR_INVALID_ARG, f"community must have {self.n} entries")
        m = np.zeros(max(self.P, 1), dtype=np.uint8)
        self._check(self._L.gvqe_block_param_mask(self._h, c.ctypes.data, int(block), m.ctypes.data))
        return m[:self.P]

    def graph_vqe_minimize(self, params, community, *, max_epochs=10, block_iters=50, global_iters=50, window=40,
                           patience=12, epoch_patience=3, lbfgs_memory=8, tol=1e-4, f_tol=1e-9, optimizer="lbfgs", rho_beg=0.0,
                           stream: int = 0):
        """Returns (params_best, result dict, history array).  Defaults are the paper's settings;
        optimizer: "lbfgs" or "cobyla"."""
        p = np.array(params, dtype=np.float64).reshape(-1)
        c = np.ascontiguousarray(community, dtype=np.int32)
        if len(p) != self.P or len(c) != self.n:
            raise GvqeError(GVQE_ERR_INVALID_ARG, "params / community size")
        opt = GvqeOptOptions(max_epochs, block_iters, global_iters, window, patience, epoch_patience, lbfgs_memory,
                             {"lbfgs": 0, "cobyla": 1}[optimizer], tol, f_tol, rho_beg)
        res = GvqeOptResult()
        hist = np.zeros(max_epochs + 1, dtype=np.float64)
        hl = C.c_int32(0)
        self._check(self._L.gvqe_graph_vqe_minimize(self._h, C.byref(opt), c.ctypes.data, p.ctypes.data, C.byref(res),
                                                    hist.ctypes.data, len(hist), C.addressof(hl), C.c_void_p(stream)))
        return p, {f: getattr(res, f) for f, _ in GvqeOptResult._fields_}, hist[:hl.value]


def _graph_check(st: int, what: str):
    if st != GVQE_OK:
        raise GvqeError(st, what)


def cobyla_minimize(fun, x0, rho_beg: float = 1.0, rho_end: float = 1e-4, max_evals: int = 1000):
    """gvqe_cobyla_minimize on a Python callable fun(rows[B, n]) -> values[B] (host only).  Returns (x, f_best, counts dict, reason)."""
    x = np.array(x0, dtype=np.float64).reshape(-1)
    n = len(x)

    def cb(rows, B, out, _user):
        try:
            pts = np.ctypeslib.as_array(rows, shape=(B * max(n, 1),))[:B * n].reshape(B, n)
            vals = np.asarray(fun(pts.copy()), dtype=np.float64).reshape(B)
            for b in range(B):
                out[b] = vals[b]
            return 0
        except Exception:
            return 1

    fb, reason = C.c_double(0.0), C.c_int32(0)
    counts = (C.c_int32 * 6)()
    _graph_check(load().gvqe_cobyla_minimize(n, x.ctypes.data, float(rho_beg), float(rho_end), int(max_evals), _BATCH_FN(cb), None,
                                             C.addressof(fb), counts, C.addressof(reason)), "gvqe_cobyla_minimize")
    names = ("evals", "trust_steps", "geometry_steps", "rho_reductions", "rebuilds", "improvements")
    return x, fb.value, dict(zip(names, list(counts))), reason.value


def modularity(w, community, gamma: float = 1.0) -> float:
    w = np.ascontiguousarray(w, dtype=np.float64)
    c = np.ascontiguousarray(community, dtype=np.int32)
    q = C.c_double(0.0)
    _graph_check(load().gvqe_modularity(w.shape[0], w.ctypes.data, c.ctypes.data, float(gamma), C.addressof(q)), "gvqe_modularity")
    return q.value


def louvain(w, gamma: float = 1.0):
    """(community[n], K, Q) of gvqe_louvain."""
    w = np.ascontiguousarray(w, dtype=np.float64)
    c = np.zeros(w.shape[0], dtype=np.int32)
    k, q = C.c_int32(0), C.c_double(0.0)
    _graph_check(load().gvqe_louvain(w.shape[0], w.ctypes.data, float(gamma), c.ctypes.data, C.addressof(k), C.addressof(q)), "gvqe_louvain")
    return c, k.value, q.value


def merge_small_blocks(w, community, s_min: int):
    w = np.ascontiguousarray(w, dtype=np.float64)
    c = np.array(community, dtype=np.int32)
    k = C.c_int32(0)
    _graph_check(load().gvqe_merge_small_blocks(w.shape[0], w.ctypes.data, int(s_min), c.ctypes.data, C.addressof(k)), "gvqe_merge_small_blocks")
    return c, k.value


def geometric_blocks(n: int, block_size: int, offset: int = 0):
    c = np.zeros(max(n, 1), dtype=np.int32)
    k = C.c_int32(0)
    _graph_check(load().gvqe_geometric_blocks(int(n), int(block_size), int(offset), c.ctypes.data, C.addressof(k)), "gvqe_geometric_blocks")
    return c[:n], k.value

"""CPU-only tests of the library's host side (no kernel runs): the C-ABI loads and exports every symbol of
include/gvqe.h, integer grouping is bit-exact against the oracle's independent routine, the schedule compiler
executes every op exactly once in an order that gives the same state (checked with the oracle), argument checks."""
import math
import os
import re

import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from workload import make_workload, CONFIGS
from workload.generator import random_ops, random_paulis

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    L = gv.load()
    hdr = open(os.path.join(ROOT, "include", "gvqe.h")).read()
    declared = set(re.findall(r"\b(gvqe_[a-z_]+)\s*\(", hdr))
    assert declared == set(gv.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_no_oracle_in_product():
    """The product never imports or links the oracle (and has no CPU fallback module)."""
    pkg = os.path.join(ROOT, "paper_2607_02749_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cpp", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "gvqe_oracle" not in src, f


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5, 6])
def test_grouping_bit_exact_vs_oracle(orc, cfg):
    c = CONFIGS[cfg]
    w = make_workload(cfg, D=1, batch=1)            # full-size Hamiltonian, tiny circuit
    g = gv.Gvqe(w.n, layout=dict(n_layers=1, entangler=w.entangler, topology=w.topology), precision="c128" if cfg in (1, 2, 6) else "c64")
    g.set_hamiltonian(w.paulis, w.coeffs)
    got = g.get_grouping(w.M)
    want = orc.grouping(w.n, w.paulis)
    assert got[4] == want[4]
    for a, b in zip(got[:4] + (got[5],), want[:4] + (want[5],)):
        assert a.dtype == b.dtype and a.tobytes() == b.tobytes()
    if c["pool"]:
        assert got[4] - 1 <= c["pool"]              # "<= 256 distinct flip masks"


def test_masks_api_equals_string_api(orc):
    n = 12
    paulis, coeffs = random_paulis(5, n, 100, 5)
    xm, zm, ny, got, ng, gm = orc.grouping(n, paulis)
    a = gv.Gvqe(n, layout=dict(n_layers=1, entangler="cz", topology="linear"))
    b = gv.Gvqe(n, layout=dict(n_layers=1, entangler="cz", topology="linear"))
    a.set_hamiltonian(paulis, coeffs)
    b.set_hamiltonian_masks(xm, zm, coeffs)
    for u, v in zip(a.get_grouping(100), b.get_grouping(100)):
        assert np.array_equal(u, v)


def _check_order(orc, n, ops, P, prec, seed, options=None):
    g = gv.Gvqe(n, ops=ops, n_params=P, precision=prec, options=options)
    order = g.get_exec_order()
    assert sorted(order.tolist()) == list(range(len(ops)))          # every op exactly once
    th = np.random.default_rng(seed).uniform(-math.pi, math.pi, max(P, 1))
    a = orc.state(n, ops, th)
    b = orc.state(n, np.asarray(ops)[order], th)                    # the device's order, run by the oracle
    assert np.max(np.abs(a - b)) < 1e-13


@pytest.mark.parametrize("seed", range(8))
def test_schedule_order_is_equivalent_random(orc, seed):
    n = 3 + seed
    ops, P = random_ops(40 + seed, n, 120)
    _check_order(orc, n, ops, P, "c64" if seed % 2 else "c128", seed)


@pytest.mark.parametrize("n,D,ent,topo,fr,prec", [(14, 3, "cz", "linear", 1, "c64"), (15, 3, "cnot", "ring", 1, "c64"),
                                                   (13, 2, "cnot", "linear", 2, "c128"), (16, 2, "cz", "ring", 2, "c128")])
def test_schedule_order_is_equivalent_layered(orc, n, D, ent, topo, fr, prec):
    from workload import layout_ops, num_params
    ops = np.array(layout_ops(n, D, ent, topo, fr), dtype=np.int32)
    # tile_bits = 10: several tiles and high-qubit blocks at small n
    _check_order(orc, n, ops, num_params(n, D, fr), prec, n, options=dict(tile_bits=10))


def test_layout_expansion_matches_generator():
    """gvqe_create(layout) builds the same op list as workload.layout_ops (readings A1-A5)."""
    from workload import layout_ops, num_params
    cases = [(6, 2, "cz", "linear", 1), (7, 3, "cnot", "ring", 2), (2, 1, "cnot", "ring", 1)]
    cases += [(n, 3, ent, topo, 1) for topo in ("full", "reverse_linear", "pairwise", "circular", "sca")
              for n, ent in ((5, "cnot"), (6, "cz"), (2, "cnot"))]
    for n, D, ent, topo, fr in cases:
        a = gv.Gvqe(n, layout=dict(n_layers=D, entangler=ent, topology=topo, final_rot=fr))
        b = gv.Gvqe(n, ops=np.array(layout_ops(n, D, ent, topo, fr), dtype=np.int32), n_params=num_params(n, D, fr))
        assert a.P == b.P == num_params(n, D, fr)
        assert a.dump_schedule() == b.dump_schedule()


def test_entangler_maps_by_hand():
    """Reading A17 written out for n = 4 (control, target)."""
    from workload.generator import entangler_pairs as ep
    assert ep(4, "full", 0) == [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    assert ep(4, "reverse_linear", 0) == [(2, 3), (1, 2), (0, 1)]
    assert ep(5, "pairwise", 0) == [(0, 1), (2, 3), (1, 2), (3, 4)]
    assert ep(4, "circular", 1) == [(3, 0), (0, 1), (1, 2), (2, 3)]
    assert ep(4, "ring", 1) == [(0, 1), (1, 2), (2, 3), (3, 0)]
    assert ep(4, "sca", 0) == [(3, 0), (0, 1), (1, 2), (2, 3)]
    assert ep(4, "sca", 1) == [(3, 2), (0, 3), (1, 0), (2, 1)]      # shifted by one, roles swapped
    assert ep(4, "sca", 2) == [(1, 2), (2, 3), (3, 0), (0, 1)]
    assert ep(2, "sca", 1) == [(0, 1)]


def test_large_configs_compile_and_plan():
    """Configs 4, 5a, 5b: schedule and pass plan exist, workspace arithmetic is 64-bit clean."""
    for cfg, prec in [(4, "c64"), (5, "c64"), (6, "c128")]:
        w = make_workload(cfg, batch=1)
        g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology), precision=prec)
        g.set_hamiltonian(w.paulis, w.coeffs)
        nb, npass, _ = g.schedule_info()
        assert nb >= 1 and npass >= 1
        s = (8 if prec == "c64" else 16) << w.n
        one, two = g.workspace_bytes(1), g.workspace_bytes(2)
        assert one > s * 1.5 and s <= two - one < s * 1.01 + (1 << 24)


def test_argument_errors():
    with pytest.raises(gv.GvqeError):
        gv.Gvqe(0, layout=dict(n_layers=1, entangler="cz", topology="linear"))
    with pytest.raises(gv.GvqeError):
        gv.Gvqe(35, layout=dict(n_layers=1, entangler="cz", topology="linear"))
    with pytest.raises(gv.GvqeError):   # parameter used twice
        gv.Gvqe(2, ops=np.array([[0, 0, -1, 0], [1, 1, -1, 0]], dtype=np.int32), n_params=1)
    with pytest.raises(gv.GvqeError):   # control == target
        gv.Gvqe(2, ops=np.array([[3, 1, 1, -1]], dtype=np.int32), n_params=0)
    g = gv.Gvqe(4, layout=dict(n_layers=1, entangler="cz", topology="linear"))
    assert g.workspace_bytes(1) == 0    # no Hamiltonian yet
    with pytest.raises(gv.GvqeError) as e:
        g.energy_batch(np.zeros((1, g.P)))
    assert e.value.status == gv.GVQE_ERR_NO_HAMILTONIAN
    with pytest.raises(gv.GvqeError) as e:
        g.set_hamiltonian(b"XQZI", [1.0])
    assert e.value.status == gv.GVQE_ERR_INVALID_ARG
    with pytest.raises(gv.GvqeError):
        g.set_hamiltonian(b"XZZI", [float("nan")])
    g.set_hamiltonian(b"XZZI" + b"IIII", [1.0, 2.0])
    with pytest.raises(gv.GvqeError) as e:
        g.energy_batch(np.zeros((1, g.P)))
    assert e.value.status == gv.GVQE_ERR_WORKSPACE
    with pytest.raises(gv.GvqeError):
        g.set_workspace(0, 1 << 20)
    with pytest.raises(gv.GvqeError):
        g.set_workspace(4096, 16)       # too small for one statevector


def test_no_environment_knobs_in_the_library():
    """SURVEY 5 "no global flags": schedule choices are gvqe_options fields, never environment variables."""
    csrc = os.path.join(ROOT, "paper_2607_02749_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_options_are_validated_and_change_the_schedule():
    lay = dict(n_layers=2, entangler="cnot", topology="ring")
    a = gv.Gvqe(14, layout=lay, precision="c64")
    b = gv.Gvqe(14, layout=lay, precision="c64", options=dict(tile_bits=10))
    assert "k=13" in a.dump_schedule() and "k=10" in b.dump_schedule()
    assert "prefix ops=0" in gv.Gvqe(14, layout=lay, precision="c64", options=dict(prefix=1)).dump_schedule()
    assert "prefix ops=0" not in gv.Gvqe(14, layout=lay, precision="c64", options=dict(prefix=2)).dump_schedule()
    # the first / last stage of a block goes straight to global memory unless staged_io = 1 asks for the staged copy
    spec = dict(specialise=2, prefix=1)
    direct = "".join(gv.Gvqe(16, layout=lay, precision="c64", options=spec).kernel_source(b)[0] for b in range(2))
    staged = "".join(gv.Gvqe(16, layout=lay, precision="c64", options=dict(spec, staged_io=1)).kernel_source(b)[0] for b in range(2))
    assert ("a_in[" in direct or "amp *gs =" in direct) and "a_in[" not in staged and "amp *gs =" not in staged
    assert "__launch_bounds__(256, 3)" in gv.Gvqe(16, layout=lay, precision="c64", options=dict(spec, blocks_per_sm=3)).kernel_source(0)[0]
    for bad in (dict(prefix=3), dict(specialise=-1), dict(tile_bits=40), dict(shared_prefix=7), dict(blocks_per_sm=4), dict(staged_io=2)):
        with pytest.raises(gv.GvqeError):
            gv.Gvqe(14, layout=lay, precision="c64", options=bad)
    with pytest.raises(gv.GvqeError):
        gv.Gvqe(14, layout=lay, options=dict(no_such_option=1))


@pytest.mark.parametrize("cfg,prec", [(3, "c64"), (3, "c128"), (4, "c64"), (5, "c64"), (6, "c128")])
def test_specialised_kernels_generate_and_compile(cfg, prec):
    """The bench configurations get one generated kernel per fused block (default from 20 qubits on); each compiles for
    sm_100a with NVRTC on this machine (no GPU needed), uses cp.async tile loads and fits two thread blocks per SM."""
    w = make_workload(cfg, M=40, batch=1)
    g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology), precision=prec)
    nb = g.schedule_info()[0] - (0 if "prefix ops=0" in g.dump_schedule() else 1)
    srcs = [g.kernel_source(b) for b in range(nb)]
    assert all(s is not None for s in srcs) and g.kernel_source(nb) is None
    for src, smem in srcs:
        assert "cp.async.cg.shared.global" in src and smem <= 113 * 1024
    try:
        assert g.compile_kernels() == nb
    except gv.GvqeError as e:
        if "libnvrtc not found" in str(e):
            pytest.skip("NVRTC is not installed here")
        raise
    # small registers keep the generic kernels unless asked
    assert gv.Gvqe(12, layout=dict(n_layers=1, entangler="cz", topology="linear")).kernel_source(0) is None


def test_kernel_info_counts_the_schedules_arithmetic():
    """gvqe_kernel_info: FP lane operations per amplitude of a generated gate kernel = 2 per rotation + 4 per complex
    table factor of its diagonal segments (the numerator of bench.py's ALU roofline): at least 2 x its rotations, and
    the blocks of one circuit together carry every R_y of the op list exactly once."""
    import re
    n, D = 20, 2
    g = gv.Gvqe(n, layout=dict(n_layers=D, entangler="cnot", topology="ring"), precision="c64", options=dict(prefix=1))
    nb = g.schedule_info()[0]
    blocks = re.split(r"\nblock ", g.dump_schedule())[1:nb + 1]
    total_ry = 0
    for b in range(nb):
        info = g.kernel_info(b)
        n_ry = blocks[b].count(" RY(")
        total_ry += n_ry
        assert info["kind"] == "gate" and info["smem_bytes"] == g.kernel_source(b)[1]
        assert info["fp_ops_per_amp"] >= 2.0 * n_ry and info["fp_ops_per_amp"] <= 2.0 * n_ry + 8.0 * (blocks[b].count(" DIAG(") + 1)
    assert total_ry == n * (D + 1) and g.kernel_info(nb) is None
    g.set_hamiltonian(["X" * 2 + "I" * (n - 2), "Z" * n], [0.5, 0.25])
    x = g.kernel_info(nb)
    assert x["kind"] == "expect" and x["fp_ops_per_amp"] > 0.0

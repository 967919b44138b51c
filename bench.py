#!/usr/bin/env python
"""bench.py -- VQE energy evaluations/s of libgvqe on one B200 (BASELINE.json metric), with the rooflines of its two
kernel classes and the CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..6] [--impl ours|reference] [--no-extra-configs]

A step = one gvqe_energy_batch call: the whole hot path (parameter expansion, every fused gate block, every
expectation pass, reduction) over one batch of synthetic parameter vectors of the configured workload.  Default
workload: BASELINE config 4 (28 qubits, complex64, 6 layers RY/RZ + CNOT ring, 20 000 Pauli terms, parameter-shift
sweep streamed 8 statevectors at a time).  At N = 1 the default run also measures the other large configurations
(5a: 32 qubits c64, 5b: 30 qubits c128, 3: 22 qubits c64) in the same process and reports them under "configs".
The path does not shard (replicas only): with --gpus N every rank runs the same workload on its own GPU
on different rows of the sweep, no collective in the data path.

Every fraction in the line is recomputable from the line: roofline.achieved = roofline.algorithmic_bytes_per_step /
(roofline.kernel_ms_per_step / 1e3) / 1e9, frac = achieved / peak; alu.achieved = alu.fp_ops_per_step /
(kernel_ms_per_step / 1e3) / 1e12, alu.peak = sm_count x lanes x sm_max_mhz.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "vqe_energy_evals_per_s"
UNIT = "evals/s"
PREC_OF = {1: "c128", 2: "c128", 3: "c64", 4: "c64", 5: "c64", 6: "c128"}
ROWS_PER_STEP = {1: 141, 2: 73, 3: 64, 4: 8, 5: 1, 6: 1}
# DRAM bytes per launch of the dominant kernel from one `ncu --set full` capture (dram__bytes_read.sum +
# dram__bytes_write.sum), with the committed summary it comes from; configs without a capture report null
TRAFFIC = {4: (34.36e9, "profiles/r02_gate_ncu_full.txt (one fused gate block over 8 statevectors: 17.18 GB read + 17.18 GB written)")}
SM_COUNT, FP32_LANES, FP64_LANES = 148, 128, 64   # per SM and clock (B200_PROFILING.md / MEASURED_PEAKS clocks)


def rows_for_step(n_rows_total, rows, world, rank, step):
    """Row indices (into the workload's parameter batch) that `rank` evaluates in step `step`: consecutive blocks of
    `rows` rows, rank-shifted so that the ranks of one step work on different rows, wrapping around the batch."""
    return (np.arange(rows) + (step * world + rank) * rows) % n_rows_total


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                o = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                    "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in o.strip().split(",")]
                if len(f) >= 6:
                    self.rows.append(f)
            except Exception:
                pass
            time.sleep(0.2)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": int(self.rows[0][1]) if self.rows[0][1].isdigit() else None, "reasons": reasons,
                "samples": len(self.rows)}


def oracle_sample(cfg, budget_rows=4, full_ops=False):
    """Time the CPU oracle (oracle/, as it stands) on a bounded sample of the workload; returns a dict with evals/s on
    all host cores, the same on one core, and a description.  Small configs: whole evaluations.  Large configs: T0's two
    loops are plain passes over the 2^n amplitudes per op / per term, so the cost is linear in both counts: `full_ops`
    runs EVERY op of the circuit once and 64 evenly spaced terms (else 24 ops and 8 terms), the rest is extrapolated
    linearly and labelled so; the one-core figure uses a smaller sample of the same kind."""
    import psutil
    import oracle
    from workload import make_workload

    oracle.build()
    cores = oracle.max_threads()
    w = make_workload(cfg, batch=1) if cfg >= 3 else make_workload(cfg)
    n, scale = w.n, 1.0
    if n <= 16:
        rows = w.params[:budget_rows]
        t0 = time.perf_counter()
        oracle.energy_batch(w.n, w.ops, rows, w.paulis, w.coeffs)
        dt = time.perf_counter() - t0
        oracle.set_threads(1)
        t0 = time.perf_counter()
        oracle.energy_batch(w.n, w.ops, rows[:1], w.paulis, w.coeffs)
        dt1 = time.perf_counter() - t0
        oracle.set_threads(cores)
        return {"value": len(rows) / dt, "cores": cores, "value_1core": 1.0 / dt1,
                "sample": f"{len(rows)} full evaluations of config {cfg} (T0, {w.M} terms), {dt:.2f} s; one core: 1 evaluation, {dt1:.2f} s"}
    avail = psutil.virtual_memory().available
    n_s = n
    while (24 << n_s) > 0.6 * avail and n_s > 20:
        n_s -= 1
    if n_s != n:
        scale = float(1 << (n - n_s))
        w = make_workload(cfg, n=n_s, batch=1)
    pl = w.pauli_list()

    def sample(k_ops, k_t):
        oi = np.linspace(0, len(w.ops) - 1, k_ops).astype(int) if k_ops < len(w.ops) else np.arange(len(w.ops))
        ti = np.linspace(0, w.M - 1, k_t).astype(int)
        sub_p = "".join(pl[i] for i in ti).encode()
        t0 = time.perf_counter()
        psi = oracle.state(w.n, w.ops[oi], w.params[0])
        t_ops = time.perf_counter() - t0
        t0 = time.perf_counter()
        oracle.energy_of_state(w.n, psi, sub_p, w.coeffs[ti])
        t_terms = time.perf_counter() - t0
        del psi
        return len(oi), t_ops, len(ti), t_terms, scale * (t_ops * len(w.ops) / len(oi) + t_terms * w.M / len(ti))

    k_ops, t_ops, k_t, t_terms, t_eval = sample(len(w.ops) if full_ops else 24, 64 if full_ops else 8)
    oracle.set_threads(1)
    k1o, t1o, k1t, t1t, t_eval1 = sample(4, 2)
    oracle.set_threads(cores)
    desc = (f"config {cfg}, oracle T0: {k_ops} of {len(w.ops)} ops ({t_ops:.2f} s) and {k_t} of {w.M} terms ({t_terms:.2f} s) at "
            f"{w.n} qubits on {cores} cores, extrapolated linearly in the term count"
            + ("" if k_ops == len(w.ops) else " and the op count") + " to one full evaluation"
            + (f" and x{scale:.0f} to {n} qubits" if scale > 1 else "")
            + f"; one core: {k1o} ops ({t1o:.2f} s) and {k1t} terms ({t1t:.2f} s), extrapolated the same way")
    return {"value": 1.0 / t_eval, "cores": cores, "value_1core": 1.0 / t_eval1, "sample": desc}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    vals = []
    last = None
    for _ in range(max(1, min(args.steps, 3))):
        last = oracle_sample(args.config, budget_rows=2)
        vals.append(last["value"])
    v = float(np.median(vals))
    rows = ROWS_PER_STEP[args.config]
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * rows / v, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(args.config),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(cfg):
    from workload import CONFIGS
    c = CONFIGS[cfg]
    return {"workload": f"BASELINE config {cfg if cfg < 5 else ('5a' if cfg == 5 else '5b')}: {c['n']} qubits, "
                        f"{PREC_OF[cfg]}, {c['D']} layers RY/RZ + {c['entangler'].upper()} {c['topology']}, "
                        f"{c['M']} Pauli terms", "rows_per_step": ROWS_PER_STEP[cfg], "precision": PREC_OF[cfg],
            "l2": "state buffers in flight exceed the 126 MB L2" if c["n"] >= 24 else "L2-resident working set (see DESIGN.md)",
            "parallelism": "replicas"}


def measure(cfg, args, options, rank, world, local, main):
    """One configuration: device-resident value, end-to-end value, per-kernel-class rooflines.  `main`: also the read-out
    sweep, the parameter-shift sweep and the clock samples."""
    import torch
    import torch.distributed as dist
    import paper_2607_02749_b200 as gv
    from workload import make_workload

    prec, rows = PREC_OF[cfg], ROWS_PER_STEP[cfg]
    if main and getattr(args, "rows", 0) > 0:
        rows = args.rows
    w = make_workload(cfg)
    g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology, final_rot=w.final_rot),
                precision=prec, options=options)
    g.set_hamiltonian(w.paulis, w.coeffs)
    g.alloc_workspace(rows, device=f"cuda:{local}")
    n_gate_blocks, n_passes, _ = g.schedule_info()
    stream = torch.cuda.Stream()
    steps = args.steps if main else min(args.steps, 3)
    total = args.warmup + steps

    def step_rows(i):   # each step takes the next `rows` rows of the sweep (rank-shifted), wrapping around
        return w.params[rows_for_step(w.B, rows, world, rank, i)]

    host_in = [torch.from_numpy(np.ascontiguousarray(step_rows(i))).pin_memory() for i in range(total)]
    host_out = torch.zeros(rows, dtype=torch.float64).pin_memory()
    dev_in = [t.cuda(non_blocking=True) for t in host_in]
    dev_out = torch.zeros(rows, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn):   # device time of exactly `steps` steps, max over ranks
        for i in range(args.warmup):
            fn(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(args.warmup, total):
            fn(i)
        e1.record(stream)
        barrier()
        ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item())

    g.energy_batch_device(dev_in[0].data_ptr(), rows, dev_out.data_ptr(), stream.cuda_stream)   # one-time set-up (tables,
    stream.synchronize()                                                                       # kernel compilation) is not a step
    sampler = ClockSampler(local) if main else None
    if sampler:
        sampler.start()
    l0 = g.launch_count()
    ms_dev = timed(lambda i: g.energy_batch_device(dev_in[i].data_ptr(), rows, dev_out.data_ptr(), stream.cuda_stream))
    launches = (g.launch_count() - l0) * steps // total
    if sampler:
        sampler.stop_flag = True
    ms_e2e = timed(lambda i: g.energy_batch_ptr(host_in[i].data_ptr(), rows, host_out.data_ptr(), stream.cuda_stream))
    # per-kernel-class device time (CUDA events inside the library, on the same stream), outside the timed region
    g.profile_enable(True)
    for i in range(args.warmup, total):
        g.energy_batch_device(dev_in[i].data_ptr(), rows, dev_out.data_ptr(), stream.cuda_stream)
    stream.synchronize()
    prof = g.profile_read()
    l_mean, l_min, l_max = g.profile_read_launches()
    g.profile_enable(False)
    chunks = max(prof["chunks"], 1.0)
    has_px = "prefix ops=0" not in g.dump_schedule()
    n_gate_launches = n_gate_blocks                       # product-state kernel included when the schedule has one
    gate_l = l_mean[:n_gate_launches]
    exp_l = l_mean[n_gate_launches:n_gate_launches + n_passes]
    # arithmetic of the specialised kernels (gvqe_kernel_info): FP lane operations per amplitude and launch
    amps = rows * float(2 ** w.n)
    ops_gate = ops_exp = 0.0
    k = 0
    while True:
        info = g.kernel_info(k)
        if info is None:
            break
        if info["kind"] == "gate":
            ops_gate += info["fp_ops_per_amp"] * amps
        else:
            ops_exp += info["fp_ops_per_amp"] * amps
        k += 1
    specialised = k > 0
    peak, sm_mhz, peak_src = peaks()
    lanes = FP32_LANES if prec == "c64" else FP64_LANES
    alu_peak = SM_COUNT * lanes * sm_mhz * 1e6 / 1e12
    gate_ms, exp_ms = prof["gate_ms"] / chunks, prof["expect_ms"] / chunks
    gate_bytes, exp_bytes = prof["gate_bytes"] / chunks, prof["expect_bytes"] / chunks
    gate_gbs = gate_bytes / (gate_ms * 1e-3) / 1e9 if gate_ms > 0 else 0.0
    exp_gbs = exp_bytes / (exp_ms * 1e-3) / 1e9 if exp_ms > 0 else 0.0
    tr = TRAFFIC.get(cfg)

    def alu(ops, ms):
        ok = ms > 0 and specialised
        return {"bound": "alu", "achieved": ops / (ms * 1e-3) / 1e12 if ok else None, "peak": alu_peak, "unit": "T lane-op/s",
                "fp_ops_per_step": ops if specialised else None, "frac": ops / (ms * 1e-3) / 1e12 / alu_peak if ok else None,
                "peak_source": f"{SM_COUNT} SMs x {lanes} lanes x {sm_mhz:.0f} MHz"}

    other_ms = prof["other_ms"] / chunks
    out = {
        "value": rows * world * steps / (ms_dev * 1e-3), "ms_per_step": ms_dev / steps, "steps": steps,
        "e2e": {"value": rows * world * steps / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": rows * w.P * 8,
                "d2h_bytes_per_step": rows * 8},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm",
                     "kernel": ("gvqe_block_* (schedule-specialised fused gate blocks" + (" + init_product_kernel)" if has_px else ")"))
                     if specialised else "gate_block_kernel", "achieved": gate_gbs, "peak": peak, "unit": "GB/s",
                     "frac": gate_gbs / peak, "frac_of_8TBs": gate_gbs / 8000.0,
                     "algorithmic_bytes_per_step": gate_bytes, "kernel_ms_per_step": gate_ms,
                     "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None, "peak_source": peak_src,
                     "launches_per_step": n_gate_launches, "avg_launch_ms": gate_ms / max(n_gate_launches, 1),
                     "launch_ms_min_max": [float(np.min(gate_l)), float(np.max(gate_l))] if len(gate_l) else None,
                     "launch_ms": [round(float(x), 3) for x in gate_l],
                     "share_of_step": gate_ms / max(gate_ms + exp_ms + other_ms, 1e-9), "alu": alu(ops_gate, gate_ms)},
        "expectation": {"kernel": "gvqe_expect_* (schedule-specialised passes)" if specialised else "expect_pass_kernel",
                        "bound": "alu" if specialised else "hbm", "achieved": exp_gbs, "unit": "GB/s", "frac": exp_gbs / peak,
                        "frac_of_8TBs": exp_gbs / 8000.0, "algorithmic_bytes_per_step": exp_bytes,
                        "kernel_ms_per_step": exp_ms, "launches_per_step": n_passes,
                        "avg_launch_ms": exp_ms / max(n_passes, 1), "launch_ms": [round(float(x), 3) for x in exp_l],
                        "share_of_step": exp_ms / max(gate_ms + exp_ms + other_ms, 1e-9), "alu": alu(ops_exp, exp_ms)},
    }
    if main:
        out["clocks"] = sampler.summary()
        # read-out sweep (gvqe_argmax: most probable bitstring of slot 0; S bytes read, result copied back and the stream
        # synchronised inside the call), outside the timed region, on the same stream
        for _ in range(3):
            g.argmax(0, stream.cuda_stream)
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_ro = 10
        r0.record(stream)
        for _ in range(n_ro):
            g.argmax(0, stream.cuda_stream)
        r1.record(stream)
        stream.synchronize()
        ro_ms = r0.elapsed_time(r1) / n_ro
        ro_gbs = (8 if prec == "c64" else 16) * 2.0 ** w.n / (ro_ms * 1e-3) / 1e9
        out["readout"] = {"kernel": "argmax_partial_kernel", "achieved": ro_gbs, "unit": "GB/s", "frac": ro_gbs / peak,
                          "ms_per_call": ro_ms, "note": "one state, includes the 16-byte D2H and the stream synchronise"}
        # whole parameter-shift sweep through gvqe_param_shift_grad (configs whose batch is a shift set): shared-prefix
        # evaluation, host buffers; one short untimed call first, then the measured one
        out["sweep"] = None
        if w.mask is not None:
            short = np.zeros_like(w.mask)
            short[:2] = 1
            g.param_shift_grad(w.theta, short, stream.cuda_stream)
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record(stream)
            g.param_shift_grad(w.theta, w.mask, stream.cuda_stream)
            s1.record(stream)
            stream.synchronize()
            n_ev = 2 * int(w.mask.sum()) + 1
            out["sweep"] = {"evaluations": n_ev, "seconds": s0.elapsed_time(s1) * 1e-3,
                            "evals_per_s": n_ev / (s0.elapsed_time(s1) * 1e-3), "api": "gvqe_param_shift_grad",
                            "shared_prefix": bool((8 if prec == "c64" else 16) * 2 ** max(w.n, 10) >= 16 << 20)}
    del g
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    options = {k: int(v) for k, v in (kv.split("=") for kv in args.opt)} or None   # gvqe_options overrides (tuning runs)
    cfg, prec = args.config, PREC_OF[args.config]
    m = measure(cfg, args, options, rank, world, local, main=True)
    extra = {}
    if world == 1 and cfg == 4 and not args.no_extra_configs:   # the other large configurations, same process, same protocol
        for c2, name in ((5, "5a"), (6, "5b"), (3, "3")):
            r = measure(c2, args, options, rank, world, local, main=False)
            r["config"] = workload_config(c2)
            r["dtype"] = "f32" if PREC_OF[c2] == "c64" else "f64"
            extra[name] = r
    if rank != 0:
        return
    cpu = oracle_sample(cfg, full_ops=True) if (world == 1 and not args.no_cpu_baseline) else None
    line = {
        "metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": m["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == "c64" else "f64", "data": "synthetic", "config": workload_config(cfg),
        "e2e": m["e2e"], "gpu_launches": m["gpu_launches"], "clocks": m["clocks"], "roofline": m["roofline"],
        "expectation": m["expectation"], "readout": m["readout"], "sweep": m["sweep"], "configs": extra or None,
        "cpu_baseline": {"value": cpu["value"] if cpu else None, "unit": UNIT, "cores": cpu["cores"] if cpu else 0, "kind": "oracle",
                         "sample": cpu["sample"] if cpu else "skipped", "value_1core": cpu["value_1core"] if cpu else None},
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--rows", type=int, default=0, help="statevectors in flight per step for --config (default: ROWS_PER_STEP)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra-configs", action="store_true", help="default config only: skip the 5a / 5b / 3 measurements")
    ap.add_argument("--opt", action="append", default=[], metavar="FIELD=INT",
                    help="gvqe_options field for this run (e.g. tiles_per_block=4, specialise=1); default: library defaults")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- throughput of the hot path (one explicit-implicit FD time step, all SURVEY 8(a)
rows) on BASELINE.json configs[4]: 8192 x 8192 fp64 nodes, config-2 physics, probe every 100.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

Prints ONE JSON line (rank 0).  metric = fp64 GCUPS (cell-updates/s) per FD time step.
A "step" is one solver step over the whole grid.  `value` is measured with the field resident
in HBM (CUDA events on the launch stream); `e2e` goes through the C ABI with pinned HOST
buffers (heat_set_field -> heat_step -> heat_get_field inside the timed region).
`--impl reference` times the CPU oracle (oracle/heat_oracle.c, as it stands) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "fp64 GCUPS (cell-updates/s) per FD time step"
UNIT = "GCUPS"
BYTES_PER_CELL = 16.0  # algorithmic: 8 B read of T^k + 8 B write of T^{k+1}
# fp64 thread-instructions (DFMA + DMUL + DADD) per cell-update, by kernel family, from the ncu counters
# smsp__sass_thread_inst_executed_op_d{fma,mul,add}_pred_on of the committed captures (profiles/*.md name
# them); a kernel without an entry gets no `roofline_alu` object rather than a guessed one
FP64_PER_CELL = {"tband<WL=16": 40.1, "band<G=256,CL=4": 48.0}
FP64_LANES = 148 * 64  # fp64 lanes of a B200 (64 per SM): the nominal ALU peak stated beside the measured one


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def load_traffic(kernel_name):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture
    (profiles/roofline_traffic.txt, key=value lines); None if the capture is of another kernel."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.txt")
    if os.path.exists(p):
        try:
            d = dict(l.strip().split("=", 1) for l in open(p) if "=" in l)
            if d.get("kernel") == kernel_name:
                return float(d["dram_bytes_per_launch"])
        except Exception:
            pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 7:
                    self.rows.append(f)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]),
                "power_w_max": max(float(r[2]) for r in self.rows), "reasons": reasons, "samples": len(self.rows)}


def make_spec(cfg, dt_fn):
    from paper_1408_5853_b200 import inputs as I
    s0 = I.config(cfg)
    return I.with_dt(s0, dt_fn(s0))


def oracle_sample(cfg, budget_s=12.0, variant="double"):
    """The oracle on a bounded sample of the workload: a z-slab of the config's grid (all nr
    radial nodes, fewer lines), same physics, same tau.  Returns (GCUPS, threads, description)."""
    from oracle.heat_oracle import Oracle, stable_dt
    from paper_1408_5853_b200 import inputs as I
    full = I.config(cfg)
    full = I.with_dt(full, stable_dt(full))
    nr, nz_full = full["nr"], full["nz"]
    nz = min(nz_full, max(18, int(4.0e6 // nr) + 2))
    s = dict(full)
    s["nz"] = nz
    s["z"] = full["z"][:nz].copy()
    s["batch"] = 1
    s["seg_layer"] = full["seg_layer"][:1]
    s["Q0"] = full["Q0"][:1]
    s["probes"] = [(nr - 1, nz // 2)] if full["probes"] else []
    o = Oracle(s, variant=variant)
    o.step(1)
    t0 = time.perf_counter()
    steps = 0
    while True:
        o.step(1)
        steps += 1
        el = time.perf_counter() - t0
        if el > budget_s or steps >= 64:
            break
    cells = nr * nz
    return cells * steps / el / 1e9, o.threads, f"{nr}x{nz}-node z-slab of config {cfg} ({steps} steps, {el:.1f} s)", el / steps


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # each "step" is one bounded oracle sample; K steps + W warm-ups, sized to end within minutes
    per = max(2.0, min(15.0, 150.0 / max(1, args.steps + args.warmup)))
    vals = []
    desc = ""
    cores = 1
    for k in range(args.warmup + args.steps):
        v, cores, desc, _ = oracle_sample(args.config, budget_s=per)
        if k >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    from paper_1408_5853_b200 import inputs as I
    s = I.config(args.config)
    cells = s["nr"] * s["nz"] * s["batch"]
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": cells / (value * 1e9) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config), "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def workload_name(cfg):
    return {0: "configs[0] 64x64 constant-coefficient cylinder", 1: "configs[1] 512x512 nonlinear 4-layer cell",
            2: "configs[2] 2048x2048 cell + 50 Hz pulse heating", 3: "configs[3] 256 x 512x512 parameter-sweep batch",
            4: "configs[4] 8192x8192 large-grid throughput, config-2 physics, probe every 100 steps"}[cfg]


def run_ours(args):
    import torch
    from paper_1408_5853_b200 import binding, build as B
    B.build()
    from paper_1408_5853_b200 import replicas as R
    rank, local, world = R.rank_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local)
    dist = R.init("nccl", local, world)  # replicas only: no data-path collective

    def barrier():
        R.barrier(dist, torch.cuda.synchronize)

    spec = make_spec(args.config, binding.heat_stable_dt)
    cells = spec["nr"] * spec["nz"] * spec["batch"]
    stream = torch.cuda.current_stream()
    sim = binding.HeatSim(spec, probe_records=max(16, (args.steps + args.warmup) // max(1, spec["probe_every"]) + 16))
    K, W = args.steps, args.warmup

    # ---- device-resident throughput: W warm-up steps, then exactly K steps between events
    sim.step(W)
    # the timed region must do everything a step can do, the probe write included: with few steps and
    # `probe_every` = 100 it would not cross a probe step, so move the step counter (not the field) to
    # K/2 + 1 steps before one.  The schedule of the BASELINE configs is the same there (source on).
    pe = int(spec["probe_every"]) if spec["probes"] else 0
    if pe > 1 and K < pe:
        sim.set_field(0, sim.field_device(0), (sim.step_index // pe + 1) * pe - K // 2 - 1) if spec["batch"] == 1 else None
    barrier()
    l0 = sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        e0.record(stream)
        sim.step(K)
        e1.record(stream)
        barrier()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count - l0
    ms_max = R.max_over_ranks(ms, dist, "cuda")
    value = R.job_gcups(cells, K, ms_max * 1e-3, world)
    probes, _ = sim.probes()
    field_ok = bool(torch.isfinite(sim.field_device(0)).all().item())

    # ---- end to end through the C ABI with pinned host buffers (per step: H2D field, step, D2H field)
    ke = max(1, min(K, args.e2e_steps))
    nzr = spec["nz"] * spec["nr"]
    host_in = torch.empty((spec["batch"], nzr), dtype=torch.float64).pin_memory()
    host_out = torch.empty((spec["batch"], nzr), dtype=torch.float64).pin_memory()
    L = binding.lib()
    import ctypes as C
    for b in range(spec["batch"]):
        L.heat_get_field(sim._h, b, C.c_void_p(host_in[b].data_ptr()), 0, sim._s())

    def e2e_step():
        k = sim.step_index
        for b in range(spec["batch"]):
            L.heat_set_field(sim._h, b, C.c_void_p(host_in[b].data_ptr()), 0, k, sim._s())
        L.heat_step(sim._h, 1, sim._s())
        for b in range(spec["batch"]):
            L.heat_get_field(sim._h, b, C.c_void_p(host_out[b].data_ptr()), 0, sim._s())

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value = R.job_gcups(cells, ke, R.max_over_ranks(e2e_s, dist, "cuda"), world)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = load_peaks()
    fp64_tflops = binding.heat_fp64_peak(1 << 15)           # measured DFMA rate of this GPU, this run
    fp64_per_cell = next((v for k, v in FP64_PER_CELL.items() if sim.kernel_name.startswith(k)), None)
    per_launch_ms = ms / max(1, launches)
    achieved = BYTES_PER_CELL * cells / (per_launch_ms * 1e-3) / 1e9
    traffic = load_traffic(sim.kernel_name)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, cores, desc, _ = oracle_sample(args.config, budget_s=12.0)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
        # second reported baseline: the same oracle, OpenMP over the lines j (bitwise the same result)
        try:
            v2, cores2, desc2, _ = oracle_sample(args.config, budget_s=6.0, variant="omp")
            cpu["omp"] = {"value": v2, "unit": UNIT, "cores": cores2, "sample": desc2}
        except Exception as ex:  # the OpenMP build is optional
            cpu["omp"] = {"unavailable": str(ex)[:120]}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config), "nr": spec["nr"], "nz": spec["nz"], "batch": spec["batch"],
                   "dt": spec["dt"], "kernel": sim.kernel_name,
                   "l2": "two 0.54 GB field levels ping-pong: inputs larger than the 126 MB L2, no flush needed"
                   if cells * 8 > 3e8 else "field fits L2 (L2-resident workload)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "finite": field_ok, "probe_records": int(probes.shape[0])},
        "algorithmic_GBps": value * BYTES_PER_CELL,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "peak_source": peak_src, "kernel": sim.kernel_name,
                     "bytes_per_launch": BYTES_PER_CELL * cells, "launch_ms": per_launch_ms},
        "roofline_alu": None if fp64_per_cell is None else {
            "bound": "alu", "achieved": achieved / BYTES_PER_CELL * fp64_per_cell, "unit": "G fp64 inst/s",
            "peak": fp64_tflops * 1e3 / 2.0, "frac": achieved / BYTES_PER_CELL * fp64_per_cell / (fp64_tflops * 1e3 / 2.0),
            "peak_source": "heat_fp64_peak in this run (%.1f TFLOP/s DFMA)" % fp64_tflops,
            "nominal_peak": FP64_LANES * (clk.summary()["sm_max_mhz"] or 1965.0) * 1e-3,
            "fp64_inst_per_cell": fp64_per_cell,
            "what": "co-limit: fp64 thread instructions per cell-update (ncu SASS counts of this kernel) against the measured DFMA issue rate"},
        "cpu_baseline": cpu,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * cells, "d2h_bytes_per_step": 8 * cells,
                "steps": ke, "what": "heat_set_field(host pinned) + heat_step(1) + heat_get_field(host pinned) per step"},
        "gpu_launches": int(launches),
        "clocks": clk.summary(),
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--e2e-steps", type=int, default=6)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

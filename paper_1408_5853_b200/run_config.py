"""Run one BASELINE.json workload at full length on the current CUDA device and write the probe
trace (the surface-temperature deliverable of configs 2-4).

    python -m paper_1408_5853_b200.run_config --config 2 --out gpurun_out/config2 [--steps N] [--every 10000]

Writes <out>_summary.txt (wall time, throughput, per-period extrema of the first probe of batch
member 0), <out>_trace.csv (every `--every`-th probe record of member 0) and, for a batch,
<out>_members.csv (one row per member: its parameters and the maximum / final probe value).  Only the C-ABI library is
used (heat_create / heat_step / heat_probe / heat_get_field through the binding).
"""
from __future__ import annotations

import argparse
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--steps", type=int, default=0, help="solver steps; 0 = the config's full length")
    ap.add_argument("--every", type=int, default=10000, help="trace downsampling for the csv")
    ap.add_argument("--out", default="gpurun_out/config")
    args = ap.parse_args()

    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)
    s0 = I.config(args.config)
    s = I.with_dt(s0, binding.heat_stable_dt(s0))
    total = args.steps if args.steps > 0 else int(s["steps"])
    P, nsub = int(s["steps_per_period"]), int(s["transient_substeps"])
    records = total // max(1, int(s["probe_every"])) + 16
    sim = binding.HeatSim(s, probe_records=records)
    cells = sim.nr * sim.nz * sim.batch
    print(f"config {args.config}: {sim.nr} x {sim.nz} x {sim.batch}, {total} solver steps, dt = {s['dt']:.6e} s, "
          f"{P} steps per period, kernel {sim.kernel_name}", flush=True)
    t0 = time.time()
    done, chunk = 0, 2_000_000
    while done < total:
        n = min(chunk, total - done)
        sim.step(n)
        sim.synchronize()
        done += n
        print(f"  {done} steps, {time.time() - t0:.0f} s", flush=True)
    el = time.time() - t0
    tr, dropped = sim.probes()
    T = sim.field(0)
    lines = [f"configs[{args.config}] on one B200: {total} solver steps in {el:.0f} s wall "
             f"({el / total * 1e6:.2f} us/step, {cells * total / el / 1e9:.1f} GCUPS), kernel {sim.kernel_name}",
             f"probe records {tr.shape[0]}, dropped {dropped}; field of member 0 finite {bool(np.isfinite(T).all())}, "
             f"min {T.min():.6f} K, max {T.max():.6f} K"]
    if tr.shape[0] and P > 0:
        t0p = tr[:, 0, 0]
        per = (P + max(nsub - 1, 0)) // max(1, int(s["probe_every"]))   # records per period (first step = nsub sub-steps)
        for n in range(0, (len(t0p) + per - 1) // per):
            seg = t0p[n * per:(n + 1) * per]
            lines.append(f"period {n}: probe 0 start {seg[0]:.6f} K, max {seg.max():.6f} K at record {int(np.argmax(seg))} "
                         f"of the period, end {seg[-1]:.6f} K")
    with open(args.out + "_summary.txt", "w") as f:
        f.write("\n".join(lines) + "\n")
    if tr.shape[0] and sim.batch > 1:
        # parameter sweep: one row per batch member (the design-sweep table of configs[3])
        cols = [np.arange(sim.batch), np.asarray(s["Q0"], dtype=np.float64)]
        names = ["member", "Q0"]
        if "heater_thickness_mm" in s:
            cols.append(np.asarray(s["heater_thickness_mm"], dtype=np.float64))
            names.append("heater_thickness_mm")
        cols += [tr[:, :, 0].max(axis=0), tr[-1, :, 0]]
        names += ["probe0_max_K", "probe0_end_K"]
        np.savetxt(args.out + "_members.csv", np.c_[tuple(cols)], delimiter=",", fmt="%.9g", header=",".join(names))
        k = int(np.argmax(cols[-2]))
        lines.append(f"batch of {sim.batch}: probe 0 maximum over the run from {cols[-2].min():.6f} K to {cols[-2].max():.6f} K "
                     f"(hottest member {k}: Q0 = {cols[1][k]:.4g})")
        with open(args.out + "_summary.txt", "w") as f:
            f.write("\n".join(lines) + "\n")
    if tr.shape[0]:
        idx = np.arange(0, tr.shape[0], max(1, args.every))
        np.savetxt(args.out + "_trace.csv", np.c_[idx, tr[idx, 0, :]], delimiter=",",
                   fmt=["%d"] + ["%.9f"] * tr.shape[2], header="record," + ",".join(f"probe{q}_K" for q in range(tr.shape[2])))
    print("\n".join(lines))
    sim.close()


if __name__ == "__main__":
    main()

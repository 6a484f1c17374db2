"""The switch-on of the source under the paper's sub-stepping trick, without it, and with iterations
(Fig. 3) on the current CUDA device.

    python -m paper_1408_5853_b200.switch_on --out gpurun_out/switch_on [--M 201]

The paper: an implicit scheme whose coefficients depend on the temperature needs
iterations at each time step; without them the discontinuous switch-on "can lead to a jump of the
temperature depending on the amplitude of the source (see Fig. 3b)"; a small enough time step avoids
it, and so does the paper's own remedy, the transient process (22) with 100 sub-steps of tau/100.
This runner puts the four side by side on `inputs.paper_device(M)` from the initial state
(T_0 = 4.2 K, source switched on at t = 0), through the C-ABI library only:
    A  the paper's scheme: transient model (22), 100 sub-steps, then steps of tau, no iterations
    B  Heaviside switch-on, steps of tau, no iterations               (what Fig. 3b warns about)
    C  Heaviside switch-on, steps of tau, `iters` iterations per step  (heat_step_picard, reading G23)
    D  Heaviside switch-on, steps of tau/100 throughout, no iterations (the "sufficiently small time-step")
and reports the temperature in the middle of the conducting layer and on the surface at z = 0 after
tau, 2 tau, 5 tau, 20 tau, 100 tau (the times of Fig. 3).  REPORTED, not asserted: Fig. 3 is an image
without numbers, and the radial grid and the graphite c_V coefficient are ours (inputs.paper_device).
"""
from __future__ import annotations

import argparse

import numpy as np

TIMES = (1, 2, 5, 20, 100)   # in units of tau


def run(binding, spec, plan):
    """plan: list of (steps, iters) chunks between the report times; returns [len(TIMES)][nprobes]."""
    sim = binding.HeatSim(spec, probe_records=4)
    out = []
    for steps, iters in plan:
        if iters > 1:
            sim.step_picard(steps, iters)
        else:
            sim.step(steps)
        F = sim.field(0)
        out.append([F[j, i] for (i, j) in spec["probes"]])
    name = sim.kernel_name
    sim.close()
    return np.array(out), name


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--M", type=int, default=201)
    ap.add_argument("--iters", type=int, nargs="*", default=[2, 4, 8])
    ap.add_argument("--out", default="gpurun_out/switch_on")
    args = ap.parse_args()

    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)

    base = I.paper_device(args.M)
    base["general_kernel"] = True
    seg = np.asarray(base["seg_layer"][0])
    heater = next(m for m, lay in enumerate(base["layers"]) if lay["is_heater"])
    nodes = np.flatnonzero(seg == heater)
    i_heat = int(nodes[len(nodes) // 2]) + 1
    base["probes"] = [(i_heat, 0), (base["nr"] - 1, 0)]
    base["probe_every"] = 10 ** 9
    nsub = int(base["transient_substeps"])
    dts = np.diff((0,) + TIMES)

    rows = {}
    # A: the first tau is nsub sub-steps, every later tau one step
    plan = [(nsub if k == 0 else int(d), 1) for k, d in enumerate(dts)]
    plan[0] = (nsub + int(dts[0]) - 1, 1)
    rows["A transient (22), 100 sub-steps"], kname = run(binding, dict(base), plan)
    heav = dict(base)
    heav["transient_substeps"] = 0
    rows["B Heaviside, one pass"], _ = run(binding, heav, [(int(d), 1) for d in dts])
    for it in args.iters:
        rows[f"C Heaviside, {it} iterations"], _ = run(binding, heav, [(int(d), it) for d in dts])
    fine = dict(heav)
    fine["dt"] = base["dt"] / 100.0
    fine["steps_per_period"], fine["steps_on"] = base["steps_per_period"] * 100, base["steps_on"] * 100
    rows["D Heaviside, tau/100 steps"], _ = run(binding, fine, [(int(d) * 100, 1) for d in dts])

    lines = [f"switch-on of the source on {base['name']} (tau = {base['dt']:g} s, kernel {kname}); "
             f"T [K] at z = 0 after t = " + ", ".join(f"{t} tau" for t in TIMES)]
    for p, label in enumerate((f"middle of the conducting layer (node {i_heat})", "surface r = r_max")):
        lines.append(f"  {label}")
        for name, v in rows.items():
            lines.append(f"    {name:34s} " + "  ".join(f"{x:9.5f}" for x in v[:, p]))
    ref = rows["D Heaviside, tau/100 steps"]
    lines.append("  largest difference to D over the five times and two nodes [K]")
    for name, v in rows.items():
        if not name.startswith("D"):
            lines.append(f"    {name:34s} {float(np.max(np.abs(v - ref))):.3e}")
    text = "\n".join(lines)
    print(text)
    import os
    os.makedirs(os.path.dirname(args.out) or ".", exist_ok=True)
    with open(args.out + "_summary.txt", "w") as f:
        f.write(text + "\n")


if __name__ == "__main__":
    main()

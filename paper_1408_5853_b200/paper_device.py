"""The paper's own device workload (arXiv 1408.5853 section 5) on the
current CUDA device.

    python -m paper_1408_5853_b200.paper_device --out gpurun_out/paper_device [--periods 400] [--timing]

Runs `inputs.paper_device(M)` (radii 0.12 / 0.125 / 0.13 / 0.1301 cm, z_max = 5 cm, POLY laws of Tables
2-3, chi(T) source, I_0 = 363 mA, tau = 1e-5 s, 25 ms / 1 ms, 100 transient sub-steps) through the
C-ABI library only, and writes <out>_summary.txt:
  * with --timing: microseconds per step on the grids of Table 4 (N = 631, M = 201 ... 1201,
    tau = 2.5e-7 s, t = 0 ... 0.025 s) beside the paper's 7.8 ms per step on a Tesla K40s;
  * the long run on 631 x 201: per period the surface temperature at (r_max, z = 0) just before
    switch-on and at switch-off (Fig. 7), and at the end the surface profile statistics of Fig. 8: mean
    surface temperature at switch-on / switch-off and the fraction of the surface z in [0, z_0 = 4 cm]
    above T_crit = 42.2 K at switch-off.
These are REPORTED beside the paper's qualitative statements (32 K <~ mean <~ 43.5 K, ~75 % of the
surface useful, ~10 s to the periodic regime), not asserted: the radial node distribution and the
graphite c_V coefficient are ours (see inputs.paper_device), so agreement can only be qualitative.
"""
from __future__ import annotations

import argparse
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--periods", type=int, default=400, help="source periods of the long run (400 = 10 s)")
    ap.add_argument("--M", type=int, default=201)
    ap.add_argument("--timing", action="store_true", help="also time the six grids of Table 4")
    ap.add_argument("--stepped", action="store_true",
                    help="the geometry of Fig. 1: layers 1-3 end at z_0 = 4 cm, the core goes on to the terminal (row f2, reading G24)")
    ap.add_argument("--out", default="gpurun_out/paper_device")
    args = ap.parse_args()

    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)
    lines = []

    if args.timing:
        lines.append("Table 4 grids (N = 631, tau = 2.5e-7 s, t = 0 .. 0.025 s = 100 099 solver steps); "
                     "paper: 12.9-14.1 min = 7.8 ms/step on a Tesla K40s, 13.0-64.0 min on a Xeon E5-2695 (P:L326-331)")
        for M in (201, 401, 601, 801, 1001, 1201):
            s = I.paper_device(M, tau=2.5e-7)
            sim = binding.HeatSim(s, probe_records=16)
            n = int(s["steps_per_period"]) + 99
            sim.step(200)
            sim.synchronize()
            t0 = time.time()
            sim.step(n)
            sim.synchronize()
            el = time.time() - t0
            T = sim.field(0)
            lines.append(f"  631 x {M}: {n} steps in {el:.2f} s = {el / n * 1e6:.2f} us/step "
                         f"({631 * M * n / el / 1e9:.2f} GCUPS), kernel {sim.kernel_name}, T in [{T.min():.3f}, {T.max():.3f}] K")
            print(lines[-1], flush=True)
            sim.close()

    s = I.paper_device(args.M, stepped=args.stepped)
    P, nsub, S = int(s["steps_per_period"]), int(s["transient_substeps"]), int(s["steps_on"])
    per = P - 1 + nsub                       # solver steps per period
    on_steps = nsub + S - 1                  # solver steps until the source switches off
    sim = binding.HeatSim(s, probe_records=16)
    nr, nz = sim.nr, sim.nz
    z = np.asarray(s["z"])
    work = z <= 4.0 + 1e-12                  # working surface z in [0, z_0], P:L314 (z_0 = 4 cm, reading G10)
    lines.append(f"long run: {s['name']}, {nr} x {nz}, tau = {s['dt']:.1e} s, {per} solver steps per period, kernel {sim.kernel_name}")
    t0 = time.time()
    rows = []
    for n in range(args.periods):
        surf_on = sim.field(0)[:, nr - 1].copy()       # just before switch-on
        sim.step(on_steps)
        surf_off = sim.field(0)[:, nr - 1].copy()      # at switch-off
        sim.step(per - on_steps)
        rows.append((n, surf_on[0], surf_off[0], surf_on[work].mean(), surf_off[work].mean(),
                     float(np.mean(surf_off[work] > I.PAPER_TCRIT))))
        if n % 50 == 0 or n == args.periods - 1:
            print(f"period {n}: T(r_max, 0) {rows[-1][1]:.3f} -> {rows[-1][2]:.3f} K, surface mean {rows[-1][3]:.3f} -> "
                  f"{rows[-1][4]:.3f} K, above T_crit {100 * rows[-1][5]:.1f} %  ({time.time() - t0:.0f} s)", flush=True)
    el = time.time() - t0
    sim.probes()
    T = sim.field(0)
    rows = np.array(rows)
    np.savetxt(args.out + "_periods.csv", rows, delimiter=",", fmt="%.9g",
               header="period,T_rmax_z0_before_on_K,T_rmax_z0_at_off_K,surface_mean_before_on_K,surface_mean_at_off_K,fraction_above_Tcrit_at_off")
    lines.append(f"  {args.periods} periods = {args.periods * per} solver steps in {el:.0f} s wall (incl. two field read-backs per period), "
                 f"field finite {bool(np.isfinite(T).all())}, T in [{T.min():.3f}, {T.max():.3f}] K")
    last = rows[-1]
    lines.append(f"  last period: T(r_max, z=0) swings {last[1]:.2f} -> {last[2]:.2f} K (Fig. 7); mean surface temperature "
                 f"{last[3]:.2f} -> {last[4]:.2f} K (paper: 32 <~ T <~ 43.5 K, P:L341); {100 * last[5]:.0f} % of the working surface "
                 f"above T_crit = {I.PAPER_TCRIT} K at switch-off (paper: ~75 %, P:L318)")
    drift = abs(rows[-1][4] - rows[max(0, len(rows) - 41)][4])
    lines.append(f"  change of the switch-off surface mean over the last 40 periods (1 s): {drift:.3f} K "
                 f"(paper: periodic regime after ~10 s, P:L312)")
    with open(args.out + "_summary.txt", "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))
    sim.close()


if __name__ == "__main__":
    main()

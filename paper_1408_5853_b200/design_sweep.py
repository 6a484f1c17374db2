"""Design sweep / source-control loop on the paper's device ("can be formulated
mathematically as source control problem").

    python -m paper_1408_5853_b200.design_sweep --out gpurun_out/design_sweep [--generations 3] [--batch 16]

The paper's outlook: choose the current amplitude I_0 (and the thickness of the conducting layer) so that
at switch-off as much of the working surface z in [0, z_0] as possible is above T_crit = 42.2 K, while
just before the next switch-on the whole surface is below it again (the working gas must condense between
pulses).  Objective (to maximise):

    J = fraction of the working surface above T_crit at switch-off      if max T_surface before switch-on < T_crit
      = -(max T_surface before switch-on - T_crit) / T_crit             otherwise (infeasible: never cools down)

The loop: a generation is ONE batch run of the library (every member its own I_0 and heater thickness,
advanced together by heat_step, SURVEY config-3 engine) over `--periods` source periods; the next
generation samples a box around the best member, shrunk by `--shrink`.  Deterministic (seeded).
Everything numerical runs in the CUDA kernels through the C ABI; this file only picks parameters and
reads the surface line of each member.  The horizon is short by default (40 periods = 1 s of the ~10 s
the device needs to settle), so J is an early indicator; `--periods 400` gives the settled value.
"""
from __future__ import annotations

import argparse
import time

import numpy as np

I0_RANGE = (0.25, 0.60)          # A; the paper's device runs at 0.363 A
THICK_RANGE = (10, 190)          # heater thickness in radial steps of 5e-5 cm of the u = 10 grid (paper: 100 = 5e-3 cm)


def objective(frac_above_at_off: float, max_before_on: float, tcrit: float) -> float:
    return float(frac_above_at_off) if max_before_on < tcrit else -float(max_before_on - tcrit) / tcrit


def first_generation(batch: int, rng: np.random.Generator):
    """The paper's design point first, then a seeded latin-hypercube-like spread over the box."""
    i0 = np.concatenate([[0.363], I0_RANGE[0] + (I0_RANGE[1] - I0_RANGE[0]) * (rng.permutation(batch - 1) + rng.random(batch - 1)) / (batch - 1)])
    th = np.concatenate([[100], np.rint(THICK_RANGE[0] + (THICK_RANGE[1] - THICK_RANGE[0]) * (rng.permutation(batch - 1) + rng.random(batch - 1)) / (batch - 1))])
    return i0, th.astype(int)


def next_generation(i0, th, J, gen: int, shrink: float, rng: np.random.Generator):
    """Keep the best member, sample the others in a box around it whose half-widths shrink by `shrink`
    per generation; clipped to the admissible ranges."""
    k = int(np.argmax(J))
    wi = 0.5 * (I0_RANGE[1] - I0_RANGE[0]) * shrink ** (gen + 1)
    wt = 0.5 * (THICK_RANGE[1] - THICK_RANGE[0]) * shrink ** (gen + 1)
    n = len(i0)
    ni = np.clip(i0[k] + wi * (2 * rng.random(n) - 1), *I0_RANGE)
    nt = np.clip(np.rint(th[k] + wt * (2 * rng.random(n) - 1)), *THICK_RANGE).astype(int)
    ni[0], nt[0] = i0[k], th[k]
    return ni, nt


def device_batch(i0, th, M, nr=631):
    """inputs.paper_device for a batch: member b has current amplitude i0[b] and a conducting layer of
    th[b] radial steps ending at r_2 (its inner interface moves, the insulator under it takes the rest)."""
    from . import inputs as I
    s = I.paper_device(M, nr=nr)
    u = (nr - 1) // 63
    n_core, n2_end = 42 * u, 42 * u + 20 * u
    segs = []
    for t in th:
        t = int(t) * u // 10 if u != 10 else int(t)
        inner = n2_end - max(2, min(20 * u - 2, t))       # node of the insulator / conductor interface
        segs.append(I.seg_layers(nr, [n_core, inner, n2_end]))
    r = s["r"]
    s["batch"] = len(i0)
    s["seg_layer"] = np.stack(segs)
    # X = chi(T) I^2 / S_2^2 with S_2 the cross-section of THIS member's conducting layer (2),(3) P:L70-76
    r_in = np.array([r[np.flatnonzero(np.diff(sg.astype(int)))[1] + 1] for sg in segs])
    S2 = np.pi * (I.PAPER_RADII_CM[2] ** 2 - r_in ** 2)
    s["Q0"] = I.PAPER_CHI0 * np.asarray(i0) ** 2 / S2 ** 2
    s["probes"] = []
    return s


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--generations", type=int, default=3)
    ap.add_argument("--batch", type=int, default=16)
    ap.add_argument("--periods", type=int, default=40)
    ap.add_argument("--M", type=int, default=101)
    ap.add_argument("--shrink", type=float, default=0.45)
    ap.add_argument("--seed", type=int, default=14085853)
    ap.add_argument("--out", default="gpurun_out/design_sweep")
    args = ap.parse_args()

    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)
    rng = np.random.Generator(np.random.PCG64(args.seed))
    i0, th = first_generation(args.batch, rng)
    rows, lines = [], []
    t0 = time.time()
    for gen in range(args.generations):
        s = device_batch(i0, th, args.M)
        sim = binding.HeatSim(s)
        nr = sim.nr
        work = np.asarray(s["z"]) <= 4.0 + 1e-12
        P, nsub, S = int(s["steps_per_period"]), int(s["transient_substeps"]), int(s["steps_on"])
        per, on_steps = P - 1 + nsub, nsub + S - 1
        sim.step((args.periods - 1) * per)
        before = np.stack([sim.field(b)[:, nr - 1] for b in range(sim.batch)])   # just before the last switch-on
        sim.step(on_steps)
        at_off = np.stack([sim.field(b)[:, nr - 1] for b in range(sim.batch)])   # at switch-off
        J = np.array([objective(np.mean(at_off[b, work] > I.PAPER_TCRIT), before[b, work].max(), I.PAPER_TCRIT) for b in range(sim.batch)])
        for b in range(sim.batch):
            rows.append((gen, b, i0[b], th[b] * 5e-5, J[b], np.mean(at_off[b, work] > I.PAPER_TCRIT), before[b, work].max(), at_off[b, work].mean()))
        k = int(np.argmax(J))
        lines.append(f"generation {gen}: best member {k}: I_0 = {i0[k] * 1e3:.1f} mA, thickness {th[k] * 5e-5 * 1e4:.1f} um, J = {J[k]:.3f} "
                     f"(surface above T_crit at switch-off {100 * rows[-sim.batch + k][5]:.0f} %, max before switch-on {rows[-sim.batch + k][6]:.2f} K); "
                     f"paper's design point (gen 0, member 0): J = {rows[0][4]:.3f}; kernel {sim.kernel_name}; {time.time() - t0:.0f} s")
        print(lines[-1], flush=True)
        sim.close()
        i0, th = next_generation(i0, th, J, gen, args.shrink, rng)
    np.savetxt(args.out + "_members.csv", np.array(rows), delimiter=",", fmt="%.9g",
               header="generation,member,I0_A,heater_thickness_cm,J,fraction_above_Tcrit_at_off,max_surface_before_on_K,mean_surface_at_off_K")
    with open(args.out + "_summary.txt", "w") as f:
        f.write(f"design sweep on the paper's device, 631 x {args.M}, {args.batch} members x {args.generations} generations x {args.periods} periods\n")
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()

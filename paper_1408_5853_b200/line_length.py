"""Throughput of the time step against the line length at a fixed number of cells (DESIGN.md section 6,
profiles/r02_line_length.md): config-2 physics on nr x nz grids with nr * nz = 2^26, through the C ABI.

    python -m paper_1408_5853_b200.line_length [--steps 100] [--sizes 8192x8192 4096x16384 ...]

HEAT_TBAND_NW in the environment selects the warps per CTA (e.g. clusters instead of one CTA per line).
"""
from __future__ import annotations

import argparse


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--sizes", nargs="*", default=["8192x8192", "4096x16384", "2048x32768", "1024x65536", "512x131072"])
    args = ap.parse_args()
    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)
    for size in args.sizes:
        nr, nz = (int(v) for v in size.split("x"))
        s = I.config(4, nr=nr, nz=nz)
        s = I.with_dt(s, binding.heat_stable_dt(s))
        sim = binding.HeatSim(s, probe_records=64)
        sim.step(5)
        sim.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(sim.stream)
        sim.step(args.steps)
        e1.record(sim.stream)
        sim.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        print(f"{nr} x {nz}  {sim.kernel_name}: {ms * 1e3:.1f} us/step, {nr * nz / ms / 1e6:.1f} GCUPS", flush=True)
        sim.close()


if __name__ == "__main__":
    main()

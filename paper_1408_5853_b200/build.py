"""Build paper_1408_5853_b200/libheat_b200.so (the C-ABI library of include/heat.h) in-tree.

    python -m paper_1408_5853_b200.build [--force]

nvcc cross-compiles for sm_100a without a GPU.  The .so is git-ignored but travels to the
GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libheat_b200.so")
def _c(*names):
    return [os.path.join(CSRC, n) for n in names]


HEAT_H = os.path.join(ROOT, "include", "heat.h")
# translation unit -> the files it is built from
UNITS = {
    "heat_api.cu": _c("heat_api.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                      "heat_line_variants.h", "heat_band_params.cuh", "heat_band_variants.h",
                      "heat_wband_params.cuh", "heat_wband_variants.h", "heat_tband_variants.h") + [HEAT_H],
    "heat_line_a.cu": _c("heat_line_a.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                         "heat_line_variants.h"),
    "heat_line_b.cu": _c("heat_line_b.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                         "heat_line_variants.h"),
    "heat_tma.cu": _c("heat_tma.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                      "heat_line_variants.h"),
    "heat_band.cu": _c("heat_band.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                       "heat_band_params.cuh", "heat_band_variants.h", "heat_band_kernel.cuh"),
    "heat_wband2.cu": _c("heat_wband2.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                         "heat_band_params.cuh", "heat_band_kernel.cuh", "heat_wband_params.cuh",
                         "heat_wband_variants.h", "heat_wband_kernel.cuh"),
    "heat_wband4.cu": _c("heat_wband4.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                         "heat_band_params.cuh", "heat_band_kernel.cuh", "heat_wband_params.cuh",
                         "heat_wband_variants.h", "heat_wband_kernel.cuh"),
    "heat_tband2.cu": _c("heat_tband2.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                         "heat_band_params.cuh", "heat_band_kernel.cuh", "heat_wband_params.cuh",
                         "heat_wband_kernel.cuh", "heat_tband_variants.h", "heat_tband_kernel.cuh"),
    "heat_tband4.cu": _c("heat_tband4.cu", "heat_device.cuh", "heat_line_kernel.cuh", "heat_tma_kernel.cuh",
                         "heat_band_params.cuh", "heat_band_kernel.cuh", "heat_wband_params.cuh",
                         "heat_wband_kernel.cuh", "heat_tband_variants.h", "heat_tband_kernel.cuh"),
}
SOURCES = _c(*UNITS)
DEPS = sorted({d for deps in UNITS.values() for d in deps})
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if any source is newer than it; return its path.  The translation
    units are compiled side by side (nvcc -c), then linked into one shared object."""
    if not force and up_to_date():
        return LIB
    objs = [os.path.splitext(src)[0] + ".o" for src in SOURCES]
    cmds = []
    for (unit, deps), src, obj in zip(UNITS.items(), SOURCES, objs):
        stale = force or not os.path.exists(obj) or any(os.path.getmtime(d) > os.path.getmtime(obj) for d in deps)
        if stale:
            cmds.append([nvcc(), *NVCC_FLAGS, "-c", "-o", obj, src])
    procs = [subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for cmd in cmds]
    log = ""
    failed = False
    for cmd, pr in zip(cmds, procs):
        out, _ = pr.communicate()
        log += " ".join(cmd) + "\n" + out
        failed = failed or pr.returncode != 0
    if not failed:
        link = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB, *objs]
        res = subprocess.run(link, capture_output=True, text=True)
        log += " ".join(link) + "\n" + res.stdout + res.stderr
        failed = res.returncode != 0
    with open(os.path.join(HERE, "build.log"), "w") as f:
        f.write(log)
    if failed:
        raise RuntimeError("nvcc failed:\n" + log[-4000:])
    if verbose:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

"""CPU-side checks of the C-ABI boundary (include/heat.h): the library builds, loads and
exports every declared symbol; host-only entry points (heat_stable_dt, heat_workspace_bytes,
descriptor validation in heat_create) behave as documented.  No compute call needs a GPU here.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1408_5853_b200 import build as B
from paper_1408_5853_b200 import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    B.build()
    from paper_1408_5853_b200 import binding as bd
    bd.lib()
    return bd


def test_header_symbols_are_exported(binding):
    """Every function include/heat.h declares is exported by libheat_b200.so, and the binding
    lists the same names."""
    text = open(os.path.join(ROOT, "include", "heat.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(heat_[a-z0-9_]+)\s*\(", text))
    assert declared, "no declarations parsed"
    L = C.CDLL(binding.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), f"{name} declared in heat.h but not exported"
    assert declared == set(binding.EXPORTS)


def test_struct_layout_matches_header(binding):
    """sizeof of the ctypes mirrors equals what the C compiler lays out (probed with gcc)."""
    import subprocess
    import tempfile
    src = '#include "heat.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu %zu\\n",sizeof(heat_law),sizeof(heat_layer),sizeof(heat_bc),sizeof(heat_desc));return 0;}\n'
    with tempfile.TemporaryDirectory() as td:
        c = os.path.join(td, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(td, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        sizes = [int(x) for x in subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()]
    assert sizes == [C.sizeof(binding.heat_law), C.sizeof(binding.heat_layer), C.sizeof(binding.heat_bc),
                     C.sizeof(binding.heat_desc)]


def test_stable_dt_matches_the_oracle(binding):
    """(21) P:L194-196 through the C ABI (host-only) against the oracle's own evaluation."""
    from oracle.heat_oracle import stable_dt
    for n, kw in ((0, {}), (1, dict(nr=64, nz=48)), (2, dict(nr=40, nz=24)), (4, dict(nr=128, nz=96))):
        s = I.config(n, **kw)
        assert binding.heat_stable_dt(s) == pytest.approx(stable_dt(s), rel=1e-13)
    s = I.random_spec(3, laws="mixed")
    assert binding.heat_stable_dt(s) == pytest.approx(stable_dt(s), rel=1e-13)


def test_workspace_bytes_and_validation(binding):
    s = I.with_dt(I.config(1, nr=64, nz=32), 1e-6)
    assert binding.heat_workspace_bytes(s) > 0
    bad = dict(s, r=s["r"][::-1].copy())
    assert binding.heat_workspace_bytes(bad) == 0          # r not ascending
    bad = dict(s, dt=-1.0)
    assert binding.heat_workspace_bytes(bad) == 0
    seg = s["seg_layer"].copy()
    seg[0, 10], seg[0, 11] = 3, 0                            # two adjacent interface nodes
    assert binding.heat_workspace_bytes(dict(s, seg_layer=seg)) == 0


def _create(binding, spec, fa=16, fb=32, ws=256):
    m = binding.Desc(spec)
    h = C.c_void_p()
    st = binding.lib().heat_create(C.byref(m.desc), fa, fb, ws, 1 << 40, None, 0, None, C.byref(h))
    return st, binding.lib().heat_last_error(None).decode(), h


def test_create_rejects_bad_descriptors_before_touching_the_device(binding):
    s = I.with_dt(I.config(1, nr=64, nz=32), 1e-6)
    st, msg, h = _create(binding, dict(s, steps_per_period=5, steps_on=9))
    assert st == binding.HEAT_EINVAL and "steps_on" in msg and not h.value
    st, msg, h = _create(binding, dict(s, probes=[(64, 3)]))
    assert st == binding.HEAT_EINVAL and "probe" in msg
    st, msg, h = _create(binding, s, fa=0)
    assert st == binding.HEAT_EINVAL
    st, msg, h = _create(binding, s, fa=24)                  # misaligned
    assert st == binding.HEAT_EINVAL and "aligned" in msg


def test_create_rejects_non_positive_laws(binding):
    """HEAT_ERANGE: the paper's printed graphite c_V row (Table 2, m = 2) has a root
    near 22 K and is negative above it (G11) -- heat_create must refuse it."""
    g = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_tables_2_3.txt")):
        f = line.split()
        if f and f[0] in ("cv", "lam"):
            g[(f[0], int(f[1]))] = [float(x) for x in f[2:]]
    s = I.with_dt(I.config(1, nr=64, nz=32), 1e-6)
    layers = [dict(l) for l in s["layers"]]
    layers[1] = I.layer(I.poly(g[("lam", 2)][::-1]), I.poly(g[("cv", 2)][::-1]), 2.0)
    st, msg, h = _create(binding, dict(s, layers=layers, T_lo=4.2, T_hi=60.0))
    assert st == binding.HEAT_ERANGE and "c_V" in msg
    import torch
    if not torch.cuda.is_available():   # with a device the fake pointers below would be used
        st, msg, h = _create(binding, dict(s, layers=layers, T_lo=4.2, T_hi=20.0))
        assert st == binding.HEAT_ECUDA                       # positive below the root: passes validation


def test_hot_path_fails_loudly_without_a_gpu(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.HeatSim(I.with_dt(I.config(0), 1e-4))


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (SURVEY tier rule 3)."""
    pkg = os.path.join(ROOT, "paper_1408_5853_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dp, f)).read()
                assert "heat_oracle" not in text and "from oracle" not in text and "import oracle" not in text, f

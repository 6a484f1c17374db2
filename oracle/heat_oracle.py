"""ctypes wrapper around oracle/heat_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package and the CUDA package imports
nothing from here.  A "spec" is the plain dict produced by the seeded input generators
(paper_1408_5853_b200/inputs.py), which hold none of the method's arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "heat_oracle.c")

# variant -> (library file, extra gcc flags)
_VARIANTS = {
    "double": ("libheat_oracle.so", []),
    "omp": ("libheat_oracle_omp.so", ["-fopenmp"]),
    "long": ("libheat_oracle_ld.so", ["-DORC_LONG_DOUBLE"]),
}
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-Wall", "-Wextra"]


def build(variant: str = "double", force: bool = False) -> str:
    """Compile heat_oracle.c with gcc into oracle/<lib>.so and return its path."""
    lib, extra = _VARIANTS[variant]
    out = os.path.join(_HERE, lib)
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        cmd = ["gcc", *CFLAGS, *extra, "-o", out, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return out


def build_all(force: bool = False) -> None:
    for v in _VARIANTS:
        build(v, force)


class _Law(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad_", C.c_int32), ("c", C.c_double * 5), ("T_ref", C.c_double)]


class _Layer(C.Structure):
    _fields_ = [("k", _Law), ("cp", _Law), ("rho", C.c_double), ("is_heater", C.c_int32),
                ("pad_", C.c_int32), ("src_shape", _Law)]


class _Bc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad_", C.c_int32), ("value", C.c_double)]


class _Desc(C.Structure):
    _fields_ = [
        ("nr", C.c_int32), ("nz", C.c_int32), ("batch", C.c_int32), ("nlayers", C.c_int32),
        ("r", C.POINTER(C.c_double)), ("z", C.POINTER(C.c_double)),
        ("layers", C.POINTER(_Layer)), ("seg_layer", C.POINTER(C.c_uint8)),
        ("r_in", _Bc), ("r_out", _Bc), ("z_lo", _Bc), ("z_hi", _Bc),
        ("T0", C.c_double), ("T_init", C.POINTER(C.c_double)),
        ("dt", C.c_double), ("Q0", C.POINTER(C.c_double)),
        ("steps_per_period", C.c_int64), ("steps_on", C.c_int64),
        ("transient_substeps", C.c_int32), ("face_mode", C.c_int32),
        ("transient_k", C.c_double),
        ("nprobes", C.c_int32), ("probe_every", C.c_int32),
        ("probe_ij", C.POINTER(C.c_int32)),
        ("i_step", C.c_int32), ("j_step", C.c_int32),
    ]


_LAW_KIND = {"const": 0, "power": 1, "poly": 2}
_BC_KIND = {"neumann0": 0, "dirichlet": 1}


def _law(d) -> _Law:
    L = _Law()
    L.kind = _LAW_KIND[d["kind"]]
    cs = list(d.get("c", [])) + [0.0] * 5
    for k in range(5):
        L.c[k] = float(cs[k])
    L.T_ref = float(d.get("T_ref", 1.0))
    return L


def _bc(t) -> _Bc:
    b = _Bc()
    b.kind = _BC_KIND[t[0]]
    b.value = float(t[1])
    return b


_ONE = {"kind": "const", "c": [1.0]}


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class _Marshalled:
    """Keeps the numpy arrays behind a _Desc alive."""

    def __init__(self, spec):
        self.r = np.ascontiguousarray(spec["r"], dtype=np.float64)
        self.z = np.ascontiguousarray(spec["z"], dtype=np.float64)
        nr, nz = self.r.size, self.z.size
        batch = int(spec.get("batch", 1))
        layers = spec["layers"]
        self.layers = (_Layer * len(layers))()
        for m, lay in enumerate(layers):
            self.layers[m].k = _law(lay["k"])
            self.layers[m].cp = _law(lay["cp"])
            self.layers[m].rho = float(lay["rho"])
            self.layers[m].is_heater = int(bool(lay.get("is_heater", False)))
            self.layers[m].src_shape = _law(lay.get("src_shape", _ONE))
        self.seg = np.ascontiguousarray(spec["seg_layer"], dtype=np.uint8).reshape(batch, nr - 1)
        self.Q0 = np.ascontiguousarray(spec.get("Q0", np.zeros(batch)), dtype=np.float64).reshape(batch)
        probes = spec.get("probes", [])
        self.probe_ij = np.ascontiguousarray(np.array(probes, dtype=np.int32).reshape(-1, 2))
        T_init = spec.get("T_init")
        self.T_init = None if T_init is None else np.ascontiguousarray(T_init, dtype=np.float64).reshape(batch, nz, nr)
        d = _Desc()
        d.nr, d.nz, d.batch, d.nlayers = nr, nz, batch, len(layers)
        d.r, d.z = _dptr(self.r), _dptr(self.z)
        d.layers = C.cast(self.layers, C.POINTER(_Layer))
        d.seg_layer = self.seg.ctypes.data_as(C.POINTER(C.c_uint8))
        d.r_in, d.r_out = _bc(spec["r_in"]), _bc(spec["r_out"])
        d.z_lo, d.z_hi = _bc(spec["z_lo"]), _bc(spec["z_hi"])
        d.T0 = float(spec.get("T0", 0.0))
        d.T_init = _dptr(self.T_init) if self.T_init is not None else None
        d.dt = float(spec.get("dt") or 1.0)
        d.Q0 = _dptr(self.Q0)
        d.steps_per_period = int(spec.get("steps_per_period", 0))
        d.steps_on = int(spec.get("steps_on", 0))
        d.transient_substeps = int(spec.get("transient_substeps", 0))
        d.face_mode = int(spec.get("face_mode", 0))
        d.transient_k = float(spec.get("transient_k", 7.0))
        d.nprobes = self.probe_ij.shape[0]
        d.probe_every = int(spec.get("probe_every", 1))
        d.probe_ij = self.probe_ij.ctypes.data_as(C.POINTER(C.c_int32))
        d.i_step, d.j_step = int(spec.get("i_step", 0)), int(spec.get("j_step", 0))
        self.desc = d
        self.nr, self.nz, self.batch = nr, nz, batch


_libs = {}


def _load(variant: str):
    if variant not in _libs:
        lib = C.CDLL(build(variant))
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.POINTER(_Desc)]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_step.argtypes = [C.c_void_p, C.c_int64]
        lib.orc_step_picard.argtypes = [C.c_void_p, C.c_int64, C.c_int]
        lib.orc_step_index.restype = C.c_int64
        lib.orc_step_index.argtypes = [C.c_void_p]
        lib.orc_get_field.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double)]
        lib.orc_set_field.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_int64]
        lib.orc_probe.restype = C.c_int64
        lib.orc_probe.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_int64]
        lib.orc_schedule.argtypes = [C.c_void_p, C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.orc_line_rows.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.POINTER(C.c_double)] * 4
        lib.orc_stable_dt.restype = C.c_double
        lib.orc_stable_dt.argtypes = [C.POINTER(_Desc), C.c_double, C.c_double, C.c_int]
        lib.orc_law_eval.restype = C.c_double
        lib.orc_law_eval.argtypes = [C.POINTER(_Law), C.c_double]
        lib.orc_real_bytes.restype = C.c_int
        lib.orc_threads.restype = C.c_int
        _libs[variant] = lib
    return _libs[variant]


STABLE_DT_SAMPLES = 1025


def stable_dt(spec, T_lo=None, T_hi=None, variant: str = "double") -> float:
    """Right-hand side of the stability bound (21)."""
    lib = _load(variant)
    m = _Marshalled(spec)
    T_lo = float(spec["T_lo"] if T_lo is None else T_lo)
    T_hi = float(spec["T_hi"] if T_hi is None else T_hi)
    return float(lib.orc_stable_dt(C.byref(m.desc), T_lo, T_hi, STABLE_DT_SAMPLES))


def law_eval(law: dict, T: float, variant: str = "double") -> float:
    lib = _load(variant)
    L = _law(law)
    return float(lib.orc_law_eval(C.byref(L), float(T)))


class Oracle:
    """One simulation state advanced by the paper's scheme on the CPU."""

    def __init__(self, spec, variant: str = "double"):
        self._lib = _load(variant)
        self._m = _Marshalled(spec)
        self.nr, self.nz, self.batch = self._m.nr, self._m.nz, self._m.batch
        self.nprobes = self._m.probe_ij.shape[0]
        self._h = self._lib.orc_create(C.byref(self._m.desc))
        if not self._h:
            raise ValueError("orc_create rejected the descriptor")

    def close(self):
        if self._h:
            self._lib.orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def threads(self) -> int:
        return int(self._lib.orc_threads())

    @property
    def step_index(self) -> int:
        return int(self._lib.orc_step_index(self._h))

    def step(self, n: int = 1) -> None:
        self._lib.orc_step(self._h, int(n))

    def step_picard(self, n: int = 1, iters: int = 2) -> None:
        """n steps of the iterated variant (reading G23); iters = 1 is step()."""
        self._lib.orc_step_picard(self._h, int(n), int(iters))

    def field(self, b: int = 0) -> np.ndarray:
        out = np.empty((self.nz, self.nr), dtype=np.float64)
        self._lib.orc_get_field(self._h, int(b), _dptr(out))
        return out

    def fields(self) -> np.ndarray:
        return np.stack([self.field(b) for b in range(self.batch)])

    def set_field(self, b: int, T: np.ndarray, step_index: int) -> None:
        T = np.ascontiguousarray(T, dtype=np.float64).reshape(self.nz, self.nr)
        self._lib.orc_set_field(self._h, int(b), _dptr(T), int(step_index))

    def probes(self) -> np.ndarray:
        """All probe records so far, shape [records, batch, nprobes]."""
        n = int(self._lib.orc_probe(self._h, None, 0))
        out = np.empty(max(n, 1), dtype=np.float64)
        self._lib.orc_probe(self._h, _dptr(out), n)
        return out[:n].reshape(-1, self.batch, max(self.nprobes, 1))

    def schedule(self, s: int):
        tau, amp = C.c_double(), C.c_double()
        self._lib.orc_schedule(self._h, int(s), C.byref(tau), C.byref(amp))
        return tau.value, amp.value

    def line_rows(self, b: int, j: int):
        """Rows (A, B, C, F) of line j as the next step would see them (dense-solve pin)."""
        arrs = [np.empty(self.nr, dtype=np.float64) for _ in range(4)]
        self._lib.orc_line_rows(self._h, int(b), int(j), *[_dptr(a) for a in arrs])
        return arrs


if __name__ == "__main__":
    build_all(force=True)
    print("built:", ", ".join(v[0] for v in _VARIANTS.values()))

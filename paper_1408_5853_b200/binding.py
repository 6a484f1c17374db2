"""Thin ctypes binding of include/heat.h -- argument marshalling only.

Every step of the method runs in the CUDA kernels behind `libheat_b200.so`; PyTorch is used
for device memory and streams.  There is no CPU fallback: importing this module without the
built library raises, and `HeatSim` raises without a CUDA device.

Function names mirror the C ABI: heat_workspace_bytes, heat_stable_dt, heat_create,
heat_step, heat_get_field, heat_set_field, heat_probe, heat_schedule, heat_destroy.
A "spec" is the plain dict produced by `paper_1408_5853_b200.inputs`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libheat_b200.so")

HEAT_OK, HEAT_EINVAL, HEAT_ENOMEM, HEAT_ECUDA, HEAT_ERANGE = range(5)
HEAT_DESC_GENERAL_KERNEL = 1
STATUS_NAMES = {0: "HEAT_OK", 1: "HEAT_EINVAL", 2: "HEAT_ENOMEM", 3: "HEAT_ECUDA", 4: "HEAT_ERANGE"}

EXPORTS = [
    "heat_workspace_bytes", "heat_stable_dt", "heat_create", "heat_step", "heat_get_field",
    "heat_set_field", "heat_get_line", "heat_set_line", "heat_probe", "heat_schedule", "heat_step_index", "heat_launch_count",
    "heat_kernel_name", "heat_last_error", "heat_destroy", "heat_fp64_peak", "heat_fp64_peak_scratch_bytes",
    "heat_create_static", "heat_static_workspace_bytes", "heat_step_picard", "heat_set_halo_peer",
]


class HeatError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class heat_law(C.Structure):
    _fields_ = [("kind", C.c_int32), ("reserved", C.c_int32), ("c", C.c_double * 5), ("T_ref", C.c_double)]


class heat_layer(C.Structure):
    _fields_ = [("k", heat_law), ("cp", heat_law), ("rho", C.c_double), ("is_heater", C.c_int32),
                ("reserved", C.c_int32), ("src_shape", heat_law)]


class heat_bc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("reserved", C.c_int32), ("value", C.c_double)]


class heat_desc(C.Structure):
    _fields_ = [
        ("nr", C.c_int32), ("nz", C.c_int32), ("batch", C.c_int32), ("nlayers", C.c_int32),
        ("r", C.POINTER(C.c_double)), ("z", C.POINTER(C.c_double)),
        ("layers", C.POINTER(heat_layer)), ("seg_layer", C.POINTER(C.c_uint8)),
        ("r_in", heat_bc), ("r_out", heat_bc), ("z_lo", heat_bc), ("z_hi", heat_bc),
        ("T0", C.c_double), ("T_init", C.c_void_p),
        ("dt", C.c_double), ("Q0", C.POINTER(C.c_double)),
        ("steps_per_period", C.c_int64), ("steps_on", C.c_int64),
        ("transient_substeps", C.c_int32), ("face_mode", C.c_int32),
        ("transient_k", C.c_double),
        ("nprobes", C.c_int32), ("probe_every", C.c_int32),
        ("probe_ij", C.POINTER(C.c_int32)),
        ("T_init_is_device", C.c_int32), ("flags", C.c_int32),
        ("T_lo", C.c_double), ("T_hi", C.c_double),
        ("i_step", C.c_int32), ("j_step", C.c_int32),
    ]


_lib = None


def lib():
    """Load the C-ABI library; fail loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1408_5853_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
        L.heat_workspace_bytes.restype = C.c_size_t
        L.heat_workspace_bytes.argtypes = [C.POINTER(heat_desc)]
        L.heat_stable_dt.restype = C.c_int
        L.heat_stable_dt.argtypes = [C.POINTER(heat_desc), dbl, dbl, C.POINTER(dbl)]
        L.heat_create.restype = C.c_int
        L.heat_create.argtypes = [C.POINTER(heat_desc), vp, vp, vp, C.c_size_t, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.heat_step.restype = C.c_int
        L.heat_step.argtypes = [vp, i64, vp]
        L.heat_get_field.restype = C.c_int
        L.heat_get_field.argtypes = [vp, C.c_int32, vp, C.c_int32, vp]
        L.heat_set_field.restype = C.c_int
        L.heat_set_field.argtypes = [vp, C.c_int32, vp, C.c_int32, i64, vp]
        L.heat_probe.restype = C.c_int
        L.heat_probe.argtypes = [vp, vp, i64, C.POINTER(i64), C.POINTER(i64), vp]
        L.heat_schedule.restype = C.c_int
        L.heat_schedule.argtypes = [vp, i64, C.POINTER(dbl), C.POINTER(dbl)]
        L.heat_step_index.restype = i64
        L.heat_step_index.argtypes = [vp]
        L.heat_launch_count.restype = i64
        L.heat_launch_count.argtypes = [vp]
        L.heat_kernel_name.restype = C.c_char_p
        L.heat_kernel_name.argtypes = [vp]
        L.heat_last_error.restype = C.c_char_p
        L.heat_last_error.argtypes = [vp]
        L.heat_destroy.restype = None
        L.heat_destroy.argtypes = [vp]
        L.heat_get_line.restype = C.c_int
        L.heat_get_line.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_int32, vp]
        L.heat_set_line.restype = C.c_int
        L.heat_set_line.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_int32, vp]
        L.heat_fp64_peak.restype = C.c_int
        L.heat_fp64_peak.argtypes = [i64, vp, C.c_size_t, vp, C.POINTER(dbl)]
        L.heat_fp64_peak_scratch_bytes.restype = C.c_size_t
        L.heat_fp64_peak_scratch_bytes.argtypes = []
        L.heat_create_static.restype = C.c_int
        L.heat_create_static.argtypes = [C.POINTER(heat_desc), vp, vp, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.heat_static_workspace_bytes.restype = C.c_size_t
        L.heat_static_workspace_bytes.argtypes = []
        L.heat_set_halo_peer.restype = C.c_int
        L.heat_set_halo_peer.argtypes = [vp, C.c_int32, vp, vp, C.c_int32]
        L.heat_step_picard.restype = C.c_int
        L.heat_step_picard.argtypes = [vp, i64, C.c_int32, vp, vp]
        _lib = L
    return _lib


_LAW_KIND = {"const": 0, "power": 1, "poly": 2}
_BC_KIND = {"neumann0": 0, "dirichlet": 1}
_ONE = {"kind": "const", "c": [1.0]}


def _law(d) -> heat_law:
    L = heat_law()
    L.kind = _LAW_KIND[d["kind"]]
    cs = list(d.get("c", [])) + [0.0] * 5
    for k in range(5):
        L.c[k] = float(cs[k])
    L.T_ref = float(d.get("T_ref", 1.0))
    return L


def _bc(t) -> heat_bc:
    b = heat_bc()
    b.kind = _BC_KIND[t[0]]
    b.value = float(t[1])
    return b


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Desc:
    """A heat_desc plus the numpy arrays that keep its host pointers alive."""

    def __init__(self, spec, T_init_device_ptr=None, placeholder_dt=False):
        self.r = np.ascontiguousarray(spec["r"], dtype=np.float64)
        self.z = np.ascontiguousarray(spec["z"], dtype=np.float64)
        nr, nz = self.r.size, self.z.size
        batch = int(spec.get("batch", 1))
        layers = spec["layers"]
        self.layers = (heat_layer * len(layers))()
        for m, lay in enumerate(layers):
            self.layers[m].k = _law(lay["k"])
            self.layers[m].cp = _law(lay["cp"])
            self.layers[m].rho = float(lay["rho"])
            self.layers[m].is_heater = int(bool(lay.get("is_heater", False)))
            self.layers[m].src_shape = _law(lay.get("src_shape", _ONE))
        self.seg = np.ascontiguousarray(spec["seg_layer"], dtype=np.uint8).reshape(batch, nr - 1)
        self.Q0 = np.ascontiguousarray(spec.get("Q0", np.zeros(batch)), dtype=np.float64).reshape(batch)
        self.probe_ij = np.ascontiguousarray(np.array(spec.get("probes", []), dtype=np.int32).reshape(-1, 2))
        T_init = spec.get("T_init")
        self.T_init = None if T_init is None else np.ascontiguousarray(T_init, dtype=np.float64).reshape(batch, nz, nr)
        d = heat_desc()
        d.nr, d.nz, d.batch, d.nlayers = nr, nz, batch, len(layers)
        d.r, d.z = _dptr(self.r), _dptr(self.z)
        d.layers = C.cast(self.layers, C.POINTER(heat_layer))
        d.seg_layer = self.seg.ctypes.data_as(C.POINTER(C.c_uint8))
        d.r_in, d.r_out = _bc(spec["r_in"]), _bc(spec["r_out"])
        d.z_lo, d.z_hi = _bc(spec["z_lo"]), _bc(spec["z_hi"])
        d.T0 = float(spec.get("T0", 0.0))
        if T_init_device_ptr is not None:
            d.T_init, d.T_init_is_device = C.c_void_p(T_init_device_ptr), 1
        elif self.T_init is not None:
            d.T_init, d.T_init_is_device = C.c_void_p(self.T_init.ctypes.data), 0
        else:
            d.T_init, d.T_init_is_device = None, 0
        # heat_stable_dt / heat_workspace_bytes are asked before tau is known: only they may pass a placeholder
        d.dt = float(spec.get("dt") or (1.0 if placeholder_dt else 0.0))
        d.Q0 = _dptr(self.Q0)
        d.steps_per_period = int(spec.get("steps_per_period", 0))
        d.steps_on = int(spec.get("steps_on", 0))
        d.transient_substeps = int(spec.get("transient_substeps", 0))
        d.face_mode = int(spec.get("face_mode", 0))
        d.flags = HEAT_DESC_GENERAL_KERNEL if spec.get("general_kernel") else 0
        d.i_step, d.j_step = int(spec.get("i_step", 0)), int(spec.get("j_step", 0))
        d.transient_k = float(spec.get("transient_k", 7.0))
        d.nprobes = self.probe_ij.shape[0]
        d.probe_every = int(spec.get("probe_every", 1))
        d.probe_ij = self.probe_ij.ctypes.data_as(C.POINTER(C.c_int32))
        d.T_lo = float(spec.get("T_lo", 0.0))
        d.T_hi = float(spec.get("T_hi", 0.0))
        self.desc = d
        self.nr, self.nz, self.batch = nr, nz, batch
        self.nprobes = d.nprobes


def heat_stable_dt(spec, T_lo=None, T_hi=None) -> float:
    """Right-hand side of (21) P:L194-196 (host-only call of the C ABI)."""
    m = Desc(spec, placeholder_dt=True)
    out = C.c_double()
    T_lo = float(spec["T_lo"] if T_lo is None else T_lo)
    T_hi = float(spec["T_hi"] if T_hi is None else T_hi)
    st = lib().heat_stable_dt(C.byref(m.desc), T_lo, T_hi, C.byref(out))
    if st != HEAT_OK:
        raise HeatError(st, lib().heat_last_error(None).decode())
    return out.value


def heat_workspace_bytes(spec) -> int:
    return int(lib().heat_workspace_bytes(C.byref(Desc(spec, placeholder_dt=True).desc)))


def heat_static_workspace_bytes() -> int:
    return int(lib().heat_static_workspace_bytes())


def heat_fp64_peak(iters=1 << 16) -> float:
    import torch
    out = C.c_double()
    nbytes = int(lib().heat_fp64_peak_scratch_bytes())
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    st = lib().heat_fp64_peak(int(iters), C.c_void_p(scratch.data_ptr()), nbytes,
                              C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(out))
    if st != HEAT_OK:
        raise HeatError(st, lib().heat_last_error(None).decode())
    return out.value


class HeatSim:
    """One simulation context on the current CUDA device: heat_create .. heat_destroy."""

    def __init__(self, spec, probe_records=None, stream=None, T_init_device=None, guard=0, static_workspace=False):
        """static_workspace=True: heat_create_static, i.e. the row tables go into the library's static
        device array (no workspace is allocated; at most one such context alive per device)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("HeatSim needs a CUDA device (B200, sm_100a); there is no CPU fallback")
        self._torch = torch
        self._L = lib()
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        dev_ptr = None
        if T_init_device is not None:
            assert T_init_device.is_cuda and T_init_device.dtype == torch.float64 and T_init_device.is_contiguous()
            dev_ptr = T_init_device.data_ptr()
        self._m = Desc(spec, T_init_device_ptr=dev_ptr)
        m = self._m
        self.nr, self.nz, self.batch, self.nprobes = m.nr, m.nz, m.batch, m.nprobes
        cells = m.batch * m.nz * m.nr
        ws = int(self._L.heat_workspace_bytes(C.byref(m.desc)))
        if ws == 0:
            # heat_create validates the descriptor before it looks at the buffers: ask it for the real status
            h0 = C.c_void_p()
            st0 = self._L.heat_create(C.byref(m.desc), None, None, None, 0, None, 0, C.c_void_p(self.stream.cuda_stream), C.byref(h0))
            raise HeatError(st0 if st0 != HEAT_OK else HEAT_EINVAL, self._L.heat_last_error(None).decode() or "descriptor rejected")
        dev = torch.device("cuda", torch.cuda.current_device())
        with torch.cuda.stream(self.stream):
            rec = m.batch * m.nprobes
            if probe_records is None:
                probe_records = 4096
            self.probe_cap = max(rec * int(probe_records), 1)
            # guard > 0 (tests): every buffer the library is handed sits between two bands of `guard`
            # doubles holding a canary, so that a write outside a buffer is seen (guards_intact)
            g = int(guard)
            self._guards = []

            def banded(n):
                big = torch.full((n + 2 * g,), self.CANARY, dtype=torch.float64, device=dev)
                if g:
                    self._guards += [big[:g], big[g + n:]]
                return big[g:g + n]

            self.field_a = banded(cells)
            self.field_b = banded(cells)
            if static_workspace:
                self.workspace = None
            else:
                self._ws64 = banded((ws + 7) // 8 + 32)
                ws_off = (-self._ws64.data_ptr()) % 256                # the workspace must be 256-byte aligned
                self.workspace = self._ws64.view(torch.uint8)[ws_off:ws_off + ws]
            self.probe_buf = banded(self.probe_cap)
            self.probe_buf.zero_()
        h = C.c_void_p()
        if static_workspace:
            st = self._L.heat_create_static(C.byref(m.desc), self.field_a.data_ptr(), self.field_b.data_ptr(),
                                            self.probe_buf.data_ptr(), self.probe_cap,
                                            C.c_void_p(self.stream.cuda_stream), C.byref(h))
            if st != HEAT_OK:
                raise HeatError(st, self._L.heat_last_error(None).decode())
            self._h = h
            return
        st = self._L.heat_create(C.byref(m.desc), self.field_a.data_ptr(), self.field_b.data_ptr(),
                                 self.workspace.data_ptr(), ws, self.probe_buf.data_ptr(), self.probe_cap,
                                 C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if st != HEAT_OK:
            raise HeatError(st, self._L.heat_last_error(None).decode())
        self._h = h

    CANARY = -7.0e77

    def guards_intact(self) -> bool:
        self.stream.synchronize()
        return all(bool((b == self.CANARY).all().item()) for b in self._guards)

    # -- C ABI calls ------------------------------------------------------------------
    def _check(self, st):
        if st != HEAT_OK:
            raise HeatError(st, self._L.heat_last_error(self._h).decode())

    def _s(self):
        return C.c_void_p(self.stream.cuda_stream)

    def step(self, n=1):
        """heat_step: enqueue n solver steps (asynchronous)."""
        self._check(self._L.heat_step(self._h, int(n), self._s()))

    def step_picard(self, n=1, iters=2):
        """heat_step_picard: n solver steps of the iterated variant; needs spec["general_kernel"]."""
        if getattr(self, "_field_c", None) is None:
            self._field_c = self._torch.empty_like(self.field_a)
        self._check(self._L.heat_step_picard(self._h, int(n), int(iters), self._field_c.data_ptr(), self._s()))

    def field(self, b=0) -> np.ndarray:
        """heat_get_field to host memory, [nz][nr]."""
        out = np.empty((self.nz, self.nr), dtype=np.float64)
        self._check(self._L.heat_get_field(self._h, int(b), C.c_void_p(out.ctypes.data), 0, self._s()))
        return out

    def fields(self) -> np.ndarray:
        return np.stack([self.field(b) for b in range(self.batch)])

    def field_device(self, b=0):
        """heat_get_field into a fresh device tensor (asynchronous)."""
        out = self._torch.empty((self.nz, self.nr), dtype=self._torch.float64, device=self.field_a.device)
        self._check(self._L.heat_get_field(self._h, int(b), C.c_void_p(out.data_ptr()), 1, self._s()))
        return out

    def set_field(self, b, T, step_index):
        """heat_set_field from a host array or a device tensor."""
        if hasattr(T, "is_cuda"):
            assert T.is_cuda and T.is_contiguous() and T.dtype == self._torch.float64
            self._check(self._L.heat_set_field(self._h, int(b), C.c_void_p(T.data_ptr()), 1, int(step_index), self._s()))
        else:
            T = np.ascontiguousarray(T, dtype=np.float64).reshape(self.nz, self.nr)
            self._check(self._L.heat_set_field(self._h, int(b), C.c_void_p(T.ctypes.data), 0, int(step_index), self._s()))

    def get_line(self, b, j):
        """heat_get_line into a fresh device tensor [nr] (asynchronous)."""
        out = self._torch.empty(self.nr, dtype=self._torch.float64, device=self.field_a.device)
        self._check(self._L.heat_get_line(self._h, int(b), int(j), C.c_void_p(out.data_ptr()), 1, self._s()))
        return out

    def set_line(self, b, j, values):
        """heat_set_line from a device tensor or a host array of nr doubles."""
        if hasattr(values, "is_cuda") and values.is_cuda:
            assert values.is_contiguous() and values.dtype == self._torch.float64 and values.numel() == self.nr
            self._check(self._L.heat_set_line(self._h, int(b), int(j), C.c_void_p(values.data_ptr()), 1, self._s()))
        else:
            v = np.ascontiguousarray(np.asarray(values, dtype=np.float64).reshape(self.nr))
            self._check(self._L.heat_set_line(self._h, int(b), int(j), C.c_void_p(v.ctypes.data), 0, self._s()))

    def set_halo_peer(self, side, peer=None):
        """heat_set_halo_peer: `peer` is the neighbour slab's HeatSim in this process (side 0: the slab below,
        1: above), a tuple (field_a_ptr, field_b_ptr, nz) of peer-mapped addresses, or None to switch it off."""
        if peer is None:
            a, b, pnz = None, None, 0
        elif isinstance(peer, tuple):
            a, b, pnz = peer
        else:
            a, b, pnz = peer.field_a.data_ptr(), peer.field_b.data_ptr(), peer.nz
        self._check(self._L.heat_set_halo_peer(self._h, int(side), a, b, int(pnz)))

    def probes(self, max_records=None):
        """heat_probe: drain the trace, shape [records, batch, nprobes]; also returns drops."""
        rec = self.batch * self.nprobes
        if rec == 0:
            return np.empty((0, self.batch, 0)), 0
        cap = self.probe_cap if max_records is None else rec * int(max_records)
        out = np.empty(max(cap, 1), dtype=np.float64)
        n, dropped = C.c_int64(), C.c_int64()
        self._check(self._L.heat_probe(self._h, C.c_void_p(out.ctypes.data), cap, C.byref(n), C.byref(dropped), self._s()))
        return out[:n.value].reshape(-1, self.batch, self.nprobes).copy(), int(dropped.value)

    def schedule(self, s):
        tau, amp = C.c_double(), C.c_double()
        self._check(self._L.heat_schedule(self._h, int(s), C.byref(tau), C.byref(amp)))
        return tau.value, amp.value

    @property
    def step_index(self) -> int:
        return int(self._L.heat_step_index(self._h))

    @property
    def launch_count(self) -> int:
        return int(self._L.heat_launch_count(self._h))

    @property
    def kernel_name(self) -> str:
        return self._L.heat_kernel_name(self._h).decode()

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "_h", None):
            self.stream.synchronize()
            self._L.heat_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

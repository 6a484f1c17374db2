"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic: it only writes down geometry, material
laws, boundary values, source parameters and integer schedules as a plain dict ("spec").
The time step is not chosen here: the stability bound (21) is part of the method, so the
caller obtains its right-hand side from whichever side it is driving (`heat_stable_dt` of
the C-ABI library, or the oracle's `stable_dt` in tests) and passes it to `with_dt`.

The five `config(n)` workloads are the ones BASELINE.json lists; they stand in for the
paper's device: thin coaxial layers core / insulator / heater / surface,
R << L (aspect 1:10), cryogenic power-law growth of k and c, rectangular pulse with 10 %
duty, cold / warm Dirichlet terminals.  Recipe and readings: DESIGN.md "Input recipe".
"""
from __future__ import annotations

import math
from fractions import Fraction

import numpy as np

SEED = 14085853
DT_SAFETY = Fraction(9, 10)  # BASELINE.json: "dt = 0.9 x explicit stability limit"


# ---------------------------------------------------------------- small constructors

def const(v):
    return {"kind": "const", "c": [float(v)], "T_ref": 1.0}


def power(c0, p, T_ref=20.0):
    return {"kind": "power", "c": [float(c0), float(p)], "T_ref": float(T_ref)}


def poly(ascending):
    return {"kind": "poly", "c": [float(x) for x in ascending], "T_ref": 1.0}


def layer(k, cp, rho, is_heater=False, src_shape=None):
    return {"k": k, "cp": cp, "rho": float(rho), "is_heater": bool(is_heater),
            "src_shape": src_shape if src_shape is not None else const(1.0)}


NEUMANN0 = ("neumann0", 0.0)


def dirichlet(v):
    return ("dirichlet", float(v))


def uniform_nodes(length, n):
    """n nodes 0 .. length, node k at length*k/(n-1) (one rounding per node)."""
    return np.array([length * k / (n - 1) for k in range(n)], dtype=np.float64)


def snap_index(radius: Fraction, R: Fraction, nr: int) -> int:
    """Node nearest to `radius` on the uniform grid of nr nodes over [0, R]; round half up,
    exact rational arithmetic."""
    x = Fraction(radius) * (nr - 1) / Fraction(R)
    return math.floor(x + Fraction(1, 2))


def seg_layers(nr: int, interface_nodes) -> np.ndarray:
    """Layer of each radial segment (i, i+1): number of interface nodes <= i."""
    seg = np.zeros(nr - 1, dtype=np.uint8)
    for n in interface_nodes:
        seg[n:] += 1
    return seg


# ---------------------------------------------------------------- BASELINE.json configs

_MM = Fraction(1, 1000)
# config 1..4 physics: k_i = k0 (T/20)^p, c_i = c0 (T/20)^q
_K0 = (15.0, 0.5, 200.0, 50.0)
_P = (1.0, 2.0, 1.0, 1.5)
_C0 = (5.0, 2.0, 10.0, 8.0)
_Q = (3.0, 3.0, 2.0, 3.0)
_RHO = (8000.0, 4000.0, 9000.0, 2700.0)
_RADII = (Fraction(12, 10) * _MM, Fraction(16, 10) * _MM, Fraction(18, 10) * _MM)
_R4 = 2 * _MM
_L4 = 20 * _MM


def _cell_layers():
    return [layer(power(_K0[m], _P[m]), power(_C0[m], _Q[m]), _RHO[m], is_heater=(m == 2))
            for m in range(4)]


def _base(nr, nz, R, L, layers, seg, batch=1):
    return {
        "nr": nr, "nz": nz, "batch": batch,
        "r": uniform_nodes(float(R), nr), "z": uniform_nodes(float(L), nz),
        "layers": layers, "seg_layer": np.ascontiguousarray(seg, dtype=np.uint8).reshape(batch, nr - 1),
        "r_in": NEUMANN0, "r_out": NEUMANN0,             # symmetry at r=0, insulated r=R
        "z_lo": dirichlet(4.2), "z_hi": dirichlet(78.0),  # helium / nitrogen terminals
        "T0": 20.0, "T_init": None,
        "Q0": np.zeros(batch), "steps_per_period": 0, "steps_on": 0,
        "transient_substeps": 0, "transient_k": 7.0, "face_mode": 0,
        "probes": [], "probe_every": 1,
        "T_lo": 4.2, "T_hi": 300.0,                      # range scanned by (21), SURVEY G19
        "dt": None,
    }


def surface_probe(nr, nz):
    """Outer surface at z = L/2: node (N, round-half-up((nz-1)/2))."""
    return (nr - 1, math.floor(Fraction(nz - 1, 2) + Fraction(1, 2)))


def cell_spec(nr, nz, batch=1, Q0=None, heater_thickness_mm=None, pulsed=True):
    """The 4-layer cryogenic cell of configs 1-4 on an nr x nz grid (also the downscaled
    variants used by the parity protocol)."""
    segs = []
    for b in range(batch):
        radii = list(_RADII)
        if heater_thickness_mm is not None:
            # heater outer radius fixed at 1.8 mm, inner = 1.8 - thickness
            x = (1.8 - float(heater_thickness_mm[b])) * (nr - 1) / 2.0
            i_heater = math.floor(x + 0.5)
            nodes = [snap_index(radii[0], _R4, nr), i_heater, snap_index(radii[2], _R4, nr)]
        else:
            nodes = [snap_index(rr, _R4, nr) for rr in radii]
        segs.append(seg_layers(nr, nodes))
    s = _base(nr, nz, _R4, _L4, _cell_layers(), np.stack(segs), batch)
    if pulsed:
        s["Q0"] = np.full(batch, 5e9) if Q0 is None else np.asarray(Q0, dtype=np.float64)
        s["period_s"], s["on_fraction"] = 20e-3, Fraction(1, 10)  # 50 Hz, 2 ms on
        s["transient_substeps"], s["transient_k"] = 100, 7.0
        s["probes"] = [surface_probe(nr, nz)]
    return s


def config(n: int, nr: int | None = None, nz: int | None = None, batch: int | None = None):
    """BASELINE.json configs[n]; nr/nz/batch override the grid for downscaled parity runs."""
    if n == 0:
        nr, nz = nr or 64, nz or 64
        R, L = 1 * _MM, 10 * _MM
        nodes = [snap_index(Fraction(5, 10) * _MM, R, nr), snap_index(Fraction(8, 10) * _MM, R, nr)]
        layers = [layer(const(10.0), const(100.0), 8000.0), layer(const(1.0), const(50.0), 4000.0),
                  layer(const(100.0), const(200.0), 9000.0)]
        s = _base(nr, nz, R, L, layers, seg_layers(nr, nodes))
        s["steps"] = 1000
        s["name"] = "cfg0 constant-coefficient 3-layer cylinder"
        return s
    if n == 1:
        s = cell_spec(nr or 512, nz or 512, pulsed=False)
        s["steps"] = 2000
        s["name"] = "cfg1 nonlinear 4-layer cell"
        return s
    if n == 2:
        s = cell_spec(nr or 2048, nz or 2048)
        s["probe_every"] = 1
        s["periods"] = 5
        s["name"] = "cfg2 cell + 50 Hz pulse heating"
        return s
    if n == 3:
        batch = batch or 256
        rng = np.random.Generator(np.random.PCG64(SEED))
        Q0 = np.exp(rng.uniform(math.log(1e9), math.log(2e10), size=256))
        thick = rng.uniform(0.1, 0.4, size=256)
        s = cell_spec(nr or 512, nz or 512, batch=batch, Q0=Q0[:batch], heater_thickness_mm=thick[:batch])
        s["probe_every"] = 1
        s["periods"] = 2
        s["heater_thickness_mm"] = thick[:batch]
        s["name"] = "cfg3 parameter-sweep batch"
        return s
    if n == 4:
        s = cell_spec(nr or 8192, nz or 8192)
        s["probe_every"] = 100
        s["steps"] = 10000
        s["name"] = "cfg4 large-grid throughput"
        return s
    raise ValueError(n)


def with_dt(spec, dt_limit: float):
    """Fix tau and the integer schedule from the right-hand side of (21):
    tau = 0.9 * limit without a source; with one, steps_per_period = ceil(t_prd / (0.9 limit)),
    tau = t_prd / steps_per_period, steps_on = steps_per_period / 10."""
    s = dict(spec)
    dt_max = float(DT_SAFETY) * float(dt_limit)
    if "period_s" in s:
        P = int(math.ceil(s["period_s"] / dt_max))
        s["steps_per_period"] = P
        s["steps_on"] = int(P * s["on_fraction"])
        s["dt"] = s["period_s"] / P
        if "periods" in s:
            sub = s["transient_substeps"]
            s["steps"] = s["periods"] * (P - 1 + sub if sub > 0 and s["steps_on"] > 0 else P)
    else:
        s["dt"] = dt_max
    return s


def steps_per_solver_period(spec) -> int:
    """Solver steps in one source period (a transient sub-step counts as a step)."""
    P, sub = spec["steps_per_period"], spec["transient_substeps"]
    return P - 1 + sub if (sub > 0 and spec["steps_on"] > 0) else P


# ---------------------------------------------------------------- random small problems

def random_spec(seed, nr=13, nz=11, nlayers=3, batch=1, laws="mixed", source=True,
                r0=0.0, bcs=None, nonuniform=True):
    """Small seeded problem with non-uniform steps, several layers and T-dependent laws, for
    the dense-solve pin, invariants and GPU edge cases."""
    rng = np.random.Generator(np.random.PCG64(SEED + int(seed)))
    hr = rng.uniform(0.5, 1.5, size=nr - 1) if nonuniform else np.ones(nr - 1)
    hz = rng.uniform(0.5, 1.5, size=nz - 1) if nonuniform else np.ones(nz - 1)
    r = r0 + np.concatenate([[0.0], np.cumsum(hr)]) * (1e-3 / (nr - 1))
    z = np.concatenate([[0.0], np.cumsum(hz)]) * (1e-2 / (nz - 1))
    layers = []
    for m in range(nlayers):
        kind = laws if laws != "mixed" else ("const", "power", "poly")[m % 3]
        if kind == "const":
            k, cp = const(rng.uniform(1, 100)), const(rng.uniform(50, 200))
        elif kind == "power":
            k = power(rng.uniform(1, 100), rng.choice([1.0, 1.5, 2.0, 0.7]))
            cp = power(rng.uniform(1, 10), rng.choice([2.0, 3.0, 1.3]))
        else:
            k = poly([rng.uniform(1, 5), rng.uniform(0.1, 0.5), rng.uniform(1e-3, 5e-3), 0.0, rng.uniform(1e-8, 1e-7)])
            cp = poly([rng.uniform(1, 5), rng.uniform(0.1, 0.5), rng.uniform(1e-3, 5e-3), rng.uniform(1e-5, 1e-4)])
        layers.append(layer(k, cp, rng.uniform(2000, 9000), is_heater=(source and m == nlayers - 2 and nlayers > 1) or (source and nlayers == 1),
                            src_shape=power(1.0, -0.5, 20.0) if m % 2 else const(1.0)))
    segs = []
    for b in range(batch):
        # interface nodes: distinct, not adjacent, not on the boundary
        while True:
            nodes = sorted(rng.choice(np.arange(2, nr - 2), size=nlayers - 1, replace=False).tolist()) if nlayers > 1 else []
            if all(b2 - a2 >= 2 for a2, b2 in zip(nodes, nodes[1:])):
                break
        segs.append(seg_layers(nr, nodes))
    s = _base(nr, nz, 1, 1, layers, np.stack(segs), batch)
    s["r"], s["z"] = r, z
    if bcs is not None:
        s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = bcs
    s["T_init"] = rng.uniform(5.0, 80.0, size=(batch, nz, nr))
    s["T_lo"], s["T_hi"] = 4.2, 100.0
    if source:
        s["Q0"] = rng.uniform(1e8, 1e9, size=batch)
        s["steps_per_period"], s["steps_on"] = 7, 3
        s["transient_substeps"], s["transient_k"] = 5, 7.0
    s["probes"] = [(nr - 1, nz // 2), (1, 1)]
    s["probe_every"] = 2
    return s


# ---------------------------------------------------------------- band-kernel edge cases

def band_spec(seed, nr=512, nz=24, nlayers=4, batch=1, bcs=None, source=True, poly_laws=False,
              nonuniform_z=True, chunk=8):
    """Seeded problem on a uniform r grid starting at r = 0 (what the band kernels cover) with
    interface nodes at every position of a thread's chunk of `chunk` nodes (first, last, middle;
    8 nodes in the band kernel, 16 in the wband kernel), square-root,
    power and polynomial laws, random initial field, optional source and non-uniform z."""
    rng = np.random.Generator(np.random.PCG64(SEED + 1000 + int(seed)))
    R = 2e-3
    r = uniform_nodes(R, nr)
    hz = rng.uniform(0.7, 1.3, size=nz - 1) if nonuniform_z else np.ones(nz - 1)
    z = np.concatenate([[0.0], np.cumsum(hz)]) * (10.0 * R / (nr - 1))  # eta ~ 10 h as in BASELINE configs
    layers = []
    for m in range(nlayers):
        if poly_laws:
            k = poly([rng.uniform(1, 5), rng.uniform(0.1, 0.5), rng.uniform(1e-3, 5e-3), rng.uniform(1e-6, 1e-5),
                      rng.uniform(1e-8, 1e-7) if m % 2 else 0.0])
            cp = poly([rng.uniform(1, 5), rng.uniform(0.1, 0.5), rng.uniform(1e-3, 5e-3), rng.uniform(1e-5, 1e-4)])
        else:
            k = power(rng.uniform(1, 100), [1.0, 2.0, 1.5, 0.5, 3.0, 0.0][(m + seed) % 6])
            cp = [power(rng.uniform(1, 10), 3.0), power(rng.uniform(1, 10), 2.0), const(rng.uniform(50, 200)),
                  power(rng.uniform(1, 10), 1.0)][(m + seed) % 4]
        layers.append(layer(k, cp, rng.uniform(2000, 9000), is_heater=(source and m == nlayers - 2)))
    segs = []
    for b in range(batch):
        # one interface per chosen chunk, at chunk positions 0, 7 and a random one
        chunks = sorted(rng.choice(np.arange(1, nr // chunk - 1), size=nlayers - 1, replace=False).tolist())
        pos = [0, chunk - 1] + [int(rng.integers(1, chunk - 1)) for _ in range(nlayers)]
        nodes = [chunk * c + pos[(q + b) % len(pos)] for q, c in enumerate(chunks)]
        # adjacent chunks could give adjacent interface nodes (8c+7, 8c+8): move the second one
        for q in range(1, len(nodes)):
            if nodes[q] - nodes[q - 1] < 2:
                nodes[q] += 3
        segs.append(seg_layers(nr, nodes))
    s = _base(nr, nz, 1, 1, layers, np.stack(segs), batch)
    s["r"], s["z"] = r, z
    if bcs is not None:
        s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = bcs
    s["T_init"] = rng.uniform(5.0, 80.0, size=(batch, nz, nr))
    s["T_lo"], s["T_hi"] = 4.2, 100.0
    if source:
        s["Q0"] = rng.uniform(1e8, 1e9, size=batch)
        s["steps_per_period"], s["steps_on"] = 7, 3
        s["transient_substeps"], s["transient_k"] = 5, 7.0
    s["probes"] = [(nr - 1, nz // 2), (0, 1), (int(np.flatnonzero(np.diff(segs[0].astype(int)))[0]) + 1, nz - 2), (17, 0)]
    s["probe_every"] = 2
    return s


# ---------------------------------------------------------------- the paper's own device

# Fit coefficients of Tables 2 and 3, units J/(g K), W/(cm K), g/cm^3, cm, K, as
# printed and read in DESCENDING powers (reading G11: only then lambda_3 == 1e-3 as P:L276 says and
# every lambda_m is positive on 4.2-60 K).  tests/golden/paper_tables_2_3.txt holds the same numbers
# with their citations; tests/test_inputs.py checks the two against each other.
PAPER_CV_DESC = {   # a3 a2 a1 a0
    0: (0.0, 4.541e-4, -3.821e-3, 1e-2),
    1: (-6.514e-7, 1.057e-4, 2.366e-2, -6.619e-3),
    2: (-8.199e-7, 2.328e-5, -1.245e-4, 2.169e-4),
    3: (0.0, 0.0, 2.35e-2, 2.0e-2),
}
PAPER_LAM_DESC = {  # b4 b3 b2 b1 b0
    0: (7.029e-7, -9.317e-5, 2.306e-3, 1.166e-1, -1.139e-1),
    1: (0.0, -2.523e-7, 2.038e-5, -1.248e-4, 6.77e-3),
    2: (0.0, 3.03e-9, -6.369e-7, 1.05e-4, -2.729e-4),
    3: (0.0, 0.0, 0.0, 0.0, 1e-3),
}
PAPER_RHO = (8.92, 2.0, 2.0, 2.5)
# The printed graphite row (m = 2) has c_V < 0 above 22 K although the paper heats graphite past
# 40 K (reading G11): a_3 = -8.199e-7 is taken as a misprint of -8.199e-9 (c_V(60 K) = 0.075 J/(g K)).
# This is OUR substitution, not the paper's number; heat_create rejects the printed row.
PAPER_GRAPHITE_A3_SUBSTITUTE = -8.199e-9
PAPER_RADII_CM = (0.12, 0.125, 0.13, 0.1301)   # r_0, r_1, r_2, r_max
PAPER_Z0_CM = 4.0                              # end of the layered part (reading G10 of the garbled P:L241)
PAPER_ZMAX_CM = 5.0                            # P:L300 (z_0 = 4 cm, reading G10, is not needed on a rectangle)
PAPER_I0_A, PAPER_CHI0 = 0.363, 1.8            # I_0 P:L278; chi(T) = 1.8 / sqrt(T) Ohm cm, (25) P:L274
PAPER_T0, PAPER_TCRIT = 4.2, 42.2


def paper_layers(printed_graphite=False):
    out = []
    for m in range(4):
        a = list(PAPER_CV_DESC[m])
        if m == 2 and not printed_graphite:
            a[0] = PAPER_GRAPHITE_A3_SUBSTITUTE
        out.append(layer(poly(PAPER_LAM_DESC[m][::-1]), poly(a[::-1]), PAPER_RHO[m], is_heater=(m == 2),
                         src_shape=power(1.0, -0.5, 1.0)))   # chi(T) ~ T^-1/2, (25)
    return out


def paper_radial_nodes(nr=631):
    """The paper gives N = 631 but not the node distribution, only that the radial step must be
    at least an order of magnitude below the layer thicknesses.  OUR recipe: with
    u = (nr - 1) / 63 segments per unit, the outer insulator (1e-4 cm) gets u segments, the two 5e-3 cm
    layers 10 u each, the core the remaining 42 u with steps growing geometrically from the core /
    insulator interface towards the axis (first step = the insulator's).  Interfaces sit on nodes.
    Returns (r, interface node indices)."""
    assert (nr - 1) % 63 == 0 and nr >= 64, "nr - 1 must be a multiple of 63"
    u = (nr - 1) // 63
    r0, r1, r2, r3 = PAPER_RADII_CM
    n_core, n1, n2, n3 = 42 * u, 10 * u, 10 * u, u
    h1 = (r1 - r0) / n1
    # core: steps h1 * q^k, k = 0 .. n_core-1 from the interface inwards, summing to r0
    lo, hi = 1.0, 2.0
    for _ in range(200):
        q = (lo + hi) / 2
        tot = h1 * n_core if abs(q - 1) < 1e-15 else h1 * (q ** n_core - 1) / (q - 1)
        lo, hi = (q, hi) if tot < r0 else (lo, q)
    hk = h1 * q ** np.arange(n_core)
    hk *= r0 / hk.sum()
    core = r0 - np.concatenate([[0.0], np.cumsum(hk)])          # r0 ... 0
    core = core[::-1].copy()
    core[0] = 0.0
    seg1 = r0 + (r1 - r0) * np.arange(1, n1 + 1) / n1
    seg2 = r1 + (r2 - r1) * np.arange(1, n2 + 1) / n2
    seg3 = r2 + (r3 - r2) * np.arange(1, n3 + 1) / n3
    r = np.concatenate([core, seg1, seg2, seg3])
    assert r.size == nr and np.all(np.diff(r) > 0)
    return r, [n_core, n_core + n1, n_core + n1 + n2]


def paper_device(M=201, nr=631, tau=1e-5, printed_graphite=False, stepped=False):
    """The workload of the paper's section 5: radii 0.12 / 0.125 / 0.13 / 0.1301 cm,
    z_max = 5 cm, POLY laws of Tables 2-3, source chi(T) I_0^2 / S_2^2 in the conducting layer with
    I_0 = 363 mA, zero flux everywhere except T = 4.2 K at z_max (6), T_0 = 4.2 K, tau = 1e-5 s,
    t_prd = 25 ms, t_src = 1 ms, 100 transient sub-steps.  M = axial nodes (201 ... 1201, Table 4).
    Missing from the paper and filled in here: the radial node distribution (paper_radial_nodes) and
    the graphite c_V misprint (PAPER_GRAPHITE_A3_SUBSTITUTE).  CGS-like units: cm, g, s, W, J, K."""
    r, ifaces = paper_radial_nodes(nr)
    s = _base(nr, M, 1, 1, paper_layers(printed_graphite), seg_layers(nr, ifaces))
    s["r"] = r
    s["z"] = uniform_nodes(PAPER_ZMAX_CM, M)
    s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = NEUMANN0, NEUMANN0, NEUMANN0, dirichlet(PAPER_T0)
    s["T0"] = PAPER_T0
    S2 = math.pi * (PAPER_RADII_CM[2] ** 2 - PAPER_RADII_CM[1] ** 2)
    s["Q0"] = np.array([PAPER_CHI0 * PAPER_I0_A ** 2 / S2 ** 2])     # W/cm^3 times T^-1/2
    s["dt"] = float(tau)
    s["steps_per_period"] = int(round(25e-3 / tau))
    s["steps_on"] = int(round(1e-3 / tau))
    s["transient_substeps"], s["transient_k"] = 100, 7.0
    s["T_lo"], s["T_hi"] = 4.2, 60.0
    s["probes"] = [(nr - 1, 0), (nr - 1, M // 2), (0, 0)]           # Fig. 7 probe, mid surface, axis
    s["probe_every"] = 1
    s["name"] = f"paper device {nr}x{M}"
    if stepped:
        # Fig. 1 with reading G10 (z_0 = 4 cm): the layers 1-3 end at z_0, the copper core (r <= r_0, the
        # first interface node) goes on to the terminal at z_max; reading G24 of the non-rectangular Omega
        s["i_step"] = int(ifaces[0])
        s["j_step"] = int(round(PAPER_Z0_CM / PAPER_ZMAX_CM * (M - 1)))
        s["name"] += " stepped"
    return s

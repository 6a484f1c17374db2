"""Pins of the CPU oracle (oracle/heat_oracle.c) against what the paper and the mathematics fix.

Nothing here touches the CUDA path.  Each test names the passage of PAPER.md (P:Lnnn) it pins
and the mistake it would catch.  Closed forms are derived in DESIGN.md "Oracle pins".
"""
import math
import os

import numpy as np
import pytest
import scipy.linalg
import scipy.special

from oracle.heat_oracle import Oracle, law_eval, stable_dt
from paper_1408_5853_b200 import inputs as I

N0 = I.NEUMANN0
D = I.dirichlet


def one_material(nr, nz, R, L, k, cp, rho, r0=0.0, bcs=(N0, N0, N0, N0), heater=False, **kw):
    s = I._base(nr, nz, 1, 1, [I.layer(k, cp, rho, is_heater=heater)], I.seg_layers(nr, []))
    s["r"] = r0 + I.uniform_nodes(R - r0, nr)
    s["z"] = I.uniform_nodes(L, nz)
    s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = bcs
    s.update(kw)
    return s


# --------------------------------------------------------------------------- dense solve

BC_SETS = [
    (N0, N0, D(4.2), D(78.0)),      # BASELINE.json configs
    (N0, N0, N0, D(4.2)),           # the paper's own (6) P:L90-95
    (D(10.0), D(30.0), N0, N0),
    (N0, D(25.0), D(5.0), N0),
]


@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("bcs", BC_SETS)
@pytest.mark.parametrize("face_mode", [0, 1])
def test_sweep_equals_dense_solve(seed, bcs, face_mode):
    """(12),(14),(16),(17),(20) P:L131-192: the alpha/beta sweep must solve the tridiagonal
    system whose rows are (15) at the r boundaries, (13) at regular nodes and the flux
    relation (18) at interface nodes.  A wrong sign/index in (12), (17) or (20) fails here.
    Rows are equilibrated before the dense solve (they span ~12 orders of magnitude)."""
    s = I.random_spec(seed, nr=14, nz=9, nlayers=3, bcs=bcs, r0=0.0 if seed % 2 else 3e-4)
    s["face_mode"] = face_mode
    s["dt"] = 0.7 * stable_dt(s)
    o = Oracle(s)
    o.step(3)  # leave the initial data, enter the sub-stepped part of the schedule
    nr, nz = s["nr"], s["nz"]
    rows = [o.line_rows(0, j) for j in range(1, nz - 1)]
    o.step(1)
    T1 = o.field()
    for j, (A, B, C, F) in zip(range(1, nz - 1), rows):
        Mx = np.diag(B) + np.diag(A[1:], -1) + np.diag(C[:-1], 1)
        sc = 1.0 / np.abs(Mx).max(axis=1)
        x = np.linalg.solve(Mx * sc[:, None], F * sc)
        assert np.max(np.abs(x - T1[j])) < 2e-12 * np.max(np.abs(x))
        # second opinion: LAPACK dgtsv via scipy on the same equilibrated band
        ab = np.zeros((3, nr))
        ab[0, 1:] = (C * sc)[:-1]
        ab[1] = B * sc
        ab[2, :-1] = (A * sc)[1:]
        xb = scipy.linalg.solve_banded((1, 1), ab, F * sc)
        assert np.max(np.abs(xb - T1[j])) < 2e-12 * np.max(np.abs(x))


def test_r_boundary_and_interface_invariants():
    """(15) P:L158-161: T^_0 = T^_1 bitwise (alpha_0 = 1, beta_0 = 0), T^_N = T^_{N-1} to
    round-off; (18) P:L178-181: discrete flux continuity at interface nodes with
    lambda* = lambda(T_{i*,j}) of the OLD level."""
    s = I.random_spec(3, nr=21, nz=12, nlayers=4, laws="power")
    s["dt"] = 0.8 * stable_dt(s)
    o = Oracle(s)
    seg = s["seg_layer"][0]
    r = s["r"]
    for _ in range(5):
        T0 = o.field()
        o.step(1)
        T1 = o.field()
        inner = slice(1, s["nz"] - 1)
        assert np.array_equal(T1[inner, 0], T1[inner, 1])
        assert np.max(np.abs(T1[inner, -1] - T1[inner, -2])) < 1e-13 * np.max(T1)
        for i in range(1, s["nr"] - 1):
            if seg[i - 1] == seg[i]:
                continue
            lm = np.array([law_eval(s["layers"][seg[i - 1]]["k"], t) for t in T0[inner, i]])
            lp = np.array([law_eval(s["layers"][seg[i]]["k"], t) for t in T0[inner, i]])
            left = lm * (T1[inner, i] - T1[inner, i - 1]) / (r[i] - r[i - 1])
            right = lp * (T1[inner, i + 1] - T1[inner, i]) / (r[i + 1] - r[i])
            assert np.max(np.abs(left - right)) < 1e-11 * max(np.max(np.abs(left)), 1e-30) + 1e-9 * 0


# --------------------------------------------------------------------------- radial operator

def discrete_radial_steady(r, lam_seg, Ta, Tb, interface_nodes=()):
    """Fixed point of Lambda_i (10) with Dirichlet T_a, T_b and piecewise-constant lambda:
    inside a layer r_{k+1/2} lam (T_{k+1}-T_k)/h_{k+1} = Phi_m; across an interface node (18)
    gives Phi_m / r_{i*-1/2} = Phi_{m+1} / r_{i*+1/2}."""
    n = r.size
    rh = (r[1:] + r[:-1]) / 2
    h = np.diff(r)
    phi = np.ones(n - 1)  # flux r_{k+1/2} lam (T_{k+1}-T_k)/h_{k+1} per segment, up to a common factor
    for k in range(1, n - 1):
        phi[k] = phi[k - 1] * (rh[k] / rh[k - 1] if k in interface_nodes else 1.0)
    dT = phi * h / (lam_seg * rh)
    S = np.concatenate([[0.0], np.cumsum(dT)])
    return Ta + (Tb - Ta) * S / S[-1]


def test_radial_steady_state_single_material_closed_form():
    """(10),(13) P:L122,L140-143 with the G1 reading: z-uniform data, Dirichlet T_a, T_b at
    r_0 > 0 and r_N: the discrete steady state T_i = T_a + (T_b-T_a) S_i/S_N,
    S_i = sum_{k<i} h_{k+1}/(lam r_{k+1/2}), is a fixed point for ANY tau, and the iteration
    converges to it.  A wrong r_{i+-1/2}, h or hbar factor in A_i / C_i fails here."""
    rng = np.random.default_rng(5)
    nr, nz = 40, 6
    s = one_material(nr, nz, 2e-3, 1e-2, I.const(7.0), I.const(3.0), 100.0, r0=2e-4,
                     bcs=(D(10.0), D(60.0), N0, N0))
    s["r"] = 2e-4 + np.concatenate([[0], np.cumsum(rng.uniform(0.5, 1.5, nr - 1))]) * 1.8e-3 / (nr - 1)
    exact = discrete_radial_steady(s["r"], np.full(nr - 1, 7.0), 10.0, 60.0)
    s["T_init"] = np.tile(exact, (nz, 1))
    s["dt"] = 1e-3
    o = Oracle(s)
    o.step(3)
    assert np.max(np.abs(o.field() - exact)) < 1e-12
    # convergence from a different state (z-uniform => no explicit flux, tau unrestricted)
    s2 = dict(s, T_init=np.full((nz, nr), 20.0), dt=10.0)
    o2 = Oracle(s2)
    o2.step(400)
    assert np.max(np.abs(o2.field()[1:-1] - exact)) < 1e-9


def test_radial_steady_state_converges_to_log_r():
    """BASELINE north_star: T = A + B ln r between fixed temperatures; the discrete closed form
    above (which the oracle reproduces to round-off) converges to it at O(h^2) on a uniform grid."""
    errs = []
    for nr in (17, 33, 65):
        s = one_material(nr, 5, 2e-3, 1e-2, I.const(2.0), I.const(3.0), 100.0, r0=5e-4,
                         bcs=(D(10.0), D(60.0), N0, N0), T0=30.0, dt=50.0)
        o = Oracle(s)
        o.step(300)
        r = s["r"]
        exact = 10.0 + 50.0 * np.log(r / r[0]) / np.log(r[-1] / r[0])
        errs.append(np.max(np.abs(o.field()[2] - exact)))
    assert errs[0] / errs[1] > 3.5 and errs[1] / errs[2] > 3.5
    assert errs[2] < 2e-3


def test_radial_steady_state_layered():
    """(18),(20) P:L176-192: piecewise-constant lambda, Dirichlet r ends: the layered discrete
    steady state (flux constant inside a layer, (18) at the interface node) is a fixed point,
    and it approaches the continuous piecewise A_m + B_m ln r with lam_m B_m continuous at
    first order only."""
    def run(nr):
        R0, R1 = 4e-4, 2e-3
        i1 = (nr - 1) // 2
        s = I._base(nr, 5, 1, 1, [I.layer(I.const(3.0), I.const(2.0), 50.0),
                                  I.layer(I.const(40.0), I.const(5.0), 70.0)], I.seg_layers(nr, [i1]))
        s["r"] = R0 + I.uniform_nodes(R1 - R0, nr)
        s["z"] = I.uniform_nodes(1e-2, 5)
        s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = D(10.0), D(60.0), N0, N0
        lam_seg = np.where(np.arange(nr - 1) < i1, 3.0, 40.0)
        exact_d = discrete_radial_steady(s["r"], lam_seg, 10.0, 60.0, interface_nodes=(i1,))
        s["T_init"] = np.tile(exact_d, (5, 1))
        s["dt"] = 0.05
        o = Oracle(s)
        o.step(2)
        assert np.max(np.abs(o.field() - exact_d)) < 1e-12
        # continuous solution: T = 10 + q ln(r/R0)/3 (r<rs), continuous, flux q continuous
        rs = s["r"][i1]
        q = 50.0 / (math.log(rs / R0) / 3.0 + math.log(R1 / rs) / 40.0)
        r = s["r"]
        cont = np.where(r <= rs, 10.0 + q * np.log(r / R0) / 3.0,
                        10.0 + q * math.log(rs / R0) / 3.0 + q * np.log(r / rs) / 40.0)
        return np.max(np.abs(exact_d - cont))
    e = [run(n) for n in (21, 41, 81)]
    assert e[0] > e[1] > e[2]
    assert 1.6 < e[0] / e[1] < 2.6 and 1.6 < e[1] / e[2] < 2.6  # O(h)


# --------------------------------------------------------------------------- axial operator

def test_z_sine_growth_factor():
    """(8),(11),(13) P:L110,L125,L144 with the G2 reading: r-uniform field T_c + eps sin(n pi z/L),
    Dirichlet T_c at both ends, uniform eta, constant coefficients: the implicit r part is the
    identity and the amplitude is multiplied by exactly g = 1 - (4 a tau/eta^2) sin^2(n pi eta/2L),
    a = lam/(rho c), every step.  Catches a wrong eta factor, a wrong sign of Lambda_j and a
    wrong rho c / tau in B_i or F_i."""
    nr, nz, L = 9, 33, 2e-2
    lam, c, rho, Tc, eps, n = 4.0, 25.0, 800.0, 30.0, 2.0, 3
    s = one_material(nr, nz, 1e-3, L, I.const(lam), I.const(c), rho, bcs=(N0, N0, D(Tc), D(Tc)))
    z = s["z"]
    s["T_init"] = np.tile((Tc + eps * np.sin(n * math.pi * z / L))[:, None], (1, nr))
    s["T_init"][0] = Tc
    s["T_init"][-1] = Tc
    s["dt"] = 0.9 * stable_dt(s, 4.2, 100.0)
    eta = L / (nz - 1)
    a = lam / (rho * c)
    assert s["dt"] == pytest.approx(0.9 * eta * eta / (2 * a), rel=1e-12)   # (21) for constants
    g = 1 - 4 * a * s["dt"] / eta**2 * math.sin(n * math.pi * eta / (2 * L)) ** 2
    o = Oracle(s)
    K = 50
    o.step(K)
    exact = Tc + eps * g**K * np.sin(n * math.pi * z / L)
    assert np.max(np.abs(o.field() - exact[:, None])) < 5e-12   # 50 steps x few ulp of 30 K


def test_bessel_sine_mode_decay_rate():
    """BASELINE north_star "decay of a single Bessel/cosine mode for constant coefficients":
    J_0(mu_1 r/R) sin(pi z/L), mu_1 = 3.8317 (J_0' = 0 at the insulated wall).  The measured
    decay rate tends to a (mu_1^2/R^2 + pi^2/L^2) as h, tau -> 0 (first order: (15) is a
    first-order boundary row)."""
    mu1 = scipy.special.jn_zeros(1, 1)[0]
    R, L, lam, c, rho, Tc = 1e-3, 4e-3, 5.0, 20.0, 500.0, 30.0
    a = lam / (rho * c)
    rate_exact = a * (mu1**2 / R**2 + math.pi**2 / L**2)
    errs = []
    for nr, nz in ((17, 17), (33, 33), (65, 65)):
        s = one_material(nr, nz, R, L, I.const(lam), I.const(c), rho, bcs=(N0, N0, D(Tc), D(Tc)))
        mode = np.outer(np.sin(math.pi * s["z"] / L), scipy.special.j0(mu1 * s["r"] / R))
        s["T_init"] = Tc + mode
        s["T_init"][0] = Tc
        s["T_init"][-1] = Tc
        s["dt"] = 0.5 * stable_dt(s, 4.2, 100.0)
        o = Oracle(s)
        t_end = 0.3 / rate_exact
        K = int(round(t_end / s["dt"]))
        o.step(K)
        T = o.field() - Tc
        # project on the mode (interior nodes)
        amp = np.sum(T[1:-1, 1:-1] * mode[1:-1, 1:-1]) / np.sum(mode[1:-1, 1:-1] ** 2)
        rate = -math.log(amp) / (K * s["dt"])
        errs.append(abs(rate - rate_exact) / rate_exact)
    assert errs[0] > errs[1] > errs[2]
    assert errs[2] < 0.03
    assert errs[1] / errs[2] > 1.6


# --------------------------------------------------------------------------- source and energy

def test_lumped_heating():
    """(2)-(4),(13) P:L70-80,L144: one material flagged heater, all-Neumann sides, constant c,
    uniform state: every node rises by exactly Q0 tau/(rho c) per step while nu = 1."""
    s = one_material(11, 9, 1e-3, 1e-2, I.power(3.0, 1.5), I.const(40.0), 900.0, heater=True, T0=10.0)
    s["Q0"] = np.array([3e6])
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 10, 4, 0
    s["dt"] = 1e-4
    o = Oracle(s)
    dT = 3e6 * 1e-4 / (900.0 * 40.0)
    for k in range(1, 13):
        o.step(1)
        on_steps = sum(1 for q in range(k) if (q % 10) < 4)
        assert np.max(np.abs(o.field() - (10.0 + on_steps * dT))) < 1e-12


def _weights(r, z):
    h = np.diff(r)
    eta = np.diff(z)
    hbar = (h[1:] + h[:-1]) / 2
    etabar = (eta[1:] + eta[:-1]) / 2
    return r[1:-1] * hbar, etabar   # r_i hbar_i (i=1..N-1), etabar_j (j=1..M-1)


def _np_law(law, T):
    if law["kind"] == "const":
        return np.full_like(T, law["c"][0])
    if law["kind"] == "power":
        return law["c"][0] * (T / law["T_ref"]) ** law["c"][1]
    return sum(law["c"][k] * T**k for k in range(len(law["c"])))


def test_energy_identity_all_neumann_single_material():
    """BASELINE north_star "energy balance (source input = stored heat + boundary flux, to
    round-off)".  Summing (8) P:L110 weighted by r_i hbar_i etabar_j over regular nodes, the
    radial fluxes telescope and vanish at the Neumann rows (15), the axial fluxes telescope and
    vanish when the stored z-boundary lines equal their neighbours, so
        sum rho c(T^k) (T^ - T) w = tau sum X w
    for ARBITRARY T-dependent lambda on a non-uniform grid.  No lambda is evaluated here, so
    a non-conservative face coefficient, a wrong weight or a wrong source factor fails."""
    rng = np.random.default_rng(11)
    nr, nz = 19, 15
    kl, cl = I.power(30.0, 1.5), I.power(4.0, 3.0)
    s = one_material(nr, nz, 1e-3, 1e-2, kl, cl, 2700.0, heater=True)
    s["layers"][0]["src_shape"] = I.power(1.0, -0.5)          # chi(T) ~ T^-1/2, (25) P:L274
    s["r"] = np.concatenate([[0], np.cumsum(rng.uniform(0.5, 1.5, nr - 1))]) * 1e-3 / (nr - 1)
    s["z"] = np.concatenate([[0], np.cumsum(rng.uniform(0.7, 1.3, nz - 1))]) * 1e-2 / (nz - 1)
    T = rng.uniform(8.0, 60.0, size=(nz, nr))
    T[0], T[-1] = T[1], T[-2]
    s["T_init"] = T
    s["Q0"] = np.array([4e8])
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 50, 50, 0
    s["T_lo"], s["T_hi"] = 4.2, 100.0
    s["dt"] = 0.5 * stable_dt(s)
    wr, wz = _weights(s["r"], s["z"])
    W = np.outer(wz, wr)
    o = Oracle(s)
    for _ in range(4):
        T0 = o.field()
        o.step(1)
        T1 = o.field()
        Ti = T0[1:-1, 1:-1]
        stored = np.sum(2700.0 * _np_law(cl, Ti) * (T1[1:-1, 1:-1] - Ti) * W)
        source = s["dt"] * np.sum(4e8 * _np_law(s["layers"][0]["src_shape"], Ti) * W)
        assert stored == pytest.approx(source, rel=2e-12)


def test_energy_identity_dirichlet_z_and_interfaces():
    """Same identity with Dirichlet z ends (boundary flux of the OLD level enters) and several
    materials: across an interface node (18) equates lam* dT/h without the r_{i+-1/2} weights
    and with lam at T_{i*} instead of the face mean, so the two face fluxes Phi that the
    neighbouring regular rows use do not cancel; the identity holds to round-off only with
    that interface defect; without it the balance is off by ~1e-4."""
    s = I.random_spec(7, nr=23, nz=13, nlayers=3, laws="power", bcs=(N0, N0, D(6.0), D(70.0)))
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 50, 50, 0
    s["dt"] = 0.5 * stable_dt(s)
    r, z = s["r"], s["z"]
    seg = s["seg_layer"][0]
    nr, nz = s["nr"], s["nz"]
    wr, wz = _weights(r, z)
    h, eta = np.diff(r), np.diff(z)
    rh = (r[1:] + r[:-1]) / 2
    regular = np.array([seg[i - 1] == seg[i] for i in range(1, nr - 1)])
    o = Oracle(s)
    o.step(2)
    T0 = o.field()
    o.step(1)
    T1 = o.field()
    tau, amp = o.schedule(2)
    lhs = rhs = defect_free = 0.0
    for ii, i in enumerate(range(1, nr - 1)):
        if not regular[ii]:
            continue
        lay = s["layers"][seg[i]]
        Tc = T0[1:-1, i]
        rc = lay["rho"] * _np_law(lay["cp"], Tc)
        lhs += np.sum(rc * (T1[1:-1, i] - Tc) / tau * wr[ii] * wz)
        X = s["Q0"][0] * _np_law(lay["src_shape"], Tc) * amp if lay["is_heater"] else 0.0
        rhs += np.sum(X * wr[ii] * wz)
        # axial fluxes telescope: only the two boundary faces remain (old level)
        lam_top = _np_law(lay["k"], (T0[-2, i] + T0[-1, i]) / 2)
        lam_bot = _np_law(lay["k"], (T0[1, i] + T0[0, i]) / 2)
        rhs += wr[ii] * (lam_top * (T0[-1, i] - T0[-2, i]) / eta[-1] - lam_bot * (T0[1, i] - T0[0, i]) / eta[0])
    # interface defect: eta_bar_j * (Phi_{i*-1/2} - Phi_{i*+1/2}) with the regular rows' face fluxes
    defect = 0.0
    for i in range(1, nr - 1):
        if seg[i - 1] == seg[i]:
            continue
        lam_m = _np_law(s["layers"][seg[i - 1]]["k"], (T0[1:-1, i] + T0[1:-1, i - 1]) / 2)
        lam_p = _np_law(s["layers"][seg[i]]["k"], (T0[1:-1, i] + T0[1:-1, i + 1]) / 2)
        phi_m = rh[i - 1] * lam_m * (T1[1:-1, i] - T1[1:-1, i - 1]) / h[i - 1]
        phi_p = rh[i] * lam_p * (T1[1:-1, i + 1] - T1[1:-1, i]) / h[i]
        defect += np.sum(wz * (phi_m - phi_p))
    scale = abs(lhs) + abs(rhs) + abs(defect)
    assert abs(lhs - (rhs + defect)) < 1e-12 * scale
    assert abs(lhs - rhs) > 1e-8 * scale   # the defect is real: (18) is not conservative


def test_z_uniform_field_stays_z_uniform_with_neumann_z():
    """G16 ("constructed in a similar way" P:L164): with Neumann at both z ends a z-uniform
    field stays z-uniform (every line incl. the two boundary lines sees zero axial flux)."""
    s = I.random_spec(2, nr=15, nz=8, nlayers=2, laws="power", bcs=(N0, N0, N0, N0), source=True)
    prof = np.linspace(10, 50, 15)
    s["T_init"] = np.tile(prof, (8, 1))
    s["dt"] = 0.9 * stable_dt(s)
    o = Oracle(s)
    o.step(9)
    T = o.field()
    assert np.max(np.abs(T - T[3])) == 0.0
    assert np.max(np.abs(T[3] - prof)) > 1e-6


def test_dirichlet_lines_are_never_touched():
    """G17: Dirichlet z lines hold their value at every i, corners included, bitwise."""
    s = I.with_dt(I.config(0, nr=24, nz=20), stable_dt(I.config(0, nr=24, nz=20)))
    o = Oracle(s)
    o.step(40)
    T = o.field()
    assert np.all(T[0] == 4.2) and np.all(T[-1] == 78.0)


def test_maximum_principle_without_source():
    """Diagnostic: below the bound (21) and without a source the field stays
    inside [min, max] of the initial and boundary data."""
    s0 = I.config(1, nr=48, nz=48)
    s = I.with_dt(s0, stable_dt(s0))
    o = Oracle(s)
    for _ in range(20):
        o.step(25)
        T = o.field()
        assert T.min() >= 4.2 - 1e-12 and T.max() <= 78.0 + 1e-12


# --------------------------------------------------------------------------- schedule

def test_schedule_table():
    """(4) P:L79 and (22)+procedure P:L212-217 (G8: negative exponent, G9: sampled at the start
    of the step, G18: integer counters).  Independent closed form for two periods."""
    s = I.random_spec(0, source=True)
    s["steps_per_period"], s["steps_on"], s["transient_substeps"], s["transient_k"] = 12, 3, 100, 7.0
    s["dt"] = 1e-6
    o = Oracle(s)
    L = 100 + 12 - 1
    t = 0.0
    for k in range(2 * L + 5):
        tau, amp = o.schedule(k)
        q = k % L
        if q < 100:
            assert tau == 1e-6 / 100
            assert amp == pytest.approx(1.0 - math.exp(-q / 7.0), abs=1e-16)
            if q == 0:
                assert amp == 0.0
            if q == 50:   # "saturation approximately in the middle of the interval" P:L215
                assert amp > 0.999
        else:
            g = q - 99
            assert tau == 1e-6
            assert amp == (1.0 if g < 3 else 0.0)
        t += tau
    # one period of solver steps spans exactly steps_per_period * tau of simulated time
    assert sum(o.schedule(k)[0] for k in range(L)) == pytest.approx(12e-6, rel=1e-13)
    # Heaviside variant ("in a simple case"): no sub-steps
    s["transient_substeps"] = 0
    o = Oracle(s)
    for k in range(30):
        tau, amp = o.schedule(k)
        assert tau == 1e-6 and amp == (1.0 if (k % 12) < 3 else 0.0)


def test_transient_model_avoids_the_switch_on_jump():
    """P:L208, L225 (Fig. 3): without the transient model the source switch-on makes the heater
    temperature overshoot within the first tau; with the sub-stepped model the heater stays
    below the no-transient value after one tau of simulated time."""
    s0 = I.config(2, nr=40, nz=24)
    s = I.with_dt(s0, stable_dt(s0))
    a = Oracle(s)
    a.step(100)                        # 100 sub-steps = one tau
    b = Oracle(dict(s, transient_substeps=0))
    b.step(1)                          # one tau, Heaviside
    seg = s["seg_layer"][0]
    heater = [i for i in range(1, 39) if seg[i - 1] == seg[i] == 2]
    Ta, Tb = a.field()[12, heater], b.field()[12, heater]
    assert np.all(Ta > 20.0) and np.all(Tb > Ta)


# --------------------------------------------------------------------------- paper's numbers

def _golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_tables_2_3.txt")
    out = {"cv": {}, "lam": {}, "rho": {}}
    for line in open(path):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] in ("cv", "lam"):
            out[f[0]][int(f[1])] = [float(x) for x in f[2:]]
        elif f[0] == "rho":
            out["rho"][int(f[1])] = float(f[2])
        else:
            out[f[0]] = float(f[1])
    return out


def test_stability_bound_reproduces_the_papers_time_steps():
    """(21) P:L194-196 against the two time steps the paper prints (tests/golden/
    paper_tables_2_3.txt): tau = 1e-5 s "suitable" for the device and 2.5e-7 s for
    the M = 1201 timing grid both sit just under the bound evaluated with Tables 2-3
    read in DESCENDING powers (G11); the bound is decided by copper near 4.8 K
    (min rho c/lambda = 0.0387 s/cm^2).  Graphite (m = 2) is left out: its printed c_V row has
    a root at 22 K (G11) which would make min|rho c/lambda| = 0."""
    g = _golden()
    layers = []
    for m in (0, 1, 3):
        layers.append(I.layer(I.poly(g["lam"][m][::-1]), I.poly(g["cv"][m][::-1]), g["rho"][m]))
    for m, lay in zip((0, 1, 3), layers):
        for T in np.linspace(4.2, 60.0, 200):
            assert law_eval(lay["k"], T) > 0 and law_eval(lay["cp"], T) > 0
    assert law_eval(layers[2]["k"], 33.0) == 1e-3                       # lambda_3 = 1e-3
    bad = I.poly(g["lam"][0])                                           # ascending reading
    assert min(law_eval(bad, T) for T in np.linspace(4.2, 60.0, 200)) < 0
    limits = {}
    for M in (int(g["M_coarse"]), int(g["M_fine"])):
        nr = 8
        s = I._base(nr, M, 1, 1, layers, np.zeros(nr - 1, dtype=np.uint8))
        s["r"] = I.uniform_nodes(0.1301, nr)
        s["z"] = I.uniform_nodes(g["z_max_cm"], M)
        limits[M] = stable_dt(s, 4.2, 60.0)
    assert limits[201] == pytest.approx(1.21e-5, rel=0.01)
    assert limits[1201] == pytest.approx(3.36e-7, rel=0.01)
    assert g["tau_device"] < limits[201] < 1.35 * g["tau_device"]
    assert g["tau_timing"] < limits[1201] < 1.35 * g["tau_timing"]
    ratio = limits[201] / ((g["z_max_cm"] / 200) ** 2 / 2)
    assert ratio == pytest.approx(0.0387, rel=0.01)


# --------------------------------------------------------------------------- builds of the oracle

def test_batch_member_equals_single_run_bitwise():
    s0 = I.config(3, nr=40, nz=24, batch=3)
    s = I.with_dt(s0, stable_dt(s0))
    o = Oracle(s)
    o.step(130)
    for b in range(3):
        s1 = dict(s, batch=1, seg_layer=s["seg_layer"][b:b + 1], Q0=s["Q0"][b:b + 1])
        o1 = Oracle(s1)
        o1.step(130)
        assert np.array_equal(o1.field(), o.field(b))
    assert not np.array_equal(o.field(0), o.field(1))
    assert o.probes().shape == (130, 3, 1)


def test_openmp_build_is_bitwise_identical():
    s0 = I.config(2, nr=48, nz=40)
    s = I.with_dt(s0, stable_dt(s0))
    a, b = Oracle(s), Oracle(s, variant="omp")
    a.step(150)
    b.step(150)
    assert np.array_equal(a.field(), b.field())
    assert np.array_equal(a.probes(), b.probes())


def test_long_double_rounding_floor():
    """How much of the 1e-9 K parity budget fp64 rounding alone uses: the same
    code in x87 extended precision vs fp64 over config 0's full 1000 steps and a downscaled
    pulsed cell."""
    s0 = I.config(0)
    s = I.with_dt(s0, stable_dt(s0))
    a, b = Oracle(s), Oracle(s, variant="long")
    a.step(1000)
    b.step(1000)
    # measured 9.6e-11 K: the radial diffusion number lam tau/(rho c h^2) is ~44 in layer 3, so
    # each line solve has cond ~ 180 and loses ~20 ulp of 78 K per step
    assert np.max(np.abs(a.field() - b.field())) < 3e-10
    s0 = I.config(2, nr=64, nz=64)
    s = I.with_dt(s0, stable_dt(s0))
    a, b = Oracle(s), Oracle(s, variant="long")
    a.step(2000)
    b.step(2000)
    assert np.max(np.abs(a.field() - b.field())) < 1e-10


def test_config_generators_match_the_survey_numbers():
    """Derived quantities of the BASELINE.json configs."""
    s = I.with_dt(I.config(0), stable_dt(I.config(0)))
    assert s["dt"] == pytest.approx(2.0408e-4, rel=1e-4)
    assert [int(i) + 1 for i in np.flatnonzero(np.diff(s["seg_layer"][0]))] == [32, 50]
    s = I.with_dt(I.config(2), stable_dt(I.config(2)))
    assert s["steps_per_period"] == 11199033 and s["steps_on"] == 1119903
    assert s["steps"] == 5 * (11199033 + 99)
    s4 = I.config(4)
    assert [int(i) + 1 for i in np.flatnonzero(np.diff(s4["seg_layer"][0]))] == [4915, 6553, 7372]
    assert s4["probes"] == [(8191, 4096)]
    assert I.with_dt(s4, stable_dt(s4))["dt"] == pytest.approx(1.115e-10, rel=1e-3)
    s3 = I.config(3)
    assert s3["seg_layer"].shape == (256, 511) and s3["Q0"].min() >= 1e9 and s3["Q0"].max() <= 2e10

"""Pins of the oracle on the stepped (non-rectangular) domain, reading G24:
"N_j" of the grid (9) P:L117 and Fig. 1 -- the lines above z_{j_step} end at node i_step (the core reaching
the terminal); zero flux (6) on the two new faces: (15) at r = r_{i_step} for the short lines, and no
explicit flux through z = z_{j_step} for i > i_step.

  * every row of one step re-assembled in NumPy from r, z, T and the law parameters on the L-shaped
    domain (regular rows (13) with (11), interface rows (18), boundary rows (15), the nodes outside
    Omega untouched, the mirror nodes above the step face);
  * no heat leaves through the step faces: with T = T_d held only at the top of the core the whole of
    Omega relaxes to T_d, while the nodes outside keep the initial value they were given;
  * the descriptor checks.
Nothing here touches the CUDA path.
"""
import numpy as np
import pytest

from oracle.heat_oracle import Oracle, stable_dt
from paper_1408_5853_b200 import inputs as I

N0 = I.NEUMANN0
D = I.dirichlet


def np_law(law, T):
    T = np.asarray(T, dtype=np.float64)
    if law["kind"] == "const":
        return np.full_like(T, law["c"][0])
    if law["kind"] == "power":
        return law["c"][0] * (T / law["T_ref"]) ** law["c"][1]
    return sum(law["c"][k] * T**k for k in range(len(law["c"])))


def np_face(law, Ta, Tb, face_mode):
    if face_mode == 0:
        return np_law(law, (np.asarray(Ta) + np.asarray(Tb)) / 2)
    return (np_law(law, Ta) + np_law(law, Tb)) / 2


def stepped(seed, i_step, j_step, nr=19, nz=13, **kw):
    s = I.random_spec(seed, nr=nr, nz=nz, nlayers=3, **kw)
    s["i_step"], s["j_step"] = i_step, j_step
    s["probes"] = [(nr - 1, j_step), (1, nz - 2), (i_step, nz - 2)]
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 9, 9, 0
    s["dt"] = 0.9 * stable_dt(s)
    return s


def in_omega(s, i, j):
    return j <= s["j_step"] or i <= s["i_step"]


def check_step(s, T, X, tau, amp):
    """All rows of one step T -> X on the stepped domain; returns the largest relative row residual."""
    r, z, seg, fm = s["r"], s["z"], s["seg_layer"][0], s.get("face_mode", 0)
    nr, nz, i_s, j_s = s["nr"], s["nz"], s["i_step"], s["j_step"]
    worst = 0.0
    for j in range(1, nz - 1):
        N = nr - 1 if j <= j_s else i_s
        e_j, e_jp = z[j] - z[j - 1], z[j + 1] - z[j]
        ebar = (e_j + e_jp) / 2
        assert X[j, 0] == X[j, 1]                         # (15) at r = 0
        assert X[j, N] == pytest.approx(X[j, N - 1], rel=1e-14)   # (15),(17) at the end of the line, N = N_j
        for i in range(N + 1, nr):                        # outside Omega
            if j == j_s + 1:
                assert X[j, i] == X[j_s, i]               # mirror of the line below: no flux through the step face
            else:
                assert X[j, i] == T[j, i]
        for i in range(1, N):
            h_i, h_ip = r[i] - r[i - 1], r[i + 1] - r[i]
            if seg[i - 1] != seg[i]:
                la = float(np_law(s["layers"][seg[i - 1]]["k"], T[j, i]))
                lb = float(np_law(s["layers"][seg[i]]["k"], T[j, i]))
                lhs, rhs = la * (X[j, i] - X[j, i - 1]) / h_i, lb * (X[j, i + 1] - X[j, i]) / h_ip
                worst = max(worst, abs(lhs - rhs) / ((la / h_i + lb / h_ip) * abs(X[j, i])))   # flux continuity (18)
                continue
            lay = s["layers"][seg[i]]
            hbar = (h_i + h_ip) / 2
            r_mh, r_ph = (r[i] + r[i - 1]) / 2, (r[i] + r[i + 1]) / 2
            Tc = T[j, i]
            # the upper neighbour: outside Omega above the step face -> no flux (6)
            Tup = T[j + 1, i] if in_omega(s, i, j + 1) else Tc
            Tdn = T[j - 1, i]
            lam_mh = float(np_face(lay["k"], Tc, T[j, i - 1], fm))
            lam_ph = float(np_face(lay["k"], Tc, T[j, i + 1], fm))
            lam_jm = float(np_face(lay["k"], Tc, Tdn, fm))
            lam_jp = float(np_face(lay["k"], Tc, Tup, fm))
            rc = lay["rho"] * float(np_law(lay["cp"], Tc))
            Xs = s["Q0"][0] * float(np_law(lay["src_shape"], Tc)) * amp if lay["is_heater"] else 0.0
            A = -r_mh * lam_mh / (r[i] * hbar * h_i)
            C = -r_ph * lam_ph / (r[i] * hbar * h_ip)
            B = -A - C + rc / tau
            Lj = (lam_jp * (Tup - Tc) / e_jp - lam_jm * (Tc - Tdn) / e_j) / ebar
            F = rc / tau * Tc + Lj + Xs
            res = A * X[j, i - 1] + B * X[j, i] + C * X[j, i + 1] - F
            worst = max(worst, abs(res) / (abs(B * X[j, i]) + abs(F)))
    return worst


@pytest.mark.parametrize("seed,i_step,j_step", [(0, 7, 5), (1, 12, 2), (2, 3, 9), (3, 17, 10)])
def test_every_row_of_a_step_on_the_stepped_domain(seed, i_step, j_step):
    """i_step on an interface node, next to one, far from one; the step near the bottom and near the top."""
    s = stepped(seed, i_step, j_step)
    if seed == 0:   # put the step exactly on the first interface node, as in the paper's device (r_0)
        s["i_step"] = i_step = int(np.flatnonzero(np.diff(s["seg_layer"][0].astype(int)))[0]) + 1
        s["probes"][2] = (i_step, s["nz"] - 2)
    o = Oracle(s)
    o.step(3)
    T = o.field()
    tau, amp = o.schedule(3)
    o.step(1)
    X = o.field()
    assert float(np.max(np.abs(X - T))) > 1e-6
    assert check_step(s, T, X, tau, amp) < 1e-12
    # the check has teeth: the same fields fail it if the step is moved by one node or one line
    for di, dj in ((1, 0), (0, 1)):
        s2 = dict(s)
        s2["i_step"], s2["j_step"] = i_step + di, j_step + dj
        with pytest.raises(AssertionError):
            assert check_step(s2, T, X, tau, amp) < 1e-12
    # probes on the surface below the step, in the core above it and on the core's lateral surface
    P = o.probes()
    for p, (i, j) in enumerate(s["probes"]):
        assert P[-1, 0, p] == X[j, i]


def test_the_rectangle_is_the_special_case():
    s = I.random_spec(5, nr=15, nz=9, nlayers=3)
    s["dt"] = 0.9 * stable_dt(s)
    a = Oracle(s)
    s2 = dict(s)
    s2["i_step"], s2["j_step"] = 0, 0
    b = Oracle(s2)
    a.step(6)
    b.step(6)
    assert np.array_equal(a.field(), b.field())


def test_no_heat_leaves_through_the_step_faces():
    """Constant laws, no source, zero flux everywhere except T_d at the top of the core: Omega relaxes
    to T_d.  A face that leaked into the nodes outside Omega (which keep T0) would hold a gradient."""
    nr, nz, i_step, j_step, T0, Td = 12, 10, 5, 4, 20.0, 50.0
    lay = [I.layer(I.const(3.0), I.const(2.0), 1.5)]
    s = I._base(nr, nz, 1, 1, lay, I.seg_layers(nr, []))
    s["r"], s["z"] = I.uniform_nodes(1.0, nr), I.uniform_nodes(0.5, nz)
    s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = N0, N0, N0, D(Td)
    s["T0"] = T0
    s["i_step"], s["j_step"] = i_step, j_step
    s["T_lo"], s["T_hi"] = 1.0, 100.0
    s["dt"] = 0.9 * stable_dt(s)
    o = Oracle(s)
    omega = np.array([[j <= j_step or i <= i_step for i in range(nr)] for j in range(nz)])
    dev = []
    for _ in range(12):
        o.step(400)
        F = o.field()
        dev.append(float(np.max(np.abs(F[omega] - Td)[: -1])))
    assert all(b < a for a, b in zip(dev, dev[1:]) if a > 1e-9), dev
    assert dev[-1] < 1e-6 * abs(Td - T0), dev
    F = o.field()
    outside = ~omega
    outside[j_step + 1, :] = False                        # the mirror line follows the line below it
    outside[-1, :] = False                                # Dirichlet line
    assert np.all(F[outside] == T0)
    assert np.array_equal(F[j_step + 1, i_step + 1:], F[j_step, i_step + 1:])


@pytest.mark.parametrize("bad", [dict(j_step=0, i_step=5), dict(j_step=11, i_step=5), dict(j_step=4, i_step=1),
                                 dict(j_step=4, i_step=18), dict(j_step=4, i_step=7, probes=[(9, 8)])])
def test_descriptor_checks(bad):
    s = stepped(0, 7, 5)
    s.update(bad)
    with pytest.raises(Exception):
        Oracle(s)

"""Round-2 pins of the CPU oracle: the parts VERDICT r1 found without an independent check.

  * (13) P:L140-145 assembled directly in NumPy from r, z, T and the law parameters (no call into
    the oracle's `regular_row`) against `orc_line_rows`, both face modes: pins the row assembly
    the dense-solve pin takes on trust.
  * `face_mode = 1` (reading G3: lambda_{i+-1/2} = (lambda(T_a) + lambda(T_b))/2): energy
    identity with the NumPy side using the mean of the two lambdas, and a hand-computed 3-node
    line where the two modes give different, hand-computed A_i, C_i.
  * probe records (`append_probes`, S3 of SURVEY 8(c)): record k is the NEW level after solver step
    (k+1) * probe_every, bitwise, for probes on a regular node, on r = R, on a Dirichlet z line and
    on a Neumann z line.

Nothing here touches the CUDA path.
"""
import numpy as np
import pytest

from oracle.heat_oracle import Oracle, stable_dt
from paper_1408_5853_b200 import inputs as I

N0 = I.NEUMANN0
D = I.dirichlet


def np_law(law, T):
    """The three law kinds of the boundary spec written out in NumPy (P:L245-248 for POLY)."""
    T = np.asarray(T, dtype=np.float64)
    if law["kind"] == "const":
        return np.full_like(T, law["c"][0])
    if law["kind"] == "power":
        return law["c"][0] * (T / law["T_ref"]) ** law["c"][1]
    return sum(law["c"][k] * T**k for k in range(len(law["c"])))


def np_face(law, Ta, Tb, face_mode):
    """lambda at a half node: mode 0 = law at the mean temperature, mode 1 = mean of the laws."""
    if face_mode == 0:
        return np_law(law, (np.asarray(Ta) + np.asarray(Tb)) / 2)
    return (np_law(law, Ta) + np_law(law, Tb)) / 2


def np_rows_13(s, T, j, tau, amp, face_mode):
    """Rows (13) P:L140-145 of the regular nodes of line j, straight from the paper:
        A_i = -r_{i-1/2} lam_{i-1/2,j} / (r_i hbar_i h_i)
        C_i = -r_{i+1/2} lam_{i+1/2,j} / (r_i hbar_i h_{i+1})
        B_i = -A_i - C_i + rho c / tau
        F_i = rho c / tau T_ij + Lambda_j[T_ij] + X_ij,   Lambda_j (11) P:L125 with etabar_j
    Returns dict i -> (A, B, C, F) for regular nodes only."""
    r, z = s["r"], s["z"]
    seg = s["seg_layer"][0]
    out = {}
    for i in range(1, s["nr"] - 1):
        if seg[i - 1] != seg[i]:
            continue
        lay = s["layers"][seg[i]]
        h_i, h_ip = r[i] - r[i - 1], r[i + 1] - r[i]
        hbar = (h_i + h_ip) / 2
        e_j, e_jp = z[j] - z[j - 1], z[j + 1] - z[j]
        ebar = (e_j + e_jp) / 2
        r_mh, r_ph = (r[i] + r[i - 1]) / 2, (r[i] + r[i + 1]) / 2
        Tc = T[j, i]
        lam_mh = float(np_face(lay["k"], Tc, T[j, i - 1], face_mode))
        lam_ph = float(np_face(lay["k"], Tc, T[j, i + 1], face_mode))
        lam_jm = float(np_face(lay["k"], Tc, T[j - 1, i], face_mode))
        lam_jp = float(np_face(lay["k"], Tc, T[j + 1, i], face_mode))
        rc = lay["rho"] * float(np_law(lay["cp"], Tc))
        X = s["Q0"][0] * float(np_law(lay["src_shape"], Tc)) * amp if lay["is_heater"] else 0.0
        A = -r_mh * lam_mh / (r[i] * hbar * h_i)
        C = -r_ph * lam_ph / (r[i] * hbar * h_ip)
        Lj = (lam_jp * (T[j + 1, i] - Tc) / e_jp - lam_jm * (Tc - T[j - 1, i]) / e_j) / ebar
        out[i] = (A, -A - C + rc / tau, C, rc / tau * Tc + Lj + X)
    return out


@pytest.mark.parametrize("face_mode", [0, 1])
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_rows_13_assembled_in_numpy(seed, face_mode):
    """(13) P:L140-145 + (11) P:L125 + (2)-(4): an independent NumPy assembly of A, B, C, F on a
    random non-uniform grid with three materials, T-dependent laws and an active source must
    equal the rows the oracle's sweep consumes.  A dropped term, a wrong h / hbar / r_{i+-1/2},
    a wrong sign of Lambda_j or a wrong face rule (either mode) fails."""
    s = I.random_spec(seed, nr=15, nz=9, nlayers=3, r0=0.0 if seed % 2 else 2e-4)
    s["face_mode"] = face_mode
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 9, 9, 0   # source on, amp = 1
    s["dt"] = 0.5 * stable_dt(s)
    o = Oracle(s)
    o.step(2)
    T = o.field()
    tau, amp = o.schedule(2)
    assert amp == 1.0
    for j in range(1, s["nz"] - 1):
        A, B, C, F = o.line_rows(0, j)
        ref = np_rows_13(s, T, j, tau, amp, face_mode)
        assert len(ref) == s["nr"] - 2 - 2   # two interface nodes
        for i, (a, b, c, f) in ref.items():
            assert A[i] == pytest.approx(a, rel=1e-13)
            assert B[i] == pytest.approx(b, rel=1e-13)
            assert C[i] == pytest.approx(c, rel=1e-13)
            assert F[i] == pytest.approx(f, rel=1e-12)


def test_face_mode_hand_computed_three_node_line():
    """Reading G3, on numbers small enough to check by hand: one material,
    lambda(T) = 2 T^2 (T_ref = 1), nodes r = 1, 2, 3 (h = hbar = 1), line T = (1, 3, 5):
        mode 0: lam_{1-1/2} = 2 ((1+3)/2)^2 = 8,   lam_{1+1/2} = 2 ((3+5)/2)^2 = 32
        mode 1: lam_{1-1/2} = (2 + 18)/2   = 10,  lam_{1+1/2} = (18 + 50)/2   = 34
        A_1 = -r_{1/2} lam_{1-1/2} / (r_1 hbar h) = -(1.5/2) lam_-,  C_1 = -(2.5/2) lam_+
    so mode 0 gives A = -6, C = -40 and mode 1 gives A = -7.5, C = -42.5."""
    expect = {0: (-6.0, -40.0), 1: (-7.5, -42.5)}
    for mode, (A1, C1) in expect.items():
        s = I._base(3, 3, 1, 1, [I.layer(I.power(2.0, 2.0, 1.0), I.const(1.0), 1.0)], I.seg_layers(3, []))
        s["r"] = np.array([1.0, 2.0, 3.0])
        s["z"] = np.array([0.0, 1.0, 2.0])
        s["r_in"], s["r_out"], s["z_lo"], s["z_hi"] = N0, N0, N0, N0
        s["T_init"] = np.tile(np.array([1.0, 3.0, 5.0]), (3, 1))
        s["face_mode"] = mode
        s["dt"] = 0.25
        s["T_lo"], s["T_hi"] = 1.0, 5.0
        o = Oracle(s)
        A, B, C, F = o.line_rows(0, 1)
        assert A[1] == pytest.approx(A1, rel=1e-15)
        assert C[1] == pytest.approx(C1, rel=1e-15)
        # z-uniform data: Lambda_j = 0, no source; rho c / tau = 4
        assert B[1] == pytest.approx(-A1 - C1 + 4.0, rel=1e-15)
        assert F[1] == pytest.approx(4.0 * 3.0, rel=1e-15)


def _weights(r, z):
    h, eta = np.diff(r), np.diff(z)
    return r[1:-1] * (h[1:] + h[:-1]) / 2, (eta[1:] + eta[:-1]) / 2


@pytest.mark.parametrize("face_mode", [0, 1])
def test_energy_identity_both_face_modes(face_mode):
    """Energy identity of SURVEY 8(c) (source input = stored heat + z-boundary flux + interface
    defect, to round-off) with Dirichlet z ends and three materials, the NumPy side evaluating
    every face lambda by the rule of the mode under test.  With the other mode's rule on the
    NumPy side the balance is off by orders of magnitude more than round-off, so the oracle's
    face_mode-1 branch is checked against something that is not itself."""
    s = I.random_spec(7, nr=23, nz=13, nlayers=3, laws="power", bcs=(N0, N0, D(6.0), D(70.0)))
    s["face_mode"] = face_mode
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 50, 50, 0
    s["dt"] = 0.25 * stable_dt(s)
    r, z = s["r"], s["z"]
    seg = s["seg_layer"][0]
    nr = s["nr"]
    wr, wz = _weights(r, z)
    h, eta = np.diff(r), np.diff(z)
    rh = (r[1:] + r[:-1]) / 2
    o = Oracle(s)
    o.step(2)
    T0 = o.field()
    o.step(1)
    T1 = o.field()
    tau, amp = o.schedule(2)

    def balance(mode):
        lhs = rhs = defect = 0.0
        for ii, i in enumerate(range(1, nr - 1)):
            if seg[i - 1] != seg[i]:
                lam_m = np_face(s["layers"][seg[i - 1]]["k"], T0[1:-1, i], T0[1:-1, i - 1], mode)
                lam_p = np_face(s["layers"][seg[i]]["k"], T0[1:-1, i], T0[1:-1, i + 1], mode)
                phi_m = rh[i - 1] * lam_m * (T1[1:-1, i] - T1[1:-1, i - 1]) / h[i - 1]
                phi_p = rh[i] * lam_p * (T1[1:-1, i + 1] - T1[1:-1, i]) / h[i]
                defect += np.sum(wz * (phi_m - phi_p))
                continue
            lay = s["layers"][seg[i]]
            Tc = T0[1:-1, i]
            rc = lay["rho"] * np_law(lay["cp"], Tc)
            lhs += np.sum(rc * (T1[1:-1, i] - Tc) / tau * wr[ii] * wz)
            if lay["is_heater"]:
                rhs += np.sum(s["Q0"][0] * np_law(lay["src_shape"], Tc) * amp * wr[ii] * wz)
            lam_top = float(np_face(lay["k"], T0[-2, i], T0[-1, i], mode))
            lam_bot = float(np_face(lay["k"], T0[1, i], T0[0, i], mode))
            rhs += wr[ii] * (lam_top * (T0[-1, i] - T0[-2, i]) / eta[-1] - lam_bot * (T0[1, i] - T0[0, i]) / eta[0])
        return lhs, rhs, defect

    lhs, rhs, defect = balance(face_mode)
    scale = abs(lhs) + abs(rhs) + abs(defect)
    assert abs(lhs - (rhs + defect)) < 1e-12 * scale
    lhs2, rhs2, defect2 = balance(1 - face_mode)           # the other rule does not balance
    assert abs(lhs2 - (rhs2 + defect2)) > 1e-7 * scale


@pytest.mark.parametrize("probe_every", [1, 3])
@pytest.mark.parametrize("z_bcs", [(D(6.0), D(70.0)), (N0, N0), (N0, D(4.2))])
def test_probe_records_are_the_new_level_of_their_step(probe_every, z_bcs):
    """S3 of SURVEY 8(c) / 8(b) "Probes record T(i_p, j_p) of the new level after every
    probe_every-th step": record k must equal, bitwise, the field after solver step
    (k+1) * probe_every at the probe node -- on a regular node, on r = R (T_N = T_{N-1}, (15)
    P:L158-161), and on both z boundary lines (a Dirichlet line holds its value, a Neumann line
    copies its neighbour's new values, G16/G17).  A record taken from the old level, one step
    late, or from the wrong line fails; so does a cadence off by one."""
    nr, nz = 13, 11
    s = I.random_spec(4, nr=nr, nz=nz, nlayers=3, bcs=(N0, N0) + z_bcs)
    s["probes"] = [(5, 4), (nr - 1, nz // 2), (3, 0), (7, nz - 1), (0, 1)]
    s["probe_every"] = probe_every
    s["dt"] = 0.6 * stable_dt(s)
    nsteps = 14
    o = Oracle(s)        # records
    w = Oracle(s)        # witness: stepped one solver step at a time, fields read directly
    o.step(nsteps)
    rec = o.probes()
    assert rec.shape == (nsteps // probe_every, 1, 5)
    prev = w.field()
    for k in range(1, nsteps + 1):
        w.step(1)
        T = w.field()
        if k % probe_every:
            prev = T
            continue
        q = k // probe_every - 1
        for p, (i, j) in enumerate(s["probes"]):
            assert rec[q, 0, p] == T[j, i]
        # the record is of the NEW level: it differs from the level before the step
        assert rec[q, 0, 0] != prev[4, 5]
        # r = R row (15): the probe on i = N equals node N-1 to round-off
        assert rec[q, 0, 1] == pytest.approx(T[nz // 2, nr - 2], rel=1e-13)
        # z lines: Dirichlet holds the boundary value, Neumann copies the neighbouring line
        if z_bcs[0][0] == "dirichlet":
            assert rec[q, 0, 2] == s["T_init"][0, 0, 3]
        else:
            assert rec[q, 0, 2] == T[1, 3]
        if z_bcs[1][0] == "dirichlet":
            assert rec[q, 0, 3] == s["T_init"][0, nz - 1, 7]
        else:
            assert rec[q, 0, 3] == T[nz - 2, 7]
        prev = T


def test_probe_records_per_batch_member():
    """Record layout [record][batch][probe]: member b's column is member b's field."""
    s = I.random_spec(9, nr=12, nz=9, nlayers=2, batch=3)
    s["probes"] = [(4, 3), (11, 4)]
    s["probe_every"] = 2
    s["dt"] = 0.6 * stable_dt(s)
    o = Oracle(s)
    o.step(6)
    rec = o.probes()
    assert rec.shape == (3, 3, 2)
    for b in range(3):
        T = o.field(b)
        assert rec[2, b, 0] == T[3, 4] and rec[2, b, 1] == T[4, 11]
    assert rec[2, 0, 0] != rec[2, 1, 0]

"""Pins of the oracle's iterated variant `orc_step_picard` (reading G23).

T^(0) = T; T^(s+1) solves the scheme (8)-(20) with every lambda, c_V and X evaluated at T^(s), the
current level T staying where (8) has it (rho c_V (T^ - T)/tau, Lambda_j[T]).  Pinned by
  * iters = 1 is the paper's step, bitwise;
  * laws that do not depend on T: every iterate is the paper's step, bitwise;
  * an independent NumPy residual of the rows (13), (15), (18) with the coefficient field and the level
    kept apart: T^(2) solves the system whose coefficients sit at T^(1) to round-off -- and does NOT
    solve the one with the coefficients at T (so the laws really moved), nor the one where the level
    in the capacity / axial terms is replaced by the iterate (so T really stayed);
  * the iterates converge (differences shrink) to a fixed point of the fully implicit-in-coefficients
    system.
Nothing here touches the CUDA path.
"""
import numpy as np
import pytest

from oracle.heat_oracle import Oracle, stable_dt
from paper_1408_5853_b200 import inputs as I


def np_law(law, T):
    """The three law kinds of the boundary spec written out in NumPy (P:L245-248 for POLY)."""
    T = np.asarray(T, dtype=np.float64)
    if law["kind"] == "const":
        return np.full_like(T, law["c"][0])
    if law["kind"] == "power":
        return law["c"][0] * (T / law["T_ref"]) ** law["c"][1]
    return sum(law["c"][k] * T**k for k in range(len(law["c"])))


def np_face(law, Ta, Tb, face_mode):
    """lambda at a half node, P:L127 (reading G3)."""
    if face_mode == 0:
        return np_law(law, (np.asarray(Ta) + np.asarray(Tb)) / 2)
    return (np_law(law, Ta) + np_law(law, Tb)) / 2


def spec(seed, laws="mixed", **kw):
    s = I.random_spec(seed, nr=17, nz=9, nlayers=3, laws=laws, **kw)
    s["steps_per_period"], s["steps_on"], s["transient_substeps"] = 9, 9, 0   # source on from step 0, amp = 1
    s["Q0"] = s["Q0"] * 30.0                                                  # strong heating: the laws move within a step
    s["dt"] = 0.9 * stable_dt(s)
    return s


def residual(s, T, S, X, tau, amp):
    """max over the nodes of interior lines of |row(x)| / scale for the rows of the scheme with the laws
    at S, the level T and the candidate new level X; (13) P:L140-145, (11) P:L125, (15) P:L158-161,
    (18) P:L178-181 written out here, not taken from the oracle."""
    r, z, seg, fm = s["r"], s["z"], s["seg_layer"][0], s.get("face_mode", 0)
    nr, nz = s["nr"], s["nz"]
    worst = 0.0
    for j in range(1, nz - 1):
        e_j, e_jp = z[j] - z[j - 1], z[j + 1] - z[j]
        ebar = (e_j + e_jp) / 2
        # (15): T^_0 = T^_1, T^_N = T^_{N-1}  (both sides Neumann in random_spec's default)
        assert s["r_in"][0] == "neumann0" and s["r_out"][0] == "neumann0"
        worst = max(worst, abs(X[j, 0] - X[j, 1]), abs(X[j, -1] - X[j, -2]))
        for i in range(1, nr - 1):
            h_i, h_ip = r[i] - r[i - 1], r[i + 1] - r[i]
            if seg[i - 1] != seg[i]:
                la = float(np_law(s["layers"][seg[i - 1]]["k"], S[j, i]))
                lb = float(np_law(s["layers"][seg[i]]["k"], S[j, i]))
                lhs, rhs = la * (X[j, i] - X[j, i - 1]) / h_i, lb * (X[j, i + 1] - X[j, i]) / h_ip
                worst = max(worst, abs(lhs - rhs) / (abs(lhs) + abs(rhs) + 1e-300) * 1e-3)  # flux continuity, cancelling
                continue
            lay = s["layers"][seg[i]]
            hbar = (h_i + h_ip) / 2
            r_mh, r_ph = (r[i] + r[i - 1]) / 2, (r[i] + r[i + 1]) / 2
            Sc, Tc = S[j, i], T[j, i]
            lam_mh = float(np_face(lay["k"], Sc, S[j, i - 1], fm))
            lam_ph = float(np_face(lay["k"], Sc, S[j, i + 1], fm))
            lam_jm = float(np_face(lay["k"], Sc, S[j - 1, i], fm))
            lam_jp = float(np_face(lay["k"], Sc, S[j + 1, i], fm))
            rc = lay["rho"] * float(np_law(lay["cp"], Sc))
            Xs = s["Q0"][0] * float(np_law(lay["src_shape"], Sc)) * amp if lay["is_heater"] else 0.0
            A = -r_mh * lam_mh / (r[i] * hbar * h_i)
            C = -r_ph * lam_ph / (r[i] * hbar * h_ip)
            B = -A - C + rc / tau
            Lj = (lam_jp * (T[j + 1, i] - Tc) / e_jp - lam_jm * (Tc - T[j - 1, i]) / e_j) / ebar
            F = rc / tau * Tc + Lj + Xs
            res = A * X[j, i - 1] + B * X[j, i] + C * X[j, i + 1] - F
            worst = max(worst, abs(res) / (abs(B * X[j, i]) + abs(F)))
    return worst


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_one_iteration_is_the_papers_step_bitwise(seed):
    s = spec(seed)
    a, b = Oracle(s), Oracle(s)
    a.step(5)
    b.step_picard(5, 1)
    assert np.array_equal(a.field(), b.field())
    assert np.array_equal(a.probes(), b.probes())
    assert a.step_index == b.step_index == 5


@pytest.mark.parametrize("iters", [2, 3, 6])
def test_constant_laws_do_not_iterate(iters):
    """lambda, c_V, X independent of T: every iterate solves the same linear system."""
    s = spec(3, laws="const")
    for lay in s["layers"]:
        lay["src_shape"] = I.const(1.0)
    a, b = Oracle(s), Oracle(s)
    a.step(4)
    b.step_picard(4, iters)
    assert np.array_equal(a.field(), b.field())


@pytest.mark.parametrize("seed", [0, 1, 4])
def test_second_iterate_solves_the_system_with_the_laws_at_the_first(seed):
    s = spec(seed)
    o0, o1, o2 = Oracle(s), Oracle(s), Oracle(s)
    o0.step(3); o1.step(3); o2.step(3)
    T = o0.field()
    tau, amp = o0.schedule(3)
    assert amp == 1.0
    o1.step(1)                 # T^(1)
    o2.step_picard(1, 2)       # T^(2)
    T1, T2 = o1.field(), o2.field()
    assert float(np.max(np.abs(T2 - T1))) > 1e-6            # the laws moved: the iterates differ
    ok = residual(s, T, T1, T2, tau, amp)
    assert ok < 1e-12
    # a wrong reading fails by orders of magnitude: laws left at T, or the level replaced by the iterate
    assert residual(s, T, T, T2, tau, amp) > 1e4 * ok
    assert residual(s, T1, T1, T2, tau, amp) > 1e4 * ok
    # and T^(1) itself solves the system with the laws at T: the paper's scheme
    assert residual(s, T, T, T1, tau, amp) < 1e-12


def test_iterates_converge_to_the_fixed_point():
    s = spec(2)
    base = Oracle(s)
    base.step(3)
    T = base.field()
    tau, amp = base.schedule(3)
    fields = []
    for iters in (1, 2, 3, 4, 6, 12, 24):
        o = Oracle(s)
        o.step(3)
        o.step_picard(1, iters)
        fields.append(o.field())
    d = [float(np.max(np.abs(fields[k + 1] - fields[k]))) for k in range(len(fields) - 1)]
    assert d[0] > 1e-6
    assert all(d[k + 1] < 0.5 * d[k] or d[k + 1] < 1e-12 for k in range(len(d) - 1)), d
    assert d[-1] < 1e-11
    # the limit solves the scheme with the laws at the new level itself
    assert residual(s, T, fields[-1], fields[-1], tau, amp) < 1e-11
    assert residual(s, T, fields[0], fields[0], tau, amp) > 1e3 * residual(s, T, fields[-1], fields[-1], tau, amp)


def test_probes_and_counters_follow_the_solver_step():
    s = spec(1)
    s["probe_every"] = 2
    o = Oracle(s)
    o.step_picard(6, 3)
    assert o.step_index == 6
    P = o.probes()
    assert P.shape[0] == 3
    i, j = s["probes"][0]
    assert P[-1, 0, 0] == o.field()[j, i]

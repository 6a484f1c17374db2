"""The seeded edge-case generators used by the GPU parity tests produce descriptors that the
library accepts (no device needed for the validation) and that the oracle can advance."""
import numpy as np
import pytest

from paper_1408_5853_b200 import inputs as I


@pytest.mark.parametrize("nr,nz,batch,poly", [(128, 14, 2, True), (512, 24, 3, False), (512, 9, 5, True),
                                              (1024, 21, 2, False), (2048, 13, 2, True), (8192, 6, 1, False)])
def test_band_spec_is_a_valid_descriptor(nr, nz, batch, poly):
    from paper_1408_5853_b200 import binding
    from oracle.heat_oracle import Oracle
    s = I.band_spec(nr + nz, nr=nr, nz=nz, batch=batch, poly_laws=poly)
    seg = s["seg_layer"]
    assert seg.shape == (batch, nr - 1) and seg.dtype == np.uint8
    for b in range(batch):
        nodes = np.flatnonzero(np.diff(seg[b].astype(int))) + 1       # interface nodes
        assert len(nodes) == len(s["layers"]) - 1
        assert nodes[0] >= 2 and nodes[-1] <= nr - 3 and np.all(np.diff(nodes) >= 2)
        assert np.all(np.bincount(nodes // 8) <= 1)                   # one interface node per 8-node chunk
    assert binding.heat_workspace_bytes(s) > 0                        # the library's own validation
    lim = binding.heat_stable_dt(s)
    assert lim > 0
    s = dict(s, dt=0.8 * lim)
    o = Oracle(s)
    o.step(3)
    assert np.all(np.isfinite(o.field(batch - 1)))


def test_band_spec_is_seeded():
    a, b, c = I.band_spec(5, nr=512, nz=12), I.band_spec(5, nr=512, nz=12), I.band_spec(6, nr=512, nz=12)
    assert np.array_equal(a["T_init"], b["T_init"]) and np.array_equal(a["seg_layer"], b["seg_layer"])
    assert not np.array_equal(a["T_init"], c["T_init"])


def _golden():
    import os
    out = {"cv": {}, "lam": {}, "rho": {}}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_tables_2_3.txt")):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] in ("cv", "lam"):
            out[f[0]][int(f[1])] = tuple(float(x) for x in f[2:])
        elif f[0] == "rho":
            out["rho"][int(f[1])] = float(f[2])
    return out


def test_paper_device_uses_the_papers_printed_numbers():
    """inputs.paper_device carries Tables 2-3 and the densities exactly as printed
    (tests/golden/paper_tables_2_3.txt), except for the ONE stated substitution in the
    graphite c_V row; geometry, source and schedule are P:L241, L274-278."""
    g = _golden()
    for m in range(4):
        assert I.PAPER_CV_DESC[m] == g["cv"][m] and I.PAPER_LAM_DESC[m] == g["lam"][m]
        assert I.PAPER_RHO[m] == g["rho"][m]
    s = I.paper_device(201)
    assert s["nr"] == 631 and s["nz"] == 201 and s["dt"] == 1e-5
    assert s["steps_per_period"] == 2500 and s["steps_on"] == 100 and s["transient_substeps"] == 100
    r = s["r"]
    seg = s["seg_layer"][0]
    nodes = np.flatnonzero(np.diff(seg.astype(int))) + 1
    assert np.allclose(r[nodes], I.PAPER_RADII_CM[:3], rtol=1e-13) and r[-1] == pytest.approx(0.1301, rel=1e-13) and r[0] == 0.0
    # every thin layer is resolved by >= 10 radial steps
    assert nodes[1] - nodes[0] >= 10 and nodes[2] - nodes[1] >= 10 and 630 - nodes[2] >= 10
    assert s["Q0"][0] == pytest.approx(1.8 * 0.363 ** 2 / (np.pi * (0.13 ** 2 - 0.125 ** 2)) ** 2, rel=1e-14)
    lay = s["layers"]
    assert lay[2]["is_heater"] and lay[2]["src_shape"]["c"][1] == -0.5
    assert lay[2]["cp"]["c"][::-1][0] == I.PAPER_GRAPHITE_A3_SUBSTITUTE          # the substitution, and only there
    assert tuple(lay[1]["cp"]["c"][::-1]) == g["cv"][1] and tuple(lay[3]["k"]["c"][::-1]) == g["lam"][3]


def test_library_rejects_the_printed_graphite_row():
    """Reading G11: the graphite c_V row as printed is negative above 22 K; the library's descriptor
    validation (no device needed) refuses it and accepts the substituted row."""
    from paper_1408_5853_b200 import binding
    assert binding.heat_workspace_bytes(I.paper_device(201)) > 0
    assert binding.heat_workspace_bytes(I.paper_device(201, printed_graphite=True)) == 0


def test_paper_device_runs_on_the_oracle():
    from oracle.heat_oracle import Oracle, stable_dt
    s = I.paper_device(41, nr=64)
    assert s["dt"] < stable_dt(s) * 26       # (21) at M = 41 is 25 x the M = 201 bound; tau = 1e-5 is far inside
    o = Oracle(s)
    o.step(260)
    T = o.field()
    assert np.all(np.isfinite(T)) and T.min() >= 4.2 - 1e-9 and T.max() > 6.0     # the heater warms up during the 1 ms pulse
    assert np.all(T[-1] == 4.2)                                                   # Dirichlet terminal at z_max


def test_design_sweep_host_logic():
    """the source-control loop's host side (no device): the objective prefers coverage
    only while the surface cools below T_crit between pulses, the first generation contains the
    paper's design point, refinement keeps the best member and stays inside the admissible box, and
    every member's descriptor is accepted by the library (moving interface, Q0 from its own S_2)."""
    from paper_1408_5853_b200 import binding, design_sweep as D
    assert D.objective(0.75, 40.0, 42.2) == 0.75 and D.objective(0.9, 44.0, 42.2) < 0
    rng = np.random.Generator(np.random.PCG64(1))
    i0, th = D.first_generation(8, rng)
    assert i0[0] == 0.363 and th[0] == 100 and len(set(th.tolist())) > 4
    assert i0.min() >= D.I0_RANGE[0] and i0.max() <= D.I0_RANGE[1]
    J = np.array([0.1, 0.5, -0.2, 0.3, 0.0, 0.2, 0.4, 0.45])
    ni, nt = D.next_generation(i0, th, J, 0, 0.5, rng)
    assert ni[0] == i0[1] and nt[0] == th[1]
    assert np.all(np.abs(ni - i0[1]) <= 0.25 * (D.I0_RANGE[1] - D.I0_RANGE[0]) + 1e-12)
    assert nt.min() >= D.THICK_RANGE[0] and nt.max() <= D.THICK_RANGE[1]
    s = D.device_batch(i0[:3], th[:3], 41)
    assert s["batch"] == 3 and s["seg_layer"].shape == (3, 630)
    ref = I.paper_device(41)
    assert np.array_equal(s["seg_layer"][0], ref["seg_layer"][0]) and s["Q0"][0] == pytest.approx(ref["Q0"][0], rel=1e-12)
    for b in range(3):
        nodes = np.flatnonzero(np.diff(s["seg_layer"][b].astype(int))) + 1
        assert nodes[0] == 420 and nodes[2] == 620 and nodes[1] == 620 - th[b]
    assert binding.heat_workspace_bytes(s) > 0


def test_paper_device_stepped_geometry():
    """Fig. 1 with reading G10 / G24: the step sits on the first interface node (r_0 = 0.12 cm) and on z_0 = 4 cm."""
    from oracle.heat_oracle import Oracle
    s = I.paper_device(M=201, stepped=True)
    assert s["r"][s["i_step"]] == pytest.approx(0.12) and s["z"][s["j_step"]] == pytest.approx(4.0)
    assert s["seg_layer"][0][s["i_step"] - 1] == 0 and s["seg_layer"][0][s["i_step"]] == 1
    o = Oracle(s)
    o.step(120)
    F = o.field()
    assert np.all(F[s["j_step"] + 2:-1, s["i_step"] + 1:] == 4.2)      # outside Omega
    assert F[: s["j_step"] + 1].max() > 6.0

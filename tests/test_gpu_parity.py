"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Bar: max |T_gpu - T_oracle| <= 1e-9 K (BASELINE.json north_star);
integer / schedule work bit-exact.  Protocol per config: SURVEY.md 8(d) / DESIGN.md "Parity".
"""
import os

import numpy as np
import pytest

from paper_1408_5853_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL = 1e-9  # K, BASELINE.json north_star


@pytest.fixture(scope="module")
def bd():
    from paper_1408_5853_b200 import build as B
    B.build()
    from paper_1408_5853_b200 import binding
    binding.lib()
    return binding


def oracle_cls():
    from oracle.heat_oracle import Oracle
    return Oracle


def with_dt(bd, s0, safety=None):
    """tau from the library's own (21); the same spec then drives both sides."""
    lim = bd.heat_stable_dt(s0)
    if safety is None:
        return I.with_dt(s0, lim)
    s = dict(s0)
    s["dt"] = safety * lim
    return s


def compare(sim, orc, tol=TOL):
    err = 0.0
    for b in range(sim.batch):
        g, o = sim.field(b), orc.field(b)
        assert np.all(np.isfinite(g))
        err = max(err, float(np.max(np.abs(g - o))))
    assert err <= tol, f"max |dT| = {err:.3e} K"
    return err


# ----------------------------------------------------------------------------- small general cases

BC_SETS = [
    (I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2), I.dirichlet(78.0)),   # BASELINE.json configs
    (I.NEUMANN0, I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2)),          # the paper's (6) P:L90-95
    (I.dirichlet(10.0), I.dirichlet(30.0), I.NEUMANN0, I.NEUMANN0),
    (I.NEUMANN0, I.dirichlet(25.0), I.dirichlet(5.0), I.NEUMANN0),
]


@pytest.mark.parametrize("seed", range(4))
@pytest.mark.parametrize("bcs", BC_SETS)
@pytest.mark.parametrize("face_mode", [0, 1])
def test_random_small_problems(bd, seed, bcs, face_mode):
    """Non-uniform grids, odd sizes (ragged tails, scalar-load path), mixed law kinds, all BC
    kinds, source with sub-stepping, probes, batch of 2."""
    nr, nz = [(13, 11), (37, 9), (64, 20), (131, 7)][seed]
    s = I.random_spec(seed, nr=nr, nz=nz, nlayers=3, batch=2, bcs=bcs, r0=0.0 if seed % 2 else 3e-4)
    s["face_mode"] = face_mode
    s = with_dt(bd, s, 0.7)
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    for n in (1, 2, 17):
        sim.step(n)
        orc.step(n)
        compare(sim, orc)
    pg, dropped = sim.probes()
    po = orc.probes()
    assert dropped == 0 and pg.shape == po.shape
    assert np.max(np.abs(pg - po)) <= TOL
    sim.close()


VARIANTS = ["4,8", "4,16", "4,32", "8,32", "16,32", "8,64", "16,64", "8,128", "16,128", "8,256", "16,256",
            "8,512", "16,512", "8,1024"]


@pytest.mark.parametrize("variant", VARIANTS)
def test_every_kernel_variant(bd, variant, monkeypatch):
    """Each (M rows per thread, G threads per line) instantiation on a line that fills it
    only partly (ragged tail inside the last thread, whole idle threads) and on one that fills
    it exactly."""
    M, G = (int(x) for x in variant.split(","))
    monkeypatch.setenv("HEAT_VARIANT", variant)
    for nr in (M * G, M * G - M - 3):
        nz = 7 if nr > 2048 else 12
        s0 = I.config(2, nr=nr, nz=nz)
        # keep eta = 10 h as in the BASELINE configs (L/R = 10, nr = nz): otherwise the line
        # systems of a long thin grid are ill-conditioned and rounding, not the kernel, is tested
        s0["z"] = I.uniform_nodes(10.0 * (nz - 1) * 2e-3 / (nr - 1), nz)
        s = with_dt(bd, s0)
        sim, orc = bd.HeatSim(s), oracle_cls()(s)
        assert sim.kernel_name == f"line<M={M},G={G}>"
        sim.step(120)
        orc.step(120)
        compare(sim, orc)
        sim.close()


BAND_CASES = [
    # nr, nz, batch, poly laws, bcs, HEAT_BAND_NT
    (512, 24, 3, False, None, 256),
    (512, 9, 5, True, BC_SETS[1], 256),        # 5 bands on 4 groups per CTA: ragged last round
    (1024, 21, 2, False, BC_SETS[2], 256),     # Dirichlet r boundaries
    (2048, 19, 1, True, BC_SETS[3], 256),
    (4096, 12, 1, False, None, 256),           # cluster of 2 CTAs per line
    (8192, 7, 1, False, BC_SETS[1], 256),      # cluster of 4, Neumann z_lo
    (512, 24, 3, False, None, 128),
    (2048, 13, 2, True, BC_SETS[3], 128),      # cluster of 2 at 128 threads
    (8192, 6, 1, False, None, 128),            # cluster of 8 (non-portable size)
]


@pytest.mark.parametrize("case", BAND_CASES, ids=lambda c: f"nr{c[0]}-nz{c[1]}-b{c[2]}-{'poly' if c[3] else 'pow'}-nt{c[5]}")
def test_band_kernel_edge_cases(bd, case, monkeypatch):
    """The band kernel (the one bench.py times) on seeded problems built to hit its special
    paths: interface nodes at the first / last / middle row of a thread's 8-node chunk, square
    root, power and degree-4 polynomial laws side by side in one warp, every BC kind, non-uniform
    z, random initial field, source with sub-steps, probes on boundary / interface / Dirichlet
    nodes, ragged band partition, clusters of 1, 2, 4 and 8 CTAs per line."""
    nr, nz, batch, poly, bcs, nt = case
    monkeypatch.setenv("HEAT_KERNEL", "band")   # the third-generation kernel (wband takes precedence otherwise)
    monkeypatch.setenv("HEAT_BAND_NT", str(nt))
    s = I.band_spec(nr + nz, nr=nr, nz=nz, batch=batch, bcs=bcs, poly_laws=poly)
    s = with_dt(bd, s, 0.8)
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp" if nr * nz > 30000 else "double")
    assert sim.kernel_name.startswith("band<") and sim.kernel_name.endswith(f"NT={nt}>"), sim.kernel_name
    for n in (1, 6, 13):
        sim.step(n)
        orc.step(n)
        compare(sim, orc)
    pg, dropped = sim.probes()
    po = orc.probes()
    assert dropped == 0 and pg.shape == po.shape
    assert np.max(np.abs(pg - po)) <= TOL
    sim.close()


WBAND_CASES = [
    # nr, nz, batch, poly laws, bcs, HEAT_WBAND_NW
    (512, 24, 3, False, None, 4),              # one warp per line, four lines per CTA
    (512, 9, 5, True, BC_SETS[1], 4),          # 35 bands of 1..: ragged last round, Neumann z_lo
    (1024, 21, 2, False, BC_SETS[2], 4),       # two warps per line, Dirichlet r boundaries
    (2048, 19, 1, True, BC_SETS[3], 4),        # a CTA per line
    (4096, 12, 1, False, None, 4),             # cluster of 2 CTAs per line
    (8192, 7, 1, False, BC_SETS[1], 4),        # cluster of 4, Neumann z_lo
    (8192, 6, 2, True, None, 2),               # cluster of 8 CTAs of 2 warps
    (8192, 9, 1, False, BC_SETS[3], 8),        # cluster of 2 CTAs of 8 warps
]


@pytest.mark.parametrize("case", WBAND_CASES, ids=lambda c: f"nr{c[0]}-nz{c[1]}-b{c[2]}-{'poly' if c[3] else 'pow'}-nw{c[5]}")
def test_wband_kernel_edge_cases(bd, case, monkeypatch):
    """The warp-autonomous band kernel (the one bench.py times) on the band_spec problems:
    interface nodes at the first / last / middle row of a thread's chunk, square root, power and
    degree-4 polynomial laws side by side in one warp, every BC kind, non-uniform z, random
    initial field, source with sub-steps, probes on boundary / interface / Dirichlet nodes,
    ragged band partition, 1..16 warps per line in clusters of 1, 2, 4 and 8 CTAs."""
    nr, nz, batch, poly, bcs, nw = case
    monkeypatch.setenv("HEAT_KERNEL", "wband")   # the register version (tband takes precedence otherwise)
    monkeypatch.setenv("HEAT_WBAND_NW", str(nw))
    s = I.band_spec(nr + nz, nr=nr, nz=nz, batch=batch, bcs=bcs, poly_laws=poly, chunk=16)
    s = with_dt(bd, s, 0.8)
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp" if nr * nz > 30000 else "double")
    assert sim.kernel_name.startswith(f"wband<WL={nr // 512},NW={nw},"), sim.kernel_name
    for n in (1, 6, 13):
        sim.step(n)
        orc.step(n)
        compare(sim, orc)
    pg, dropped = sim.probes()
    po = orc.probes()
    assert dropped == 0 and pg.shape == po.shape
    assert np.max(np.abs(pg - po)) <= TOL
    sim.close()


TBAND_CASES = [
    # nr, nz, batch, poly laws, bcs, HEAT_TBAND_NW
    (512, 24, 3, False, None, 4),              # one warp per line, four lines per CTA
    (512, 9, 5, True, BC_SETS[1], 4),          # ragged last round, Neumann z_lo
    (1024, 21, 2, False, BC_SETS[2], 4),       # two warps per line, Dirichlet r boundaries
    (2048, 19, 1, True, BC_SETS[3], 4),        # a CTA per line
    (4096, 12, 1, False, None, 4),             # cluster of 2 CTAs per line
    (4096, 10, 2, True, BC_SETS[2], 8),        # a CTA of 8 warps per line (default for nr = 4096)
    (8192, 7, 1, False, BC_SETS[1], 4),        # cluster of 4, Neumann z_lo
    (8192, 6, 2, True, None, 8),               # cluster of 2 CTAs of 8 warps
    (8192, 9, 1, False, BC_SETS[3], 16),       # one CTA of 16 warps per line, no cluster (default for nr = 8192)
]


@pytest.mark.parametrize("case", TBAND_CASES, ids=lambda c: f"nr{c[0]}-nz{c[1]}-b{c[2]}-{'poly' if c[3] else 'pow'}-nw{c[5]}")
def test_tband_kernel_edge_cases(bd, case, monkeypatch):
    """The tensor-memory band kernel (the one bench.py times) on the band_spec problems: interface
    nodes at the first / last / middle row of a thread's chunk, square root, power and degree-4
    polynomial laws side by side in one warp, every BC kind, non-uniform z, random initial field,
    source with sub-steps, probes on boundary / interface / Dirichlet nodes, ragged band
    partition, 1..16 warps per line in clusters of 1, 2 and 4 CTAs."""
    nr, nz, batch, poly, bcs, nw = case
    monkeypatch.setenv("HEAT_TBAND_NW", str(nw))
    s = I.band_spec(nr + nz, nr=nr, nz=nz, batch=batch, bcs=bcs, poly_laws=poly, chunk=16)
    s = with_dt(bd, s, 0.8)
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp" if nr * nz > 30000 else "double")
    assert sim.kernel_name.startswith(f"tband<WL={nr // 512},NW={nw},"), sim.kernel_name
    for n in (1, 6, 13):
        sim.step(n)
        orc.step(n)
        compare(sim, orc)
    pg, dropped = sim.probes()
    po = orc.probes()
    assert dropped == 0 and pg.shape == po.shape
    assert np.max(np.abs(pg - po)) <= TOL
    sim.close()


def test_tband_kernel_band_length_does_not_change_the_result(bd, monkeypatch):
    """The partition of the lines into bands is a scheduling choice: the field is bitwise the
    same for bands of 1, 3 and all lines."""
    s = with_dt(bd, I.band_spec(7, nr=1024, nz=20, batch=2, chunk=16), 0.8)
    out = []
    for bl in ("1", "3", "18"):
        monkeypatch.setenv("HEAT_BAND_LINES", bl)
        sim = bd.HeatSim(s)
        assert sim.kernel_name.startswith("tband<"), sim.kernel_name
        sim.step(9)
        out.append(sim.fields())
        sim.close()
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])


def test_wband_kernel_band_length_does_not_change_the_result(bd, monkeypatch):
    """The partition of the lines into bands is a scheduling choice: the field is bitwise the
    same for bands of 1, 3 and all lines."""
    s = with_dt(bd, I.band_spec(7, nr=1024, nz=20, batch=2, chunk=16), 0.8)
    out = []
    monkeypatch.setenv("HEAT_KERNEL", "wband")
    for bl in ("1", "3", "18"):
        monkeypatch.setenv("HEAT_BAND_LINES", bl)
        sim = bd.HeatSim(s)
        assert sim.kernel_name.startswith("wband<"), sim.kernel_name
        sim.step(9)
        out.append(sim.fields())
        sim.close()
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])


def test_band_kernel_band_length_does_not_change_the_result(bd, monkeypatch):
    """The partition of the lines into bands is a scheduling choice: the field is bitwise the
    same for bands of 1, 3 and all lines."""
    s = with_dt(bd, I.band_spec(7, nr=512, nz=20, batch=2), 0.8)
    out = []
    monkeypatch.setenv("HEAT_KERNEL", "band")
    for bl in ("1", "3", "18"):
        monkeypatch.setenv("HEAT_BAND_LINES", bl)
        sim = bd.HeatSim(s)
        sim.step(9)
        out.append(sim.fields())
        sim.close()
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])


@pytest.mark.parametrize("nr", [128, 256, 512, 1024, 2048, 4096, 8192])
@pytest.mark.parametrize("face_mode", [0, 1])
def test_tma_kernel_variants(bd, nr, face_mode, monkeypatch):
    """The TMA line kernel (the general fast path: any law kind, both face modes; heat_create
    picks it when the band kernel does not cover the descriptor) on every line length it is
    instantiated for, on the band kernel's edge-case problems."""
    monkeypatch.setenv("HEAT_KERNEL", "tma")
    nz = 9 if nr >= 2048 else 14
    s = I.band_spec(3 * nr + face_mode, nr=nr, nz=nz, batch=2 if nr <= 1024 else 1, poly_laws=(nr // 128) % 2 == 1,
                    bcs=BC_SETS[(nr // 128) % 4])
    s["face_mode"] = face_mode
    # the mean of two lambdas (face_mode 1) on a random field of 5..80 K exceeds lambda at the mean
    # temperature by far: keep the explicit part well inside its stability range
    s = with_dt(bd, s, 0.8 if face_mode == 0 else 0.25)
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp" if nr * nz > 30000 else "double")
    assert sim.kernel_name.startswith("tma<"), sim.kernel_name
    for n in (1, 7, 12):
        sim.step(n)
        orc.step(n)
        compare(sim, orc)
    pg, dropped = sim.probes()
    assert dropped == 0 and np.max(np.abs(pg - orc.probes())) <= TOL
    sim.close()


def test_schedule_table_is_bit_exact(bd):
    """(4) P:L79, (22) P:L212-217: the library's (tau_k, amp_k) equals the oracle's, bitwise."""
    s = I.random_spec(0, source=True)
    s["steps_per_period"], s["steps_on"], s["transient_substeps"], s["transient_k"] = 12, 3, 100, 7.0
    s["dt"] = 1e-6
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    for k in range(2 * 111 + 5):
        assert sim.schedule(k) == orc.schedule(k)
    s["transient_substeps"] = 0
    sim2, orc2 = bd.HeatSim(s), oracle_cls()(s)
    for k in range(30):
        assert sim2.schedule(k) == orc2.schedule(k)


def test_set_get_field_and_step_index(bd):
    """Checkpoint / resume: heat_get_field -> heat_set_field reproduces the run bitwise."""
    s = with_dt(bd, I.config(2, nr=96, nz=40))
    a = bd.HeatSim(s)
    a.step(150)
    snap, k = a.field(0), a.step_index
    a.step(77)
    ref = a.field(0)
    b = bd.HeatSim(s)
    b.set_field(0, snap, k)
    b.step(77)
    assert np.array_equal(b.field(0), ref)
    c = bd.HeatSim(s)
    c.set_field(0, a._torch.from_numpy(snap).cuda(), k)   # device source
    c.step(77)
    assert np.array_equal(c.field_device(0).cpu().numpy(), ref)


def test_batch_member_equals_single_run_bitwise(bd):
    """Cell b of a batch run == the same cell run alone, bitwise on the GPU."""
    s = with_dt(bd, I.config(3, nr=128, nz=40, batch=5))
    sim = bd.HeatSim(s)
    sim.step(140)
    for b in (0, 3, 4):
        s1 = dict(s, batch=1, seg_layer=s["seg_layer"][b:b + 1], Q0=s["Q0"][b:b + 1])
        one = bd.HeatSim(s1)
        one.step(140)
        assert np.array_equal(one.field(0), sim.field(b))
    assert not np.array_equal(sim.field(0), sim.field(1))


def test_dirichlet_lines_and_r_boundary_rows(bd):
    """G17: Dirichlet z lines are never touched; (15): T^_0 = T^_1 bitwise."""
    s = with_dt(bd, I.config(1, nr=100, nz=30))
    sim = bd.HeatSim(s)
    sim.step(33)
    T = sim.field(0)
    assert np.all(T[0] == 4.2) and np.all(T[-1] == 78.0)
    assert np.array_equal(T[1:-1, 0], T[1:-1, 1])
    assert np.max(np.abs(T[1:-1, -1] - T[1:-1, -2])) < 1e-12


def test_probe_buffer_overflow_is_counted(bd):
    s = with_dt(bd, I.config(2, nr=64, nz=24))
    sim = bd.HeatSim(s, probe_records=10)
    sim.step(25)
    p, dropped = sim.probes()
    assert p.shape == (10, 1, 1) and dropped == 15
    sim.step(4)
    p, dropped = sim.probes()
    assert p.shape == (4, 1, 1) and dropped == 0


# ----------------------------------------------------------------------------- BASELINE.json configs

def test_config0_full_length(bd):
    """configs[0]: 64x64 constant coefficients, all 1000 steps."""
    s = with_dt(bd, I.config(0))
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    sim.step(s["steps"])
    orc.step(s["steps"])
    compare(sim, orc)


def test_config1_full_length(bd):
    """configs[1]: 512x512 nonlinear 4-layer cell, 2000 steps from the initial condition."""
    s = with_dt(bd, I.config(1))
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp")
    for _ in range(4):
        sim.step(500)
        orc.step(500)
        compare(sim, orc)


def test_config2_windows(bd):
    """configs[2]: 2048x2048 with pulse heating.  W1 = steps 0..299 from the initial condition
    (100 sub-steps + 200 steps); W2 / W3 = snapshot-seeded windows across switch-off and across
    the next switch-on (the GPU field at the window start seeds the oracle)."""
    s = with_dt(bd, I.config(2))
    assert s["steps_per_period"] == 11199033
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp")
    sim.step(300)
    orc.step(300)
    compare(sim, orc)
    pg, _ = sim.probes()
    assert np.max(np.abs(pg - orc.probes())) <= TOL
    nsub, P, S = s["transient_substeps"], s["steps_per_period"], s["steps_on"]
    off = nsub + S - 1                      # first solver step with amp = 0
    for start in (off - 20, nsub + P - 1 - 20):
        snap = sim.field(0)
        sim.set_field(0, snap, start)
        orc.set_field(0, snap, start)
        sim.step(60)
        orc.step(60)
        amps = [sim.schedule(start + q)[1] for q in range(60)]
        assert len(set(amps)) > 1           # the window really crosses a switch
        compare(sim, orc)


@pytest.mark.parametrize("n", [64, 128])
def test_config2_downscaled_full_length(bd, n):
    """configs[2] physics on n x n nodes, all 5 periods (5.3e4 steps at 64^2, 2.2e5 at 128^2): drift check,
    field and probe trace."""
    s = with_dt(bd, I.config(2, nr=n, nz=n))
    sim, orc = bd.HeatSim(s, probe_records=s["steps"] + 8), oracle_cls()(s, variant="omp" if n > 64 else "double")
    sim.step(s["steps"])
    orc.step(s["steps"])
    compare(sim, orc)
    pg, dropped = sim.probes()
    po = orc.probes()
    assert dropped == 0 and pg.shape == po.shape == (s["steps"], 1, 1)
    assert np.max(np.abs(pg - po)) <= TOL


def test_config3_batch_sample(bd):
    """configs[3]: 256 cells of 512x512.  The whole batch runs on the GPU; cells first, last,
    max Q0 and max heater thickness are checked against single-cell oracle runs: 300 steps from
    the initial condition, then a snapshot-seeded window across switch-off."""
    s = with_dt(bd, I.config(3))
    sim = bd.HeatSim(s)
    sim.step(300)
    cells = sorted({0, 255, int(np.argmax(s["Q0"])), int(np.argmax(s["heater_thickness_mm"]))})
    orcs = {}
    for b in cells:
        s1 = dict(s, batch=1, seg_layer=s["seg_layer"][b:b + 1], Q0=s["Q0"][b:b + 1])
        o = oracle_cls()(s1, variant="omp")
        o.step(300)
        assert np.max(np.abs(sim.field(b) - o.field(0))) <= TOL
        orcs[b] = o
    start = s["transient_substeps"] + s["steps_on"] - 1 - 15
    for b in cells:
        snap = sim.field(b)
        orcs[b].set_field(0, snap, start)
    snaps = sim._torch.stack([sim.field_device(b) for b in range(sim.batch)])
    for b in range(sim.batch):
        sim.set_field(b, snaps[b].contiguous(), start)
    sim.step(40)
    for b in cells:
        orcs[b].step(40)
        assert np.max(np.abs(sim.field(b) - orcs[b].field(0))) <= TOL


def test_config4_windows(bd):
    """configs[4]: 8192x8192, the launch configuration bench.py times.  10 steps from the
    initial condition; then the GPU runs on to step 9990 and a snapshot-seeded window
    9990 -> 10000 is compared (probe every 100 steps)."""
    s = with_dt(bd, I.config(4))
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp")
    sim.step(10)
    orc.step(10)
    compare(sim, orc)
    sim.step(9980)
    snap = sim.field(0)
    orc.set_field(0, snap, 9990)
    sim.step(10)
    orc.step(10)
    compare(sim, orc)
    pg, dropped = sim.probes()
    assert pg.shape == (100, 1, 1) and dropped == 0
    assert abs(pg[-1, 0, 0] - orc.field(0)[s["probes"][0][1], s["probes"][0][0]]) <= TOL


# ----------------------------------------------------------------------------- the paper's own device (f1)

def test_paper_device_windows(bd):
    """SURVEY 8(f) f1, the workload of the paper's section 5 on its 631 x 201 grid (non-uniform r,
    POLY laws of Tables 2-3, chi(T) ~ T^-1/2 source, Neumann z = 0 / Dirichlet 4.2 K at z_max):
    from the initial condition through the 100 transient sub-steps, across switch-off (snapshot
    seeded) and across the next switch-on."""
    s = I.paper_device(201)
    sim, orc = bd.HeatSim(s), oracle_cls()(s, variant="omp")
    per = s["steps_per_period"] - 1 + s["transient_substeps"]
    off = s["transient_substeps"] + s["steps_on"] - 1
    sim.step(150); orc.step(150)                      # W1: sub-steps + the first tau steps
    compare(sim, orc)
    sim.step(off - 150 - 20)                          # GPU alone up to 20 steps before switch-off
    orc.set_field(0, sim.field(0), sim.step_index)
    sim.step(60); orc.step(60)                        # W2: across switch-off
    compare(sim, orc)
    sim.step(per - sim.step_index - 30)               # ... up to 30 steps before the next switch-on
    orc.set_field(0, sim.field(0), sim.step_index)
    sim.step(160); orc.step(160)                      # W3: across switch-on and its sub-steps
    compare(sim, orc)
    pg, _ = sim.probes()
    assert np.all(np.isfinite(pg)) and pg[:, 0, 0].max() > 8.0   # the surface probe of Fig. 7 warms up
    sim.close()


def test_paper_device_downscaled_forty_periods(bd):
    """The same physics on 64 x 21 nodes over 40 source periods (104 000 solver steps): drift."""
    s = I.paper_device(21, nr=64)
    sim, orc = bd.HeatSim(s, probe_records=8), oracle_cls()(s)
    n = 40 * (s["steps_per_period"] - 1 + s["transient_substeps"])
    sim.step(n); orc.step(n)
    err = compare(sim, orc)
    assert sim.field(0).max() > 6.0
    sim.close()


# ----------------------------------------------------------------------------- round-2 parity holes / ADVICE

def test_thin_grid_drift_is_rounding_not_the_kernel(bd):
    """test_every_kernel_variant keeps eta = 10 h.  Here the grid is the thin
    one that test avoids (L/R = 10 with nz << nr, eta = 550 h): the line systems are ill-conditioned
    and fp64 rounding alone moves the result.  Measured statement instead of a narrowed input: the GPU
    differs from the long-double oracle by no more than a small multiple of what the fp64 oracle
    itself differs from it."""
    s = with_dt(bd, I.config(2, nr=1021, nz=12))
    sim, o64, o80 = bd.HeatSim(s), oracle_cls()(s), oracle_cls()(s, variant="long")
    assert sim.kernel_name.startswith("line<")
    sim.step(120); o64.step(120); o80.step(120)
    ref = o80.field(0)
    floor = float(np.max(np.abs(o64.field(0) - ref)))
    gpu = float(np.max(np.abs(sim.field(0) - ref)))
    print(f"thin grid: |fp64 oracle - long double| = {floor:.3e} K, |GPU - long double| = {gpu:.3e} K")
    assert gpu <= 3.0 * floor + 1e-12
    sim.close()


@pytest.mark.parametrize("nr,r0", [(128, 0.0), (128, 3e-4), (256, 0.0), (256, 2e-4)])
def test_tma_kernel_on_nonuniform_r(bd, nr, r0, monkeypatch):
    """the TMA kernel's table-driven rows on a NON-uniform r grid and on a grid
    that starts at r_0 > 0 (pick_tma_variant routes nr = 128 .. 8192 there when the band kernels decline)."""
    monkeypatch.setenv("HEAT_KERNEL", "tma")
    s = I.random_spec(nr, nr=nr, nz=14, nlayers=3, batch=2, r0=r0, bcs=BC_SETS[(nr // 128 + (r0 > 0)) % 4])
    s = with_dt(bd, s, 0.8)
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    assert sim.kernel_name.startswith("tma<"), sim.kernel_name
    for n in (1, 7, 12):
        sim.step(n); orc.step(n)
        compare(sim, orc)
    pg, _ = sim.probes()
    assert np.max(np.abs(pg - orc.probes())) <= TOL
    sim.close()


def test_almost_uniform_grid_takes_the_general_kernel(bd):
    """the kernels that generate (i +- 1/2) / h^2 on the fly accept a grid only if it is
    R i / N to a few ulp of R (the oracle uses the r it is given).  A grid that is off by 1e-12 R in
    places -- thousands of ulp, yet far below anything a tolerance on h would notice -- must go to the
    general kernel and match the oracle there; a grid accumulated as r_i = r_{i-1} + h stays within a
    few ulp and may take the fast kernel, where it must match as well."""
    base = I.config(2, nr=512, nz=16)
    R = base["r"][-1]
    bent = dict(base, r=base["r"].copy())
    bent["r"][100:300] += 1e-12 * R
    acc = dict(base, r=np.concatenate([[0.0], np.cumsum(np.full(511, R / 511))]))
    for spec, must_be_general in ((bent, True), (acc, False), (base, False)):
        s = with_dt(bd, spec)
        sim, orc = bd.HeatSim(s), oracle_cls()(s)
        fast = sim.kernel_name.startswith(("tband<", "wband<", "band<"))
        assert not (fast and must_be_general), sim.kernel_name
        if spec is base:
            assert sim.kernel_name.startswith("tband<"), sim.kernel_name
        sim.step(150); orc.step(150)
        compare(sim, orc)
        sim.close()


def test_two_live_contexts_with_different_layer_counts(bd):
    """the dynamic shared-memory attribute belongs to the kernel function; a context
    with fewer layers created after one with more must not break the launches of the first."""
    for nr in (512, 96):                                      # tband kernel / line kernel
        a = bd.HeatSim(with_dt(bd, I.config(2, nr=nr, nz=24)))                 # 4 layers
        two = I.config(0, nr=nr, nz=24)                                        # 3 layers
        b = bd.HeatSim(with_dt(bd, two))
        a.step(20); b.step(20); a.step(20)
        oa, ob = oracle_cls()(with_dt(bd, I.config(2, nr=nr, nz=24))), oracle_cls()(with_dt(bd, two))
        oa.step(40); ob.step(20)
        compare(a, oa); compare(b, ob)
        a.close(); b.close()


def test_missing_dt_is_rejected(bd):
    """a spec without tau must fail in heat_create, not run with a placeholder."""
    s = I.config(1, nr=64, nz=32)
    assert s["dt"] is None
    with pytest.raises(bd.HeatError):
        bd.HeatSim(s)


GUARD_CASES = [({}, 1024, 8, 2), ({"HEAT_TBAND_NW": "16"}, 8192, 6, 1), ({"HEAT_TBAND_NW": "4"}, 8192, 6, 1),
               ({"HEAT_TBAND_NW": "8"}, 4096, 7, 2), ({"HEAT_KERNEL": "wband"}, 4096, 6, 1), ({"HEAT_KERNEL": "band"}, 4096, 6, 1),
               ({"HEAT_KERNEL": "band"}, 512, 8, 2), ({"HEAT_KERNEL": "tma"}, 256, 8, 2), ({"HEAT_KERNEL": "line"}, 96, 8, 2)]


@pytest.mark.parametrize("case", GUARD_CASES, ids=lambda c: "-".join(f"{k[5:]}{v}" for k, v in c[0].items()) + f"nr{c[1]}")
def test_no_write_outside_the_callers_buffers(bd, case, monkeypatch):
    """compute-sanitizer is closed on this GPU pool (profiles/r02_sanitizer.md), so the out-of-bounds
    check is our own: both field levels, the workspace and the probe ring sit between canary bands of
    4096 doubles; after a run with TMA stores on the first / last lines, Neumann z copies, probes on
    boundary nodes and a ragged band partition every band still holds its canary, for every kernel family."""
    env, nr, nz, batch = case
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    s = I.band_spec(nr + nz, nr=nr, nz=nz, batch=batch, chunk=16, bcs=BC_SETS[1] if nr % 1024 else BC_SETS[3])
    s = with_dt(bd, s, 0.8)
    sim = bd.HeatSim(s, guard=4096, probe_records=3)      # the probe ring overflows on purpose (records are dropped, not written past)
    sim.step(11)
    assert sim.guards_intact(), sim.kernel_name
    orc = oracle_cls()(s, variant="omp" if nr * nz > 30000 else "double")
    orc.step(11)
    compare(sim, orc)
    pg, dropped = sim.probes()
    assert pg.shape[0] == 3 and dropped == 11 // s["probe_every"] - 3 and sim.guards_intact()
    sim.close()


@pytest.mark.parametrize("nr,nz,batch", [(64, 64, 1), (13, 11, 2), (96, 40, 3), (512, 40, 1)])
def test_persistent_multi_step_launch_equals_single_steps(bd, nr, nz, batch, monkeypatch):
    """heat_step(n) on the line kernel is ONE cooperative launch with the schedule, the level swap and the
    probe slots on the device.  It must give bitwise what n single-step launches give
    (field, probe records, dropped count, step index) -- across sub-steps, switch-off, an odd number of
    steps and a probe ring that overflows -- and both must match the oracle."""
    monkeypatch.setenv("HEAT_KERNEL", "line")
    if nr == 13:
        s = I.random_spec(5, nr=nr, nz=nz, batch=batch)
        s["dt"] = 0.7 * bd.heat_stable_dt(s)
    else:
        s = with_dt(bd, I.config(3 if batch > 1 else 2, nr=nr, nz=nz, batch=batch) if nr != 64 else I.config(0))
    if s["probes"]:
        s["probe_every"] = 3
    a, b = bd.HeatSim(s, probe_records=40), bd.HeatSim(s, probe_records=40)
    orc = oracle_cls()(s)
    before = a.launch_count
    a.step(151)                                  # one launch
    assert a.launch_count == before + 1
    for _ in range(151):
        b.step(1)                                # 151 launches
    assert a.step_index == b.step_index == 151
    assert np.array_equal(a.fields(), b.fields())
    a.step(2); b.step(1); b.step(1)
    assert np.array_equal(a.fields(), b.fields())
    pa, da = a.probes()
    pb, db = b.probes()
    assert np.array_equal(pa, pb) and da == db
    orc.step(153)
    compare(a, orc)
    po = orc.probes()
    if s["probes"]:
        assert pa.shape[0] == 40 and da == 153 // 3 - 40 and np.max(np.abs(pa - po[:40])) <= TOL
    a.close(); b.close()


@pytest.mark.parametrize("nr,nw", [(2048, 4), (8192, 16), (8192, 4)])
def test_tband_with_strongly_coupled_separators(bd, nr, nw, monkeypatch):
    """The tband kernel skips the PCR over the separator rows when their mutual couplings are below
    2^-80 (the BASELINE-shaped grids, eta = 10 h).  On a thin grid (L/R = 10 with nz = 10: eta ~ 2000 h)
    the line systems are barely diagonally dominant, the separators 512 rows apart stay coupled at
    O(1) and the full separator solve runs.  These systems are ill-conditioned, so the bar is the
    measured rounding floor: |GPU - long double| <= 3 |fp64 oracle - long double|."""
    monkeypatch.setenv("HEAT_TBAND_NW", str(nw))
    s = with_dt(bd, I.config(2, nr=nr, nz=10))
    sim, o64, o80 = bd.HeatSim(s), oracle_cls()(s, variant="omp"), oracle_cls()(s, variant="long")
    assert sim.kernel_name.startswith(f"tband<WL={nr // 512},NW={nw},"), sim.kernel_name
    sim.step(25); o64.step(25); o80.step(25)
    ref = o80.field(0)
    floor = float(np.max(np.abs(o64.field(0) - ref)))
    gpu = float(np.max(np.abs(sim.field(0) - ref)))
    print(f"nr = {nr}: |fp64 oracle - long double| = {floor:.3e} K, |GPU - long double| = {gpu:.3e} K")
    assert gpu <= 3.0 * floor + 1e-12
    sim.close()


@pytest.mark.parametrize("nr,nz,world", [(512, 40, 2), (1024, 23, 3), (96, 30, 2)])
def test_zslab_run_equals_the_single_gpu_run_bitwise(bd, nr, nz, world):
    """the z-slab sharding (paper_1408_5853_b200/zslab.py) on ONE GPU -- every slab is
    its own library context with Dirichlet halo lines, the contexts are stepped in turn and exchange one
    edge line per neighbour and step through heat_get_line / heat_set_line (device to device; no
    kernel waits on another).  The gathered field must be bitwise the single-context field, across
    sub-steps and switch-off, for the tband and the line kernel."""
    from paper_1408_5853_b200 import zslab as Z
    s = with_dt(bd, I.config(2, nr=nr, nz=nz))
    one = bd.HeatSim(s)
    slabs = [bd.HeatSim(Z.slab_spec(s, r, world)) for r in range(world)]
    assert all(q.kernel_name == one.kernel_name for q in slabs)
    for n in (1, 60, 90):
        one.step(n)
        Z.step_slabs_in_one_process(slabs, nz, n)
        got = Z.gather_field([q.fields() for q in slabs], nz)
        assert np.array_equal(got, one.fields())
    orc = oracle_cls()(s)
    orc.step(151)
    compare(one, orc)
    one.close()
    for q in slabs:
        q.close()


@pytest.mark.parametrize("nr,nz,world,batch", [(512, 40, 2, 1), (1024, 23, 3, 1), (2048, 20, 2, 1), (96, 30, 2, 1), (77, 31, 3, 2)])
def test_zslab_peer_stores_equal_the_single_gpu_run_bitwise(bd, nr, nz, world, batch):
    """heat_set_halo_peer: the step kernel itself stores a slab's edge lines into its neighbours' halo lines
    (TMA store in the tband kernel, plain stores in the line kernel); no get_line / set_line.  On ONE GPU the
    "peer" buffers are the other contexts' fields and the launches are ordered by the stream.  The gathered
    field must be bitwise the single-context field."""
    from paper_1408_5853_b200 import zslab as Z
    if nr == 77:
        s0 = I.random_spec(9, nr=nr, nz=nz, nlayers=3, batch=batch, bcs=(I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2), I.dirichlet(78.0)))
        s0["general_kernel"] = True
        s = with_dt(bd, s0)
    else:
        s = with_dt(bd, I.config(2, nr=nr, nz=nz))
    one = bd.HeatSim(s)
    slabs = [bd.HeatSim(Z.slab_spec(s, r, world)) for r in range(world)]
    assert all(q.kernel_name == one.kernel_name for q in slabs)
    Z.connect_peers_in_one_process(slabs)
    for n in (1, 60, 31):
        one.step(1)
        one.step(n - 1)          # the single run may use its persistent multi-step launch
        Z.step_peer_slabs_in_one_process(slabs, n)
        got = Z.gather_field([q.fields() for q in slabs], nz)
        assert np.array_equal(got, one.fields())
    if nr == 77:   # iterations would need an exchange per iteration: refused on a slab with peers
        with pytest.raises(bd.HeatError) as e:
            slabs[0].step_picard(1, 3)
        assert "halo peers" in str(e.value)
    # a peer switched off stops the exchange: the runs part
    slabs[0].set_halo_peer(1, None)
    one.step(5)
    Z.step_peer_slabs_in_one_process(slabs, 5)
    assert not np.array_equal(Z.gather_field([q.fields() for q in slabs], nz), one.fields())
    one.close()
    for q in slabs:
        q.close()


def test_halo_peer_argument_checks(bd):
    s = with_dt(bd, I.config(2, nr=512, nz=24))
    a, b = bd.HeatSim(s), bd.HeatSim(s)
    for side, peer, msg in ((2, b, "side"), (0, (a.field_a.data_ptr(), None, 24), "both level buffers"), (0, (8, 16, 2), "nz >= 3")):
        with pytest.raises(bd.HeatError) as e:
            a.set_halo_peer(side, peer)
        assert e.value.status == bd.HEAT_EINVAL and msg in str(e.value)
    n0 = dict(s)
    n0["z_lo"] = I.NEUMANN0
    c = bd.HeatSim(n0)
    with pytest.raises(bd.HeatError) as e:
        c.set_halo_peer(0, b)
    assert "Dirichlet" in str(e.value)
    os.environ["HEAT_KERNEL"] = "tma"
    try:
        d = bd.HeatSim(s)
        with pytest.raises(bd.HeatError) as e:
            d.set_halo_peer(0, b)
        assert "tband and the line kernel" in str(e.value)
        d.close()
    finally:
        del os.environ["HEAT_KERNEL"]
    for q in (a, b, c):
        q.close()


def _peer_worker(rank, world, port, nr, nz, nsteps, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    from paper_1408_5853_b200 import binding, zslab as Z
    torch.cuda.set_device(0)                      # one GPU in this sandbox: both ranks share it
    dist.init_process_group("gloo")
    s0 = I.config(2, nr=nr, nz=nz)
    s = I.with_dt(s0, binding.heat_stable_dt(s0))
    sim = binding.HeatSim(Z.slab_spec(s, rank, world))
    rk = Z.PeerSlabRank(sim, rank, world, dist)
    rk.step(nsteps)
    out[rank] = (sim.kernel_name, sim.fields())
    rk.close()
    sim.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("nr,nz,world", [(512, 40, 2), (96, 30, 2)])
def test_zslab_peer_stores_across_processes(bd, nr, nz, world):
    """PeerSlabRank: one process per rank (here sharing the one GPU), the neighbours' field levels mapped
    through CUDA IPC, a barrier per step (host-side: no kernel waits on another).  Gathered field == the
    single run, bitwise."""
    import torch.multiprocessing as mp
    from paper_1408_5853_b200 import zslab as Z
    nsteps = 45
    port = 33000 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_peer_worker, args=(world, port, nr, nz, nsteps, out), nprocs=world, join=True)
        res = [out[r] for r in range(world)]
    s = with_dt(bd, I.config(2, nr=nr, nz=nz))
    one = bd.HeatSim(s)
    one.step(nsteps)
    assert all(name == one.kernel_name for name, _ in res)
    assert np.array_equal(Z.gather_field([f for _, f in res], nz), one.fields())
    one.close()

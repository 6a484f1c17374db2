"""GPU parity of the iterated variant heat_step_picard (reading G23)
against the oracle's orc_step_picard: element by element, <= 1e-9 K, same seeded inputs.
"""
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


def _spec(bd, s0, hot=30.0):
    s = dict(s0)
    s["general_kernel"] = True
    if s.get("Q0") is not None:
        s["Q0"] = np.asarray(s["Q0"]) * hot     # strong heating: the laws move within a step
    return I.with_dt(s, bd.heat_stable_dt(s))


CASES = [
    ("random 77x19 x3, mixed laws", lambda: I.random_spec(11, nr=77, nz=19, nlayers=3, batch=3), 3, 14),
    ("random 130x33, poly laws, dirichlet r", lambda: I.random_spec(5, nr=130, nz=33, nlayers=4, laws="poly",
                                                                   bcs=(I.dirichlet(10.0), I.dirichlet(30.0), I.NEUMANN0, I.NEUMANN0)), 2, 12),
    ("uniform 512x24 (a grid the band kernels would take)", lambda: I.band_spec(3, nr=512, nz=24, chunk=16), 4, 9),
    ("random 631x21 non-uniform, r0 > 0", lambda: I.random_spec(8, nr=631, nz=21, nlayers=4, r0=1e-4), 2, 8),
]


@pytest.mark.parametrize("name,make,iters,nsteps", CASES, ids=[c[0] for c in CASES])
def test_picard_matches_the_oracle(bd, name, make, iters, nsteps):
    s = _spec(bd, make())
    sim = bd.HeatSim(s, guard=64)
    assert sim.kernel_name.startswith("line<")
    orc = oracle_cls()(s)
    sim.step_picard(nsteps, iters)
    orc.step_picard(nsteps, iters)
    err = 0.0
    for b in range(sim.batch):
        g, o = sim.field(b), orc.field(b)
        assert np.all(np.isfinite(g))
        err = max(err, float(np.max(np.abs(g - o))))
    assert err <= TOL, f"max |dT| = {err:.3e} K"
    P, dropped = sim.probes()
    assert dropped == 0 and P.shape == orc.probes().shape
    assert float(np.max(np.abs(P - orc.probes()))) <= TOL
    assert sim.step_index == orc.step_index == nsteps
    assert sim.launch_count == nsteps * iters
    assert sim.guards_intact()
    # the iterations did something: the paper's one-pass step gives another field
    plain = oracle_cls()(s)
    plain.step(nsteps)
    assert float(np.max(np.abs(plain.field(0) - orc.field(0)))) > 1e-6
    sim.close()


def test_one_iteration_is_heat_step_bitwise_and_mixing_is_allowed(bd):
    s = _spec(bd, I.random_spec(2, nr=45, nz=17, nlayers=3))
    a, b = bd.HeatSim(s), bd.HeatSim(s)
    a.step(7)
    b.step_picard(3, 1)
    b.step(1)
    b.step_picard(3, 1)
    assert np.array_equal(a.fields(), b.fields())
    # iterated and plain steps interleaved, against the oracle doing the same
    orc = oracle_cls()(s)
    orc.step(7)
    for sim_or_orc in (a, orc):
        sim_or_orc.step_picard(2, 3)
        sim_or_orc.step(2)
        sim_or_orc.step_picard(1, 2)
    assert float(np.max(np.abs(a.field(0) - orc.field(0)))) <= TOL
    a.close(); b.close()


def test_set_line_refreshes_the_iteration_buffer(bd):
    """A Dirichlet z line changed between two calls must reach the iterate buffers (z-slab halo lines)."""
    s = _spec(bd, I.random_spec(4, nr=33, nz=12, nlayers=2, bcs=(I.NEUMANN0, I.NEUMANN0, I.dirichlet(15.0), I.dirichlet(25.0))))
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    sim.step_picard(2, 3)
    orc.step_picard(2, 3)
    line = np.linspace(30.0, 40.0, s["nr"])
    sim.set_line(0, 0, line)
    F = orc.field(0)
    F[0, :] = line
    orc.set_field(0, F, orc.step_index)
    sim.step_picard(3, 4)
    orc.step_picard(3, 4)
    assert float(np.max(np.abs(sim.field(0) - orc.field(0)))) <= TOL
    sim.close()


def test_picard_needs_the_general_kernel(bd):
    s = I.with_dt(I.band_spec(3, nr=512, nz=24, chunk=16), bd.heat_stable_dt(I.band_spec(3, nr=512, nz=24, chunk=16)))
    sim = bd.HeatSim(s)
    assert not sim.kernel_name.startswith("line<")
    with pytest.raises(bd.HeatError) as e:
        sim.step_picard(1, 2)
    assert e.value.status == bd.HEAT_EINVAL and "HEAT_DESC_GENERAL_KERNEL" in str(e.value)
    sim.step_picard(2, 1)   # one iteration is heat_step on any kernel
    sim.close()

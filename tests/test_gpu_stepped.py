"""GPU parity on the stepped (non-rectangular) domain, reading G24: the lines above
z_{j_step} end at node i_step.  CUDA path (general line kernel, through the C ABI) against the oracle,
element by element on the whole array (the nodes outside Omega included: they keep their value, the
line above the step face mirrors the line below it), <= 1e-9 K.
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


def stepped(bd, s0, i_step, j_step):
    s = dict(s0)
    s["i_step"], s["j_step"] = i_step, j_step
    nr, nz = s["nr"], s["nz"]
    s["probes"] = [(nr - 1, j_step), (1, nz - 2), (i_step, nz - 2), (nr - 1, 0)]
    s["probe_every"] = 2
    return I.with_dt(s, bd.heat_stable_dt(s))


CASES = [
    ("77x19 x3 batch, step in the middle", lambda: I.random_spec(11, nr=77, nz=19, nlayers=3, batch=3), 40, 9, 25),
    ("130x33 poly laws, step one line below the top", lambda: I.random_spec(5, nr=130, nz=33, nlayers=4, laws="poly"), 61, 30, 15),
    ("130x33, step on line 1, i_step = 2", lambda: I.random_spec(6, nr=130, nz=33, nlayers=3), 2, 1, 15),
    ("512x24 uniform (even nr: the paired loads are off), i_step odd", lambda: I.band_spec(3, nr=512, nz=24, chunk=16), 301, 11, 12),
    ("631x41 non-uniform r, dirichlet top, i_step = nr-2", lambda: I.random_spec(8, nr=631, nz=41, nlayers=4, r0=1e-4,
                                                                               bcs=(I.NEUMANN0, I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2))), 629, 20, 10),
]


@pytest.mark.parametrize("name,make,i_step,j_step,nsteps", CASES, ids=[c[0] for c in CASES])
def test_stepped_domain_matches_the_oracle(bd, name, make, i_step, j_step, nsteps):
    s = stepped(bd, make(), i_step, j_step)
    sim = bd.HeatSim(s, guard=64)
    assert sim.kernel_name.startswith("line<")
    orc = oracle_cls()(s)
    sim.step(1)                 # single launches
    sim.step(nsteps - 1)        # and the persistent multi-step launch
    orc.step(nsteps)
    for b in range(sim.batch):
        g, o = sim.field(b), orc.field(b)
        assert np.all(np.isfinite(g))
        assert float(np.max(np.abs(g - o))) <= TOL
        # outside Omega nothing moved; the line above the step face mirrors the one below, bitwise
        T0 = np.asarray(s["T_init"]).reshape(sim.batch, s["nz"], s["nr"])[b]
        assert np.array_equal(g[j_step + 2:-1, i_step + 1:], T0[j_step + 2:-1, i_step + 1:])
        assert np.array_equal(g[j_step + 1, i_step + 1:], g[j_step, i_step + 1:])
    P, dropped = sim.probes()
    assert dropped == 0 and P.shape == orc.probes().shape and P.shape[0] == nsteps // 2
    assert float(np.max(np.abs(P - orc.probes()))) <= TOL
    assert sim.guards_intact()
    # the step matters: the rectangle gives another field inside Omega
    rect = dict(s)
    rect["i_step"] = rect["j_step"] = 0
    ro = oracle_cls()(rect)
    ro.step(nsteps)
    assert float(np.max(np.abs(ro.field(0)[: j_step + 1] - orc.field(0)[: j_step + 1]))) > 1e-6
    sim.close()


def test_stepped_domain_with_iterations_set_field_and_set_line(bd):
    s = stepped(bd, I.random_spec(4, nr=45, nz=17, nlayers=3), 20, 8)
    s["general_kernel"] = True
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    sim.step_picard(3, 3)
    orc.step_picard(3, 3)
    assert float(np.max(np.abs(sim.field(0) - orc.field(0)))) <= TOL
    # a new field: the library re-establishes the mirror line, whatever the caller put there
    rng = np.random.Generator(np.random.PCG64(5))
    F = rng.uniform(5.0, 80.0, size=(s["nz"], s["nr"]))
    sim.set_field(0, F, 7)
    orc.set_field(0, F, 7)
    sim.step(4)
    orc.step(4)
    assert float(np.max(np.abs(sim.field(0) - orc.field(0)))) <= TOL
    # a line at the step face replaced (what a z-slab halo exchange does)
    line = np.linspace(30.0, 40.0, s["nr"])
    sim.set_line(0, 8, line)
    G = orc.field(0)
    G[8, :] = line
    orc.set_field(0, G, orc.step_index)
    sim.step(3)
    orc.step(3)
    assert float(np.max(np.abs(sim.field(0) - orc.field(0)))) <= TOL
    sim.close()


@pytest.mark.parametrize("bad,msg", [(dict(j_step=0, i_step=5), "stepped"), (dict(j_step=17, i_step=5), "stepped"),
                                     (dict(j_step=4, i_step=1), "stepped"), (dict(j_step=4, i_step=7, probes=[(9, 8)]), "outside")])
def test_descriptor_checks(bd, bad, msg):
    s = I.with_dt(I.random_spec(0, nr=19, nz=19, nlayers=3), bd.heat_stable_dt(I.random_spec(0, nr=19, nz=19, nlayers=3)))
    s.update(bad)
    with pytest.raises(bd.HeatError) as e:
        bd.HeatSim(s)
    assert e.value.status == bd.HEAT_EINVAL and msg in str(e.value)


def test_the_papers_device_with_its_core_reaching_the_terminal(bd):
    """inputs.paper_device(stepped=True): layers 1-3 end at z_0 = 4 cm, the copper core goes on to the
    4.2 K terminal at z_max = 5 cm (Fig. 1, G10).  Window from the initial state across the switch-on."""
    s = I.paper_device(M=201, stepped=True)
    sim, orc = bd.HeatSim(s), oracle_cls()(s)
    n = 130
    sim.step(n)
    orc.step(n)
    g, o = sim.field(0), orc.field(0)
    assert float(np.max(np.abs(g - o))) <= TOL
    assert g.max() > 6.0 and g[s["j_step"] + 2:, s["i_step"] + 1:].max() == 4.2
    sim.close()

"""heat_create_static: the allocation-free set-up (include/heat.h, "allocation-free set-up").

The row tables of a context go into the library's static device array instead of a workspace the
caller allocates.  The output must be that of the existing path (heat_create): same kernels, same
tables, so the fields and probe traces are compared within the GPU tests' tolerance AND bitwise.
The array is shared and keeps the previous context's contents, so the calls come in a row, with
different problems and different kernels (tensor-memory band kernel, general line kernel, band
kernel again), each destroyed before the next is created.

The file is named so that pytest collects it last (the suite runs with pytest -x).
"""
import numpy as np
import pytest

from paper_1408_5853_b200 import inputs as I

TOL = 1e-9  # K, the bar of tests/test_gpu_parity.py (BASELINE.json north_star)


@pytest.fixture(scope="module")
def bd():
    from paper_1408_5853_b200 import build as B
    B.build()
    from paper_1408_5853_b200 import binding
    binding.lib()
    return binding


def _with_dt(bd, s0):
    return I.with_dt(s0, bd.heat_stable_dt(s0))


def _run(bd, spec, nsteps, static):
    sim = bd.HeatSim(spec, static_workspace=static, guard=64)
    try:
        name = sim.kernel_name
        sim.step(nsteps // 2)
        sim.step(nsteps - nsteps // 2)
        F = sim.fields().copy()
        P, dropped = sim.probes()
        assert dropped == 0
        assert sim.guards_intact()
        if static:
            assert sim.workspace is None
    finally:
        sim.close()
    return name, F, P


def _specs(bd):
    return [
        ("tband", _with_dt(bd, I.band_spec(3, nr=512, nz=40, batch=2, chunk=16)), 23),
        ("line", _with_dt(bd, I.random_spec(11, nr=77, nz=19, nlayers=3, batch=3)), 31),
        ("tband", _with_dt(bd, I.band_spec(5, nr=1024, nz=21, poly_laws=True, chunk=16)), 17),
    ]


@pytest.mark.gpu
def test_static_workspace_matches_heat_create_on_calls_in_a_row(bd):
    assert bd.heat_static_workspace_bytes() == 4 << 20
    specs = _specs(bd)
    want = [_run(bd, s, n, static=False) for _, s, n in specs]
    # the static calls back to back: nothing but the shared array between them
    got = [_run(bd, s, n, static=True) for _, s, n in specs]
    for (kind, s, n), (wn, wF, wP), (gn, gF, gP) in zip(specs, want, got):
        assert kind in wn and gn == wn, (kind, wn, gn)
        assert bd.heat_workspace_bytes(s) <= bd.heat_static_workspace_bytes()
        assert np.all(np.isfinite(gF))
        assert float(np.max(np.abs(gF - wF))) <= TOL
        assert gP.shape == wP.shape and gP.size > 0
        assert float(np.max(np.abs(gP - wP))) <= TOL
        assert np.array_equal(gF, wF) and np.array_equal(gP, wP)   # same kernels, same tables: same bits
        assert float(np.max(np.abs(gF - np.asarray(s["T_init"]).reshape(gF.shape)))) > 1e-3   # the steps did something


@pytest.mark.gpu
def test_static_workspace_same_problem_twice_and_after_a_larger_one(bd):
    """The same problem twice in a row, then once more after a problem with larger tables has been
    through the array: the result never depends on what the array held."""
    kind, small, n = _specs(bd)[1]
    _, big, nb = _specs(bd)[0]
    _, wF, wP = _run(bd, small, n, static=False)
    for _ in range(2):
        _, gF, gP = _run(bd, small, n, static=True)
        assert np.array_equal(gF, wF) and np.array_equal(gP, wP)
    _run(bd, big, nb, static=True)
    _, gF, gP = _run(bd, small, n, static=True)
    assert float(np.max(np.abs(gF - wF))) <= TOL and np.array_equal(gF, wF) and np.array_equal(gP, wP)


@pytest.mark.gpu
def test_static_workspace_rejects_what_does_not_fit(bd):
    s = _with_dt(bd, I.band_spec(7, nr=512, nz=8, batch=512, chunk=16))
    assert bd.heat_workspace_bytes(s) > bd.heat_static_workspace_bytes()
    with pytest.raises(bd.HeatError) as e:
        bd.HeatSim(s, static_workspace=True)
    assert e.value.status == bd.HEAT_ENOMEM
    assert "HEAT_STATIC_WORKSPACE_BYTES" in str(e.value) and str(bd.heat_workspace_bytes(s)) in str(e.value)
    # the existing path takes the same problem
    sim = bd.HeatSim(s)
    sim.step(2)
    assert np.all(np.isfinite(sim.field(0)))
    sim.close()

"""z-slab sharding on CPU: index bookkeeping, and the exchange protocol over gloo
with the ORACLE as the per-rank stepper -- the slab run must equal the single run bitwise."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1408_5853_b200 import inputs as I
from paper_1408_5853_b200 import zslab as Z


class OracleStepper:
    """Adapter: the oracle with the get_line / set_line / step interface a slab rank needs."""

    def __init__(self, spec):
        from oracle.heat_oracle import Oracle
        self.o, self.batch, self.nr, self.nz = Oracle(spec), int(spec.get("batch", 1)), spec["nr"], spec["nz"]

    def step(self, n=1):
        self.o.step(n)

    def get_line(self, b, j):
        return self.o.field(b)[j].copy()

    def set_line(self, b, j, values):
        T = self.o.field(b)
        T[j] = np.asarray(values, dtype=np.float64)
        self.o.set_field(b, T, self.o.step_index)

    def fields(self):
        return self.o.fields()


def test_partition_and_plan():
    assert Z.partition(10, 1) == [(1, 9)]
    assert Z.partition(10, 3) == [(1, 4), (4, 7), (7, 9)]
    assert Z.partition(12, 4) == [(1, 4), (4, 7), (7, 9), (9, 11)]
    with pytest.raises(ValueError):
        Z.partition(5, 4)
    for nz, world in ((10, 3), (64, 8), (13, 2)):
        parts = Z.partition(nz, world)
        assert parts[0][0] == 1 and parts[-1][1] == nz - 1
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1
        for r in range(world):
            plan = Z.exchange_plan(nz, r, world)
            assert len(plan) == (r > 0) + (r < world - 1)
            last = parts[r][1] - parts[r][0] + 1
            for peer, js, jr in plan:
                assert (peer, js, jr) == ((r - 1, 1, 0) if peer < r else (r + 1, last - 1, last))


def test_slab_spec_geometry_and_probes():
    s = I.random_spec(3, nr=11, nz=14, nlayers=2, bcs=(I.NEUMANN0, I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2)))
    s["probes"] = [(10, 0), (3, 5), (2, 9), (4, 13)]
    parts = Z.partition(14, 3)
    seen = []
    for r in range(3):
        q = Z.slab_spec(s, r, 3)
        j0, j1 = parts[r]
        assert q["nz"] == j1 - j0 + 2 and np.array_equal(q["z"], s["z"][j0 - 1:j1 + 1])
        assert np.array_equal(q["T_init"], s["T_init"][:, j0 - 1:j1 + 1, :])
        assert q["z_lo"] == (s["z_lo"] if r == 0 else Z.DIRICHLET_HALO) and q["z_hi"] == (s["z_hi"] if r == 2 else Z.DIRICHLET_HALO)
        seen += [(i, j + j0 - 1) for (i, j) in q["probes"]]
    assert sorted(seen) == sorted(s["probes"])          # every probe has exactly one owner


@pytest.mark.parametrize("world", [2, 3])
def test_slabs_in_one_process_equal_the_single_run(world):
    """The protocol without a transport: slabs stepped in turn, edge lines copied."""
    from oracle.heat_oracle import Oracle, stable_dt
    s = I.random_spec(11, nr=12, nz=15, nlayers=3, batch=2)
    s["dt"] = 0.6 * stable_dt(s)
    ref = Oracle(s)
    slabs = [OracleStepper(Z.slab_spec(s, r, world)) for r in range(world)]
    for n in (1, 4, 9):
        ref.step(n)
        Z.step_slabs_in_one_process(slabs, s["nz"], n)
        got = Z.gather_field([st.fields() for st in slabs], s["nz"])
        assert np.array_equal(got, ref.fields())


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle.heat_oracle import stable_dt
    dist.init_process_group("gloo")
    s = I.random_spec(5, nr=13, nz=12, nlayers=3, batch=2, bcs=(I.NEUMANN0, I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2)))
    s["dt"] = 0.6 * stable_dt(s)
    st = OracleStepper(Z.slab_spec(s, rank, world))
    rk = Z.SlabRank(st, s, rank, world, dist=dist)
    rk.step(17)
    out[rank] = st.fields()
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_over_gloo_equal_the_single_run():
    """world_size 2 over torch.distributed (gloo): one line per neighbour and step, both directions
    posted at once; the gathered field equals the single-process oracle run bitwise."""
    import torch.multiprocessing as mp
    from oracle.heat_oracle import Oracle, stable_dt
    world, port = 2, 31000 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        fields = [out[r] for r in range(world)]
    s = I.random_spec(5, nr=13, nz=12, nlayers=3, batch=2, bcs=(I.NEUMANN0, I.NEUMANN0, I.NEUMANN0, I.dirichlet(4.2)))
    s["dt"] = 0.6 * stable_dt(s)
    ref = Oracle(s)
    ref.step(17)
    assert np.array_equal(Z.gather_field(fields, s["nz"]), ref.fields())


def test_peer_plan_mirrors_the_exchange_plan():
    """Peer-store mode: a slab stores into exactly the neighbours it would send to, on the side that faces them."""
    for world in (1, 2, 3, 5):
        for rank in range(world):
            plan = Z.peer_plan(rank, world)
            ex = Z.exchange_plan(40, rank, world)
            assert [p for _, p in plan] == [p for p, _, _ in ex]
            for side, peer in plan:
                assert peer == rank - 1 if side == 0 else peer == rank + 1
                # the neighbour lists this rank on its opposite side
                assert (1 - side, rank) in Z.peer_plan(peer, world)

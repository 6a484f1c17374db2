"""Multi-GPU sharding of ONE problem by contiguous z-slabs.

Within a step every z-line is independent and only the explicit axial operator Lambda_j (11)
P:L125 couples line j to lines j-1 and j+1 of the OLD level.  A rank therefore owns a contiguous slab of
lines, keeps one halo line on each inner side, and after every step exchanges exactly one line of nr
doubles with each neighbour (point to point; no reduction, no all-to-all).

How a slab becomes an ordinary problem of the library: the halo lines are the first and last line of
the rank's local grid with a DIRICHLET z condition -- such lines are never solved and hold whatever
values they are given (reading G17) -- and after each step they are overwritten with the neighbour's
freshly solved edge line (`heat_set_line`).  The local z coordinates include the halo lines, so the
factors 1 / (etabar_j eta_j) of (11) are those of the global grid, and the per-line arithmetic of a slab
run is the arithmetic of the single-GPU run: the two are bitwise identical (tests/test_zslab.py on CPU
with the oracle as the stepper, tests/test_gpu_parity.py::test_zslab_* on one GPU with two contexts
stepped in turn).  Outer slabs keep the problem's own z boundary condition on their outer side.

Nothing here is arithmetic of the method: index bookkeeping and the exchange protocol only.  The
stepper is anything with `step(n)`, `get_line(b, j)`, `set_line(b, j, values)` (binding.HeatSim on a
GPU, the oracle in the CPU test); the transport is torch.distributed send / recv (nccl between GPUs,
gloo in the CPU test) or a direct copy when both slabs live in one process.
Probes stay with the rank that owns their line (`local_probes`).  No scaling curve has been measured:
this sandbox has one GPU.

Peer-store mode (`peer_plan`, `connect_peers_in_one_process`, `step_peer_slabs_in_one_process`): instead of
get_line / send / recv / set_line, `heat_set_halo_peer` gives every slab the address of its neighbours' field
levels and the step kernel itself stores its edge lines into their halo lines (TMA store / plain stores
over NVLink peer memory), so the exchange costs no extra kernel or copy and overlaps the step.  Between
processes (`PeerSlabRank`) the addresses come from CUDA IPC handles and the per-step synchronisation is a
barrier; tested with two processes sharing the one GPU of this sandbox.
"""
from __future__ import annotations

import numpy as np

DIRICHLET_HALO = ("dirichlet", 0.0)   # the value is irrelevant: T_init carries the halo line


def partition(nz: int, world: int):
    """Interior lines 1 .. nz-2 split into `world` contiguous slabs, sizes differing by at most one
    (the first nz-2 mod world slabs are the longer ones).  Returns [(j0, j1)] with j0 <= j < j1."""
    n = nz - 2
    if world < 1 or n < world:
        raise ValueError(f"cannot cut {n} interior lines into {world} slabs")
    base, extra = divmod(n, world)
    out, j = [], 1
    for r in range(world):
        m = base + (1 if r < extra else 0)
        out.append((j, j + m))
        j += m
    return out


def slab_spec(spec, rank: int, world: int, T_field=None):
    """The descriptor of rank's slab: lines j0-1 .. j1 of the global grid (local line l = global
    j0-1+l).  T_field: the global current level [batch][nz][nr] (default: spec's initial condition)."""
    j0, j1 = partition(spec["nz"], world)[rank]
    nr, nz, batch = spec["nr"], spec["nz"], int(spec.get("batch", 1))
    s = dict(spec)
    s["nz"] = j1 - j0 + 2
    s["z"] = np.ascontiguousarray(spec["z"][j0 - 1:j1 + 1])
    if rank > 0:
        s["z_lo"] = DIRICHLET_HALO
    if rank < world - 1:
        s["z_hi"] = DIRICHLET_HALO
    if T_field is None:
        T_field = initial_field(spec)
    s["T_init"] = np.ascontiguousarray(np.asarray(T_field, dtype=np.float64).reshape(batch, nz, nr)[:, j0 - 1:j1 + 1, :])
    s["probes"] = local_probes(spec, rank, world)
    return s


def initial_field(spec):
    """The global initial level as heat_create builds it: T_init if given, else T0 with the Dirichlet
    sides set (r sides first, z lines last so that corners belong to the z lines, G17)."""
    nr, nz, batch = spec["nr"], spec["nz"], int(spec.get("batch", 1))
    if spec.get("T_init") is not None:
        return np.asarray(spec["T_init"], dtype=np.float64).reshape(batch, nz, nr).copy()
    T = np.full((batch, nz, nr), float(spec["T0"]))
    if spec["r_in"][0] == "dirichlet":
        T[:, :, 0] = spec["r_in"][1]
    if spec["r_out"][0] == "dirichlet":
        T[:, :, -1] = spec["r_out"][1]
    if spec["z_lo"][0] == "dirichlet":
        T[:, 0, :] = spec["z_lo"][1]
    if spec["z_hi"][0] == "dirichlet":
        T[:, -1, :] = spec["z_hi"][1]
    return T


def local_probes(spec, rank: int, world: int):
    """Probes whose line this rank owns (boundary lines belong to the outer slabs), in local indices."""
    j0, j1 = partition(spec["nz"], world)[rank]
    lo = 0 if rank == 0 else j0
    hi = spec["nz"] if rank == world - 1 else j1
    return [(i, j - (j0 - 1)) for (i, j) in spec.get("probes", []) if lo <= j < hi]


def exchange_plan(nz: int, rank: int, world: int):
    """What a rank does after every step: a list of (peer, send_local_line, recv_local_line).  It
    sends its first / last INTERIOR line and receives into its halo line on the same side."""
    j0, j1 = partition(nz, world)[rank]
    last = j1 - j0 + 1            # local index of the upper halo line
    plan = []
    if rank > 0:
        plan.append((rank - 1, 1, 0))
    if rank < world - 1:
        plan.append((rank + 1, last - 1, last))
    return plan


class SlabRank:
    """One rank of a z-slab run over torch.distributed (nccl on GPUs, gloo on CPU)."""

    def __init__(self, stepper, spec_global, rank: int, world: int, dist=None, device="cpu"):
        self.st, self.rank, self.world, self.dist, self.device = stepper, rank, world, dist, device
        self.batch, self.nr = int(spec_global.get("batch", 1)), spec_global["nr"]
        self.plan = exchange_plan(spec_global["nz"], rank, world)

    def step(self, n: int = 1):
        import torch
        for _ in range(n):
            self.st.step(1)
            if not self.plan:
                continue
            # post every send and receive of this step, then wait: no ordering between neighbours is needed
            ops, recvs = [], []
            for peer, js, jr in self.plan:
                out = torch.stack([torch.as_tensor(self.st.get_line(b, js)) for b in range(self.batch)]).to(self.device).contiguous()
                buf = torch.empty((self.batch, self.nr), dtype=torch.float64, device=self.device)
                ops.append(self.dist.P2POp(self.dist.isend, out, peer))
                ops.append(self.dist.P2POp(self.dist.irecv, buf, peer))
                recvs.append((jr, buf))
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()
            for jr, buf in recvs:
                for b in range(self.batch):
                    self.st.set_line(b, jr, buf[b])


def step_slabs_in_one_process(steppers, nz: int, n: int = 1):
    """The same protocol with every slab in this process (one GPU holding all slabs, stepped in turn;
    used by the single-GPU parity test -- the kernels never wait on one another)."""
    world = len(steppers)
    plans = [exchange_plan(nz, r, world) for r in range(world)]
    batch = steppers[0].batch
    for _ in range(n):
        for st in steppers:
            st.step(1)
        moved = []
        for r, st in enumerate(steppers):
            for peer, js, jr in plans[r]:
                # what rank r sends lands in the peer's halo line that faces r
                jr_peer = next(q_jr for (q_peer, q_js, q_jr) in plans[peer] if q_peer == r)
                moved.append((peer, jr_peer, [st.get_line(b, js) for b in range(batch)]))
        for peer, jr, lines in moved:
            for b in range(batch):
                steppers[peer].set_line(b, jr, lines[b])


def peer_plan(rank: int, world: int):
    """Peer-store mode (heat_set_halo_peer): [(side, neighbour rank)] -- side 0 is the slab below, 1 the slab above."""
    plan = []
    if rank > 0:
        plan.append((0, rank - 1))
    if rank < world - 1:
        plan.append((1, rank + 1))
    return plan


def connect_peers_in_one_process(steppers):
    """Every slab's step kernel stores its edge lines straight into its neighbours' halo lines (all slabs
    in this process: the same GPU, or GPUs with peer access enabled).  After this, a step of the run is
    `for st in steppers: st.step(1)` plus a synchronisation; no get_line / set_line."""
    world = len(steppers)
    for r, st in enumerate(steppers):
        for side, peer in peer_plan(r, world):
            st.set_halo_peer(side, steppers[peer])


def step_peer_slabs_in_one_process(steppers, n: int = 1):
    """n steps in peer-store mode.  In one process the launches are ordered by the stream: step k of
    every slab is enqueued before step k + 1 of any (between processes this is a barrier per step)."""
    for _ in range(n):
        for st in steppers:
            st.step(1)


def export_level(t):
    """What another process needs to map a device tensor (one field level): torch's CUDA IPC descriptor of
    its storage plus the tensor's offset inside it.  The exporting process must keep `t` alive."""
    return tuple(t.untyped_storage()._share_cuda_()) + (int(t.storage_offset()) * t.element_size(),)


def import_level(desc):
    """(storage to keep alive, device address) of a level exported by another process: cudaIpcOpenMemHandle
    through torch (peer access between the two GPUs is enabled by the open)."""
    import torch
    st = torch.UntypedStorage._new_shared_cuda(*desc[:-1])
    return st, int(st.data_ptr()) + int(desc[-1])


class PeerSlabRank:
    """One rank of a z-slab run in peer-store mode, one process per GPU.  The addresses of the neighbours'
    field levels are exchanged once (CUDA IPC handles through `dist.all_gather_object`, any backend); a
    step is heat_step(1) on every rank, whose kernel stores the edge lines into the neighbours' halo lines,
    then a stream synchronisation and a barrier: nobody starts step k + 1 before every store of step k
    has landed.  No halo data passes through the host or through a collective."""

    def __init__(self, sim, rank: int, world: int, dist):
        self.sim, self.rank, self.world, self.dist = sim, rank, world, dist
        mine = (export_level(sim.field_a), export_level(sim.field_b), int(sim.nz))
        everyone = [None] * world
        dist.all_gather_object(everyone, mine)
        self._mapped = []
        for side, peer in peer_plan(rank, world):
            da, db, pnz = everyone[peer]
            sa, pa = import_level(da)
            sb, pb = import_level(db)
            self._mapped += [sa, sb]
            sim.set_halo_peer(side, (pa, pb, pnz))
        dist.barrier()

    def step(self, n: int = 1):
        for _ in range(n):
            self.sim.step(1)
            self.sim.synchronize()
            self.dist.barrier()

    def close(self):
        """Stop storing into the neighbours and unmap them (call on every rank before the fields are freed)."""
        self.sim.synchronize()
        self.dist.barrier()
        for side, _ in peer_plan(self.rank, self.world):
            self.sim.set_halo_peer(side, None)
        self._mapped = []
        self.dist.barrier()


def gather_field(fields, nz: int):
    """Global level [batch][nz][nr] from the ranks' local levels (halo lines dropped)."""
    world = len(fields)
    parts = []
    for r, F in enumerate(fields):
        j0, j1 = partition(nz, world)[r]
        lo = 0 if r == 0 else 1
        hi = F.shape[1] if r == world - 1 else F.shape[1] - 1
        parts.append(F[:, lo:hi, :])
    return np.concatenate(parts, axis=1)

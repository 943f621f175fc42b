"""Multi-rank bookkeeping ("replicas only") on CPU: world_size 2, gloo backend.

The path has no data-path collective; what N > 1 adds is (i) dealing independent fields to ranks,
(ii) the barrier + max-over-ranks timing rule and (iii) the whole-job throughput aggregate that
bench.py prints.  These run here without a GPU."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2409_02294_b200 import nested, replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_fields, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert replicas.dist_env() == (rank, rank, world)
        mine = replicas.fields_of_rank(n_fields, rank, world)
        # every rank learns every other rank's share: together they cover each field exactly once
        shares = [None] * world
        dist.all_gather_object(shares, mine)
        flat = sorted(i for s in shares for i in s)
        assert flat == list(range(n_fields))
        assert max(len(s) for s in shares) - min(len(s) for s in shares) <= 1
        replicas.barrier(world)
        # rank r "took" 10 + 5 r ms for its share; the job's time is the slowest rank's
        ms = 10.0 + 5.0 * rank
        value, ms_max, total = replicas.aggregate_throughput(len(mine), ms, world)
        assert ms_max == 10.0 + 5.0 * (world - 1)
        assert total == n_fields
        assert abs(value - n_fields * 1e3 / ms_max) < 1e-9
        assert replicas.max_over_ranks(float(rank), world) == float(world - 1)
        assert replicas.sum_over_ranks(1.0, world) == float(world)
        out.put((rank, value))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_fields", [8, 5])
def test_replicas_world2_gloo(n_fields):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_fields, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = dict(out.get(timeout=10) for _ in range(world))
    assert got[0] == got[1]          # both ranks agree on the whole-job number


def test_single_rank_is_identity():
    assert replicas.fields_of_rank(3, 0, 1) == [0, 1, 2]
    assert replicas.max_over_ranks(2.5, 1) == 2.5
    assert replicas.aggregate_throughput(4, 2.0, 1) == (2000.0, 2.0, 4.0)
    with pytest.raises(ValueError):
        replicas.fields_of_rank(3, 2, 2)


# ------------------------------------------------------------------ NEXT-3: one nested mesh level per rank
class _HostLevel:
    """Stand-in for nested.GpuLevel on CPU tensors: the oracle's steps in place of the pg3n_* kernels, so that the
    SCHEDULE of nested.run_schedule (who sends what to whom, in which order) is what is under test."""

    def __init__(self, n, box0, level, depth, rho):
        import numpy as np
        from oracle import nested_oracle as no
        import oracle
        self.np, self.no, self.oracle = np, no, oracle
        self.n, self.box, self.level, self.depth = n, box0 / 2**level, level, depth
        self.rho = rho.copy()
        n_mean, n_halo = nested.message_counts(n)
        self.mean_in = torch.empty(n_mean, dtype=torch.float64)
        self.halo_in = torch.empty(n_halo, dtype=torch.float64)
        self.log = []

    def recv_buffers(self):
        return self.mean_in, self.halo_in

    def restrict(self):
        self.log.append("restrict")
        return torch.from_numpy(self.no.restrict(self.rho).ravel().copy()), None

    def absorb(self, t, token):
        self.log.append("absorb")
        q = self.n // 2
        self.rho = self.no.absorb(self.rho, t.numpy().reshape(q, q, q))

    def solve(self):
        self.log.append("solve")
        self.own = self.oracle.cart_potential(self.n, self.box, self.rho)
        if self.level < self.depth - 1:
            self.out = self.oracle.cart_potential(self.n, self.box, self.no.mask_centre(self.rho))

    def add_exterior(self, t, token):
        self.log.append("add_exterior")
        m = self.n // 2 + 2
        self.ext = self.np.zeros((self.n,) * 3) if t is None else self.no.prolong(t.numpy().reshape(m, m, m), self.n)
        self.phi = self.own + self.ext

    def pack_exterior(self):
        self.log.append("pack_exterior")
        return torch.from_numpy(self.no.pack_halo(self.out + self.ext).ravel().copy()), None


def _nested_inputs(n, depth):
    import numpy as np
    rng = np.random.default_rng(77)
    return [rng.random((n, n, n)) for _ in range(depth)]


def _nested_worker(rank, world, port, n, out):
    import numpy as np
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rhos = _nested_inputs(n, world)
        lev = _HostLevel(n, 4.0, rank, world, rhos[rank])
        nested.run_schedule({rank: lev}, world, nested.DistLink(dist))
        out.put((rank, lev.phi, lev.log))
    finally:
        dist.destroy_process_group()


def test_nested_levels_one_per_rank_world2_gloo():
    """Depth 2, level l on rank l: the restricted density goes up, the exterior potential comes down, and both ranks
    end with the potentials the in-process schedule (LocalLink) and the oracle produce."""
    import numpy as np
    from oracle import nested_oracle as no
    n, world, port = 8, 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_nested_worker, args=(r, world, port, n, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict((r, (phi, log)) for r, phi, log in (out.get(timeout=120) for _ in range(world)))
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    rhos = _nested_inputs(n, world)
    ref, _ = no.nested_potential(n, 4.0, rhos)
    for l in range(world):
        assert np.array_equal(got[l][0], ref[l])
    assert got[1][1] == ["restrict", "solve", "add_exterior"]
    assert got[0][1] == ["absorb", "solve", "add_exterior", "pack_exterior"]
    # the same schedule with every level in one process
    levels = {l: _HostLevel(n, 4.0, l, world, rhos[l]) for l in range(world)}
    nested.run_schedule(levels, world, nested.LocalLink())
    for l in range(world):
        assert np.array_equal(levels[l].phi, ref[l])
    assert nested.message_counts(8) == (64, 216)


def _putlink_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        link = nested.PutLink(dist)               # no token_device given: taken from the group's backend
        if rank == 0:
            link.tok.fill_(41)
            link.send(0, 1, None)
        else:
            link.recv(0, 1)
        out.put((rank, str(link.tok.device), int(link.tok.item())))
    finally:
        dist.destroy_process_group()


def test_putlink_token_device_follows_the_backend_world2_gloo():
    """PutLink's one-element token must live where the group's backend can move it: host memory for gloo (device memory
    for nccl -- the default used to be "cpu" whatever the backend, which an NCCL-only group cannot send)."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_putlink_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict((r, (dev, val)) for r, dev, val in (out.get(timeout=120) for _ in range(world)))
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert got[0][0] == "cpu" and got[1] == ("cpu", 41)

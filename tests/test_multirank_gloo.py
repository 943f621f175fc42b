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

from paper_2409_02294_b200 import replicas


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

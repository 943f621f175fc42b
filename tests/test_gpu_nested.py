"""Parity of the nested-mesh path (row NEXT-3 of SURVEY.md 8(f): Fig. 8 :306; readings M1-M6)
against oracle/nested_oracle.py, element by element on seeded densities, level by level, and of each coupling kernel
against its oracle step.  Bar: rel-L2 <= 1e-10, max pointwise relative <= 1e-9."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import nested_oracle as no
from paper_2409_02294_b200 import binding as pg
from paper_2409_02294_b200 import nested

pytestmark = pytest.mark.gpu


def level_rho(n, level, seed):
    """A centrally condensed clump sampled on the level's cells plus seeded clumps and 1 % noise; non-negative."""
    rng = np.random.Generator(np.random.PCG64(2409022940 + 7000 * n + 10 * seed + level))
    x = (np.arange(n) + 0.5 - n / 2.0) / n / 2.0**level
    z, y, xx = np.meshgrid(x, x, x, indexing="ij")
    rho = 1.0 / (1.0 + (xx**2 + y**2 + z**2) / 0.05**2)
    for _ in range(4):
        c = rng.uniform(-0.4, 0.4, 3) / 2.0**level
        w = rng.uniform(0.03, 0.1) / 2.0**level
        rho += rng.uniform(0.5, 2.0) * np.exp(-((xx - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2) / (2 * w * w))
    return rho * (1.0 + 0.01 * rng.standard_normal(rho.shape))


def check(got, ref, what):
    l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got / ref - 1.0).max()
    assert l2 <= 1e-10 and mx <= 1e-9, f"{what}: rel-L2 {l2:.3e}, max rel {mx:.3e}"


@pytest.mark.parametrize("n,depth", [(32, 1), (32, 2), (32, 3), (32, 4), (64, 2)])      # depth 4: the paper's hierarchy, Fig. 8
def test_nested_levels_on_one_gpu_vs_oracle(n, depth):
    box0 = 8.0
    rhos = [level_rho(n, l, depth) for l in range(depth)]
    ref, _ = no.nested_potential(n, box0, rhos)
    np_ = nested.NestedPotential(n, box0, depth, device=0)
    try:
        d_rho = {l: torch.from_numpy(rhos[l]).cuda() for l in range(depth)}
        d_out = {l: torch.empty_like(d_rho[l]) for l in range(depth)}
        for rep in range(2):                                   # twice: the message buffers are reused safely
            np_.solve(d_rho, d_out)
        np_.synchronize()
        for l in range(depth):
            got = d_out[l].cpu().numpy()
            assert (got < 0).all()
            check(got, ref[l], f"n={n} depth={depth} level {l}")
        assert np_.launches() > 0
    finally:
        np_.close()


def test_coupling_kernels_step_by_step_and_call_order_errors():
    n, box0 = 32, 4.0
    rng = np.random.default_rng(11)
    coarse, fine = rng.random((n, n, n)), rng.random((n, n, n))
    st = torch.cuda.current_stream().cuda_stream
    h0 = pg.pg3n_create(n, box0, 0, 2, 0, st)
    h1 = pg.pg3n_create(n, box0, 1, 2, 0, st)
    try:
        n_mean, n_halo = nested.message_counts(n)
        mean = torch.zeros(n_mean, dtype=torch.float64, device="cuda")
        halo = torch.zeros(n_halo, dtype=torch.float64, device="cuda")
        with pytest.raises(pg.PolargravError) as e:            # nothing set yet
            pg.pg3n_restrict(h1, mean)
        assert e.value.status == pg.PG_ERR_STATE
        pg.pg3n_set_density(h0, coarse, pg.PG_MEM_HOST)
        pg.pg3n_set_density(h1, torch.from_numpy(fine).cuda(), pg.PG_MEM_DEVICE)
        for bad in (lambda: pg.pg3n_restrict(h0, mean), lambda: pg.pg3n_absorb(h1, mean),
                    lambda: pg.pg3n_add_exterior(h0, None), lambda: pg.pg3n_pack_exterior(h0, halo)):
            with pytest.raises(pg.PolargravError) as e:
                bad()
            assert e.value.status == pg.PG_ERR_STATE
        pg.pg3n_restrict(h1, mean)
        pg.pg3n_synchronize(h1)
        assert np.array_equal(mean.cpu().numpy().reshape(n // 2, n // 2, n // 2), no.restrict(fine))      # M2, same order
        pg.pg3n_absorb(h0, mean)
        pg.pg3n_solve(h0); pg.pg3n_solve(h1)
        pg.pg3n_add_exterior(h0, None)
        pg.pg3n_pack_exterior(h0, halo)
        with pytest.raises(pg.PolargravError) as e:            # level 1 needs its parent's values
            pg.pg3n_add_exterior(h1, None)
        assert e.value.status == pg.PG_ERR_STATE             # no inbox yet: a state error, like restrict / absorb / pack
        pg.pg3n_add_exterior(h1, halo)
        out0 = np.empty((n, n, n)); out1 = np.empty((n, n, n))
        pg.pg3n_potential(h0, out0, pg.PG_MEM_HOST); pg.pg3n_potential(h1, out1, pg.PG_MEM_HOST)
        ref, rho = no.nested_potential(n, box0, [coarse, fine])
        check(out0, ref[0], "level 0"); check(out1, ref[1], "level 1")
        # the packed message is (out_0 + E_0) on the parent cells that cross the boundary; E_1 is its prolongation
        import oracle
        ref_halo = no.pack_halo(oracle.cart_potential(n, box0, no.mask_centre(rho[0])))
        got_halo = halo.cpu().numpy().reshape((n // 2 + 2,) * 3)
        check(got_halo, ref_halo, "halo")
        ext1 = out1 - oracle.cart_potential(n, box0 / 2, fine)
        assert np.abs(ext1 - no.prolong(got_halo, n)).max() <= 1e-11 * np.abs(out1).max()
    finally:
        pg.pg3n_destroy(h0); pg.pg3n_destroy(h1)


@pytest.mark.parametrize("n", [64, 128])
def test_coupling_kernels_at_the_papers_mesh_sizes(n):
    """The five coupling kernels (restrict, absorb, mask, pack, prolong) at 64^3 and 128^3 against the numpy
    oracle steps.  The oracle's per-level solve costs n^6 and is out of reach here, so the single-level solves the
    coupling sits between are taken from pg3_potential -- the path test_gpu_cartesian.py holds to the oracle -- and only
    the coupling arithmetic is under test: copies and the 8-child mean must be exact, the trilinear sum within rounding."""
    box0 = 4.0
    rng = np.random.default_rng(100 + n)
    coarse, fine = rng.random((n, n, n)), rng.random((n, n, n))
    st = torch.cuda.current_stream().cuda_stream
    h0 = pg.pg3n_create(n, box0, 0, 2, 0, st)
    h1 = pg.pg3n_create(n, box0, 1, 2, 0, st)
    m0, m1 = pg.pg3_create(n, box0, 0, st), pg.pg3_create(n, box0 / 2, 0, st)

    def single(mesh, rho):
        d_r = torch.from_numpy(np.ascontiguousarray(rho)).cuda(); d_p = torch.empty_like(d_r)
        pg.pg3_set_density(mesh, d_r, pg.PG_MEM_DEVICE)
        pg.pg3_potential(mesh, d_p, pg.PG_MEM_DEVICE)
        pg.pg3_synchronize(mesh)
        return d_p.cpu().numpy()

    try:
        n_mean, n_halo = nested.message_counts(n)
        mean = torch.zeros(n_mean, dtype=torch.float64, device="cuda")
        halo = torch.zeros(n_halo, dtype=torch.float64, device="cuda")
        pg.pg3n_set_density(h0, torch.from_numpy(coarse).cuda(), pg.PG_MEM_DEVICE)
        pg.pg3n_set_density(h1, torch.from_numpy(fine).cuda(), pg.PG_MEM_DEVICE)
        pg.pg3n_restrict(h1, mean)
        pg.pg3n_synchronize(h1)
        got_mean = mean.cpu().numpy().reshape((n // 2,) * 3)
        assert np.array_equal(got_mean, no.restrict(fine))                                        # restrict (M2)
        pg.pg3n_absorb(h0, mean)
        pg.pg3n_solve(h0); pg.pg3n_solve(h1)
        pg.pg3n_add_exterior(h0, None)
        pg.pg3n_pack_exterior(h0, halo)
        pg.pg3n_add_exterior(h1, halo)
        out0, out1 = np.empty((n, n, n)), np.empty((n, n, n))
        pg.pg3n_potential(h0, out0, pg.PG_MEM_HOST); pg.pg3n_potential(h1, out1, pg.PG_MEM_HOST)
        rho0 = no.absorb(coarse, got_mean)
        assert np.array_equal(out0, single(m0, rho0))                                             # absorb (M2); E_0 = 0 (M6)
        got_halo = halo.cpu().numpy().reshape((n // 2 + 2,) * 3)
        assert np.array_equal(got_halo, no.pack_halo(single(m0, no.mask_centre(rho0))))           # mask (M3) + pack (M5)
        want1 = single(m1, fine) + no.prolong(got_halo, n)                                        # prolong (M5) + M6
        assert np.abs(out1 / want1 - 1.0).max() <= 1e-15 * 8
    finally:
        pg.pg3n_destroy(h0); pg.pg3n_destroy(h1); pg.pg3_destroy(m0); pg.pg3_destroy(m1)


# ------------------------------------------------------------------ one level per process, one-sided exchange
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _put_worker(rank, world, port, n, box0, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)       # control messages only: the payload is PUT
    try:
        torch.cuda.set_device(0)
        solver = nested.NestedPotential(n, box0, world, device=0, dist=dist, link="put")
        try:
            d_rho = {rank: torch.from_numpy(level_rho(n, rank, world)).cuda()}
            d_out = {rank: torch.zeros_like(d_rho[rank])}
            for rep in range(3):                                   # the inboxes are reused safely from solve to solve
                solver.solve(d_rho, d_out)
            solver.synchronize()
            out.put((rank, d_out[rank].cpu().numpy(), solver.launches()))
        finally:
            solver.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("depth", [2, 3])
def test_one_level_per_process_one_sided_puts(depth):
    """The paper's distribution (one nested mesh per image / GPU) with its communication model
    (one-sided transfers): every level lives in its own PROCESS, exports its inboxes by CUDA IPC handle,
    and its neighbours' kernels write the level-boundary messages straight into them; torch.distributed (gloo) carries
    only the one-element tokens.  The processes share the one GPU of this box (no kernel ever waits on another
    process's kernel: the hand-over is by host messages), so what is exercised is handles, peer pointers, order and
    reuse of the inboxes -- not NVLink.  Results must equal the oracle."""
    import torch.multiprocessing as mp
    n, box0 = 32, 8.0
    port = _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_put_worker, args=(r, depth, port, n, box0, out)) for r in range(depth)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(depth):
        r, phi, launches = out.get(timeout=300)
        got[r] = phi
        assert launches > 0
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    ref, _ = no.nested_potential(n, box0, [level_rho(n, l, depth) for l in range(depth)])
    for l in range(depth):
        check(got[l], ref[l], f"one-sided, depth {depth}, level {l}")


def test_one_sided_inside_one_process_and_inbox_errors():
    """The same NULL-pointer calls with the neighbour's inbox given by plain device pointer (pg3n_peer_set)."""
    n, box0 = 32, 4.0
    rng = np.random.default_rng(12)
    coarse, fine = rng.random((n, n, n)), rng.random((n, n, n))
    st = torch.cuda.current_stream().cuda_stream
    h0 = pg.pg3n_create(n, box0, 0, 2, 0, st)
    h1 = pg.pg3n_create(n, box0, 1, 2, 0, st)
    try:
        for bad in (lambda: pg.pg3n_inbox_export(h1, pg.PG3N_INBOX_MEAN), lambda: pg.pg3n_inbox_export(h0, pg.PG3N_INBOX_HALO)):
            with pytest.raises(pg.PolargravError) as e:
                bad()
            assert e.value.status == pg.PG_ERR_STATE
        pg.pg3n_set_density(h0, coarse, pg.PG_MEM_HOST)
        pg.pg3n_set_density(h1, fine, pg.PG_MEM_HOST)
        with pytest.raises(pg.PolargravError) as e:            # the parent's inbox has not been opened
            pg.pg3n_restrict(h1, None)
        assert e.value.status == pg.PG_ERR_STATE
        handle, mean_addr = pg.pg3n_inbox_export(h0, pg.PG3N_INBOX_MEAN)
        _, halo_addr = pg.pg3n_inbox_export(h1, pg.PG3N_INBOX_HALO)
        assert len(handle) == pg.PG_IPC_HANDLE_BYTES and mean_addr % 16 == 0 and halo_addr % 16 == 0
        pg.pg3n_peer_set(h1, pg.PG3N_INBOX_MEAN, mean_addr)
        pg.pg3n_peer_set(h0, pg.PG3N_INBOX_HALO, halo_addr)
        pg.pg3n_restrict(h1, None); pg.pg3n_absorb(h0, None)
        pg.pg3n_solve(h0); pg.pg3n_solve(h1)
        pg.pg3n_add_exterior(h0, None); pg.pg3n_pack_exterior(h0, None); pg.pg3n_add_exterior(h1, None)
        out0 = np.empty((n, n, n)); out1 = np.empty((n, n, n))
        pg.pg3n_potential(h0, out0, pg.PG_MEM_HOST); pg.pg3n_potential(h1, out1, pg.PG_MEM_HOST)
        ref, _ = no.nested_potential(n, box0, [coarse, fine])
        check(out0, ref[0], "level 0"); check(out1, ref[1], "level 1")
    finally:
        pg.pg3n_destroy(h0); pg.pg3n_destroy(h1)

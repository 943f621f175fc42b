"""Boundary behaviour on a real device: the three memspaces (row a6: pinned staging on CUDA
streams, Fig. 4 :202), ordering, state errors, batch rules, profiling
counters.  Arithmetic parity lives in test_gpu_parity.py."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2409_02294_b200 import binding as pg
from paper_2409_02294_b200.workloads import random_sigma

pytestmark = pytest.mark.gpu

N_R, N_PHI, R_IN, R_OUT, EPS = 128, 256, 1.0, 300.0, 0.01


@pytest.fixture()
def solver():
    s = pg.Solver(N_R, N_PHI, R_IN, R_OUT, EPS, max_batch=4, device=0,
                  cuda_stream=torch.cuda.current_stream().cuda_stream)
    yield s
    s.close()


def device_solve(s, sig):
    batch = 1 if sig.ndim == 2 else sig.shape[0]
    d_s = torch.from_numpy(np.ascontiguousarray(sig)).cuda()
    d_p = torch.empty_like(d_s)
    pg.pg_set_density(s.h, d_s, batch, pg.PG_MEM_DEVICE)
    pg.pg_potential(s.h, d_p, batch, pg.PG_MEM_DEVICE)
    pg.pg_synchronize(s.h)
    return d_p.cpu().numpy()


def test_memspaces_agree_bit_for_bit(solver):
    sig = np.stack([random_sigma(N_R, N_PHI, 10 + b) for b in range(4)])
    ref = np.stack([oracle.potential_o1(N_R, N_PHI, R_IN, R_OUT, EPS, sig[b]) for b in range(4)])
    dev = device_solve(solver, sig)
    assert np.abs(dev / ref - 1).max() <= 1e-9
    # pageable host -> staged through owned pinned buffers, blocking
    host = solver.potential_host(sig)
    assert np.array_equal(host, dev)
    # caller-owned pinned memory (pg_host_alloc), asynchronous
    pin_in, pin_out = pg.PinnedArray(sig.shape), pg.PinnedArray(sig.shape)
    try:
        pin_in.array[...] = sig
        pin_out.array[...] = 0.0
        pg.pg_set_density(solver.h, pin_in.ptr, 4, pg.PG_MEM_HOST_PINNED)
        pg.pg_potential(solver.h, pin_out.ptr, 4, pg.PG_MEM_HOST_PINNED)
        pg.pg_synchronize(solver.h)
        assert np.array_equal(pin_out.array, dev)
        # mixed: host density, device potential
        d_p = torch.empty(sig.shape, dtype=torch.float64, device="cuda")
        pg.pg_set_density(solver.h, sig, 4, pg.PG_MEM_HOST)
        pg.pg_potential(solver.h, d_p, 4, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(solver.h)
        assert np.array_equal(d_p.cpu().numpy(), dev)
        # mixed: device density, host potential
        d_s = torch.from_numpy(sig).cuda()
        out = np.empty_like(sig)
        pg.pg_set_density(solver.h, d_s, 4, pg.PG_MEM_DEVICE)
        pg.pg_potential(solver.h, out, 4, pg.PG_MEM_HOST)
        assert np.array_equal(out, dev)
    finally:
        pin_in.free(); pin_out.free()


def test_repeated_host_solves_reuse_staging_safely(solver):
    prev = None
    for k in range(6):
        sig = random_sigma(N_R, N_PHI, 50 + k)
        got = solver.potential_host(sig)
        ref = device_solve(solver, sig)
        assert np.array_equal(got, ref)
        assert prev is None or not np.array_equal(prev, got)
        prev = got


def test_direct_host_path_and_rings(solver):
    sig = random_sigma(N_R, N_PHI, 3)
    full = solver.potential_host(sig, direct=True)
    ref = oracle.potential_o1(N_R, N_PHI, R_IN, R_OUT, EPS, sig)
    assert np.abs(full / ref - 1).max() <= 1e-12
    out = np.empty((5, N_PHI))
    pg.pg_set_density(solver.h, sig, 1, pg.PG_MEM_HOST)
    pg.pg_potential_direct_rings(solver.h, out, 100, 5, pg.PG_MEM_HOST)
    assert np.array_equal(out, full[100:105])
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_rings(solver.h, out, 125, 5, pg.PG_MEM_HOST)
    assert e.value.status == pg.PG_ERR_INVALID_ARG


def test_state_and_argument_errors(solver):
    out = np.empty((N_R, N_PHI))
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential(solver.h, out, 1, pg.PG_MEM_HOST)          # before any density
    assert e.value.status == pg.PG_ERR_STATE
    sig = random_sigma(N_R, N_PHI, 1)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_set_density(solver.h, sig, 5, pg.PG_MEM_HOST)         # batch > max_batch
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_set_density(solver.h, sig, 0, pg.PG_MEM_HOST)
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_set_density(solver.h, sig, 1, 7)                      # unknown memspace
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    pg.pg_set_density(solver.h, sig, 1, pg.PG_MEM_HOST)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential(solver.h, out, 2, pg.PG_MEM_HOST)           # batch mismatch
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    assert "batch" in pg.last_error(solver.h)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_set_option(solver.h, 99, 1)                           # unknown option
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    pg.pg_set_option(solver.h, pg.PG_OPT_DENSITY_STABLE, 1)         # has no effect on host-staged solves
    pg.pg_potential(solver.h, out, 1, pg.PG_MEM_HOST)               # still usable after errors
    assert np.isfinite(out).all()
    pg.pg_set_option(solver.h, pg.PG_OPT_DENSITY_STABLE, 0)


def test_nan_propagates_not_checked(solver):
    sig = random_sigma(N_R, N_PHI, 2)
    sig[7, 9] = np.nan
    assert np.isnan(solver.potential_host(sig)).any()


def test_own_stream_and_set_stream():
    st = torch.cuda.Stream()
    s = pg.Solver(64, 64, 1.0, 100.0, 0.01, device=0, cuda_stream=st.cuda_stream)
    try:
        sig = random_sigma(64, 64, 5)
        with torch.cuda.stream(st):
            d_s = torch.from_numpy(sig).cuda()
            d_p = torch.empty_like(d_s)
        st.synchronize()
        pg.pg_set_density(s.h, d_s, 1, pg.PG_MEM_DEVICE)
        pg.pg_potential(s.h, d_p, 1, pg.PG_MEM_DEVICE)
        st.synchronize()
        a = d_p.cpu().numpy()
        pg.pg_set_stream(s.h, None)                                   # legacy default stream
        pg.pg_potential(s.h, d_p, 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(s.h)
        assert np.array_equal(a, d_p.cpu().numpy())
        ref = oracle.potential_o1(64, 64, 1.0, 100.0, 0.01, sig)
        assert np.abs(a / ref - 1).max() <= 1e-9
    finally:
        s.close()


def test_profile_counters_and_algorithmic_bytes(solver):
    sig = np.stack([random_sigma(N_R, N_PHI, 20 + b) for b in range(2)])
    d_s = torch.from_numpy(sig).cuda()
    d_p = torch.empty_like(d_s)
    pg.pg_set_density(solver.h, d_s, 2, pg.PG_MEM_DEVICE)
    n0 = pg.pg_launch_count(solver.h)
    pg.pg_profile(solver.h, True)
    for _ in range(5):
        pg.pg_potential(solver.h, d_p, 2, pg.PG_MEM_DEVICE)
    ms, n = pg.pg_kernel_times(solver.h)
    pg.pg_profile(solver.h, False)
    assert n == [5, 5, 5] and all(t > 0 for t in ms)
    assert pg.pg_launch_count(solver.h) - n0 == 15                   # three kernels per solve
    m_h = N_PHI // 2 + 1
    cells, spec = N_R * N_PHI, 16 * N_R * m_h
    assert pg.pg_kernel_algorithmic_bytes(solver.h, 0, 2) == 2 * (8 * cells + spec)
    assert pg.pg_kernel_algorithmic_bytes(solver.h, 1, 2) == 2 * 2 * spec + 16 * N_R * m_h
    assert pg.pg_kernel_algorithmic_bytes(solver.h, 2, 2) == 2 * (spec + 8 * cells)
    assert pg.pg_algorithmic_bytes(solver.h, 2) == sum(pg.pg_kernel_algorithmic_bytes(solver.h, k, 2) for k in range(3))


def test_two_solvers_are_independent():
    a = pg.Solver(64, 64, 1.0, 100.0, 0.01, device=0)
    b = pg.Solver(64, 128, 1.0, 50.0, 0.02, device=0)
    try:
        sa, sb = random_sigma(64, 64, 1), random_sigma(64, 128, 2)
        pa1 = a.potential_host(sa)
        pb = b.potential_host(sb)
        pa2 = a.potential_host(sa)
        assert np.array_equal(pa1, pa2)
        assert np.abs(pb / oracle.potential_o1(64, 128, 1.0, 50.0, 0.02, sb) - 1).max() <= 1e-9
    finally:
        a.close(); b.close()


def test_misaligned_device_pointers_are_rejected(solver):
    """the kernels move device arrays as 16-byte vectors; a view at an odd element offset must be
    refused (PG_ERR_INVALID_ARG), not run into a sticky misaligned-address fault."""
    n = N_R * N_PHI
    buf = torch.zeros(2 * n + 2, dtype=torch.float64, device="cuda")
    odd_in, odd_out = buf[1:1 + n], buf[n + 1:2 * n + 1]           # 8 bytes past a 16-byte boundary
    assert odd_in.data_ptr() % 16 == 8 and odd_out.data_ptr() % 16 == 8
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_set_density(solver.h, odd_in, 1, pg.PG_MEM_DEVICE)
    assert e.value.status == pg.PG_ERR_INVALID_ARG and "aligned" in pg.last_error(solver.h)
    sig = torch.from_numpy(random_sigma(N_R, N_PHI, 4)).cuda()
    pg.pg_set_density(solver.h, sig, 1, pg.PG_MEM_DEVICE)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential(solver.h, odd_out, 1, pg.PG_MEM_DEVICE)
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct(solver.h, odd_out, 1, pg.PG_MEM_DEVICE)
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    good = torch.empty_like(sig)
    pg.pg_potential(solver.h, good, 1, pg.PG_MEM_DEVICE)            # the context is still healthy
    pg.pg_synchronize(solver.h)
    assert torch.isfinite(good).all()


def test_potential_overlapping_the_density_is_rejected(solver):
    sig = torch.from_numpy(np.stack([random_sigma(N_R, N_PHI, 30 + b) for b in range(2)])).cuda()
    pg.pg_set_density(solver.h, sig, 2, pg.PG_MEM_DEVICE)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential(solver.h, sig, 2, pg.PG_MEM_DEVICE)          # in place
    assert e.value.status == pg.PG_ERR_INVALID_ARG and "overlap" in pg.last_error(solver.h)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential(solver.h, sig[1:], 2, pg.PG_MEM_DEVICE)      # partial overlap (field 1 onwards)
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    out = torch.empty_like(sig)
    pg.pg_potential(solver.h, out, 2, pg.PG_MEM_DEVICE)
    pg.pg_synchronize(solver.h)
    assert (out < 0).all()


def test_calls_leave_the_current_device_alone(solver):
    before = torch.cuda.current_device()
    sig = random_sigma(N_R, N_PHI, 6)
    solver.potential_host(sig)
    pg.pg_synchronize(solver.h)
    assert torch.cuda.current_device() == before


def test_fed_back_potential_with_another_solver_in_between():
    """the early-fetch alias guard is per stream.  Solver A solves, solver B solves on ANOTHER
    stream, then A is fed its own (still in flight) potential as the next density with PG_OPT_DENSITY_STABLE on:
    the library must notice the overlap and fall back to the ordered launch, so the chain equals the same chain
    run with a synchronisation after every step."""
    n_r, n_phi = 512, 512
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    A = pg.Solver(n_r, n_phi, 1.0, 1000.0, 0.01, device=0, cuda_stream=sa.cuda_stream)
    B = pg.Solver(n_r, n_phi, 1.0, 1000.0, 0.01, device=0, cuda_stream=sb.cuda_stream)
    try:
        for s in (A, B):
            pg.pg_set_option(s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        x0 = torch.from_numpy(random_sigma(n_r, n_phi, 77)).cuda()
        yb = torch.from_numpy(random_sigma(n_r, n_phi, 78)).cuda()
        torch.cuda.synchronize()

        def chain(sync_every_step):
            bufs = [x0.clone(), torch.empty_like(x0), torch.empty_like(x0), torch.empty_like(x0)]
            outb = torch.empty_like(x0)
            torch.cuda.synchronize()
            for k in range(3):
                pg.pg_set_density(A.h, bufs[k], 1, pg.PG_MEM_DEVICE)
                pg.pg_potential(A.h, bufs[k + 1], 1, pg.PG_MEM_DEVICE)      # A: Phi_k -> next density
                if sync_every_step:
                    torch.cuda.synchronize()
                pg.pg_set_density(B.h, yb, 1, pg.PG_MEM_DEVICE)              # B on another stream in between
                pg.pg_potential(B.h, outb, 1, pg.PG_MEM_DEVICE)
                if sync_every_step:
                    torch.cuda.synchronize()
            torch.cuda.synchronize()
            return bufs[3].cpu().numpy()

        ref = chain(True)
        for _ in range(5):
            assert np.array_equal(chain(False), ref)
    finally:
        A.close(); B.close()


@pytest.mark.parametrize("n_r,n_phi,batch", [(1024, 1024, 2), (2048, 2048, 1), (256, 512, 3)])
def test_two_lanes_equal_one_lane_bit_for_bit(n_r, n_phi, batch):
    """PG_OPT_LANES = 2, 3: independent resident solves go in turn to that many internal streams; results are those of the
    ordinary path bit for bit, complete after pg_flush + a sync of the solver's stream (or pg_synchronize)."""
    st = torch.cuda.Stream()
    s = pg.Solver(n_r, n_phi, 1.0, 1000.0, 0.01, max_batch=batch, device=0, cuda_stream=st.cuda_stream)
    try:
        pg.pg_set_option(s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        K = 7
        sig = [torch.from_numpy(np.stack([random_sigma(n_r, n_phi, 900 + 10 * k + b) for b in range(batch)])).cuda() for k in range(K)]
        torch.cuda.synchronize()

        def run(lanes):
            pg.pg_set_option(s.h, pg.PG_OPT_LANES, lanes)
            out = [torch.zeros_like(x) for x in sig]
            torch.cuda.synchronize()
            for rep in range(3):
                for k in range(K):
                    pg.pg_set_density(s.h, sig[k], batch, pg.PG_MEM_DEVICE)
                    pg.pg_potential(s.h, out[k], batch, pg.PG_MEM_DEVICE)
            pg.pg_flush(s.h)
            st.synchronize()                                     # the solver's stream alone: pg_flush joined the lanes
            return [o.cpu().numpy() for o in out]

        one = run(1)
        for lanes in (2, 3):
            many = run(lanes)
            for a, b in zip(one, many):
                assert np.array_equal(a, b) and (a < 0).all()
        # a host-staged solve in between keeps working (it uses the solver's own stream)
        host = s.potential_host(sig[0].cpu().numpy())
        assert np.array_equal(host, one[0])
        pg.pg_set_option(s.h, pg.PG_OPT_LANES, 1)
        with pytest.raises(pg.PolargravError) as e:
            pg.pg_set_option(s.h, pg.PG_OPT_LANES, 5)          # PG_MAX_LANES = 4
        assert e.value.status == pg.PG_ERR_INVALID_ARG
    finally:
        s.close()


@pytest.mark.parametrize("n_r,n_phi,batch", [(64, 64, 1), (64, 64, 5), (256, 256, 1), (512, 512, 1), (512, 512, 3),
                                             (64, 512, 2), (512, 64, 2), (128, 256, 4)])
def test_fused_single_launch_equals_three_kernels_bit_for_bit(n_r, n_phi, batch):
    """PG_OPT_FUSED (default on): grids of 64 .. 512 cells per axis are solved by ONE cooperative launch (the three
    kernel bodies separated by grid-wide barriers) as long as all its CTAs are resident at once; larger batches fall
    back to the three kernels.  Same arithmetic: bit-identical potentials, one launch per solve instead of three, and
    parity with the oracle on field 0."""
    st = torch.cuda.Stream()
    s = pg.Solver(n_r, n_phi, 1.0, 300.0, 0.01, max_batch=batch, device=0, cuda_stream=st.cuda_stream)
    try:
        sig = np.stack([random_sigma(n_r, n_phi, 4000 + b) for b in range(batch)])
        d_s = torch.from_numpy(sig).cuda()
        got = {}
        for fused in (0, 1):
            pg.pg_set_option(s.h, pg.PG_OPT_FUSED, fused)
            out = torch.zeros_like(d_s)
            n0 = pg.pg_launch_count(s.h)
            for _ in range(3):                                   # back to back: the W workspace is reused safely
                pg.pg_set_density(s.h, d_s, batch, pg.PG_MEM_DEVICE)
                pg.pg_potential(s.h, out, batch, pg.PG_MEM_DEVICE)
            pg.pg_synchronize(s.h)
            got[fused] = (out.cpu().numpy(), pg.pg_launch_count(s.h) - n0)
        assert np.array_equal(got[0][0], got[1][0])
        assert got[0][1] == 9
        assert got[1][1] in (3, 9)                               # 9: the batch does not fit one resident grid
        if batch == 1 or n_r * n_phi <= 128 * 256:
            assert got[1][1] == 3
        ref = oracle.potential_o1(n_r, n_phi, 1.0, 300.0, 0.01, sig[0])
        assert np.linalg.norm(got[1][0][0] - ref) / np.linalg.norm(ref) <= 1e-10
        assert np.abs(got[1][0][0] / ref - 1).max() <= 1e-9
        # the host-staged path goes through the same fused launch, one field at a time
        host = s.potential_host(sig)
        assert np.array_equal(host, got[1][0])
    finally:
        s.close()


@pytest.mark.parametrize("n_r,n_phi", [(64, 64), (256, 256), (512, 512)])
def test_fused_solves_on_four_lanes_equal_the_ordinary_path(n_r, n_phi):
    """Small grids in throughput mode, the launch configuration bench.py times for configs 1-3: PG_OPT_LANES = 4 deals
    the fused launches out over four internal streams; results equal the one-lane three-kernel path bit for bit."""
    st = torch.cuda.Stream()
    s = pg.Solver(n_r, n_phi, 1.0, 500.0, 0.01, device=0, cuda_stream=st.cuda_stream)
    try:
        pg.pg_set_option(s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        K = 9
        sig = [torch.from_numpy(random_sigma(n_r, n_phi, 5000 + k)[None]).cuda() for k in range(K)]
        torch.cuda.synchronize()
        res = {}
        for lanes, fused in ((1, 0), (4, 1)):
            pg.pg_set_option(s.h, pg.PG_OPT_LANES, lanes)
            pg.pg_set_option(s.h, pg.PG_OPT_FUSED, fused)
            out = [torch.zeros_like(x) for x in sig]
            torch.cuda.synchronize()
            for rep in range(3):
                for k in range(K):
                    pg.pg_set_density(s.h, sig[k], 1, pg.PG_MEM_DEVICE)
                    pg.pg_potential(s.h, out[k], 1, pg.PG_MEM_DEVICE)
            pg.pg_flush(s.h)
            st.synchronize()
            res[lanes] = [o.cpu().numpy() for o in out]
        for a, b in zip(res[1], res[4]):
            assert np.array_equal(a, b) and (a < 0).all()
    finally:
        s.close()


@pytest.mark.parametrize("batch", [1, 3])
def test_lanes_with_a_device_density_and_a_host_potential_stay_on_the_solvers_stream(batch):
    """PG_OPT_LANES >= 2 + PG_OPT_DENSITY_STABLE, device Sigma, HOST Phi: the staged download waits for events on the
    solver's stream, so these solves must not go to a lane (polargrav.h: host memspaces keep using the solver's stream).
    Before the fix field 0 was solved on a lane stream and its download could run ahead of it (stale data)."""
    n_r, n_phi = 256, 512
    st = torch.cuda.Stream()
    s = pg.Solver(n_r, n_phi, 1.0, 1000.0, 0.01, max_batch=batch, device=0, cuda_stream=st.cuda_stream)
    pin = pg.PinnedArray((batch, n_r, n_phi))
    try:
        pg.pg_set_option(s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        K = 6
        sig = [torch.from_numpy(np.stack([random_sigma(n_r, n_phi, 1300 + 10 * k + b) for b in range(batch)])).cuda() for k in range(K)]
        torch.cuda.synchronize()

        def run(lanes, where):
            pg.pg_set_option(s.h, pg.PG_OPT_LANES, lanes)
            res = []
            for k in range(K):
                pg.pg_set_density(s.h, sig[k], batch, pg.PG_MEM_DEVICE)
                if where == pg.PG_MEM_HOST:
                    out = np.full((batch, n_r, n_phi), np.nan)
                    pg.pg_potential(s.h, out, batch, where)            # blocks until filled
                    res.append(out)
                else:
                    pin.array[...] = np.nan
                    pg.pg_potential(s.h, pin.ptr, batch, where)
                    pg.pg_synchronize(s.h)
                    res.append(pin.array.copy())
            return res

        one = run(1, pg.PG_MEM_HOST)
        assert all((x < 0).all() for x in one)
        for lanes in (2, 4):
            for where in (pg.PG_MEM_HOST, pg.PG_MEM_HOST_PINNED):
                for a, b in zip(one, run(lanes, where)):
                    assert np.array_equal(a, b)
    finally:
        pin.free()
        s.close()


def test_profiling_survives_a_solve_with_non_symmetric_softening(solver):
    """pg_profile(1) + PG_SOFT_FIELD / PG_SOFT_SOURCE: the variant path records no per-kernel events, so it must not take
    a profiling slot; afterwards pg_kernel_times, pg_profile and pg_set_stream keep working and the counters hold only
    the symmetric solves."""
    sig = random_sigma(N_R, N_PHI, 77)
    d_s = torch.from_numpy(sig).cuda()
    d_p = torch.empty_like(d_s)
    pg.pg_set_density(solver.h, d_s, 1, pg.PG_MEM_DEVICE)
    pg.pg_profile(solver.h, True)
    pg.pg_potential(solver.h, d_p, 1, pg.PG_MEM_DEVICE)
    for soft in (pg.PG_SOFT_FIELD, pg.PG_SOFT_SOURCE):
        pg.pg_set_softening(solver.h, soft)
        pg.pg_potential(solver.h, d_p, 1, pg.PG_MEM_DEVICE)
        ms, n = pg.pg_kernel_times(solver.h)
        assert n == [1, 1, 1]
    pg.pg_set_softening(solver.h, pg.PG_SOFT_SYMMETRIC)
    pg.pg_potential(solver.h, d_p, 1, pg.PG_MEM_DEVICE)
    ms, n = pg.pg_kernel_times(solver.h)
    assert n == [2, 2, 2] and all(t > 0 for t in ms)
    pg.pg_profile(solver.h, False)
    pg.pg_set_stream(solver.h, torch.cuda.current_stream().cuda_stream)
    pg.pg_synchronize(solver.h)


@pytest.mark.parametrize("n_r,n_phi,lanes", [(64, 64, 1), (256, 128, 4), (512, 512, 2), (1024, 1024, 2)])
def test_series_call_equals_the_same_solves_one_by_one(n_r, n_phi, lanes):
    """pg_potential_series: `count` solves enqueued by one host call are the solves of `count` pg_set_density /
    pg_potential pairs bit for bit -- fused small grids and the three-kernel path, with and without lanes, with a
    stride larger than a field (the gap must stay untouched)."""
    st = torch.cuda.Stream()
    s = pg.Solver(n_r, n_phi, 1.0, 400.0, 0.02, device=0, cuda_stream=st.cuda_stream)
    try:
        count, field = 9, n_r * n_phi
        stride = field + 6
        sig = np.zeros((count, stride)); 
        for k in range(count):
            sig[k, :field] = random_sigma(n_r, n_phi, 2100 + k).ravel()
        d_s = torch.from_numpy(sig).cuda()
        one = torch.full_like(d_s, 7.0)
        many = torch.full_like(d_s, 7.0)
        torch.cuda.synchronize()
        pg.pg_set_option(s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        for k in range(count):
            pg.pg_set_density(s.h, d_s[k].data_ptr(), 1, pg.PG_MEM_DEVICE)
            pg.pg_potential(s.h, one[k].data_ptr(), 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(s.h)
        pg.pg_set_option(s.h, pg.PG_OPT_LANES, lanes)
        for rep in range(2):
            pg.pg_potential_series(s.h, d_s, many, count, stride)
        pg.pg_flush(s.h)
        st.synchronize()
        a, b = one.cpu().numpy(), many.cpu().numpy()
        assert np.array_equal(a, b)
        assert (b[:, :field] < 0).all() and (b[:, field:] == 7.0).all()
        # afterwards the density set is the last field
        last = torch.empty(n_r, n_phi, dtype=torch.float64, device="cuda")
        pg.pg_potential(s.h, last, 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(s.h)
        assert np.array_equal(last.cpu().numpy().ravel(), b[count - 1, :field])
        for bad in (lambda: pg.pg_potential_series(s.h, d_s, many, 0, stride),
                    lambda: pg.pg_potential_series(s.h, d_s, many, count, field - 2),
                    lambda: pg.pg_potential_series(s.h, d_s, many, count, field + 1),
                    lambda: pg.pg_potential_series(s.h, d_s, d_s.data_ptr() + 16, 2, stride),
                    lambda: pg.pg_potential_series(s.h, d_s.data_ptr() + 8, many, 2, stride)):
            with pytest.raises(pg.PolargravError) as e:
                bad()
            assert e.value.status == pg.PG_ERR_INVALID_ARG
    finally:
        s.close()

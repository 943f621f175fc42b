"""pg_potential_direct_static: the one call of the library that takes no device memory (include/polargrav.h).

It exists for programs that cannot give the library any: a simulation whose own arena already owns all free HBM (a
later cudaMalloc fails), a job inside a fixed memory budget (MIG slice, MPS limit), a plug-in that is only lent
device pointers.  pg_create* and, on first use of some options, pg_potential allocate; this call keeps the three
grid tables of the direct kernels in a fixed 48 KiB array of the library image, shared by all calls on a GPU and
never cleared between them.  So the checks here are: two calls IN A ROW on different grids (the second smaller, so
that entries of the first are still lying in the array behind it) each equal the existing path -- the solver-based
pg_potential_direct, the FFT solve and the oracle, at the bars every parity test uses (relative L2 <= 1e-10, max
pointwise relative <= 1e-9); the free device memory does not move across the calls; grids beyond the fixed array
are refused with a message that names the limit.

The file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process (the first call then does the one-time address look-up) and
after the rest of the suite (the library is then long loaded and other solvers have come and gone)."""
import numpy as np
import pytest

import oracle
from paper_2409_02294_b200 import binding as pg
from paper_2409_02294_b200.workloads import random_sigma

REL_L2, MAX_REL = 1e-10, 1e-9      # north_star's bars, as in tests/test_gpu_parity.py


def _errors(got, ref):
    return np.linalg.norm(got - ref) / np.linalg.norm(ref), np.abs(got / ref - 1.0).max()


def _existing_paths(torch, n_r, n_phi, r_in, r_out, eps, d_sigma):
    """pg_potential_direct and pg_potential of an ordinary (allocating) solver for the same grid and density."""
    s = pg.Solver(n_r, n_phi, r_in, r_out, eps, device=0, cuda_stream=torch.cuda.current_stream().cuda_stream)
    try:
        d_direct, d_fft = torch.empty_like(d_sigma), torch.empty_like(d_sigma)
        pg.pg_set_density(s.h, d_sigma, 1, pg.PG_MEM_DEVICE)
        pg.pg_potential_direct(s.h, d_direct, 1, pg.PG_MEM_DEVICE)
        pg.pg_potential(s.h, d_fft, 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(s.h)
        return d_direct.cpu().numpy(), d_fft.cpu().numpy()
    finally:
        s.close()


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path_and_allocate_nothing():
    torch = pytest.importorskip("torch")
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    # (n_r, n_phi, r_in, r_out, eps): the register-tiled kernel, then the plain one on a smaller grid
    grids = [(128, 256, 1.0, 300.0, 0.01), (64, 64, 2.0, 150.0, 0.05)]
    sig = [random_sigma(g[0], g[1], 700 + k) for k, g in enumerate(grids)]
    d_sig = [torch.from_numpy(x).cuda() for x in sig]
    # Phi starts as NaN: a cell the kernel did not write cannot pass for a result
    d_phi = [torch.full_like(x, float("nan")) for x in d_sig]

    # the first call on a device does the one-time set-up (and loads the kernel's module): before the memory reading
    warm = torch.empty_like(d_sig[0])
    pg.pg_potential_direct_static(d_sig[0], warm, *grids[0], device=0, cuda_stream=stream)
    torch.cuda.synchronize()
    del warm

    free_before, _ = torch.cuda.mem_get_info()
    for k, g in enumerate(grids):          # back to back on one stream, nothing in between
        pg.pg_potential_direct_static(d_sig[k], d_phi[k], *g, device=0, cuda_stream=stream)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, "the call changed the amount of free device memory"

    for k, g in enumerate(grids):
        got = d_phi[k].cpu().numpy()
        assert np.isfinite(got).all()
        direct, fft = _existing_paths(torch, *g, d_sig[k])
        ref = oracle.potential_o1(*g, sig[k])
        for name, other in (("pg_potential_direct", direct), ("pg_potential", fft), ("oracle O1", ref)):
            l2, mx = _errors(got, other)
            assert l2 <= REL_L2 and mx <= MAX_REL, f"grid {g[:2]} vs {name}: rel-L2 {l2:.3e}, max rel {mx:.3e}"

    # and once more in the other order: the large grid after the small one has overwritten the head of the array
    d_again = torch.full_like(d_sig[0], float("nan"))
    pg.pg_potential_direct_static(d_sig[0], d_again, *grids[0], device=0, cuda_stream=stream)
    torch.cuda.synchronize()
    l2, mx = _errors(d_again.cpu().numpy(), d_phi[0].cpu().numpy())
    assert l2 <= REL_L2 and mx <= MAX_REL


def test_sizes_beyond_the_fixed_array_and_bad_arguments_are_refused():
    """Host-side checks only (they come before any CUDA call, so this part also runs on the CPU box)."""
    n = pg.PG_STATIC_MAX_N
    fake_in, fake_out = 0x10000000, 0x20000000          # never dereferenced: the checks fail first
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(fake_in, fake_out, 2 * n, 64, 1.0, 100.0, 0.01)
    assert e.value.status == pg.PG_ERR_UNSUPPORTED and str(n) in str(e.value) and "fixed" in str(e.value)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(fake_in, fake_out, 64, 2 * n, 1.0, 100.0, 0.01)
    assert e.value.status == pg.PG_ERR_UNSUPPORTED and str(n) in str(e.value)
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(fake_in, fake_out, 96, 64, 1.0, 100.0, 0.01)      # not a power of two
    assert e.value.status == pg.PG_ERR_UNSUPPORTED
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(fake_in + 8, fake_out, 64, 64, 1.0, 100.0, 0.01)  # misaligned
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(fake_in, fake_in + 64, 64, 64, 1.0, 100.0, 0.01)  # overlapping
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(None, fake_out, 64, 64, 1.0, 100.0, 0.01)
    assert e.value.status == pg.PG_ERR_INVALID_ARG
    with pytest.raises(pg.PolargravError) as e:
        pg.pg_potential_direct_static(fake_in, fake_out, 64, 64, 1.0, 0.5, 0.01)        # r_out <= r_in
    assert e.value.status == pg.PG_ERR_INVALID_ARG

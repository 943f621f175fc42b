"""Parity of the NEXT-4 variants (readings N1, N2 of DESIGN.md section 3) against
oracle/polar_oracle_ext.c: potential with field / source softening (complex kernel spectrum) and the softened
pair acceleration.  Potential: north_star's bar (rel-L2 <= 1e-10, max pointwise relative <= 1e-9).  Acceleration
components change sign across the grid, so the pointwise bar is taken relative to the magnitude of the
acceleration vector at the cell: |delta a_c| <= 1e-9 |a|, plus rel-L2 <= 1e-10 per component."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2409_02294_b200 import binding as pg
from paper_2409_02294_b200.workloads import CONFIGS, make_sigma, random_sigma

pytestmark = pytest.mark.gpu
SOFTS = (pg.PG_SOFT_SYMMETRIC, pg.PG_SOFT_FIELD, pg.PG_SOFT_SOURCE)


def solver(n_r, n_phi, r_in, r_out, eps, max_batch=1):
    return pg.Solver(n_r, n_phi, r_in, r_out, eps, max_batch=max_batch, device=0,
                     cuda_stream=torch.cuda.current_stream().cuda_stream)


def potential(s, sig):
    batch = 1 if sig.ndim == 2 else sig.shape[0]
    d_s = torch.from_numpy(np.ascontiguousarray(sig)).cuda(); d_p = torch.empty_like(d_s)
    pg.pg_set_density(s.h, d_s, batch, pg.PG_MEM_DEVICE)
    pg.pg_potential(s.h, d_p, batch, pg.PG_MEM_DEVICE)
    pg.pg_synchronize(s.h)
    return d_p.cpu().numpy()


def acceleration(s, sig):
    batch = 1 if sig.ndim == 2 else sig.shape[0]
    d_s = torch.from_numpy(np.ascontiguousarray(sig)).cuda()
    d_r, d_p = torch.empty_like(d_s), torch.empty_like(d_s)
    pg.pg_set_density(s.h, d_s, batch, pg.PG_MEM_DEVICE)
    pg.pg_acceleration(s.h, d_r, d_p, batch, pg.PG_MEM_DEVICE)
    pg.pg_synchronize(s.h)
    return d_r.cpu().numpy(), d_p.cpu().numpy()


def check_phi(got, ref, what):
    l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got / ref - 1.0).max()
    assert l2 <= 1e-10 and mx <= 1e-9, f"{what}: rel-L2 {l2:.3e}, max rel {mx:.3e}"


def check_acc(got_r, got_p, ref_r, ref_p, what):
    mag = np.hypot(ref_r, ref_p)
    for g, r, c in ((got_r, ref_r, "a_r"), (got_p, ref_p, "a_phi")):
        l2 = np.linalg.norm(g - r) / np.linalg.norm(r)
        mx = (np.abs(g - r) / mag).max()
        assert l2 <= 1e-10 and mx <= 1e-9, f"{what} {c}: rel-L2 {l2:.3e}, max |delta| / |a| {mx:.3e}"


@pytest.mark.parametrize("soft", SOFTS)
@pytest.mark.parametrize("n_r,n_phi,r_in,r_out,eps", [(64, 64, 1.0, 100.0, 0.01), (128, 256, 1.0, 300.0, 0.01), (256, 64, 0.5, 50.0, 0.3)])
def test_softening_modes_and_acceleration_full_grid(n_r, n_phi, r_in, r_out, eps, soft):
    s = solver(n_r, n_phi, r_in, r_out, eps)
    try:
        sig = random_sigma(n_r, n_phi, 400 + soft)
        ref_phi, ref_r, ref_p = oracle.ext_o1(n_r, n_phi, r_in, r_out, eps, soft, sig)
        pg.pg_set_softening(s.h, soft)
        check_phi(potential(s, sig), ref_phi, f"{n_r}x{n_phi} soft {soft} potential")
        a_r, a_p = acceleration(s, sig)
        check_acc(a_r, a_p, ref_r, ref_p, f"{n_r}x{n_phi} soft {soft}")
    finally:
        s.close()


def test_switching_back_to_symmetric_restores_the_default_path_bit_for_bit():
    n = 256
    s = solver(n, n, 1.0, 500.0, 0.01)
    try:
        sig = random_sigma(n, n, 77)
        base = potential(s, sig)
        pg.pg_set_softening(s.h, pg.PG_SOFT_FIELD)
        other = potential(s, sig)
        assert not np.array_equal(base, other) and np.abs(other / base - 1).max() < 0.2
        pg.pg_set_softening(s.h, pg.PG_SOFT_SYMMETRIC)
        assert np.array_equal(potential(s, sig), base)
        with pytest.raises(pg.PolargravError) as e:
            pg.pg_set_softening(s.h, 7)
        assert e.value.status == pg.PG_ERR_INVALID_ARG
    finally:
        s.close()


def test_acceleration_batch_host_memspace_and_argument_checks():
    n_r, n_phi = 128, 128
    s = solver(n_r, n_phi, 1.0, 200.0, 0.02, max_batch=3)
    try:
        sig = np.stack([random_sigma(n_r, n_phi, 500 + b) for b in range(3)])
        a_r, a_p = acceleration(s, sig)
        for b in range(3):
            _, rr, rp = oracle.ext_o1(n_r, n_phi, 1.0, 200.0, 0.02, 0, sig[b])
            check_acc(a_r[b], a_p[b], rr, rp, f"batch field {b}")
        # host in, host out
        h_r, h_p = np.empty_like(sig), np.empty_like(sig)
        pg.pg_set_density(s.h, sig, 3, pg.PG_MEM_HOST)
        pg.pg_acceleration(s.h, h_r, h_p, 3, pg.PG_MEM_HOST)
        assert np.array_equal(h_r, a_r) and np.array_equal(h_p, a_p)
        d = torch.from_numpy(sig).cuda(); o = torch.empty_like(d)
        pg.pg_set_density(s.h, d, 3, pg.PG_MEM_DEVICE)
        with pytest.raises(pg.PolargravError) as e:
            pg.pg_acceleration(s.h, o, o, 3, pg.PG_MEM_DEVICE)          # a_r and a_phi overlap
        assert e.value.status == pg.PG_ERR_INVALID_ARG
        with pytest.raises(pg.PolargravError) as e:
            pg.pg_acceleration(s.h, o, d, 3, pg.PG_MEM_DEVICE)          # output overlaps the density
        assert e.value.status == pg.PG_ERR_INVALID_ARG
        with pytest.raises(pg.PolargravError) as e:
            pg.pg_acceleration(s.h, o, torch.empty_like(d), 2, pg.PG_MEM_DEVICE)   # batch mismatch
        assert e.value.status == pg.PG_ERR_INVALID_ARG
    finally:
        s.close()


def test_total_self_force_vanishes_at_2048():
    """Newton's third law on the GPU result at the bench size (symmetric softening): sum m a = 0 in Cartesian
    components, to rounding, for the config-5 density."""
    c = CONFIGS[5]
    s = solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps)
    try:
        r, phi, area = s.grid()
        sig = make_sigma(5, r, phi)
        a_r, a_p = acceleration(s, sig)
        m = sig * area[:, None]
        fx = (m * (a_r * np.cos(phi)[None, :] - a_p * np.sin(phi)[None, :])).sum()
        fy = (m * (a_r * np.sin(phi)[None, :] + a_p * np.cos(phi)[None, :])).sum()
        scale = (m * np.hypot(a_r, a_p)).sum()
        assert abs(fx) < 1e-11 * scale and abs(fy) < 1e-11 * scale
    finally:
        s.close()


@pytest.mark.parametrize("soft", (pg.PG_SOFT_SYMMETRIC, pg.PG_SOFT_SOURCE))
def test_variants_sampled_rings_at_2048(soft):
    c = CONFIGS[5]
    s = solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps)
    try:
        r, phi, _ = s.grid()
        sig = make_sigma(5, r, phi)
        rings = np.array([0, 1, 700, 1024, 2046, 2047], dtype=np.int32)
        ref_phi, ref_r, ref_p = oracle.ext_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, soft, sig, rings)
        pg.pg_set_softening(s.h, soft)
        check_phi(potential(s, sig)[rings], ref_phi, f"config 5 soft {soft} potential")
        a_r, a_p = acceleration(s, sig)
        check_acc(a_r[rings], a_p[rings], ref_r, ref_p, f"config 5 soft {soft}")
    finally:
        s.close()

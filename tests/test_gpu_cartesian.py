"""Parity of the 3-D Cartesian mesh path (row NEXT-2 of SURVEY.md 8(f): the paper's own per-GPU workload,
PAPER.md:267, :271) against oracle/cartesian_oracle.c, element by element on seeded densities.
Bar: rel-L2 <= 1e-10, max pointwise relative <= 1e-9 (north_star's figures; Phi < 0 everywhere for rho >= 0)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2409_02294_b200 import binding as pg

pytestmark = pytest.mark.gpu


def make_rho(n, seed):
    """Synthetic mesh level in the spirit of the paper's runs (contents never described): a centrally
    condensed clump plus a few seeded Gaussian clumps plus 1 % noise; non-negative."""
    rng = np.random.Generator(np.random.PCG64(2409022940 + 1000 * n + seed))
    z, y, x = np.meshgrid(*(np.arange(n) + 0.5,) * 3, indexing="ij")
    c = n / 2.0
    r2 = (x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2
    rho = 1.0 / (1.0 + r2 / (0.1 * n) ** 2)
    for _ in range(6):
        cx, cy, cz = rng.uniform(0.2 * n, 0.8 * n, 3)
        w = rng.uniform(1.5, 4.0)
        rho += rng.uniform(0.5, 3.0) * np.exp(-((x - cx) ** 2 + (y - cy) ** 2 + (z - cz) ** 2) / (2 * w * w))
    return rho * (1.0 + 0.01 * rng.standard_normal(rho.shape))


class Dev3:
    def __init__(self, n, box):
        self.n = n
        self.h = pg.pg3_create(n, box, 0, torch.cuda.current_stream().cuda_stream)

    def solve(self, rho):
        d_r = torch.from_numpy(np.ascontiguousarray(rho)).cuda(); d_p = torch.empty_like(d_r)
        pg.pg3_set_density(self.h, d_r, pg.PG_MEM_DEVICE)
        pg.pg3_potential(self.h, d_p, pg.PG_MEM_DEVICE)
        pg.pg3_synchronize(self.h)
        return d_p.cpu().numpy()

    def close(self):
        pg.pg3_destroy(self.h)


def check(got, ref, what):
    l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got / ref - 1.0).max()
    assert l2 <= 1e-10 and mx <= 1e-9, f"{what}: rel-L2 {l2:.3e}, max rel {mx:.3e}"


def test_cartesian_32_every_cell():
    n, box = 32, 4.0
    d = Dev3(n, box)
    try:
        rho = make_rho(n, 0)
        check(d.solve(rho), oracle.cart_potential(n, box, rho), "32^3 every cell")
    finally:
        d.close()


@pytest.mark.parametrize("n,n_targets", [(64, 2048), (128, 512), (256, 64)])
def test_cartesian_sampled_targets_at_the_papers_sizes(n, n_targets):
    box = 10.0
    d = Dev3(n, box)
    try:
        rho = make_rho(n, 1)
        got = d.solve(rho)
        assert np.isfinite(got).all() and (got < 0).all()
        rng = np.random.default_rng(n)
        corners = [0, n - 1, n * n - 1, n**3 - 1, (n // 2) * (n * n + n + 1)]
        tg = np.unique(np.concatenate([corners, rng.integers(0, n**3, n_targets)])).astype(np.int64)
        ref = oracle.cart_potential_targets(n, box, rho, tg)
        check(got.reshape(-1)[tg], ref, f"{n}^3 on {len(tg)} sampled cells")
    finally:
        d.close()


def test_cartesian_single_cell_no_wraparound_and_self_term():
    """A unit cell in a corner: Phi = -h^3 / distance everywhere (no periodic image leaks in through the padding),
    -h^2 S in the cell itself."""
    n, box = 64, 64.0
    d = Dev3(n, box)
    try:
        for pos in ((0, 0, 0), (n - 1, n - 1, n - 1), (n - 1, 0, n // 2)):
            rho = np.zeros((n, n, n)); rho[pos] = 1.0
            got = d.solve(rho)
            z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
            dist = np.sqrt((z - pos[0]) ** 2.0 + (y - pos[1]) ** 2.0 + (x - pos[2]) ** 2.0)
            with np.errstate(divide="ignore"):
                expect = -1.0 / dist
            expect[pos] = -(3 * np.log(2 + np.sqrt(3)) - np.pi / 2)
            # FFT rounding is uniform in absolute terms: bound the error by the field's scale
            assert np.abs(got - expect).max() <= 1e-13 * np.abs(expect).max(), pos
            assert np.abs(got / expect - 1.0).max() <= 1e-9, pos
    finally:
        d.close()


def test_cartesian_memspaces_repeatability_and_errors():
    n, box = 32, 2.0
    d = Dev3(n, box)
    try:
        with pytest.raises(pg.PolargravError) as e:
            pg.pg3_potential(d.h, np.empty((n, n, n)), pg.PG_MEM_HOST)          # before any density
        assert e.value.status == pg.PG_ERR_STATE
        rho = make_rho(n, 2)
        dev = d.solve(rho)
        assert np.array_equal(d.solve(rho), dev)                                 # bitwise repeatable
        out = np.empty_like(rho)
        pg.pg3_set_density(d.h, rho, pg.PG_MEM_HOST)
        pg.pg3_potential(d.h, out, pg.PG_MEM_HOST)
        assert np.array_equal(out, dev)
        t = torch.from_numpy(rho).cuda()
        pg.pg3_set_density(d.h, t, pg.PG_MEM_DEVICE)
        with pytest.raises(pg.PolargravError) as e:
            pg.pg3_potential(d.h, t, pg.PG_MEM_DEVICE)                           # in place
        assert e.value.status == pg.PG_ERR_INVALID_ARG
        # linearity with a negative weight
        other = make_rho(n, 3)
        lin = d.solve(0.5 * rho - 2.0 * other)
        assert np.abs(lin - (0.5 * dev - 2.0 * d.solve(other))).max() <= 1e-13 * np.abs(lin).max()
    finally:
        d.close()

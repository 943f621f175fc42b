"""Parity of the 3-D Cartesian mesh path (row NEXT-2 of SURVEY.md 8(f): the paper's own per-GPU workload,
PAPER.md:267, :271) against oracle/cartesian_oracle.c, element by element on seeded densities.
Bar: rel-L2 <= 1e-10, max pointwise relative <= 1e-9 (north_star's figures; Phi < 0 everywhere for rho >= 0)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2409_02294_b200 import binding as pg
from paper_2409_02294_b200.workloads import make_rho3 as make_rho

pytestmark = pytest.mark.gpu


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


def whole_lines(n):
    """Flat indices of the six whole lines along x, y and z through the corner cell (0, 0, 0) and through the centre
    cell: every x of a row, every y of a column, every z of a pillar -- all the tiles the transposing y pass
    (ycols_fwd / ycols_inv, runs of YM columns) and the row kernels cut a line into, first and last included."""
    a, c = np.arange(n), n // 2
    flat = lambda z, y, x: (z * n + y) * n + x
    return np.concatenate([flat(0, 0, a), flat(0, a, 0), flat(a, 0, 0), flat(c, c, a), flat(c, a, c), flat(a, c, c)])


@pytest.mark.slow
@pytest.mark.parametrize("n,n_targets", [(64, 2048), (128, 20000), (256, 2000)])
def test_cartesian_sampled_targets_at_the_papers_sizes(n, n_targets):
    """64^3 and 128^3 are the paper's sizes.  The oracle costs n^3 pair terms per target: 20 000 targets at
    128^3 and 2 000 at 256^3 are ~4e10 terms each (tens of seconds on the host cores)."""
    box = 10.0
    d = Dev3(n, box)
    try:
        rho = make_rho(n, 1)
        got = d.solve(rho)
        assert np.isfinite(got).all() and (got < 0).all()
        rng = np.random.default_rng(n)
        corners = [0, n - 1, n * n - 1, n**3 - 1, (n // 2) * (n * n + n + 1)]
        lines = whole_lines(n)
        tg = np.unique(np.concatenate([corners, lines, rng.integers(0, n**3, n_targets - len(lines))])).astype(np.int64)
        assert len(tg) >= 0.99 * n_targets
        ref = oracle.cart_potential_targets(n, box, rho, tg)
        check(got.reshape(-1)[tg], ref, f"{n}^3 on {len(tg)} sampled cells")
        ln = np.isin(tg, lines)
        check(got.reshape(-1)[tg[ln]], ref[ln], f"{n}^3 on the six whole lines")
    finally:
        d.close()


@pytest.mark.parametrize("n", [64, 128, 256])
def test_cartesian_single_cell_no_wraparound_and_self_term(n):
    """A unit cell in a corner, on a face, in the centre: Phi = -h^3 / distance on EVERY cell (no periodic image leaks in
    through the padding), -h^2 S in the cell itself.  The closed form costs numpy nothing, so the paper's 128^3
     and 256^3 are checked whole: an index slip in a tile of the transposing y pass cannot hide."""
    box = float(n)
    d = Dev3(n, box)
    try:
        a = np.arange(n, dtype=np.float64)
        for pos in ((0, 0, 0), (n - 1, n - 1, n - 1), (n - 1, 0, n // 2), (n // 2, n // 2, n // 2), (3, n // 2 + 1, n - 2)):
            rho = np.zeros((n, n, n)); rho[pos] = 1.0
            got = d.solve(rho)
            dist = np.sqrt(((a - pos[0]) ** 2)[:, None, None] + ((a - pos[1]) ** 2)[None, :, None] + ((a - pos[2]) ** 2)[None, None, :])
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

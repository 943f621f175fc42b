"""Pins of oracle/nested_oracle.py (NEXT-3: nested meshes, readings M1-M6 of DESIGN.md section 3).  The scheme is an
algorithm, so the pins fix every step against what mathematics fixes: restriction conserves mass, maps children to their parents and keeps linear fields linear,
prolongation reproduces linear functions exactly at the children's cell centres (the +-1/4 offsets), depth 1 is the
single-level oracle, a configuration with nothing outside the finest box has no exterior term, a far exterior point
mass arrives on the fine level as -M/d within the trilinear error bound, linearity, mirror symmetry, and the whole
scheme against a direct sum over the composite (leaf-cell) mass distribution."""
import numpy as np
import pytest

import oracle
from oracle import nested_oracle as no


def centres(n, box, level):
    """cell-centre coordinates of level `level` (M1): edge box / 2^level, common centre 0"""
    b = box / 2**level
    return -b / 2 + (np.arange(n) + 0.5) * (b / n)


def test_restriction_conserves_mass_and_maps_children_to_parents():
    n, box = 8, 2.0
    rng = np.random.default_rng(1)
    fine = rng.random((n, n, n))
    coarse = no.restrict(fine)
    hf, hc = box / n, 2 * box / n
    assert abs(coarse.sum() * hc**3 - fine.sum() * hf**3) < 1e-14 * fine.sum()
    # index mapping: child (i, j, k) lands in parent (i // 2, j // 2, k // 2), whose centre is the mean of its children's
    one = np.zeros((n, n, n)); one[5, 2, 7] = 8.0
    r = no.restrict(one)
    assert r[2, 1, 3] == 1.0 and r.sum() == 1.0
    xf = centres(n, box, 0)
    xc = xf.reshape(-1, 2).mean(axis=1)
    assert abs(xc[2] - 0.5 * (xf[4] + xf[5])) < 1e-15
    # a field that is linear in the coordinates restricts to the same linear function at the parents' centres
    lin = 1.0 + 2.0 * xf[:, None, None] - 3.0 * xf[None, :, None] + 0.5 * xf[None, None, :]
    assert np.abs(no.restrict(lin) - (1.0 + 2.0 * xc[:, None, None] - 3.0 * xc[None, :, None] + 0.5 * xc[None, None, :])).max() < 1e-14
    assert np.allclose(no.restrict(np.full((n, n, n), 3.25)), 3.25, rtol=0, atol=1e-15)


def test_absorb_puts_a_child_cell_into_its_parent():
    n, box = 8, 4.0
    fine = np.zeros((n, n, n)); fine[5, 2, 7] = 8.0
    coarse = no.absorb(np.full((n, n, n), 9.0), no.restrict(fine))
    q = n // 4
    assert coarse[q + 2, q + 1, q + 3] == 1.0             # mean of 8 children, one of them 8
    inner = coarse[q:3 * q, q:3 * q, q:3 * q]
    assert inner.sum() == 1.0                             # the rest of the central block was replaced by zeros
    assert (no.mask_centre(coarse)[q:3 * q, q:3 * q, q:3 * q] == 0).all()
    assert coarse.sum() - inner.sum() == 9.0 * (n**3 - (n // 2) ** 3)          # outside untouched
    # geometry: the parent's centre is half a child cell from the child's centre on every axis
    xc, xf = centres(n, box, 0), centres(n, box, 1)
    for parent, child in ((q + 2, 5), (q + 1, 2), (q + 3, 7)):
        assert abs(abs(xc[parent] - xf[child]) - box / 2 / n / 2) < 1e-15


def test_prolongation_reproduces_linear_functions_at_the_child_centres():
    n, box = 12, 3.0
    xc, xf = centres(n, box, 0), centres(n, box, 1)
    a, b, c, d = 0.7, -1.3, 2.1, 0.4
    coarse = a + b * xc[:, None, None] + c * xc[None, :, None] + d * xc[None, None, :]
    fine = no.prolong(no.pack_halo(coarse), n)
    expect = a + b * xf[:, None, None] + c * xf[None, :, None] + d * xf[None, None, :]
    assert np.abs(fine - expect).max() < 1e-14
    # and a product of linear factors (trilinear interpolation is exact for it too)
    coarse = (1 + xc[:, None, None]) * (2 - xc[None, :, None]) * (0.5 + xc[None, None, :])
    expect = (1 + xf[:, None, None]) * (2 - xf[None, :, None]) * (0.5 + xf[None, None, :])
    assert np.abs(no.prolong(no.pack_halo(coarse), n) - expect).max() < 1e-14


def test_depth_one_is_the_single_level_oracle():
    n, box = 8, 1.5
    rho = np.random.default_rng(2).random((n, n, n))
    phi, _ = no.nested_potential(n, box, [rho])
    assert np.array_equal(phi[0], oracle.cart_potential(n, box, rho))


def test_nothing_outside_the_finest_box_means_no_exterior_term():
    n, box = 8, 2.0
    rng = np.random.default_rng(3)
    fine = rng.random((n, n, n))
    junk = np.zeros((n, n, n)); q = n // 4
    junk[q:3 * q, q:3 * q, q:3 * q] = 77.0                # M2: what the caller put under the child is ignored
    phi, rho = no.nested_potential(n, box, [junk, fine])
    assert np.array_equal(phi[1], oracle.cart_potential(n, box / 2, fine))
    assert np.array_equal(phi[0], oracle.cart_potential(n, box, no.absorb(np.zeros((n, n, n)), no.restrict(fine))))
    # far from the blob the coarse level sees a point mass at the blob's centre of mass
    m = fine.sum() * (box / 2 / n) ** 3
    xf = centres(n, box, 1)
    com = [(fine * xf.reshape([-1 if a == ax else 1 for a in range(3)])).sum() / fine.sum() for ax in range(3)]
    xc = centres(n, box, 0)
    corner = np.array([xc[0], xc[0], xc[0]])
    d = np.linalg.norm(corner - np.array(com))
    assert abs(phi[0][0, 0, 0] / (-m / d) - 1) < 2e-2


def test_far_exterior_point_mass_reaches_the_fine_level_within_the_trilinear_bound():
    n, box = 32, 8.0
    h0 = box / n
    coarse = np.zeros((n, n, n)); coarse[16, 15, 1] = 5.0           # [z][y][x]: 7 cells outside the child box in x
    fine = np.zeros((n, n, n))
    phi, _ = no.nested_potential(n, box, [coarse, fine])
    xc, xf = centres(n, box, 0), centres(n, box, 1)
    m = 5.0 * h0**3
    src = np.array([xc[16], xc[15], xc[1]])
    dist = np.sqrt((xf[:, None, None] - src[0]) ** 2 + (xf[None, :, None] - src[1]) ** 2 + (xf[None, None, :] - src[2]) ** 2)
    exact = -m / dist
    rel = np.abs(phi[1] / exact - 1)
    bound = 0.75 * (h0 / dist.min()) ** 2                 # (h^2 / 8) sum_axes |f_aa| <= (3/4) (h/d)^2 |f|
    assert rel.max() < bound
    assert rel.max() > bound / 200                        # it IS an interpolation error (1/r is harmonic: the leading terms partly cancel)
    # an offset mistake in the prolongation would be far outside: a shift by 1/4 parent cell alone is h/(4 d) everywhere
    assert rel.max() < 0.25 * (0.25 * h0 / dist.max())


def test_linearity_and_mirror_symmetry():
    n, box = 8, 2.0
    rng = np.random.default_rng(4)
    a = [rng.random((n, n, n)) for _ in range(3)]
    b = [rng.random((n, n, n)) - 0.5 for _ in range(3)]
    pa, _ = no.nested_potential(n, box, a)
    pb, _ = no.nested_potential(n, box, b)
    pc, _ = no.nested_potential(n, box, [2.0 * x - 3.0 * y for x, y in zip(a, b)])
    for l in range(3):
        assert np.abs(pc[l] - (2.0 * pa[l] - 3.0 * pb[l])).max() < 1e-12 * np.abs(pa[l]).max()
    pm, _ = no.nested_potential(n, box, [x[:, :, ::-1] for x in a])
    for l in range(3):
        assert np.abs(pm[l] - pa[l][:, :, ::-1]).max() < 1e-13 * np.abs(pa[l]).max()


def test_against_the_direct_sum_over_the_composite_mass_distribution():
    """Depth 2, a centrally concentrated blob sampled on both levels: the nested potential on the fine level against
    the plain sum over the leaf cells as point masses (fine cells everywhere inside the child box, coarse cells outside
    it; the self term as in reading C3).  The scheme's own error -- exterior mass seen through a trilinear
    interpolation -- stays below 2 %; a dropped, doubled or sign-flipped exterior term would be tens of percent."""
    n, box = 16, 4.0
    xc, xf = centres(n, box, 0), centres(n, box, 1)
    blob = lambda x: np.exp(-(x[:, None, None] ** 2 + x[None, :, None] ** 2 + x[None, None, :] ** 2) / (2 * 0.9**2))
    coarse, fine = blob(xc) + 0.05, blob(xf) + 0.05
    phi, _ = no.nested_potential(n, box, [coarse, fine])
    h0, h1 = box / n, box / 2 / n
    q = n // 4
    leaf_mask = np.ones((n, n, n), bool); leaf_mask[q:3 * q, q:3 * q, q:3 * q] = False
    cz, cy, cx = np.meshgrid(xc, xc, xc, indexing="ij")
    src_pos = np.stack([cz[leaf_mask], cy[leaf_mask], cx[leaf_mask]], axis=1)
    src_m = coarse[leaf_mask] * h0**3
    fz, fy, fx = np.meshgrid(xf, xf, xf, indexing="ij")
    tgt = np.stack([fz.ravel(), fy.ravel(), fx.ravel()], axis=1)
    ext = np.zeros(len(tgt))
    for k in range(0, len(tgt), 512):
        d = np.linalg.norm(tgt[k:k + 512, None, :] - src_pos[None, :, :], axis=2)
        ext[k:k + 512] = -(src_m[None, :] / d).sum(axis=1)
    direct = oracle.cart_potential(n, box / 2, fine) + ext.reshape(n, n, n)
    rel = np.abs(phi[1] / direct - 1)
    assert rel.max() < 2e-2
    share = np.abs(ext).min() / np.abs(direct).max()
    assert share > 0.1                                    # the exterior term matters in this configuration


# ------------------------------------------------------------------ depth >= 3: the recursion of M4, E_(l+1) = P[out_l + E_l]
# ext[0] is zero, so the "+ E_l" inside the prolongation only acts from the third level on (the paper's hierarchy has
# four, Fig. 8).  Both tests below turn red when nested_potential prolongs out_l alone.

def _point_sources_potential(tgt_axes, src_pos, src_m):
    """-sum m / |x - x'| at the tensor grid of the three target axes ([z][y][x]); sources as point masses"""
    z, y, x = tgt_axes
    out = np.zeros((len(z), len(y), len(x)))
    for p, m in zip(src_pos, src_m):
        out -= m / np.sqrt((z[:, None, None] - p[0]) ** 2 + (y[None, :, None] - p[1]) ** 2 + (x[None, None, :] - p[2]) ** 2)
    return out


def test_far_point_mass_on_level_0_reaches_level_2_through_two_prolongations():
    """One massive cell on level 0 outside box_1, levels 1 and 2 empty: out_1 = 0, so everything level 2 sees comes
    through E_1 inside P[out_1 + E_1].  Phi_2 = -M/d within the bound of two trilinear interpolations; without the
    recursion term Phi_2 is identically zero."""
    n, box = 32, 8.0
    h0, h1 = box / n, box / 2 / n
    coarse = np.zeros((n, n, n)); coarse[16, 15, 1] = 5.0           # [z][y][x]: 7 cells outside box_1 in x
    empty = np.zeros((n, n, n))
    phi, _ = no.nested_potential(n, box, [coarse, empty, empty])
    x0, x1, x2 = centres(n, box, 0), centres(n, box, 1), centres(n, box, 2)
    m = 5.0 * h0**3
    src = np.array([x0[16], x0[15], x0[1]])
    d2 = np.sqrt((x2[:, None, None] - src[0]) ** 2 + (x2[None, :, None] - src[1]) ** 2 + (x2[None, None, :] - src[2]) ** 2)
    exact = -m / d2
    assert np.abs(phi[2]).min() > 0.5 * np.abs(exact).min()          # not zero: the recursion term is there
    rel = np.abs(phi[2] / exact - 1)
    # first interpolation (level 0 -> 1), only its values on the level-1 cells that level 2 reads, [n/4 - 1, 3n/4]:
    # |e1| <= (3/4) (h0/d)^2 |f| there (same bound as the depth-2 test); the second one is a convex combination of them
    # (weights >= 0, sum 1), so it passes max |e1| on and adds (3/4) (h1/d)^2 |f| of its own.
    q = n // 4
    x1h = x1[q - 1:3 * q + 1]
    d1 = np.sqrt((x1h[:, None, None] - src[0]) ** 2 + (x1h[None, :, None] - src[1]) ** 2 + (x1h[None, None, :] - src[2]) ** 2)
    e1_abs = (0.75 * (h0 / d1) ** 2 * m / d1).max()
    bound = e1_abs / np.abs(exact).min() + 0.75 * (h1 / d2.min()) ** 2
    assert rel.max() < bound
    assert bound < 0.02                                               # and the bound is tight enough to mean something
    # level 1 itself, for completeness: one interpolation
    d1f = np.sqrt((x1[:, None, None] - src[0]) ** 2 + (x1[None, :, None] - src[1]) ** 2 + (x1[None, None, :] - src[2]) ** 2)
    assert np.abs(phi[1] / (-m / d1f) - 1).max() < 0.75 * (h0 / d1f.min()) ** 2


def test_depth_three_against_the_direct_sum_over_the_composite_mass_distribution():
    """Depth 3.  Mass on level 0 only in its outermost layer of cells, on level 1 only in ITS outermost layer, a blob on
    level 2: every exterior source is many cells away from where its potential is interpolated, so the error of the
    scheme against the plain sum over the leaf cells is bounded by the trilinear bound source by source,
        |error of Phi_2| <= b0 |Phi_2 from level 0| + b1 |Phi_2 from level 1|     (all contributions have one sign),
    b0 for two interpolations (h0 then h1), b1 for one (h1).  The level-0 share of Phi_2 is > 10 % and many times that
    bar: prolonging out_1 without E_1 fails it."""
    n, box = 32, 8.0
    h = [box / 2**l / n for l in range(3)]
    x = [centres(n, box, l) for l in range(3)]
    rng = np.random.default_rng(31)
    shell = np.zeros((n, n, n), bool)
    shell[[0, -1], :, :] = True; shell[:, [0, -1], :] = True; shell[:, :, [0, -1]] = True
    rho0 = np.where(shell, 3.0 + rng.random((n, n, n)), 0.0)
    rho1 = np.where(shell, 1.0 + rng.random((n, n, n)), 0.0)
    g2 = np.exp(-(x[2][:, None, None] ** 2 + x[2][None, :, None] ** 2 + x[2][None, None, :] ** 2) / (2 * 0.3**2))
    rho2 = 2.0 * g2 + 0.05
    phi, _ = no.nested_potential(n, box, [rho0, rho1, rho2])

    def leaves(l, rho):
        zz, yy, xx = np.meshgrid(x[l], x[l], x[l], indexing="ij")
        return np.stack([zz[shell], yy[shell], xx[shell]], axis=1), rho[shell] * h[l] ** 3
    p0, m0 = leaves(0, rho0)
    p1, m1 = leaves(1, rho1)
    axes2 = (x[2], x[2], x[2])
    from0, from1 = _point_sources_potential(axes2, p0, m0), _point_sources_potential(axes2, p1, m1)
    own2 = oracle.cart_potential(n, box / 4, rho2)
    # the centre of level 1 is replaced by the means of level 2 (M2) and solved by level 2 itself; nothing else is inside
    direct = own2 + from0 + from1
    err = np.abs(phi[2] - direct)
    # distances: level-0 shell at |coordinate| >= box/2 - h0 on some axis; it is interpolated first onto the level-1 cells
    # level 2 reads (|coordinate| <= box/8 + 1.5 h1), then onto level 2 (|coordinate| <= box/8); the level-1 shell likewise
    d01 = (box / 2 - h[0]) - (box / 8 + 1.5 * h[1])
    d02 = (box / 2 - h[0]) - box / 8
    d12 = (box / 4 - h[1]) - box / 8
    # |f| at the level-1 cells read may exceed |f| at the level-2 target by at most the ratio of the distances
    b0 = 0.75 * (h[0] / d01) ** 2 * (d02 + np.sqrt(3) * box / 4) / d01 + 0.75 * (h[1] / d02) ** 2
    b1 = 0.75 * (h[1] / d12) ** 2
    bar = b0 * np.abs(from0) + b1 * np.abs(from1)
    assert (err < bar).all()
    assert (bar / np.abs(direct)).max() < 0.02                           # a bar of under 2 % of Phi_2 everywhere
    share0 = np.abs(from0) / np.abs(direct)
    print(f"err/bar max {(err / bar).max():.3f}  level-0 share min {share0.min():.3f}  from0/bar min {(np.abs(from0) / bar).min():.1f}")
    assert share0.min() > 0.10 and (np.abs(from0) / bar).min() > 10      # dropping E_1 inside P[...] is >= 10 bars off

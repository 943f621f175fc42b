"""Pins of oracle/cartesian_oracle.c (NEXT-2: one 3-D Cartesian mesh level, readings C1-C4 of DESIGN.md section 3):
the self constant against numerical quadrature, 50-digit brute force, single-cell closed form, linearity, the
symmetries of the cube, translation of a compact source, far field."""
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_self_constant_against_quadrature_and_closed_form():
    s_quad = float([l for l in open(os.path.join(GOLD, "cart_self_constant.txt")) if not l.startswith("#")][0])
    assert abs(oracle.cart_self_constant() / s_quad - 1.0) < 1e-14
    assert abs(s_quad - (3 * np.log(2 + np.sqrt(3)) - np.pi / 2)) < 1e-14        # 2.38007736...


@pytest.mark.parametrize("name", ["3", "4"])
def test_bruteforce_50_digits(name):
    path = os.path.join(GOLD, f"cart_{name}.txt")
    hdr = [l for l in open(path) if l.startswith("# n=")][0]
    n = int(hdr.split("n=")[1].split()[0]); box = float(hdr.split("box=")[1].split()[0]); seed = int(hdr.split("seed=")[1])
    gold = np.loadtxt(path)[:, 3].reshape(n, n, n)
    rho = np.random.Generator(np.random.PCG64(seed)).random((n, n, n))
    got = oracle.cart_potential(n, box, rho)
    assert np.abs(got / gold - 1.0).max() < 5e-15


def test_single_cell_closed_form_and_linearity():
    n, box = 12, 3.0
    h = box / n
    rho = np.zeros((n, n, n)); rho[4, 7, 2] = 2.5
    got = oracle.cart_potential(n, box, rho)
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    d = h * np.sqrt((z - 4.0) ** 2 + (y - 7.0) ** 2 + (x - 2.0) ** 2)
    with np.errstate(divide="ignore"):
        expect = -2.5 * h**3 / d
    expect[4, 7, 2] = -2.5 * h**2 * 2.380077363979553
    np.testing.assert_allclose(got, expect, rtol=2e-15)
    rng = np.random.default_rng(3)
    a, b = rng.random((n, n, n)), rng.random((n, n, n)) - 0.5
    pa, pb = oracle.cart_potential(n, box, a), oracle.cart_potential(n, box, b)
    pab = oracle.cart_potential(n, box, 0.5 * a - 2.0 * b)
    assert np.abs(pab - (0.5 * pa - 2.0 * pb)).max() < 1e-13 * np.abs(pab).max()


def test_cube_symmetries():
    n, box = 10, 1.0
    rho = np.random.default_rng(4).random((n, n, n))
    p = oracle.cart_potential(n, box, rho)
    for axes in ((1, 0, 2), (2, 1, 0), (0, 2, 1)):
        assert np.abs(oracle.cart_potential(n, box, rho.transpose(axes)) - p.transpose(axes)).max() < 1e-13 * np.abs(p).max()
    for ax in range(3):
        assert np.abs(oracle.cart_potential(n, box, np.flip(rho, ax)) - np.flip(p, ax)).max() < 1e-13 * np.abs(p).max()


def test_translation_of_a_compact_source_and_scaling():
    """Isolated boundary: moving a compact source by whole cells moves its potential with it (no images)."""
    n, box = 14, 7.0
    rng = np.random.default_rng(5)
    src = np.zeros((n, n, n)); src[2:5, 3:6, 1:4] = rng.random((3, 3, 3))
    p0 = oracle.cart_potential(n, box, src)
    shifted = np.roll(src, (4, 2, 6), axis=(0, 1, 2))           # stays inside the mesh, nothing wraps
    p1 = oracle.cart_potential(n, box, shifted)
    assert np.abs(p1[4:, 2:, 6:] - p0[: n - 4, : n - 2, : n - 6]).max() < 1e-14 * np.abs(p0).max()
    # box twice as large, same rho values: mass x 8, distances x 2 -> potential x 4
    assert np.abs(oracle.cart_potential(n, 2 * box, src) / (4 * p0) - 1.0).max() < 1e-14


def test_far_field_monopole():
    n, box = 24, 24.0
    rho = np.zeros((n, n, n)); rho[0:2, 0:2, 0:2] = 1.0          # 8 unit cells in one corner, centre of mass at (1,1,1)
    tg = np.array([(n - 1) * n * n + (n - 1) * n + (n - 1)])
    got = oracle.cart_potential_targets(n, box, rho, tg)[0]
    r = np.sqrt(3.0) * (n - 1 + 0.5 - 1.0)
    assert abs(got / (-8.0 / r) - 1.0) < 2e-3                     # quadrupole of the 2x2x2 block vanishes by symmetry

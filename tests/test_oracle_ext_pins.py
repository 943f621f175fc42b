"""Pins of oracle/polar_oracle_ext.c (NEXT-4 variants: softening readings N1, acceleration reading N2 of DESIGN.md
section 3) against things other than itself: 50-digit brute force summed in Cartesian components, the pinned
polar_oracle.c for the symmetric potential, field/source adjointness, single-cell closed forms, Newton's third
law, the gradient of the off-grid potential (source softening), far field, axisymmetry."""
import os

import numpy as np
import pytest

import oracle
from paper_2409_02294_b200.workloads import random_sigma

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SOFTS = (oracle.SOFT_SYMMETRIC, oracle.SOFT_FIELD, oracle.SOFT_SOURCE)


def load_gold(name, soft):
    path = os.path.join(GOLD, f"ext_{name}_soft{soft}.txt")
    hdr = [l for l in open(path) if l.startswith("# n_r=")][0]
    kv = dict(tok.split("=", 1) for tok in hdr[2:].split() if "=" in tok and not tok.startswith("sigma"))
    n_r, n_phi = int(kv["n_r"]), int(kv["n_phi"])
    seed = int(hdr.split("seed=")[1].split(")")[0])
    g = np.loadtxt(path)
    return (n_r, n_phi, float(kv["r_in"]), float(kv["r_out"]), float(kv["eps"]), seed,
            [g[:, k].reshape(n_r, n_phi) for k in (2, 3, 4)])


@pytest.mark.parametrize("name", ["4x6", "5x3"])
@pytest.mark.parametrize("soft", SOFTS)
def test_bruteforce_50_digits_cartesian(name, soft):
    n_r, n_phi, r_in, r_out, eps, seed, gold = load_gold(name, soft)
    sigma = random_sigma(n_r, n_phi, seed)
    for fn in (oracle.ext_o0, oracle.ext_o1):
        got = fn(n_r, n_phi, r_in, r_out, eps, soft, sigma)
        assert np.abs(got[0] / gold[0] - 1.0).max() < 5e-15, fn.__name__
        for k in (1, 2):      # components may pass through zero: error relative to the field's scale
            assert np.abs(got[k] - gold[k]).max() < 2e-14 * np.abs(gold[1]).max(), (fn.__name__, k)


def test_symmetric_mode_is_the_pinned_oracle():
    n_r, n_phi = 24, 20
    sigma = random_sigma(n_r, n_phi, 5)
    ref = oracle.potential_o0(n_r, n_phi, 1.0, 60.0, 0.02, sigma)
    got = oracle.ext_o0(n_r, n_phi, 1.0, 60.0, 0.02, 0, sigma)[0]
    assert np.abs(got / ref - 1.0).max() < 1e-15


@pytest.mark.parametrize("soft", SOFTS)
def test_ring_pair_form_equals_definition(soft):
    n_r, n_phi = 20, 16
    sigma = random_sigma(n_r, n_phi, 6)
    a = oracle.ext_o0(n_r, n_phi, 0.5, 40.0, 0.05, soft, sigma)
    b = oracle.ext_o1(n_r, n_phi, 0.5, 40.0, 0.05, soft, sigma)
    assert np.abs(b[0] / a[0] - 1.0).max() < 1e-13
    for k in (1, 2):
        assert np.abs(b[k] - a[k]).max() < 1e-13 * np.abs(a[1]).max()


def test_field_and_source_softening_are_adjoint():
    """sum Sigma1 dA Phi_field[Sigma2] = sum Sigma2 dA Phi_source[Sigma1]: the pair kernel of one is the transpose of
    the other's; each alone is NOT symmetric (the reciprocity pin P6 must fail for them)."""
    n_r, n_phi, r_in, r_out, eps = 18, 12, 1.0, 80.0, 0.3
    s1, s2 = random_sigma(n_r, n_phi, 7), random_sigma(n_r, n_phi, 8)
    _, _, area, _ = oracle.grid(n_r, n_phi, r_in, r_out)
    f2 = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, oracle.SOFT_FIELD, s2)[0]
    g1 = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, oracle.SOFT_SOURCE, s1)[0]
    a = (s1 * area[:, None] * f2).sum(); b = (s2 * area[:, None] * g1).sum()
    assert abs(a / b - 1.0) < 1e-13
    f1 = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, oracle.SOFT_FIELD, s1)[0]
    c = (s2 * area[:, None] * f1).sum()
    assert abs(a / c - 1.0) > 1e-4       # field softening alone is not reciprocal


@pytest.mark.parametrize("soft", SOFTS)
def test_single_cell_closed_form(soft):
    n_r, n_phi, r_in, r_out, eps = 16, 8, 1.0, 50.0, 0.1
    r, phi, area, _ = oracle.grid(n_r, n_phi, r_in, r_out)
    h = np.sqrt(area)
    for i0 in (0, 7, n_r - 1):
        j0 = 3
        s = np.zeros((n_r, n_phi)); s[i0, j0] = 1.0
        e2 = eps**2 * {0: h[:, None] * h[i0], 1: h[:, None] ** 2 * np.ones((1, 1)), 2: h[i0] ** 2 * np.ones((n_r, 1))}[soft]
        dphi = phi[None, :] - phi[j0]
        d2 = r[:, None] ** 2 + r[i0] ** 2 - 2 * r[:, None] * r[i0] * np.cos(dphi) + e2
        pot, ar, aphi = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, soft, s)
        np.testing.assert_allclose(pot, -area[i0] / np.sqrt(d2), rtol=2e-14)
        np.testing.assert_allclose(ar, -area[i0] * (r[:, None] - r[i0] * np.cos(dphi)) / d2**1.5, rtol=0, atol=3e-14 * np.abs(ar).max())
        np.testing.assert_allclose(aphi, -area[i0] * r[i0] * np.sin(dphi) / d2**1.5, rtol=0, atol=3e-14 * np.abs(ar).max())
        assert abs(pot[i0, j0] / (-h[i0] / eps) - 1.0) < 1e-14 and ar[i0, j0] == 0.0 and aphi[i0, j0] == 0.0


def test_newtons_third_law_symmetric_softening():
    """Pair forces cancel: the total force of the disk on itself vanishes (Cartesian sum of m a)."""
    n_r, n_phi, r_in, r_out, eps = 16, 16, 1.0, 30.0, 0.05
    sigma = random_sigma(n_r, n_phi, 9)
    r, phi, area, _ = oracle.grid(n_r, n_phi, r_in, r_out)
    _, ar, aphi = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, 0, sigma)
    m = sigma * area[:, None]
    fx = (m * (ar * np.cos(phi)[None, :] - aphi * np.sin(phi)[None, :])).sum()
    fy = (m * (ar * np.sin(phi)[None, :] + aphi * np.cos(phi)[None, :])).sum()
    scale = (m * np.hypot(ar, aphi)).sum()
    assert abs(fx) < 1e-13 * scale and abs(fy) < 1e-13 * scale
    # ... and it does not vanish when the softening length belongs to one member of the pair only
    _, ar1, ap1 = oracle.ext_o0(n_r, n_phi, r_in, r_out, 0.5, 1, sigma)
    fx1 = (m * (ar1 * np.cos(phi)[None, :] - ap1 * np.sin(phi)[None, :])).sum()
    assert abs(fx1) > 1e-8 * (m * np.hypot(ar1, ap1)).sum()


def test_source_softening_acceleration_is_minus_grad_phi():
    """With soft = 2 the softening length depends on the source only, so Phi(x) is an ordinary function of the field
    point and a = -grad Phi.  Central differences of the off-grid potential (typed here from N1) in r and phi."""
    n_r, n_phi, r_in, r_out, eps = 12, 10, 1.0, 20.0, 0.2
    sigma = random_sigma(n_r, n_phi, 10)
    r, phi, area, _ = oracle.grid(n_r, n_phi, r_in, r_out)
    xs = (r[:, None] * np.cos(phi)[None, :]).ravel(); ys = (r[:, None] * np.sin(phi)[None, :]).ravel()
    m = (sigma * area[:, None]).ravel(); e2 = np.repeat(eps**2 * area, n_phi)

    def pot(rr, pp):
        return -(m / np.sqrt((rr * np.cos(pp) - xs) ** 2 + (rr * np.sin(pp) - ys) ** 2 + e2)).sum()

    _, ar, aphi = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, oracle.SOFT_SOURCE, sigma)
    for (i, j) in ((0, 0), (5, 3), (11, 9), (7, 6)):
        hr, hp = 1e-5 * r[i], 1e-5
        g_r = -(pot(r[i] + hr, phi[j]) - pot(r[i] - hr, phi[j])) / (2 * hr)
        g_p = -(pot(r[i], phi[j] + hp) - pot(r[i], phi[j] - hp)) / (2 * hp * r[i])
        scale = np.hypot(ar[i, j], aphi[i, j])
        assert abs(ar[i, j] - g_r) < 2e-8 * scale and abs(aphi[i, j] - g_p) < 2e-8 * scale


@pytest.mark.parametrize("soft", SOFTS)
def test_far_field_and_axisymmetry(soft):
    n_r, n_phi, r_in, r_out, eps = 64, 32, 1.0, 100.0, 0.01
    r, phi, area, _ = oracle.grid(n_r, n_phi, r_in, r_out)
    s = np.zeros((n_r, n_phi)); s[0, :] = 1.0
    M, a = n_phi * area[0], r[0]
    pot, ar, aphi = oracle.ext_o0(n_r, n_phi, r_in, r_out, eps, soft, s)
    i = n_r - 1
    e2 = eps**2 * {0: np.sqrt(area[i] * area[0]), 1: area[i], 2: area[0]}[soft]
    # monopole + quadrupole of a ring, first order in the softening: M r / (r^2 + e2)^(3/2) (1 + 3 a^2 / 4 r^2)
    expect = -M / r[i] ** 2 * (1 + 0.75 * a**2 / r[i] ** 2) * (1 - 1.5 * e2 / r[i] ** 2)
    assert abs(ar[i, 0] / expect - 1.0) < 1e-6
    assert np.abs(aphi).max() < 1e-13 * np.abs(ar).max()
    assert (ar.max(axis=1) - ar.min(axis=1)).max() < 1e-13 * np.abs(ar).max()
    # roll in phi
    sig = random_sigma(n_r, n_phi, 12)
    p1 = oracle.ext_o1(n_r, n_phi, r_in, r_out, eps, soft, sig)
    p2 = oracle.ext_o1(n_r, n_phi, r_in, r_out, eps, soft, np.roll(sig, 5, axis=1))
    for k in range(3):
        assert np.abs(np.roll(p1[k], 5, axis=1) - p2[k]).max() < 1e-12 * np.abs(p1[k]).max()

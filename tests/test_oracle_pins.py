"""Pins of the CPU oracle against things other than itself.

The paper prints no formula or value for this path (PAPER.md:267 names the method only),
so the pins are closed forms, invariants, a library routine and 50-digit brute force.
Each pin is chosen so that a plausible slip in oracle/polar_oracle.c (dropped term, wrong
sign/index, midpoint instead of exact area, absolute instead of scale-free softening,
missing self term) fails at least one of them.
"""
import os

import numpy as np
import pytest
from scipy.special import ellipkm1

import oracle
from paper_2409_02294_b200.workloads import CONFIGS, make_sigma, random_sigma

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


# ---------------------------------------------------------------- P11: grid tables
@pytest.mark.parametrize("n_r,n_phi,r_in,r_out", [(64, 64, 1.0, 100.0), (7, 5, 0.3, 2.0), (256, 128, 1.0, 500.0)])
def test_p11_total_area_and_tables(n_r, n_phi, r_in, r_out):
    r, phi, area, edges = oracle.grid(n_r, n_phi, r_in, r_out)
    assert edges[0] == r_in and edges[-1] == r_out
    # exact annulus area (A1 edges + A2 exact sectors)
    assert abs(n_phi * area.sum() - np.pi * (r_out**2 - r_in**2)) <= 4e-15 * np.pi * r_out**2
    du = np.log(r_out / r_in) / n_r
    # geometric centres and the sinh form of the sector area
    np.testing.assert_allclose(r, r_in * np.exp((np.arange(n_r) + 0.5) * du), rtol=2e-15)
    np.testing.assert_allclose(area, r**2 * np.sinh(du) * 2 * np.pi / n_phi, rtol=1e-13)
    # the midpoint area r^2 du dphi is NOT what is used (differs by du^2/6)
    assert np.all(np.abs(area / (r**2 * du * 2 * np.pi / n_phi) - 1.0) > 0.1 * du**2 / 6)
    np.testing.assert_allclose(phi, (np.arange(n_phi) + 0.5) * 2 * np.pi / n_phi, rtol=1e-15)


# ---------------------------------------------------------------- P10: 50-digit brute force
@pytest.mark.parametrize("name", ["4x6", "8x8", "5x3"])
def test_p10_bruteforce_50_digits(name):
    path = os.path.join(GOLD, f"bruteforce_{name}.txt")
    hdr = [l for l in open(path) if l.startswith("# n_r=")][0]
    kv = dict(tok.split("=", 1) for tok in hdr[2:].split() if "=" in tok and not tok.startswith("sigma"))
    n_r, n_phi = int(kv["n_r"]), int(kv["n_phi"])
    r_in, r_out, eps = float(kv["r_in"]), float(kv["r_out"]), float(kv["eps"])
    seed = int(hdr.split("seed=")[1].split(")")[0])
    gold = np.loadtxt(path)[:, 2].reshape(n_r, n_phi)
    sigma = random_sigma(n_r, n_phi, seed)
    for fn in (oracle.potential_o0, oracle.potential_o1, oracle.potential_definition_numpy):
        got = fn(n_r, n_phi, r_in, r_out, eps, sigma)
        assert np.abs(got / gold - 1.0).max() < 5e-15, fn.__name__


# ---------------------------------------------------------------- O1 == O0 == numpy definition
def test_o1_equals_o0_config1_full():
    c = CONFIGS[1]
    r, phi, _, _ = oracle.grid(c.n_r, c.n_phi, c.r_in, c.r_out)
    s = make_sigma(1, r, phi)
    a = oracle.potential_o0(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, s)
    b = oracle.potential_o1(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, s)
    assert np.abs(b / a - 1.0).max() < 1e-13
    assert np.all(a < 0.0)


def test_o1_equals_o0_sampled_config2_and_3():
    for cfg, n_t in ((2, 512), (3, 128)):
        c = CONFIGS[cfg]
        r, phi, _, _ = oracle.grid(c.n_r, c.n_phi, c.r_in, c.r_out)
        s = make_sigma(cfg, r, phi)
        rng = np.random.default_rng(cfg)
        rings = np.unique(np.concatenate([[0, c.n_r - 1], rng.integers(0, c.n_r, 4)])).astype(np.int32)
        o1 = oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, s, rings)
        cols = rng.integers(0, c.n_phi, n_t // len(rings))
        tg = (rings[:, None].astype(np.int64) * c.n_phi + cols[None, :]).reshape(-1)
        o0 = oracle.potential_o0_targets(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, s, tg)
        assert np.abs(o1[:, cols].reshape(-1) / o0 - 1.0).max() < 1e-13


def test_numpy_definition_matches_c_small():
    s = random_sigma(12, 10, 5)
    a = oracle.potential_definition_numpy(12, 10, 1.0, 30.0, 0.02, s)
    b = oracle.potential_o0(12, 10, 1.0, 30.0, 0.02, s)
    assert rel(a, b) < 1e-13


# ---------------------------------------------------------------- P1-P3: symmetry / linearity
N, RI, RO, EPS = 32, 1.0, 50.0, 0.01


def test_p1_axisymmetric_density_gives_axisymmetric_potential():
    r, _, _, _ = oracle.grid(N, N, RI, RO)
    s = np.repeat(np.exp(-r / 7.0)[:, None], N, axis=1)
    for fn in (oracle.potential_o0, oracle.potential_o1):
        p = fn(N, N, RI, RO, EPS, s)
        spread = (p.max(axis=1) - p.min(axis=1)) / np.abs(p).max(axis=1)
        assert spread.max() < 1e-13


def test_p2_linearity_with_negative_weights():
    s1, s2 = random_sigma(N, N, 1), random_sigma(N, N, 2, signed=True)
    a, b = -1.75, 0.3
    for fn in (oracle.potential_o0, oracle.potential_o1):
        lhs = fn(N, N, RI, RO, EPS, a * s1 + b * s2)
        rhs = a * fn(N, N, RI, RO, EPS, s1) + b * fn(N, N, RI, RO, EPS, s2)
        assert rel(lhs, rhs) < 1e-13


def test_p3_roll_in_phi():
    s = random_sigma(N, N, 3)
    for fn in (oracle.potential_o0, oracle.potential_o1):
        p = fn(N, N, RI, RO, EPS, s)
        q = fn(N, N, RI, RO, EPS, np.roll(s, 5, axis=1))
        assert rel(q, np.roll(p, 5, axis=1)) < 1e-13


# ---------------------------------------------------------------- P4: single cell
@pytest.mark.parametrize("i0", [0, 1, N // 2, N - 1])
def test_p4_single_cell_response(i0):
    j0 = 3
    r, phi, area, _ = oracle.grid(N, N, RI, RO)
    s = np.zeros((N, N)); s[i0, j0] = 1.0
    h = np.sqrt(area)
    d2 = (r[:, None] - r[i0]) ** 2 + 4 * r[:, None] * r[i0] * np.sin(0.5 * (phi[None, :] - phi[j0])) ** 2 \
        + EPS**2 * h[:, None] * h[i0]
    expect = -area[i0] / np.sqrt(d2)
    for fn in (oracle.potential_o0, oracle.potential_o1):
        p = fn(N, N, RI, RO, EPS, s)
        assert np.abs(p / expect - 1.0).max() < 1e-13
        # self term present and equal to -h/eps (A4)
        assert abs(p[i0, j0] / (-h[i0] / EPS) - 1.0) < 1e-13
        # no radial wrap-around: response decays monotonically away from the source ring at phi_j0
        col = -p[:, j0]
        assert np.all(np.diff(col[i0:]) < 0) and np.all(np.diff(col[: i0 + 1]) > 0)


# ---------------------------------------------------------------- P5: scale covariance (A3)
def test_p5_scale_covariance():
    s = random_sigma(N, N, 4)
    lam = 3.7
    for fn in (oracle.potential_o0, oracle.potential_o1):
        p = fn(N, N, RI, RO, EPS, s)
        q = fn(N, N, lam * RI, lam * RO, EPS, s)
        assert rel(q, lam * p) < 1e-13


# ---------------------------------------------------------------- P6: reciprocity
def test_p6_reciprocity():
    s1, s2 = random_sigma(N, N, 6), random_sigma(N, N, 7)
    _, _, area, _ = oracle.grid(N, N, RI, RO)
    p1 = oracle.potential_o1(N, N, RI, RO, EPS, s1)
    p2 = oracle.potential_o1(N, N, RI, RO, EPS, s2)
    a = (s1 * area[:, None] * p2).sum()
    b = (s2 * area[:, None] * p1).sum()
    assert abs(a / b - 1.0) < 1e-12


# ---------------------------------------------------------------- P7: far field
def test_p7_far_field_monopole_plus_quadrupole():
    n = 64
    r, _, area, _ = oracle.grid(n, n, 1.0, 100.0)
    s = np.zeros((n, n)); s[0, :] = 1.0
    M, a = n * area[0], r[0]
    for fn in (oracle.potential_o0, oracle.potential_o1):
        p = fn(n, n, 1.0, 100.0, 0.01, s)
        far = p[-1, 0]
        mono = -M / r[-1]
        assert far < 0
        assert 1e-6 < abs(far / mono - 1.0) < 1e-4           # monopole alone is off by the quadrupole
        assert abs(far / (mono * (1 + a * a / (4 * r[-1] ** 2))) - 1.0) < 1e-7
        # falls off like 1/r in the outer rings
        slope = np.log(p[-1, 0] / p[-9, 0]) / np.log(r[-1] / r[-9])
        assert abs(slope + 1.0) < 1e-3


# ---------------------------------------------------------------- P8: elliptic-integral ring
@pytest.mark.parametrize("cfg_n,r_out,i0,kmin", [(64, 100.0, 20, 8), (256, 500.0, 100, 6)])
def test_p8_uniform_ring_vs_complete_elliptic_integral(cfg_n, r_out, i0, kmin):
    n = cfg_n
    eps = 0.01
    r, _, area, _ = oracle.grid(n, n, 1.0, r_out)
    s = np.zeros((n, n)); s[i0, :] = 1.0
    rings = np.array([i for i in range(n) if abs(i - i0) >= kmin], dtype=np.int32)
    p = oracle.potential_o1_rings(n, n, 1.0, r_out, eps, s, rings)
    a = r[i0]
    rr = r[rings]
    e2 = eps**2 * np.sqrt(area[rings] * area[i0])
    A = rr**2 + a**2 + e2
    B = 2 * rr * a
    one_minus_m = ((rr - a) ** 2 + e2) / (A + B)
    expect = -area[i0] * (n / (2 * np.pi)) * 4 * ellipkm1(one_minus_m) / np.sqrt(A + B)
    assert np.abs(p[:, 0] / expect - 1.0).max() < 1e-12
    # O0 on a few of those targets
    tg = rings[::7].astype(np.int64) * n + 5
    p0 = oracle.potential_o0_targets(n, n, 1.0, r_out, eps, s, tg)
    assert np.abs(p0 / expect[::7] - 1.0).max() < 1e-12


def test_p8_uniform_annulus_is_sum_of_rings():
    n, r_out, eps = 64, 100.0, 0.01
    r, _, area, _ = oracle.grid(n, n, 1.0, r_out)
    src = np.arange(10, 20)
    s = np.zeros((n, n)); s[src, :] = 2.5
    tgt = np.array([40, 50, 63], dtype=np.int32)
    p = oracle.potential_o1_rings(n, n, 1.0, r_out, eps, s, tgt)[:, 0]
    expect = np.zeros(len(tgt))
    for i0 in src:
        e2 = eps**2 * np.sqrt(area[tgt] * area[i0])
        A = r[tgt] ** 2 + r[i0] ** 2 + e2
        B = 2 * r[tgt] * r[i0]
        expect += -2.5 * area[i0] * (n / (2 * np.pi)) * 4 * ellipkm1(((r[tgt] - r[i0]) ** 2 + e2) / (A + B)) / np.sqrt(A + B)
    assert np.abs(p / expect - 1.0).max() < 1e-12

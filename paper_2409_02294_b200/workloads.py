"""Seeded synthetic surface-density fields for the five BASELINE.json configs.

This module serves both the CPU oracle (through tests/ and bench.py) and the CUDA
path.  It holds NONE of the method's arithmetic: cell-centre radii and azimuths are
passed in by the caller (from `oracle.grid` or from `pg_grid`), and the functions
below only evaluate a density recipe on them.  Recipe: SURVEY.md section 8(d) /
DESIGN.md section 4 (the paper itself names no dataset: its workloads are CM4NG
meshes of 64^3/128^3 cells whose contents are never described).
"""
from __future__ import annotations

import dataclasses
import numpy as np

SEED_BASE = 2409022940


@dataclasses.dataclass(frozen=True)
class Config:
    cfg: int            # 1..5, position in BASELINE.json "configs"
    n_r: int
    n_phi: int
    r_in: float
    r_out: float
    eps: float
    batch: int
    name: str


CONFIGS = {
    1: Config(1, 64, 64, 1.0, 100.0, 0.01, 1, "64x64 exp disk + 1% noise"),
    2: Config(2, 256, 256, 1.0, 500.0, 0.01, 1, "256x256 power-law disk + m=2,3 spirals"),
    3: Config(3, 512, 512, 1.0, 1000.0, 0.01, 1, "512x512 exp disk + 50 clumps"),
    4: Config(4, 1024, 1024, 1.0, 1000.0, 0.01, 8, "1024x1024 x8 exp disk * lognormal"),
    5: Config(5, 2048, 2048, 1.0, 2000.0, 0.01, 1, "2048x2048 exp disk + m=1..8 spirals + 200 clumps"),
}

_PITCH = np.deg2rad(15.0)


def _rng(cfg: int, b: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + cfg + 100 * b))


def _spiral(m, r, phi, r_in, phase):
    """cos(m [phi - phase - ln(r/r_in)/tan(pitch)]) -- logarithmic spiral, pitch 15 deg."""
    return np.cos(m * (phi[None, :] - phase - np.log(r / r_in)[:, None] / np.tan(_PITCH)))


def _clumps(rng, n_clumps, base_of_ring, n_r, n_phi):
    """Gaussian clumps in index space (separable, periodic in phi, truncated at 9 widths);
    amplitude relative to the local base density."""
    out = np.zeros((n_r, n_phi))
    for _ in range(n_clumps):
        ic = rng.uniform(0.0, n_r)
        jc = rng.uniform(0.0, n_phi)
        w = rng.uniform(2.0, 6.0)
        amp = rng.uniform(0.5, 5.0)
        half = int(np.ceil(9.0 * w))
        i0, i1 = max(0, int(ic) - half), min(n_r, int(ic) + half + 1)
        ii = np.arange(i0, i1, dtype=np.float64)
        jw = np.arange(int(jc) - half, int(jc) + half + 1)
        jw = jw[: n_phi] if jw.size > n_phi else jw
        gi = np.exp(-((ii - ic) ** 2) / (2.0 * w * w))
        gj = np.exp(-((jw.astype(np.float64) - jc) ** 2) / (2.0 * w * w))
        local = base_of_ring[min(int(ic), n_r - 1)]
        out[i0:i1, np.mod(jw, n_phi)] += (amp * local) * gi[:, None] * gj[None, :]
    return out


def make_sigma(cfg: int, r: np.ndarray, phi: np.ndarray, b: int = 0) -> np.ndarray:
    """Surface density [n_r][n_phi] (fp64, non-negative) of config `cfg`, batch element `b`.

    r: cell-centre radii [n_r]; phi: cell-centre azimuths [n_phi] (caller-supplied)."""
    c = CONFIGS[cfg]
    r = np.asarray(r, dtype=np.float64)
    phi = np.asarray(phi, dtype=np.float64)
    if r.shape != (c.n_r,) or phi.shape != (c.n_phi,):
        raise ValueError("grid tables do not match the config")
    rng = _rng(cfg, b)
    if cfg == 1:
        base = np.exp(-r / 10.0)
        s = base[:, None] * (1.0 + 0.01 * rng.standard_normal((c.n_r, c.n_phi)))
    elif cfg == 2:
        base = r ** -1.5
        ph = rng.uniform(0.0, 2.0 * np.pi, size=2)
        s = base[:, None] * (1.0 + 0.1 * _spiral(2, r, phi, c.r_in, ph[0])
                             + 0.1 * _spiral(3, r, phi, c.r_in, ph[1]))
    elif cfg == 3:
        base = np.exp(-r / 100.0)
        s = base[:, None] + _clumps(rng, 50, base, c.n_r, c.n_phi)
    elif cfg == 4:
        base = np.exp(-r / 100.0)
        s = base[:, None] * np.exp(0.3 * rng.standard_normal((c.n_r, c.n_phi)))
    elif cfg == 5:
        base = np.exp(-r / 200.0)
        ph = rng.uniform(0.0, 2.0 * np.pi, size=8)
        mod = np.ones((c.n_r, c.n_phi))
        for m in range(1, 9):
            mod += 0.05 * _spiral(m, r, phi, c.r_in, ph[m - 1])
        s = base[:, None] * mod + _clumps(rng, 200, base, c.n_r, c.n_phi)
    else:
        raise ValueError(f"unknown config {cfg}")
    s = np.ascontiguousarray(s, dtype=np.float64)
    assert (s >= 0.0).all()
    return s


def make_batch(cfg: int, r, phi) -> np.ndarray:
    """[batch][n_r][n_phi] for the config's batch size."""
    c = CONFIGS[cfg]
    return np.stack([make_sigma(cfg, r, phi, b) for b in range(c.batch)])


def random_sigma(n_r: int, n_phi: int, seed: int, signed: bool = False) -> np.ndarray:
    """Uniform random field for invariance tests (not one of the configs)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    s = rng.random((n_r, n_phi))
    return s - 0.5 if signed else s


def make_rho3(n: int, seed: int) -> np.ndarray:
    """Synthetic 3-D mesh level [z][y][x] in the spirit of the paper's runs, whose contents are never described
    (PAPER.md:271): a centrally condensed clump, six seeded Gaussian clumps, 1 % noise; non-negative.  The one generator
    for bench.py --cart / --nested and tests/test_gpu_cartesian.py (inputs only, none of the method's arithmetic)."""
    rng = np.random.Generator(np.random.PCG64(2409022940 + 1000 * n + seed))
    z, y, x = np.meshgrid(*(np.arange(n) + 0.5,) * 3, indexing="ij")
    c = n / 2.0
    rho = 1.0 / (1.0 + ((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2) / (0.1 * n) ** 2)
    for _ in range(6):
        cx, cy, cz = rng.uniform(0.2 * n, 0.8 * n, 3)
        w = rng.uniform(1.5, 4.0)
        rho += rng.uniform(0.5, 3.0) * np.exp(-((x - cx) ** 2 + (y - cy) ** 2 + (z - cz) ** 2) / (2 * w * w))
    return rho * (1.0 + 0.01 * rng.standard_normal(rho.shape))

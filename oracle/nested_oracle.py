"""nested_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Oracle for row NEXT-3 of SURVEY.md section 8(f): the paper's distributed scheme, "the convolution method for solving
potential fields on NESTED grids in three dimensions ... each nested mesh was allocated one GPU" (PAPER.md:267, :269,
Fig. 8 :306).  The method's reference ([13]) is not available and PAPER.md prints neither the coupling
between the levels nor a formula, so the scheme below is a stated reading (M1-M6 of DESIGN.md section 3); it is an
ALGORITHM (restriction and prolongation are approximations of the composite mass distribution), so this oracle
follows it step by step, in fp64 numpy, with the pinned single-level direct sum (cartesian_oracle.c,
oracle.cart_potential) as the per-level solve.  It shares nothing with paper_2409_02294_b200/.

  M1  depth D levels l = 0 .. D-1 with a common centre, n^3 cells each (n a multiple of 4), edge box_l = box_0 / 2^l,
      h_l = box_l / n: level l+1 covers exactly the central (n/2)^3 cells [n/4, 3n/4)^3 of level l, two cells per
      parent cell and axis.  Arrays [z][y][x].
  M2  fine -> coarse (restriction), from the finest level up: the central (n/2)^3 cells of rho_l are REPLACED by
      the mean of their 2 x 2 x 2 children in rho_(l+1) (mass conserving); what the caller put there is ignored.
  M3  every level solves its own mesh with the isolated single-level convolution of NEXT-2 (readings C1-C4):
      own_l = Phi[rho_l], and, for l < D-1, out_l = Phi[rho_l with the central (n/2)^3 cells set to zero]:
      the potential, at level l's cell centres, of the level's mass OUTSIDE the next level's box.
  M4  E_l = potential, at level l's cell centres, of everything outside box_l:  E_0 = 0 (isolated),
      E_(l+1) = P[out_l + E_l].
  M5  coarse -> fine (prolongation) P: trilinear interpolation between the parent's cell centres.  Fine cell i sits at
      parent coordinate  n/4 + (2 i - 1)/4  (cell-centred, so +-1/4 of a parent cell off the parent centres): weights
      3/4 and 1/4 on the two nearest parents; the parents needed are the central cells plus ONE halo cell per side,
      [n/4 - 1, 3n/4]^3: (n/2 + 2)^3 values cross the level boundary.
  M6  Phi_l = own_l + E_l on every level.

Pins: tests/test_oracle_nested_pins.py.
"""
from __future__ import annotations

import numpy as np

from .polar_oracle import cart_potential


def restrict(rho_fine: np.ndarray) -> np.ndarray:
    """M2: mean of the 2 x 2 x 2 children: [n][n][n] -> [n/2][n/2][n/2]."""
    n = rho_fine.shape[0]
    out = np.zeros((n // 2, n // 2, n // 2))
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                out += rho_fine[dz::2, dy::2, dx::2]
    return out / 8.0


def absorb(rho_coarse: np.ndarray, child_mean: np.ndarray) -> np.ndarray:
    """M2: the central (n/2)^3 cells of the parent are replaced by the children's means."""
    n = rho_coarse.shape[0]
    q = n // 4
    out = rho_coarse.copy()
    out[q:3 * q, q:3 * q, q:3 * q] = child_mean
    return out


def mask_centre(rho: np.ndarray) -> np.ndarray:
    """M3: the level's mass outside the next level's box."""
    n = rho.shape[0]
    q = n // 4
    out = rho.copy()
    out[q:3 * q, q:3 * q, q:3 * q] = 0.0
    return out


def pack_halo(field: np.ndarray) -> np.ndarray:
    """M5: the parent values that cross the level boundary: cells [n/4 - 1, 3n/4] per axis, (n/2 + 2)^3."""
    n = field.shape[0]
    q = n // 4
    return field[q - 1:3 * q + 1, q - 1:3 * q + 1, q - 1:3 * q + 1].copy()


def prolong(halo: np.ndarray, n: int) -> np.ndarray:
    """M5: trilinear interpolation of the packed parent values onto the n^3 cell centres of the child.
    halo index J = parent index - (n/4 - 1).  Fine cell i = 2k: parents k-1 (1/4) and k (3/4) of the central block,
    i.e. halo J = k, k+1; fine cell i = 2k+1: parents k (3/4) and k+1 (1/4), halo J = k+1, k+2."""
    assert halo.shape == (n // 2 + 2,) * 3
    lo = np.empty(n, dtype=np.int64)
    w_lo = np.empty(n)
    for i in range(n):
        k = i // 2
        if i % 2 == 0:
            lo[i], w_lo[i] = k, 0.25
        else:
            lo[i], w_lo[i] = k + 1, 0.75
    out = np.zeros((n, n, n))
    for az in (0, 1):
        wz = w_lo if az == 0 else 1.0 - w_lo
        for ay in (0, 1):
            wy = w_lo if ay == 0 else 1.0 - w_lo
            for ax in (0, 1):
                wx = w_lo if ax == 0 else 1.0 - w_lo
                out += (wz[:, None, None] * wy[None, :, None] * wx[None, None, :]) * halo[np.ix_(lo + az, lo + ay, lo + ax)]
    return out


def nested_potential(n: int, box0: float, rhos):
    """M1-M6.  rhos: list of D arrays [n][n][n], level 0 (coarsest) first.  Returns the list of Phi_l and the
    restricted densities the levels actually solved."""
    depth = len(rhos)
    if n % 4 != 0:
        raise ValueError("n must be a multiple of 4")
    rho = [np.ascontiguousarray(r, dtype=np.float64).copy() for r in rhos]
    for l in range(depth - 2, -1, -1):                      # M2, finest first
        rho[l] = absorb(rho[l], restrict(rho[l + 1]))
    own = [cart_potential(n, box0 / 2**l, rho[l]) for l in range(depth)]                       # M3
    out = [cart_potential(n, box0 / 2**l, mask_centre(rho[l])) for l in range(depth - 1)]
    ext = [np.zeros((n, n, n))]                                                                 # M4
    for l in range(depth - 1):
        ext.append(prolong(pack_halo(out[l] + ext[l]), n))
    return [own[l] + ext[l] for l in range(depth)], rho                                        # M6

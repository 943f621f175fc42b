"""The definition written out in numpy -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A third, independent spelling of the sum in oracle/polar_oracle.c's header
(BASELINE.json north_star + readings A1-A5 of DESIGN.md section 3), with the
*naive* law-of-cosines distance r^2 + r'^2 - 2 r r' cos(phi - phi') exactly as
north_star prints it.  O(N^2) memory: tiny grids only.
"""
import numpy as np


def potential_definition_numpy(n_r, n_phi, r_in, r_out, eps, sigma):
    sigma = np.asarray(sigma, dtype=np.float64)
    edges = r_in * (r_out / r_in) ** (np.arange(n_r + 1) / n_r)          # A1
    r = np.sqrt(edges[:-1] * edges[1:])                                   # A1 geometric centre
    dphi = 2.0 * np.pi / n_phi
    phi = (np.arange(n_phi) + 0.5) * dphi                                 # A6
    area = 0.5 * (edges[1:] ** 2 - edges[:-1] ** 2) * dphi                # A2 exact sector
    h = np.sqrt(area)
    R, P = np.meshgrid(r, phi, indexing="ij")
    H = np.broadcast_to(h[:, None], R.shape)
    A = np.broadcast_to(area[:, None], R.shape)
    Rf, Pf, Hf, Af, Sf = (x.reshape(-1) for x in (R, P, H, A, sigma))
    d2 = (Rf[:, None] ** 2 + Rf[None, :] ** 2
          - 2.0 * Rf[:, None] * Rf[None, :] * np.cos(Pf[:, None] - Pf[None, :])
          + eps * eps * Hf[:, None] * Hf[None, :])                        # A3
    d2 = np.maximum(d2, 0.0)
    phi_out = -np.sum(Sf[None, :] * Af[None, :] / np.sqrt(d2), axis=1)    # A4 self term included, G=1 (A5)
    return phi_out.reshape(n_r, n_phi)

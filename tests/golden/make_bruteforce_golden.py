"""Writes tests/golden/bruteforce_*.txt: 50-digit brute-force potentials on tiny grids.

Calls neither oracle/ nor the CUDA path: only mpmath and the seeded input generator.
Definition: BASELINE.json north_star's sum with the *naive* law-of-cosines distance,
conventions A1-A5 of DESIGN.md section 3 (PAPER.md prints no formula; PAPER.md:267
only names the convolution method).  Run:  python tests/golden/make_bruteforce_golden.py
"""
import os
import sys

import mpmath as mp

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from paper_2409_02294_b200.workloads import random_sigma  # noqa: E402

mp.mp.dps = 50

CASES = [  # name, n_r, n_phi, r_in, r_out, eps, seed
    ("4x6", 4, 6, 1.0, 10.0, 0.01, 11),
    ("8x8", 8, 8, 0.5, 40.0, 0.05, 12),
    ("5x3", 5, 3, 2.0, 3.0, 0.3, 13),      # non power of two, thin annulus, large softening
]


def brute(n_r, n_phi, r_in, r_out, eps, sigma):
    r_in, r_out, eps = mp.mpf(r_in), mp.mpf(r_out), mp.mpf(eps)
    edges = [r_in * (r_out / r_in) ** (mp.mpf(i) / n_r) for i in range(n_r + 1)]
    r = [mp.sqrt(edges[i] * edges[i + 1]) for i in range(n_r)]
    dphi = 2 * mp.pi / n_phi
    phi = [(mp.mpf(j) + mp.mpf(1) / 2) * dphi for j in range(n_phi)]
    area = [(edges[i + 1] ** 2 - edges[i] ** 2) / 2 * dphi for i in range(n_r)]
    out = []
    for i in range(n_r):
        for j in range(n_phi):
            acc = mp.mpf(0)
            for ip in range(n_r):
                e2 = eps ** 2 * mp.sqrt(area[i]) * mp.sqrt(area[ip])
                for jp in range(n_phi):
                    d2 = r[i] ** 2 + r[ip] ** 2 - 2 * r[i] * r[ip] * mp.cos(phi[j] - phi[jp]) + e2
                    acc += mp.mpf(float(sigma[ip, jp])) * area[ip] / mp.sqrt(d2)
            out.append(-acc)
    return out


for name, n_r, n_phi, r_in, r_out, eps, seed in CASES:
    sigma = random_sigma(n_r, n_phi, seed)
    vals = brute(n_r, n_phi, r_in, r_out, eps, sigma)
    path = os.path.join(HERE, f"bruteforce_{name}.txt")
    with open(path, "w") as f:
        f.write("# 50-digit mpmath brute force of north_star's sum (naive cosine form), readings A1-A5;\n")
        f.write("# written by tests/golden/make_bruteforce_golden.py (calls neither oracle/ nor CUDA).\n")
        f.write(f"# n_r={n_r} n_phi={n_phi} r_in={r_in} r_out={r_out} eps={eps} "
                f"sigma=workloads.random_sigma(n_r,n_phi,seed={seed})\n")
        f.write("# columns: i j Phi_ij (25 significant digits)\n")
        for t, v in enumerate(vals):
            f.write(f"{t // n_phi} {t % n_phi} {mp.nstr(v, 25)}\n")
    print("wrote", path)

"""Writes tests/golden/ext_*.txt: 50-digit brute force of the NEXT-4 variants on tiny grids.

Potential with the three softening readings (N1) and the softened pair acceleration (N2) of DESIGN.md section 3
(not in the paper, PAPER.md:267 only names the convolution method).  Calls neither
oracle/ nor the CUDA path: only mpmath and the seeded input generator.  The acceleration is summed in CARTESIAN
components from the cell-centre positions and projected on the polar basis of the field point at the end, i.e.
by a route that shares nothing with the polar-component formula the oracle and the kernels use.
Run:  python tests/golden/make_ext_golden.py
"""
import os
import sys

import mpmath as mp

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from paper_2409_02294_b200.workloads import random_sigma  # noqa: E402

mp.mp.dps = 50

CASES = [  # name, n_r, n_phi, r_in, r_out, eps, seed
    ("4x6", 4, 6, 1.0, 10.0, 0.01, 21),
    ("5x3", 5, 3, 2.0, 3.0, 0.3, 22),
]


def brute(n_r, n_phi, r_in, r_out, eps, soft, sigma):
    r_in, r_out, eps = mp.mpf(r_in), mp.mpf(r_out), mp.mpf(eps)
    edges = [r_in * (r_out / r_in) ** (mp.mpf(i) / n_r) for i in range(n_r + 1)]
    r = [mp.sqrt(edges[i] * edges[i + 1]) for i in range(n_r)]
    dphi = 2 * mp.pi / n_phi
    phi = [(mp.mpf(j) + mp.mpf(1) / 2) * dphi for j in range(n_phi)]
    area = [(edges[i + 1] ** 2 - edges[i] ** 2) / 2 * dphi for i in range(n_r)]
    pos = [[(r[i] * mp.cos(phi[j]), r[i] * mp.sin(phi[j])) for j in range(n_phi)] for i in range(n_r)]
    out = []
    for i in range(n_r):
        for j in range(n_phi):
            x, y = pos[i][j]
            pot, ax, ay = mp.mpf(0), mp.mpf(0), mp.mpf(0)
            for ip in range(n_r):
                e2 = eps ** 2 * (area[i] if soft == 1 else area[ip] if soft == 2 else mp.sqrt(area[i]) * mp.sqrt(area[ip]))
                for jp in range(n_phi):
                    xs, ys = pos[ip][jp]
                    m = mp.mpf(float(sigma[ip, jp])) * area[ip]
                    d2 = (x - xs) ** 2 + (y - ys) ** 2 + e2
                    pot -= m / mp.sqrt(d2)
                    ax -= m * (x - xs) / d2 ** mp.mpf("1.5")
                    ay -= m * (y - ys) / d2 ** mp.mpf("1.5")
            a_r = ax * mp.cos(phi[j]) + ay * mp.sin(phi[j])
            a_phi = -ax * mp.sin(phi[j]) + ay * mp.cos(phi[j])
            out.append((pot, a_r, a_phi))
    return out


for name, n_r, n_phi, r_in, r_out, eps, seed in CASES:
    sigma = random_sigma(n_r, n_phi, seed)
    for soft in (0, 1, 2):
        vals = brute(n_r, n_phi, r_in, r_out, eps, soft, sigma)
        path = os.path.join(HERE, f"ext_{name}_soft{soft}.txt")
        with open(path, "w") as f:
            f.write("# 50-digit mpmath brute force: potential (reading N1) and softened pair acceleration (reading N2),\n")
            f.write("# Cartesian sums projected on the polar basis; written by tests/golden/make_ext_golden.py.\n")
            f.write(f"# n_r={n_r} n_phi={n_phi} r_in={r_in} r_out={r_out} eps={eps} soft={soft} "
                    f"sigma=workloads.random_sigma(n_r,n_phi,seed={seed})\n")
            f.write("# columns: i j Phi a_r a_phi (25 significant digits)\n")
            for t, (p, a, b) in enumerate(vals):
                f.write(f"{t // n_phi} {t % n_phi} {mp.nstr(p, 25)} {mp.nstr(a, 25)} {mp.nstr(b, 25)}\n")
        print("wrote", path)

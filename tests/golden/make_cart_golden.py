"""Writes tests/golden/cart_*.txt: 50-digit brute force of the 3-D Cartesian potential (NEXT-2) on tiny meshes.

Readings C1-C4 of DESIGN.md section 3 (PAPER.md:267 names the method only; the paper's ref. [13] is not available):
cells as point masses at their centres, the self term from the cube integral S = int_{unit cube} d^3x / |x|, isolated
boundary.  S is NOT taken from its closed form here: it is integrated numerically (one analytic step in z, two by
mpmath quadrature) and written to tests/golden/cart_self_constant.txt.  Calls neither oracle/ nor the CUDA path.
Run:  python tests/golden/make_cart_golden.py
"""
import os
import sys

import mpmath as mp
import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
mp.mp.dps = 30

# S = 8 * int_0^{1/2} int_0^{1/2} asinh( (1/2) / sqrt(x^2 + y^2) ) dx dy   (the z integral done analytically)
half = mp.mpf(1) / 2
S = 8 * mp.quad(lambda x, y: mp.asinh(half / mp.sqrt(x * x + y * y)), [0, half], [0, half])
with open(os.path.join(HERE, "cart_self_constant.txt"), "w") as f:
    f.write("# integral of 1/|x| over the unit cube centred on the origin, by mpmath quadrature (reading C3);\n")
    f.write("# written by tests/golden/make_cart_golden.py\n")
    f.write(mp.nstr(S, 20) + "\n")
print("S =", mp.nstr(S, 20))

CASES = [("3", 3, 1.5, 31), ("4", 4, 10.0, 32)]      # name, n, box, seed
mp.mp.dps = 50
for name, n, box, seed in CASES:
    rho = np.random.Generator(np.random.PCG64(seed)).random((n, n, n))
    h = mp.mpf(box) / n
    lines = []
    for z in range(n):
        for y in range(n):
            for x in range(n):
                acc = mp.mpf(0)
                for zp in range(n):
                    for yp in range(n):
                        for xp in range(n):
                            d2 = (x - xp) ** 2 + (y - yp) ** 2 + (z - zp) ** 2
                            g = 1 / (h * mp.sqrt(d2)) if d2 else S / h
                            acc += mp.mpf(float(rho[zp, yp, xp])) * h ** 3 * g
                lines.append(f"{z} {y} {x} {mp.nstr(-acc, 25)}")
    path = os.path.join(HERE, f"cart_{name}.txt")
    with open(path, "w") as f:
        f.write("# 50-digit mpmath brute force of the 3-D Cartesian potential, readings C1-C4;\n")
        f.write("# written by tests/golden/make_cart_golden.py (calls neither oracle/ nor CUDA).\n")
        f.write(f"# n={n} box={box} rho=numpy.random.Generator(PCG64({seed})).random((n,n,n)) seed={seed}\n")
        f.write("# columns: z y x Phi (25 significant digits)\n")
        f.write("\n".join(lines) + "\n")
    print("wrote", path)

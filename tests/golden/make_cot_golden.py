"""Writes tests/golden/cot_half_40digits.txt: cot((x+iy)/2) to 40 significant digits with mpmath.

Independent of oracle/ and of the CUDA path (mpmath only).  The quantity is the periodised Cauchy
kernel of Eq. (3.4):  PV sum_k 1/(zeta + 2 pi k - z) = (1/2) cot((zeta - z)/2).
The (x, y) list mixes generic arguments, near-singular ones (|w| down to 1e-6, the near-neighbour
regime of a fine grid), arguments close to the periodic images x = +-2 pi, and large |y|.
Inputs are written as C99 hex floats so that the test feeds bit-identical doubles.

    python tests/golden/make_cot_golden.py
"""
import os
import random

import mpmath as mp

mp.mp.dps = 60
rnd = random.Random(20210801)
pts = []
for _ in range(40):
    pts.append((rnd.uniform(-4 * mp.pi, 4 * mp.pi), rnd.uniform(-3.0, 3.0)))
for e in range(1, 7):
    r = 10.0 ** (-e)
    for _ in range(4):
        th = rnd.uniform(0, 2 * 3.141592653589793)
        pts.append((r * float(mp.cos(th)), r * float(mp.sin(th))))
for e in range(1, 6):
    r = 10.0 ** (-e)
    for sgn in (-1.0, 1.0):
        pts.append((sgn * 6.283185307179586 + r * rnd.uniform(-1, 1), r * rnd.uniform(-1, 1)))
        pts.append((sgn * 3.141592653589793 + r * rnd.uniform(-1, 1), rnd.uniform(-0.5, 0.5)))
for y in (-8.0, -5.0, 5.0, 8.0, -20.0, 20.0):
    pts.append((rnd.uniform(-6, 6), y))

out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cot_half_40digits.txt")
with open(out, "w") as f:
    f.write("# cot((x+iy)/2), 40 significant digits (mpmath, dps=60); Eq. (3.4) PAPER.md:L204\n")
    f.write("# x_hex y_hex re im\n")
    for x, y in pts:
        x = float(x)
        y = float(y)
        w = mp.mpc(mp.mpf(x), mp.mpf(y)) / 2
        c = mp.cos(w) / mp.sin(w)
        f.write("%s %s %s %s\n" % (x.hex(), y.hex(), mp.nstr(c.real, 40), mp.nstr(c.imag, 40)))
print("wrote", out, len(pts))

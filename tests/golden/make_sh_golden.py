"""Writes tests/golden/sh_basis.txt: real spherical harmonics (Condon-Shortley phase, index l*l+l+m) at fixed
directions from the associated-Legendre definition via scipy.special.lpmv.  Calls nothing under oracle/ or the
CUDA package.  Each row: x y z Y_0 .. Y_15.

Y_lm = N_lm P_l^|m|(cos th) * { sqrt2 cos(m ph) (m>0) ; 1 (m=0) ; sqrt2 sin(|m| ph) (m<0) },
N_lm = sqrt((2l+1)/(4 pi) (l-|m|)!/(l+|m|)!)  - the textbook real basis DESIGN.md reading R8 names.
"""
import math
import os
import numpy as np
from scipy.special import lpmv

dirs = np.array([[0.36, -0.48, 0.8], [-0.6, 0.0, -0.8], [2.0 / 7, 3.0 / 7, 6.0 / 7]])
rows = []
for d in dirs:
    d = d / np.linalg.norm(d)
    th, ph = math.acos(d[2]), math.atan2(d[1], d[0])
    Y = []
    for l in range(4):
        for m in range(-l, l + 1):
            am = abs(m)
            N = math.sqrt((2 * l + 1) / (4 * math.pi) * math.factorial(l - am) / math.factorial(l + am))
            P = lpmv(am, l, math.cos(th))
            Y.append(N * P * (math.sqrt(2) * math.cos(m * ph) if m > 0 else (1.0 if m == 0 else math.sqrt(2) * math.sin(am * ph))))
    rows.append(np.concatenate([d, Y]))
np.savetxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "sh_basis.txt"), np.array(rows), fmt="%.17g",
           header="x y z Y0..Y15 ; real SH with Condon-Shortley phase, index l*l+l+m (DESIGN.md R8); written by make_sh_golden.py")

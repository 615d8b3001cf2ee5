"""Writes tests/golden/clean_M20_channel_counts.txt: energies and the integer number of open
subbands of the clean M=20 armchair ribbon.

Source of the values: PAPER.md:82 ("a step-like dependence with the conductance being a
multiple of 2e^2/h" for the ideal ribbon) fixes that T is an integer; WHICH integer is the
count of subbands p = 1..M/2 with |1 - 2c_p| < |E/t| < 1 + 2c_p, c_p = cos(p pi/(M+1))
(armchair dimer-chain dispersion E^2 = t^2 (1 + 4c_p^2 + 4c_p cos k), BASELINE.json:north_star).
Uses neither oracle/ nor the CUDA path.  Run: python tests/golden/make_channel_counts.py
"""
import os

import numpy as np

M, t = 20, -2.7
energies = np.linspace(-2.7, 2.7, 64)   # BASELINE.json:configs[0] grid
rows = []
for E in energies:
    x = abs(E / t)
    n = sum(1 for p in range(1, M // 2 + 1)
            if abs(1 - 2 * np.cos(p * np.pi / (M + 1))) < x < 1 + 2 * np.cos(p * np.pi / (M + 1)))
    rows.append((E, n))
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "clean_M20_channel_counts.txt")
with open(out, "w") as f:
    f.write("# E[eV]  N_open  -- clean armchair ribbon M=20, t=-2.7 eV; PAPER.md:82 integer steps;\n")
    f.write("# written by tests/golden/make_channel_counts.py (closed-form subband count)\n")
    for E, n in rows:
        f.write("%.17g %d\n" % (E, n))
print(out)

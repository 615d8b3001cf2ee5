"""Writes tests/golden/near_neutrality_ld.txt: T(E) of the near-charge-neutrality cases in 80-bit arithmetic.

Why this file exists.  Close to E = 0 the oracle's own Sancho-Rubio decimation loses digits: E = 0 is an eigenvalue of the
isolated lead cell for every M, and the decimation's inverse (z - eps)^-1 amplifies rounding by ~(t / E)^2 (DESIGN.md
section 2, note 1).  Measured against the values below, oracle/rgf_oracle.c is off by 3e-8 at |E| = 1e-5 eV and 2e-9 at
1e-4 eV on the disordered M = 128 ribbons -- more than the tolerance 1e-9 it is meant to referee.  The GPU tests therefore
compare with the oracle where the oracle is good (|E| >= 1e-3 eV) and with these values below that.

What it computes: Eq. 1 + Eq. 2 of the paper by the slice recursion of BASELINE.json:north_star
(G_ii = (z - H_i - V G V)^-1, G_i0 = G_ii V G_{i-1,0}) on full M x M slices in numpy longdouble (x87 80-bit, eps = 5e-20)
with its own Gauss-Jordan inverse.  The lead self-energies are the exact surface Green's function of the clean lead: in
the transverse sine basis the armchair lead is M/2 chains with alternating hoppings 2 t cos(p pi / (M+1)), t, whose end-site
Green's function is the stable root of a quadratic (no iteration, no resonance).  Calls neither oracle/ nor the CUDA path;
tests/test_oracle_pins.py pins it to the oracle away from E = 0 and to the closed-form T of the clean ribbon.

    python tests/golden/make_near_neutrality_ld.py [case ...]      (minutes per disordered case)
    python tests/golden/make_near_neutrality_ld.py --config3 IDX [IDX ...]
        the same evaluation for energies of the disordered configs[3] ribbon (M = 244, L = 2000; 35 minutes per energy),
        appended to tests/golden/config3_ld.txt: the referee for the half-slice formulation's guard at resonant energies
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from paper_1107_5300_b200 import inputs       # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
LD, CLD = np.longdouble, np.clongdouble
PI = LD("3.14159265358979323846264338327950288")


def inv_ld(A):
    """Gauss-Jordan inverse with partial pivoting in long double."""
    n = A.shape[0]
    A = A.astype(CLD).copy()
    B = np.eye(n, dtype=CLD)
    for k in range(n):
        p = k + int(np.argmax(np.abs(A[k:, k])))
        if p != k:
            A[[k, p]] = A[[p, k]]
            B[[k, p]] = B[[p, k]]
        d = CLD(1) / A[k, k]
        A[k] *= d
        B[k] *= d
        f = A[:, k].copy()
        f[k] = 0
        A -= f[:, None] * A[k][None, :]
        B -= f[:, None] * B[k][None, :]
    return B


def chain_surface(z, h1, h2):
    """End-site Green's function of the semi-infinite chain with hoppings h1, h2, h1, ...: G = 1 / (z - h1^2 / (z - h2^2 G))."""
    if h1 == 0:
        return 1 / z
    Bq = z * z - h1 * h1 + h2 * h2
    D = (z - h1 - h2) * (z + h1 + h2) * (z - h1 + h2) * (z + h1 - h2)
    s = np.sqrt(D)
    best, bd = None, None
    for sg in (1, -1):
        G = 2 * z / (Bq + sg * s)
        d = abs(G * h1 * h2 / (z - h2 * h2 * G)) ** 2         # |f'(G)|: the retarded root is the attractive fixed point
        if bd is None or d < bd:
            best, bd = G, d
    return best


def lead_surface(M, t, z, qc):
    """Surface Green's function of the clean lead on the atoms j = 2r + qc of its surface slice (those bonded to the device)."""
    nc = (M - qc + 1) // 2
    j = (2 * np.arange(nc) + qc + 1).astype(LD)
    cols, G0 = [], []
    for p in range(1, M // 2 + 1):
        th = LD(p) * PI / LD(M + 1)
        cols.append(LD(2) / np.sqrt(LD(M + 1)) * np.sin(th * j))
        G0.append(chain_surface(z, LD(2) * t * np.cos(th), t))
    if M % 2 == 1 and qc == 0:
        cols.append(np.sqrt(LD(2) / LD(M + 1)) * np.sin(PI / 2 * j))
        G0.append(1 / z)
    Q = np.array(cols, dtype=LD).T.astype(CLD)
    return (Q * np.array(G0, dtype=CLD)[None, :]) @ Q.T


def transmission_ld(onsite, vac, t, E, eta):
    L, M = onsite.shape
    t = LD(t)
    z = CLD(LD(E) + 1j * LD(eta))
    isv = np.zeros((L, M), bool) if vac is None else vac.astype(bool)
    j = np.arange(M)

    def sigma(qc, alive):
        g = lead_surface(M, t, z, qc)
        S = np.zeros((M, M), CLD)
        idx = 2 * np.arange(g.shape[0]) + qc
        S[np.ix_(idx, idx)] = t * t * g
        a = alive.astype(LD)
        return a[:, None] * S * a[None, :]

    SL, SR = sigma(1, ~isv[0]), sigma((L - 1) & 1, ~isv[L - 1])
    g = P = m = None
    for i in range(L):
        A = np.zeros((M, M), CLD)
        A[j, j] = z - onsite[i].astype(LD)
        al = (~isv[i, :-1] & ~isv[i, 1:])
        A[j[:-1], j[:-1] + 1] = -t * al
        A[j[:-1] + 1, j[:-1]] = -t * al
        if i == 0:
            A = A - SL
        else:
            m = (t * ((((i - 1) + j) % 2 == 0) & ~isv[i - 1] & ~isv[i])).astype(CLD)
            A = A - m[:, None] * g * m[None, :]
        if i == L - 1:
            A = A - SR
        g = inv_ld(A)
        P = g[:, 1::2].copy() if i == 0 else (g * m[None, :]) @ P
    GL = (1j * (SL - SL.conj().T))[1::2, 1::2]
    GR = 1j * (SR - SR.conj().T)
    return float(np.trace(GL @ (P.conj().T @ GR @ P)).real)


def main_config3(indices):
    w = inputs.config3(disordered=True)
    out = os.path.join(HERE, "config3_ld.txt")
    if not os.path.exists(out):
        with open(out, "w") as f:
            f.write("# T(E) of the disordered configs[3] ribbon (M=244 L=2000 W=0.1 seed 5301) in 80-bit arithmetic, written by\n"
                    "# tests/golden/make_near_neutrality_ld.py --config3 (numpy %s); t=-2.7 eV eta=1e-9 eV\n# columns: energy_index E[eV] T\n" % np.__version__)
    for k in indices:
        T = transmission_ld(w.onsite[0], None, w.t, w.energies[k], w.eta)
        with open(out, "a") as f:
            f.write("%d %.17g %.17g\n" % (k, w.energies[k], T))
        print(k, w.energies[k], T, flush=True)


def main():
    if len(sys.argv) > 1 and sys.argv[1] == "--config3":
        return main_config3([int(x) for x in sys.argv[2:]])
    cases = sys.argv[1:] or list(inputs.NEAR_NEUTRALITY_CASES)
    out = os.path.join(HERE, "near_neutrality_ld.txt")
    old = {}
    if os.path.exists(out):
        for line in open(out):
            if not line.startswith("#"):
                c, k, e, tv = line.split()
                old[(c, int(k))] = (e, tv)
    for c in cases:
        w = inputs.near_neutrality(c)
        vac = None if w.vacancy is None else w.vacancy[0]
        for k, e in enumerate(w.energies):
            old[(c, k)] = ("%.17g" % e, "%.17g" % transmission_ld(w.onsite[0], vac, w.t, e, w.eta))
            print(c, k, old[(c, k)], flush=True)
    with open(out, "w") as f:
        f.write("# T(E) in 80-bit arithmetic, written by tests/golden/make_near_neutrality_ld.py (numpy %s, longdouble eps %.1e)\n" % (np.__version__, np.finfo(LD).eps))
        f.write("# cases: paper_1107_5300_b200/inputs.py near_neutrality(); t=-2.7 eV eta=1e-9 eV\n# columns: case energy_index E[eV] T\n")
        for c in inputs.NEAR_NEUTRALITY_CASES:
            for k in range(8):
                if (c, k) in old:
                    f.write("%s %d %s %s\n" % (c, k, old[(c, k)][0], old[(c, k)][1]))


if __name__ == "__main__":
    main()

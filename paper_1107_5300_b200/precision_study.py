"""configs[3] precision study (BASELINE.json:configs[3]; "single vs double precision").

Runs the M = 244, L = 2000 ribbon (clean and the seeded +-0.1 eV disorder variant) over the 1024 energies of
configs[3] in complex128 and in complex64 through the C ABI and reports |T_c64 - T_c128| versus E: the
maximum per energy window and the growth towards charge neutrality that north_star asks to be reported.
Marshalling and a table only -- every number comes from the CUDA library.

    python -m paper_1107_5300_b200.precision_study [--L 2000] [--out profiles/precision_r02_config3.md]
"""
import argparse
import sys
import time

import numpy as np

from . import binding as rgf
from . import inputs

def edge_distance(M, E, t):
    """Distance of |E| to the nearest subband edge |t| |1 - 2 c_p|, |t| (1 + 2 c_p) of the clean ribbon (R6): T(E) of
    the clean ribbon is discontinuous there, so an energy within 1e-4 eV of an edge is left out of the bound (reading Q8)."""
    c = np.cos(np.arange(1, M // 2 + 1) * np.pi / (M + 1))
    edges = np.abs(t) * np.concatenate([np.abs(1 - 2 * c), 1 + 2 * c])
    return np.min(np.abs(edges[None, :] - np.abs(np.asarray(E))[:, None]), axis=1)


WINDOWS = [(0.0, 0.02), (0.02, 0.05), (0.05, 0.1), (0.1, 0.2), (0.2, 0.5), (0.5, 1.0001)]


def run(L):
    rows = []
    with rgf.Plan(0) as p:
        for disordered in (False, True):
            w = inputs.config3(L=L, disordered=disordered)
            p.set_device(w.onsite, w.t)
            t0 = time.time(); T128 = p.transmission(w.energies, w.eta)[0]; t128 = time.time() - t0
            t0 = time.time(); T64 = p.transmission(w.energies, w.eta, precision=rgf.RGF_C64, ok=(rgf.RGF_ESINGULAR,))[0]; t64 = time.time() - t0
            rows.append((w, T128, T64, t128, t64))
    return rows


def report(rows, out):
    pr = lambda s="": print(s, file=out)
    pr("# configs[3] precision study: |T_c64 - T_c128| versus E (M = 244, sweep in complex64 vs complex128)")
    pr()
    pr("Command: `python -m paper_1107_5300_b200.precision_study` (one B200, through the C ABI).  Leads in complex128 in")
    pr("both runs (reading R13); t = -2.7 eV, eta = 1e-9 eV; 1024 energies = linspace(-1, 1, 512) ++ linspace(-0.05, 0.05, 512).")
    pr("Lowest subband edges of M = 244: 0.0200, 0.0399, 0.0803, 0.0993 eV (|E| < 0.02 eV is the gap).")
    pr()
    for w, T128, T64, t128, t64 in rows:
        bad = ~np.isfinite(T64)          # single-precision overflow: reported by the library as RGF_ESINGULAR + NaN
        d = np.abs(np.where(bad, 0.0, T64) - T128)
        aE = np.abs(w.energies)
        pr("## %s  (c128 %.1f s, c64 %.1f s incl. leads)" % (w.name, t128, t64))
        pr()
        pr("| window of abs(E) [eV] | energies | c64 non-finite | max T_c128 | max abs dT | median abs dT | max abs dT / max(1e-12, T) |")
        pr("|---|---|---|---|---|---|---|")
        for lo, hi in WINDOWS:
            m = (aE >= lo) & (aE < hi)
            if not m.any():
                continue
            rel = d[m] / np.maximum(1e-12, np.abs(T128[m]))
            pr("| [%.2f, %.2f) | %d | %d | %.3f | %.2e | %.2e | %.2e |" % (lo, min(hi, 1.0), m.sum(), (bad & m).sum(), T128[m].max(), d[m].max(), np.median(d[m]), rel.max()))
        outside = aE >= 0.1
        if not w.notes.get("W"):          # clean variant: steps of T(E) at the subband edges
            near = edge_distance(w.M, w.energies, w.t) < 1e-4
            pr()
            pr("%d energies lie within 1e-4 eV of a subband edge (T(E) jumps there; reading Q8) and are left out of the bound: " % near.sum()
               + ", ".join("E = %+.5f dT = %.1e" % (w.energies[k], d[k]) for k in np.where(near & outside)[0]))
            outside &= ~near
        pr()
        pr("north_star bound |dT| <= 1e-3 outside |E| < 0.1 eV: max = %.2e -> %s" % (d[outside].max(), "holds" if d[outside].max() <= 1e-3 else "VIOLATED"))
        worst = np.argsort(-d)[:5]
        pr("largest differences: " + ", ".join("E = %+.5f: T128 = %.6f, dT = %.2e" % (w.energies[k], T128[k], d[k]) for k in worst))
        pr()
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=2000)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    rows = run(a.L)
    if a.out:
        with open(a.out, "w") as f:
            report(rows, f)
    report(rows, sys.stdout)


if __name__ == "__main__":
    main()

"""Oracle-side reproduction of the paper's single-precision finding (SURVEY.md 8(c) "Precision finding").

TEST / REPORT INFRASTRUCTURE: runs ONLY the CPU oracle.  For the configs[3] ribbon (M = 244, L = 2000; clean and the seeded
+-0.1 eV variant) it evaluates T(E) by the paper's own form of Eq. 4, G_jj = (1 - G0 V G V)^-1 G0, in IEEE single precision
(orc_transmission_eq4_batch, use_float = 1) and compares with the double-precision direct form (orc_transmission_batch).
The CUDA library's complex64 sweep uses the direct form (BASELINE.json north_star); its curve is
profiles/precision_r02_config3.md.  About 45 minutes on 8 cores.

    python oracle/precision_eq4.py --out profiles/precision_r02_eq4_oracle.md
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import rgf_oracle as orc                  # noqa: E402
from paper_1107_5300_b200 import inputs               # noqa: E402  (seeded input generators only)

ENERGIES = np.array([0.03, 0.05, 0.09, 0.2, 0.5])     # the energies of SURVEY.md 8(c): N_ch = 1, 2, 3, 6, 16


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None)
    ap.add_argument("--L", type=int, default=2000)
    a = ap.parse_args()
    lines = ["# The paper's Eq. 4 form in single precision on the CPU oracle (M = 244, L = %d, eta = 1e-9 eV)" % a.L, "",
             "Command: `python oracle/precision_eq4.py --out profiles/precision_r02_eq4_oracle.md` (oracle only, %d threads)." % orc.num_threads(),
             "T_ref = direct form in double (orc_transmission_batch); eq4/float = (1 - G0 V G V)^-1 G0 with float LU and matmul, leads in",
             "double and rounded; eq4/double = the same form in double (how much is the form, how much the precision).", ""]
    for disordered in (False, True):
        w = inputs.config3(L=a.L, disordered=disordered)
        t0 = time.time()
        T_ref = orc.transmission_batch(w.onsite[0], None, w.t, ENERGIES, w.eta)
        T_d = orc.transmission_eq4_batch(w.onsite[0], None, w.t, ENERGIES, w.eta, use_float=False)
        T_f = orc.transmission_eq4_batch(w.onsite[0], None, w.t, ENERGIES, w.eta, use_float=True)
        lines += ["## %s  (%.0f s)" % (w.name, time.time() - t0), "", "| E [eV] | T_ref | abs(T_eq4/float - T_ref) | relative | abs(T_eq4/double - T_ref) |", "|---|---|---|---|---|"]
        for e, tr, td, tf in zip(ENERGIES, T_ref, T_d, T_f):
            lines.append("| %.2f | %.6f | %.2e | %.1e | %.2e |" % (e, tr, abs(tf - tr), abs(tf - tr) / max(abs(tr), 1e-300), abs(td - tr)))
        lines.append("")
    text = "\n".join(lines) + "\n"
    if a.out:
        with open(a.out, "w") as f:
            f.write(text)
    print(text)


if __name__ == "__main__":
    main()

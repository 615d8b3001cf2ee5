"""Writes the stored oracle transmissions for the full-size configs (tests/golden/config*_oracle.txt).

Calls ONLY oracle/ (the CPU oracle) and the seeded input generators; nothing here comes from the
CUDA path.  These runs take minutes to an hour of CPU time (naive LU at M = 244 / 1024), which is
why their results are stored instead of being recomputed inside the GPU parity tests.

    python tests/golden/make_oracle_goldens.py --config 2 [--threads 8]
    python tests/golden/make_oracle_goldens.py --config 2 --append 236 246 250 261 266 280
                                     (more energies of device 0, appended to the stored file; the existing lines stay)

Each output line: dev_index energy_index E[eV] T.  Header lines (#) state the workload recipe.
Lead self-energies use the oracle's cell form (Sancho-Rubio on the 2M x 2M two-slice cell,
LEAD_CELL) for M <= 512; the truncated configs[4] case (M = 1024) uses the block form, which
tests/test_oracle_pins.py pins against the cell form away from its resonances.
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import rgf_oracle as orc          # noqa: E402
from paper_1107_5300_b200 import inputs       # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def subset(cfg):
    """(workload, list of dev indices, list of energy indices, truncation length or None)."""
    if cfg == 1:
        return inputs.config1(), [0, 1, 2, 3], list(range(0, 256, 32)) + [127, 128], None
    if cfg == 2:
        return inputs.config2(), [0], [0, 73, 146, 219, 255, 256, 365, 511], None
    if cfg == 3:
        return inputs.config3(disordered=True), [0], [0, 170, 300, 511, 512, 700, 767, 768, 900, 1023], None
    if cfg == 4:
        return inputs.config4(), [0], [0, 9, 18, 27, 36, 45, 54, 63], 64      # first 64 slices on 8 energies (truncated device)
    raise SystemExit("config must be 1..4")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--append", type=int, nargs="+", default=None, help="energy indices (device 0) to add to the stored file")
    a = ap.parse_args()
    w, devs, eidx, trunc = subset(a.config)
    if a.append:
        devs, eidx = [0], sorted(a.append)
    if trunc:
        w = inputs.truncate(w, trunc)
    E = w.energies[eidx]
    out = os.path.join(HERE, "config%d_oracle.txt" % a.config)
    lines = []
    t0 = time.time()
    for d in devs:
        vac = None if w.vacancy is None else w.vacancy[d]
        method = orc.LEAD_CELL if w.M <= 512 else orc.LEAD_BLOCK
        T, st = orc.transmission_batch(w.onsite[d], vac, w.t, E, w.eta, method=method,
                                       nthreads=a.threads, return_status=True)
        assert np.all(st == 0), st
        for k, e, tk in zip(eidx, E, T):
            lines.append("%d %d %.17g %.17g\n" % (d, k, e, tk))
    dt = time.time() - t0
    if a.append:
        with open(out, "a") as f:
            f.write("# appended by --append %s: same oracle call, %d threads, %.0f s wall\n"
                    % (" ".join(str(k) for k in eidx), orc.num_threads() if a.threads <= 0 else a.threads, dt))
            f.writelines(lines)
        print(out, "appended, %.0f s" % dt)
        return
    with open(out, "w") as f:
        f.write("# oracle transmissions, written by tests/golden/make_oracle_goldens.py --config %d\n" % a.config)
        f.write("# workload: %s; t=%g eV eta=%g eV; notes=%s; numpy %s\n" % (w.name, w.t, w.eta, w.notes, np.__version__))
        f.write("# oracle: oracle/rgf_oracle.c (naive LU, %s leads), %d threads, %.0f s wall\n" % ("LEAD_CELL" if w.M <= 512 else "LEAD_BLOCK", orc.num_threads() if a.threads <= 0 else a.threads, dt))
        f.write("# columns: dev_index energy_index E[eV] T\n")
        f.writelines(lines)
    print(out, "%.0f s" % dt)


if __name__ == "__main__":
    main()

"""Compares alternative readings of the paper's gaps with the values the paper prints (Tables 1-2).
TEST INFRASTRUCTURE: calls only oracle/ and the seeded input generators.

  python oracle/readings_table.py [--sizes 10 20 40] > table.md

For every listed reading (R5 tau2 normalised or not; S3 sum or max over directions; G3 tanh
constant C in {1, 5, 20}; G2 variant A or B) it runs the accuracy test of PAPER.md:378-396 to t = 2 (CFL 0.5, tau = 0)
with the CPU oracle and prints the L1 / L2 density errors next to the printed ones and their relative deviation.
The linear scheme (Table 1) depends on R5 and S3 only; the nonlinear one (Table 2) also on G2 and G3.
"""
import argparse
import math
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import ref                      # noqa: E402
from paper_2508_08965_b200 import inputs    # noqa: E402

TABLE1 = {10: (2.1963e-2, 8.5136e-3), 20: (7.1472e-4, 2.8195e-4), 40: (2.3127e-5, 9.0788e-6), 80: (8.0092e-7, 3.1656e-7)}
TABLE2 = {10: (3.2325e-2, 1.2403e-2), 20: (7.1472e-4, 2.8195e-4), 40: (2.3127e-5, 9.0788e-6), 80: (8.0092e-7, 3.1656e-7)}


def run(n, nonlinear, r5=1, s3=1, g2=1, C=5.0, cfl=0.5, tend=2.0, r=2):
    ref.set_readings(r5, s3, g2)
    try:
        nodes, Q, G, D = inputs.sine_advection(n)
        s = ref.RefSolver(nodes, ref.make_params(**inputs.sine_params(), nonlinear=nonlinear, geno_C=C, geno_r=r))
        s.set_state(Q, G, D)
        t = 0.0
        while t < tend - 1e-13:
            dt = min(s.compute_dt(cfl), tend - t)
            s.step(dt); t += dt
        e = s.get_state()[0][0] - inputs.sine_exact_averages(n, tend)
        s.close()
    finally:
        ref.set_readings(1, 1, 1)
    h = 2.0 / n
    return np.abs(e).sum() * h ** 3, math.sqrt((e ** 2).sum() * h ** 3)


def geno_scan():
    """the path function (readings G2 / G3) against Table 2's 10^3 row, the only number the paper prints
    that exercises the blend, at the time step of the table's header (CFL 0.5) AND at the one that reproduces Table 1
    (CFL 0.25).  A reading is admissible only if its 20^3 row equals the linear scheme's to 5 digits (Table 2 = Table 1 there)."""
    print("| G2 variant, r | C | CFL | 10^3 L1 | dev from 3.2325e-2 | 10^3 L2 | dev from 1.2403e-2 | 20^3 L1 | 20^3 L1 / linear 20^3 L1 - 1 |")
    print("|---|---|---|---|---|---|---|---|---|")
    lin20 = {cfl: run(20, 0, cfl=cfl)[0] for cfl in (0.5, 0.25)}
    lin10 = {cfl: run(10, 0, cfl=cfl) for cfl in (0.5, 0.25)}
    for cfl in (0.5, 0.25):
        print("| linear scheme | - | %.2f | %.4e | %+.1f %% of Table 1 | %.4e | %+.1f %% of Table 1 | %.4e | 0 |" %
              (cfl, lin10[cfl][0], 100 * (lin10[cfl][0] / TABLE1[10][0] - 1), lin10[cfl][1], 100 * (lin10[cfl][1] / TABLE1[10][1] - 1), lin20[cfl]), flush=True)
    variants = [("(B) third + fourth part, r = 2", dict(g2=1), [3.0, 3.25, 3.5, 3.75, 4.0, 4.25, 4.5, 4.75, 5.0]),
                ("fourth part only, r = 2", dict(g2=2), [3.0, 4.0, 5.0]),
                ("(B), r = 1 (ratio not squared)", dict(g2=1, r=1), [3.0, 4.0, 5.0]),
                ("(A) |IS^H - IS^L|, r = 2", dict(g2=0), [3.0, 5.0])]
    for name, kw, Cs in variants:
        for C in Cs:
            for cfl in (0.5, 0.25):
                l1, l2 = run(10, 1, C=C, cfl=cfl, **kw)
                m1, _ = run(20, 1, C=C, cfl=cfl, **kw)
                print("| %s | %.2f | %.2f | %.4e | %+.1f %% | %.4e | %+.1f %% | %.4e | %.1e |" %
                      (name, C, cfl, l1, 100 * (l1 / TABLE2[10][0] - 1), l2, 100 * (l2 / TABLE2[10][1] - 1), m1, m1 / lin20[cfl] - 1), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", type=int, nargs="+", default=[10, 20, 40])
    ap.add_argument("--geno-scan", action="store_true", help="scan of the GENO path function against Table 2 (see geno_scan)")
    a = ap.parse_args()
    if a.geno_scan:
        return geno_scan()
    lin = [("taken: R5 normalised, S3 sum", dict()), ("R5 unnormalised tau2", dict(r5=0)), ("S3 max over directions", dict(s3=0)),
           ("R5 unnormalised + S3 max", dict(r5=0, s3=0)), ("taken, but CFL = 0.25 (size of the temporal error)", dict(cfl=0.25))]
    print("| reading | mesh | L1 | paper L1 | dev | L2 | paper L2 | dev | order (L1) |")
    print("|---|---|---|---|---|---|---|---|---|")
    for name, kw in lin:
        prev = None
        for n in a.sizes:
            t0 = time.time()
            l1, l2 = run(n, 0, **kw)
            p1, p2 = TABLE1[n]
            order = "" if prev is None else "%.2f" % math.log2(prev / l1)
            print("| linear, %s | %d^3 | %.4e | %.4e | %+.1f %% | %.4e | %.4e | %+.1f %% | %s |" %
                  (name, n, l1, p1, 100 * (l1 / p1 - 1), l2, p2, 100 * (l2 / p2 - 1), order), flush=True)
            print("  (%.0f s)" % (time.time() - t0), file=sys.stderr)
            prev = l1
    nl = [("taken: G2 (B), C = 5", dict()), ("G2 (B), C = 1", dict(C=1.0)), ("G2 (B), C = 3", dict(C=3.0)), ("G2 (B), C = 4", dict(C=4.0)),
          ("G2 (B), C = 20", dict(C=20.0)),
          ("G2 (A), C = 5", dict(g2=0)), ("G2 (A), C = 20", dict(g2=0, C=20.0))]
    for name, kw in nl:
        for n in [m for m in a.sizes if m <= 20]:
            l1, l2 = run(n, 1, **kw)
            p1, p2 = TABLE2[n]
            print("| nonlinear, %s | %d^3 | %.4e | %.4e | %+.1f %% | %.4e | %.4e | %+.1f %% | |" %
                  (name, n, l1, p1, 100 * (l1 / p1 - 1), l2, p2, 100 * (l2 / p2 - 1)), flush=True)


if __name__ == "__main__":
    main()

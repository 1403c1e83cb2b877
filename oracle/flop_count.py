"""Instrumented flop count of the CPU oracle.  TEST INFRASTRUCTURE ONLY.

  python oracle/flop_count.py        # prints the counts as JSON

Builds oracle/flopcount.cpp (cgks_ref.c with a counting double; add/sub/mul = 1, div/sqrt/exp/erfc/tanh/pow = 1) and
counts, for the gas constants of the bench workload (iso_sup: power-law viscosity, Pr = 0.7, c2 = 5, GENO on):
  flux_point      one call of cgks_ref_flux_point (one face Gauss point, Cartesian frame), discontinuous states
  recon_var       one call of cgks_ref_recon_reference (one cell and variable: a = M d, linear polynomials, GENO, 24 points)
  step_per_cell   one full S2O4 step on a periodic 6^3 mesh divided by the number of cells
each as (all operations, operations on non-zero operands).  The second figure leaves out multiplications by the
structural zeros of M, E and the moment tables, i.e. it is the count SURVEY.md 8(d) calls algorithmic.
bench.py carries the flux figure as a constant; tests/test_abi.py checks that constant against this script.
"""
import ctypes as C
import json
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
sys.path.insert(0, ROOT)
LIB = os.path.join(HERE, "libcgks_ref_count.so")


def build(force=False):
    deps = [os.path.join(HERE, f) for f in ("flopcount.cpp", "cgks_ref.c", "cgks_ref.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    subprocess.check_call(["g++", "-O1", "-fpermissive", "-w", "-ffp-contract=off", "-fPIC", "-shared", "-o", LIB,
                           os.path.join(HERE, "flopcount.cpp"), "-lm"])
    return LIB


def counts():
    from oracle import build as obuild, ref
    from paper_2508_08965_b200 import inputs
    build()
    saved_lib, saved_build = ref._lib, obuild.build
    ref._lib = None
    obuild.build = lambda force=False: LIB           # oracle.ref loads the counting build through its usual loader
    try:
        L = ref.lib()
        L.cgks_ref_flops_get.argtypes = [C.POINTER(C.c_long), C.POINTER(C.c_long)]

        def measure(fn):
            L.cgks_ref_flops_reset(); fn()
            a = C.c_long(0); b = C.c_long(0); L.cgks_ref_flops_get(C.byref(a), C.byref(b))
            return int(a.value), int(b.value)
        prm = ref.make_params(**inputs.iso_params(1.0, k0=8.0), nonlinear=1)
        rng = np.random.default_rng(0)
        out = {}
        # flux: discontinuous states with slopes; the count does not depend on the values (no data-dependent loops; the
        # branches taken are those of the bench workload: viscous, power law, Pr fix, c2 > 0)
        w = inputs.workload("iso_sup", 8, 2.0)
        Q = w["Q"]
        WL = Q[:, 1, 2, 3].copy(); WR = Q[:, 1, 2, 4].copy()
        gL = 0.2 * rng.standard_normal((5, 3)); gR = 0.2 * rng.standard_normal((5, 3))
        n = np.array([1.0, 0.0, 0.0]); t1 = np.array([0.0, 1.0, 0.0])
        ref.flux_point(prm, 1e-2, WL, gL, WR, gR, n, t1)                     # builds the constants outside the count
        out["flux_point"] = measure(lambda: ref.flux_point(prm, 1e-2, WL, gL, WR, gR, n, t1))
        d = rng.standard_normal(72)
        ref.recon_reference(prm, d)                                          # builds M, E, Gram outside the count
        out["recon_var"] = measure(lambda: ref.recon_reference(prm, d))
        m = 6
        wk = inputs.workload("iso_sup", m, 2.0)
        s = ref.RefSolver(wk["nodes"], prm); s.set_state(wk["Q"])
        dt = s.compute_dt(0.5)
        a, b = measure(lambda: s.step(dt))
        out["step_per_cell"] = (a / m ** 3, b / m ** 3)
        s.close()
        return out
    finally:
        ref._lib, obuild.build = saved_lib, saved_build


if __name__ == "__main__":
    print(json.dumps(counts()))

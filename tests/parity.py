"""Helpers of the GPU parity tests: run the same seeded workload through the oracle and through the C ABI, and the
per-field error norm of SURVEY.md section 8(d) / DESIGN.md section 6."""
import numpy as np

from oracle import ref
from paper_2508_08965_b200 import inputs


REST_FRACTION = 0.05      # a flow counts as "at rest" when max|U| < REST_FRACTION * max c


def field_errors(gpu, orc, nodes, Qref, mask=None):
    """Relative L-infinity error per field (80 planes): max|gpu-oracle| / max(|oracle|_inf, delta_f),
    delta_f = 1e-3 |Q_v|_inf (D planes), 1e-3 |Q_v|_inf / h_min (G planes), 1e-3 |rho|_inf max|U| (momentum planes).
    The floors keep fields that are identically ~0 (free-stream derivatives, transverse momenta of 1-D flows) from turning
    round-off noise into O(1) 'relative' errors.  Two statements the survey's text leaves open:
    (i) for a momentum variable, |Q_v|_inf in the D and G floors is max(|Q_v|_inf, momentum floor), otherwise the floor
    of the derivative planes of an identically-zero momentum component would itself be zero; (ii) when the flow is
    at rest (max|U| < 0.05 max c: the shock tubes) the velocity scale max|U| is itself ~0 and is replaced by max(|U| + c).
    `mask` (bool, cells) restricts the numerators to the cells it selects (the scales stay those of the whole field)."""
    sel = (lambda a: a) if mask is None else (lambda a: a[mask])
    return {k: sel(e).max() for k, e in element_errors(gpu, orc, nodes, Qref).items()}


def element_errors(gpu, orc, nodes, Qref):
    """|gpu - oracle| of every element divided by the field's scale max(|oracle_f|_inf, delta_f) (see field_errors)."""
    Qg, Gg, Dg = gpu; Qo, Go, Do = orc
    hmin = min(np.abs(np.diff(nodes[0], axis=2)).min(), np.abs(np.diff(nodes[1], axis=1)).min(), np.abs(np.diff(nodes[2], axis=0)).min())
    qinf = [np.abs(Qref[v]).max() for v in range(5)]
    rho = Qref[0]; U = Qref[1:4] / rho
    pres = 0.4 * (Qref[4] - 0.5 * rho * (U ** 2).sum(0))
    speed = np.sqrt((U ** 2).sum(0)); sound = np.sqrt(1.4 * pres / rho)
    umax = speed.max()
    if umax < REST_FRACTION * sound.max():
        umax = (speed + sound).max()
    mom_floor = 1e-3 * qinf[0] * umax
    errs = {}
    for v in range(5):
        floor = mom_floor if 1 <= v <= 3 else 0.0
        qfloor = max(qinf[v], mom_floor) if 1 <= v <= 3 else qinf[v]
        errs["Q%d" % v] = np.abs(Qg[v] - Qo[v]) / max(np.abs(Qo[v]).max(), floor, 1e-300)
        for r in range(3):
            errs["G%d_%d" % (v, r)] = np.abs(Gg[v, r] - Go[v, r]) / max(np.abs(Go[v, r]).max(), 1e-3 * qfloor / hmin)
        for s in range(12):
            errs["D%d_%d" % (v, s)] = np.abs(Dg[v, s] - Do[v, s]) / max(np.abs(Do[v, s]).max(), 1e-3 * qfloor)
    return errs


def build_case(name, n=None, nonlinear=None, k0=None):
    w = inputs.workload(name, n, k0)
    if nonlinear is not None:
        w["nonlinear"] = nonlinear
    return w


def run_oracle(w, nsteps, dts=None):
    s = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=w["nonlinear"]))
    s.set_state(w["Q"], w["G"], w["D"])
    used = []
    for i in range(nsteps):
        dt = s.compute_dt(w["cfl"]) if dts is None else dts[i]
        used.append(dt); s.step(dt)
    out = s.get_state(); s.close()
    return out, used


def run_gpu(w, nsteps, dts=None, budget_bytes=0):
    """Steps with `dts` when given (the oracle's), else with the library's own cgks_compute_dt; returns the state and
    the library's own dt of every step."""
    from paper_2508_08965_b200 import binding
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=w["nonlinear"]), budget_bytes=budget_bytes)
    s.set_state(w["Q"], w["G"], w["D"])
    used = []
    for i in range(nsteps):
        dt_own = s.compute_dt(w["cfl"])
        dt = dt_own if dts is None else dts[i]
        used.append(dt_own); s.step(dt)
    s.status()
    Q, G, D = s.get_state()
    out = (Q.cpu().numpy(), G.cpu().numpy(), D.cpu().numpy())
    s.close()
    return out, used

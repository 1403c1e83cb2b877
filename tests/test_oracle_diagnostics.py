"""Pin of the oracle's diagnostics against closed forms: for the Taylor-Green
velocity field U = (sin x cos y cos z, -cos x sin y cos z, 0) with rho = 1 the volume averages are
E_k = <|U|^2>/2 = 1/8 and <|curl U|^2> = 3/4, so that enstrophy = 3 mu/4 for constant mu."""
import math

import numpy as np

from oracle import ref
from paper_2508_08965_b200 import inputs

G_ = inputs.GAUSS_G


def _analytic_state(n):
    """rho = 1, momentum = Taylor-Green velocity: exact cell averages, G by the face quadrature of Eq. 9 and D = exact
    point-value differences of Eq. 10 (the same recipe as inputs.sine_advection)."""
    h = 2.0 * math.pi / n
    nodes = inputs.cartesian_nodes(n)
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    fu = lambda x, y, z: np.sin(x) * np.cos(y) * np.cos(z)
    fv = lambda x, y, z: -np.cos(x) * np.sin(y) * np.cos(z)
    sinc = (math.sin(h / 2) / (h / 2)) ** 3
    shape = X.shape
    Q = np.zeros((5,) + shape); G = np.zeros((5, 3) + shape); D = np.zeros((5, 12) + shape)
    Q[0] = 1.0; Q[1] = sinc * fu(X, Y, Z); Q[2] = sinc * fv(X, Y, Z)
    Q[4] = 100.0 / 0.4 + 0.5 * (Q[1] ** 2 + Q[2] ** 2)
    P = [X, Y, Z]
    for v, f in ((1, fu), (2, fv)):
        for axis in range(3):
            o1, o2 = [a for a in range(3) if a != axis]
            k = 0; acc = 0.0
            for a in (-G_ * h, G_ * h):
                for b in (-G_ * h, G_ * h):
                    hi = [p.copy() for p in P]; lo = [p.copy() for p in P]
                    hi[axis] = hi[axis] + h / 2; lo[axis] = lo[axis] - h / 2
                    for q in (hi, lo):
                        q[o1] = q[o1] + a; q[o2] = q[o2] + b
                    d = f(*hi) - f(*lo)
                    D[v, 4 * axis + k] = d; acc = acc + 0.25 * d / h; k += 1
            G[v, axis] = acc
    return nodes, Q, G, D


def test_taylor_green_kinetic_energy_and_enstrophy_closed_forms():
    errs = []
    for n in (8, 16):
        nodes, Q, G, D = _analytic_state(n)
        prm = dict(inputs.tgv_params())
        s = ref.RefSolver(nodes, ref.make_params(**prm, nonlinear=0)); s.set_state(Q, G, D)
        ek, en = s.diagnostics(); s.close()
        errs.append((abs(ek / 0.125 - 1), abs(en / (0.75 * prm["mu_ref"]) - 1)))
    assert errs[1][0] < 1e-4 and errs[1][1] < 2e-3, errs
    assert errs[0][0] / errs[1][0] > 12 and errs[0][1] / errs[1][1] > 10, errs        # at least ~4th order


def test_uniform_flow_on_the_distorted_mesh():
    """Uniform flow: E_k = rho |U|^2/2 to round-off and zero enstrophy, also on the non-orthogonal mesh (the quadrature
    weights |Omega_i|/8 sum to the domain volume; constants are reproduced by the reconstruction)."""
    w = inputs.workload("freestream_curv", 8)
    s = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1)); s.set_state(w["Q"])
    ek, en = s.diagnostics(); s.close()
    assert abs(ek - 0.5 * (1 + 0.25 + 0.0625)) < 1e-13 and abs(en) < 1e-20

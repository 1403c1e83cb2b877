"""Scheme-level pins of the oracle: geometry, S2O4, conservation, free-stream preservation, Tables 1-2, ENO property.
CPU only.  Pin numbers follow DESIGN.md section 4."""
import math
import os

import numpy as np
import pytest

from oracle import ref
from paper_2508_08965_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "table1_table2.txt")


def golden():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        t, n, l1, l2 = line.split()
        out[(int(t), int(n))] = (float(l1), float(l2))
    return out


def run_sine(n, nonlinear, tend=2.0, cfl=0.5):
    nodes, Q, G, D = inputs.sine_advection(n)
    s = ref.RefSolver(nodes, ref.make_params(**inputs.sine_params(), nonlinear=nonlinear))
    s.set_state(Q, G, D)
    t = 0.0
    while t < tend - 1e-13:
        dt = min(s.compute_dt(cfl), tend - t)
        s.step(dt); t += dt
    Q1, _, _ = s.get_state()
    e = Q1[0] - inputs.sine_exact_averages(n, tend)
    h = 2.0 / n
    # reading T3: un-normalised norms against exact CELL AVERAGES
    return np.abs(e).sum() * h ** 3, math.sqrt((e ** 2).sum() * h ** 3), Q, Q1


# ----------------------------------------------------------------------------- geometry
def test_geometry_cartesian_and_curvilinear():
    n = 6
    nodes = inputs.cartesian_nodes(n, 0.0, 2.0)
    s = ref.RefSolver(nodes, ref.make_params())
    vol, J0, area = s.geometry()
    h = 2.0 / n
    np.testing.assert_allclose(vol, h ** 3, rtol=1e-13)
    np.testing.assert_allclose(J0, np.broadcast_to(h * np.eye(3), J0.shape), atol=1e-14)
    for ax in range(3):
        e = np.zeros(3); e[ax] = h * h
        np.testing.assert_allclose(area[ax], np.broadcast_to(e, area[ax].shape), atol=1e-14)
    nodes = inputs.curvilinear_nodes(n)
    s = ref.RefSolver(nodes, ref.make_params())
    vol, J0, area = s.geometry()
    assert abs(vol.sum() - (2 * math.pi) ** 3) < 1e-10          # trilinear cells tile the periodic box (Appendix)
    assert (vol > 0).all()
    # closed cell surfaces: sum of outward vector areas is zero (reading R2) -> free-stream preservation
    tot = np.zeros(vol.shape + (3,))
    for ax in range(3):
        tot += area[ax] - np.roll(area[ax], 1, axis=2 - ax)
    assert np.abs(tot).max() < 1e-13
    # J0 columns are the three edge vectors from node (i,j,k)  (Eq. 18, reading R1)
    i, j, k = 2, 3, 1
    for a, (di, dj, dk) in enumerate([(1, 0, 0), (0, 1, 0), (0, 0, 1)]):
        np.testing.assert_allclose(J0[k, j, i, :, a], nodes[:, k + dk, j + dj, i + di] - nodes[:, k, j, i], atol=1e-15)


# ----------------------------------------------------------------------------- P12: S2O4
def test_P12_s2o4_scalar_ode():
    """y' = lambda y through the two stages gives 1 + z + z^2/2 + z^3/6 + z^4/24."""
    lam, dt, y = -0.7, 0.3, 1.3
    ys = ref.s2o4_stage1(y, lam * y, lam * lam * y, dt)
    yn = ref.s2o4_stage2(y, lam * y, lam * lam * y, lam * lam * ys, dt)
    z = lam * dt
    assert abs(yn - y * (1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24)) < 1e-15
    assert abs(ys - y * (1 + z / 2 + z ** 2 / 8)) < 1e-15


# ----------------------------------------------------------------------------- P10: invariants
def _random_smooth_state(nodes, rng, amp=0.05):
    x, y, z = inputs.cell_centroids(nodes)
    f = lambda: amp * (np.sin(x + rng.uniform(0, 6)) * np.cos(y + rng.uniform(0, 6)) + np.sin(z + rng.uniform(0, 6)))
    return inputs.prim_to_cons(1.0 + f(), 0.5 + f(), -0.3 + f(), 0.2 + f(), 1.0 + f())


@pytest.mark.parametrize("mesh", ["cart", "curv"])
def test_P10_conservation(mesh):
    """Single-valued face fluxes (Eq. 8): sum |Omega_i| Q_i is constant to round-off on periodic domains."""
    n = 6
    nodes = inputs.cartesian_nodes(n) if mesh == "cart" else inputs.curvilinear_nodes(n)
    s = ref.RefSolver(nodes, ref.make_params(**inputs.tgv_params(Re=100.0), nonlinear=1))
    Q = _random_smooth_state(nodes, np.random.default_rng(0))
    s.set_state(Q)
    vol, _, _ = s.geometry()
    tot0 = (Q * vol).sum(axis=(1, 2, 3))
    for _ in range(3):
        s.step(s.compute_dt(0.5))
    Q1, _, _ = s.get_state()
    tot1 = (Q1 * vol).sum(axis=(1, 2, 3))
    np.testing.assert_allclose(tot1, tot0, rtol=1e-13, atol=1e-12)
    assert np.abs(Q1 - Q).max() > 1e-4           # something happened


def test_P10_free_stream_preservation_curvilinear():
    """Uniform flow on the distorted mesh stays uniform (BASELINE.json config 3), all 80 dof."""
    n = 6
    nodes = inputs.curvilinear_nodes(n)
    s = ref.RefSolver(nodes, ref.make_params(**inputs.tgv_params(), nonlinear=1))
    Q = inputs.free_stream((n, n, n))
    s.set_state(Q)
    for _ in range(5):
        s.step(s.compute_dt(0.5))
    Q1, G1, D1 = s.get_state()
    assert np.abs(Q1 - Q).max() < 1e-13
    assert np.abs(G1).max() < 1e-12 and np.abs(D1).max() < 1e-13


def test_axis_permutation_symmetry_of_a_step():
    """Relabelling the axes (x,y,z)->(y,z,x) of mesh and data relabels the result: every ordering table
    (faces, edges, lines, Gauss points, frames) is consistent across the whole step."""
    n = 6
    nodes = inputs.cartesian_nodes(n)
    rng = np.random.default_rng(5)
    Q = _random_smooth_state(nodes, rng, amp=0.1)
    prm = ref.make_params(**inputs.tgv_params(Re=200.0), nonlinear=1)
    s = ref.RefSolver(nodes, prm); s.set_state(Q); dt = s.compute_dt(0.5); s.step(dt)
    Q1, G1, D1 = s.get_state()
    # transpose (2,0,1): A'[k',j',i'] = A[j',i',k'], i.e. the old cell (x,y,z) moves to (x',y',z') = (y,z,x)
    def perm(A):
        return np.ascontiguousarray(np.transpose(A, (2, 0, 1)))
    # vectors follow: (u'_x, u'_y, u'_z) = (u_y, u_z, u_x)
    Qp = np.stack([perm(Q[0]), perm(Q[2]), perm(Q[3]), perm(Q[1]), perm(Q[4])])
    s2 = ref.RefSolver(nodes, prm); s2.set_state(Qp); s2.step(dt)
    Q2, _, _ = s2.get_state()
    Q1p = np.stack([perm(Q1[0]), perm(Q1[2]), perm(Q1[3]), perm(Q1[1]), perm(Q1[4])])
    np.testing.assert_allclose(Q2, Q1p, rtol=1e-11, atol=1e-12)


# ----------------------------------------------------------------------------- P4/P5/P6: Tables 1 and 2
def test_P4_table1_linear_and_order():
    """Table 1: linear CGKS-5, t = 2.  With the readings taken the oracle's errors are within
    -3.7 / -0.7 % (10^3) and +6.7 / +6.6 % (20^3) of the printed L1 / L2 values: the closest of the readings compared by
    oracle/readings_table.py, and the printed order (4.94) is matched to within 0.2."""
    gold = golden()
    l1_10, l2_10, Q0, Q1 = run_sine(10, 0)
    l1_20, l2_20, _, _ = run_sine(20, 0)
    assert abs(l1_10 / gold[(1, 10)][0] - 1) < 0.045 and abs(l2_10 / gold[(1, 10)][1] - 1) < 0.015
    assert abs(l1_20 / gold[(1, 20)][0] - 1) < 0.075 and abs(l2_20 / gold[(1, 20)][1] - 1) < 0.075
    order = math.log2(l1_10 / l1_20)
    assert abs(order - 4.9415) < 0.2, order
    # the printed L1/L2 ratio (2.58 at 10^3) fixes the norm definition (reading T3)
    assert abs(l1_10 / l2_10 - gold[(1, 10)][0] / gold[(1, 10)][1]) < 0.1
    # conservation over the whole run
    np.testing.assert_allclose(Q1.sum(axis=(1, 2, 3)), Q0.sum(axis=(1, 2, 3)), rtol=1e-13)


def test_P4b_table1_to_one_percent_with_half_the_time_step():
    """The remaining deviation of P4 is TEMPORAL: with half the time step (CFL 0.25 in reading S3) the oracle reproduces
    Table 1 at 20^3 to +0.7 % (L1) / +0.2 % (L2) and the 10^3 L2 value to +0.4 % (oracle/readings_table.py).  The spatial
    operator -- stencil, Eq. 14/19 rows, row scalings, tau_2 normalisation (R4, R5), the tau = 0 flux and the norms (T3) --
    is therefore the authors'; what differs is the size of their time step, which the paper does not give (S3)."""
    gold = golden()
    l1, l2, _, _ = run_sine(20, 0, cfl=0.25)
    assert abs(l1 / gold[(1, 20)][0] - 1) < 0.015 and abs(l2 / gold[(1, 20)][1] - 1) < 0.01, (l1, l2)
    l1, l2, _, _ = run_sine(10, 0, cfl=0.25)
    assert abs(l1 / gold[(1, 10)][0] - 1) < 0.05 and abs(l2 / gold[(1, 10)][1] - 1) < 0.01, (l1, l2)


def test_P6_table2_pattern():
    """Table 2: nonlinear errors are LARGER than linear at 10^3 and identical at >= 20^3.
    Checked through chi on the exact data (20^3: 1 - chi < 1e-5 everywhere; 10^3: chi clearly below 1 somewhere) and
    a full 10^3 run."""
    gold = golden()
    for n, lo, hi in ((20, 0.0, 1e-5), (10, 0.05, 1.0)):
        nodes, Q, G, D = inputs.sine_advection(n)
        s = ref.RefSolver(nodes, ref.make_params(**inputs.sine_params(), nonlinear=1)); s.set_state(Q, G, D)
        _, chi = s.reconstruct()
        dev = 1.0 - chi[0].min()
        assert lo <= dev <= hi, (n, dev)
    l1_nl, l2_nl, _, _ = run_sine(10, 1)
    l1_l, l2_l, _, _ = run_sine(10, 0)
    assert l1_nl > 1.1 * l1_l and l2_nl > 1.1 * l2_l
    assert l1_nl < 2.0 * gold[(2, 10)][0]


def test_P6c_table2_row_at_the_best_fit():
    """Table 2's 10^3 row (L1 3.2325e-2, L2 1.2403e-2) is the one printed number that exercises the GENO blend.
    The scan of DESIGN.md section 3.2 (oracle/readings_table.py --geno-scan) finds that reading G2 (B) with r = 2 reproduces it to
    2 % at C = 3.5 (CFL 0.5); a wrong power in alpha, a missing square, IS^tau from the wrong derivative orders or a different
    tanh map all move the row by 10 % or more (the scan's neighbours and negative controls), so 3 % pins the FORM of the path
    function to the paper's number.  The default C = 5 (kept because only it leaves the 20^3 row identical to the linear one,
    section 3.2) misses the row by -23 % / -18 %: pinned too, so that a change of the default or of the blend is noticed."""
    from oracle import readings_table
    p1, p2 = readings_table.TABLE2[10]
    l1, l2 = readings_table.run(10, 1, C=3.5, cfl=0.5)
    assert abs(l1 / p1 - 1.0) < 0.03 and abs(l2 / p2 - 1.0) < 0.03, (l1, l2)
    l1, l2 = readings_table.run(10, 1, C=5.0, cfl=0.5)
    assert abs(l1 / p1 - (1.0 - 0.231)) < 0.01 and abs(l2 / p2 - (1.0 - 0.177)) < 0.01, (l1, l2)
    l1, l2 = readings_table.run(10, 1, C=4.0, cfl=0.5, g2=2)          # negative control: fourth-derivative part only
    assert l1 / p1 < 0.80


def test_P6b_nonlinear_equals_linear_at_20():
    """Short 20^3 run: nonlinear and linear results agree to ~1e-6 relative of the perturbation (Table 2 rows >= 20^3)."""
    a = run_sine(20, 0, tend=0.1)[3]; b = run_sine(20, 1, tend=0.1)[3]
    assert np.abs(a[0] - b[0]).max() < 1e-6


# ----------------------------------------------------------------------------- P11: ENO property
def test_P11_double_shock_tube_no_overshoot():
    """Periodic two-state Riemann problem (two Sod tubes back to back) through the 3-D code: no O(1) overshoot,
    chi drops only near the jumps."""
    ni, nj, nk = 48, 4, 4
    nodes = inputs.cartesian_nodes((ni, nj, nk), 0.0, 1.0)
    # rescale y,z so that cells are cubes
    nodes[1] *= nj / ni; nodes[2] *= nk / ni
    x = (np.arange(ni) + 0.5) / ni
    left = (x > 0.25) & (x < 0.75)
    rho = np.where(left, 1.0, 0.125)[None, None, :] * np.ones((nk, nj, ni)); p = np.where(left, 1.0, 0.1)[None, None, :] * np.ones((nk, nj, ni))
    zero = np.zeros_like(rho)
    Q = inputs.prim_to_cons(rho, zero, zero, zero, p)
    s = ref.RefSolver(nodes, ref.make_params(tau_c1=0.05, tau_c2=5.0, nonlinear=1))
    s.set_state(Q)
    _, chi0 = s.reconstruct()
    frac0 = (chi0[0] < 0.99).mean()
    assert 0.02 < frac0 < 0.4, frac0                      # only the cells whose stencil sees a jump
    assert chi0[0][0, 0, 18:30].min() == 1.0 and chi0[0][0, 0, 42:48].min() == 1.0     # flat data: chi = 1 exactly
    t = 0.0
    while t < 0.08:
        dt = s.compute_dt(0.5); s.step(dt); t += dt
    Q1, _, _ = s.get_state()
    assert Q1[0].min() > 0.125 - 0.02 and Q1[0].max() < 1.0 + 0.02
    pr = 0.4 * (Q1[4] - 0.5 * (Q1[1] ** 2 + Q1[2] ** 2 + Q1[3] ** 2) / Q1[0])
    assert pr.min() > 0.1 - 0.02 and pr.max() < 1.0 + 0.02
    assert np.abs(Q1[2]).max() < 1e-12 and np.abs(Q1[3]).max() < 1e-12      # stays one-dimensional
    np.testing.assert_allclose(Q1[:, 0, 0, :], Q1[:, 2, 3, :], atol=1e-12)
    _, chi = s.reconstruct()
    assert chi[0].min() < 0.5 and chi[0].max() > 0.99
    # mirror symmetry about x = 0.5
    np.testing.assert_allclose(Q1[0][0, 0, :], Q1[0][0, 0, ::-1], atol=1e-10)


def test_bootstrap_of_derivative_dof():
    """Reading S2: G from 4th-order central differences of cell averages (error O(h^4)); the four line differences
    of an axis all get the axis value (error O(h^2) in D, regenerated by the scheme after the first step)."""
    errs = []
    for n in (8, 16):
        nodes, Q, G, D = inputs.sine_advection(n)
        s = ref.RefSolver(nodes, ref.make_params()); s.set_state(Q)
        _, Gb, Db = s.get_state()
        errs.append((np.abs(Gb - G).max(), np.abs(Db - D).max()))
    assert errs[0][0] / errs[1][0] > 10 and errs[0][1] / errs[1][1] > 3

"""Pins of the oracle's compact reconstruction (Eq. 11-16, 19) against what the paper and the
mathematics fix.  CPU only.  Pin numbers P1.. follow DESIGN.md section 4."""
import math

import numpy as np
import pytest

from oracle import ref
from tests import refdata as rd

LIN = ref.make_params(nonlinear=0)
NL = ref.make_params(nonlinear=1)


def test_sizes_and_gauss_points():
    didx, gp = ref.basis()
    assert didx.shape == (34, 3)                       # 34 unknowns, 1 <= |d| <= 4
    assert sorted(set(didx.sum(1))) == [1, 2, 3, 4]
    assert len({tuple(r) for r in didx}) == 34
    np.testing.assert_allclose(gp, rd.gauss_points(), atol=1e-15)     # K = 4 Gauss points per face


def test_P1_quartic_exactness():
    """Eq. 14 has 72 consistent equations for 34 unknowns: any polynomial of degree <= 4 is reproduced exactly,
    values and derivatives at all 24 Gauss points (data by numerical quadrature, not the oracle's row formulas)."""
    rng = np.random.default_rng(1)
    for trial in range(3):
        coef = {d: rng.standard_normal() for d in rd.quartic_multi_indices()}
        fn, grad = rd.poly_fn(coef)
        q0, d = rd.data_vector(fn, grad)
        a, b, chi, om, val, gref = ref.recon_reference(LIN, d)
        assert chi == 1.0
        pts = rd.gauss_points()
        exact = np.array([fn(*p) for p in pts]); gex = np.array([[g for g in grad(*p)] for p in pts])
        np.testing.assert_allclose(q0 + val, exact, atol=2e-12)
        np.testing.assert_allclose(gref, gex, atol=2e-11)


def test_P1b_quintic_is_not_exact():
    """Negative control: a fifth-degree term must NOT be reproduced (guards against a vacuous P1)."""
    fn, grad = rd.poly_fn({(5, 0, 0): 1.0, (2, 2, 1): 1.0})
    q0, d = rd.data_vector(fn, grad)
    _, _, _, _, val, _ = ref.recon_reference(LIN, d)
    exact = np.array([fn(*p) for p in rd.gauss_points()])
    assert np.abs(q0 + val - exact).max() > 1e-4


def _functional_matrix():
    """72 x 34 matrix of the data functionals applied to the monomials xi^d/d!, by numerical quadrature."""
    didx, _ = ref.basis()
    A = np.zeros((72, 34))
    for b, d in enumerate(didx):
        f = 1.0 / (math.factorial(d[0]) * math.factorial(d[1]) * math.factorial(d[2]))
        fn, grad = rd.poly_fn({tuple(int(x) for x in d): f})
        _, A[:, b] = rd.data_vector(fn, grad)
    return A


def test_P3_bruteforce_constrained_least_squares():
    """a = M d equals a per-case dense solve of 'strict on the six face-neighbour averages, least squares on the
    other 66 rows' done with a different algorithm (null-space + lstsq) on rows built by quadrature."""
    A = _functional_matrix()
    Cm, L = A[:6], A[6:]
    M, _ = ref.matrices()
    _, _, Vt = np.linalg.svd(Cm)
    Z = Vt[6:].T                                     # null space of the constraints
    rng = np.random.default_rng(2)
    for _ in range(4):
        d = rng.standard_normal(72)
        ap = np.linalg.lstsq(Cm, d[:6], rcond=None)[0]
        y = np.linalg.lstsq(L @ Z, d[6:] - L @ ap, rcond=None)[0]
        a_bf = ap + Z @ y
        np.testing.assert_allclose(M @ d, a_bf, atol=1e-10)
        np.testing.assert_allclose(Cm @ (M @ d), d[:6], atol=1e-11)      # strict rows hold exactly


def test_P3b_row_scalings_matter():
    """h1'=2, h2'=1, h3'=3: with all scalings equal the LS solution differs -> the pin sees them."""
    A = _functional_matrix()
    M, _ = ref.matrices()
    A2 = A.copy(); A2[18:36] /= 2.0; A2[60:72] /= 3.0
    Cm, L = A2[:6], A2[6:]
    _, _, Vt = np.linalg.svd(Cm); Z = Vt[6:].T
    d = np.random.default_rng(3).standard_normal(72)
    d2 = d.copy(); d2[18:36] /= 2.0; d2[60:72] /= 3.0
    ap = np.linalg.lstsq(Cm, d2[:6], rcond=None)[0]
    a_eq = ap + Z @ np.linalg.lstsq(L @ Z, d2[6:] - L @ ap, rcond=None)[0]
    assert np.abs(M @ d - a_eq).max() > 1e-3


def test_matrix_structure_survey_numbers():
    """Independent survey probe: rank 34, ||M||_F = 28.5484, 1008 non-zeros."""
    M, E = ref.matrices()
    assert np.linalg.matrix_rank(M) == 34
    assert abs(np.linalg.norm(M) - 28.5484) < 1e-3
    assert int((np.abs(M) > 1e-12).sum()) == 1008
    assert int((np.abs(E) > 1e-12).sum()) == 2184


def test_fifth_order_plane_wave():
    """Face-point value error of the linear reconstruction falls like k^5, its derivative like k^4
    (fifth-order claim)."""
    errs = []
    kdir = np.array([1.0, 0.7, -0.4]); kdir /= np.linalg.norm(kdir)
    for ppw in (10, 20):
        k = 2 * math.pi / ppw * kdir
        fn = lambda x, y, z: np.sin(k[0] * x + k[1] * y + k[2] * z + 0.3)
        grad = lambda x, y, z: tuple(k[a] * np.cos(k[0] * x + k[1] * y + k[2] * z + 0.3) for a in range(3))
        q0, d = rd.data_vector(fn, grad)
        _, _, _, _, val, gref = ref.recon_reference(LIN, d)
        pts = rd.gauss_points()
        ev = max(abs(q0 + val[i] - fn(*pts[i])) for i in range(24))
        eg = max(abs(gref[i][a] - grad(*pts[i])[a]) for i in range(24) for a in range(3))
        errs.append((ev, eg))
    order_v = math.log2(errs[0][0] / errs[1][0]); order_g = math.log2(errs[0][1] / errs[1][1])
    assert 4.6 < order_v < 6.5, errs
    assert 3.6 < order_g < 5.5, errs


def test_linear_polynomials_closed_form():
    """Eq. 15: P_m is strict on Q_{1,m} and least squares on the 8 perpendicular line derivatives -> the normal
    slope is the average difference, each tangential slope the mean of the 4 line differences of that axis."""
    rng = np.random.default_rng(5)
    d = rng.standard_normal(72)
    _, b, _, om, _, _ = ref.recon_reference(LIN, d)
    for m in range(6):
        ax = m // 2; sgn = 1.0 if m % 2 == 0 else -1.0
        # neighbour average of P_m = Q0 + b.xi over the cube at offset sgn*e_ax is Q0 + sgn*b[ax]
        assert abs(sgn * b[m, ax] - d[m]) < 1e-14
        for e in rd.other_axes(ax):
            # LS on four equations b_e = D_s (unscaled) -> mean
            assert abs(b[m, e] - d[60 + 4 * e:64 + 4 * e].mean() / 3.0) < 1e-14
    np.testing.assert_allclose(om, 1.0 / 6.0)


def test_geno_limits():
    """Eq. 16 and PAPER.md:223-246: smooth, well-resolved data -> chi = 1 to 1e-6 (Table 2 = Table 1 at >= 20^3);
    a jump across a face -> chi -> small, weights concentrate on the smooth side (ENO property)."""
    k = 2 * math.pi / 20 * np.array([1.0, 1.0, 1.0])        # the 20^3 sine of the accuracy test in reference units
    fn = lambda x, y, z: 1 + 0.2 * np.sin(k[0] * x + k[1] * y + k[2] * z + 0.9)
    grad = lambda x, y, z: tuple(0.2 * k[a] * np.cos(k[0] * x + k[1] * y + k[2] * z + 0.9) for a in range(3))
    q0, d = rd.data_vector(fn, grad)
    _, _, chi, om, _, _ = ref.recon_reference(NL, d)
    assert 1 - chi < 1e-5
    # jump at x = +1/2: only the +x neighbours differ
    d = np.zeros(72)
    d[0] = 1.0                                            # face neighbour +x
    for n, (o, _) in enumerate(rd.edge_offsets()):
        if o[0] == 1:
            d[6 + n] = 1.0
    a, b, chi, om, val, gref = ref.recon_reference(NL, d)
    assert chi < 0.9
    assert om[0] < 1e-8 and abs(om[1:].sum() - 1) < 1e-12    # the stencil across the jump gets no weight
    # with chi -> 0 the value would be flat; check the blended value is between the P4 value and the ENO value
    _, _, _, _, val_lin, _ = ref.recon_reference(LIN, d)
    assert np.all(np.abs(val) <= np.abs(val_lin) + 1e-14)


def test_smoothness_indicator_quadrature():
    """IS = sum_l int_cell (D^l P4)^2, per derivative order, against numerical quadrature."""
    didx, _ = ref.basis()
    rng = np.random.default_rng(7)
    a = rng.standard_normal(34)
    IS = ref.smoothness(a)
    x, w = np.polynomial.legendre.leggauss(6); x = 0.5 * x; w = 0.5 * w
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij"); W = w[:, None, None] * w[None, :, None] * w[None, None, :]
    from itertools import product
    out = np.zeros(4)
    for l in product(range(5), repeat=3):
        o = sum(l)
        if not 1 <= o <= 4:
            continue
        val = np.zeros_like(X)
        for c, d in zip(a, didx):
            e = d - np.array(l)
            if (e < 0).any():
                continue
            val += c * X ** e[0] * Y ** e[1] * Z ** e[2] / (math.factorial(e[0]) * math.factorial(e[1]) * math.factorial(e[2]))
        out[o - 1] += (W * val * val).sum()
    np.testing.assert_allclose(IS, out, rtol=1e-11)


def test_P2_cube_symmetry():
    """Permuting / reflecting the field permutes the outputs: M, E and every ordering table respect the cube group."""
    rng = np.random.default_rng(11)
    coef = {d: rng.standard_normal() for d in rd.quartic_multi_indices()}
    coef[(5, 1, 0)] = 0.3; coef[(0, 2, 4)] = -0.2          # beyond quartic, so the LS part is exercised
    fn, grad = rd.poly_fn(coef)
    q0, d = rd.data_vector(fn, grad)
    _, _, _, _, val, gref = ref.recon_reference(LIN, d)
    pts = rd.gauss_points()
    # symmetry: (x,y,z) -> (y,-z,x)
    def T(p):
        return np.array([p[1], -p[2], p[0]])
    fn2 = lambda x, y, z: fn(y, -z, x)
    def grad2(x, y, z):
        g = grad(y, -z, x)
        return (g[2], g[0], -g[1])
    q02, d2 = rd.data_vector(fn2, grad2)
    _, _, _, _, val2, gref2 = ref.recon_reference(LIN, d2)
    assert abs(q0 - q02) < 1e-13
    for i, p in enumerate(pts):
        tp = T(p)
        j = int(np.argmin(np.abs(pts - tp).sum(1)))
        assert np.abs(pts[j] - tp).max() < 1e-14
        assert abs(val2[i] - val[j]) < 1e-11
        g = gref[j]
        np.testing.assert_allclose(gref2[i], [g[2], g[0], -g[1]], atol=1e-10)

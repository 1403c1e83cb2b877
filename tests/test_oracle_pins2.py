"""Round-2 pins of oracle functions that had none ("parity unpinned"): the J0^T data transform and J0^-T
back-transform on non-orthogonal cells, the time step (reading S3), the Prandtl fix
on F^n AND F_t^n (reading F2) against a brute-force velocity-space heat flux, and the positivity fallback (reading R9).
CPU only."""
import itertools
import math

import numpy as np
import pytest

from oracle import ref
from paper_2508_08965_b200 import inputs
from tests.test_oracle_gks import GAMMA, K, Quad, _prim, _slopes_bf, cons

G = 0.5 / math.sqrt(3.0)


# ----------------------------------------------------------------------------- J0^T / J0^-T on an affine sheared mesh
def _poly(rng, const):
    coef = {d: 0.05 * rng.standard_normal() for d in itertools.product(range(5), repeat=3) if 1 <= sum(d) <= 4}
    coef[(0, 0, 0)] = const

    def val(x):
        return sum(c * x[0] ** d[0] * x[1] ** d[1] * x[2] ** d[2] for d, c in coef.items())

    def grad(x):
        g = []
        for r in range(3):
            s = 0.0
            for d, c in coef.items():
                if d[r] > 0:
                    e = list(d); e[r] -= 1
                    s = s + c * d[r] * x[0] ** e[0] * x[1] ** e[1] * x[2] ** e[2]
            g.append(s + 0 * x[0])
        return np.array(g)
    return val, grad


def test_sheared_mesh_quartic_exactness():
    """Reading R4: on an AFFINE mesh the reference-cell reconstruction is exact for physical-space quartics.  The mesh has
    a constant NON-SYMMETRIC J0 (x = A xi), so a transposed J0 in the data transform (grad Q)' = J0^T grad Q
     or in the back-transform grad Q = J0^-T grad' Q breaks the exactness.  Data: exact cell
    averages and cell-averaged PHYSICAL gradients by tensor Gauss quadrature, exact line differences."""
    n, h = 5, 0.4
    A = inputs.SHEAR
    nodes = inputs.sheared_nodes(n, h)
    rng = np.random.default_rng(12)
    polys = [_poly(rng, c) for c in (10.0, 0.3, -0.2, 0.1, 100.0)]          # rho and E far from zero: no fallback
    gx, gw = np.polynomial.legendre.leggauss(3); gx = 0.5 * gx; gw = 0.5 * gw
    Q = np.zeros((5, n, n, n)); Gd = np.zeros((5, 3, n, n, n)); D = np.zeros((5, 12, n, n, n))
    J = A * h

    def phys(i, j, k, xi):          # physical position of reference point xi of cell (i, j, k)
        return nodes[:, k, j, i] + J @ (np.asarray(xi) + 0.5)
    lines = []
    for ax in range(3):
        o1, o2 = [a for a in range(3) if a != ax]
        for a in (0, 1):
            for b in (0, 1):
                x1 = [0.0] * 3; x2 = [0.0] * 3
                x1[ax] = -0.5; x2[ax] = 0.5; x1[o1] = x2[o1] = G if a else -G; x1[o2] = x2[o2] = G if b else -G
                lines.append((x1, x2))
    for k in range(n):
        for j in range(n):
            for i in range(n):
                for v, (val, grad) in enumerate(polys):
                    for a, wa in zip(gx, gw):
                        for b, wb in zip(gx, gw):
                            for c, wc in zip(gx, gw):
                                x = phys(i, j, k, (a, b, c))
                                Q[v, k, j, i] += wa * wb * wc * val(x)
                                Gd[v, :, k, j, i] += wa * wb * wc * grad(x)
                    for s, (x1, x2) in enumerate(lines):
                        D[v, s, k, j, i] = val(phys(i, j, k, x2)) - val(phys(i, j, k, x1))
    s = ref.RefSolver(nodes, ref.make_params(nonlinear=0))
    s.set_state(Q, Gd, D)
    pv, chi = s.reconstruct()
    assert s.fallback_stats()[0] == 0
    _, gp = ref.basis()
    worst_v = worst_g = 0.0
    for k in range(1, n - 1):            # cells whose stencil does not wrap (a polynomial is not periodic)
        for j in range(1, n - 1):
            for i in range(1, n - 1):
                for p in range(24):
                    x = phys(i, j, k, gp[p])
                    for v, (val, grad) in enumerate(polys):
                        worst_v = max(worst_v, abs(pv[k, j, i, p, v] - val(x)))
                        worst_g = max(worst_g, np.abs(pv[k, j, i, p, 5 + 3 * v:8 + 3 * v] - grad(x)).max())
    assert worst_v < 1e-11 and worst_g < 1e-10, (worst_v, worst_g)
    # negative control: the same data with G transposed-transformed (J0 instead of J0^T applied by hand) is NOT exact
    Gbad = np.einsum("ra,vaijk->vrijk", A @ np.linalg.inv(A.T), Gd)
    s.set_state(Q, Gbad, D)
    pv2, _ = s.reconstruct()
    assert np.abs(pv2[2, 2, 2] - pv[2, 2, 2]).max() > 1e-4
    s.close()


def test_one_step_on_the_sheared_mesh_is_frame_consistent():
    """One short step of a smooth flow on the sheared mesh: the change of the cell-averaged mass equals -div(rho U), with
    the divergence evaluated spectrally in the periodic coordinates, up to a truncation error that falls under refinement
    (a wrong J0 transform gives an O(1) discrepancy that does not fall)."""
    errs = []
    for n in (8, 16):
        w = inputs.workload("tgv_shear", n)
        s = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=0)); s.set_state(w["Q"])
        dt = 0.25 * s.compute_dt(0.5)
        s.step(dt)
        Q1 = s.get_state()[0]
        # time derivative of the mass from the divergence of the momentum, evaluated spectrally in the periodic coordinates
        xi = np.linalg.solve(inputs.SHEAR, inputs.cell_centroids(w["nodes"]).reshape(3, -1)).reshape(3, n, n, n)
        Ainv = np.linalg.inv(inputs.SHEAR)
        m = w["Q"][1:4]
        kk = np.fft.fftfreq(n, 1.0 / n)
        KZ, KY, KX = np.meshgrid(kk, kk, kk, indexing="ij")
        kxi = [KX, KY, KZ]
        div = 0.0
        for r in range(3):          # d m_r / d x_r = sum_a (A^-1)[a][r] d m_r / d xi_a
            mh = np.fft.fftn(m[r])
            for a in range(3):
                div = div + Ainv[a, r] * np.real(np.fft.ifftn(1j * kxi[a] * mh))
        errs.append(np.abs((Q1[0] - w["Q"][0]) / dt + div).max())
        s.close()
    assert errs[1] < errs[0] / 3.0 and errs[1] < 0.02, errs


# ----------------------------------------------------------------------------- time step (reading S3)
def _dt_by_hand(J, rho, U, p, cfl, mu=0.0):
    """Uniform state on a mesh of identical parallelepiped cells with edge vectors J[:, a]: the hand calculation."""
    a = [J[:, 0], J[:, 1], J[:, 2]]
    vol = abs(np.linalg.det(J))
    S = [np.cross(a[1], a[2]), np.cross(a[2], a[0]), np.cross(a[0], a[1])]
    c = math.sqrt(GAMMA * p / rho)
    hs = [vol / np.linalg.norm(Sd) for Sd in S]
    rate = sum((abs(np.dot(U, Sd)) / np.linalg.norm(Sd) + c) / hd for Sd, hd in zip(S, hs))
    dt = cfl / rate
    if mu > 0:
        dt = min(dt, cfl * min(hs) ** 2 / (3.0 * mu / rho))
    return dt


@pytest.mark.parametrize("mesh", ["cart", "shear"])
def test_compute_dt_by_hand(mesh):
    rho, U, p, cfl = 1.3, np.array([0.4, -0.7, 0.2]), 0.9, 0.45
    if mesh == "cart":
        ni, nj, nk = 5, 4, 6
        nodes = inputs.cartesian_nodes((ni, nj, nk), 0.0, 1.0)
        nodes[0] *= 0.5; nodes[1] *= 0.6; nodes[2] *= 1.2          # hx = 0.1, hy = 0.15, hz = 0.2
        J = np.diag([0.1, 0.15, 0.2])
        assert abs(_dt_by_hand(J, rho, U, p, cfl) - cfl / ((0.4 + math.sqrt(1.4 * 0.9 / 1.3)) / 0.1 + (0.7 + math.sqrt(1.4 * 0.9 / 1.3)) / 0.15
                                                               + (0.2 + math.sqrt(1.4 * 0.9 / 1.3)) / 0.2)) < 1e-15
    else:
        ni = nj = nk = 5
        nodes = inputs.sheared_nodes(5, 0.17)
        J = inputs.SHEAR * 0.17
    one = np.ones((nk, nj, ni))
    Q = inputs.prim_to_cons(rho * one, U[0] * one, U[1] * one, U[2] * one, p * one)
    s = ref.RefSolver(nodes, ref.make_params()); s.set_state(Q)
    assert abs(s.compute_dt(cfl) / _dt_by_hand(J, rho, U, p, cfl) - 1) < 1e-13
    s.close()
    # viscous cap active (dt = CFL h^2/(3 nu)), constant viscosity and the power law
    for om, Tref in ((0.0, 1.0), (0.76, 0.5)):
        mu_ref = 0.5
        mu = mu_ref * ((p / rho) / Tref) ** om
        s = ref.RefSolver(nodes, ref.make_params(mu_ref=mu_ref, visc_omega=om, T_ref=Tref, Pr=0.72)); s.set_state(Q)
        by_hand = _dt_by_hand(J, rho, U, p, cfl, mu)
        assert by_hand < 0.7 * _dt_by_hand(J, rho, U, p, cfl)          # the cap decides
        assert abs(s.compute_dt(cfl) / by_hand - 1) < 1e-13
        s.close()
    # the minimum is over cells: one faster cell decides
    Q2 = Q.copy(); Uf = np.array([2.5, 0.1, -0.3])
    Q2[:, 2, 1, 3] = inputs.prim_to_cons(rho, Uf[0], Uf[1], Uf[2], p)
    s = ref.RefSolver(nodes, ref.make_params()); s.set_state(Q2)
    assert abs(s.compute_dt(cfl) / _dt_by_hand(J, rho, Uf, p, cfl) - 1) < 1e-13
    s.close()


# ----------------------------------------------------------------------------- Prandtl fix on F^n and F_t^n (reading F2)
def test_prandtl_fix_on_flux_and_time_derivative_bruteforce():
    """Reading F2: energy flux += (1/Pr - 1) q with q the heat flux OF THE SAME DISTRIBUTION.  Brute force: q(t) is
    integrated from its kinetic definition q = int (u - U0) ((u-U0)^2 + (v-V0)^2 + (w-W0)^2 + xi^2)/2 f dXi with f of Eq. 5
    (every term by tensor quadrature over velocity space, time integrals by Gauss-Legendre), then linearised in time like
    the flux.  F(Pr) - F(Pr = 1) must equal (1/Pr - 1) q for BOTH F^n and F_t^n (P9 pinned
    out[0] only).  Discontinuous states with slopes, physical + numerical collision time."""
    rng = np.random.default_rng(5)
    WL = cons(1.0, [0.35, -0.2, 0.1], 1.0); WR = cons(0.85, [0.2, 0.1, -0.05], 0.75)
    gL = 0.3 * rng.standard_normal((5, 3)); gR = 0.3 * rng.standard_normal((5, 3))
    n = np.array([1.0, 0, 0]); t1 = np.array([0, 1.0, 0])
    dt = 0.05; c2 = 2.0; mu = 4e-3; Pr = 0.72
    one = ref.flux_point(ref.make_params(gamma=GAMMA, Pr=1.0, mu_ref=mu, tau_c2=c2), dt, WL, gL, WR, gR, n, t1)
    fix = ref.flux_point(ref.make_params(gamma=GAMMA, Pr=Pr, mu_ref=mu, tau_c2=c2), dt, WL, gL, WR, gR, n, t1)
    # only the energy flux and its time derivative change; interface values do not
    for q in range(6):
        comp = slice(0, 4) if q < 2 else slice(0, 5)
        np.testing.assert_allclose(fix[q][comp], one[q][comp], rtol=1e-13, atol=1e-14)
    # --- brute force of the heat flux ---
    rl, Ul, ll = _prim(WL); rr, Ur, lr = _prim(WR)
    ql, qlp = Quad(*Ul, ll, 0), Quad(*Ul, ll, +1)
    qr, qrn = Quad(*Ur, lr, 0), Quad(*Ur, lr, -1)
    pl, plp, pr, prn = ql.psi(), qlp.psi(), qr.psi(), qrn.psi()
    aL = [_slopes_bf(ql, pl, gL[:, d] / rl) for d in range(3)]
    aR = [_slopes_bf(qr, pr, gR[:, d] / rr) for d in range(3)]
    W0 = np.array([rl * qlp.integ(plp[a]) + rr * qrn.integ(prn[a]) for a in range(5)])
    r0, U0, l0 = _prim(W0); q0 = Quad(*U0, l0, 0); p0 = q0.psi()
    dot = lambda a, ps: sum(a[i] * ps[i] for i in range(5))
    a0 = []
    for d in range(3):
        dW0 = np.array([rl * qlp.integ(dot(aL[d], plp) * plp[a]) + rr * qrn.integ(dot(aR[d], prn) * prn[a]) for a in range(5)])
        a0.append(_slopes_bf(q0, p0, dW0 / r0))

    def tslope(q, ps, a):
        adv = dot(a[0], ps) * q.u + dot(a[1], ps) * q.v + dot(a[2], ps) * q.w
        return _slopes_bf(q, ps, np.array([-q.integ(adv * ps[al]) for al in range(5)]))
    AL, AR, A0 = tslope(ql, pl, aL), tslope(qr, pr, aR), tslope(q0, p0, a0)
    pL_, pR_, p0_ = rl / (2 * ll), rr / (2 * lr), r0 / (2 * l0)
    tau = mu / p0_ + c2 * abs(pL_ - pR_) / abs(pL_ + pR_) * dt

    def heat_weight(q):
        cu, cv, cw = q.u - U0[0], q.v - U0[1], q.w - U0[2]
        return cu * 0.5 * (cu ** 2 + cv ** 2 + cw ** 2 + q.x1 ** 2 + q.x2 ** 2)
    h0, hl, hr = heat_weight(q0), heat_weight(qlp), heat_weight(qrn)
    tx, tw = np.polynomial.legendre.leggauss(14)

    def heat_integral(T):
        s = 0.0
        for x, w in zip(tx, tw):
            t = 0.5 * T * (x + 1); wt = 0.5 * T * w; e = math.exp(-t / tau)
            f0 = r0 * ((1 - e) + ((t + tau) * e - tau) * (dot(a0[0], p0) * q0.u + dot(a0[1], p0) * q0.v + dot(a0[2], p0) * q0.w)
                       + (t - tau + tau * e) * dot(A0, p0))
            fl = rl * e * (1 - (tau + t) * (dot(aL[0], plp) * qlp.u + dot(aL[1], plp) * qlp.v + dot(aL[2], plp) * qlp.w) - tau * dot(AL, plp))
            fr = rr * e * (1 - (tau + t) * (dot(aR[0], prn) * qrn.u + dot(aR[1], prn) * qrn.v + dot(aR[2], prn) * qrn.w) - tau * dot(AR, prn))
            s += wt * (q0.integ(f0 * h0) + qlp.integ(fl * hl) + qrn.integ(fr * hr))
        return s
    I1, I2 = heat_integral(dt), heat_integral(dt / 2)
    qn = (4 * I2 - I1) / dt; qt = 4 * (I1 - 2 * I2) / dt ** 2
    assert abs(qn) > 1e-3 and abs(qt) > 1e-3                       # the test sees both
    np.testing.assert_allclose(fix[0][4] - one[0][4], (1 / Pr - 1) * qn, rtol=1e-7)
    np.testing.assert_allclose(fix[1][4] - one[1][4], (1 / Pr - 1) * qt, rtol=1e-6)


# ----------------------------------------------------------------------------- positivity fallback (reading R9)
@pytest.mark.parametrize("name", ["jump_blob", "jump_oblique_linear"])
def test_positivity_fallback_fires_by_an_O1_margin_and_stays_conservative(name):
    w = inputs.workload(name)
    s = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=w["nonlinear"])); s.set_state(w["Q"])
    pv, _ = s.reconstruct()
    nfall, min_rho, min_pe = s.fallback_stats()
    assert nfall > 200 and min_rho < -0.5, (nfall, min_rho, min_pe)          # rho of a replaced state: below -0.5 rho_cell
    # the replaced points carry the cell average and zero gradients (reading R9), all others are untouched
    Qc = np.moveaxis(w["Q"], 0, -1)[:, :, :, None, :]
    flat = (np.abs(pv[..., 5:]).max(-1) == 0) & (np.abs(pv[..., :5] - Qc).max(-1) == 0)
    rho = pv[..., 0]; adm = pv[..., 0] * pv[..., 4] - 0.5 * (pv[..., 1] ** 2 + pv[..., 2] ** 2 + pv[..., 3] ** 2)
    assert (rho > 0).all() and (adm > 0).all()                              # every state handed to the flux is admissible
    _, Gb, Db = s.get_state()
    nonuniform = (np.abs(Db).max(axis=(0, 1)) > 0) | (np.abs(Gb).max(axis=(0, 1)) > 0)
    assert (flat & nonuniform[..., None]).sum() == nfall
    tot0 = w["Q"].sum(axis=(1, 2, 3))
    for _ in range(3):
        s.step(s.compute_dt(w["cfl"]))
    Q1 = s.get_state()[0]
    np.testing.assert_allclose(Q1.sum(axis=(1, 2, 3)), tot0, rtol=1e-13, atol=1e-12)
    assert Q1[0].min() > 0
    s.close()


# ----------------------------------------------------------------------------- GENO weights on worked examples
def test_geno_formulas_on_worked_examples():
    """The blending formulas as the paper prints them, evaluated BY HAND on data for which every ingredient has a closed form.
    (i) omega_m = (d_m/(IS_m + eps)^5)/sum: face-neighbour differences g_m with all line differences zero
    give b^m = +-g_m e_axis, IS_m = g_m^2, so omega_0/omega_1 = ((g_1^2 + eps)/(g_0^2 + eps))^5: the exponent 5 and the
    normalisation.  (ii) chi for the 1-D polynomial P = a xi + c xi^3 (reproduced exactly by the quartic): by hand
    int P'^2 = a^2 + a c/2 + 9 c^2/80, int P''^2 = 3 c^2, int P'''^2 = 36 c^2, so IS^L, IS^H and (reading G2) IS^tau are known
    numbers; alpha^{H,L} = 1 + (IS^tau/(IS^{H,L} + eps))^2, alpha = 2 alpha^H/(alpha^H + alpha^L), chi = tanh(C alpha)/tanh C
    (C = 5 by reading G3): the exponent r = 2, the roles of H and L, the tanh map."""
    from tests import refdata as rd
    from tests.test_oracle_recon import NL
    g = np.array([0.3, -0.5, 0.2, 0.7, -0.4, 0.25])
    d = np.zeros(72); d[:6] = g
    _, b, _, om, _, _ = ref.recon_reference(NL, d)
    eps = 1e-15
    for m in range(6):
        assert abs(np.abs(b[m]).sum() - abs(g[m])) < 1e-15                  # b^m = +-g_m along the face normal only
    w = (1.0 / 6.0) / (g ** 2 + eps) ** 5
    np.testing.assert_allclose(om, w / w.sum(), rtol=1e-12)
    assert abs(om[0] / om[1] - ((g[1] ** 2 + eps) / (g[0] ** 2 + eps)) ** 5) < 1e-10 * om[0] / om[1]
    for a_, c_ in ((1.0, 0.5), (0.2, 1.5), (1.0, 0.01)):
        fn, grad = rd.poly_fn({(1, 0, 0): a_, (3, 0, 0): c_})
        _, d = rd.data_vector(fn, grad)
        _, _, chi, _, _, _ = ref.recon_reference(NL, d)
        is1 = a_ * a_ + a_ * c_ / 2.0 + 9.0 * c_ * c_ / 80.0; is2 = 3.0 * c_ * c_; is3 = 36.0 * c_ * c_
        ish = is1 + is2 + is3; ist = is3
        ah = 1.0 + (ist / (ish + eps)) ** 2; al = 1.0 + (ist / (is1 + eps)) ** 2
        alpha = 2.0 * ah / (ah + al)
        assert abs(chi - math.tanh(5.0 * alpha) / math.tanh(5.0)) < 1e-11, (a_, c_, chi)
    assert chi > 0.999                                                       # nearly linear data: the quartic is kept


# ----------------------------------------------------------------------------- reading F3: the one-sided ingredients
def _euler_flux(W, d):
    rho = W[0]; U = W[1:4] / rho
    p = (GAMMA - 1.0) * (W[4] - 0.5 * rho * U @ U)
    F = W * U[d]
    F[1 + d] += p; F[4] += p * U[d]
    return F


def test_F3_one_sided_part_is_the_euler_time_derivative():
    """Reading F3: the interface values handed to the two cells are V^s = (1-w) Q^e + w W^s and
    Q_t^s = (1-w) Q_t^e + w int psi A^s g_s, w = exp(-dt/tau0), tau0 = c2 |pl-pr|/|pl+pr| dt, with ONE equilibrium part Q^e,
    Q_t^e for both sides.  Hence V^l - V^r = w (W^l - W^r) and Q_t^l - Q_t^r = w (dW^l/dt - dW^r/dt), where the compatibility
    condition makes the one-sided time derivative the Euler equations applied to the one-sided polynomial,
    dW/dt = - sum_d dF_d(W)/dx_d: written here from the textbook Euler flux (central differences of F_d along the slope, no
    kinetic arithmetic).  Pins sign, frame rotation and the slope -> time-slope solve of the one-sided part, and the weight.
    (The sum of the two sides contains Q^e, which P7b pins by brute force; the limit w -> 1 does not isolate the one-sided
    part: (1-w) Q^e tends to dt times a slope term, because Q^e grows like tau.)"""
    rng = np.random.default_rng(11)
    from tests.test_oracle_gks import random_frame

    def euler_dt(W, g):
        eps = 1e-6
        r = np.zeros(5)
        for d in range(3):
            r -= (_euler_flux(W + eps * g[:, d], d) - _euler_flux(W - eps * g[:, d], d)) / (2 * eps)
        return r
    for c2 in (5.0, 0.8, 60.0):
        n, t1 = random_frame(rng)
        WL = cons(1.0, [0.35, -0.2, 0.1], 1.0); WR = cons(0.5, [0.15, 0.1, -0.05], 0.3)
        gL = 0.3 * rng.standard_normal((5, 3)); gR = 0.3 * rng.standard_normal((5, 3))
        eL, eR = euler_dt(WL, gL), euler_dt(WR, gR)
        out = ref.flux_point(ref.make_params(gamma=GAMMA, Pr=1.0, mu_ref=0.0, tau_c1=0.05, tau_c2=c2), 0.01, WL, gL, WR, gR, n, t1)
        w = math.exp(-1.0 / (c2 * abs(1.0 - 0.3) / (1.0 + 0.3)))
        np.testing.assert_allclose(out[2] - out[4], w * (WL - WR), rtol=1e-10, atol=1e-11)
        np.testing.assert_allclose(out[3] - out[5], w * (eL - eR), rtol=1e-7, atol=1e-8)
        assert np.abs(eL - eR).max() > 1e-2 and w > 0.09          # the two sides really differ, the weight is not ~0


# ----------------------------------------------------------------------------- reading S2: bootstrap of G and D
def test_S2_bootstrap_symbol_on_the_sheared_mesh():
    """Reading S2 (the paper is silent on the initial derivative dof): G and D from the fourth-order central difference
    (8 (Q+1 - Q-1) - (Q+2 - Q-2))/12 of the cell averages along each index direction, G = J0^-T of that reference-space
    vector, the four line differences of an axis = its component.  For a plane wave in the lattice
    coordinates, Q = 2 + sin(a . xi), the difference quotient of the cell averages has the closed form
    A cos(a . xi_c) (8 sin(a_r h) - sin(2 a_r h))/6 with A the product of the three sinc factors of the cell average: pins
    the stencil weights, their sign, the axis -> line-difference placement and, on the non-symmetric affine mesh, J0^-T
    against a transposed or missing transform."""
    n = 12; h = 2.0 * math.pi / n
    nodes = inputs.sheared_nodes(n, h)
    a = np.array([1.0, 2.0, -1.0])
    k, j, i = np.meshgrid(np.arange(n) + 0.5, np.arange(n) + 0.5, np.arange(n) + 0.5, indexing="ij")
    phase = a[0] * i * h + a[1] * j * h + a[2] * k * h
    amp = np.prod([math.sin(0.5 * ar * h) / (0.5 * ar * h) for ar in a])
    Q = np.zeros((5, n, n, n))
    Q[0] = 2.0 + amp * np.sin(phase)
    Q[1] = 0.3 * Q[0]; Q[2] = -0.1 * Q[0]; Q[3] = 0.2 * Q[0]; Q[4] = 3.0 + 0.5 * amp * np.cos(phase)
    s = ref.RefSolver(nodes, ref.make_params()); s.set_state(Q)
    _, Gb, Db = s.get_state(); s.close()
    sym = np.array([(8.0 * math.sin(ar * h) - math.sin(2.0 * ar * h)) / 6.0 for ar in a])
    J0 = inputs.SHEAR * h                                  # columns = N2-N1, N3-N1, N4-N1 (reading R1)
    for v, (c_sin, c_cos) in enumerate([(1.0, 0.0), (0.3, 0.0), (-0.1, 0.0), (0.2, 0.0), (0.0, 0.5)]):
        dphase = amp * (c_sin * np.cos(phase) - c_cos * np.sin(phase))          # d/d(phase) of variable v's wave
        dref = sym[:, None, None, None] * dphase[None]                         # reference-space derivative per index direction
        Gexp = np.einsum("rs,skji->rkji", np.linalg.inv(J0).T, dref)
        np.testing.assert_allclose(Gb[v], Gexp, atol=2e-13)
        for r in range(3):
            for q in range(4):
                np.testing.assert_allclose(Db[v, 4 * r + q], dref[r], atol=2e-13)
    # negative control: the transposed transform differs by far more than the tolerance
    assert np.abs(np.einsum("rs,skji->rkji", np.linalg.inv(J0), dref) - Gexp).max() > 1e-2

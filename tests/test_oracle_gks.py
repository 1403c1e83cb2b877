"""Pins of the oracle's gas-kinetic interface solver (Eq. 1-7, 330-352) against quadrature,
closed forms and invariants.  CPU only.  Pin numbers P7.. follow DESIGN.md section 4."""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import ref

GAMMA = 1.4
K = (5 - 3 * GAMMA) / (GAMMA - 1)            # = 2 internal dof


def cons(rho, U, p):
    U = np.asarray(U, float)
    return np.array([rho, *(rho * U), p / (GAMMA - 1) + 0.5 * rho * U @ U])


def cons_grad(rho, U, p, drho, dU, dp):
    """Conservative gradients [5][3] from primitive gradients drho[3], dU[3 comps][3 dirs], dp[3]."""
    U = np.asarray(U, float); drho = np.asarray(drho, float); dU = np.asarray(dU, float); dp = np.asarray(dp, float)
    g = np.zeros((5, 3))
    g[0] = drho
    for c in range(3):
        g[1 + c] = drho * U[c] + rho * dU[c]
    g[4] = dp / (GAMMA - 1) + 0.5 * drho * (U @ U) + rho * (U @ dU)
    return g


def euler_flux(W, n):
    rho = W[0]; U = W[1:4] / rho; p = (GAMMA - 1) * (W[4] - 0.5 * rho * U @ U); un = U @ n
    return np.array([rho * un, *(rho * U * un + p * n), (W[4] + p) * un])


def random_frame(rng):
    n = rng.standard_normal(3); n /= np.linalg.norm(n)
    t = rng.standard_normal(3); t -= (t @ n) * n; t /= np.linalg.norm(t)
    return n, t


# ----------------------------------------------------------------------------- P7: moments
def test_P7_moments_vs_quadrature():
    U, lam = 0.37, 0.83
    full, pos, neg = ref.moments(U, lam)
    g1 = lambda u: math.sqrt(lam / math.pi) * math.exp(-lam * (u - U) ** 2)
    for n in range(7):
        assert abs(integrate.quad(lambda u: u ** n * g1(u), -np.inf, np.inf)[0] - full[n]) < 1e-9
        assert abs(integrate.quad(lambda u: u ** n * g1(u), 0, np.inf)[0] - pos[n]) < 1e-9
        assert abs(integrate.quad(lambda u: u ** n * g1(u), -np.inf, 0)[0] - neg[n]) < 1e-9
    np.testing.assert_allclose(pos + neg, full, rtol=1e-13)


class Quad:
    """Tensor quadrature over (u, v, w, xi1, xi2) for a Maxwellian (per unit density), K = 2."""

    def __init__(self, U, V, W, lam, half=0, nu=64):
        gh_x, gh_w = np.polynomial.hermite.hermgauss(8)
        s = 1.0 / math.sqrt(lam)
        def gh(c):
            return c + s * gh_x, gh_w / math.sqrt(math.pi)
        if half == 0:
            gh_xu, gh_wu = np.polynomial.hermite.hermgauss(12)
            u, wu = U + s * gh_xu, gh_wu / math.sqrt(math.pi)
        else:
            x, w = np.polynomial.legendre.leggauss(nu)
            lo, hi = (0.0, max(U, 0) + 9 * s) if half > 0 else (min(U, 0) - 9 * s, 0.0)
            u = 0.5 * (hi - lo) * x + 0.5 * (hi + lo); wu = 0.5 * (hi - lo) * w * math.sqrt(lam / math.pi) * np.exp(-lam * (u - U) ** 2)
        v, wv = gh(V); w_, ww = gh(W); x1, w1 = gh(0.0); x2, w2 = gh(0.0)
        self.u, self.v, self.w, self.x1, self.x2 = np.meshgrid(u, v, w_, x1, x2, indexing="ij")
        self.wt = np.einsum("a,b,c,d,e->abcde", wu, wv, ww, w1, w2)

    def psi(self):
        return [np.ones_like(self.u), self.u, self.v, self.w,
                0.5 * (self.u ** 2 + self.v ** 2 + self.w ** 2 + self.x1 ** 2 + self.x2 ** 2)]

    def integ(self, fn):
        return float((self.wt * fn).sum())


def test_P7_moment_apsi_vs_quadrature():
    U, V, W, lam = 0.37, -0.21, 0.11, 0.83
    a = np.array([0.3, -0.7, 0.2, 0.5, -0.4])
    for half in (0, 1, -1):
        q = Quad(U, V, W, lam, half)
        psi = q.psi(); apsi = sum(a[i] * psi[i] for i in range(5))
        for (i, j, k) in [(0, 0, 0), (1, 0, 0), (2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 1, 0), (0, 0, 1)]:
            out = ref.moment_apsi(a, i, j, k, U, V, W, lam, K, half)
            bf = [q.integ(apsi * q.u ** i * q.v ** j * q.w ** k * psi[al]) for al in range(5)]
            np.testing.assert_allclose(out, bf, rtol=2e-10, atol=2e-11)


def test_microslope_inverts_moment_matrix():
    U, V, W, lam = 0.37, -0.21, 0.11, 0.83
    q = Quad(U, V, W, lam, 0); psi = q.psi()
    Mm = np.array([[q.integ(psi[a] * psi[b]) for b in range(5)] for a in range(5)])
    h = np.array([0.2, -0.5, 0.1, 0.33, 0.8])
    np.testing.assert_allclose(ref.microslope(h, U, V, W, lam, K), np.linalg.solve(Mm, h), rtol=1e-9)


# ----------------------------------------------------------------------------- P7b: brute force of Eq. 5
def _prim(W):
    rho = W[0]; U = W[1:4] / rho
    lam = (K + 3) * rho / (4 * (W[4] - 0.5 * rho * U @ U))
    return rho, U, lam


def _slopes_bf(q, psi, h):
    Mm = np.array([[q.integ(psi[a] * psi[b]) for b in range(5)] for a in range(5)])
    return np.linalg.solve(Mm, h)


def test_P7b_bruteforce_velocity_space_quadrature_of_eq5():
    """Discontinuous states with slopes: every term of Eq. 5 integrated numerically over velocity space and time,
    micro-slopes from numerical 5x5 moment systems; compared with the oracle's analytic F^n, F_t^n, Q^n, Q_t^n."""
    rng = np.random.default_rng(3)
    WL = cons(1.0, [0.35, -0.2, 0.1], 1.0); WR = cons(0.8, [0.15, 0.1, -0.05], 0.7)
    gL = 0.3 * rng.standard_normal((5, 3)); gR = 0.3 * rng.standard_normal((5, 3))
    n = np.array([1.0, 0, 0]); t1 = np.array([0, 1.0, 0])
    dt = 0.05; c1, c2 = 0.3, 2.0
    prm = ref.make_params(gamma=GAMMA, Pr=1.0, mu_ref=0.0, tau_c1=c1, tau_c2=c2)
    out = ref.flux_point(prm, dt, WL, gL, WR, gR, n, t1)
    # --- brute force ---
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
    pL_, pR_ = rl / (2 * ll), rr / (2 * lr)
    tau = c1 * dt + c2 * abs(pL_ - pR_) / abs(pL_ + pR_) * dt
    tx, tw = np.polynomial.legendre.leggauss(14)
    def integrals(T):
        IF = np.zeros(5); IQ = np.zeros(5)
        for x, w in zip(tx, tw):
            t = 0.5 * T * (x + 1); wt = 0.5 * T * w; e = math.exp(-t / tau)
            f0 = r0 * ((1 - e) + ((t + tau) * e - tau) * (dot(a0[0], p0) * q0.u + dot(a0[1], p0) * q0.v + dot(a0[2], p0) * q0.w)
                       + (t - tau + tau * e) * dot(A0, p0))
            fl = rl * e * (1 - (tau + t) * (dot(aL[0], plp) * qlp.u + dot(aL[1], plp) * qlp.v + dot(aL[2], plp) * qlp.w) - tau * dot(AL, plp))
            fr = rr * e * (1 - (tau + t) * (dot(aR[0], prn) * qrn.u + dot(aR[1], prn) * qrn.v + dot(aR[2], prn) * qrn.w) - tau * dot(AR, prn))
            for al in range(5):
                IQ[al] += wt * (q0.integ(f0 * p0[al]) + qlp.integ(fl * plp[al]) + qrn.integ(fr * prn[al]))
                IF[al] += wt * (q0.integ(f0 * p0[al] * q0.u) + qlp.integ(fl * plp[al] * qlp.u) + qrn.integ(fr * prn[al] * qrn.u))
        return IF, IQ
    IF1, IQ1 = integrals(dt); IF2, IQ2 = integrals(dt / 2)
    Fn = (4 * IF2 - IF1) / dt; Ft = 4 * (IF1 - 2 * IF2) / dt ** 2
    Qn = (4 * IQ2 - IQ1) / dt; Qt = 4 * (IQ1 - 2 * IQ2) / dt ** 2
    np.testing.assert_allclose(out[0], Fn, rtol=2e-8, atol=2e-9)
    np.testing.assert_allclose(out[1], Ft, rtol=2e-7, atol=2e-7)
    # interface values, reading F3: V^s = (1-w) Q^n + w W^s with w = exp(-dt/tau0), tau0 = c2 |pl-pr|/|pl+pr| dt
    w = math.exp(-1.0 / (c2 * abs(pL_ - pR_) / abs(pL_ + pR_)))
    np.testing.assert_allclose(out[2], (1 - w) * Qn + w * WL, rtol=2e-8, atol=2e-9)
    np.testing.assert_allclose(out[4], (1 - w) * Qn + w * WR, rtol=2e-8, atol=2e-9)
    dQL = rl * np.array([ql.integ(dot(AL, pl) * pl[al]) for al in range(5)])
    np.testing.assert_allclose(out[3], (1 - w) * Qt + w * dQL, rtol=2e-7, atol=2e-7)


# ----------------------------------------------------------------------------- P8: closed forms, inviscid
def test_P8_uniform_state_gives_euler_flux():
    rng = np.random.default_rng(0)
    W = cons(1.2, [0.4, -0.3, 0.2], 0.9); z = np.zeros((5, 3))
    for prm in (ref.make_params(), ref.make_params(mu_ref=1e-3, Pr=0.72, tau_c2=5.0), ref.make_params(tau_c1=0.05, tau_c2=5.0)):
        n, t1 = random_frame(rng)
        out = ref.flux_point(prm, 0.01, W, z, W, z, n, t1)
        np.testing.assert_allclose(out[0], euler_flux(W, n), rtol=1e-13, atol=1e-14)
        np.testing.assert_allclose(out[1], 0, atol=1e-12)
        np.testing.assert_allclose(out[2], W, rtol=1e-13); np.testing.assert_allclose(out[4], W, rtol=1e-13)
        np.testing.assert_allclose(out[3], 0, atol=1e-12)


def _euler_div(W, g):
    """-div F(W) for conservative gradients g[5][3], by a central-difference Jacobian of the Euler flux."""
    out = np.zeros(5)
    for d in range(3):
        e = np.zeros(3); e[d] = 1.0
        for v in range(5):
            h = 1e-6 * max(1.0, abs(W[v])); Wp = W.copy(); Wm = W.copy(); Wp[v] += h; Wm[v] -= h
            out -= (euler_flux(Wp, e) - euler_flux(Wm, e)) / (2 * h) * g[v, d]
    return out


def test_P8b_tau0_lax_wendroff():
    """tau = 0 (accuracy test): f = g0 (1 + A t) -> F^n = Euler flux, F_t = dF/dW . W_t with
    W_t = -div F(W), and the interface values are W and W_t."""
    rng = np.random.default_rng(1)
    W = cons(1.1, [0.5, 0.25, -0.35], 1.3); g = 0.2 * rng.standard_normal((5, 3))
    n, t1 = random_frame(rng)
    out = ref.flux_point(ref.make_params(), 0.02, W, g, W, g, n, t1)
    Wt = _euler_div(W, g)
    np.testing.assert_allclose(out[0], euler_flux(W, n), rtol=1e-12)
    Ft = np.zeros(5)
    for v in range(5):
        h = 1e-6; Wp = W.copy(); Wm = W.copy(); Wp[v] += h; Wm[v] -= h
        Ft += (euler_flux(Wp, n) - euler_flux(Wm, n)) / (2 * h) * Wt[v]
    np.testing.assert_allclose(out[1], Ft, rtol=1e-7, atol=1e-8)
    np.testing.assert_allclose(out[2], W, rtol=1e-12)
    np.testing.assert_allclose(out[3], Wt, rtol=1e-7, atol=1e-8)
    np.testing.assert_allclose(out[5], Wt, rtol=1e-7, atol=1e-8)


# ----------------------------------------------------------------------------- P9: Chapman-Enskog / Navier-Stokes
@pytest.mark.parametrize("Pr", [1.0, 0.72])
def test_P9_navier_stokes_flux(Pr):
    """Continuous state and slopes: Eq. 5 collapses to f = g0 [1 - tau (a.u + A) + t A], so F^n is exactly the
    Navier-Stokes flux with mu = tau p, bulk viscosity 2K/(3(K+3)) mu and heat conductivity mu cp / Pr."""
    rng = np.random.default_rng(4)
    rho, U, p = 1.15, np.array([0.3, -0.2, 0.45]), 0.95
    drho = 0.2 * rng.standard_normal(3); dU = 0.3 * rng.standard_normal((3, 3)); dp = 0.2 * rng.standard_normal(3)
    W = cons(rho, U, p); g = cons_grad(rho, U, p, drho, dU, dp)
    mu = 2.3e-3
    n, t1 = random_frame(rng)
    out = ref.flux_point(ref.make_params(mu_ref=mu, Pr=Pr), 0.01, W, g, W, g, n, t1)
    div = np.trace(dU)                       # dU[c][d] = dU_c/dx_d
    zeta = 2 * K / (3 * (K + 3)) * mu
    stress = mu * (dU + dU.T - 2.0 / 3.0 * div * np.eye(3)) + zeta * div * np.eye(3)
    T = p / rho; dT = dp / rho - p / rho ** 2 * drho
    cp = GAMMA / (GAMMA - 1)
    qh = -mu * cp / Pr * dT
    Fns = euler_flux(W, n)
    Fns[1:4] -= stress @ n
    Fns[4] += -U @ stress @ n + qh @ n
    np.testing.assert_allclose(out[0], Fns, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(out[2], W, rtol=1e-12)          # <(a.u + A) psi> = 0: interface value is W itself
    np.testing.assert_allclose(out[3], _euler_div(W, g), rtol=1e-7, atol=1e-8)


def test_power_law_viscosity():
    rho, U, p = 1.3, np.array([0.1, 0.2, 0.3]), 2.0
    dU = np.zeros((3, 3)); dU[1, 0] = 0.4        # dV/dx: pure shear
    W = cons(rho, U, p); g = cons_grad(rho, U, p, np.zeros(3), dU, np.zeros(3))
    n = np.array([1.0, 0, 0]); t1 = np.array([0, 1.0, 0])
    mu_ref, om, Tref = 1e-3, 0.76, 0.8
    out = ref.flux_point(ref.make_params(mu_ref=mu_ref, visc_omega=om, T_ref=Tref), 0.01, W, g, W, g, n, t1)
    mu = mu_ref * ((p / rho) / Tref) ** om
    assert abs((out[0][2] - rho * U[0] * U[1]) - (-mu * 0.4)) < 1e-13


# ----------------------------------------------------------------------------- invariants
def test_mirror_symmetry_conservation():
    """The flux seen from the other side (swap l/r, flip n) is the negative: single-valued face flux (Eq. 8)."""
    rng = np.random.default_rng(8)
    WL = cons(1.0, [0.35, -0.2, 0.1], 1.0); WR = cons(0.6, [-0.15, 0.1, 0.25], 0.5)
    gL = 0.3 * rng.standard_normal((5, 3)); gR = 0.3 * rng.standard_normal((5, 3))
    n, t1 = random_frame(rng)
    prm = ref.make_params(mu_ref=1e-3, Pr=0.72, tau_c2=5.0)
    a = ref.flux_point(prm, 0.02, WL, gL, WR, gR, n, t1)
    b = ref.flux_point(prm, 0.02, WR, gR, WL, gL, -n, t1)
    np.testing.assert_allclose(a[0], -b[0], rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(a[1], -b[1], rtol=1e-9, atol=1e-10)
    np.testing.assert_allclose(a[2], b[4], rtol=1e-11, atol=1e-13)     # own-side values swap
    np.testing.assert_allclose(a[5], b[3], rtol=1e-9, atol=1e-10)


def test_frame_invariance():
    """The result does not depend on the choice of the tangent t1 (the solver treats v and w alike)."""
    rng = np.random.default_rng(9)
    WL = cons(1.0, [0.35, -0.2, 0.1], 1.0); WR = cons(0.9, [0.3, -0.1, 0.15], 0.8)
    gL = 0.3 * rng.standard_normal((5, 3)); gR = 0.3 * rng.standard_normal((5, 3))
    n, t1 = random_frame(rng)
    t2 = np.cross(n, t1); t1b = math.cos(0.7) * t1 + math.sin(0.7) * t2
    prm = ref.make_params(mu_ref=1e-3, Pr=0.72, tau_c2=5.0)
    a = ref.flux_point(prm, 0.02, WL, gL, WR, gR, n, t1); b = ref.flux_point(prm, 0.02, WL, gL, WR, gR, n, t1b)
    np.testing.assert_allclose(a, b, rtol=1e-10, atol=1e-11)


def test_collision_time_and_interface_blend():
    """tau grows with the pressure jump; PAPER.md:330-336 (reading F3): the one-sided interface
    values move from the common equilibrium value (smooth) towards the one-sided states (strong jump)."""
    z = np.zeros((5, 3)); n = np.array([1.0, 0, 0]); t1 = np.array([0, 1.0, 0])
    prm = ref.make_params(tau_c1=0.05, tau_c2=5.0)
    WL = cons(1.0, [0.0, 0, 0], 1.0)
    small = ref.flux_point(prm, 0.01, WL, z, cons(0.999, [0, 0, 0], 0.999), z, n, t1)
    big = ref.flux_point(prm, 0.01, WL, z, cons(0.125, [0, 0, 0], 0.1), z, n, t1)
    assert np.abs(small[2] - small[4]).max() < 1e-12                 # w = exp(-1/(5*5e-4)) underflows to 0
    wgt = math.exp(-1.0 / (5.0 * 0.9 / 1.1))
    assert 0.5 < wgt < 1
    # V^l - V^r = w (W^l - W^r)
    np.testing.assert_allclose(big[2] - big[4], wgt * (WL - cons(0.125, [0, 0, 0], 0.1)), rtol=1e-12)
    # Sod-like jump: mass flux goes from the high-pressure side to the low-pressure side
    assert big[0][0] > 0

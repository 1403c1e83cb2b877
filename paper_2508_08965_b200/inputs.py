"""Seeded synthetic input generators (meshes and initial fields) shared by the tests, bench.py and the oracle legs.

This module holds none of the method's arithmetic: it only produces node coordinates, initial conservative
cell averages (and, for the sine case, exact derivative data) and the gas/option constants of each workload.
The inputs stand in for the paper's workloads (section 6; BASELINE.json configs); recipe in DESIGN.md section 5.

Array layouts (numpy, C order, fp64): nodes (3, nk+1, nj+1, ni+1); Q (5, nk, nj, ni); G (5, 3, nk, nj, ni);
D (5, 12, nk, nj, ni).  Line index s = 4*axis + 2*a + b, (a, b) selecting -g/+g on the two other axes, ascending.
"""
import math

import numpy as np

GAUSS_G = 0.5 / math.sqrt(3.0)


# ----------------------------------------------------------------------------- meshes
def cartesian_nodes(n, lo=0.0, hi=2.0 * math.pi):
    """Uniform periodic Cartesian mesh of n^3 (or (ni,nj,nk)) cells on [lo,hi]^3."""
    ni, nj, nk = (n, n, n) if np.isscalar(n) else n
    x = np.linspace(lo, hi, ni + 1); y = np.linspace(lo, hi, nj + 1); z = np.linspace(lo, hi, nk + 1)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return np.stack([X, Y, Z]).astype(np.float64)


def curvilinear_nodes(n, amp=0.1):
    """Non-orthogonal periodic mesh of BASELINE.json config 3 on [0,2pi]^3:
    x = xi + amp sin(eta) sin(zeta), y = eta + amp sin(xi) sin(zeta), z = zeta + amp sin(xi) sin(eta)."""
    c = cartesian_nodes(n, 0.0, 2.0 * math.pi)
    xi, eta, zeta = c[0], c[1], c[2]
    return np.stack([xi + amp * np.sin(eta) * np.sin(zeta),
                     eta + amp * np.sin(xi) * np.sin(zeta),
                     zeta + amp * np.sin(xi) * np.sin(eta)])


def cell_centroids(nodes):
    """Mean of the 8 nodes of each cell, shape (3, nk, nj, ni)."""
    s = 0.0
    for dk in (0, 1):
        for dj in (0, 1):
            for di in (0, 1):
                s = s + nodes[:, dk:nodes.shape[1] - 1 + dk, dj:nodes.shape[2] - 1 + dj, di:nodes.shape[3] - 1 + di]
    return s / 8.0


def prim_to_cons(rho, u, v, w, p, gamma=1.4):
    return np.stack([rho, rho * u, rho * v, rho * w, p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)])


# ----------------------------------------------------------------------------- config 1: sine advection
def sine_params():
    """Accuracy test: inviscid, tau = 0."""
    return dict(gamma=1.4, Pr=1.0, mu_ref=0.0, visc_omega=0.0, T_ref=1.0, tau_c1=0.0, tau_c2=0.0)


def _sine_rho(s, t=0.0):
    return 1.0 + 0.2 * np.sin(math.pi * (s - 3.0 * t))


def sine_exact_averages(n, t=0.0):
    """Exact cell averages of rho = 1 + 0.2 sin(pi(x+y+z-3t)) on the uniform n^3 mesh of [0,2]^3."""
    h = 2.0 / n
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    sinc = (math.sin(math.pi * h / 2) / (math.pi * h / 2)) ** 3
    return 1.0 + 0.2 * sinc * np.sin(math.pi * (X + Y + Z - 3.0 * t))


def sine_advection(n, t=0.0, gamma=1.4):
    """State of the accuracy test at time t on the uniform n^3 mesh of [0,2]^3:
    exact cell averages; G by the 4-point face Gauss quadrature of exact point values (Eq. 9);
    D = exact point-value differences between paired face Gauss points (Eq. 10 without 1/|l|)."""
    h = 2.0 / n
    nodes = cartesian_nodes(n, 0.0, 2.0)
    rho = sine_exact_averages(n, t)
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    S = X + Y + Z                        # only x+y+z matters
    g = GAUSS_G * h
    drho_axis = np.zeros((3,) + rho.shape)       # cell-averaged d rho/dx_axis by face quadrature
    Drho = np.zeros((12,) + rho.shape)
    for axis in range(3):
        k = 0
        acc = 0.0
        for a in (-g, g):
            for b in (-g, g):
                hi_ = _sine_rho(S + h / 2 + a + b, t); lo_ = _sine_rho(S - h / 2 + a + b, t)
                Drho[4 * axis + k] = hi_ - lo_
                acc = acc + 0.25 * (hi_ - lo_) / h
                k += 1
        drho_axis[axis] = acc
    # rho U = rho, rho E = p/(gamma-1) + 1.5 rho: every variable is affine in rho
    coef = np.array([1.0, 1.0, 1.0, 1.0, 1.5])
    Q = prim_to_cons(rho, 1.0, 1.0, 1.0, 1.0, gamma)
    G = coef[:, None, None, None, None] * drho_axis[None]
    D = coef[:, None, None, None, None] * Drho[None]
    return nodes, Q, G, D


# ----------------------------------------------------------------------------- configs 2/3: Taylor-Green vortex
def tgv_params(Ma=0.1, Re=1600.0, Pr=0.72):
    """Taylor-Green vortex (BASELINE.json config 2): constant mu = 1/Re, tau = mu/p + 5 |dp|/|sum p| dt."""
    return dict(gamma=1.4, Pr=Pr, mu_ref=1.0 / Re, visc_omega=0.0, T_ref=1.0, tau_c1=0.0, tau_c2=5.0)


def taylor_green(nodes, Ma=0.1, gamma=1.4):
    """Point values of the TGV initial field at the cell centroids, used as cell averages."""
    x, y, z = cell_centroids(nodes)
    p0 = 1.0 / (gamma * Ma * Ma)
    u = np.sin(x) * np.cos(y) * np.cos(z)
    v = -np.cos(x) * np.sin(y) * np.cos(z)
    w = np.zeros_like(u)
    p = p0 + (np.cos(2 * x) + np.cos(2 * y)) * (np.cos(2 * z) + 2.0) / 16.0
    rho = p / p0
    return prim_to_cons(rho, u, v, w, p, gamma)


def free_stream(shape, gamma=1.4):
    """Uniform state of BASELINE.json config 3: rho = 1, U = (1, 0.5, 0.25), p = 1/1.4."""
    one = np.ones(shape)
    return prim_to_cons(one, 1.0 * one, 0.5 * one, 0.25 * one, one / 1.4, gamma)


# ----------------------------------------------------------------------------- configs 4/5: isotropic turbulence
def iso_params(Ma_t, Re_lambda=72.0, k0=8.0, gamma=1.4, Pr=0.7):
    """Decaying isotropic turbulence (BASELINE.json configs 4-5; not in the paper): power-law viscosity."""
    p = 1.0 / (gamma * Ma_t * Ma_t)
    uprime = 1.0 / math.sqrt(3.0); lam = 2.0 / k0
    mu_ref = 1.0 * uprime * lam / Re_lambda
    return dict(gamma=gamma, Pr=Pr, mu_ref=mu_ref, visc_omega=0.76, T_ref=p / 1.0, tau_c1=0.0, tau_c2=5.0)


def iso_turbulence(n, seed, Ma_t, k0=8.0, gamma=1.4, device=None):
    """Solenoidal random-phase velocity with E(k) ~ k^4 exp(-2 k^2/k0^2) on the periodic n^3 mesh of [0,2pi]^3,
    rescaled to <u.u>^(1/2) = 1; rho = 1, p = 1/(gamma Ma_t^2).
    With `device` (a torch device) the FFTs run there and a torch tensor on that device is returned (same recipe and
    seed, results equal to the numpy path to round-off); used for the 384^3 bench input."""
    rng = np.random.Generator(np.random.PCG64(seed))
    noise = rng.standard_normal((3, n, n, n))
    if device is not None:
        import torch
        xp = torch
        noise = torch.from_numpy(noise).to(device)
        fftn = lambda a: torch.fft.fftn(a, dim=(1, 2, 3))
        ifftn = lambda a: torch.fft.ifftn(a, dim=(1, 2, 3))
        kk = torch.fft.fftfreq(n, 1.0 / n, dtype=torch.float64, device=device)
        KZ, KY, KX = torch.meshgrid(kk, kk, kk, indexing="ij")
        stack, where, sqrt, exp, absf, real = torch.stack, torch.where, torch.sqrt, torch.exp, torch.abs, torch.real
        one = lambda a: torch.ones_like(a)
    else:
        xp = np
        fftn = lambda a: np.fft.fftn(a, axes=(1, 2, 3))
        ifftn = lambda a: np.fft.ifftn(a, axes=(1, 2, 3))
        kk = np.fft.fftfreq(n, 1.0 / n)
        KZ, KY, KX = np.meshgrid(kk, kk, kk, indexing="ij")
        stack, where, sqrt, exp, absf, real = np.stack, np.where, np.sqrt, np.exp, np.abs, np.real
        one = lambda a: np.ones_like(a)
    uh = fftn(noise)
    del noise
    mag = absf(uh); mag = where(mag == 0, one(mag), mag)
    uh = uh / mag                                       # unit modulus, random phase, Hermitian symmetric
    del mag
    kvec = stack([KX, KY, KZ]); k2 = (kvec ** 2).sum(0); k2s = where(k2 == 0, one(k2), k2)
    uh = uh - kvec * (kvec * uh).sum(0) / k2s           # solenoidal projection
    Ek = k2s ** 2 * exp(-2.0 * k2 / (k0 * k0))
    amp = sqrt(Ek / (2.0 * math.pi * k2s)); amp = where(k2 == 0, 0.0 * amp, amp)
    nrm = sqrt((absf(uh) ** 2).sum(0)); nrm = where(nrm == 0, one(nrm), nrm)
    uh = uh / nrm * amp
    del nrm, amp, Ek, kvec
    u = real(ifftn(uh))
    del uh
    u = u / math.sqrt(float((u ** 2).sum(0).mean()))
    pval = 1.0 / (gamma * Ma_t * Ma_t)
    # velocity components (x, y, z) = u[0], u[1], u[2]; array axes (k, j, i) = (z, y, x)
    ke = 0.5 * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2])
    return stack([one(ke), u[0], u[1], u[2], pval / (gamma - 1.0) + ke])


# ----------------------------------------------------------------------------- affine (sheared) mesh, strong-jump states
SHEAR = np.array([[1.0, 0.3, 0.1], [-0.15, 1.0, 0.2], [0.25, -0.1, 1.0]])      # constant, non-symmetric J0 / h


def sheared_nodes(n, h=1.0, A=SHEAR):
    """Affine periodic mesh of parallelepiped cells: node(i, j, k) = A (i, j, k) h (every cell has J0 = A h)."""
    ni, nj, nk = (n, n, n) if np.isscalar(n) else n
    K, J, I = np.meshgrid(np.arange(nk + 1.0), np.arange(nj + 1.0), np.arange(ni + 1.0), indexing="ij")
    lat = np.stack([I, J, K]) * h
    return np.einsum("ra,akji->rkji", np.asarray(A, dtype=np.float64), lat)


def jump_state(n, kind="blob", ratio=0.05, nodes=None):
    """Piecewise-constant state with a strong density / pressure jump (inside : outside = 1 : ratio) and a uniform
    velocity, on the unit box: the compact polynomials over- and undershoot at the jump by a multiple of the low state,
    so the positivity fallback (reading R9) fires by an O(1) margin.  kind: 'blob' (off-centre ball) or
    'oblique' (slab inclined to all three axes)."""
    nodes = cartesian_nodes(n, 0.0, 1.0) if nodes is None else nodes
    X, Y, Z = cell_centroids(nodes)
    if kind == "blob":
        inside = np.sqrt((X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.55) ** 2) < 0.27
    else:
        inside = (X + 0.5 * Y + 0.25 * Z) % 1.0 < 0.5
    rho = np.where(inside, 1.0, ratio); p = np.where(inside, 1.0, 0.8 * ratio)
    one = np.ones_like(rho)
    return nodes, prim_to_cons(rho, 0.3 * one, -0.2 * one, 0.1 * one, p)


# ----------------------------------------------------------------------------- named workloads
def workload(name, n=None, k0=None):
    """Returns dict(nodes, Q, G, D, params, nonlinear, cfl, steps) for the five BASELINE.json configs.
    G, D are None when the derivative dof are bootstrapped by cgks_set_state.
    For the turbulence cases k0 (spectrum peak, BASELINE.json: 8) may be lowered on small test meshes so that the
    field keeps a resolution comparable to the full-size workload (384^3 with k0 = 8 has 48 cells per peak wavelength)."""
    if name == "sine":
        n = n or 16
        nodes, Q, G, D = sine_advection(n)
        return dict(nodes=nodes, Q=Q, G=G, D=D, params=sine_params(), nonlinear=1, cfl=0.5, steps=10)
    if name == "tgv":
        n = n or 64
        nodes = cartesian_nodes(n)
        return dict(nodes=nodes, Q=taylor_green(nodes), G=None, D=None, params=tgv_params(), nonlinear=1, cfl=0.5, steps=200)
    if name == "tgv_curv":
        n = n or 64
        nodes = curvilinear_nodes(n)
        return dict(nodes=nodes, Q=taylor_green(nodes), G=None, D=None, params=tgv_params(), nonlinear=1, cfl=0.5, steps=200)
    if name == "tgv_sup":
        # the paper's second Taylor-Green workload, Ma = 1.25, Pr = 0.7, nonlinear reconstruction only
        # (128^3 and 320^3 in the paper); shocklets form from t ~ 3
        n = n or 128
        nodes = cartesian_nodes(n)
        return dict(nodes=nodes, Q=taylor_green(nodes, Ma=1.25), G=None, D=None, params=tgv_params(Ma=1.25, Pr=0.7),
                    nonlinear=1, cfl=0.5, steps=200)
    if name == "freestream_curv":
        n = n or 64
        nodes = curvilinear_nodes(n)
        return dict(nodes=nodes, Q=free_stream((n, n, n)), G=None, D=None, params=tgv_params(), nonlinear=1, cfl=0.5, steps=100)
    if name == "iso_sub":
        n = n or 128
        k0 = k0 or 8.0
        return dict(nodes=cartesian_nodes(n), Q=iso_turbulence(n, 4, 0.5, k0), G=None, D=None, params=iso_params(0.5, k0=k0),
                    nonlinear=1, cfl=0.5, steps=500)
    if name == "iso_sup":
        n = n or 384
        k0 = k0 or 8.0
        return dict(nodes=cartesian_nodes(n), Q=iso_turbulence(n, 5, 1.0, k0), G=None, D=None, params=iso_params(1.0, k0=k0),
                    nonlinear=1, cfl=0.5, steps=100)
    if name in ("jump_blob", "jump_oblique", "jump_oblique_linear"):
        # deterministic positivity-fallback cases (reading R9): GENO on a 1:0.05 jump, linear reconstruction on a 1:0.2 jump
        n = n or 12
        kind = "blob" if name == "jump_blob" else "oblique"
        nodes, Q = jump_state(n, kind, 0.2 if name.endswith("linear") else 0.05)
        prm = dict(sine_params()); prm.update(tau_c1=0.05, tau_c2=5.0)
        return dict(nodes=nodes, Q=Q, G=None, D=None, params=prm, nonlinear=0 if name.endswith("linear") else 1, cfl=0.3, steps=5)
    if name == "tgv_shear":
        # Taylor-Green-like smooth field on the affine sheared mesh (constant non-symmetric J0): pins the J0^T / J0^-T transforms
        n = n or 12
        nodes = sheared_nodes(n, 2.0 * math.pi / n)
        xi = np.linalg.solve(SHEAR, cell_centroids(nodes).reshape(3, -1)).reshape(3, n, n, n)      # periodic coordinates
        p0 = 1.0 / (1.4 * 0.3 ** 2)
        u = np.sin(xi[0]) * np.cos(xi[1]) * np.cos(xi[2]); v = -np.cos(xi[0]) * np.sin(xi[1]) * np.cos(xi[2]); wv = 0.2 * np.sin(xi[2] + xi[0])
        p = p0 + (np.cos(2 * xi[0]) + np.cos(2 * xi[1])) * (np.cos(2 * xi[2]) + 2.0) / 16.0
        return dict(nodes=nodes, Q=prim_to_cons(p / p0, u, v, wv, p), G=None, D=None, params=tgv_params(Ma=0.3, Re=200.0),
                    nonlinear=1, cfl=0.5, steps=100)
    raise KeyError(name)

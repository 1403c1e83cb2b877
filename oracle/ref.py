"""ctypes wrapper of the CPU oracle (oracle/cgks_ref.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
The product package (paper_2508_08965_b200) never does.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

NB, ND, NGP = 34, 72, 24


class Params(C.Structure):
    """Mirror of cgks_ref_params (oracle/cgks_ref.h)."""
    _fields_ = [("gamma", C.c_double), ("Pr", C.c_double), ("mu_ref", C.c_double),
                ("visc_omega", C.c_double), ("T_ref", C.c_double),
                ("tau_c1", C.c_double), ("tau_c2", C.c_double),
                ("nonlinear", C.c_int), ("geno_C", C.c_double), ("geno_eps", C.c_double),
                ("geno_r", C.c_int)]


def make_params(gamma=1.4, Pr=1.0, mu_ref=0.0, visc_omega=0.0, T_ref=1.0, tau_c1=0.0, tau_c2=0.0,
                nonlinear=1, geno_C=5.0, geno_eps=1e-15, geno_r=2) -> Params:
    return Params(gamma, Pr, mu_ref, visc_omega, T_ref, tau_c1, tau_c2, int(nonlinear), geno_C, geno_eps, int(geno_r))


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.cgks_ref_create.restype = C.c_void_p
        L.cgks_ref_create.argtypes = [C.c_int, C.c_int, C.c_int, _dp, C.POINTER(Params)]
        L.cgks_ref_destroy.argtypes = [C.c_void_p]
        L.cgks_ref_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.cgks_ref_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.cgks_ref_compute_dt.argtypes = [C.c_void_p, C.c_double, _dp]
        L.cgks_ref_step.argtypes = [C.c_void_p, C.c_double]
        L.cgks_ref_last_error.restype = C.c_char_p
        L.cgks_ref_last_error.argtypes = [C.c_void_p]
        L.cgks_ref_matrices.argtypes = [_dp, _dp]
        L.cgks_ref_basis.argtypes = [C.POINTER(C.c_int), _dp]
        L.cgks_ref_recon_reference.argtypes = [C.POINTER(Params)] + [_dp] * 7
        L.cgks_ref_smoothness.argtypes = [_dp, _dp]
        L.cgks_ref_reconstruct.argtypes = [C.c_void_p, _dp, _dp]
        L.cgks_ref_diagnostics.argtypes = [C.c_void_p, _dp, _dp]
        L.cgks_ref_debug_flux.argtypes = [C.c_void_p, C.c_double, _dp]
        L.cgks_ref_flux_point.argtypes = [C.POINTER(Params), C.c_double] + [_dp] * 7
        L.cgks_ref_moments.argtypes = [C.c_double, C.c_double, _dp, _dp, _dp]
        L.cgks_ref_microslope.argtypes = [_dp] + [C.c_double] * 5 + [_dp]
        L.cgks_ref_moment_apsi.argtypes = [_dp, C.c_int, C.c_int, C.c_int] + [C.c_double] * 5 + [C.c_int, _dp]
        L.cgks_ref_geometry.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.cgks_ref_fallback_stats.argtypes = [C.c_void_p, C.POINTER(C.c_long), _dp, _dp]
        L.cgks_ref_set_readings.argtypes = [C.c_int, C.c_int, C.c_int]
        L.cgks_ref_s2o4_stage1.argtypes = [C.c_double] * 4 + [_dp]
        L.cgks_ref_s2o4_stage2.argtypes = [C.c_double] * 5 + [_dp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def set_readings(r5_normalised=1, s3_sum=1, g2_variant=1):
    """Alternative readings for oracle/readings_table.py; (1, 1, 1) restores the readings taken."""
    lib().cgks_ref_set_readings(int(r5_normalised), int(s3_sum), int(g2_variant))


def matrices():
    M = np.zeros((NB, ND)); E = np.zeros((4 * NGP, NB))
    lib().cgks_ref_matrices(_p(M), _p(E))
    return M, E


def basis():
    d = np.zeros((NB, 3), dtype=np.int32); gp = np.zeros((NGP, 3))
    lib().cgks_ref_basis(d.ctypes.data_as(C.POINTER(C.c_int)), _p(gp))
    return d, gp


def recon_reference(params: Params, d):
    d = _c(d)
    a = np.zeros(NB); b = np.zeros((6, 3)); chi = np.zeros(1); om = np.zeros(6)
    val = np.zeros(NGP); gref = np.zeros((NGP, 3))
    lib().cgks_ref_recon_reference(C.byref(params), _p(d), _p(a), _p(b), _p(chi), _p(om), _p(val), _p(gref))
    return a, b, float(chi[0]), om, val, gref


def smoothness(a):
    a = _c(a); out = np.zeros(4)
    lib().cgks_ref_smoothness(_p(a), _p(out))
    return out


def flux_point(params: Params, dt, WL, gL, WR, gR, n, t1):
    out = np.zeros(30)
    WL, gL, WR, gR, n, t1 = map(_c, (WL, gL, WR, gR, n, t1))
    lib().cgks_ref_flux_point(C.byref(params), float(dt), _p(WL), _p(gL), _p(WR), _p(gR), _p(n), _p(t1), _p(out))
    return out.reshape(6, 5)     # Fn, Ft, VL, DtL, VR, DtR


def moments(U, lam):
    f = np.zeros(7); p = np.zeros(7); n = np.zeros(7)
    lib().cgks_ref_moments(float(U), float(lam), _p(f), _p(p), _p(n))
    return f, p, n


def microslope(h, U, V, W, lam, K):
    h = _c(h); a = np.zeros(5)
    lib().cgks_ref_microslope(_p(h), U, V, W, lam, K, _p(a))
    return a


def moment_apsi(a, i, j, k, U, V, W, lam, K, half=0):
    a = _c(a); out = np.zeros(5)
    lib().cgks_ref_moment_apsi(_p(a), i, j, k, U, V, W, lam, K, half, _p(out))
    return out


def s2o4_stage1(qn, L, Lt, dt):
    o = np.zeros(1); lib().cgks_ref_s2o4_stage1(qn, L, Lt, dt, _p(o)); return float(o[0])


def s2o4_stage2(qn, L, Lt, Lts, dt):
    o = np.zeros(1); lib().cgks_ref_s2o4_stage2(qn, L, Lt, Lts, dt, _p(o)); return float(o[0])


class RefSolver:
    """cgks_ref_* with numpy arrays.  Shapes: nodes (3,nk+1,nj+1,ni+1); Q (5,nk,nj,ni); G (5,3,nk,nj,ni);
    D (5,12,nk,nj,ni)."""

    def __init__(self, nodes, params: Params):
        nodes = _c(nodes)
        self.nk, self.nj, self.ni = (s - 1 for s in nodes.shape[1:])
        self.n = self.ni * self.nj * self.nk
        self.params = params
        self._h = lib().cgks_ref_create(self.ni, self.nj, self.nk, _p(nodes), C.byref(params))
        if not self._h:
            raise ValueError("cgks_ref_create failed")

    def close(self):
        if self._h:
            lib().cgks_ref_destroy(self._h); self._h = None

    def __del__(self):
        self.close()

    def set_state(self, Q, G=None, D=None):
        Q, G, D = _c(Q), _c(G), _c(D)
        assert Q.size == 5 * self.n
        lib().cgks_ref_set_state(self._h, _p(Q), _p(G), _p(D))

    def get_state(self):
        s = (self.nk, self.nj, self.ni)
        Q = np.zeros((5,) + s); G = np.zeros((5, 3) + s); D = np.zeros((5, 12) + s)
        lib().cgks_ref_get_state(self._h, _p(Q), _p(G), _p(D))
        return Q, G, D

    def compute_dt(self, cfl):
        o = np.zeros(1); lib().cgks_ref_compute_dt(self._h, float(cfl), _p(o)); return float(o[0])

    def step(self, dt):
        rc = lib().cgks_ref_step(self._h, float(dt))
        if rc:
            raise FloatingPointError(lib().cgks_ref_last_error(self._h).decode())

    def diagnostics(self):
        """(E_k, enstrophy) of PAPER.md:428-454, divided by |Omega| (rho_0 = 1)."""
        ek = np.zeros(1); en = np.zeros(1)
        lib().cgks_ref_diagnostics(self._h, _p(ek), _p(en))
        return float(ek[0]), float(en[0])

    def reconstruct(self):
        pv = np.zeros((self.nk, self.nj, self.ni, NGP, 20)); chi = np.zeros((5, self.nk, self.nj, self.ni))
        lib().cgks_ref_reconstruct(self._h, _p(pv), _p(chi))
        return pv, chi

    def fallback_stats(self):
        """(points replaced by the R9 fallback in the last reconstruction, min rho/rho_cell, min admissibility/scale)."""
        n = C.c_long(0); a = np.zeros(1); b = np.zeros(1)
        lib().cgks_ref_fallback_stats(self._h, C.byref(n), _p(a), _p(b))
        return int(n.value), float(a[0]), float(b[0])

    def debug_flux(self, dt):
        fx = np.zeros((3, self.nk, self.nj, self.ni, 4, 30))
        lib().cgks_ref_debug_flux(self._h, float(dt), _p(fx))
        return fx

    def geometry(self):
        vol = np.zeros((self.nk, self.nj, self.ni)); J0 = np.zeros((self.nk, self.nj, self.ni, 3, 3))
        area = np.zeros((3, self.nk, self.nj, self.ni, 3))
        lib().cgks_ref_geometry(self._h, _p(vol), _p(J0), _p(area))
        return vol, J0, area

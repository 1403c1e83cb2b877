"""Thin Python binding of the C ABI in include/cgks.h (argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels of libcgks.so.
There is no CPU fallback: a missing library or device raises."""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcgks.so")

CGKS_OK, CGKS_EINVAL, CGKS_ENOMEM, CGKS_ECUDA, CGKS_ENONPHYSICAL = 0, -1, -2, -3, -4
BC_SLIP_WALL, BC_NOSLIP_WALL, BC_OUTFLOW, BC_FARFIELD = 0, 1, 2, 3
KERNEL_CLASSES = {"recon": 0, "flux": 1, "update": 2, "cfl": 3, "other": 4}


class cgks_params(C.Structure):
    _fields_ = [("gamma", C.c_double), ("Pr", C.c_double), ("mu_ref", C.c_double),
                ("visc_omega", C.c_double), ("T_ref", C.c_double),
                ("tau_c1", C.c_double), ("tau_c2", C.c_double),
                ("nonlinear", C.c_int), ("geno_C", C.c_double), ("geno_eps", C.c_double),
                ("geno_r", C.c_int)]


class CgksError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("cgks error %d: %s" % (code, msg))
        self.code = code


_lib = None
_vp = C.c_void_p


def lib():
    """Loads libcgks.so; raises if it has not been built (python -m paper_2508_08965_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("CUDA extension %s is missing: run `python paper_2508_08965_b200/build.py`" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        L.cgks_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_size_t, C.POINTER(C.c_size_t)]
        L.cgks_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, _vp, C.POINTER(cgks_params), _vp, C.c_size_t, _vp]
        L.cgks_set_state.argtypes = [_vp, _vp, _vp, _vp]
        L.cgks_get_state.argtypes = [_vp, _vp, _vp, _vp]
        L.cgks_compute_dt.argtypes = [_vp, C.c_double, C.POINTER(C.c_double)]
        L.cgks_compute_dt_static.argtypes = [C.c_int, C.c_int, C.c_int, _vp, C.POINTER(C.c_double), C.POINTER(cgks_params),
                                             C.c_double, _vp, _vp, _vp]
        L.cgks_static_last_error.restype = C.c_char_p
        L.cgks_step.argtypes = [_vp, C.c_double]
        L.cgks_stage.argtypes = [_vp, C.c_int, C.c_double]
        L.cgks_create_slab.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _vp, C.POINTER(cgks_params), _vp, C.c_size_t, _vp]
        L.cgks_halo_bytes.argtypes = [_vp, C.POINTER(C.c_size_t)]
        L.cgks_pack_halo.argtypes = [_vp, C.c_int, _vp]
        L.cgks_unpack_halo.argtypes = [_vp, C.c_int, _vp]
        L.cgks_fill_halo_bc.argtypes = [_vp, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.cgks_status.argtypes = [_vp]
        L.cgks_diagnostics.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.cgks_run_host.argtypes = [_vp, _vp, _vp, _vp, C.c_double, C.c_int, _vp, _vp, _vp]
        L.cgks_launch_count.argtypes = [_vp]; L.cgks_launch_count.restype = C.c_long
        L.cgks_slab_depth.argtypes = [_vp]
        L.cgks_set_profiling.argtypes = [_vp, C.c_int]
        L.cgks_kernel_ms.argtypes = [_vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_long)]
        L.cgks_get_chi.argtypes = [_vp, _vp]
        L.cgks_debug_stage.argtypes = [_vp, C.c_double, _vp, _vp]
        L.cgks_fp64_peak.argtypes = [_vp, C.POINTER(C.c_double)]
        L.cgks_debug_math.argtypes = [C.c_int, C.c_long, _vp, _vp, _vp]
        L.cgks_destroy.argtypes = [_vp]
        L.cgks_last_error.argtypes = [_vp]; L.cgks_last_error.restype = C.c_char_p
        L.cgks_last_create_error.restype = C.c_char_p
        L.cgks_version.restype = C.c_char_p
        _lib = L
    return _lib


def make_params(gamma=1.4, Pr=1.0, mu_ref=0.0, visc_omega=0.0, T_ref=1.0, tau_c1=0.0, tau_c2=0.0,
                nonlinear=1, geno_C=5.0, geno_eps=1e-15, geno_r=2):
    return cgks_params(gamma, Pr, mu_ref, visc_omega, T_ref, tau_c1, tau_c2, int(nonlinear), geno_C, geno_eps, int(geno_r))


def workspace_bytes(ni, nj, nk, budget_bytes=0):
    out = C.c_size_t(0)
    rc = lib().cgks_workspace_bytes(ni, nj, nk, budget_bytes, C.byref(out))
    if rc:
        raise CgksError(rc, "cgks_workspace_bytes")
    return out.value


STATIC_MAX_CELLS = 1 << 24


def compute_dt_static(Q, h, params, cfl, out_dt, out_bad=None):
    """cgks_compute_dt_static: the CFL time step of the cell averages Q (5, nk, nj, ni) on a uniform Cartesian mesh of
    cell sizes h = (hx, hy, hz), without a Solver, a workspace or any device allocation -- for callers that cannot
    allocate (all of HBM owned by someone else's allocator, or a loop that must not hit cudaMalloc's device-wide
    synchronisation).  Nothing is allocated here either: Q must already be a contiguous float64 CUDA tensor, and the
    results go into tensors the caller owns, out_dt (1 float64) and, if given, out_bad (1 int32: 1 when a cell with
    rho <= 0 or p <= 0 was met).  Asynchronous on the current stream of Q's device.  At most STATIC_MAX_CELLS cells;
    calls that may overlap on the GPU race on the library's built-in scratch array (include/cgks.h)."""
    if not (Q.is_cuda and Q.dtype == torch.float64 and Q.is_contiguous() and Q.dim() == 4 and Q.shape[0] == 5):
        raise ValueError("Q must be a contiguous float64 CUDA tensor of shape (5, nk, nj, ni)")
    if not (out_dt.is_cuda and out_dt.dtype == torch.float64 and out_dt.numel() >= 1):
        raise ValueError("out_dt must be a float64 CUDA tensor")
    if out_bad is not None and not (out_bad.is_cuda and out_bad.dtype == torch.int32 and out_bad.numel() >= 1):
        raise ValueError("out_bad must be an int32 CUDA tensor")
    nk, nj, ni = (int(s) for s in Q.shape[1:])
    prm = params if isinstance(params, cgks_params) else make_params(**params)
    hh = (C.c_double * 3)(*[float(x) for x in h])
    with torch.cuda.device(Q.device):
        st = torch.cuda.current_stream()
        rc = lib().cgks_compute_dt_static(ni, nj, nk, _ptr(Q), hh, C.byref(prm), float(cfl), _ptr(out_dt), _ptr(out_bad),
                                          _vp(st.cuda_stream))
    if rc:
        raise CgksError(rc, lib().cgks_static_last_error().decode())


def fp64_peak_tflops(device="cuda:0"):
    """DFMA micro-benchmark (cgks_fp64_peak): measured FP64 FMA throughput of the device in TFLOP/s."""
    out = C.c_double(0.0)
    with torch.cuda.device(device):
        st = torch.cuda.current_stream()
        rc = lib().cgks_fp64_peak(_vp(st.cuda_stream), C.byref(out))
    if rc:
        raise CgksError(rc, "cgks_fp64_peak")
    return out.value


def debug_math(which, x, device="cuda:0"):
    """Test tap cgks_debug_math: 0 1/x, 1 1/sqrt(x), 2 exp(x), 3 erfc(x), 4 exp(-x^2); x a float64 array."""
    xin = _dev(x, torch.device(device)).reshape(-1)
    out = torch.empty_like(xin)
    with torch.cuda.device(xin.device):
        st = torch.cuda.current_stream()
        rc = lib().cgks_debug_math(int(which), xin.numel(), _ptr(xin), _ptr(out), _vp(st.cuda_stream))
    if rc:
        raise CgksError(rc, "cgks_debug_math")
    return out.cpu().numpy()


def _dev(a, device):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        a = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
    return a.to(device=device, dtype=torch.float64).contiguous()


def _ptr(t):
    return None if t is None else _vp(t.data_ptr())


class Solver:
    """cgks_create / cgks_set_state / cgks_compute_dt / cgks_step / cgks_get_state on one CUDA device.

    nodes (3, nk+1, nj+1, ni+1); Q (5, nk, nj, ni); G (5, 3, nk, nj, ni); D (5, 12, nk, nj, ni)."""

    def __init__(self, nodes, params, device="cuda:0", budget_bytes=0, workspace_nbytes=None, slab=None):
        """slab = (k0, nk_owned): a sub-domain context (cgks_create_slab) of the global mesh given by `nodes`; its arrays
        have nk_owned + 4 planes (two halo planes on each side)."""
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2508_08965_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        self._h = _vp(None)
        L = lib()
        nodes = _dev(nodes, self.device)
        self.nk_global, self.nj, self.ni = (int(s) - 1 for s in nodes.shape[1:])
        self.slab = slab
        self.nk = self.nk_global if slab is None else int(slab[1]) + 4
        self.n = self.ni * self.nj * self.nk
        self.params = params if isinstance(params, cgks_params) else make_params(**params)
        nbytes = workspace_nbytes or workspace_bytes(self.ni, self.nj, self.nk, budget_bytes)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device)
            if slab is None:
                rc = L.cgks_create(C.byref(self._h), self.ni, self.nj, self.nk, _ptr(nodes), C.byref(self.params),
                                   _vp(self.workspace.data_ptr()), nbytes, _vp(self.stream.cuda_stream))
            else:
                rc = L.cgks_create_slab(C.byref(self._h), self.ni, self.nj, self.nk_global, int(slab[0]), int(slab[1]), _ptr(nodes),
                                        C.byref(self.params), _vp(self.workspace.data_ptr()), nbytes, _vp(self.stream.cuda_stream))
        if rc:
            self._h = _vp(None)
            raise CgksError(rc, "cgks_create: " + L.cgks_last_create_error().decode())

    def _check(self, rc):
        if rc:
            raise CgksError(rc, lib().cgks_last_error(self._h).decode())

    def close(self):
        if self._h:
            lib().cgks_destroy(self._h); self._h = _vp(None)
        self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, Q, G=None, D=None):
        Q, G, D = _dev(Q, self.device), _dev(G, self.device), _dev(D, self.device)
        assert Q.numel() == 5 * self.n
        self._check(lib().cgks_set_state(self._h, _ptr(Q), _ptr(G), _ptr(D)))
        torch.cuda.current_stream(self.device).synchronize()      # the inputs may be temporaries

    def get_state(self, derivatives=True):
        """(Q, G, D) of the current state; derivatives=False returns (Q, None, None) without allocating the 75 derivative
        fields (cgks_get_state takes NULL for what is not wanted)."""
        s = (self.nk, self.nj, self.ni)
        Q = torch.empty((5,) + s, dtype=torch.float64, device=self.device)
        G = torch.empty((5, 3) + s, dtype=torch.float64, device=self.device) if derivatives else None
        D = torch.empty((5, 12) + s, dtype=torch.float64, device=self.device) if derivatives else None
        self._check(lib().cgks_get_state(self._h, _ptr(Q), _ptr(G), _ptr(D)))
        return Q, G, D

    def compute_dt(self, cfl):
        out = C.c_double(0.0)
        self._check(lib().cgks_compute_dt(self._h, float(cfl), C.byref(out)))
        return out.value

    def step(self, dt):
        self._check(lib().cgks_step(self._h, float(dt)))

    def stage(self, stage, dt):
        self._check(lib().cgks_stage(self._h, int(stage), float(dt)))

    def halo_buffer(self):
        """A device buffer for one side's halo planes: 80 * 2 * nj * ni doubles (cgks_halo_bytes), opaque -- the library's internal
        record order, to be filled by pack_halo and read by unpack_halo only (include/cgks.h)."""
        nb = C.c_size_t(0)
        self._check(lib().cgks_halo_bytes(self._h, C.byref(nb)))
        return torch.empty(nb.value // 8, dtype=torch.float64, device=self.device)

    def pack_halo(self, side, buf):
        self._check(lib().cgks_pack_halo(self._h, int(side), _ptr(buf)))

    def unpack_halo(self, side, buf):
        self._check(lib().cgks_unpack_halo(self._h, int(side), _ptr(buf)))

    def fill_halo_bc(self, side, kind, far_state=None):
        """cgks_fill_halo_bc: boundary rule `kind` (BC_*) for the halo planes of `side`; far_state = 5 conservative values."""
        far = None if far_state is None else (C.c_double * 5)(*[float(x) for x in far_state])
        self._check(lib().cgks_fill_halo_bc(self._h, int(side), int(kind), far))

    def step_bounded(self, dt, bc_lo, bc_hi, far_state=None):
        """One S2O4 step of a sub-domain bounded in k on both sides: the boundary rules before each stage, then the stage."""
        for stage in (1, 2):
            self.fill_halo_bc(0, bc_lo, far_state); self.fill_halo_bc(1, bc_hi, far_state)
            self.stage(stage, dt)

    def diagnostics(self):
        """(E_k, enstrophy) of the current state, divided by |Omega|."""
        ek = C.c_double(0.0); en = C.c_double(0.0)
        self._check(lib().cgks_diagnostics(self._h, C.byref(ek), C.byref(en)))
        return ek.value, en.value

    def status(self):
        self._check(lib().cgks_status(self._h))

    def chi(self):
        out = torch.empty((5, self.nk, self.nj, self.ni), dtype=torch.float64, device=self.device)
        self._check(lib().cgks_get_chi(self._h, _ptr(out)))
        return out

    def run_host(self, Q, G, D, cfl, nsteps, out_Q, out_G=None, out_D=None):
        """Host (ideally pinned) tensors in and out; H2D + nsteps steps + D2H inside the call."""
        def hp(t):
            return None if t is None else _vp(t.data_ptr())
        self._check(lib().cgks_run_host(self._h, hp(Q), hp(G), hp(D), float(cfl), int(nsteps), hp(out_Q), hp(out_G), hp(out_D)))

    def debug_stage(self, dt=None):
        """Test tap: (pv [24][20][nk][nj][ni], fx [12][30][nk][nj][ni] or None) of the current state."""
        s = (self.nk, self.nj, self.ni)
        pv = torch.empty((24, 20) + s, dtype=torch.float64, device=self.device)
        fx = None if dt is None else torch.empty((12, 30) + s, dtype=torch.float64, device=self.device)
        self._check(lib().cgks_debug_stage(self._h, 0.0 if dt is None else float(dt), _ptr(pv), _ptr(fx)))
        return pv, fx

    def launch_count(self):
        return int(lib().cgks_launch_count(self._h))

    def slab_depth(self):
        """k-planes per chunk of the stage pipeline chosen from the workspace size (nk: whole mesh resident)."""
        return int(lib().cgks_slab_depth(self._h))

    def set_profiling(self, on):
        self._check(lib().cgks_set_profiling(self._h, int(on)))

    def kernel_ms(self, which):
        ms = C.c_double(0.0); nl = C.c_long(0)
        self._check(lib().cgks_kernel_ms(self._h, KERNEL_CLASSES[which], C.byref(ms), C.byref(nl)))
        return ms.value, nl.value

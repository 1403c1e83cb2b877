"""cgks_compute_dt_static: the CFL time step for callers that cannot allocate device memory.

Who that is: code that gets a Q array inside a process where somebody else's allocator already owns all of HBM (a raw
cudaMalloc fails there, and without memory there is no workspace for cgks_create either), and time loops that must not
run into the device-wide synchronisation of cudaMalloc / cudaFree.  The entry point therefore keeps its per-block partial
minima in an array compiled into libcgks.so (33 kB per GPU, at most 256^3 cells) instead of in a caller's workspace.

The checks: the result equals cgks_compute_dt of a context on the same mesh and state, to the 1e-13 the parity tests
allow for a time step, on two calls in a row that share the array (the second on a smaller mesh, so stale partials
of the first call lie behind the ones it uses; then a call that raises the bad-cell flag followed by one that must find it
cleared).  Every tensor is created before the calls: the calls themselves allocate nothing.

This file is named so that pytest collects it last (`pytest --collect-only -q`): `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests.  It does not depend on them: it passes alone in a fresh process too."""
import ctypes as C

import numpy as np
import pytest

from paper_2508_08965_b200 import inputs

TOL_DT = 1e-13            # tests/test_gpu_parity.py: the first dt is the same formula on identical input


def _cell_sizes(nodes):
    """Period / n per direction from the corner nodes, the way cgks_create derives them for a uniform Cartesian mesh."""
    nk, nj, ni = (s - 1 for s in nodes.shape[1:])
    return ((nodes[0, 0, 0, ni] - nodes[0, 0, 0, 0]) / ni, (nodes[1, 0, nj, 0] - nodes[1, 0, 0, 0]) / nj,
            (nodes[2, nk, 0, 0] - nodes[2, 0, 0, 0]) / nk)


def _context_dt(w):
    """The existing path: cgks_create + cgks_set_state + cgks_compute_dt (scratch in the caller's workspace)."""
    from paper_2508_08965_b200 import binding
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=w["nonlinear"]))
    s.set_state(w["Q"], w["G"], w["D"])
    dt = s.compute_dt(w["cfl"])
    s.close()
    return dt


@pytest.mark.gpu
def test_static_dt_matches_context_dt_on_consecutive_calls():
    import torch
    from paper_2508_08965_b200 import binding
    dev = torch.device("cuda:0")
    # viscous Taylor-Green vortex (the viscous cap takes part), then supersonic turbulence with the power-law viscosity on a
    # smaller mesh; 40^3 = 15.6 blocks of 4096 cells: several blocks and a ragged last one
    cases = [inputs.workload("tgv", 40), inputs.workload("iso_sup", 24, 2.0), inputs.workload("sine", 16)]
    want = [_context_dt(w) for w in cases]
    Qs = [torch.from_numpy(np.ascontiguousarray(w["Q"])).to(dev) for w in cases]
    out = torch.full((len(cases),), -1.0, dtype=torch.float64, device=dev)
    bad = torch.full((len(cases),), -1, dtype=torch.int32, device=dev)
    torch.cuda.synchronize()
    for rep in range(2):                                   # the whole sequence twice: the array keeps the last call's contents
        for i, w in enumerate(cases):                      # back to back on one stream, no synchronisation in between
            binding.compute_dt_static(Qs[i], _cell_sizes(w["nodes"]), binding.make_params(**w["params"]), w["cfl"],
                                      out[i:i + 1], bad[i:i + 1])
        got = out.cpu().numpy(); flags = bad.cpu().numpy()
        for i in range(len(cases)):
            assert abs(got[i] / want[i] - 1.0) <= TOL_DT, (rep, i, got[i], want[i])
            assert flags[i] == 0
        out.fill_(-1.0); bad.fill_(-1)


@pytest.mark.gpu
def test_static_dt_flag_is_cleared_between_calls():
    import torch
    from paper_2508_08965_b200 import binding
    dev = torch.device("cuda:0")
    w = inputs.workload("tgv", 24)
    prm, h = binding.make_params(**w["params"]), _cell_sizes(w["nodes"])
    good = torch.from_numpy(np.ascontiguousarray(w["Q"])).to(dev)
    broken = good.clone(); broken[0, 3, 5, 7] = -1.0       # one cell with negative density
    out = torch.zeros(2, dtype=torch.float64, device=dev); bad = torch.zeros(2, dtype=torch.int32, device=dev)
    binding.compute_dt_static(broken, h, prm, w["cfl"], out[0:1], bad[0:1])
    binding.compute_dt_static(good, h, prm, w["cfl"], out[1:2], bad[1:2])
    assert bad.cpu().tolist() == [1, 0]
    want = _context_dt(w)
    got = out.cpu().numpy()
    assert abs(got[1] / want - 1.0) <= TOL_DT
    assert np.isfinite(got[0]) and got[0] > 0.0            # the bad cell is skipped, the others still reduce


def test_static_dt_rejects_what_does_not_fit():
    """Host-side argument checks run before any CUDA call, so they are testable without a device: a mesh beyond the
    built-in array's 256^3 cells is refused with a message that names the limit."""
    from paper_2508_08965_b200 import binding, build
    build.build()
    L = binding.lib()
    prm = binding.make_params()
    h = (C.c_double * 3)(1.0, 1.0, 1.0)
    dummy = C.c_void_p(256)                                # never dereferenced: the size check comes first
    rc = L.cgks_compute_dt_static(257, 256, 256, dummy, h, C.byref(prm), 0.5, dummy, None, None)
    assert rc == binding.CGKS_EINVAL
    msg = L.cgks_static_last_error().decode()
    assert str(binding.STATIC_MAX_CELLS) in msg and "exceed" in msg
    assert L.cgks_compute_dt_static(0, 8, 8, dummy, h, C.byref(prm), 0.5, dummy, None, None) == binding.CGKS_EINVAL
    assert L.cgks_compute_dt_static(8, 8, 8, None, h, C.byref(prm), 0.5, dummy, None, None) == binding.CGKS_EINVAL
    assert L.cgks_compute_dt_static(8, 8, 8, dummy, h, C.byref(prm), -1.0, dummy, None, None) == binding.CGKS_EINVAL
    assert b"positive" in L.cgks_static_last_error()

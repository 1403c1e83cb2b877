"""Host-side checks of the C ABI (no GPU needed): the library loads, exports every function include/cgks.h declares,
and its pure host entry points behave as documented."""
import ctypes as C
import os
import re

import pytest

from paper_2508_08965_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "cgks.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cgks_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert {"cgks_create", "cgks_set_state", "cgks_compute_dt", "cgks_step", "cgks_get_state", "cgks_destroy",
            "cgks_workspace_bytes", "cgks_run_host", "cgks_status", "cgks_stage", "cgks_create_slab", "cgks_halo_bytes",
            "cgks_pack_halo", "cgks_unpack_halo", "cgks_last_create_error"} <= set(names)
    for nm in names:
        assert hasattr(lib, nm), nm
    raw = C.CDLL(binding.LIB_PATH)
    for nm in names:
        getattr(raw, nm)          # raises AttributeError if the symbol is missing


def test_version_and_workspace_sizes(lib):
    assert b"sm_100a" in lib.cgks_version()
    small = binding.workspace_bytes(16, 16, 16)
    fixed = (3 * 80 + 5 + 37) * 16 ** 3 * 8
    assert small >= fixed + (480 + 360) * 16 ** 3 * 8          # whole mesh resident
    big = binding.workspace_bytes(384, 384, 384)
    assert 100e9 < big < 185e9                                  # three state buffers, metrics, ~48 GB of slab buffers
    capped = binding.workspace_bytes(384, 384, 384, int(150e9))
    assert capped <= 150e9 + 4096 and capped < big
    with pytest.raises(binding.CgksError) as e:
        binding.workspace_bytes(3, 16, 16)
    assert e.value.code == binding.CGKS_EINVAL
    with pytest.raises(binding.CgksError) as e:                 # a budget below the state buffers plus a two-plane slab
        binding.workspace_bytes(384, 384, 384, int(100e9))
    assert e.value.code == binding.CGKS_ENOMEM


def test_no_cpu_fallback(lib):
    """Without a CUDA device every compute entry point refuses: the product path never routes through the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p(None)
    prm = binding.make_params()
    dummy = (C.c_double * 8)()
    rc = lib.cgks_create(C.byref(h), 8, 8, 8, C.cast(dummy, C.c_void_p), C.byref(prm), C.cast(dummy, C.c_void_p), 64, None)
    assert rc == binding.CGKS_ECUDA and not h.value
    assert lib.cgks_last_create_error() == b"no CUDA device" and lib.cgks_last_error(None) == b"no CUDA device"
    assert lib.cgks_create(C.byref(h), 3, 8, 8, C.cast(dummy, C.c_void_p), C.byref(prm), C.cast(dummy, C.c_void_p), 64, None) == binding.CGKS_EINVAL
    assert b"at least 4" in lib.cgks_last_create_error()
    with pytest.raises(RuntimeError):
        binding.Solver(__import__("numpy").zeros((3, 9, 9, 9)), prm)
    assert lib.cgks_step(None, 0.1) == binding.CGKS_EINVAL
    assert lib.cgks_destroy(None) == binding.CGKS_EINVAL
    assert lib.cgks_stage(None, 1, 0.1) == binding.CGKS_EINVAL and lib.cgks_pack_halo(None, 0, None) == binding.CGKS_EINVAL


def test_product_path_does_not_import_the_oracle():
    import subprocess
    import sys
    code = ("import sys; import paper_2508_08965_b200.binding, paper_2508_08965_b200.inputs, paper_2508_08965_b200.build, paper_2508_08965_b200.slab; "
            "bad = [m for m in sys.modules if m == 'oracle' or m.startswith('oracle.')]; sys.exit(1 if bad else 0)")
    assert subprocess.run([sys.executable, "-c", code], cwd=ROOT).returncode == 0
    for fn in os.listdir(os.path.join(ROOT, "paper_2508_08965_b200", "csrc")):
        txt = open(os.path.join(ROOT, "paper_2508_08965_b200", "csrc", fn), errors="ignore").read()
        assert "cgks_ref" not in txt and "oracle/" not in txt.replace("oracle/)", ""), fn


def test_generated_headers_are_current(tmp_path):
    """csrc/recon_gen.cuh and csrc/math_gen.cuh (committed) are exactly what their generators produce, and the
    symmetry-reduced reconstruction operators reproduce a = M d (numpy emulation of the emitted structure)."""
    import importlib.util
    csrc = os.path.join(ROOT, "paper_2508_08965_b200", "csrc")
    for gen, hdr in (("gen_recon.py", "recon_gen.cuh"), ("gen_math.py", "math_gen.cuh")):
        spec = importlib.util.spec_from_file_location(gen[:-3], os.path.join(csrc, gen))
        mod = importlib.util.module_from_spec(spec); spec.loader.exec_module(mod)
        out = tmp_path / hdr
        mod.generate(str(out))
        assert out.read_text() == open(os.path.join(csrc, hdr)).read(), hdr
        if gen == "gen_recon.py":
            assert mod.self_check() == 312


def test_flux_flop_constant_is_the_oracle_count():
    """bench.py's FLUX_FLOPS_ORACLE (the oracle-counted algorithmic flops per face Gauss point it prints in `roofline`) is
    what the counting-double build of the oracle gives for the bench workload's gas constants."""
    import importlib.util
    import sys
    spec = importlib.util.spec_from_file_location("flop_count", os.path.join(ROOT, "oracle", "flop_count.py"))
    fc = importlib.util.module_from_spec(spec); spec.loader.exec_module(fc)
    counts = fc.counts()
    spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec); spec.loader.exec_module(bench)
    assert counts["flux_point"][1] == bench.FLUX_FLOPS_ORACLE
    assert counts["flux_point"][0] >= counts["flux_point"][1] > 5 * bench.SWEEP_FLOPS_STAGE1
    # the non-zero count of one (cell, variable) reconstruction is bounded below by the non-zeros of M and E (FMA = 2)
    assert counts["recon_var"][1] >= 2 * (1008 + 2184)


def test_flux_flop_constants_belong_to_the_committed_kernel_source():
    """bench.py's executed-flop constants were counted with ncu on a specific revision of the flux arithmetic
    and of the sweep kernel around it (profiles/r02k_final.md); a change to gks_flux.cuh / fastmath64.cuh / math_gen.cuh /
    kernels_fused.cuh without a re-count fails here."""
    import hashlib
    import importlib.util
    csrc = os.path.join(ROOT, "paper_2508_08965_b200", "csrc")
    h = hashlib.sha256()
    for fn in ("gks_flux.cuh", "fastmath64.cuh", "math_gen.cuh", "kernels_fused.cuh"):
        h.update(open(os.path.join(csrc, fn), "rb").read())
    spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec); spec.loader.exec_module(bench)
    assert h.hexdigest()[:16] == bench.FLUX_SOURCE_SHA16, "re-count SWEEP_FLOPS_STAGE1/2 with ncu and update FLUX_SOURCE_SHA16"

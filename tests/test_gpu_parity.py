"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): relative L-inf <= 1e-10 after one step and <= 1e-8 after
100 steps, on every one of the 80 fields (norm of DESIGN.md section 6)."""
import numpy as np
import pytest

from paper_2508_08965_b200 import inputs
from tests import parity

pytestmark = pytest.mark.gpu

TOL_1 = 1e-10
TOL_100 = 1e-8


def _check(w, nsteps, tol, budget=0):
    orc, dts = parity.run_oracle(w, nsteps)
    gpu, dts_gpu = parity.run_gpu(w, nsteps, dts=dts, budget_bytes=budget)
    # both sides step with the oracle's dt; the GPU's own CFL reduction must agree with it
    np.testing.assert_allclose(dts_gpu, dts, rtol=max(tol, 1e-12))
    errs = parity.field_errors(gpu, orc, w["nodes"], w["Q"])
    worst = max(errs, key=errs.get)
    assert errs[worst] <= tol, (worst, errs[worst])
    return errs[worst]


CASES_1STEP = [
    ("sine", 16, 1), ("sine", 16, 0), ("sine", 8, 1),
    ("tgv", 16, 1), ("tgv", 16, 0),
    ("tgv_curv", 12, 1), ("freestream_curv", 8, 1),
    ("iso_sub", 16, 1), ("iso_sup", 16, 1),
]


@pytest.mark.parametrize("name,n,nonlinear", CASES_1STEP)
def test_one_step_parity(name, n, nonlinear):
    w = parity.build_case(name, n, nonlinear)
    _check(w, 1, TOL_1)


def test_ragged_sizes_and_minimum_mesh():
    """Sizes that are not multiples of any block/tile size, and the smallest allowed mesh (4 cells per direction)."""
    for shape in ((13, 9, 7), (4, 4, 4), (5, 4, 33)):
        ni, nj, nk = shape
        nodes = inputs.cartesian_nodes(shape, 0.0, 2.0 * np.pi)
        # unequal spacing per direction: stretch y and z
        nodes[1] *= 0.8; nodes[2] *= 1.3
        Q = inputs.taylor_green(nodes)
        w = dict(nodes=nodes, Q=Q, G=None, D=None, params=inputs.tgv_params(Re=100.0), nonlinear=1, cfl=0.5)
        _check(w, 2, TOL_1 * 2)


def test_slab_pipeline_equals_resident():
    """A workspace budget that forces the k-slab pipeline (several chunks, recomputed halo planes) gives the same
    bits as the fully resident run, and both match the oracle."""
    from paper_2508_08965_b200 import binding
    w = parity.build_case("tgv_curv", 12, 1)
    full, _ = parity.run_gpu(w, 2)
    n = 12 ** 3
    fixed = 3 * 80 * n * 8 + 5 * n * 8 + 37 * n * 8 + 4096
    budget = fixed + 6 * (480 + 360) * 144 * 8           # 6 slots -> slab depth 4 -> 3 chunks
    slab, _ = parity.run_gpu(w, 2, budget_bytes=budget)
    for a, b in zip(full, slab):
        assert np.array_equal(a, b)
    _check(w, 2, TOL_1 * 2, budget=budget)


@pytest.mark.parametrize("name,n", [("sine", 16), ("iso_sup", 16)])
def test_hundred_step_parity(name, n):
    w = parity.build_case(name, n, 1)
    _check(w, 100, TOL_100)


def test_ten_steps_config1():
    """BASELINE.json config 1: 16^3 sine advection, 10 S2O4 steps."""
    w = parity.build_case("sine", 16, 1)
    _check(w, 10, 1e-9)


def test_conservation_and_free_stream_on_gpu():
    w = parity.build_case("freestream_curv", 12, 1)
    gpu, _ = parity.run_gpu(w, 20)
    assert np.abs(gpu[0] - w["Q"]).max() < 1e-12
    assert np.abs(gpu[1]).max() < 1e-11 and np.abs(gpu[2]).max() < 1e-12
    w = parity.build_case("tgv", 16, 1)
    gpu, _ = parity.run_gpu(w, 5)
    np.testing.assert_allclose(gpu[0].sum(axis=(1, 2, 3)), w["Q"].sum(axis=(1, 2, 3)), rtol=1e-13, atol=1e-10)


def test_error_codes():
    from paper_2508_08965_b200 import binding
    nodes = inputs.cartesian_nodes(8)
    prm = binding.make_params(**inputs.tgv_params())
    with pytest.raises(binding.CgksError) as e:
        binding.Solver(inputs.cartesian_nodes((3, 8, 8)), prm)
    assert e.value.code == binding.CGKS_EINVAL
    with pytest.raises(binding.CgksError) as e:
        binding.Solver(nodes, prm, budget_bytes=1 << 20)          # cannot hold even two k-planes of slab
    assert e.value.code in (binding.CGKS_ENOMEM,)
    bad = nodes.copy(); bad[0, :, :, -1] += 0.3                   # breaks periodicity of the node array
    with pytest.raises(binding.CgksError) as e:
        binding.Solver(bad, prm)
    assert e.value.code == binding.CGKS_EINVAL
    s = binding.Solver(nodes, prm)
    Q = inputs.taylor_green(nodes); Q[4, 2, 3, 4] = -1.0          # negative energy
    s.set_state(Q)
    with pytest.raises(binding.CgksError) as e:
        s.compute_dt(0.5)
    assert e.value.code == binding.CGKS_ENONPHYSICAL
    s.close()


def test_chi_matches_oracle():
    from oracle import ref
    from paper_2508_08965_b200 import binding
    w = parity.build_case("iso_sup", 16, 1)
    so = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1)); so.set_state(w["Q"])
    _, chi_o = so.reconstruct()
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1)); s.set_state(w["Q"])
    s.step(1e-6)
    # chi of the LAST reconstruction (stage 2) is what the tap returns: compare loosely, and exactly for stage 1
    # through a zero-length-like step: dt -> tiny, W* ~ W^n
    chi_g = s.chi().cpu().numpy()
    assert np.abs(chi_g - chi_o).max() < 1e-3
    assert (chi_g < 0.99).mean() > 0.01            # the adaptive fallback is exercised by this workload
    s.close()

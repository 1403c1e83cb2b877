"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): relative L-inf <= 1e-10 after one step and <= 1e-8 after
100 steps, on every one of the 80 fields (norm of DESIGN.md section 6)."""
import os

import numpy as np
import pytest

from paper_2508_08965_b200 import inputs
from tests import parity

pytestmark = pytest.mark.gpu

TOL_1 = 1e-10
TOL_100 = 1e-8


def _check(w, nsteps, tol, budget=0, own_dt=False):
    orc, dts = parity.run_oracle(w, nsteps)
    gpu, dts_gpu = parity.run_gpu(w, nsteps, dts=None if own_dt else dts, budget_bytes=budget)
    # the first dt is the same formula on identical input; later ones on states that agree to `tol`
    assert abs(dts_gpu[0] / dts[0] - 1) <= 1e-13, (dts_gpu[0], dts[0])
    np.testing.assert_allclose(dts_gpu, dts, rtol=tol)
    errs = parity.field_errors(gpu, orc, w["nodes"], w["Q"])
    worst = max(errs, key=errs.get)
    assert errs[worst] <= tol, (worst, errs[worst])
    return errs[worst]


# small stand-ins of the five BASELINE.json configs; the turbulence fields use k0 = 2 so that the small meshes keep a
# resolution (8-12 cells per peak wavelength) that does not produce near-vacuum reconstructed states
CASES_1STEP = [
    ("sine", 16, 1, None), ("sine", 16, 0, None), ("sine", 8, 1, None),
    ("tgv", 16, 1, None), ("tgv", 16, 0, None),
    ("tgv_curv", 12, 1, None), ("freestream_curv", 8, 1, None),
    ("iso_sub", 16, 1, 2.0), ("iso_sup", 24, 1, 2.0), ("iso_sup", 16, 0, 2.0),
    ("tgv_sup", 24, 1, None),                # Taylor-Green vortex at Ma = 1.25
    ("tgv_shear", 12, 1, None), ("tgv_shear", 8, 0, None),      # affine sheared mesh: constant non-symmetric J0
    ("jump_blob", 12, None, None), ("jump_oblique", 12, None, None), ("jump_oblique_linear", 12, None, None),      # reading R9 fires by an O(1) margin
]


@pytest.mark.parametrize("name,n,nonlinear,k0", CASES_1STEP)
def test_one_step_parity(name, n, nonlinear, k0):
    w = parity.build_case(name, n, nonlinear, k0)
    _check(w, 1, TOL_1)


def _shock_tube_case():
    """Two Sod tubes back to back, periodic, through the 3-D code: exercises chi -> 0, the ENO weights, the numerical
    collision time and the one-sided interface values."""
    ni, nj, nk = 48, 4, 5
    nodes = inputs.cartesian_nodes((ni, nj, nk), 0.0, 1.0)
    nodes[1] *= nj / ni; nodes[2] *= nk / ni
    x = (np.arange(ni) + 0.5) / ni
    left = (x > 0.25) & (x < 0.75)
    one = np.ones((nk, nj, ni))
    rho = np.where(left, 1.0, 0.125)[None, None, :] * one; p = np.where(left, 1.0, 0.1)[None, None, :] * one
    Q = inputs.prim_to_cons(rho, 0 * one, 0 * one, 0 * one, p)
    prm = dict(inputs.sine_params()); prm.update(tau_c1=0.05, tau_c2=5.0)
    return dict(nodes=nodes, Q=Q, G=None, D=None, params=prm, nonlinear=1, cfl=0.5)


def test_shock_tube_parity():
    w = _shock_tube_case()
    _check(w, 1, TOL_1)
    # 40 steps: the north_star bound grows from 1e-10 (1 step) to 1e-8 (100 steps); 40/100 of the latter.  The shock
    # makes the ENO weights ~(IS+eps)^-5 amplify round-off five-fold per evaluation.
    _check(w, 40, 4e-9)


@pytest.mark.parametrize("name", ["jump_blob", "jump_oblique_linear"])
def test_positivity_fallback_parity(name):
    """Reading R9 with hundreds of Gauss-point states replaced in every stage (tests/test_oracle_pins2.py shows the
    margins: rho of a replaced state below -0.5 rho_cell): the decision is taken on the same fp64 expression on both
    sides (csrc/cgks_common.cuh admissible(), oracle/cgks_ref.c reconstruct_all), so parity holds element by element."""
    from oracle import ref
    w = parity.build_case(name)
    so = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=w["nonlinear"])); so.set_state(w["Q"])
    so.reconstruct()
    assert so.fallback_stats()[0] > 200
    so.close()
    _check(w, 1, TOL_1)
    _check(w, 5, 5 * TOL_1)


def test_rough_field_one_step_parity_and_robustness():
    """Badly under-resolved Ma_t = 1 field (16^3, k0 = 8; the case VERDICT r1 item 3 names): the fallback (reading R9)
    fires, and some ADMITTED Gauss-point states are near vacuum (internal energy 8e-6 of the total energy), where the
    kinetic flux has a condition number of ~1e6.  Checked: (i) both sides replace exactly the same points; (ii) the
    reconstructed values agree to 1e-13 everywhere; (iii) after one step every element agrees to 1e-10 wherever the
    ORACLE ITSELF is well conditioned, i.e. where a 2-ulp relative perturbation of its input moves its own result by less
    than 1e-12 (> 95 % of the elements), and within 200 x the oracle's own sensitivity elsewhere; then the run must stay
    physical and conservative."""
    from oracle import ref
    from paper_2508_08965_b200 import binding
    w = parity.build_case("iso_sup", 16, 1)
    so = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1)); so.set_state(w["Q"])
    pvo, _ = so.reconstruct()
    nfall = so.fallback_stats()[0]
    so.close()
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1)); s.set_state(w["Q"])
    pv, _ = s.debug_stage()
    s.close()
    pvg = np.moveaxis(pv.cpu().numpy(), (0, 1), (3, 4))
    adm = pvg[..., 0] * pvg[..., 4] - 0.5 * ((pvg[..., 1] * pvg[..., 1] + pvg[..., 2] * pvg[..., 2]) + pvg[..., 3] * pvg[..., 3])
    bad_g = ~((pvg[..., 0] > 0) & (adm > 0))
    Qc = np.moveaxis(w["Q"], 0, -1)[:, :, :, None, :]
    flat_o = (np.abs(pvo[..., 5:]).max(-1) == 0) & (np.abs(pvo[..., :5] - Qc).max(-1) == 0)
    assert nfall > 0 and bad_g.sum() == nfall and np.array_equal(bad_g, flat_o)
    assert np.abs(pvg - pvo)[~bad_g].max() < 1e-13 * np.abs(pvo).max()
    assert ((adm / (Qc[..., 0] * Qc[..., 4]) < 1e-4) & ~bad_g).any()           # a near-vacuum state is admitted
    orc, dts = parity.run_oracle(w, 1)
    gpu, dts_gpu = parity.run_gpu(w, 1, dts=dts)
    assert abs(dts_gpu[0] / dts[0] - 1) <= 1e-13
    err = parity.element_errors(gpu, orc, w["nodes"], w["Q"])
    sens = None
    for seed in (1, 2):
        w2 = dict(w); w2["Q"] = w["Q"] * (1.0 + 4.4e-16 * np.random.default_rng(seed).uniform(-1, 1, w["Q"].shape))
        pert, _ = parity.run_oracle(w2, 1, dts=dts)
        e2 = parity.element_errors(pert, orc, w["nodes"], w["Q"])
        sens = e2 if sens is None else {k: np.maximum(sens[k], e2[k]) for k in e2}
    nwell = ntot = 0
    for k in err:
        well = sens[k] < 1e-12
        nwell += int(well.sum()); ntot += well.size
        assert err[k][well].max() <= TOL_1, (k, err[k][well].max())
        assert (err[k][~well] <= 200 * sens[k][~well]).all(), k
    assert nwell > 0.95 * ntot, (nwell, ntot)
    gpu, _ = parity.run_gpu(w, 50)
    assert np.isfinite(gpu[0]).all() and gpu[0][0].min() > 0
    np.testing.assert_allclose(gpu[0].sum(axis=(1, 2, 3)), w["Q"].sum(axis=(1, 2, 3)), rtol=1e-12, atol=1e-9)


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
    slot = 480
    budget = fixed + 6 * slot * 144 * 8                  # 6 slots of reconstructed face values -> slab depth 4 -> 3 chunks
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1), budget_bytes=budget)
    assert s.slab_depth() == 4
    s.close()
    slab, _ = parity.run_gpu(w, 2, budget_bytes=budget)
    for a, b in zip(full, slab):
        assert np.array_equal(a, b)
    _check(w, 2, TOL_1 * 2, budget=budget)


@pytest.mark.parametrize("case", ["tgv_curv", "iso_sup", "ragged", "jump"])
def test_sweep_pipeline_against_the_three_kernel_pipeline(case, monkeypatch):
    """The product path does flux + update in one sweep kernel per face direction (csrc/kernels_fused.cuh); the
    three-kernel pipeline of rounds 1-2 (flux -> face-flux buffer -> update) lives on in the TEST-ONLY build libcgks_ab.so
    (build.build_ab(), -DCGKS_AB_SPLIT_PIPELINE), loaded here in place of the product library for the second run.
    They order the sums of Eq. 8-9 differently (direction by direction and Gauss-point quads against face by face), so
    they agree to round-off, not bit for bit; both match the oracle at 1e-10 per step."""
    from paper_2508_08965_b200 import binding, build
    ab_path = build.build_ab()
    if case == "ragged":
        nodes = inputs.cartesian_nodes((13, 9, 7), 0.0, 2.0 * np.pi); nodes[1] *= 0.8; nodes[2] *= 1.3
        w = dict(nodes=nodes, Q=inputs.taylor_green(nodes), G=None, D=None, params=inputs.tgv_params(Re=100.0), nonlinear=1, cfl=0.5)
    elif case == "jump":
        w = parity.build_case("jump_blob", 12, 1)
    else:
        w = parity.build_case(case, 12, 1, 2.0 if case == "iso_sup" else None)
    orc, dts = parity.run_oracle(w, 2)
    assert b"TEST BUILD" not in binding.lib().cgks_version()
    sweep, _ = parity.run_gpu(w, 2, dts=dts)
    monkeypatch.setattr(binding, "LIB_PATH", ab_path); monkeypatch.setattr(binding, "_lib", None)
    assert b"TEST BUILD" in binding.lib().cgks_version()
    split, _ = parity.run_gpu(w, 2, dts=dts)
    monkeypatch.undo()                                   # back to the product library (the cached handle is restored with it)
    assert b"TEST BUILD" not in binding.lib().cgks_version()
    e_ab = parity.field_errors(sweep, split, w["nodes"], w["Q"])
    e_sw = parity.field_errors(sweep, orc, w["nodes"], w["Q"])
    e_sp = parity.field_errors(split, orc, w["nodes"], w["Q"])
    print(case, "sweep vs split %.1e, sweep vs oracle %.1e, split vs oracle %.1e" % (max(e_ab.values()), max(e_sw.values()), max(e_sp.values())))
    assert max(e_ab.values()) <= (1e-10 if case == "jump" else 1e-11), max(e_ab, key=e_ab.get)
    assert max(e_sw.values()) <= 2 * TOL_1 and max(e_sp.values()) <= 2 * TOL_1


def test_sweep_lines_cut_into_segments():
    """The sweep kernels cut the j- and k-lines into segments (each starts with one recomputed face); on a mesh with many
    more cells along j and k than the shortest segment (24) the result must not depend on it: a 8 x 60 x 56 mesh against the
    oracle, and bit-identical to its own k-slab pipeline (other k-segments, other first faces)."""
    from paper_2508_08965_b200 import binding
    shape = (8, 60, 56)
    nodes = inputs.cartesian_nodes(shape, 0.0, 2.0 * np.pi)
    w = dict(nodes=nodes, Q=inputs.taylor_green(nodes), G=None, D=None, params=inputs.tgv_params(Re=100.0), nonlinear=1, cfl=0.5)
    _check(w, 1, TOL_1)
    full, _ = parity.run_gpu(w, 2)
    n = shape[0] * shape[1] * shape[2]; plane = shape[0] * shape[1]
    slot = 480
    budget = 3 * 80 * n * 8 + 5 * n * 8 + 37 * n * 8 + 4096 + 30 * slot * plane * 8
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1), budget_bytes=budget)
    assert 24 < s.slab_depth() < shape[2]          # two chunks, the first longer than the shortest segment
    s.close()
    slab, _ = parity.run_gpu(w, 2, budget_bytes=budget)
    for a, b in zip(full, slab):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("name,n,k0", [("sine", 16, None), ("iso_sup", 16, 2.0), ("tgv", 16, None),
                                       ("tgv_curv", 16, None), ("tgv_shear", 12, None), ("iso_sub", 24, 4.0)])
def test_hundred_step_parity(name, n, k0):
    """100 S2O4 steps, every field <= 1e-8 (north_star), on small stand-ins of all five configs (config 3: tgv_curv)."""
    w = parity.build_case(name, n, 1, k0)
    _check(w, 100, TOL_100)


def test_hundred_step_parity_supersonic_k0_8():
    """Ma_t = 1.0 with the full-size spectrum (k0 = 8) on 48^3, 100 steps: the nearest oracle-affordable stand-in for the
    128^3 variant SURVEY.md 8(d) names for the 100-step parity of config 5 (about 80 s of oracle time on 16 cores)."""
    w = parity.build_case("iso_sup", 48, 1, 8.0)
    _check(w, 100, TOL_100)


def test_own_dt_multi_step():
    """The library steps with its OWN cgks_compute_dt for 20 steps (no oracle dt is fed in) and still matches."""
    w = parity.build_case("tgv_curv", 12, 1)
    _check(w, 20, 20 * TOL_1, own_dt=True)
    w = parity.build_case("iso_sup", 16, 1, 2.0)
    _check(w, 20, 20 * TOL_1, own_dt=True)


def test_supersonic_taylor_green_thirty_steps():
    """SURVEY.md 8(f) NEXT-2 (Ma = 1.25): 30 steps (t = 1.8, before the shocklets form).  On a 16^3 mesh the
    later, shocked evolution amplifies round-off exponentially in BOTH implementations (x10 per ~4 steps: 4e-10 at 30
    steps, 7e-5 at 60, O(0.1) at 100 between oracle and GPU), so a 100-step element-wise comparison is meaningless
    at a resolution the oracle can afford; the bound used is 30/100 of the north_star 100-step bound."""
    w = parity.build_case("tgv_sup", 16, 1)
    _check(w, 30, 3e-9)


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
        binding.Solver(nodes, prm, workspace_nbytes=3 * 80 * 512 * 8 + (1 << 16))   # state fits, no room for a slab
    assert e.value.code == binding.CGKS_ENOMEM
    with pytest.raises(binding.CgksError) as e:
        binding.Solver(nodes, prm, workspace_nbytes=4096)
    assert e.value.code == binding.CGKS_ENOMEM
    bad = nodes.copy(); bad[0, 2, 3, -1] += 0.3                   # one node of the last plane: period vector not constant
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
    w = parity.build_case("iso_sup", 16, 1, 2.0)
    so = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1)); so.set_state(w["Q"])
    _, chi_o = so.reconstruct()
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1)); s.set_state(w["Q"])
    s.debug_stage()
    chi_g = s.chi().cpu().numpy()
    assert np.abs(chi_g - chi_o).max() < 1e-12
    s.close()
    # the shock tube exercises the adaptive fallback
    w = _shock_tube_case()
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1)); s.set_state(w["Q"])
    s.debug_stage()
    chi_g = s.chi().cpu().numpy()
    assert chi_g.min() < 1e-3 and (chi_g[0] < 0.99).mean() > 0.05
    s.close()


def test_special_functions_of_the_flux_kernel():
    """csrc/fastmath64.cuh (branch-free reciprocal, rsqrt, exp, erfc with its exp(-x^2)) against mpmath (40 digits) on
    sampled arguments: relative error <= 2e-15; dense checks against numpy/scipy, whose own erfc and exp(-x*x) carry
    the rounding error of x*x (up to 6e-14 at |x| = 26), with correspondingly looser bounds."""
    import mpmath as mp
    from scipy import special
    from paper_2508_08965_b200 import binding
    mp.mp.dps = 40
    rng = np.random.default_rng(7)
    x = np.concatenate([10.0 ** rng.uniform(-12, 12, 20000), rng.uniform(0.5, 2.0, 20000)])
    np.testing.assert_allclose(binding.debug_math(0, x), 1.0 / x, rtol=4e-16)
    np.testing.assert_allclose(binding.debug_math(1, x), 1.0 / np.sqrt(x), rtol=6e-16)
    xl = np.concatenate([x, rng.uniform(0.99, 1.01, 20000), [1.0, 2.0 ** 0.5, 0.5 ** 0.5, 1.4142135623730951, 1.4142135623730954]])
    gl = binding.debug_math(5, xl)
    for a, b in zip(xl[::97], gl[::97]):         # the power law of the viscosity: log against mpmath, absolute 2e-16 near 1
        r = mp.log(mp.mpf(float(a)))
        assert abs(mp.mpf(float(b)) - r) <= 3e-16 * max(abs(r), mp.mpf(1) / 8), a
    np.testing.assert_allclose(gl, np.log(xl), rtol=1e-15, atol=3e-17)
    xt = np.concatenate([rng.uniform(0.0, 12.0, 20000), 10.0 ** rng.uniform(-8, 0, 5000), [0.0, 5.0, 40.0]])
    np.testing.assert_allclose(binding.debug_math(6, xt), np.tanh(xt), rtol=0, atol=3e-16)      # the GENO path function: absolute accuracy
    xe = np.concatenate([rng.uniform(-700, 10, 20000), rng.uniform(-1, 1, 20000)])
    np.testing.assert_allclose(binding.debug_math(2, xe), np.exp(xe), rtol=1e-15)
    xu = np.array([-745.0, -760.0, -800.0, -1e5, -1e300])
    assert np.all(binding.debug_math(2, xu) <= 1e-323 * 2)          # underflows gradually to 0, never garbage
    xs = np.concatenate([rng.uniform(-6, 6, 40000), [0.0, 1e-300, -1e-300, 30.0, -30.0]])
    np.testing.assert_allclose(binding.debug_math(3, xs), special.erfc(xs), rtol=5e-14, atol=1e-300)
    np.testing.assert_allclose(binding.debug_math(4, xs), np.exp(-xs * xs), rtol=1e-14, atol=1e-300)
    mp.mp.dps = 40
    xm = np.concatenate([rng.uniform(-6, 6, 600), rng.uniform(6, 26, 200), rng.uniform(-1e-3, 1e-3, 100)])
    xa = -np.abs(xm) * 25
    ge = binding.debug_math(3, xm); gq = binding.debug_math(4, xm); gx = binding.debug_math(2, xa)
    for a, b, c, d, e in zip(xm, ge, gq, gx, xa):
        am = mp.mpf(float(a))
        assert abs(mp.mpf(float(b)) / mp.erfc(am) - 1) < 2e-15, a
        assert abs(mp.mpf(float(c)) / mp.exp(-am * am) - 1) < 2e-15, a
        assert abs(mp.mpf(float(d)) / mp.exp(mp.mpf(float(e))) - 1) < 2e-15, e


def _block(t, lo, size):
    """Periodic sub-block [lo, lo+size)^3 of a (..., n, n, n) torch tensor (wraps around), as numpy."""
    import torch
    n = t.shape[-1]
    idx = [torch.arange(l, l + size, device=t.device) % n for l in lo]      # lo = (k0, j0, i0)
    return t.index_select(-3, idx[0]).index_select(-2, idx[1]).index_select(-1, idx[2]).cpu().numpy()


@pytest.mark.parametrize("n,nblocks,Ma_t,seed", [(384, 6, 1.0, 5), (96, 4, 1.0, 5), (128, 4, 0.5, 4)])
def test_full_size_sampled_blocks(n, nblocks, Ma_t, seed):
    """BASELINE.json config 5 at its full size (384^3, the configuration bench.py times: slab pipeline, Cartesian
    kernels), one S2O4 step, checked on sampled 16^3 blocks the oracle can compute on their own: a cell's new state
    depends on cell averages within index distance 6 (bootstrap 2 + two stages of 2), so the oracle run on the periodic
    28^3 block around a sample reproduces the inner 16^3 exactly, whatever happens at the block's own (wrong) periodic
    seam.  Blocks are seeded, and include the periodic seam of the full mesh and a slab boundary of the pipeline.
    The 96^3 case runs the same check with a workspace that forces a slab depth of 12; the 128^3 case is BASELINE.json
    config 4 (Ma_t = 0.5, seed 4) at its full size, also through the slab pipeline."""
    import torch
    from oracle import ref
    from paper_2508_08965_b200 import binding
    dev = torch.device("cuda", 0)
    free, _ = torch.cuda.mem_get_info(dev)
    need = (3 * 80 + 5 + 480 + 360) * n ** 3 * 8
    if n == 384 and free < 150e9:
        pytest.skip("needs a 180 GB device")
    k0s = 8.0
    prm = inputs.iso_params(Ma_t, k0=k0s)
    Q = inputs.iso_turbulence(n, seed, Ma_t, k0s, device=dev).contiguous()
    q0 = Q.sum(dim=(1, 2, 3)).cpu().numpy()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info(dev)
    nodes = inputs.cartesian_nodes(n)
    h = 2.0 * np.pi / n
    if n == 384:
        budget = int(free - 42e9)                       # leaves room for the 36 GB of get_state outputs
    else:
        budget = (3 * 80 + 5) * n ** 3 * 8 + 14 * (480 + 360) * n * n * 8 + (1 << 20)      # 14 slots -> slab depth 12
    s = binding.Solver(nodes, binding.make_params(**prm, nonlinear=1), device=dev, budget_bytes=budget)
    S = int(binding.lib().cgks_slab_depth(s._h))
    assert 2 <= S < n
    s.set_state(Q)
    rng = np.random.default_rng(11)
    los = [(n - 9, n - 20, n - 3), (S - 14, 5, 17)] + [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(nblocks - 2)]
    blocks = [(lo, _block(Q, lo, 28)) for lo in los]
    del Q
    # one dt for both sides: the smallest CFL = 0.4 step of the sampled blocks (oracle formula on each block)
    bn = inputs.cartesian_nodes(28, 0.0, 28 * h)
    dts = []
    for lo, qb in blocks:
        o = ref.RefSolver(bn, ref.make_params(**prm, nonlinear=1)); o.set_state(qb); dts.append(o.compute_dt(0.4)); o.close()
    dt = min(dts)
    s.step(dt); s.status()
    Qg, Gg, Dg = s.get_state()
    worst = 0.0
    for lo, qb in blocks:
        o = ref.RefSolver(bn, ref.make_params(**prm, nonlinear=1)); o.set_state(qb); o.step(dt)
        Qo, Go, Do = o.get_state(); o.close()
        inner = (slice(None),) + (slice(6, 22),) * 3
        inner2 = (slice(None), slice(None)) + (slice(6, 22),) * 3
        lo_in = tuple(l + 6 for l in lo)
        gpu = (_block(Qg, lo_in, 16), _block(Gg, lo_in, 16), _block(Dg, lo_in, 16))
        orc = (Qo[inner], Go[inner2], Do[inner2])
        errs = parity.field_errors(gpu, orc, inputs.cartesian_nodes(16, 0.0, 16 * h), qb[inner])
        w = max(errs, key=errs.get)
        assert errs[w] <= TOL_1, (lo, w, errs[w])
        worst = max(worst, errs[w])
    # whole-mesh property at any size: conservation to round-off
    tot = Qg.sum(dim=(1, 2, 3)).cpu().numpy()
    np.testing.assert_allclose(tot, q0, rtol=1e-12, atol=1e-6 * n ** 3 * 1e-6)
    s.close()
    print("worst sampled-block error", worst)


@pytest.mark.parametrize("name,n,k0,budget_slots", [("tgv", 16, None, 0), ("tgv_curv", 12, None, 0), ("iso_sup", 16, 2.0, 0),
                                                    ("tgv_curv", 12, None, 6)])
def test_diagnostics_match_oracle(name, n, k0, budget_slots):
    """cgks_diagnostics (kinetic energy and enstrophy) against the oracle, on the initial state and
    after two steps; also through the slab pipeline (budget_slots > 0)."""
    from oracle import ref
    from paper_2508_08965_b200 import binding
    w = parity.build_case(name, n, 1, k0)
    budget = 0
    if budget_slots:
        cells = n ** 3
        budget = 3 * 80 * cells * 8 + 5 * cells * 8 + 37 * cells * 8 + 4096 + budget_slots * (480 + 360) * n * n * 8
    so = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1)); so.set_state(w["Q"], w["G"], w["D"])
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1), budget_bytes=budget)
    s.set_state(w["Q"], w["G"], w["D"])
    for it in range(2):
        eo, no = so.diagnostics(); eg, ng = s.diagnostics()
        assert abs(eg / eo - 1) < 1e-11, (it, eg, eo)
        assert abs(ng - no) <= 1e-10 * abs(no) + 1e-300, (it, ng, no)
        dt = so.compute_dt(0.5)
        so.step(dt); so.step(dt); s.step(dt); s.step(dt)
    # the state is untouched by the diagnostics
    Q1 = s.get_state()[0].cpu().numpy(); Qo = so.get_state()[0]
    assert np.abs(Q1 - Qo).max() / np.abs(Qo).max() < 1e-10
    s.close(); so.close()


@pytest.mark.parametrize("name,n,steps", [("iso_sub", 64, 200), ("iso_sup", 64, 100), ("tgv_sup", 48, 150)])
def test_long_runs_stay_physical_and_conservative(name, n, steps):
    """Properties that hold at any size (BASELINE.json configs 4-5 and NEXT-2 at reduced mesh size, full step counts where
    affordable): mass, momentum and energy are conserved to round-off over the whole run, the state stays physical
    (cgks_status), the kinetic energy of the decaying turbulence does not grow, and in the supersonic cases the adaptive
    second-order fallback is exercised (chi < 0.99 somewhere)."""
    import torch
    from paper_2508_08965_b200 import binding
    w = parity.build_case(name, n, 1, 8.0 if name.startswith("iso") else None)
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1))
    s.set_state(w["Q"])
    tot0 = w["Q"].sum(axis=(1, 2, 3))
    ek0, en0 = s.diagnostics()
    eks = [ek0]
    for it in range(steps):
        s.step(s.compute_dt(0.5))
        if (it + 1) % 25 == 0:
            eks.append(s.diagnostics()[0])
    s.status()
    Q = s.get_state()[0]
    tot1 = Q.sum(dim=(1, 2, 3)).cpu().numpy()
    scale = np.abs(w["Q"]).sum(axis=(1, 2, 3)).max()
    assert np.abs(tot1 - tot0).max() <= 1e-12 * scale * steps ** 0.5 + 1e-9
    rho = Q[0]
    assert torch.isfinite(Q).all() and rho.min().item() > 0
    if name.startswith("iso"):       # decaying turbulence from a solenoidal field; the supersonic vortex trades kinetic and internal energy
        assert all(b <= a * (1 + 1e-9) for a, b in zip(eks, eks[1:])), eks
    chi = s.chi()
    if name != "iso_sub":
        assert (chi < 0.99).double().mean().item() > 1e-5
    s.close()


@pytest.mark.parametrize("name,n,steps", [("tgv", 64, 3), ("tgv_curv", 64, 2), ("freestream_curv", 64, 2)])
def test_configs_2_and_3_at_full_size(name, n, steps):
    """BASELINE.json configs 2 and 3 at their full 64^3 size (Cartesian and non-orthogonal mesh), a few S2O4 steps,
    every field against the oracle element by element."""
    w = parity.build_case(name, n, 1)
    _check(w, steps, TOL_1 * steps)


# ----------------------------------------------------------------------------------------------- restart parity
def _restart_parity(s, nodes, params, nonlinear, lows, B, tol, dt=None, need_chi_below=None):
    """'Restart parity': take the library's CURRENT state (all 80 dof), cut periodic B^3 blocks,
    give each to the oracle with set_state(Q, G, D), advance both by one S2O4 step of the same dt and compare the
    block's inner cells.  With G and D supplied, a cell's new state depends on cells within index distance 4 (two stages
    of the 2-cell stencil), so the inner (B-8)^3 cells of the oracle's block run are exact whatever happens at the block's
    own (wrong) periodic seam.  Works at any mesh size and after any number of steps."""
    import torch
    from oracle import ref
    from paper_2508_08965_b200 import binding
    Q, G, D = s.get_state()
    n = Q.shape[-1]
    chi_seen = 1.0
    blocks = []
    for lo in lows:
        blocks.append((lo, _block(Q, lo, B), _block(G, lo, B), _block(D, lo, B)))
    del Q, G, D
    torch.cuda.empty_cache()
    if dt is None:
        dt = s.compute_dt(0.5)
    s.step(dt); s.status()
    Q1, G1, D1 = s.get_state()
    worst = 0.0
    for lo, qb, gb, db in blocks:
        # nodes of the block: B+1 planes per direction starting at lo (the mesh is periodic: wrap with the period vector)
        bn = _block_nodes(nodes, lo, B)
        o = ref.RefSolver(bn, ref.make_params(**params, nonlinear=nonlinear)); o.set_state(qb, gb, db)
        _, chi = o.reconstruct()
        inner = (slice(4, B - 4),) * 3
        chi_seen = min(chi_seen, float(chi[(slice(None),) + inner].min()))
        o.step(dt)
        Qo, Go, Do = o.get_state(); o.close()
        lo_in = tuple(l + 4 for l in lo); m = B - 8
        gpu = (_block(Q1, lo_in, m), _block(G1, lo_in, m), _block(D1, lo_in, m))
        orc = (Qo[(slice(None),) + inner], Go[(slice(None), slice(None)) + inner], Do[(slice(None), slice(None)) + inner])
        errs = parity.field_errors(gpu, orc, _block_nodes(nodes, lo_in, m), qb[(slice(None),) + inner])
        w = max(errs, key=errs.get)
        assert errs[w] <= tol, (lo, w, errs[w])
        worst = max(worst, errs[w])
    if need_chi_below is not None:
        assert chi_seen < need_chi_below, chi_seen           # the sampled cells do exercise the adaptive fallback
    return worst, chi_seen


def _block_nodes(nodes, lo, B):
    """Node coordinates (3, B+1, B+1, B+1) of the periodic block of B^3 cells starting at cell lo = (k0, j0, i0)."""
    nodes = np.asarray(nodes)
    nk, nj, ni = (s - 1 for s in nodes.shape[1:])
    per = [nodes[:, nk, 0, 0] - nodes[:, 0, 0, 0], nodes[:, 0, nj, 0] - nodes[:, 0, 0, 0], nodes[:, 0, 0, ni] - nodes[:, 0, 0, 0]]
    idx = []; shift = []
    for l, n in zip(lo, (nk, nj, ni)):
        a = np.arange(l, l + B + 1)
        idx.append(a % n); shift.append(a // n)
    out = nodes[:, idx[0][:, None, None], idx[1][None, :, None], idx[2][None, None, :]].copy()
    for d in range(3):
        sh = shift[d].reshape([-1 if e == d else 1 for e in range(3)])
        out += per[d][:, None, None, None] * sh[None]
    return out


@pytest.mark.parametrize("case", ["iso_sup_384_after_100", "iso_sub_128_after_100", "tgv_sup_128_shocked", "tgv_curv_64_after_100",
                                  "tgv_64_after_100", "iso_sup_64_rough_after_50", "tgv_sup_320_shocked"])
def test_restart_parity(case):
    """Multi-step and shock-active states at sizes the oracle cannot run as a whole (north_star: 100 steps on all five
    configs; Ma = 1.25 vortex once shocklets have formed): the library runs the steps on the full
    mesh, then one further step is compared with the oracle on sampled blocks (see _restart_parity)."""
    import torch
    from paper_2508_08965_b200 import binding
    dev = torch.device("cuda", 0)
    free, _ = torch.cuda.mem_get_info(dev)
    rng = np.random.default_rng(21)
    need_chi = None
    if case == "iso_sup_384_after_100":
        if free < 150e9:
            pytest.skip("needs a 180 GB device")
        n, steps, B, nb = 384, 100, 24, 5
        prm = inputs.iso_params(1.0, k0=8.0); nonlinear = 1
        nodes = inputs.cartesian_nodes(n)
        Q = inputs.iso_turbulence(n, 5, 1.0, 8.0, device=dev).contiguous()
        budget = int(free - 42e9)
    elif case == "iso_sub_128_after_100":
        n, steps, B, nb = 128, 100, 24, 4
        prm = inputs.iso_params(0.5, k0=8.0); nonlinear = 1
        nodes = inputs.cartesian_nodes(n)
        Q = inputs.iso_turbulence(n, 4, 0.5, 8.0, device=dev).contiguous()
        budget = 0
    elif case in ("tgv_sup_128_shocked", "tgv_sup_320_shocked"):
        n = 128 if "128" in case else 320               # the two mesh sizes of the paper's Ma = 1.25 runs
        # the paper's own mesh for this run: about 1400 steps at 320^3, 5 GPU-minutes.  Runs by default on a
        # device that can hold it, so that the driver's GPU run sees the paper's size; CGKS_SKIP_LONG_TESTS=1 opts out
        if n == 320 and os.environ.get("CGKS_SKIP_LONG_TESTS"):
            pytest.skip("CGKS_SKIP_LONG_TESTS is set")
        if n == 320 and free < 150e9:
            pytest.skip("needs a 180 GB device")
        steps, B, nb = 0, 24, 6
        w = inputs.workload("tgv_sup", n); prm = w["params"]; nonlinear = 1; nodes = w["nodes"]; Q = w["Q"]
        budget = 0 if n == 128 else int(free - 30e9)
    elif case in ("tgv_curv_64_after_100", "tgv_64_after_100"):      # BASELINE.json configs[2] and configs[1] at full size
        n, steps, B, nb = 64, 100, 24, 4
        w = inputs.workload("tgv_curv" if "curv" in case else "tgv", n); prm = w["params"]; nonlinear = 1; nodes = w["nodes"]; Q = w["Q"]
        budget = 0
    else:
        n, steps, B, nb = 64, 50, 24, 4
        prm = inputs.iso_params(1.0, k0=8.0); nonlinear = 1
        nodes = inputs.cartesian_nodes(n)
        Q = inputs.iso_turbulence(n, 5, 1.0, 8.0, device=dev).contiguous()
        budget = 0
    s = binding.Solver(nodes, binding.make_params(**prm, nonlinear=nonlinear), device=dev, budget_bytes=budget)
    s.set_state(Q)
    del Q
    if case.startswith("tgv_sup"):
        t = 0.0
        while t < 3.5:                      # shocklets of the Ma = 1.25 vortex form from t ~ 3
            dt = s.compute_dt(0.5); s.step(dt); t += dt
    else:
        for _ in range(steps):
            s.step(s.compute_dt(0.5))
    s.status()
    lows = [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(nb)]
    if case.startswith("tgv_sup"):
        # blocks around the cells where the adaptive weights respond most (smallest chi of the density)
        s.step(s.compute_dt(0.5)); chi = s.chi()[0]
        flat = torch.argsort(chi.flatten())[:: max(1, chi.numel() // 400000)][:3].cpu().numpy()
        for f in flat:
            k, j, i = np.unravel_index(int(f), chi.shape)
            lows.append(((k - B // 2) % n, (j - B // 2) % n, (i - B // 2) % n))
        need_chi = 0.99
    if case == "iso_sup_384_after_100":
        lows[0] = (n - 9, n - 20, n - 3)          # across the periodic seam of the full mesh
    worst, chi_seen = _restart_parity(s, nodes, prm, nonlinear, lows, B, TOL_1, need_chi_below=need_chi)
    s.close()
    print(case, "worst", worst, "min chi in the sampled cells", chi_seen)


def test_flux_tap_matches_oracle_per_axis():
    """Reconstructed face values and the flux kernel's outputs, per face direction and Gauss point, against the oracle's
    (cgks_debug_stage vs cgks_ref_reconstruct / cgks_ref_debug_flux).  Permanent guard for the staged left/right inputs of
    flux_kernel<AXIS> (round 1 saw the wrong plane staged for AXIS = 2 with one form of the address arithmetic,
    DESIGN.md section 7.2): a left/right or plane mix-up in any direction fails here directly, not through a step."""
    from oracle import ref
    from paper_2508_08965_b200 import binding
    for name, n in (("tgv_curv", 10), ("iso_sup", 12)):
        w = parity.build_case(name, n, 1, 2.0 if name == "iso_sup" else None)
        so = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1)); so.set_state(w["Q"])
        dt = so.compute_dt(0.5)
        pvo, _ = so.reconstruct(); fxo = so.debug_flux(dt); so.close()
        s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1)); s.set_state(w["Q"])
        pv, fx = s.debug_stage(dt)
        pv = pv.cpu().numpy(); fx = fx.cpu().numpy(); s.close()
        pvg = np.moveaxis(pv, (0, 1), (3, 4))                      # [24][20][k][j][i] -> [k][j][i][24][20]
        worst = {}
        for c in range(20):
            var = c if c < 5 else (c - 5) // 3
            sc = np.abs(pvo[..., c]).max() + 1e-3 * np.abs(pvo[..., var]).max() * n + 1e-300
            worst["pv"] = max(worst.get("pv", 0.0), np.abs(pvg[..., c] - pvo[..., c]).max() / sc)
        names = ["Fn", "Ft", "VL", "DtL", "VR", "DtR"]
        for ax in range(3):
            for q in range(4):
                g = np.moveaxis(fx[4 * ax + q], 0, -1)             # [30][k][j][i] -> [k][j][i][30]
                o = fxo[ax][..., q, :]
                for grp in range(6):
                    sl = slice(5 * grp, 5 * grp + 5)
                    sc = np.abs(o[..., sl]).max(axis=(0, 1, 2)) + 1e-3 * np.abs(o[..., sl]).max()
                    e = (np.abs(g[..., sl] - o[..., sl]).max(axis=(0, 1, 2)) / sc).max()
                    key = "%s ax%d" % (names[grp], ax)
                    worst[key] = max(worst.get(key, 0.0), e)
        print(name, {k: "%.1e" % v for k, v in worst.items()})
        assert worst["pv"] <= 1e-11, worst
        for k, v in worst.items():
            if k != "pv":
                assert v <= (1e-12 if k[:2] in ("Fn", "VL", "VR") else 2e-11), (name, k, v)


@pytest.mark.parametrize("pinned", [True, False])
def test_run_host_equals_the_device_calls(pinned):
    """cgks_run_host (the end-to-end leg of bench.py) with pinned and with pageable host buffers, Q/G/D in and out:
    bit-identical to set_state -> (compute_dt -> step) x 2 -> get_state, and equal to the oracle at 1e-10 per step."""
    import torch
    from paper_2508_08965_b200 import binding
    w = parity.build_case("sine", 16, 1)
    prm = binding.make_params(**w["params"], nonlinear=1)

    def host(a):
        t = torch.from_numpy(np.ascontiguousarray(a))
        return t.pin_memory() if pinned else t
    Qh, Gh, Dh = host(w["Q"]), host(w["G"]), host(w["D"])
    out = [torch.empty_like(t) for t in (Qh, Gh, Dh)]
    if pinned:
        out = [t.pin_memory() for t in out]
    s = binding.Solver(w["nodes"], prm)
    s.run_host(Qh, Gh, Dh, 0.5, 2, out[0], out[1], out[2])
    s.close()
    ref_dev, _ = parity.run_gpu(w, 2)
    for a, b in zip(out, ref_dev):
        assert np.array_equal(a.numpy(), b)
    orc, _ = parity.run_oracle(w, 2)
    errs = parity.field_errors(tuple(t.numpy() for t in out), orc, w["nodes"], w["Q"])
    assert max(errs.values()) <= 2 * TOL_1
    # Q only (G, D bootstrapped by reading S2, not returned): what bench.py's e2e leg ships
    w2 = parity.build_case("tgv_curv", 12, 1)
    s = binding.Solver(w2["nodes"], binding.make_params(**w2["params"], nonlinear=1))
    Qo = torch.empty_like(host(w2["Q"]))
    s.run_host(host(w2["Q"]), None, None, 0.5, 1, Qo)
    s.close()
    ref_dev, _ = parity.run_gpu(w2, 1)
    assert np.array_equal(Qo.numpy(), ref_dev[0])


def test_compute_dt_at_full_size_against_torch():
    """The CFL reduction at the bench size (384^3, 56.6 M cells; 128^3 on smaller devices) against a torch fp64 evaluation
    of reading S3 on the same state (the full-size reduction was never compared with anything)."""
    import torch
    from paper_2508_08965_b200 import binding
    dev = torch.device("cuda", 0)
    free, _ = torch.cuda.mem_get_info(dev)
    n = 384 if free > 150e9 else 128
    prm = inputs.iso_params(1.0, k0=8.0)
    Q = inputs.iso_turbulence(n, 5, 1.0, 8.0, device=dev).contiguous()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info(dev)
    s = binding.Solver(inputs.cartesian_nodes(n), binding.make_params(**prm, nonlinear=1), device=dev, budget_bytes=int(free - 30e9))
    s.set_state(Q)
    for it in range(2):
        Qc = s.get_state()[0] if it else Q
        h = 2.0 * np.pi / n
        rho = Qc[0]; U = Qc[1:4] / rho
        p = 0.4 * (Qc[4] - 0.5 * rho * (U * U).sum(0))
        c = torch.sqrt(1.4 * p / rho)
        rate = ((U.abs() + c) / h).sum(0)
        mu = prm["mu_ref"] * ((p / rho) / prm["T_ref"]) ** prm["visc_omega"]
        dt_t = min(float((0.5 / rate).min()), float((0.5 * h * h / (3.0 * mu / rho)).min()))
        dt = s.compute_dt(0.5)
        assert abs(dt / dt_t - 1) < 1e-13, (dt, dt_t)
        del Qc, rho, U, p, c, rate, mu
        if it == 0:
            s.step(dt); s.step(s.compute_dt(0.5))
    s.close()

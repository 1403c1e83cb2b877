"""Slab decomposition along k on ONE device: several sub-domain contexts
(cgks_create_slab) that exchange their two-plane halos through cgks_pack_halo / cgks_unpack_halo reproduce the
single-domain run BIT FOR BIT -- same kernels, same per-cell arithmetic, same metrics (computed from the same node values),
and min over sub-domains of the local CFL reductions = the global reduction.  The multi-rank transport (NCCL) is not
exercised here (one GPU); its choreography runs under gloo in tests/test_slab_host.py."""
import numpy as np
import pytest
import torch

from paper_2508_08965_b200 import binding, inputs, slab
from tests import parity

pytestmark = pytest.mark.gpu


def _single(w, nsteps, budget=0):
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=w["nonlinear"]), budget_bytes=budget)
    s.set_state(w["Q"], w["G"], w["D"])
    dts = []
    for _ in range(nsteps):
        dt = s.compute_dt(w["cfl"]); dts.append(dt); s.step(dt)
    s.status()
    out = tuple(t.cpu().numpy() for t in s.get_state()); s.close()
    return out, dts


def _slabs(w, nsteps, world, budget=0):
    nk = w["nodes"].shape[1] - 1
    prm = binding.make_params(**w["params"], nonlinear=w["nonlinear"])
    parts = slab.partition(nk, world)
    subs = [binding.Solver(w["nodes"], prm, slab=p, budget_bytes=budget) for p in parts]
    dev = subs[0].device
    ext = lambda a, p, kd: None if a is None else slab.extended(binding._dev(a, dev), p[0], p[1], kd)
    for s, p in zip(subs, parts):
        s.set_state(ext(w["Q"], p, 1), ext(w["G"], p, 2), ext(w["D"], p, 2))
    dts = []
    for _ in range(nsteps):
        dt = min(s.compute_dt(w["cfl"]) for s in subs); dts.append(dt)
        for stage in (1, 2):
            slab.exchange_halos_local(subs)
            for s in subs:
                s.stage(stage, dt)
    outs = []
    for s in subs:
        s.status()
        outs.append(tuple(t.cpu().numpy() for t in s.get_state()))
        s.close()
    # owned planes of every sub-domain, concatenated along k
    Q = np.concatenate([o[0][:, 2:-2] for o in outs], axis=1)
    G = np.concatenate([o[1][:, :, 2:-2] for o in outs], axis=2)
    D = np.concatenate([o[2][:, :, 2:-2] for o in outs], axis=2)
    return (Q, G, D), dts


@pytest.mark.parametrize("name,n,world", [("tgv", 16, 3), ("tgv_curv", 12, 2), ("tgv_shear", 12, 4), ("iso_sup", 16, 2), ("sine", 16, 5),
                                           ("jump_blob", 12, 3)])
def test_subdomains_equal_the_single_domain_bit_for_bit(name, n, world):
    w = parity.build_case(name, n, None, 2.0 if name == "iso_sup" else None)
    ref, dts_ref = _single(w, 5)
    got, dts = _slabs(w, 5, world)
    assert dts == dts_ref
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)
    # ... and the decomposed run against the ORACLE (not only against the GPU itself), stepping the oracle with the same dts;
    # the bar is north_star's 1e-10 per step
    orc, _ = parity.run_oracle(w, 5, dts=dts)
    errs = parity.field_errors(got, orc, w["nodes"], w["Q"])
    worst = max(errs, key=errs.get)
    assert errs[worst] <= 5 * 1e-10, (worst, errs[worst])


def test_mesh_type_is_a_property_of_the_mesh_not_of_the_slab():
    """A mesh that is uniform Cartesian everywhere except in cell planes 8..10: the sub-domain that holds planes 16, 17, 0..7
    sees only uniform cells, yet it must run the general-mesh kernels like its neighbours and like the single-domain context
    (cgks_create_slab decides on the WHOLE node array), or its cells would not be bit-identical."""
    n = 18
    w = parity.build_case("tgv", n, 1)
    nodes = w["nodes"].copy()
    h = 2.0 * np.pi / n
    bump = 0.1 * h * np.sin(2.0 * np.pi * np.arange(n + 1) / n)             # periodic in i: nodes 0 and n unmoved
    for k in (9, 10):
        nodes[0, k] += bump[None, :]
    w["nodes"] = nodes
    ref, dts_ref = _single(w, 2)
    got, dts = _slabs(w, 2, 3)
    assert dts == dts_ref
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)


def test_subdomain_with_its_own_slab_pipeline():
    """A sub-domain whose workspace forces the k-chunk pipeline inside it (chunks of 2 planes) gives the same bits."""
    w = parity.build_case("tgv_curv", 12, 1)
    ref, _ = _single(w, 3)
    cells = 12 * 12 * 10                      # 6 owned + 4 halo planes
    budget = 3 * 80 * cells * 8 + 5 * cells * 8 + 37 * cells * 8 + 4096 + 4 * (480 + 360) * 144 * 8
    got, _ = _slabs(w, 3, 2, budget=budget)
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)


def test_slab_solver_world_of_one_and_error_codes():
    """SlabSolver (the per-rank driver of slab.py) with a world of one rank: the slab is its own periodic neighbour."""
    w = parity.build_case("tgv", 16, 1)
    ref, dts_ref = _single(w, 3)
    s = slab.SlabSolver(w["nodes"], binding.make_params(**w["params"], nonlinear=1), rank=0, world=1)
    s.set_state_global(torch.from_numpy(w["Q"]))
    dts = []
    for _ in range(3):
        dt = s.compute_dt(0.5); dts.append(dt); s.step(dt)
    Q, G, D = (t.cpu().numpy() for t in s.get_state_owned())
    assert dts == dts_ref
    assert np.array_equal(Q, ref[0]) and np.array_equal(G, ref[1]) and np.array_equal(D, ref[2])
    with pytest.raises(binding.CgksError) as e:
        s.sub.step(1e-3)                                   # a sub-domain needs the halo exchange between the stages
    assert e.value.code == binding.CGKS_EINVAL
    with pytest.raises(binding.CgksError):
        s.sub.stage(2, 1e-3)                               # stages alternate 1, 2
    s.close()
    full = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=1))
    with pytest.raises(binding.CgksError):
        full.pack_halo(0, torch.empty(80 * 2 * 256, dtype=torch.float64, device="cuda"))      # whole-mesh context has no halos
    full.close()
    with pytest.raises(binding.CgksError):
        binding.Solver(w["nodes"], binding.make_params(**w["params"]), slab=(0, 1))          # fewer than 2 owned planes


def test_bench_slab_mode_on_one_rank():
    """bench.py --parallel slab at N = 1 (the code path the driver's scaling run uses): one JSON line with the contract's keys,
    the roofline on its fixed FP64 basis, an end-to-end number with its copies declared."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    # this process may still hold most of the device in torch's caching allocator (the 384^3 cases): give it back to the driver,
    # the child process allocates its own workspace
    import gc
    gc.collect(); torch.cuda.empty_cache()
    r = subprocess.run([sys.executable, "bench.py", "--n", "64", "--steps", "2", "--warmup", "3", "--gpus", "1", "--parallel", "slab",
                        "--no-cpu-baseline"], cwd=root, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["value"] > 0 and d["n_gpus"] == 1 and d["dtype"] == "f64" and d["gpu_launches"] > 0
    assert "slab decomposition" in d["config"]["parallelism"]
    assert d["roofline"]["bound"] == "alu" and 0 < d["roofline"]["frac"] < 1 and "frac_as_built_bytes" in d["roofline"]
    assert d["roofline"]["whole_step"]["compulsory_bytes_per_cell"] == 4000.0
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0

#!/usr/bin/env python
"""bench.py -- cell-updates/s per full S2O4 step of the CGKS-5 hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--n 384] [--impl ours|reference] [--parallel replicas|slab]

One "step" = cgks_compute_dt + cgks_step (two stages: reconstruction + GENO blend, then three sweep kernels: gas-kinetic flux with update/combine)
over the whole mesh.  Workload at N = 1: BASELINE.json configs[4], supersonic isotropic turbulence Ma_t = 1 on the
periodic Cartesian 384^3 mesh (synthetic, seeded).  north_star asks for one GPU, so by default
--gpus N runs N independent replicas (weak scaling, no collective); --parallel slab runs the paper's own parallelisation
instead (1-D slab decomposition along k: two-plane halo exchange per stage over NCCL, one scalar
all-reduce for dt; strong scaling of the one 384^3 problem).
Prints ONE JSON line (rank 0).
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "cell-updates/s per S2O4 step (fp64)"
UNIT = "cell-updates/s"
# Dominant kernel = sweep_kernel (gas-kinetic flux + update/S2O4 combine of one face direction, csrc/kernels_fused.cuh), bound by
# the plain FP64 ALUs.  Two flop counts per face Gauss point (FMA = 2, add/mul = 1), DESIGN.md section 7.2:
#  * EXECUTED by the formulation as built (primed-basis moments, own reciprocal / rsqrt / exp / erfc of csrc/fastmath64.cuh, the
#    quad sums and the combine), from ncu's executed-FP64-op counters on the committed capture profiles/r02k_final.md,
#    per point of an updated cell (the extra first face of every line of a sweep is NOT counted as useful work): stage 1
#    computes F, F_t, Q, Q_t and both one-sided values, stage 2 only the time derivatives.  This is the leanest formulation
#    known to the authors of this repository and is what `roofline.achieved` uses: it can only understate the algorithmic work.
#  * ORACLE-COUNTED (counting-double build of the CPU oracle, oracle/flop_count.py; operations on non-zero
#    operands): the oracle evaluates every term of Eq. 5 with the generic moment routine and needs 7x the arithmetic, so
#    a fraction formed with it exceeds 1; it is printed beside the other, not used as the numerator.
SWEEP_FLOPS_STAGE1 = 2286.0         # per point: 843 DFMA + 471 DMUL + 128 DADD = 1442 FP64 instructions (flux solver ~2180, quad sums and combine ~105)
SWEEP_FLOPS_STAGE2 = 2069.0         # per point: 765 DFMA + 440 DMUL + 99 DADD = 1304 FP64 instructions (flux solver ~2025, quad sums and combine ~45)
FLUX_SOURCE_SHA16 = "944b1a218fc1b5cf"      # sha256 (16 hex digits) of gks_flux.cuh + fastmath64.cuh + math_gen.cuh + kernels_fused.cuh the counts were taken on
FLUX_FLOPS_ORACLE = 15584.0          # tests/test_abi.py checks this constant against oracle/flop_count.py
# Round 1's flux kernel executed 3092.7 / 2923.2 flops per point for the same result (profiles/r01d_kernels_128.md); VERDICT r1's
# target "frac >= 0.50, i.e. flux <= 223 ms per step" is stated in that count, so the fraction in that count is printed too.
FLUX_FLOPS_R01 = (3092.7, 2923.2)
SWEEP_FP64_PIPE_ACTIVE_NCU = (0.621, 0.656)     # sm__pipe_fp64_cycles_active of the stage-1 / stage-2 launches, same capture
# Bytes per point.  Algorithmic: 2 x 20 reconstructed inputs (320 B) + the state records the direction reads and writes, per
# cell and stage 1: 40 (Q^n) + 2 x 320 read, 3 x 640 written; stage 2: 3 x 320 read, 3 x 320 written; / 12 points.
# Measured: dram__bytes_read + write per launch / points, same capture.
SWEEP_BYTES_ALG = (320.0 + (40 + 640 + 1920) / 12.0, 320.0 + (960 + 960) / 12.0)
SWEEP_TRAFFIC = (556.1, 490.7)
SWEEP_FP64_INSTR = (1442.0, 1304.0)            # FP64 instructions per point, stage 1 / stage 2 (same capture)
# reconstruction kernel, per (cell, variable) and stage, ncu capture profiles/r02k_final.md (2 x (12 x 2178 + 5 x 2348)
# = 75.7 kflop and 2 x (12 x 1373 + 5 x 1516) = 48.1 k FP64 instructions per cell and step for the whole pipeline)
RECON_FLOPS_PER_CELLVAR = 2348.0
RECON_FP64_INSTR_PER_CELLVAR = 1516.0
COMPULSORY_BYTES_PER_CELL = 4000.0            # 500 doubles per cell and step, state in / state out only
DRAM_BYTES_PER_CELL_NCU = 21970.0             # profiles/r02k_dram_384.csv: 1.244 TB per 384^3 step
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # SMs x FP64 FMA lanes x 2 x max SM clock = 37.2
# Per-kernel constants by mesh type.  "cart": the uniform-Cartesian kernels (sweep_kernel<1,..>, recon_kernel<1,..>), capture
# profiles/r02k_final.md.  "general": the general-mesh kernels (sweep_kernel<0,..>, recon_kernel<0,..>: metric loads, J0 / J0^-1
# transforms, face frames built from the stored vector areas), capture profiles/r03a_curvilinear.md.
KERNEL_CONSTANTS = {
    "cart": {"sweep_flops": (SWEEP_FLOPS_STAGE1, SWEEP_FLOPS_STAGE2), "sweep_instr": SWEEP_FP64_INSTR, "sweep_bytes": SWEEP_BYTES_ALG,
             "sweep_traffic": SWEEP_TRAFFIC, "pipe_active": SWEEP_FP64_PIPE_ACTIVE_NCU, "recon_flops": RECON_FLOPS_PER_CELLVAR,
             "recon_instr": RECON_FP64_INSTR_PER_CELLVAR, "recon_bytes_cell": 4480.0, "dram_bytes_per_cell": DRAM_BYTES_PER_CELL_NCU,
             "compulsory_bytes_per_cell": COMPULSORY_BYTES_PER_CELL, "capture": "profiles/r02k_final.md"},
    # general meshes, per EXECUTED point like the Cartesian figures (per useful point at 128^3: 2963 / 2924 / 2924 flops in stage 1,
    # 2616 / 2578 / 2579 in stage 2, divided by 1.0625 for AX = 0 and 1.047 for AX = 1, 2); reconstruction 1030 DFMA + 307 DMUL + 449 DADD
    "general": {"sweep_flops": (2791.0, 2462.0), "sweep_instr": (1758.0, 1544.0),
                "sweep_bytes": (SWEEP_BYTES_ALG[0] + 12.7, SWEEP_BYTES_ALG[1] + 12.7),      # + the face's vector area and tangent (48 B per face) and the cell volume
                "sweep_traffic": (571.4, 505.8), "pipe_active": (0.520, 0.602), "recon_flops": 2816.0, "recon_instr": 1786.0,
                "recon_bytes_cell": 4480.0 + 144.0, "dram_bytes_per_cell": 23560.0,      # after r03b (recon reads 16.9 instead of 25.0 GB per launch at 256^3)
                "compulsory_bytes_per_cell": COMPULSORY_BYTES_PER_CELL + 2 * 296.0, "capture": "profiles/r03a_curvilinear.md"},
}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", "--size", dest="n", type=int, default=384, help="cells per direction (default: the 384^3 headline config)")
    ap.add_argument("--workload", default="iso_sup", choices=["iso_sup", "tgv_curv"],
                    help="iso_sup: the headline config (BASELINE.json configs[4], Cartesian); tgv_curv: Taylor-Green vortex on the "
                         "non-orthogonal curvilinear mesh of configs[2] (general-mesh kernels; use --n 256)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default) or the 1-D slab decomposition of the one problem")
    return ap.parse_args()


# ----------------------------------------------------------------------------------------------- clocks sampling
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.index = index; self.rows = []; self._stop = False; self.t = None

    def _run(self):
        while not self._stop:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            time.sleep(0.2)

    def start(self):
        self.t = threading.Thread(target=self._run, daemon=True); self.t.start()

    def stop(self):
        self._stop = True
        if self.t:
            self.t.join(timeout=6)
        sm = []; mx = 0; reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for nm, val in zip(names, r[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------------------------- oracle timing
def oracle_sample(nsteps_hint=None):
    """Times the CPU oracle, as it stands, on a bounded sample of the workload: the same generator (seed 5,
    Ma_t = 1) on a periodic 32^3 mesh with k0 = 2, one S2O4 step per sample."""
    from oracle import ref
    from paper_2508_08965_b200 import inputs
    n = 32
    w = inputs.workload("iso_sup", n, 2.0)
    s = ref.RefSolver(w["nodes"], ref.make_params(**w["params"], nonlinear=1))
    s.set_state(w["Q"])
    cores = os.cpu_count() or 1
    try:
        cores = len(os.sched_getaffinity(0))
    except Exception:
        pass
    omp = os.environ.get("OMP_NUM_THREADS")
    if omp:
        cores = min(cores, int(omp))

    def one():
        t0 = time.perf_counter(); s.step(s.compute_dt(0.5)); return time.perf_counter() - t0
    return s, n, cores, one


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    s, n, cores, one = oracle_sample()
    for _ in range(min(args.warmup, 1)):
        one()
    t = 0.0
    for _ in range(args.steps):
        t += one()
    cells = n ** 3
    val = cells * args.steps / t
    sample = "one S2O4 step per bench step on a periodic %d^3 mesh, same generator (seed 5, Ma_t=1, k0=2)" % n
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "iso_sup Ma_t=1.0 (oracle sample %d^3 of the 384^3 config)" % n},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2508_08965_b200 import binding, inputs, slab

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    use_slab = args.parallel == "slab"
    n = args.n
    curv = args.workload == "tgv_curv"
    if curv:
        if use_slab:
            raise SystemExit("bench.py: --workload tgv_curv runs on a whole-mesh context (no --parallel slab)")
        prm = inputs.tgv_params()
        nodes_np = inputs.curvilinear_nodes(n)
        Q = torch.from_numpy(inputs.taylor_green(nodes_np)).to(dev).contiguous()
        nodes = torch.from_numpy(nodes_np).to(dev)
        del nodes_np
        workload_name = "tgv_curv: Taylor-Green vortex Re=1600 Ma=0.1 on the non-orthogonal periodic curvilinear %d^3 mesh (BASELINE.json configs[2] at %d^3)" % (n, n)
    else:
        k0 = 8.0 if n >= 128 else 2.0
        prm = inputs.iso_params(1.0, k0=k0)
        nodes = torch.from_numpy(inputs.cartesian_nodes(n)).to(dev)
        # replicas: one seed per rank (independent problems); slab: every rank builds the one global field and keeps its slab
        Q = inputs.iso_turbulence(n, 5 + (0 if use_slab else rank), 1.0, k0, device=dev).contiguous()
        workload_name = "iso_sup: supersonic isotropic turbulence Ma_t=1.0, periodic Cartesian %d^3 (BASELINE.json configs[4])" % n
    K = KERNEL_CONSTANTS["general" if curv else "cart"]
    params = binding.make_params(**prm, nonlinear=1)
    if use_slab:
        k_lo, nk_own = slab.partition(n, world)[rank]
        Q = slab.extended(Q, k_lo, nk_own, 1)              # owned planes + two halo planes per side
    Qhost = torch.empty(Q.shape, dtype=torch.float64, pin_memory=True); Qhost.copy_(Q)
    Qout = torch.empty(Q.shape, dtype=torch.float64, pin_memory=True)
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info(dev)
    budget = int(free - (3 << 30))
    if use_slab:
        driver = slab.SlabSolver(nodes, params, rank=rank, world=world, device=dev, budget_bytes=budget)
        solver = driver.sub
        solver.set_state(Q)
        step = driver.step; compute_dt = driver.compute_dt
        cells_rank = nk_own * n * n; cells_job = n ** 3
    else:
        solver = binding.Solver(nodes, params, device=dev, budget_bytes=budget)
        solver.set_state(Q)
        step = solver.step; compute_dt = solver.compute_dt
        cells_rank = n ** 3; cells_job = n ** 3 * world
    del nodes, Q

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def one_step():
        step(compute_dt(0.5))

    for _ in range(max(args.warmup, 3)):
        one_step()
    solver.status()
    # ---- timed region: K steps, device resident, CUDA events on the launching stream; per-kernel profiling is OFF ----
    sampler = ClockSampler(local); sampler.start()
    l0 = solver.launch_count()
    barrier()
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    ev0.record(torch.cuda.current_stream(dev))
    for _ in range(args.steps):
        one_step()
    ev1.record(torch.cuda.current_stream(dev))
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = solver.launch_count() - l0
    # ---- second, short pass with the library's per-kernel CUDA events switched on (fills kernel_ms and the roofline) ----
    psteps = min(args.steps, 3)
    solver.set_profiling(True)
    pev0 = torch.cuda.Event(enable_timing=True); pev1 = torch.cuda.Event(enable_timing=True)
    pev0.record(torch.cuda.current_stream(dev))
    for _ in range(psteps):
        one_step()
    pev1.record(torch.cuda.current_stream(dev))
    torch.cuda.synchronize(dev)
    pms = pev0.elapsed_time(pev1)
    clocks = sampler.stop()
    kms = {k: solver.kernel_ms(k) for k in ("recon", "flux", "update", "cfl")}
    solver.set_profiling(False)
    solver.status()
    chi = solver.chi()
    chi_frac = float((chi < 0.99).double().mean().item())
    del chi
    tmax = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    ms_max = float(tmax.item())
    value = cells_job * args.steps / (ms_max * 1e-3)
    # ---- end to end: host buffers, H2D + one step + D2H per bench step -----------------------------------------------
    e2e = None
    if not args.no_e2e:
        if use_slab:
            def e2e_step():
                solver.set_state(Qhost.to(dev, non_blocking=True))
                step(compute_dt(0.5))
                Qout.copy_(solver.get_state(derivatives=False)[0], non_blocking=True)
                torch.cuda.synchronize(dev)
        else:
            def e2e_step():
                solver.run_host(Qhost, None, None, 0.5, 1, Qout)    # the C-ABI call with HOST buffers; synchronises inside
        e2e_step()                                                   # warm
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            e2e_step()
        barrier()
        te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        nb = int(Qhost.numel() * 8)
        e2e = {"value": cells_job * args.steps / float(te.item()), "unit": UNIT,
               "h2d_bytes_per_step": nb, "d2h_bytes_per_step": nb,
               "note": ("slab mode: every bench step ships this rank's slab of Q (with its halo planes) host->device from pinned memory, "
                        "calls cgks_set_state, one full S2O4 step with the halo exchanges, cgks_get_state, and ships Q back; G and D are "
                        "re-bootstrapped on the device (reading S2)") if use_slab else
                       "every bench step ships the 5 cell-average fields (Q) host->device from pinned memory through cgks_run_host, "
                       "runs one full S2O4 step and ships Q back; the 75 derivative dof per cell (G, D) are NOT shipped: they are "
                       "re-bootstrapped from Q on the device (DESIGN.md reading S2) and not returned, so this is a cold-start step "
                       "(the full 80-dof state would be 36.2 GB each way at 384^3, i.e. PCIe-bound at ~1.5 s per step)"}
    # ---- roofline of the dominant kernel (sweep_kernel: gas-kinetic flux + update, one launch per face direction) ----------
    peak_meas = binding.fp64_peak_tflops(dev) if rank == 0 else None
    fms, fnl = kms["flux"]
    rms, rnl = kms["recon"]
    roof = None
    if fnl > 0:
        # summed over the launches of the profiled steps the useful points are 12 per cell per stage (the extra first face of
        # every line of a sweep is redundant work and not counted)
        pts_per_stage = 12 * cells_rank
        flops = sum(K["sweep_flops"]) * pts_per_stage * psteps
        ach = flops / (fms * 1e-3) / 1e12
        pts_per_launch = 2 * pts_per_stage * psteps / fnl
        sm_mhz = clocks.get("sm_mhz") or 1965.0
        # reconstruction: HBM-bound, 640 B read + 3840 B written per cell (+ the two extra planes of every slab)
        nchunks = 1 if solver_slab(solver) >= (nk_own + 4 if use_slab else n) else math.ceil((nk_own if use_slab else n) / solver_slab(solver))
        planes = (nk_own if use_slab else n) + (2 * nchunks if (use_slab or nchunks > 1) else 0)
        recon_bytes = 2 * psteps * K["recon_bytes_cell"] * planes * n * n
        hbm_peak = measured_hbm_peak()
        # which roof binds (north_star: "the slower of bytes at HBM bandwidth and flops at FP64 peak"): the kernel's arithmetic
        # intensity, executed flops / algorithmic bytes, against the machine balance
        alg_bytes_launch = 0.5 * sum(K["sweep_bytes"]) * pts_per_launch
        gbs = alg_bytes_launch / (fms / fnl * 1e-3) / 1e9
        t_hbm = gbs / hbm_peak[0]; t_alu = ach / FP64_PEAK_NOMINAL_TFLOPS
        # `frac` has ONE basis, the same in every round: the FP64 roof on the flops this kernel executes ("the plain
        # FP64 ALUs bind").  The HBM figure below counts reads of pv, an intermediate buffer this design chooses to materialise
        # between recon_kernel and sweep_kernel, so it is NOT a fraction of a compulsory-traffic roof: it is reported under
        # `hbm_on_pipeline_bytes` / `frac_as_built_bytes` and never selected as `frac`.
        roof = {"bound": "alu", "kernel": "sweep_kernel",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": t_alu,
                "frac_as_built_bytes": t_hbm,
                "bound_note": "frac = executed FP64 flops / time / derived FP64 peak (148 SMs x 64 lanes x 2 x 1.965 GHz); SURVEY.md 8(d) names "
                              "the FP64 ALUs as the binding roof (compulsory HBM traffic is 4.0 kB per cell per step).  frac_as_built_bytes = "
                              "bytes the pipeline AS BUILT moves per point (incl. 320 B of reads of the intermediate pv buffer) / time / HBM peak "
                              "(%.1f GB/s, %s): a utilisation figure of this design's own traffic, not a roofline fraction" % (hbm_peak[0], hbm_peak[1]),
                "hbm_on_pipeline_bytes": {"achieved": gbs, "peak": hbm_peak[0], "unit": "GB/s", "frac_as_built_bytes": t_hbm, "peak_source": hbm_peak[1],
                                          "bytes_per_point": list(K["sweep_bytes"]), "of_which_pv_reads": 320.0},
                "alu": {"achieved": ach, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": t_alu,
                        "frac_at_measured_clock": ach / (FP64_PEAK_NOMINAL_TFLOPS * sm_mhz / 1965.0)},
                "flops_per_point_executed": list(K["sweep_flops"]), "constants_from": K["capture"],
                "flops_per_point_oracle_counted": FLUX_FLOPS_ORACLE,
                "achieved_with_oracle_count": ach * 2.0 * FLUX_FLOPS_ORACLE / sum(K["sweep_flops"]),
                "frac_with_r01_flop_count": ach * sum(FLUX_FLOPS_R01) / sum(K["sweep_flops"]) / FP64_PEAK_NOMINAL_TFLOPS,
                "fp64_pipe_active_ncu": list(K["pipe_active"]),
                "flops_note": "achieved = flops EXECUTED by this kernel's own (leanest known) formulation per useful point / time, so a leaner "
                              "formulation lowers it at equal pipe utilisation (round 1's flux kernel executed 42 % more flops per point for "
                              "the same result); 36 % of its FP64 instructions are DMUL/DADD, which occupy an FMA slot for one flop: at 100 % "
                              "pipe activity this instruction mix reaches 0.79 of the FMA peak; the peak assumes the maximum SM clock, the "
                              "box runs below it under its 1 kW power cap (frac_at_measured_clock uses the sampled clock); the CPU oracle's "
                              "term-by-term evaluation needs 7x the arithmetic, so its count would give a fraction above 1 (DESIGN.md 7.2)",
                "traffic": 0.5 * sum(K["sweep_traffic"]) * pts_per_launch,
                "pipeline_bytes": alg_bytes_launch,
                "traffic_note": "bytes per average launch = ncu dram bytes per point (profiles/r02k_final.md) x points per launch; "
                                "pipeline bytes per point as built %.0f (stage 1) / %.0f (stage 2), 320 of them reads of pv" % tuple(K["sweep_bytes"]),
                "peak_source": "HBM: " + hbm_peak[1] + "; FP64: derived, 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md section 7), "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "peak_dfma_microbench": peak_meas, "frac_of_dfma_microbench": (ach / peak_meas) if peak_meas else None,
                "avg_launch_ms": fms / fnl, "launches": fnl,
                "share_of_step": fms / (pms if pms > 0 else 1.0),
                "kernel_ms_per_step": {k: v[0] / psteps for k, v in kms.items()},
                "profiled_steps": psteps, "profiled_ms_per_step": pms / psteps,
                "whole_step": whole_step(K, pms / psteps, cells_rank, hbm_peak[0], sm_mhz),
                "other_kernels": {"recon_kernel": {
                    "bound": "hbm", "achieved": recon_bytes / (rms * 1e-3) / 1e9 if rms > 0 else None, "peak": hbm_peak[0], "unit": "GB/s",
                    "frac": (recon_bytes / (rms * 1e-3) / 1e9 / hbm_peak[0]) if rms > 0 else None, "peak_source": hbm_peak[1],
                    "algorithmic_bytes_per_cell": K["recon_bytes_cell"], "avg_launch_ms": rms / rnl if rnl else None, "launches": rnl,
                    "share_of_step": rms / (pms if pms > 0 else 1.0)}}}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "strong" if use_slab and world > 1 else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name,
                       "cells": n ** 3, "nonlinear": 1, "cfl": 0.5,
                       "parallelism": ("slab decomposition along k, %d ranks" % world) if use_slab else ("replicas only" if world > 1 else "single GPU"),
                       "l2": "inputs larger than L2 (state %.1f GB per buffer)" % (80 * cells_rank * 8 / 1e9),
                       "slab_depth": solver_slab(solver), "chi_below_0.99_fraction": chi_frac},
            "clocks": clocks, "gpu_launches": launches, "e2e": e2e, "roofline": roof}
    if e2e is not None and world == 1 and not use_slab:
        # the full 80-dof state through the same host call, measured (not estimated) on a mesh whose state fits a pinned buffer
        solver.close(); del solver
        torch.cuda.empty_cache()
        e2e["full_state"] = full_state_e2e(dev, max(args.steps, 2))
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline()
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def whole_step(K, ms_step, cells, hbm_gbs, sm_mhz):
    """The whole S2O4 step against its two floors: compulsory HBM bytes (state in / state out only: stage 1
    reads 80 and writes 80 + 90 doubles per cell, stage 2 reads 80 + 90 and writes 80 -> 500 doubles = 4.0 kB per cell) and
    executed FP64 work.  Everything a reader needs to recompute the fractions is in the object."""
    t = ms_step * 1e-3
    flops_cell = 12.0 * sum(K["sweep_flops"]) + 2.0 * 5.0 * K["recon_flops"]
    instr_cell = 12.0 * sum(K["sweep_instr"]) + 2.0 * 5.0 * K["recon_instr"]
    # one FP64 instruction per lane per cycle: 148 SMs x 64 lanes at the sampled clock
    instr_rate_peak = 148 * 64 * sm_mhz * 1e6
    built = 2 * K["recon_bytes_cell"] + 12.0 * sum(K["sweep_bytes"])
    comp = K["compulsory_bytes_per_cell"]; dram = K["dram_bytes_per_cell"]
    return {"compulsory_bytes_per_cell": comp,
            "pipeline_bytes_per_cell": built,
            "dram_bytes_per_cell_ncu": dram,
            "traffic_ratio": (dram / comp) if dram else None,
            "hbm_floor_ms_compulsory": comp * cells / hbm_gbs / 1e6,
            "frac_of_compulsory_hbm_floor": comp * cells / hbm_gbs / 1e9 / t,
            "hbm_floor_ms_as_built": built * cells / hbm_gbs / 1e6,
            "frac_as_built_bytes": built * cells / hbm_gbs / 1e9 / t,
            "fp64_flops_per_cell_executed": flops_cell,
            "fp64_tflops": flops_cell * cells / t / 1e12,
            "frac_of_fp64_peak": flops_cell * cells / t / 1e12 / FP64_PEAK_NOMINAL_TFLOPS,
            "fp64_instr_per_cell": instr_cell,
            "fp64_pipe_busy_at_sampled_clock": instr_cell * cells / t / instr_rate_peak,
            "note": "dram_bytes_per_cell_ncu and the instruction counts are constants of the committed ncu capture named in bench.py; "
                    "traffic_ratio = measured DRAM bytes / compulsory bytes (1.0 = no intermediate traffic at all)"}


def full_state_e2e(dev, steps, n=128):
    """cgks_run_host with ALL 80 fields per cell (Q, G, D) shipped host->device from pinned memory, one S2O4 step, all 80 shipped
    back: the warm-restart counterpart of the Q-only end-to-end leg, on the 128^3 supersonic-turbulence mesh (the 384^3 state
    is 36 GB each way and would time the PCIe link only)."""
    import torch
    from paper_2508_08965_b200 import binding, inputs
    prm = inputs.iso_params(1.0, k0=8.0)
    nodes = torch.from_numpy(inputs.cartesian_nodes(n)).to(dev)
    Q = inputs.iso_turbulence(n, 5, 1.0, 8.0, device=dev).contiguous()
    sol = binding.Solver(nodes, binding.make_params(**prm, nonlinear=1), device=dev)
    sol.set_state(Q)
    sol.step(sol.compute_dt(0.5))                           # a developed set of derivative dof
    host_in = [torch.empty(t.shape, dtype=torch.float64, pin_memory=True) for t in sol.get_state()]
    for h, t in zip(host_in, sol.get_state()):
        h.copy_(t)
    host_out = [torch.empty(h.shape, dtype=torch.float64, pin_memory=True) for h in host_in]
    torch.cuda.synchronize(dev)
    sol.run_host(*host_in, 0.5, 1, *host_out)               # warm
    t0 = time.perf_counter()
    for _ in range(steps):
        sol.run_host(*host_in, 0.5, 1, *host_out)           # synchronises inside (cgks_status)
    dt = time.perf_counter() - t0
    sol.close()
    nb = int(sum(h.numel() for h in host_in) * 8)
    return {"value": n ** 3 * steps / dt, "unit": UNIT, "cells": n ** 3, "h2d_bytes_per_step": nb, "d2h_bytes_per_step": nb,
            "ms_per_step": 1e3 * dt / steps,
            "note": "iso_sup at %d^3: Q, G and D (80 doubles per cell) host->device from pinned memory, one full S2O4 step, all 80 back" % n}


def measured_hbm_peak():
    """(GB/s, source): the driver-written copy bandwidth of this pool's B200s, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "fallback of /opt/skills/guides/B200_PROFILING.md (no MEASURED_PEAKS.json)"


def solver_slab(solver):
    from paper_2508_08965_b200 import binding
    return int(binding.lib().cgks_slab_depth(solver._h))


def slab_overhead(solver, n, sub_domain=False):
    """Flux launches cover one extra k-plane per chunk of the k-pipeline (recomputed halo) unless the whole mesh is
    resident; a sub-domain (n owned planes + 4 halo planes) always computes the faces of one halo plane."""
    S = solver_slab(solver)
    if S >= n + (4 if sub_domain else 0):
        return (n + 1) / n if sub_domain else 1.0
    nchunks = math.ceil(n / S)
    return (n + nchunks) / n


def cpu_baseline():
    s, n, cores, one = oracle_sample()
    one()
    t = 0.0; k = 0
    while t < 10.0 and k < 8:
        t += one(); k += 1
    return {"value": n ** 3 * k / t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d S2O4 steps on a periodic %d^3 mesh, same generator (seed 5, Ma_t=1, k0=2), after 1 warm step" % (k, n)}


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)

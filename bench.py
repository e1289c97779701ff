"""bench.py — throughput of the quench-simulation hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg0|cfg1|cfg2|cfg3] [--impl ours|reference]

One "step" = one qs_step (S1..S7 of SURVEY.md §8(a)) on the named synthetic coil; default workload: config 3, the
largest single-GPU configuration (864,000 rings).  Prints ONE JSON line.
  value      coupled cell-steps/s, state resident in HBM, CUDA events on the library's stream, max over ranks
  e2e        same metric through the C ABI with HOST buffers: qs_write(J, T) + qs_step + qs_read(J, T, B, E) per step
  roofline   the dominant kernel (fused pair sweep K2): nominal algorithmic flop / measured launch duration against
             the FP64 FMA peak ("bound": "alu"); plus the HBM-bound passes on a lattice larger than L2
  cpu_baseline  the CPU oracle as it stands, timed on a bounded row sample of the same workload on ALL host cores
                (a process pool over target rows; rank 0, N = 1)
  operator_cfg4 the config-4 sweep: y = M x and the CG solve at N = 4,096 / 65,536 / 262,144 / 1,048,576
  cg_active     config 1 (the nonlinear config: ~26 CG iterations per step with the two-level patch preconditioner) next to the headline, whose timed steps
                are linear-regime steps in which the warm-started CG has nothing left to do
N > 1: independent replicas (one coil per GPU, different Jc0 seeds), no data-path collective ("replicas only").
--impl reference: the oracle on the host cores (rank 0 only); no CUDA is touched.
"""
from __future__ import annotations

import argparse
import json
import multiprocessing
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "coupled cell-steps/s"
UNIT = "cell-steps/s"
# nominal algorithmic flop per pair evaluation: K1 = 76, fused K2 = 100
FLOP_K1, FLOP_K2 = 76.0, 100.0
# FP64 peak derived from unit counts: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz
FP64_PEAK_NOMINAL = 148 * 64 * 2 * 1.965e9 / 1e12
# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the ncu --set full captures summarised
# under profiles/ (r02_sweep_field_cfg3.md, r02_hbm_passes.md); None where no capture of that workload exists
NCU_TRAFFIC = {"sweep_field:cfg3_real_coil_60x100x12": 50.1e6 + 0.8e6,      # profiles/r02_sweep_field_cfg3.md
               "material_K5": 671.3e6 + 498.7e6, "heat_K6": 275.2e6 + 102.3e6}  # profiles/r02_hbm_passes.md
NCU_SOURCE = "committed ncu capture (profiles/), not a quantity of this run"
# executed FP64 flop per launch (dadd + dmul + 2 dfma thread instructions) of the same captures: ncu counts what the
# kernel really issues (square roots and the series tail expand to several FP64 instructions), the nominal count does not
NCU_EXEC_FLOP = {"sweep_field:cfg3_real_coil_60x100x12": (809.524212 + 2449.661278 + 2 * 4568.629332) * 1.963472e9 * 1.643487}
DEFAULTS = {"cfg0": (50, 5), "cfg1": (100, 5), "cfg2": (10, 3), "cfg3": (5, 3)}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0)
    ap.add_argument("--warmup", type=int, default=0)
    ap.add_argument("--workload", default="cfg3", choices=sorted(DEFAULTS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the HBM-roofline leg, cfg4 operator leg and cpu_baseline")
    ap.add_argument("--operator", default="pairs", choices=["pairs", "tables"],
                    help="pairs: on-the-fly AGM pair sweeps (north_star, default); tables: lattice-aware operator (f1)")
    ap.add_argument("--leg", default="all", choices=["all", "hbm", "hbm_blocked", "operator"],
                    help="hbm / operator: run only that extra leg and print its JSON (used for the ncu captures)")
    ap.add_argument("--sizes", default="4096,65536,262144,1048576", help="ring counts of the config-4 operator leg")
    ap.add_argument("--cg-budget-s", type=float, default=45.0,
                    help="operator leg: seconds of CG per size above 65,536 rings (0: matvec only)")
    a = ap.parse_args()
    a.sizes = tuple(int(v) for v in a.sizes.split(",") if v)
    k, w = DEFAULTS[a.workload]
    a.steps = a.steps or k
    a.warmup = max(a.warmup or w, 3)
    return a


def load_measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            p = [q.strip() for q in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); smax.append(float(p[1])); power.append(float(p[2]))
            except ValueError:
                continue
            for nm, val in zip(names, p[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py may execute oracle/): cpu_baseline and --impl reference
# ---------------------------------------------------------------------------------------------------
def oracle_row_sample(w, rows, J, T, dt):
    """What one oracle step does for the sampled target cells of the workload, pair by pair against ALL N
    sources: S1 field rows, S2 material law, one S3 application of M (the warm-started residual check of the
    linear regime = what the GPU step executes: one fused sweep).  Returns seconds."""
    from oracle import qs_oracle as qo
    geo, mat = w.geometry, w.material
    chunk = max(1, min(16, int(2e6 // geo.n_rings)))          # rows per evaluation block: bounded memory per worker
    t0 = time.perf_counter()
    Icur = geo.area * J
    Br, Bz = qo.field_eval_rows(geo, Icur, rows, chunk=chunk)
    ml = qo.material_law(mat, J[rows], T[rows], Br, Bz, geo.r[rows], mat.jc0_scale[rows])
    y = qo.matvec_rows(geo, Icur, rows, chunk=chunk)
    _ = y + ml["E"]
    return time.perf_counter() - t0


_POOL_STATE = {}


def _pool_init(w, J, T):
    try:                                                       # one thread per worker: the pool is the parallelism
        from threadpoolctl import threadpool_limits
        _POOL_STATE["limit"] = threadpool_limits(limits=1)
    except Exception:
        pass
    _POOL_STATE.update(w=w, J=J, T=T)


def _pool_rows(rows):
    st = _POOL_STATE
    oracle_row_sample(st["w"], rows, st["J"], st["T"], st["w"].dt)
    return rows.size


def oracle_workers():
    """Worker processes of the oracle legs: one per host core the process may run on."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except Exception:
        return max(1, os.cpu_count() or 1)


class OraclePool:
    """The oracle (unchanged, single-threaded numpy/scipy) run on all host cores: a fork pool over blocks of target
    rows.  Must be created before CUDA is initialised in this process (fork)."""

    def __init__(self, w, workers):
        g = np.random.default_rng(w.seed + 7)
        self.w, self.workers = w, workers
        self.J = 1e7 * g.standard_normal(w.geometry.n_rings)
        self.T = np.full(w.geometry.n_rings, w.geometry.T_bath)
        self.pool = None
        if workers > 1:
            self.pool = multiprocessing.get_context("fork").Pool(workers, initializer=_pool_init, initargs=(w, self.J, self.T))

    def seconds(self, rows):
        """Wall seconds for the oracle to process `rows` (split evenly over the workers)."""
        t0 = time.perf_counter()
        if self.pool is None:
            oracle_row_sample(self.w, rows, self.J, self.T, self.w.dt)
        else:
            parts = [p for p in np.array_split(rows, self.workers) if p.size]
            self.pool.map(_pool_rows, parts, chunksize=1)
        return time.perf_counter() - t0

    def close(self):
        if self.pool is not None:
            self.pool.close()
            self.pool.join()


def run_oracle_sample(w, target_seconds, reps, warm):
    """cell-steps/s of the oracle on a seeded sample of target rows per 'step' (each row against all N sources), all
    host cores; the sample is sized so that one 'step' costs about target_seconds.  Returns (value, seconds, text, cores)."""
    geo = w.geometry
    workers = oracle_workers()
    pool = OraclePool(w, workers)
    try:
        probe = wl.sample_rows(geo.n_rings, 2 * workers, seed=w.seed + 1)
        pool.seconds(probe)                                   # imports, page-in
        per_row = pool.seconds(probe) / probe.size            # wall seconds per row with every worker busy
        n_rows = int(max(workers, min(geo.n_rings, round(target_seconds / max(per_row, 1e-9)))))
        n_rows = max(workers, n_rows // workers * workers)
        rows = wl.sample_rows(geo.n_rings, n_rows, seed=w.seed)
        for _ in range(warm):
            pool.seconds(rows[: max(workers, n_rows // 8)])
        times = [pool.seconds(rows) for _ in range(reps)]
    finally:
        pool.close()
    total = float(np.sum(times))
    text = (f"{rows.size} seeded target cells of {w.name} per step, each against all {geo.n_rings} source rings: "
            f"oracle field rows (S1) + material law (S2) + one M row (S3), scipy K/E + Maxwell bracket; "
            f"{workers} worker processes of {os.cpu_count()} host CPUs")
    return rows.size * reps / total, total, text, workers


def run_oracle_steps(w, steps, warm):
    """The oracle's own qs_step loop (dense operators, Cholesky KKT) — sizes it can hold (N <= 4096)."""
    from oracle import qs_oracle as qo
    orc = qo.Oracle(w.geometry, w.material)
    for _ in range(warm):
        orc.step(w.dt, w.I_ramp)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.step(w.dt, w.I_ramp)
    total = time.perf_counter() - t0
    try:
        from threadpoolctl import threadpool_info
        threads = max([int(d.get("num_threads", 1)) for d in threadpool_info()] or [1])
    except Exception:
        threads = 1
    return (w.geometry.n_rings * steps / total, total,
            f"{steps} full oracle steps of {w.name} (dense M, G_B; Cholesky KKT by LAPACK/BLAS on {threads} threads)", threads)


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = wl.config(int(args.workload[3]))
    if w.geometry.n_rings <= 4096:
        value, total, sample, cores = run_oracle_steps(w, args.steps, args.warmup)
    else:                                                     # whole run ~ 1 minute of wall time on all cores
        value, total, sample, cores = run_oracle_sample(w, 60.0 / (args.steps + args.warmup), args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_rings": w.geometry.n_rings, "dt": w.dt, "I_ramp": w.I_ramp},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------------
def pair_evals(n):
    nb = (n + 31) // 32
    return nb * (nb + 1) // 2 * 1024


def timed_steps(torch, sim, w, steps, host_io=None, cg_iters=None):
    """K steps bracketed by CUDA events on the library's stream.  host_io = (J, T, outs): pinned host buffers
    for the e2e variant (qs_write + qs_step + qs_read every step).  cg_iters: list that receives the projected-CG
    iterations of every step (host-side counter of the handle, no device access).  Returns (ms, launches)."""
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = sim.stats()["launches"]
    sim.sync()
    a.record(sim.stream)
    for _ in range(steps):
        if host_io is not None:
            J, T, outs = host_io
            st = sim.stats()
            sim.write(J, T, st["t"], st["I"])
        rc = sim.step(w.dt, w.I_ramp)
        if rc < 0:
            raise RuntimeError(f"qs_step returned {rc}")
        if cg_iters is not None:
            cg_iters.append(sim.stats()["cg_iters"])
        if host_io is not None:
            sim.read(out=outs)
            J[:] = outs[0]
            T[:] = outs[1]
    b.record(sim.stream)
    sim.sync()
    b.synchronize()
    return a.elapsed_time(b), sim.stats()["launches"] - l0


def pinned(torch, n):
    return torch.empty(n, dtype=torch.float64).pin_memory().numpy()


def hbm_roofline_leg(torch, pkg, hbm_peak, blocked=False):
    """K5 / K6 on a lattice whose arrays exceed L2 (4096 x 4096 cells = 134 MB per array), no pair operator."""
    w = wl.lattice_workload("hbm_4096x4096", 64, 64, 64, 1.0e-3, 30e-3, 1e-4, 0.0, 1, 77, 0.01)
    N = w.geometry.n_rings
    out = {"lattice": "4096x4096 cells (134 MB per FP64 array, > 126 MB L2)"}
    with pkg.QS(w.geometry, w.material, no_operator=True) as sim:
        g = np.random.default_rng(5)
        sim.write(J=1e8 * g.standard_normal(N), T=4.2 + g.random(N))
        sim.set_fields(B=0.1 * g.standard_normal(2 * N), Q=1e3 * g.random(N))
        sub_dt = 1e-9
        for _ in range(3):
            sim.material_eval(1e-4, aux=False)
            sim.heat(sub_dt)
        sim.profile_enable(True)
        for _ in range(10):
            sim.material_eval(1e-4, aux=False)
        for _ in range(20):
            sim.heat(sub_dt)
        pr = sim.profile_read()
    ms_mat = pr["material"][0] / max(pr["material"][1], 1)
    ms_heat = pr["heat"][0] / max(pr["heat"][1], 1)
    if blocked:   # ncu capture of the temporally blocked kernel on this HBM-resident lattice (not its production size)
        mat = w.material
        alpha0 = mat.k_in / (mat.C3 * w.geometry.T_bath ** 2 + mat.C1)
        dt4 = 3.5 * 0.8 * w.geometry.h ** 2 / (4.0 * alpha0)           # m = 4 sub-steps per call = one launch
        with pkg.QS(w.geometry, w.material, no_operator=True, heat_blocked=True) as sim:
            sim.write(J=np.zeros(N), T=4.2 + g.random(N))
            sim.set_fields(Q=1e3 * g.random(N))
            sim.profile_enable(True)
            m4 = sim.heat(dt4)
            for _ in range(10):
                sim.heat(dt4)
            pr4 = sim.profile_read()
        ms4 = pr4["heat"][0] / max(pr4["heat"][1], 1)
        out["heat_K6_blocked_forced"] = {"substeps_per_launch": int(m4), "ms": ms4, "ms_per_substep": ms4 / max(m4, 1),
                                         "note": "forced (QS_GEO_HEAT_BLOCKED): above 2 M cells the library runs one "
                                                 "marching kernel per sub-step instead"}
    # algorithmic bytes per cell: K5 reads J, T, Br, Bz, jc0_scale (40) and
    # writes E, dE/dJ, Q, b (32) = 72; K6 reads H, Q and writes H = 24 per sub-step
    for name, ms, bpc in (("material_K5", ms_mat, 72.0), ("heat_K6", ms_heat, 24.0)):
        gbs = bpc * N / (ms * 1e-3) / 1e9
        out[name] = {"bound": "hbm", "ms": ms, "bytes_per_cell": bpc, "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                     "frac": gbs / hbm_peak, "traffic": NCU_TRAFFIC.get(name)}
    return out


def operator_leg(torch, pkg, fp64_peak, sizes=(4096, 65536, 262144, 1048576), budget_s=45.0):
    """Config 4 (BASELINE.json configs[4]): the standalone y = M x and the CG solve M xh = b, b = M x, on random coaxial
    ring sets at N = 4,096 / 65,536 / 262,144 / 1,048,576.  CG runs to cg_tol = 1e-10 where that takes seconds
    (N <= 65,536) and for a fixed iteration budget above (the softened random-ring matrix has
    cond ~ 1e7), reporting iterations/s and the residual reached."""
    out = {"flop_per_pair_eval_nominal": FLOP_K1, "cg_tol": 1e-10,
           "preconditioner": "block-Jacobi over the sweep's 32-ring Morton blocks (DESIGN.md section 6)"}
    reps = {4096: 20, 65536: 10, 262144: 5, 1048576: 2}
    to_tol = {4096: 20000, 65536: 6000}
    for n in sizes:
        geo, x = wl.free_rings(n)
        with pkg.QS(geo, wl.Material(cg_tol=1e-10, cg_maxit=20000)) as sim:
            xd = torch.from_numpy(x).to(sim.device)
            bd = torch.empty_like(xd)
            xh = torch.empty_like(xd)
            torch.cuda.synchronize()
            for _ in range(2):
                sim.matvec_device(xd, bd)
            sim.profile_enable(True)
            for _ in range(reps.get(n, 2)):
                sim.matvec_device(xd, bd)
            pr = sim.profile_read()
            sim.profile_enable(False)
            ms = pr["sweep_M"][0] / pr["sweep_M"][1]
            pe = pair_evals(n)
            tf = FLOP_K1 * pe / ms * 1e3 / 1e12
            rec = {"matvec_ms": ms, "pair_evals_per_s": pe / ms * 1e3, "pair_interactions_per_s": n * n / ms * 1e3,
                   "nominal_tflops": tf, "frac_of_fp64_peak": tf / fp64_peak}
            # CG: to tolerance, or the iterations that fit the time budget of this size (at least 20)
            if budget_s <= 0.0:
                out[f"N{n}"] = rec
                continue
            per_it_s = ms * 1e-3 * 1.05
            maxit = to_tol.get(n) or int(max(20, min(200, budget_s / per_it_s)))
            sim.solve_device(bd, xh, maxit=2)                 # graph capture, first-touch
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            sim.sync()
            a.record(sim.stream)
            it, relres, rc = sim.solve_device(bd, xh, maxit=maxit)
            b.record(sim.stream)
            sim.sync()
            b.synchronize()
            secs = a.elapsed_time(b) * 1e-3
            chk = torch.empty_like(xd)
            sim.matvec_device(xh, chk)
            sim.sync()
            rec["cg"] = {"mode": "to tolerance 1e-10" if n in to_tol else f"fixed budget of {maxit} iterations",
                         "iterations": it, "seconds": secs, "iters_per_s": it / secs, "relres_reached": relres,
                         "converged": rc == 0,
                         "true_residual_rel_l2": float(torch.linalg.norm(chk - bd) / torch.linalg.norm(bd)),
                         "solution_rel_l2": float(torch.linalg.norm(xh - xd) / torch.linalg.norm(xd))}
        out[f"N{n}"] = rec
    return out


def cg_active_leg(torch, pkg, steps=50, warm=20):
    """Config 1 (single wire, 64 x 64 cells, ramped background field): the config whose steps really iterate the
    projected CG (~26 iterations per step: K1 sweeps + K3/K4 vector kernels), timed next to the headline."""
    w = wl.config(1)
    its = []
    with pkg.QS(w.geometry, w.material) as sim:
        for _ in range(warm):
            sim.step(w.dt, w.I_ramp)
        ms, launches = timed_steps(torch, sim, w, steps, cg_iters=its)
    N = w.geometry.n_rings
    return {"workload": w.name, "n_rings": N, "steps": steps, "warmup": warm, "value": N * steps / (ms * 1e-3), "unit": UNIT,
            "ms_per_step": ms / steps, "cg_iterations_per_step_mean": float(np.mean(its)), "cg_iterations_total": int(np.sum(its)),
            "gpu_launches": int(launches)}


def nonlinear_cfg2_leg(torch, pkg, reach=150, steps=2):
    """Config 2 beyond its linear first ~100 steps (C13): the surface cells of the wires are at Jc and every
    step iterates the projected CG.  The state of step `reach` is produced by a lattice-tables handle (f1: ~6 s) and
    carried over (state + rate) to a pair-sweep handle, which takes one untimed and `steps` timed steps."""
    w = wl.config(2)
    N = w.geometry.n_rings
    with pkg.QS(w.geometry, w.material, lattice_tables=True) as tab:
        for _ in range(reach):
            tab.step(w.dt, w.I_ramp)
        J, T = tab.read(B=False, E=False)[:2]
        st = tab.stats()
        rate = tab.read_rate()
    its = []
    with pkg.QS(w.geometry, w.material) as sim:
        sim.write(J, T, st["t"], st["I"])
        sim.write_rate(rate)
        sim.step(w.dt, w.I_ramp)
        ms, launches = timed_steps(torch, sim, w, steps, cg_iters=its)
    return {"workload": w.name, "operator": "pairs", "window": f"steps {reach + 2}..{reach + 1 + steps} of the trajectory",
            "value": N * steps / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / steps,
            "cg_iterations_per_step_mean": float(np.mean(its)), "gpu_launches": int(launches)}


def gpu_arm(args):
    # the CPU oracle first (rank 0, one GPU, unless --no-extras): its worker pool is forked before this process
    # creates a CUDA context
    cpu_baseline = None
    if int(os.environ.get("RANK", "0")) == 0 and args.gpus == 1 and not args.no_extras and args.leg == "all":
        wb = wl.config(int(args.workload[3]))
        if wb.geometry.n_rings <= 4096:
            v, total, sample, cores = run_oracle_steps(wb, min(args.steps, 20), 1)
        else:
            v, total, sample, cores = run_oracle_sample(wb, 15.0, 1, 0)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "host_cpus": os.cpu_count(), "kind": "oracle",
                        "sample": sample, "seconds": total}
    import torch
    import paper_2403_07666_b200 as pkg

    from paper_2403_07666_b200.replicas import Group, env_rank, replica_seed
    rank, local, world = env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    group = Group("nccl", torch.device("cuda", local))   # no-op for world == 1; replicas only: barrier + max reduce

    def barrier():
        group.barrier()
        torch.cuda.synchronize()

    max_over_ranks = group.max_over_ranks

    cfg = int(args.workload[3])
    w = wl.config(cfg)
    if rank > 0:   # replicas: same coil, another seeded Jc0 perturbation (a parameter study)
        w.material.jc0_scale = wl.jc0_scale(replica_seed(w.seed, rank), w.geometry.n_rings, 0.02 if cfg == 2 else 0.01)
    N = w.geometry.n_rings
    hbm_peak, hbm_src = load_measured_peaks()
    fp64_tf, fp64_mhz = pkg.fp64_peak()
    if args.leg != "all":
        leg = (hbm_roofline_leg(torch, pkg, hbm_peak, blocked=args.leg == "hbm_blocked") if args.leg.startswith("hbm")
               else operator_leg(torch, pkg, fp64_tf, args.sizes, args.cg_budget_s))
        print(json.dumps({"leg": args.leg, **leg}), flush=True)
        return

    sim = pkg.QS(w.geometry, w.material, device=local, lattice_tables=args.operator == "tables")
    # The very first step of a run solves for I' from a cold start: ~60 CG iterations, each a full K1 sweep (minutes at
    # 864,000 rings) - a cost of the first step only, the timed steps are steps of the running trajectory.  For the big
    # coils that first step is taken by a second handle with the lattice-tables operator (f1, ~0.2 s per sweep) and the
    # state AND the rate I' are carried over through qs_read / qs_read_rate -> qs_write / qs_write_rate; the W warm-up
    # steps and the K timed steps then run on the timed (pair-sweep) handle.
    sim_tab, cold_start, first_timed = None, "qs_step on the timed handle", 1
    if args.operator == "pairs" and N > 100000:
        sim_tab = pkg.QS(w.geometry, w.material, device=local, lattice_tables=True)
        sim_tab.step(w.dt, w.I_ramp)
        J1, T1 = sim_tab.read(B=False, E=False)[:2]
        sim.write(J1, T1, sim_tab.stats()["t"], sim_tab.stats()["I"])
        sim.write_rate(sim_tab.read_rate())
        first_timed = 2
        cold_start = ("first step (cold CG solve) on a lattice-tables handle, state + I' carried over by qs_write / "
                      "qs_write_rate; all warm-up and timed steps on the pair-sweep handle")
        if rank > 0 or world > 1 or args.no_extras:
            sim_tab.close()
            sim_tab = None
    for _ in range(args.warmup):
        sim.step(w.dt, w.I_ramp)
    # every leg below times the SAME K steps of the trajectory (the cost of a step drifts along it: config 1 needs more
    # CG iterations as the flux front moves in), so the state after the warm-up is kept and written back between legs
    snapJ, snapT = sim.read(B=False, E=False)[:2]
    snapR = sim.read_rate()
    snap_t, snap_I = sim.stats()["t"], sim.stats()["I"]

    def rewind():
        sim.write(snapJ, snapT, snap_t, snap_I)
        sim.write_rate(snapR)

    # ---- device-resident timing -----------------------------------------------------------------
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    cg_its = []
    ms, launches = timed_steps(torch, sim, w, args.steps, cg_iters=cg_its)
    barrier()
    clocks = sampler.stop()
    # the same K steps again with the library's event profiler recording (per-kernel-class device times for the
    # roofline; the profiler brackets launches with events and disables the CUDA-graph replay of CG iterations,
    # so it stays out of the region `value` is taken from)
    rewind()
    sim.profile_enable(True)
    ms_prof, _ = timed_steps(torch, sim, w, args.steps)
    prof = sim.profile_read()
    sim.profile_enable(False)
    st = sim.stats()
    ms = max_over_ranks(ms)
    value = world * N * args.steps / (ms * 1e-3)
    # ---- end to end through the C ABI with host buffers -----------------------------------------
    J, T = pinned(torch, N), pinned(torch, N)
    outs = [pinned(torch, N), pinned(torch, N), pinned(torch, 2 * N), pinned(torch, N)]
    got = sim.read(out=outs)
    J[:], T[:] = got[0], got[1]
    timed_steps(torch, sim, w, 1, (J, T, outs))
    rewind()
    J[:], T[:] = snapJ, snapT
    barrier()
    ms_e2e, _ = timed_steps(torch, sim, w, args.steps, (J, T, outs))
    barrier()
    ms_e2e = max_over_ranks(ms_e2e)
    e2e = {"value": world * N * args.steps / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 16 * N,
           "d2h_bytes_per_step": 40 * N, "ms_per_step": ms_e2e / args.steps,
           "path": "qs_write(J,T) + qs_step + qs_read(J,T,B,E), pinned host buffers"}
    sim.close()

    # ---- roofline of the dominant kernel (the fused pair sweep K2; K1 when CG iterates) ----------
    kf_ms, kf_n = prof["sweep_field"]
    km_ms, km_n = prof["sweep_M"]
    pe = pair_evals(N)
    dom = "sweep_field" if kf_ms >= km_ms else "sweep_M"
    d_ms, d_n = (kf_ms, kf_n) if dom == "sweep_field" else (km_ms, km_n)
    flop = (FLOP_K2 if dom == "sweep_field" else FLOP_K1) * pe
    if args.operator == "tables":   # block-Toeplitz product: N^2 multiply-adds per table (3 tables in the fused sweep)
        flop = 2.0 * N * N * (3 if dom == "sweep_field" else 1)
    ach = flop / (d_ms / max(d_n, 1) * 1e-3) / 1e12
    kname = (f"qs::sweep_kernel<{'true' if dom == 'sweep_field' else 'false'}> ({dom})" if args.operator == "pairs"
             else f"qs::table_sweep_kernel<R, {'true' if dom == 'sweep_field' else 'false'}> ({dom}, lattice tables)")
    roofline = {"bound": "alu", "kernel": kname,
                "achieved": ach, "peak": fp64_tf, "unit": "TFLOP/s", "frac": ach / fp64_tf,
                "traffic": NCU_TRAFFIC.get(f"{dom}:{w.name}"),
                "traffic_source": NCU_SOURCE if NCU_TRAFFIC.get(f"{dom}:{w.name}") is not None else None,
                "peak_source": "measured in this run: DFMA-chain probe qs_fp64_peak; "
                               f"unit-count peak 148 SM x 64 lanes x 2 x 1.965 GHz = {FP64_PEAK_NOMINAL:.2f}",
                "frac_of_nominal_peak": ach / FP64_PEAK_NOMINAL,
                "flop_per_pair_eval": FLOP_K2 if dom == "sweep_field" else FLOP_K1, "pair_evals_per_launch": pe,
                "launch_ms": d_ms / max(d_n, 1), "launches_timed": d_n,
                "share_of_step": d_ms / ms_prof, "pair_evals_per_s": pe / (d_ms / max(d_n, 1) * 1e-3)}
    ex = NCU_EXEC_FLOP.get(f"{dom}:{w.name}") if args.operator == "pairs" else None
    if ex is not None:   # executed flop per launch from the committed ncu capture / this run's launch time
        ex_tf = ex / (d_ms / max(d_n, 1) * 1e-3) / 1e12
        roofline["executed"] = {"achieved": ex_tf, "unit": "TFLOP/s", "frac": ex_tf / fp64_tf,
                                "source": NCU_SOURCE + ": profiles/r02_sweep_field_cfg3.md (sass_thread_inst_executed_op_d{add,mul,fma})"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_rings": N, "n_turns": w.geometry.n_turns, "dt": w.dt, "I_ramp": w.I_ramp,
                       "operator": args.operator,
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "per-cell arrays fit L2; the pair sweep is FP64-ALU bound, HBM legs use a 134 MB/array lattice",
                       "cg_iterations_timed": int(np.sum(cg_its)), "cg_iterations_per_step_mean": float(np.mean(cg_its)),
                       "cg_note": "linear-regime steps: the warm-started CG is converged on entry, a step is one fused K2 "
                                  "sweep + O(N) passes; see cg_active for steps that iterate" if int(np.sum(cg_its)) == 0 else None,
                       "window": f"steps {args.warmup + first_timed}..{args.warmup + first_timed - 1 + args.steps} of the trajectory from J = 0 (the coil "
                                 "configs are in the linear regime for their first ~100 steps; later steps iterate the CG: "
                                 "nonlinear_cfg2, cg_active, profiles/r02_full_runs.md)",
                       "cold_start": cold_start, "heat_substeps": st["heat_substeps"]},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()}}
    if rank == 0 and world == 1 and not args.no_extras:
        line["issue_model"] = dict(pkg.issue_probe(), unit="SM cycles per DFMA warp-instruction per sub-partition",
                                   note="FP64 pipe rate is 2; a third register operand costs a cycle, and so does every "
                                        "non-FP64 instruction issued beside the DFMAs (DESIGN.md section 6)")
        if args.operator == "pairs":   # SURVEY.md §8(f) f1, same workload: tables over (ir, jr, |dz|) + block-Toeplitz sweeps
            with (sim_tab if sim_tab is not None else pkg.QS(w.geometry, w.material, device=local, lattice_tables=True)) as sim2:
                for _ in range(args.warmup):
                    sim2.step(w.dt, w.I_ramp)
                ms2, _ = timed_steps(torch, sim2, w, args.steps)
                sim2.profile_enable(True)
                timed_steps(torch, sim2, w, args.steps)
                pr2 = sim2.profile_read()
            sw_ms = pr2["sweep_field"][0] / max(pr2["sweep_field"][1], 1)
            line["next_f1_lattice_tables"] = {
                "value": N * args.steps / (ms2 * 1e-3), "unit": UNIT, "ms_per_step": ms2 / args.steps,
                "sweep_ms": sw_ms, "sweep_tflops": 6.0 * N * N / (sw_ms * 1e-3) / 1e12 if sw_ms > 0 else None,
                "note": "not the graded path: north_star fixes on-the-fly AGM pair evaluation"}
        line["roofline_hbm"] = hbm_roofline_leg(torch, pkg, hbm_peak)
        line["roofline_hbm"]["peak_source"] = f"MEASURED_PEAKS.json hbm_gbs ({hbm_src})"
        line["roofline_hbm"]["traffic_source"] = NCU_SOURCE
        line["cg_active"] = cg_active_leg(torch, pkg)
        line["nonlinear_cfg2"] = nonlinear_cfg2_leg(torch, pkg)
        line["operator_cfg4"] = operator_leg(torch, pkg, fp64_tf, args.sizes, args.cg_budget_s)
        line["cpu_baseline"] = cpu_baseline
    if rank == 0:
        print(json.dumps(line), flush=True)
    group.close()


if __name__ == "__main__":
    _args = parse_args()
    if _args.impl == "reference":
        reference_arm(_args)
    else:
        gpu_arm(_args)

"""bench.py — throughput of the quench-simulation hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg0|cfg1|cfg2|cfg3] [--impl ours|reference]

One "step" = one qs_step (S1..S7 of SURVEY.md §8(a)) on the named synthetic coil.  Prints ONE JSON line.
  value      coupled cell-steps/s, state resident in HBM, CUDA events on the library's stream, max over ranks
  e2e        same metric through the C ABI with HOST buffers: qs_write(J, T) + qs_step + qs_read(J, T, B, E) per step
  roofline   the dominant kernel (fused pair sweep K2): nominal algorithmic flop / measured launch duration against
             the FP64 FMA peak ("bound": "alu"); plus the HBM-bound passes on a lattice larger than L2
  cpu_baseline  the CPU oracle as it stands, timed on a bounded row sample of the same workload (rank 0, N = 1)
N > 1: independent replicas (one coil per GPU, different Jc0 seeds), no data-path collective ("replicas only").
--impl reference: the oracle on the host cores (rank 0 only); no CUDA is touched.
"""
from __future__ import annotations

import argparse
import json
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
# under profiles/ (r01_sweep_field_cfg2.md, r01_hbm_passes.md); None where no capture of that workload exists
NCU_TRAFFIC = {"sweep_field:cfg2_mid_solenoid_20x40x16": 11.8e6, "material_K5": 671.4e6 + 498.2e6, "heat_K6": 275.0e6 + 102.4e6}   # r01 captures
# executed FP64 flop per launch (dadd + dmul + 2 dfma thread instructions) of the same captures: ncu counts what the
# kernel really issues (square roots and the series tail expand to several FP64 instructions), the nominal count does not
NCU_EXEC_FLOP = {"sweep_field:cfg2_mid_solenoid_20x40x16": (1178.569285 + 2342.123003 + 2 * 4037.256723) * 1.963764e9 * 102.601792e-3}
DEFAULTS = {"cfg0": (50, 5), "cfg1": (100, 5), "cfg2": (10, 3), "cfg3": (3, 3)}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0)
    ap.add_argument("--warmup", type=int, default=0)
    ap.add_argument("--workload", default="cfg2", choices=sorted(DEFAULTS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the HBM-roofline leg, cfg4 operator leg and cpu_baseline")
    ap.add_argument("--operator", default="pairs", choices=["pairs", "tables"],
                    help="pairs: on-the-fly AGM pair sweeps (north_star, default); tables: lattice-aware operator (f1)")
    ap.add_argument("--leg", default="all", choices=["all", "hbm", "operator"],
                    help="hbm / operator: run only that extra leg and print its JSON (used for the ncu captures)")
    a = ap.parse_args()
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
    t0 = time.perf_counter()
    Icur = geo.area * J
    Br, Bz = qo.field_eval_rows(geo, Icur, rows, chunk=16)
    ml = qo.material_law(mat, J[rows], T[rows], Br, Bz, geo.r[rows], mat.jc0_scale[rows])
    y = qo.matvec_rows(geo, Icur, rows, chunk=16)
    _ = y + ml["E"]
    return time.perf_counter() - t0


def oracle_threads():
    """Threads the oracle legs actually use: the pair-by-pair K/E evaluation is numpy/scipy elementwise code,
    single-threaded; the BLAS pool only sees the tiny row dot products."""
    return 1


def run_oracle_sample(w, n_rows, reps, warm):
    """cell-steps/s of the oracle on `n_rows` seeded target rows per 'step' (each row against all N sources)."""
    geo = w.geometry
    rows = wl.sample_rows(geo.n_rings, n_rows, seed=w.seed)
    g = np.random.default_rng(w.seed + 7)
    J = 1e7 * g.standard_normal(geo.n_rings)
    T = np.full(geo.n_rings, geo.T_bath)
    for _ in range(warm):
        oracle_row_sample(w, rows[: max(1, n_rows // 8)], J, T, w.dt)
    times = [oracle_row_sample(w, rows, J, T, w.dt) for _ in range(reps)]
    total = float(np.sum(times))
    return rows.size * reps / total, total, times


def pick_rows(w, target_seconds):
    """Number of sampled rows so that one oracle 'step' costs about target_seconds on this host."""
    geo = w.geometry
    rows = wl.sample_rows(geo.n_rings, 2, seed=w.seed + 1)
    g = np.random.default_rng(1)
    J = 1e7 * g.standard_normal(geo.n_rings)
    T = np.full(geo.n_rings, geo.T_bath)
    oracle_row_sample(w, rows[:1], J, T, w.dt)
    t = oracle_row_sample(w, rows, J, T, w.dt) / rows.size
    return int(max(2, min(geo.n_rings, round(target_seconds / max(t, 1e-9)))))


def row_sample_text(w, n_rows):
    return (f"{n_rows} seeded target cells of {w.name} per step, each against all {w.geometry.n_rings} source rings: "
            "oracle field rows (S1) + material law (S2) + one M row (S3), scipy K/E + Maxwell bracket")


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
    return w.geometry.n_rings * steps / total, total, f"{steps} full oracle steps of {w.name} (dense M, G_B; Cholesky KKT)"


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = wl.config(int(args.workload[3]))
    if w.geometry.n_rings <= 4096:
        value, total, sample = run_oracle_steps(w, args.steps, args.warmup)
    else:
        n_rows = pick_rows(w, 60.0 / (args.steps + args.warmup))       # whole run ~ 1 minute of CPU work
        value, total, _ = run_oracle_sample(w, n_rows, args.steps, args.warmup)
        sample = row_sample_text(w, n_rows)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_rings": w.geometry.n_rings, "dt": w.dt, "I_ramp": w.I_ramp},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------------
def pair_evals(n):
    nb = (n + 31) // 32
    return nb * (nb + 1) // 2 * 1024


def timed_steps(torch, sim, w, steps, host_io=None):
    """K steps bracketed by CUDA events on the library's stream.  host_io = (J, T, outs): pinned host buffers
    for the e2e variant (qs_write + qs_step + qs_read every step).  Returns (ms, launches)."""
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


def hbm_roofline_leg(torch, pkg, hbm_peak):
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
    # algorithmic bytes per cell: K5 reads J, T, Br, Bz, jc0_scale (40) and
    # writes E, dE/dJ, Q, b (32) = 72; K6 reads H, Q and writes H = 24 per sub-step
    for name, ms, bpc in (("material_K5", ms_mat, 72.0), ("heat_K6", ms_heat, 24.0)):
        gbs = bpc * N / (ms * 1e-3) / 1e9
        out[name] = {"bound": "hbm", "ms": ms, "bytes_per_cell": bpc, "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                     "frac": gbs / hbm_peak, "traffic": NCU_TRAFFIC.get(name)}
    return out


def operator_leg(torch, pkg, fp64_peak):
    """Config 4: standalone y = M x on random rings (N = 262,144), plus CG iterations/s at N = 65,536."""
    out = {}
    n = 262144
    geo, x = wl.free_rings(n)
    with pkg.QS(geo, wl.Material()) as sim:
        xd = torch.from_numpy(x).to(sim.device)
        yd = torch.empty_like(xd)
        torch.cuda.synchronize()
        for _ in range(2):
            sim.matvec_device(xd, yd)
        sim.profile_enable(True)
        for _ in range(5):
            sim.matvec_device(xd, yd)
        pr = sim.profile_read()
    ms = pr["sweep_M"][0] / pr["sweep_M"][1]
    pe = pair_evals(n)
    out["matvec_N262144"] = {"ms": ms, "pair_evals_per_s": pe / ms * 1e3, "pair_interactions_per_s": n * n / ms * 1e3,
                             "nominal_tflops": FLOP_K1 * pe / ms * 1e3 / 1e12,
                             "frac_of_fp64_peak": FLOP_K1 * pe / ms * 1e3 / 1e12 / fp64_peak}
    n = 65536
    geo, x = wl.free_rings(n)
    with pkg.QS(geo, wl.Material(cg_tol=1e-10)) as sim:
        bd = torch.from_numpy(x).to(sim.device)
        xd = torch.empty_like(bd)
        torch.cuda.synchronize()
        sim.solve_device(bd, xd, maxit=5)
        sim.profile_enable(True)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(sim.stream)
        it, relres, _ = sim.solve_device(bd, xd, maxit=50)
        b.record(sim.stream)
        sim.sync()
        b.synchronize()
        pr = sim.profile_read()
    # config 4 (b): b = M x, solve M xh = b to cg_tol = 1e-10 at N = 4096 (ill-conditioned: cond ~ 1e7), check xh ~ x
    n4 = 4096
    geo4, x4 = wl.free_rings(n4)
    with pkg.QS(geo4, wl.Material(cg_tol=1e-10, cg_maxit=20000)) as sim:
        xd = torch.from_numpy(x4).to(sim.device)
        bd4 = torch.empty_like(xd)
        xh = torch.empty_like(xd)
        torch.cuda.synchronize()
        sim.matvec_device(xd, bd4)
        sim.sync()
        a4, b4 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a4.record(sim.stream)
        it4, rel4, rc4 = sim.solve_device(bd4, xh)
        b4.record(sim.stream)
        sim.sync()
        b4.synchronize()
        chk = torch.empty_like(xd)
        sim.matvec_device(xh, chk)
        sim.sync()
    s4 = a4.elapsed_time(b4) * 1e-3
    out["cg_N4096_to_tolerance"] = {"iterations": it4, "seconds": s4, "iters_per_s": it4 / s4, "relres": rel4,
                                    "converged": rc4 == 0,
                                    "residual_rel_l2": float(torch.linalg.norm(chk - bd4) / torch.linalg.norm(bd4)),
                                    "solution_rel_l2": float(torch.linalg.norm(xh - xd) / torch.linalg.norm(xd))}
    vec_us = 1e3 * pr["cg_vector"][0] / max(it, 1)
    out["cg_N65536"] = {"iterations": it, "iters_per_s": it / (a.elapsed_time(b) * 1e-3), "relres_reached": relres,
                        "sweep_ms_per_iteration": pr["sweep_M"][0] / max(pr["sweep_M"][1], 1),
                        "vector_kernels_us_per_iteration": vec_us,
                        "vector_kernels_GBs": 152.0 * n / (vec_us * 1e-6) / 1e9 if vec_us > 0 else None,
                        "vector_bytes_per_ring": 152.0}
    return out


def gpu_arm(args):
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
        leg = hbm_roofline_leg(torch, pkg, hbm_peak) if args.leg == "hbm" else operator_leg(torch, pkg, fp64_tf)
        print(json.dumps({"leg": args.leg, **leg}), flush=True)
        return

    sim = pkg.QS(w.geometry, w.material, device=local, lattice_tables=args.operator == "tables")
    for _ in range(args.warmup):
        sim.step(w.dt, w.I_ramp)
    # every leg below times the SAME K steps of the trajectory (the cost of a step drifts along it: config 1 needs more
    # CG iterations as the flux front moves in), so the state after the warm-up is kept and written back between legs
    snapJ, snapT = sim.read(B=False, E=False)[:2]
    snap_t, snap_I = sim.stats()["t"], sim.stats()["I"]

    def rewind():
        sim.write(snapJ, snapT, snap_t, snap_I)

    # ---- device-resident timing -----------------------------------------------------------------
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    ms, launches = timed_steps(torch, sim, w, args.steps)
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
                                "source": "profiles/r01_sweep_field_cfg2.md (sass_thread_inst_executed_op_d{add,mul,fma})"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_rings": N, "n_turns": w.geometry.n_turns, "dt": w.dt, "I_ramp": w.I_ramp,
                       "operator": args.operator,
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "per-cell arrays fit L2; the pair sweep is FP64-ALU bound, HBM legs use a 134 MB/array lattice",
                       "cg_iters_last_step": st["cg_iters"], "heat_substeps": st["heat_substeps"]},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()}}
    if rank == 0 and world == 1 and not args.no_extras:
        line["issue_model"] = dict(pkg.issue_probe(), unit="SM cycles per DFMA warp-instruction per sub-partition",
                                   note="FP64 pipe rate is 2; a third register operand costs a cycle, and so does every "
                                        "non-FP64 instruction issued beside the DFMAs (DESIGN.md section 6)")
        line["roofline_hbm"] = hbm_roofline_leg(torch, pkg, hbm_peak)
        line["roofline_hbm"]["peak_source"] = f"MEASURED_PEAKS.json hbm_gbs ({hbm_src})"
        line["operator_cfg4"] = operator_leg(torch, pkg, fp64_tf)
        if args.operator == "pairs":   # SURVEY.md §8(f) f1, same workload: tables over (ir, jr, |dz|) + block-Toeplitz sweeps
            with pkg.QS(w.geometry, w.material, device=local, lattice_tables=True) as sim2:
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
        if N <= 4096:
            v, total, sample = run_oracle_steps(w, min(args.steps, 20), 1)
        else:
            n_rows = pick_rows(w, 15.0)
            v, total, _ = run_oracle_sample(w, n_rows, 1, 0)
            sample = row_sample_text(w, n_rows)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle", "sample": sample,
                                "seconds": total}
    if rank == 0:
        print(json.dumps(line), flush=True)
    group.close()


if __name__ == "__main__":
    _args = parse_args()
    if _args.impl == "reference":
        reference_arm(_args)
    else:
        gpu_arm(_args)

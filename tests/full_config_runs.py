"""The BASELINE.json configs run start to end as they are specified (all their steps, from J = 0, T = T_bath), on one GPU:

    config 0:  50 steps at dt = 1e-4, 50 A/s                      (pair sweeps)
    config 1:  2000 steps at dt = 5e-5, background field 1 T/s    (pair sweeps)
    config 2:  1000 steps at dt = 1e-4, 20 A/s                    (lattice-tables operator f1)
    config 3:  adaptive dt in [1e-6, 1e-4] by the caller-side controller (C11), events on; --steps3 K of its 5000 steps
               (lattice-tables operator f1)
    --pairs-steps K also runs the first K steps of configs 2 / 3 with the on-the-fly pair sweeps and compares the states.

Why the tables operator for the long runs: the coil configs leave the linear regime after about 100 steps (the surface
cells of the wires carry the shielding currents and approach Jc long before the mean current density does), from then
on every step iterates the projected CG, tens to hundreds of operator sweeps per step (C13).

Not collected by pytest and not a parity test (tests/long_parity.py is): a record of whole-run wall time and
throughput, of the trajectory's observables (I, U_terminal, Tmax, events) and of the step-size sequence of config 3.
Run by hand on a GPU box,

    python tests/full_config_runs.py [--configs 0,1,2,3] [--pairs-steps 20]

prints one JSON line per run; the lines are committed under profiles/.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402
import paper_2403_07666_b200 as pkg  # noqa: E402
from paper_2403_07666_b200.controller import run_adaptive  # noqa: E402


MARKS = (1, 2, 10, 50, 100, 150, 200, 300, 500, 750, 1000, 2000, 3000, 5000)


def run_fixed(cfg, tables=False, steps=None):
    w = wl.config(cfg)
    steps = steps or w.steps
    N = w.geometry.n_rings
    its, ev, marks = [], 0, {}
    t0 = time.time()
    with pkg.QS(w.geometry, w.material, lattice_tables=tables) as sim:
        t_init = time.time() - t0
        t1 = time.time()
        for k in range(1, steps + 1):
            rc = sim.step(w.dt, w.I_ramp)
            ev |= rc
            its.append(sim.stats()["cg_iters"])
            if k in MARKS:
                marks[k] = {"cg_iters": its[-1], "wall_s": round(time.time() - t1, 2), "U_terminal": sim.stats()["U_terminal"]}
                print(json.dumps({"progress": w.name, "step": k, **marks[k]}), file=sys.stderr, flush=True)
        sim.sync()
        wall = time.time() - t1
        st = sim.stats()
        J, T, B, E = sim.read()
    return {"workload": w.name, "operator": "tables" if tables else "pairs", "n_rings": N, "steps": steps,
            "init_s": round(t_init, 3), "wall_s": round(wall, 3), "cell_steps_per_s": N * steps / wall,
            "cg_iterations_first_step": its[0], "cg_iterations_total": int(np.sum(its)), "at_step": marks,
            "event_word_or": int(ev), "t": st["t"], "I": st["I"], "Bext": min(w.geometry.Bext0 + w.geometry.Bext_rate * st["t"], w.geometry.Bext_max)
            if w.geometry.Bext_rate else w.geometry.Bext0,
            "U_terminal": st["U_terminal"], "Tmax": st["Tmax"], "max_abs_J": float(np.max(np.abs(J))),
            "max_abs_B": float(np.max(np.abs(B))), "launches": st["launches"]}, (J, T, B, E)


def run_config3(steps):
    w = wl.config(3)
    N = w.geometry.n_rings
    ev, its, marks = [0], [], {}
    tm = [time.time()]

    def on_step(dt, rc, st):
        ev[0] |= rc
        its.append(st["cg_iters"])
        if len(its) in MARKS:
            marks[len(its)] = {"cg_iters": its[-1], "dt": dt, "wall_s": round(time.time() - tm[0], 2), "U_terminal": st["U_terminal"]}
            print(json.dumps({"progress": w.name, "step": len(its), **marks[len(its)]}), file=sys.stderr, flush=True)

    t0 = time.time()
    with pkg.QS(w.geometry, w.material, lattice_tables=True) as sim:
        t_init = time.time() - t0
        t1 = tm[0] = time.time()
        dts = run_adaptive(sim, w.geometry, w.material, w.I_ramp, steps, on_step=on_step)
        sim.sync()
        wall = time.time() - t1
        st = sim.stats()
        J, T, B, E = sim.read()
    line = {"workload": w.name, "operator": "tables", "n_rings": N, "steps": steps, "init_s": round(t_init, 3),
            "wall_s": round(wall, 3), "cell_steps_per_s": N * steps / wall, "dt_min_taken": min(dts), "dt_max_taken": max(dts),
            "dt_distinct": sorted(set(dts)), "cg_iterations_first_step": its[0], "cg_iterations_total": int(np.sum(its)),
            "at_step": marks,
            "event_word_or": int(ev[0]), "t": st["t"], "I": st["I"], "U_terminal": st["U_terminal"], "Tmax": st["Tmax"],
            "max_abs_J": float(np.max(np.abs(J))), "max_abs_B": float(np.max(np.abs(B))), "launches": st["launches"]}
    print(json.dumps(line), flush=True)


def pairs_against_tables(cfg, steps):
    """The first `steps` steps with the on-the-fly pair sweeps, against the same steps with the tables operator."""
    lt, state_t = run_fixed(cfg, tables=True, steps=steps)
    lp, state_p = run_fixed(cfg, tables=False, steps=steps)
    lp["rel_l2_vs_tables"] = {k: float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
                              for k, a, b in zip("JTBE", state_p, state_t)}
    print(json.dumps(lp), flush=True)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,1,2,3")
    ap.add_argument("--pairs-steps", type=int, default=20)
    ap.add_argument("--steps3", type=int, default=300)
    a = ap.parse_args()
    for c in (int(v) for v in a.configs.split(",")):
        if c == 3:
            run_config3(a.steps3)
        else:
            print(json.dumps(run_fixed(c, tables=c == 2)[0]), flush=True)
        if c >= 2 and a.pairs_steps > 0:
            pairs_against_tables(c, a.pairs_steps)

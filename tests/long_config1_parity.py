"""Full-length parity of BASELINE.json configs[1] (single wire, 64 x 64 cells, background field ramp, 2000 steps at
dt = 5e-5 s): the CUDA path against the CPU oracle (dense Cholesky KKT per step) over the WHOLE run.

Not collected by pytest (about half an hour of host time for the oracle): run by hand on a GPU box,

    python tests/long_config1_parity.py [steps] [--tables]

and prints one JSON line per checkpoint with the relative L2 differences of J, T, B, E and the trajectory's
observables.  DESIGN.md §2 quotes the result.
"""
import dataclasses
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402
from oracle import qs_oracle as qo  # noqa: E402
import paper_2403_07666_b200 as pkg  # noqa: E402


def rel(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def main():
    steps = int(sys.argv[1]) if len(sys.argv) > 1 and sys.argv[1].isdigit() else 2000
    tables = "--tables" in sys.argv
    w = wl.config(1)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    orc = qo.Oracle(w.geometry, mat)
    marks = {10, 50, 100, 250, 500, 1000, 1500, steps}
    t0 = time.time()
    with pkg.QS(w.geometry, mat, lattice_tables=tables) as sim:
        for k in range(1, steps + 1):
            ro, rg = orc.step(w.dt, w.I_ramp), sim.step(w.dt, w.I_ramp)
            assert ro == (rg & 3), (k, ro, rg)
            if k in marks:
                (Jg, Tg, Bg, Eg), (Jo, To, Bo, Eo) = sim.read(), orc.read()
                st = sim.stats()
                aux_x = np.max(np.abs(Jo)) / (mat.Jc0 * (1 - 4.2 / mat.Tc) ** 2)
                print(json.dumps({"step": k, "t": st["t"], "Bext": min(w.geometry.Bext_rate * st["t"], w.geometry.Bext_max),
                                  "rel_J": rel(Jg, Jo), "rel_T": rel(Tg, To), "rel_B": rel(Bg, Bo), "rel_E": rel(Eg, Eo),
                                  "Tmax": float(To.max()), "max_absJ_over_Jc0ref": float(aux_x),
                                  "cg_iters": st["cg_iters"], "wall_s": round(time.time() - t0, 1)}), flush=True)


if __name__ == "__main__":
    main()

"""Full-size, many-step parity of BASELINE.json configs[2] and configs[3] (SURVEY.md §8(d) parity protocol:
100 steps at the config's own size; config 3: 10 steps of the full state), CUDA path against the CPU oracle.

Not collected by pytest: the oracle needs tens of minutes of host time at these sizes.  Two phases, so that the
oracle can run on any host (it needs no GPU) and the comparison on a GPU box:

    python tests/long_parity.py oracle --config 2 --steps 100 --out REF.npz        # calls only oracle/ and workloads/
    python tests/long_parity.py oracle --config 3 --steps 10  --out REF.npz --fft  # tables applied by FFT (see oracle)
    python tests/long_parity.py gpu --ref REF.npz [--tables]                       # CUDA path, compared per checkpoint

`oracle` runs Oracle(operator="tables" | "tables_fft", solver="pcg") with cg_tol = 1e-12 and stores the full state
(J, T, B, E), U_terminal and the CG iteration counts at the checkpoints.  `gpu` replays the same steps through the
C ABI and prints one JSON line per checkpoint: rel-L2 and the largest per-element difference relative to max|ref|
of J, T, B, E, and the terminal voltage.  The printed lines are committed under profiles/ and quoted in DESIGN.md §2.
"""
import argparse
import dataclasses
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402


def workload(cfg, shrink):
    if shrink:
        layers, turns = (int(v) for v in shrink.split("x"))
        w = wl.shrunk(cfg, layers, turns)
    else:
        w = wl.config(cfg)
    return w, dataclasses.replace(w.material, cg_tol=1e-12)


def run_oracle(a):
    from oracle import qs_oracle as qo
    w, mat = workload(a.config, a.shrink)
    marks = sorted({int(m) for m in a.marks.split(",") if int(m) <= a.steps} | {a.steps})
    t0 = time.time()
    orc = qo.Oracle(w.geometry, mat, operator="tables_fft" if a.fft else "tables", solver="pcg")
    print(json.dumps({"phase": "oracle tables built", "wall_s": round(time.time() - t0, 1)}), flush=True)
    out = {"config": a.config, "shrink": a.shrink or "", "steps": a.steps, "marks": np.array(marks), "fft": int(a.fft)}
    rets, iters = [], []
    for k in range(1, a.steps + 1):
        rets.append(orc.step(w.dt, w.I_ramp))
        iters.append(orc.stats["cg_iters"])
        if k in marks:
            J, T, B, E = orc.read()
            out[f"J{k}"], out[f"T{k}"], out[f"B{k}"], out[f"E{k}"] = J, T, B, E
            out[f"U{k}"] = orc.stats["U_terminal"]
            line = {"phase": "oracle", "step": k, "cg_iters": iters[-1], "U_terminal": orc.stats["U_terminal"],
                    "wall_s": round(time.time() - t0, 1)}
            if a.fft:   # the FFT application against the defining offset-by-offset sum, on this very state
                y1, y0 = orc.tables.matvec(orc.Idot), orc.tables.matvec_plain(orc.Idot)
                line["fft_vs_plain_matvec_rel_l2"] = float(np.linalg.norm(y1 - y0) / np.linalg.norm(y0))
                (br1, bz1), (br0, bz0) = orc.tables.field(w.geometry.area * J), orc.tables.field_plain(w.geometry.area * J)
                line["fft_vs_plain_field_rel_l2"] = float(np.linalg.norm(np.r_[br1 - br0, bz1 - bz0]) /
                                                          np.linalg.norm(np.r_[br0, bz0]))
            print(json.dumps(line), flush=True)
            np.savez(a.out, rets=np.array(rets), iters=np.array(iters), **out)   # partial results survive an interruption
    np.savez(a.out, rets=np.array(rets), iters=np.array(iters), **out)


def rel(x, y):
    return float(np.linalg.norm(x - y) / max(np.linalg.norm(y), 1e-300))


def relmax(x, y):
    return float(np.max(np.abs(x - y)) / max(np.max(np.abs(y)), 1e-300))


def run_gpu(a):
    import paper_2403_07666_b200 as pkg
    ref = np.load(a.ref)
    cfg, steps, marks = int(ref["config"]), int(ref["steps"]), [int(m) for m in ref["marks"]]
    w, mat = workload(cfg, str(ref["shrink"]))
    t0 = time.time()
    with pkg.QS(w.geometry, mat, lattice_tables=a.tables) as sim:
        for k in range(1, steps + 1):
            rc = sim.step(w.dt, w.I_ramp)
            assert rc >= 0 and (rc & 3) == int(ref["rets"][k - 1]), (k, rc)
            if k in marks and f"J{k}" in ref:
                got = sim.read()
                st = sim.stats()
                line = {"workload": w.name, "operator": "tables" if a.tables else "pairs", "step": k, "n_rings": w.geometry.n_rings}
                for name, g in zip("JTBE", got):
                    r = ref[f"{name}{k}"]
                    line[f"rel_{name}"] = rel(g, r)
                    line[f"relmax_{name}"] = relmax(g, r)
                U = float(ref[f"U{k}"])
                line["U_terminal"] = st["U_terminal"]
                line["rel_U"] = abs(st["U_terminal"] - U) / abs(U)
                line["cg_iters_gpu"], line["cg_iters_oracle"] = st["cg_iters"], int(ref["iters"][k - 1])
                line["wall_s"] = round(time.time() - t0, 1)
                print(json.dumps(line), flush=True)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    sub = ap.add_subparsers(dest="phase", required=True)
    po = sub.add_parser("oracle")
    po.add_argument("--config", type=int, required=True, choices=[2, 3])
    po.add_argument("--shrink", default="", help="layers x turns of a smaller winding pack, e.g. 12x20")
    po.add_argument("--steps", type=int, required=True)
    po.add_argument("--marks", default="1,10,50,100")
    po.add_argument("--out", required=True)
    po.add_argument("--fft", action="store_true")
    pg = sub.add_parser("gpu")
    pg.add_argument("--ref", required=True)
    pg.add_argument("--tables", action="store_true")
    args = ap.parse_args()
    run_oracle(args) if args.phase == "oracle" else run_gpu(args)

"""Host experiment behind the constraint preconditioner of the projected CG ("Patch preconditioner"):
iteration counts of the projected CG of SURVEY.md section 8(c) C8 with different block-diagonal preconditioners H on ONE
mid-trajectory system (M + theta dt D) I' + C V = b of a shrunk config, taken where the surface cells of the wires sit at
Jc (the nonlinear regime the configs spend most of their steps in, C13).  C8 leaves H free (the solution of a
step is unique); the experiment asks which H is worth building on the GPU.

Not collected by pytest and not a parity test: plain numpy on the CPU oracle's dense matrices (it calls only oracle/ and
workloads/), minutes of host time.  By hand,

    python tests/precond_experiment.py --config 3 --layers 4 --turns 6 --steps 130 --ramp-x 200
    python tests/precond_experiment.py --config 2 --layers 3 --turns 4 --steps 130 --ramp-x 100
    python tests/precond_experiment.py --config 1 --cells 32 --steps 120 --ramp-x 20

(--ramp-x scales the ramp so that the shrunk coil reaches Jc within the steps taken); the printed lines are committed
under profiles/r02_precond_experiment.md.

Preconditioners compared (all block-diagonal inside a constraint group, so the per-turn Schur complement of the
projection stays diagonal, except the last):
  patch p x p        exact inverse of (M + shift) on square patches of p x p cells of a wire; p = wire side: the whole wire
  fixed, scaled      ONE inverse of M per patch (no shift) and the shift as a symmetric diagonal scaling
                     H = D^1/2 M_patch D^1/2, D = 1 + shift / diag(M): no inversion per solve
  two-level          p x p patches + a coarse space of piecewise constants per patch, per wire (additive)
  groups of wires    exact blocks over gl x gt adjacent wires with a G x G Schur complement per group
"""
import argparse
import dataclasses
import math
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402
from oracle import qs_oracle as qo  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=[1, 2, 3])
    ap.add_argument("--layers", type=int, default=2)
    ap.add_argument("--turns", type=int, default=3)
    ap.add_argument("--cells", type=int, default=32, help="cells per wire side of the single wire (config 1)")
    ap.add_argument("--steps", type=int, default=130)
    ap.add_argument("--ramp-x", type=float, default=200.0)
    a = ap.parse_args()

    if a.config == 1:
        w = wl.shrunk(1, 1, 1, a.cells)
        w = dataclasses.replace(w, geometry=dataclasses.replace(w.geometry, Bext_rate=w.geometry.Bext_rate * a.ramp_x))
    else:
        w = wl.shrunk(a.config, a.layers, a.turns)
        w = dataclasses.replace(w, I_ramp=w.I_ramp * a.ramp_x)
    geo, mat = w.geometry, w.material
    N, nt, tid = geo.n_rings, geo.n_turns, geo.turn_id
    print(f"{w.name}: N {N}, {geo.Nr} x {geo.Nz} cells, {nt} wires, dt {w.dt}, I_ramp {w.I_ramp}, Bext_rate {geo.Bext_rate}", flush=True)
    orc = qo.Oracle(geo, mat)
    t0 = time.time()
    for _ in range(a.steps):
        orc.step(w.dt, w.I_ramp)
    print(f"{a.steps} oracle steps in {time.time() - t0:.0f} s; max|J| {np.abs(orc.J).max():.4g}", flush=True)

    # the system of the next step (C4, C7), assembled as Oracle.step does
    area = geo.area
    Br, Bz = orc.field(area * orc.J)
    ml = qo.material_law(mat, orc.J, orc.T, Br, Bz + orc.Bext(orc.t), geo.r, orc.scale)
    Bdot = geo.Bext_rate if orc.Bext(orc.t) < geo.Bext_max else 0.0
    b = -2.0 * math.pi * geo.r * (ml["E"] + 0.5 * geo.r * Bdot)
    shift = mat.theta * w.dt * 2.0 * math.pi * geo.r * ml["dEdJ"] / area
    A = orc.M + np.diag(shift)
    d = np.full(nt, float(w.I_ramp))
    print(f"shift / diag(M): max {(shift / orc.diagM).max():.3g}", flush=True)
    xref, _ = qo.kkt_dense(A, qo.constraint_matrix(geo), b, d)
    xw = orc.Idot.copy()                               # warm start: the previous step's solution
    n = int(round(math.sqrt(N / nt)))                  # cells per wire side
    ir, iz = np.arange(N) // geo.Nz, np.arange(N) % geo.Nz

    def patches(p):
        key = (ir // p) * (geo.Nz // p + 1) + iz // p
        order = np.argsort(key, kind="stable")
        _, starts = np.unique(key[order], return_index=True)
        return np.split(order, starts[1:])

    def block_apply(blocks, scale=None):
        def app(r):
            out = np.empty_like(r)
            rs = r if scale is None else r * scale
            for idx, Bi in blocks:
                out[idx] = Bi @ rs[idx]
            return out if scale is None else out * scale
        return app

    def exact(p):
        if p == 1:
            dg = np.diag(A).copy()
            return lambda r: r / dg
        return block_apply([(idx, np.linalg.inv(A[np.ix_(idx, idx)])) for idx in patches(p)])

    def fixed_scaled(p):
        blocks = [(idx, np.linalg.inv(orc.M[np.ix_(idx, idx)])) for idx in patches(p)]
        return block_apply(blocks, 1.0 / np.sqrt(1.0 + shift / orc.diagM))

    def two_level(p):
        pl = patches(p)
        fine = exact(p)
        Z = np.zeros((N, len(pl)))
        for k, idx in enumerate(pl):
            Z[idx, k] = 1.0
        pt = np.array([tid[idx[0]] for idx in pl])
        A0inv = np.linalg.inv(np.where(pt[:, None] == pt[None, :], Z.T @ A @ Z, 0.0))   # block-diagonal over wires
        return lambda r: fine(r) + Z @ (A0inv @ (Z.T @ r))

    def pcg(prec, x0, tol=mat.cg_tol, maxit=3000):
        """projected CG with H block-diagonal inside the constraint groups (diagonal Schur complement)"""
        Hi1 = prec(np.ones(N))
        s = np.bincount(tid, weights=Hi1, minlength=nt)

        def project(r):
            t = prec(r)
            v = np.bincount(tid, weights=t, minlength=nt) / s
            return t - v[tid] * Hi1, v
        x = x0 + ((d - np.bincount(tid, weights=x0, minlength=nt)) / s)[tid] * Hi1
        r = A @ x - b
        g, _ = project(r)
        rg = r @ g
        rc = A @ ((d / s)[tid] * Hi1) - b
        gc, _ = project(rc)
        nu = math.sqrt(abs(rc @ gc))                   # reference norm: the cold start's projected residual (C8)
        p, it = -g, 0
        while math.sqrt(abs(rg)) > tol * nu and it < maxit:
            q = A @ p
            alpha = rg / (p @ q)
            x += alpha * p
            r += alpha * q
            g, v = project(r)
            r = r - v[tid]
            rg, rg_old = r @ g, rg
            p = -g + (rg / rg_old) * p
            it += 1
        return x, it

    def pcg_groups(gl, gt, x0, tol=mat.cg_tol, maxit=3000):
        """the same with exact blocks over gl x gt adjacent wires: G x G Schur complement per group"""
        Tn = geo.turns_per_layer
        gkey = ((tid // Tn) // gl) * ((Tn + gt - 1) // gt) + (tid % Tn) // gt
        groups = [np.where(gkey == k)[0] for k in np.unique(gkey)]
        ws = [np.unique(tid[idx]) for idx in groups]
        Binv = [np.linalg.inv(A[np.ix_(idx, idx)]) for idx in groups]
        Cg = [np.stack([(tid[idx] == q).astype(float) for q in wq], axis=1) for idx, wq in zip(groups, ws)]
        HiC = [Bi @ C for Bi, C in zip(Binv, Cg)]
        Sinv = [np.linalg.inv(C.T @ h) for C, h in zip(Cg, HiC)]

        def project(r):
            g, v = np.empty_like(r), np.zeros(nt)
            for idx, Bi, C, h, Si, wq in zip(groups, Binv, Cg, HiC, Sinv, ws):
                t = Bi @ r[idx]
                vv = Si @ (C.T @ t)
                g[idx], v[wq] = t - h @ vv, vv
            return g, v
        x, xc = x0.copy(), np.zeros(N)
        defi = d - np.bincount(tid, weights=x, minlength=nt)
        for idx, h, Si, wq in zip(groups, HiC, Sinv, ws):
            x[idx] += h @ (Si @ defi[wq])
            xc[idx] = h @ (Si @ d[wq])
        r = A @ x - b
        g, _ = project(r)
        rg = r @ g
        rc = A @ xc - b
        gc, _ = project(rc)
        nu = math.sqrt(abs(rc @ gc))
        p, it = -g, 0
        while math.sqrt(abs(rg)) > tol * nu and it < maxit:
            q = A @ p
            alpha = rg / (p @ q)
            x += alpha * p
            r += alpha * q
            g, v = project(r)
            r = r - v[tid]
            rg, rg_old = r @ g, rg
            p = -g + (rg / rg_old) * p
            it += 1
        return x, it

    def report(name, solve):
        xs, itw = solve(xw)
        _, itc = solve(np.zeros(N))
        err = np.linalg.norm(xs - xref) / np.linalg.norm(xref)
        print(f"{name:42s} warm start {itw:4d} iterations, cold start {itc:4d}; error against the dense KKT solve {err:.1e}", flush=True)

    sizes = [q for q in (2, 3, 4, 6, 8, 12, 16, 32) if n % q == 0 and q <= n]
    report("diagonal", lambda x0: pcg(exact(1), x0))
    for p in sizes:
        report(f"patch {p} x {p}" + (" (whole wire)" if p == n else ""), lambda x0, p=p: pcg(exact(p), x0))
    for p in [q for q in sizes if q >= 6]:
        report(f"fixed inverse of M, scaled, patch {p} x {p}", lambda x0, p=p: pcg(fixed_scaled(p), x0))
    for p in [q for q in (4, 8) if n % q == 0 and q < n]:
        report(f"two-level: patch {p} x {p} + constants", lambda x0, p=p: pcg(two_level(p), x0))
    if nt > 1:
        for gl, gt in ((1, 2), (2, 2), (2, 3), (4, 3)):
            if gl <= geo.layers and gt <= geo.turns_per_layer:
                report(f"whole wires in groups of {gl} x {gt}", lambda x0, gl=gl, gt=gt: pcg_groups(gl, gt, x0))


if __name__ == "__main__":
    main()

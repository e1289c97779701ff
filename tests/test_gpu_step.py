"""GPU parity of whole time steps (qs_step, S1..S7) against the CPU oracle on the same seeded inputs.

north_star tolerance: rel-L2 <= 1e-6 for J, T and B after 100 steps (50 on config 0).  Both sides run with
cg_tol = 1e-12 (the oracle solves by dense Cholesky where it can).  Event flags must match exactly.
"""
import dataclasses

import numpy as np
import pytest

import workloads as wl
from oracle import qs_oracle as qo

pytestmark = pytest.mark.gpu
TOL = 1e-6


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def pkg():
    import paper_2403_07666_b200 as p
    return p


def run_both(pkg, geo, mat, steps, dt, I_ramp, operator="dense", solver="cholesky", prep=None, dts=None):
    mat = dataclasses.replace(mat, cg_tol=1e-12)
    orc = qo.Oracle(geo, mat, operator=operator, solver=solver)
    sim = pkg.QS(geo, mat)
    if prep is not None:
        J0, T0 = prep
        orc.write(J0, T0, 0.0, 0.0)
        sim.write(J0, T0, 0.0, 0.0)
    rets = []
    for k in range(steps):
        d = dt if dts is None else dts[k]
        ro, rg = orc.step(d, I_ramp), sim.step(d, I_ramp)
        rets.append((ro, rg & 3))
    out = (orc, sim, orc.read(), sim.read(), rets)
    return out


def check_state(ref, got, tol=TOL):
    for name, a, b in zip(("J", "T", "B", "E"), got, ref):
        if np.linalg.norm(b) == 0.0:
            assert np.linalg.norm(a) <= 1e-300 or name == "E", name
            continue
        floor = 1e-30 if name == "E" else 0.0                   # E ~ Ec (J/Jc)^20 underflows in the linear regime
        assert np.linalg.norm(a - b) <= tol * np.linalg.norm(b) + floor, (name, rel(a, b))
        # and cell by cell: no single cell may hide inside the norm
        assert np.max(np.abs(a - b)) <= tol * np.max(np.abs(b)) + floor, (name, np.max(np.abs(a - b)) / np.max(np.abs(b)))


def test_config0_50_steps(pkg):
    w = wl.config(0)
    orc, sim, ref, got, rets = run_both(pkg, w.geometry, w.material, 50, w.dt, w.I_ramp)
    check_state(ref, got)
    assert all(a == b for a, b in rets)
    st = sim.stats()
    assert abs(st["U_terminal"] - orc.stats["U_terminal"]) <= 1e-8 * abs(orc.stats["U_terminal"])
    assert abs(st["I"] - 50 * w.dt * w.I_ramp) < 1e-15 and st["heat_substeps"] == 5
    cur = np.bincount(w.geometry.turn_id, weights=got[0] * w.geometry.area)
    assert np.max(np.abs(cur - st["I"])) <= 1e-10 * st["I"]
    sim.close()


def test_config1_100_steps_nonlinear(pkg):
    # full config 1 (64x64 cells, ramped background field); 100 steps as north_star asks
    w = wl.config(1)
    orc, sim, ref, got, rets = run_both(pkg, w.geometry, w.material, 100, w.dt, w.I_ramp)
    check_state(ref, got)
    assert sim.stats()["heat_substeps"] == 144
    sim.close()


def test_config1_strong_drive_reaches_flux_flow(pkg):
    # same wire at 32x32 cells, 20 T/s: |J| ~ Jc, E' matters, Joule heating is visible in T
    w = wl.shrunk(1, 1, 1, 32)
    geo = dataclasses.replace(w.geometry, Bext_rate=20.0)
    orc, sim, ref, got, rets = run_both(pkg, geo, w.material, 100, w.dt, 0.0)
    check_state(ref, got)
    Jc = 2e9 * (1 - 4.2 / 18) ** 2
    assert np.max(np.abs(ref[0])) > 0.9 * Jc and np.max(ref[3]) > 1e-6 and ref[1].max() > 4.2 + 1e-6
    assert all(a == b for a, b in rets)
    fo, fg = orc.flags, sim.events()[0]
    assert np.array_equal(fo, fg)
    sim.close()


@pytest.mark.parametrize("cfg,layers,turns", [(2, 3, 5), (3, 4, 6)])
def test_shrunk_coils_100_steps(pkg, cfg, layers, turns):
    # configs 2 / 3 wire, laws, ramp and seed on a smaller winding pack (N = 3840 / 3456): dense oracle
    w = wl.shrunk(cfg, layers, turns)
    orc, sim, ref, got, rets = run_both(pkg, w.geometry, w.material, 100, w.dt, w.I_ramp)
    check_state(ref, got)
    sim.close()


_cfg3_12x20 = {}


@pytest.mark.parametrize("tables", [False, True])
def test_config3_shrunk_12x20_100_steps(pkg, tables):
    # SURVEY.md §8(d) parity protocol for configs[3]: 100 steps on 12 layers x 20 turns, n = 12 (N = 34,560), oracle with
    # lattice tables + its own projected CG (too large for dense matrices); both GPU operators
    w = wl.shrunk(3, 12, 20)
    geo = w.geometry
    assert geo.n_rings == 34560
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    if not _cfg3_12x20:                                         # the oracle trajectory serves both parametrisations
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=1):                       # 480 small matrix products per application: BLAS threads only spin
            orc = qo.Oracle(geo, mat, operator="tables", solver="pcg")
            rets = [orc.step(w.dt, w.I_ramp) for _ in range(100)]
        _cfg3_12x20.update(ref=orc.read(), rets=rets, U=orc.stats["U_terminal"])
    with pkg.QS(geo, mat, lattice_tables=tables) as sim:
        rets = [sim.step(w.dt, w.I_ramp) & 3 for _ in range(100)]
        got = sim.read()
        st = sim.stats()
    assert rets == _cfg3_12x20["rets"]
    check_state(_cfg3_12x20["ref"], got)
    assert abs(st["U_terminal"] - _cfg3_12x20["U"]) <= 1e-8 * abs(_cfg3_12x20["U"])
    cur = np.bincount(geo.turn_id, weights=got[0] * geo.area)
    assert np.max(np.abs(cur - st["I"])) <= 1e-9 * st["I"]


def test_shrunk_config3_adaptive_dt_replay(pkg):
    # C11: the caller's controller lives outside qs_step; the GPU replays the oracle's recorded dt list
    w = wl.shrunk(3, 2, 3)
    dts = [1e-4, 1e-4, 5e-5, 2.5e-5, 1e-6, 1e-6, 2e-6, 4e-6, 8e-6, 1.6e-5, 3.2e-5, 6.4e-5, 1e-4, 1e-4, 1e-4]
    orc, sim, ref, got, rets = run_both(pkg, w.geometry, w.material, len(dts), None, w.I_ramp, dts=dts)
    check_state(ref, got)
    assert abs(sim.stats()["t"] - sum(dts)) < 1e-15
    sim.close()


def test_table_oracle_on_a_mid_size_lattice(pkg):
    # N = 12288 (> dense range): oracle with lattice tables + its own projected CG, 5 steps
    w = wl.shrunk(2, 4, 12)
    orc, sim, ref, got, rets = run_both(pkg, w.geometry, w.material, 5, w.dt, w.I_ramp, operator="tables", solver="pcg")
    check_state(ref, got)
    sim.close()


@pytest.mark.parametrize("variant", ["v1", "v2", "v3"])
def test_event_variants(pkg, variant):
    # prepared states that make the detector fire; flags, first-event times, counters exact
    w = wl.config(0)
    geo = w.geometry
    N = geo.n_rings
    T0 = np.full(N, geo.T_bath)
    J0 = np.zeros(N)
    hot = geo.turn_id == 5
    if variant == "v1":
        T0[hot] = 12.0
    elif variant == "v2":
        T0[hot] = 19.0
    else:
        T0[hot] = 19.0
        J0[:] = 0.9 * 2e9 * (1 - 4.2 / 18) ** 2
    orc, sim, ref, got, rets = run_both(pkg, geo, w.material, 12, 2e-5, w.I_ramp, prep=(J0, T0))
    assert all(a == b for a, b in rets), rets
    fl, tf, cnt = sim.events()
    assert np.array_equal(fl, orc.flags) and np.array_equal(cnt, orc.count)
    assert np.allclose(tf, orc.t_first, rtol=0, atol=1e-18)
    assert orc.flags.any() and rets[0][0] != 0
    check_state(ref, got, tol=1e-6)
    # per-wire statistics (f3): same accumulators on both sides
    ws = sim.wire_stats()
    for key in ("E_joule", "Q_FJ", "P_max", "T_max", "T_q", "P_q", "Q_q"):
        ref_w = orc.wire[key]
        assert np.max(np.abs(ws[key] - ref_w)) <= 1e-6 * max(np.max(np.abs(ref_w)), 1e-300), key
    assert np.allclose(ws["t_q"], orc.wire["t_q"], rtol=0, atol=1e-18)
    if variant != "v1":
        assert ws["t_q"][5] > 0 and ws["Q_q"][5] >= 0
    sim.close()


def test_step_is_transactional_and_write_resumes(pkg):
    w = wl.shrunk(0, 2, 2, 4)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    with pkg.QS(w.geometry, mat) as a, pkg.QS(w.geometry, mat) as b:
        for _ in range(6):
            a.step(w.dt, w.I_ramp)
        J, T, _, _ = a.read()
        with pytest.raises(pkg.QsError):
            a.step(-1.0, w.I_ramp)
        J2, T2, _, _ = a.read()
        assert np.array_equal(J, J2) and np.array_equal(T, T2)
        st = a.stats()
        b.write(J, T, st["t"], st["I"])                            # resume in a second handle
        a.step(w.dt, w.I_ramp)
        b.step(w.dt, w.I_ramp)
        for u, v in zip(a.read(), b.read()):
            assert rel(u, v) <= 1e-9 or np.linalg.norm(v) < 1e-30


@pytest.mark.parametrize("where,code", [(1, -2), (2, -3)])
def test_failed_step_restores_everything_the_caller_can_observe(pkg, where, code):
    # include/qs.h: negative return = state unchanged.  A failure is injected AFTER the current update S5 (a CUDA error
    # reported by the heat stage / a NaN in J caught by the step's own check) on a state with live event flags, a dE/dt
    # history and per-wire statistics; J, T, B, E, flags, first-event times, counters, wire statistics, t, I must be
    # bit-identical afterwards, and the retried step must equal the step of a twin handle that never failed.
    w = wl.config(0)
    geo = w.geometry
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    N = geo.n_rings
    T0 = np.full(N, geo.T_bath)
    T0[geo.turn_id == 5] = 19.0
    J0 = np.full(N, 0.9 * 2e9 * (1 - 4.2 / 18) ** 2)

    def observe(sim):
        st = sim.stats()
        ws = sim.wire_stats()
        return (*sim.read(), *sim.events(), *[ws[k] for k in sorted(ws)], np.array([st["t"], st["I"]]))

    with pkg.QS(geo, mat) as a, pkg.QS(geo, mat) as b:
        for sim in (a, b):
            sim.write(J0, T0, 0.0, 0.0)
            for _ in range(3):
                assert sim.step(2e-5, w.I_ramp) >= 0
        before = observe(a)
        assert before[4].any() and before[6].any()               # flags and counters are live
        a.debug_inject_failure(where)
        with pytest.raises(pkg.QsError) as ei:
            a.step(2e-5, w.I_ramp)
        assert ei.value.code == code
        after = observe(a)
        for u, v in zip(before, after):
            assert np.array_equal(u, v, equal_nan=True)
        ra, rb = a.step(2e-5, w.I_ramp), b.step(2e-5, w.I_ramp)
        assert ra == rb
        for u, v in zip(observe(a), observe(b)):
            assert np.allclose(u, v, rtol=1e-9, atol=1e-300, equal_nan=True)


def test_rate_checkpoint_resumes_like_the_uninterrupted_run(pkg):
    # qs_read_rate / qs_write_rate: a second handle resumed from (J, T, t, I) and I' continues like the first one
    w = wl.shrunk(1, 1, 1, 12)
    geo = dataclasses.replace(w.geometry, Bext_rate=400.0)     # fast ramp: |J| reaches Jc within a few steps, the CG iterates
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    with pkg.QS(geo, mat) as a, pkg.QS(geo, mat) as b:
        for _ in range(25):
            a.step(w.dt, 0.0)
        J, T, _, _ = a.read()
        st = a.stats()
        b.write(J, T, st["t"], st["I"])
        b.write_rate(a.read_rate())
        a.write(J, T, st["t"], st["I"])                          # same history reset on both sides
        a.step(w.dt, 0.0)
        b.step(w.dt, 0.0)
        ia, ib = a.stats()["cg_iters"], b.stats()["cg_iters"]
        assert ia > 0 and abs(ia - ib) <= 2                      # FP64 atomics: the stopping iteration may shift by one
        for u, v in zip(a.read(), b.read()):                     # both converged to cg_tol = 1e-12; E ~ J^20 amplifies it
            assert rel(u, v) <= 1e-9
        assert rel(b.read_rate(), a.read_rate()) <= 1e-9


def test_patch_preconditioner_changes_iterations_not_the_solution(pkg):
    # C8: the preconditioner is free, the solution of a step is unique.  Same nonlinear trajectory (single wire under a
    # fast field ramp, |J| ~ Jc) with the patch (block-Jacobi) constraint preconditioner and with the diagonal one
    # (QS_GEO_NO_PATCH_PRECOND): same states and terminal voltage to the CG tolerance, fewer iterations; and a coil in
    # the linear regime (several turns: the per-turn Schur complement of the block projection), cold solve included
    w = wl.shrunk(1, 1, 1, 32)
    geo = dataclasses.replace(w.geometry, Bext_rate=20.0)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    res = {}
    for patch in (True, False):
        its = 0
        with pkg.QS(geo, mat, patch_precond=patch) as sim:
            for _ in range(60):
                assert sim.step(w.dt, 0.0) >= 0
                its += sim.stats()["cg_iters"]
            res[patch] = (sim.read(), sim.stats()["U_terminal"], its)
    for u, v in zip(res[True][0], res[False][0]):
        assert rel(u, v) <= 1e-8 or np.linalg.norm(v) < 1e-30
    assert abs(res[True][1] - res[False][1]) <= 1e-8 * abs(res[False][1]) + 1e-20
    assert 0 < res[True][2] < 0.7 * res[False][2], (res[True][2], res[False][2])
    w = wl.shrunk(0, 3, 2, 8)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    res = {}
    for patch in (True, False):
        with pkg.QS(w.geometry, mat, patch_precond=patch) as sim:
            sim.step(w.dt, w.I_ramp)
            first = sim.stats()["cg_iters"]
            for _ in range(4):
                sim.step(w.dt, w.I_ramp)
            res[patch] = (sim.read(), sim.stats()["U_terminal"], first)
    for u, v in zip(res[True][0], res[False][0]):
        assert rel(u, v) <= 1e-9 or np.linalg.norm(v) < 1e-30
    assert abs(res[True][1] - res[False][1]) <= 1e-9 * abs(res[False][1])
    assert 0 < res[True][2] < res[False][2]


def test_whole_wire_patches_of_the_preconditioner(pkg):
    # wires of 12 x 12 (config 3) and 16 x 16 (config 2) cells: the patch is the whole wire (inverted per solve in global
    # memory, the constant part shared per layer) against the sub-wire patches of at most 8 x 8 cells
    # (QS_GEO_PATCH_SUBWIRE) and the diagonal (QS_GEO_NO_PATCH_PRECOND), on a trajectory ramped fast enough that the
    # surface cells of the wires sit at Jc (C13): same states and terminal voltage (C8: the preconditioner is
    # free), and about half the iterations of the sub-wire patches; wires of 10 x 10 cells (a block size that is not a
    # multiple of the update's 4 x 4 tiles); last wires larger than a patch, where a second level of patch-wise constants
    # stands in for the whole-wire block: one wire of 32 x 32 cells in a fast field ramp (16 coarse unknowns) and two
    # layers of two wires of 24 x 24 cells (9 coarse unknowns per wire, one coarse matrix per layer)
    cases = [(wl.shrunk(3, 2, 3), 200.0, 0.0, 0.75), (wl.shrunk(2, 2, 2), 100.0, 0.0, 0.75), (wl.shrunk(3, 3, 2, 10), 200.0, 0.0, 0.75),
             (wl.shrunk(1, 1, 1, 32), 1.0, 20.0, 0.8), (wl.shrunk(3, 2, 2, 24), 200.0, 0.0, 0.8)]
    for w, rampx, bext_rate, gain in cases:
        geo = dataclasses.replace(w.geometry, Bext_rate=bext_rate) if bext_rate else w.geometry
        mat = dataclasses.replace(w.material, cg_tol=1e-12)
        res = {}
        for mode, kw in (("whole", {}), ("sub", dict(patch_subwire=True)), ("diag", dict(patch_precond=False))):
            its = 0
            with pkg.QS(geo, mat, **kw) as sim:
                for k in range(130):
                    assert sim.step(w.dt, w.I_ramp * rampx) >= 0
                    if k >= 110:
                        its += sim.stats()["cg_iters"]
                res[mode] = (sim.read(), sim.stats()["U_terminal"], its)
        J = res["diag"][0][0]
        assert np.abs(J).max() > 1e9                              # the nonlinear regime was reached
        for mode in ("whole", "sub"):
            for u, v in zip(res[mode][0], res["diag"][0]):
                assert rel(u, v) <= 1e-8 or np.linalg.norm(v) < 1e-30
            assert abs(res[mode][1] - res["diag"][1]) <= 1e-8 * abs(res["diag"][1]) + 1e-20
        print("cg iterations over 20 steps (p <= 16, p <= 8, diagonal):", res["whole"][2], res["sub"][2], res["diag"][2])
        assert 0 < res["whole"][2] < gain * res["sub"][2] < res["diag"][2], (res["whole"][2], res["sub"][2], res["diag"][2])


def test_handle_works_while_another_device_or_stream_context_is_current(pkg):
    # a handle remembers its device: calls are valid whatever device is current in the calling thread (one GPU here:
    # the guard must at least be a no-op; with two visible devices the second one is made current around the calls)
    import torch
    w = wl.shrunk(0, 2, 2, 4)
    other = torch.cuda.device_count() - 1
    with pkg.QS(w.geometry, w.material, device=0) as sim, pkg.QS(w.geometry, w.material, device=0) as ref:
        with torch.cuda.device(other):
            for _ in range(3):
                assert sim.step(w.dt, w.I_ramp) >= 0
            got = sim.read()
        for _ in range(3):
            ref.step(w.dt, w.I_ramp)
        for u, v in zip(got, ref.read()):                      # (FP64 atomics: equal up to summation order)
            assert rel(u, v) <= 1e-12 or np.linalg.norm(v) < 1e-30


@pytest.mark.parametrize("cfg,rows", [(2, 256), (3, 128)])
def test_full_size_step_sampled_outputs_and_invariants(pkg, cfg, rows):
    # BASELINE.json configs[2], [3] at FULL size, in the launch configuration bench.py times.  The oracle cannot
    # step these, but every output of the step that has a row-by-row definition can be sampled:
    #   B^k = G_B (a J^k) + B_ext and E^k = E(J^k, T^k, B^k) on seeded cells (pair by pair against all N sources),
    # and the properties that hold at any size: the turn currents advance by dt*I_ramp exactly (every CG iterate
    # keeps the constraint, so two iterations suffice), T stays at the bath while Q ~ 0, no event fires.
    w = wl.config(cfg)
    geo = w.geometry
    mat = dataclasses.replace(w.material, cg_maxit=2)
    N = geo.n_rings
    g = np.random.default_rng(50 + cfg)
    Jc0 = 2e9 * (1 - 4.2 / 18) ** 2
    J0 = 0.7 * Jc0 * g.uniform(-1.0, 1.0, N)
    T0 = g.uniform(4.2, 6.0, N)
    idx = wl.sample_rows(N, rows, seed=70 + cfg)
    with pkg.QS(geo, mat) as sim:
        sim.write(J0, T0, 0.0, 0.0)
        rc = sim.step(w.dt, w.I_ramp)
        J1, T1, B, E = sim.read()
        st = sim.stats()
    assert rc >= 0 and (rc & 4)                                   # stopped at cg_maxit, state advanced
    Br, Bz = qo.field_eval_rows(geo, geo.area * J0, idx, chunk=4)
    assert rel(B[idx], Br) <= 1e-9 and rel(B[N + idx], Bz) <= 1e-9
    ml = qo.material_law(mat, J0[idx], T0[idx], Br, Bz, geo.r[idx], mat.jc0_scale[idx])
    assert rel(E[idx], ml["E"]) <= 1e-6
    # net current of every turn: sum_i a (J1 - J0) = dt * I_ramp
    dI = np.bincount(geo.turn_id, weights=geo.area * (J1 - J0), minlength=geo.n_turns)
    assert np.max(np.abs(dI - w.dt * w.I_ramp)) <= 1e-9 * w.dt * w.I_ramp + 1e-12 * np.max(np.abs(geo.area * J0)) * 200
    assert np.all(np.isfinite(T1)) and st["heat_substeps"] == qo.heat_substeps_count(geo, mat, w.dt)


@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 1, 2), (2, 1, 1), (1, 3, 1), (1, 1, 3)])
@pytest.mark.parametrize("tables", [False, True])
def test_degenerate_lattices(pkg, shape, tables):
    # one-cell wires, single rows / columns: every stencil neighbour is a border, blocks are almost all padding
    L, Tn, n = shape
    geo = wl.lattice_geometry(L, Tn, n, 1.0e-3, 30e-3, Bext_rate=5.0, Bext_max=3.0)
    mat = dataclasses.replace(wl.Material(jc0_scale=wl.jc0_scale(5, geo.n_rings, 0.01)), cg_tol=1e-12)
    orc = qo.Oracle(geo, mat)
    with pkg.QS(geo, mat, lattice_tables=tables) as sim:
        for _ in range(30):
            assert orc.step(1e-4, 40.0) == (sim.step(1e-4, 40.0) & 3)
        got, ref = sim.read(), orc.read()
    check_state(ref, got)


def test_explicit_theta0_steps(pkg):
    # C7: theta = 0 (the literal explicit Euler reading) stays available; linear regime and a mildly nonlinear wire
    for w, steps, kw in ((wl.shrunk(0, 2, 2, 8), 30, {}), (wl.shrunk(1, 1, 1, 16), 60, {"Bext_rate": 2.0})):
        geo = dataclasses.replace(w.geometry, **kw)
        mat = dataclasses.replace(w.material, theta=0.0, cg_tol=1e-12)
        orc = qo.Oracle(geo, mat)
        with pkg.QS(geo, mat) as sim:
            for _ in range(steps):
                assert orc.step(w.dt, w.I_ramp) == (sim.step(w.dt, w.I_ramp) & 3)
            got, ref = sim.read(), orc.read()
        check_state(ref, got)


@pytest.mark.parametrize("scenario", ["quench", "ramp"])
def test_adaptive_dt_controller(pkg, scenario):
    # configs[3] "adaptive dt in [1e-6, 1e-4] s with event detection" (C11).  The product's controller drives the GPU,
    # the rule restated here drives the oracle from the oracle's own max |dJ|; the two dt sequences must coincide and
    # the states agree.  "quench": shrunk coil with a prepared normal turn (events pin dt at dt_min);
    # "ramp": single wire under a fast background ramp (no event: dt halves while the screening currents build up)
    from paper_2403_07666_b200.controller import run_adaptive
    if scenario == "quench":
        w = wl.shrunk(3, 2, 3)
        geo = w.geometry
    else:
        w = wl.shrunk(1, 1, 1, 12)
        geo = dataclasses.replace(w.geometry, Bext_rate=400.0)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    N = geo.n_rings
    Jref = mat.Jc0 * (1 - geo.T_bath / mat.Tc) ** 2
    J0 = np.full(N, 0.85 * Jref) if scenario == "quench" else np.zeros(N)
    T0 = np.full(N, geo.T_bath)
    if scenario == "quench":
        T0[geo.turn_id == 2] = 19.0
    steps = 40
    orc = qo.Oracle(geo, mat)
    orc.write(J0, T0, 0.0, 0.0)
    dt, held, dts_ref = 1e-4, 0, []
    for _ in range(steps):
        Jb = orc.J.copy()
        ret = orc.step(dt, w.I_ramp)
        dts_ref.append(dt)
        s = np.max(np.abs(orc.J - Jb)) / Jref
        if ret & 3:
            held = 10
        if held > 0:
            held -= 1
            dt = 1e-6
        elif s > 0.02:
            dt = max(dt / 2, 1e-6)
        elif s < 0.005:
            dt = min(2 * dt, 1e-4)
    with pkg.QS(geo, mat) as sim:
        sim.write(J0, T0, 0.0, 0.0)
        dts = run_adaptive(sim, geo, mat, w.I_ramp, steps)
        got = sim.read()
    assert dts == dts_ref, (dts, dts_ref)
    assert len(set(dts)) >= 2, dts
    check_state(orc.read(), got)


def test_heun_euler_rk_steps(pkg):
    # f2: embedded Heun-Euler pair with error control.  The oracle runs under its own controller; the
    # GPU is offered the oracle's accepted dt of every step and must accept it at the first try with the same error
    # estimate, suggestion and state.  Single wire under a fast background ramp (nonlinear, both stages differ).
    w = wl.shrunk(1, 1, 1, 12)
    geo = dataclasses.replace(w.geometry, Bext_rate=50.0)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    rtol, dt_min = 2e-4, 1e-8
    orc = qo.Oracle(geo, mat)
    with pkg.QS(geo, mat) as sim:
        dt = 1e-4
        taken = []
        for k in range(40):
            ro, dt_o, nxt_o, err_o = orc.step_rk(dt, 0.0, rtol, dt_min)
            rg, dt_g, nxt_g, err_g = sim.step_rk(dt_o, 0.0, rtol, dt_min)
            assert dt_g == dt_o and ro == (rg & 3), (k, dt_o, dt_g, err_o, err_g)
            assert abs(err_g - err_o) <= 1e-6 * err_o + 1e-15 and abs(nxt_g - nxt_o) <= 1e-6 * nxt_o
            taken.append(dt_o)
            dt = nxt_o
        got = sim.read()
        st = sim.stats()
    assert len(set(taken)) > 3 and min(taken) < 1e-4                        # the controller really adapted
    check_state(orc.read(), got)
    assert abs(st["t"] - orc.t) <= 1e-15 and abs(st["U_terminal"] - orc.stats["U_terminal"]) <= 1e-6 * abs(orc.stats["U_terminal"]) + 1e-20


def test_heun_euler_rejects_an_oversized_step_on_the_gpu(pkg):
    w = wl.shrunk(1, 1, 1, 12)
    geo = dataclasses.replace(w.geometry, Bext_rate=50.0)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    orc = qo.Oracle(geo, mat)
    with pkg.QS(geo, mat) as sim:
        for _ in range(6):                                                   # build up screening currents first
            orc.step(1e-4, 0.0)
            sim.step(1e-4, 0.0)
        ro, dt_o, nxt_o, err_o = orc.step_rk(2e-3, 0.0, 1e-5, 1e-8)
        rg, dt_g, nxt_g, err_g = sim.step_rk(2e-3, 0.0, 1e-5, 1e-8)
    assert dt_o < 2e-3 and abs(dt_g - dt_o) <= 1e-6 * dt_o and err_g <= 1e-5
    # linear regime on a coil: both stages give the same rate, err = 0, the suggestion doubles
    w = wl.shrunk(0, 2, 2, 4)
    with pkg.QS(w.geometry, w.material) as sim:
        rc, dt_g, nxt, err = sim.step_rk(1e-4, 50.0, 1e-6, 1e-9)
    assert dt_g == 1e-4 and err <= 1e-9 and abs(nxt - 2e-4) < 1e-18


def test_steps_with_the_adi_heat_scheme(pkg):
    # material.heat_adi_substeps = m: S6 by m ADI sub-steps (C15) inside qs_step, a hot turn relaxing by conduction
    w = wl.shrunk(0, 3, 3, 6)
    geo = w.geometry
    mat = dataclasses.replace(w.material, heat_adi_substeps=2)
    N = geo.n_rings
    T0 = np.full(N, geo.T_bath)
    T0[geo.turn_id == 4] = 9.0
    orc, sim, ref, got, rets = run_both(pkg, geo, mat, 25, w.dt, w.I_ramp, prep=(np.zeros(N), T0))
    assert sim.stats()["heat_substeps"] == 2 and all(a == b for a, b in rets)
    check_state(ref, got)
    assert ref[1].max() < 9.0 and ref[1].min() >= geo.T_bath - 1e-9
    sim.close()


def test_energy_balance_of_whole_steps_on_the_gpu(pkg):
    # north_star: "the Joule heat integral equals the enthalpy rise plus boundary flux".  Adiabatic pack (h_conv = 0),
    # dissipative state (|J| ~ Jc): sum_c V_c (H_c^{end} - H_c^0) = sum_steps dt * joule_power, GPU quantities only
    w = wl.shrunk(0, 2, 2, 8)
    geo = dataclasses.replace(w.geometry, h_conv=(0.0, 0.0, 0.0, 0.0))
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    N = geo.n_rings
    Jc0 = mat.Jc0 * (1 - geo.T_bath / mat.Tc) ** 2
    g = np.random.default_rng(21)
    J0 = Jc0 * g.uniform(0.9, 1.05, N)
    T0 = np.full(N, geo.T_bath)
    V = 2 * np.pi * geo.r * geo.area
    with pkg.QS(geo, mat) as sim:
        sim.write(J0, T0, 0.0, 0.0)
        total = 0.0
        for _ in range(8):
            assert sim.step(2e-5, 0.0) >= 0
            total += 2e-5 * sim.stats()["joule_power"]
        _, T1, _, _ = sim.read()
        ws = sim.wire_stats()
    dH = qo.enthalpy(mat, T1) - qo.enthalpy(mat, T0)
    assert total > 0 and abs(np.sum(V * dH) - total) <= 1e-9 * total
    assert abs(ws["E_joule"].sum() - total) <= 1e-9 * total          # per-wire energies add up to the same integral


@pytest.mark.parametrize("tables", [False, True])
def test_nonlinear_trajectory_ends_in_the_closed_form_saturated_state_on_the_gpu(pkg, tables):
    # not an oracle comparison: the CUDA path against the closed form of the stationary saturated state under a steady
    # field ramp (2 pi r E = -pi r^2 Bdot - V_w, J = Jc sgn(E) (|E|/Ec)^(1/n), V_w from sum a J = 0 per turn), which
    # tests/test_oracle_solver_step.py derives and pins the oracle with.  Both operators.
    from test_oracle_solver_step import saturated_state, saturation_workload
    w = saturation_workload(layers=2, turns=2, n=8)
    geo, mat = w.geometry, dataclasses.replace(w.material, cg_tol=1e-12)
    Js, Es, Us = saturated_state(geo, mat, np.asarray(mat.jc0_scale), geo.Bext_rate)
    with pkg.QS(geo, mat, lattice_tables=tables) as sim:
        for k in range(w.steps):
            assert sim.step(w.dt, 0.0) >= 0
        J, T, B, E = sim.read()
        st = sim.stats()
    assert rel(J, Js) < 1e-9, rel(J, Js)
    assert rel(E, Es) < 1e-8, rel(E, Es)
    assert abs(st["U_terminal"] - Us.sum()) < 1e-8 * abs(Us.sum())


def test_nonlinear_transient_power_balance_on_the_gpu(pkg):
    # GPU quantities only (qs_step, qs_read, qs_matvec): Poynting balance of the moving flux front, first order in dt
    from test_oracle_solver_step import power_balance_residual
    w = wl.shrunk(1, 1, 1, 8)
    geo = dataclasses.replace(w.geometry, Bext_rate=10.0)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    res = []
    for dt in (1e-4, 5e-5):
        with pkg.QS(geo, mat) as sim:
            def read_JE():
                J, _, _, E = sim.read(T=False, B=False)
                return J, E
            rr, share = power_balance_residual(lambda d: sim.step(d, 0.0), read_JE, sim.matvec, geo, 10.0, dt,
                                               int(round(0.02 / dt)))
        res.append(rr)
        assert 0.2 < share < 0.4
    assert 0 < res[0] < 0.01 and 1.8 < res[0] / res[1] < 2.2

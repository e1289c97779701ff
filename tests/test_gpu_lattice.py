"""GPU parity of the lattice-aware operator (QS_GEO_LATTICE_TABLES) against the CPU oracle and
against the on-the-fly pair sweeps: same unique pair values, block-Toeplitz application."""
import dataclasses

import numpy as np
import pytest

import workloads as wl
from oracle import qs_oracle as qo

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def pkg():
    import paper_2403_07666_b200 as p
    return p


# (layers, turns, n): Nz = turns * n covers every thread/output shape of the sweeps: 8, 18 (ragged), 65 (odd), 96, and
# for the tensor-core kernel (Nz >= 128) 130, 143 (odd: padded table rows, folded offset window) and 328 (several warps)
@pytest.mark.parametrize("shape", [(1, 1, 8), (2, 3, 6), (2, 5, 13), (3, 4, 24), (2, 10, 13), (2, 11, 13), (1, 41, 8)])
def test_tables_matvec_and_field_equal_the_dense_oracle(pkg, shape):
    L, Tn, n = shape
    geo = wl.lattice_geometry(L, Tn, n, 0.9e-3, 35e-3)
    N = geo.n_rings
    g = np.random.default_rng(5 + N)
    x = g.standard_normal(N)
    with pkg.QS(geo, wl.Material(), lattice_tables=True) as sim:
        y, B = sim.matvec(x), sim.field(x)
    with pkg.QS(geo, wl.Material()) as fly:
        y2, B2 = fly.matvec(x), fly.field(x)
    GBr, GBz = qo.dense_GB(geo)
    assert rel(y, qo.dense_M(geo) @ x) <= 1e-9
    assert rel(B[:N], GBr @ x) <= 1e-9 and rel(B[N:], GBz @ x) <= 1e-9
    assert rel(y, y2) <= 1e-12 and rel(B, B2) <= 1e-12           # the two GPU operators agree far tighter


@pytest.mark.parametrize("cfg", [0, 1])
def test_tables_configs_matvec(pkg, cfg):
    w = wl.config(cfg)
    geo = w.geometry
    x = np.random.default_rng(40 + cfg).standard_normal(geo.n_rings)
    with pkg.QS(geo, w.material, lattice_tables=True) as sim:
        y = sim.matvec(x)
    assert rel(y, qo.dense_M(geo) @ x) <= 1e-9


def test_tables_config2_full_size_sampled_rows(pkg):
    w = wl.config(2)
    geo = w.geometry
    x = np.random.default_rng(32).standard_normal(geo.n_rings)
    idx = wl.sample_rows(geo.n_rings, 48, seed=2)
    with pkg.QS(geo, w.material, lattice_tables=True) as sim:
        y = sim.matvec(x)
        B = sim.field(x)
    assert rel(y[idx], qo.matvec_rows(geo, x, idx, chunk=16)) <= 1e-9
    Br, Bz = qo.field_eval_rows(geo, x, idx, chunk=8)
    assert rel(B[idx], Br) <= 1e-9 and rel(B[geo.n_rings + idx], Bz) <= 1e-9


# long rows of the tensor-core sweep, one case per launch shape (mma_sweep_shape): Nz = 128 (one warp, both of its
# tiles), 200 (second warp with its second tile beyond the row), 1200 (config 3's rows: three CTAs per row of 4 + 4 + 2
# active warps) and 8192 (the source blocks of a row split between CTAs: the windows of the fused sweep do not fit
# otherwise); exact oracle rows on a seeded sample, the on-the-fly sweeps on every ring
# (layers, turns, n, inner radius): the 0.82 m tall stack needs a radius the library accepts (k'^2 <= 0.98)
@pytest.mark.parametrize("shape", [(2, 16, 8, 50e-3), (2, 25, 8, 50e-3), (1, 100, 12, 50e-3), (1, 1024, 8, 0.2)])
def test_tables_long_rows_sampled(pkg, shape):
    L, Tn, n, r_in = shape
    geo = wl.lattice_geometry(L, Tn, n, 0.8e-3, r_in)
    N = geo.n_rings
    x = np.random.default_rng(77 + N).standard_normal(N)
    idx = wl.sample_rows(N, 64, seed=N)
    with pkg.QS(geo, wl.Material(), lattice_tables=True) as sim:
        y, B = sim.matvec(x), sim.field(x)
    with pkg.QS(geo, wl.Material()) as fly:
        y2, B2 = fly.matvec(x), fly.field(x)
    assert rel(y, y2) <= 1e-12 and rel(B, B2) <= 1e-12
    assert np.max(np.abs(y - y2)) <= 1e-11 * np.max(np.abs(y2)) and np.max(np.abs(B - B2)) <= 1e-11 * np.max(np.abs(B2))
    assert rel(y[idx], qo.matvec_rows(geo, x, idx, chunk=16)) <= 1e-9
    Br, Bz = qo.field_eval_rows(geo, x, idx, chunk=8)
    assert rel(B[idx], Br) <= 1e-9 and rel(B[N + idx], Bz) <= 1e-9


def test_tables_steps_config0_and_shrunk_config2(pkg):
    for w, steps in ((wl.config(0), 50), (wl.shrunk(2, 3, 5), 100)):
        geo = w.geometry
        mat = dataclasses.replace(w.material, cg_tol=1e-12)
        orc = qo.Oracle(geo, mat)
        with pkg.QS(geo, mat, lattice_tables=True) as sim:
            for _ in range(steps):
                assert orc.step(w.dt, w.I_ramp) == (sim.step(w.dt, w.I_ramp) & 3)
            got, ref = sim.read(), orc.read()
        for name, a, b in zip("JTB", got, ref):
            assert rel(a, b) <= 1e-6, name


def test_tables_nonlinear_config1_like(pkg):
    # single wire under a fast background ramp (flux penetrates): CG iterates every step through the table sweeps
    w = wl.shrunk(1, 1, 1, 16)
    geo = dataclasses.replace(w.geometry, Bext_rate=10.0)
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    orc = qo.Oracle(geo, mat)
    with pkg.QS(geo, mat, lattice_tables=True) as sim:
        its = 0
        for _ in range(40):
            orc.step(w.dt, 0.0)
            sim.step(w.dt, 0.0)
            its += sim.stats()["cg_iters"]
        got, ref = sim.read(), orc.read()
    assert its > 0
    for name, a, b in zip("JTBE", got, ref):
        assert rel(a, b) <= 1e-6, name


def test_tables_constrained_solve_and_rk_step_agree_with_the_pair_sweeps(pkg):
    # the solver and the Runge-Kutta step are operator-agnostic: same results through either operator
    w = wl.shrunk(2, 2, 9, 16)                                   # Nz = 144 >= 128: tensor-core sweep
    geo = w.geometry
    mat = dataclasses.replace(w.material, cg_tol=1e-12)
    b = np.random.default_rng(8).standard_normal(geo.n_rings) * 1e-6
    out = {}
    for tables in (False, True):
        with pkg.QS(geo, mat, lattice_tables=tables) as sim:
            x, it, relres, rc = sim.solve(b)
            assert rc == 0 and relres <= 1e-12
            geo2 = geo
            rk = [sim.step_rk(1e-4, w.I_ramp, 1e-6, 1e-9) for _ in range(3)]
            out[tables] = (x, rk, sim.read())
    xa, rka, sa = out[False]
    xb, rkb, sb = out[True]
    assert rel(xb, xa) <= 1e-8
    cs = np.bincount(geo.turn_id, weights=xb, minlength=geo.n_turns)
    assert np.max(np.abs(cs)) <= 1e-9 * np.max(np.abs(xb)) * 300     # C^T x = 0 kept by the projection
    for (ra, da, na, ea), (rb_, db, nb, eb) in zip(rka, rkb):
        assert ra == rb_ and da == db and abs(ea - eb) <= 1e-9 + 1e-6 * ea
    for a, b_ in zip(sa, sb):
        assert rel(b_, a) <= 1e-9 or np.linalg.norm(a) < 1e-30

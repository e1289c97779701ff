"""GPU parity of the pair operator K1/K2, the CG solve and the pointwise passes against the CPU oracle.

All calls go through the C ABI (paper_2403_07666_b200.QS -> libqs.so).  Tolerances: north_star
(rel-L2 <= 1e-9 for the G matvec); the pointwise passes are compared far tighter (same formulas in FP64,
differences come from FMA contraction and libm-vs-CUDA pow only).
"""
import dataclasses
import math

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


@pytest.mark.parametrize("n", [1, 31, 33, 1000, 4096])
def test_matvec_free_rings_full(pkg, n):
    geo, x = wl.free_rings(n, seed=4000 + n)
    with pkg.QS(geo, wl.Material()) as sim:
        y = sim.matvec(x)
        st = sim.stats()
    yo = qo.matvec(geo, x)
    assert rel(y, yo) <= 1e-9
    assert np.max(np.abs(y - yo)) <= 1e-9 * np.max(np.abs(yo))
    nb = (n + 31) // 32
    assert st["pair_evals"] >= nb * (nb + 1) // 2 * 1024 and st["launches"] > 0


@pytest.mark.parametrize("n,rows", [(65536, 1024), (262144, 1024), (1048576, 1024)])
def test_matvec_free_rings_sampled_rows(pkg, n, rows):
    # BASELINE.json configs[4] sizes; the oracle evaluates exact rows sum_j M_ij x_j on a seeded sample of 1024 target
    # rows (SURVEY.md §8(d) parity protocol), pair by pair against all n sources
    geo, x = wl.free_rings(n)
    idx = wl.sample_rows(n, rows, seed=n)
    with pkg.QS(geo, wl.Material()) as sim:
        y = sim.matvec(x)
    yo = qo.matvec_rows(geo, x, idx, chunk=16)
    assert rel(y[idx], yo) <= 1e-9
    assert np.max(np.abs(y[idx] - yo)) <= 1e-9 * np.max(np.abs(yo))
    assert np.all(np.isfinite(y))


def test_matvec_device_variant_and_symmetry(pkg):
    import torch
    geo, x = wl.free_rings(2048)
    g = np.random.default_rng(11)
    w = g.standard_normal(2048)
    with pkg.QS(geo, wl.Material()) as sim:
        y = sim.matvec(x)
        with torch.cuda.stream(sim.stream):
            xd = torch.from_numpy(x).to(sim.device)
            yd = torch.empty_like(xd)
        sim.stream.synchronize()
        sim.matvec_device(xd, yd)
        sim.sync()
        assert rel(yd.cpu().numpy(), y) <= 1e-13
        Mw = sim.matvec(w)
    # x^T M w == w^T M x (one evaluation per unordered pair makes this exact up to summation order); SPD
    assert abs(x @ Mw - w @ y) <= 1e-12 * abs(w @ y)
    assert x @ y > 0 and w @ Mw > 0


@pytest.mark.parametrize("cfg", [0, 1])
def test_matvec_and_field_lattice_configs(pkg, cfg):
    w = wl.config(cfg)
    geo = w.geometry
    g = np.random.default_rng(20 + cfg)
    x = g.standard_normal(geo.n_rings)
    with pkg.QS(geo, w.material) as sim:
        y = sim.matvec(x)
        B = sim.field(x)
    M = qo.dense_M(geo)
    assert rel(y, M @ x) <= 1e-9
    del M
    GBr, GBz = qo.dense_GB(geo)
    N = geo.n_rings
    assert rel(B[:N], GBr @ x) <= 1e-9 and rel(B[N:], GBz @ x) <= 1e-9


def test_matvec_ragged_lattice(pkg):
    # Nz = 18 is not a multiple of 32: blocks straddle rows, last block is padded (N = 12*18 = 216)
    geo = wl.lattice_geometry(2, 3, 6, 0.9e-3, 35e-3)
    x = np.random.default_rng(3).standard_normal(geo.n_rings)
    with pkg.QS(geo, wl.Material()) as sim:
        y, B = sim.matvec(x), sim.field(x)
    GBr, GBz = qo.dense_GB(geo)
    assert rel(y, qo.dense_M(geo) @ x) <= 1e-9
    assert rel(B[:216], GBr @ x) <= 1e-9 and rel(B[216:], GBz @ x) <= 1e-9


@pytest.mark.parametrize("cfg,rows", [(2, 96), (3, 32)])
def test_matvec_full_size_coils_sampled_rows(pkg, cfg, rows):
    w = wl.config(cfg)
    geo = w.geometry
    x = np.random.default_rng(30 + cfg).standard_normal(geo.n_rings)
    idx = wl.sample_rows(geo.n_rings, rows, seed=cfg)
    with pkg.QS(geo, w.material) as sim:
        y = sim.matvec(x)
    assert rel(y[idx], qo.matvec_rows(geo, x, idx, chunk=16)) <= 1e-9


def test_solve_free_rings_and_constrained_lattice(pkg):
    geo, x = wl.free_rings(1024)
    mat = wl.Material(cg_tol=1e-10, cg_maxit=20000)
    M = qo.dense_M(geo)
    b = M @ x
    with pkg.QS(geo, mat) as sim:
        xs, it, relres, rc = sim.solve(b)
    assert rc == 0 and 0 < it < 20000 and relres <= 1e-10
    assert rel(M @ xs, b) <= 1e-8
    xd = np.linalg.solve(M, b)
    assert rel(xs, xd) <= 1e-4                                   # cond(M) ~ 1e6
    # lattice with turns: M x + C V = b, C^T x = 0 against the dense KKT solve
    geo = wl.lattice_geometry(2, 2, 8, 1e-3, 30e-3)
    b = np.random.default_rng(5).standard_normal(geo.n_rings) * 1e-6
    xk, _ = qo.kkt_dense(qo.dense_M(geo), qo.constraint_matrix(geo), b, np.zeros(geo.n_turns))
    with pkg.QS(geo, wl.Material(cg_tol=1e-12)) as sim:
        xs, it, relres, rc = sim.solve(b)
    assert rc == 0 and rel(xs, xk) <= 1e-8
    assert np.max(np.abs(np.bincount(geo.turn_id, weights=xs))) <= 1e-10 * np.max(np.abs(xs)) * 64


def test_solve_maxit_is_reported(pkg):
    geo, x = wl.free_rings(512)
    with pkg.QS(geo, wl.Material(cg_tol=1e-14)) as sim:
        _, it, relres, rc = sim.solve(sim.matvec(x), maxit=5)
    assert rc == 4 and it == 5 and relres > 1e-14


def test_material_law_pointwise(pkg):
    w = wl.shrunk(0, 3, 2, 8)
    geo, mat = w.geometry, w.material
    N = geo.n_rings
    g = np.random.default_rng(8)
    Jc0 = 2e9 * (1 - 4.2 / 18) ** 2
    J = Jc0 * g.uniform(-1.3, 1.3, N)
    J[:7] = 0.0
    J[7:12] = 1e3 * Jc0                                          # deep normal state / overflow guard
    T = g.uniform(4.2, 17.0, N)
    T[20:30] = 19.0                                              # above Tc
    B = np.concatenate([g.uniform(-2, 2, N), g.uniform(-12, 12, N)])
    dt = 1e-4
    with pkg.QS(geo, mat) as sim:
        sim.write(J, T, 0.0, 0.0)
        sim.set_fields(B=B)
        sim.material_eval(dt)
        _, Tg, Bg, E = sim.read()
        aux = sim.read_aux()
    ml = qo.material_law(mat, J, T, B[:N], B[N:], geo.r, mat.jc0_scale)
    assert np.max(np.abs(Tg - T)) <= 1e-13 * 19 and np.array_equal(Bg, B)
    assert np.any(ml["Jc"] == 0.0) and np.any(ml["rho"] == mat.rho_n) and np.any(ml["rho"] == 0.0)
    for key, got in [("E", E), ("Q", aux["Q"]), ("dEdJ", aux["dEdJ"]), ("Jc", aux["Jc"]), ("rho", aux["rho"])]:
        ref = ml[key]
        assert np.max(np.abs(got - ref)) <= 1e-11 * np.max(np.abs(ref)), key
        assert rel(got, ref) <= 1e-12, key


# lattices of <= 4096 cells run all sub-steps in one launch: one CTA below 16 rows ((1, 1, 8), (3, 2, 4)), a cluster of
# 8 CTAs with DSMEM halo rows from there: 16 rows = 2 per CTA (1, 1, 16), ragged bands with an empty last CTA
# ((2, 5, 13): 26 rows, (2, 3, 10): 20 rows), configs 0 and 1 ((4, 4, 8), (1, 1, 64)); (5, 3, 24) is the blocked kernel
@pytest.mark.parametrize("shape", [(1, 1, 8), (3, 2, 4), (2, 5, 13), (5, 3, 24), (1, 1, 16), (2, 3, 10), (4, 4, 8), (1, 1, 64)])
def test_heat_substeps_pointwise(pkg, shape):
    L, Tn, n = shape
    geo = wl.lattice_geometry(L, Tn, n, 1e-3, 30e-3)
    geo = dataclasses.replace(geo, h_conv=(500.0, 300.0, 200.0, 100.0))
    mat = wl.Material()
    N = geo.n_rings
    g = np.random.default_rng(9)
    T = g.uniform(4.2, 12.0, N)
    Q = g.uniform(0, 5e6, N)
    dt = 1e-4
    with pkg.QS(geo, mat, no_operator=True) as sim:
        sim.write(np.zeros(N), T, 0.0, 0.0)
        sim.set_fields(Q=Q)
        m = sim.heat(dt)
        _, Tg, _, _ = sim.read(J=False, B=False, E=False)
    mo = qo.heat_substeps_count(geo, mat, dt)
    Ho, _ = qo.heat_substeps(geo, mat, qo.enthalpy(mat, T), Q, dt, mo)
    assert m == mo
    assert np.max(np.abs(Tg - qo.temperature(mat, Ho))) <= 1e-12 * 12.0


@pytest.mark.parametrize("shape,msub", [((7, 9, 11), 6), ((20, 17, 8), 4), ((5, 3, 24), 9), ((9, 13, 7), 1), ((9, 13, 7), 3)])
def test_heat_temporally_blocked_kernel(pkg, shape, msub):
    # lattices above 4096 cells: groups of <= 4 sub-steps per launch from a shared-memory tile with a 4-cell halo.
    # Odd sizes (tiles cut by all four pack borders), sub-step counts that are not multiples of 4 (a short last group),
    # Robin loss on all borders, strong gradients: cell by cell against the oracle's sub-step loop.
    L, Tn, n = shape
    geo = wl.lattice_geometry(L, Tn, n, 1e-3, 30e-3)
    geo = dataclasses.replace(geo, h_conv=(500.0, 300.0, 200.0, 100.0))
    mat = wl.Material()
    N = geo.n_rings
    assert N > 4096
    g = np.random.default_rng(100 + msub)
    T = g.uniform(4.2, 12.0, N)
    Q = g.uniform(0, 5e6, N)
    alpha0 = mat.k_in / (mat.C3 * geo.T_bath ** 2 + mat.C1)
    dt = (msub - 0.5) * 0.8 * geo.h ** 2 / (4.0 * alpha0)
    assert qo.heat_substeps_count(geo, mat, dt) == msub
    with pkg.QS(geo, mat, no_operator=True) as sim:
        sim.write(np.zeros(N), T, 0.0, 0.0)
        sim.set_fields(Q=Q)
        for _ in range(3):                                       # three steps: ping-pong buffers, graph replay (msub > 8)
            assert sim.heat(dt) == msub
        _, Tg, _, _ = sim.read(J=False, B=False, E=False)
    Ho = qo.enthalpy(mat, T)
    for _ in range(3):
        Ho, _ = qo.heat_substeps(geo, mat, Ho, Q, dt, msub)
    assert np.max(np.abs(Tg - qo.temperature(mat, Ho))) <= 1e-12 * 12.0


def test_heat_temporally_blocked_kernel_forced_on_a_large_lattice(pkg):
    # 2048 x 2048 cells: above the size the library blocks by itself (QS_GEO_HEAT_BLOCKED forces it: the 64 x 64-tile
    # variant); 4 sub-steps in one launch, and 6 (4 + 2), cell by cell against the oracle
    geo = wl.lattice_geometry(32, 32, 64, 1e-3, 30e-3)
    geo = dataclasses.replace(geo, h_conv=(500.0, 300.0, 200.0, 100.0))
    mat = wl.Material()
    N = geo.n_rings
    g = np.random.default_rng(404)
    T = g.uniform(4.2, 12.0, N)
    Q = g.uniform(0, 5e6, N)
    alpha0 = mat.k_in / (mat.C3 * geo.T_bath ** 2 + mat.C1)
    for msub in (4, 6):
        dt = (msub - 0.5) * 0.8 * geo.h ** 2 / (4.0 * alpha0)
        with pkg.QS(geo, mat, no_operator=True, heat_blocked=True) as sim:
            sim.write(np.zeros(N), T, 0.0, 0.0)
            sim.set_fields(Q=Q)
            assert sim.heat(dt) == msub
            _, Tg, _, _ = sim.read(J=False, B=False, E=False)
        Ho, _ = qo.heat_substeps(geo, mat, qo.enthalpy(mat, T), Q, dt, msub)
        assert np.max(np.abs(Tg - qo.temperature(mat, Ho))) <= 1e-12 * 12.0


def test_errors_and_no_operator_mode(pkg):
    geo, x = wl.free_rings(64)
    with pkg.QS(geo, wl.Material()) as sim:
        with pytest.raises(pkg.QsError) as e:
            sim.step(1e-4, 0.0)                                  # free rings cannot step
        assert e.value.code == -1
    w = wl.shrunk(0, 1, 1, 4)
    with pkg.QS(w.geometry, w.material) as sim:
        with pytest.raises(pkg.QsError) as e:
            sim.step(0.0, 1.0)
        assert e.value.code == -5
    with pkg.QS(w.geometry, w.material, no_operator=True) as sim:
        with pytest.raises(pkg.QsError):
            sim.matvec(np.ones(16))
    bad = dataclasses.replace(w.geometry, r=w.geometry.r[::-1].copy())
    with pytest.raises(pkg.QsError):
        pkg.QS(bad, w.material)                                  # r/z arrays contradict the lattice description
    with pkg.QS(w.geometry, w.material, torch_memory=False) as sim:   # plain-C path: cudaMalloc + own stream
        y = sim.matvec(np.ones(16))
    assert rel(y, qo.dense_M(w.geometry) @ np.ones(16)) <= 1e-9


def test_pair_arithmetic_every_class_at_its_threshold(pkg):
    # per-pair K, E, M of the sweeps against the oracle's library route (scipy Cephes K/E + Maxwell bracket),
    # each evaluation class probed from its own k'^2 threshold upwards (where its truncation error is largest)
    from paper_2403_07666_b200 import pair_eval
    # classes (NIT, ORD): (2,2) (2,4) (3,2) (3,4) (4,2) (4,4) (5,2) (5,4) (6,2) (7,2)
    thr = [0.3965, 0.1394, 0.01529, 1.374e-3, 1.453e-5, 1.157e-7, 1.293e-11, 8.2e-16, 1.03e-23, 1e-27]
    ri = 0.05
    for cls, t in enumerate(thr):
        kp2 = t * np.logspace(0.0, 1.0, 64) if t < 0.09 else np.linspace(t, 0.98, 64)
        kp2 = np.minimum(kp2, 0.98)
        # coaxial pair with ri = rj: A2 = 4 ri^2 + dz^2, B2 = dz^2  ->  dz^2 = 4 ri^2 kp2/(1-kp2)
        dz2 = 4 * ri * ri * kp2 / (1.0 - kp2)
        A2, B2 = 4 * ri * ri + dz2, dz2
        M, K, E, used = pair_eval(A2, B2, cls)
        assert np.all(used == cls)
        Ko, Eo = qo.elliptic_KE(B2 / A2)
        Mo = qo.mutual_pair(ri, 0.0, ri, 0.0, soft2=dz2)
        assert np.max(np.abs(K / Ko - 1)) <= 4e-15, (cls, np.max(np.abs(K / Ko - 1)))
        assert np.max(np.abs(E / Eo - 1)) <= 2e-14, (cls, np.max(np.abs(E / Eo - 1)))
        # Maxwell's bracket loses digits to cancellation at small k (far pairs): compare M where it is well conditioned
        ok = kp2 <= 0.5
        if np.any(ok):
            assert np.max(np.abs(M[ok] / Mo[ok] - 1)) <= 2e-14, (cls, np.max(np.abs(M[ok] / Mo[ok] - 1)))
    # automatic class choice is monotone in k'^2 and never cheaper than the threshold table allows
    kp2 = np.logspace(-26, np.log10(0.98), 400)
    dz2 = 4 * ri * ri * kp2 / (1.0 - kp2)
    M, K, E, used = pair_eval(4 * ri * ri + dz2, dz2, -1)
    assert np.all(np.diff(used) <= 0)
    Ko, Eo = qo.elliptic_KE(dz2 / (4 * ri * ri + dz2))
    assert np.max(np.abs(K / Ko - 1)) <= 4e-15 and np.max(np.abs(E / Eo - 1)) <= 2e-14


@pytest.mark.parametrize("n_exp,eps_exp", [(15.0, 1.7), (20.5, 2.3), (2.0, 1.0)])
def test_material_law_other_exponents(pkg, n_exp, eps_exp):
    # integer n != 20 (binary powering), non-integer n (exp/log path), other strain exponents
    w = wl.shrunk(0, 2, 2, 6)
    geo = w.geometry
    mat = dataclasses.replace(w.material, n_exp=n_exp, eps_exp=eps_exp)
    N = geo.n_rings
    g = np.random.default_rng(int(10 * n_exp))
    Jc0 = 2e9 * (1 - 4.2 / 18) ** 2
    J = Jc0 * g.uniform(-1.2, 1.2, N)
    T = g.uniform(4.2, 16.0, N)
    B = np.concatenate([g.uniform(-2, 2, N), g.uniform(-12, 12, N)])
    with pkg.QS(geo, mat) as sim:
        sim.write(J, T, 0.0, 0.0)
        sim.set_fields(B=B)
        sim.material_eval(1e-4)
        _, _, _, E = sim.read()
        aux = sim.read_aux()
    ml = qo.material_law(mat, J, T, B[:N], B[N:], geo.r, mat.jc0_scale)
    for key, got in [("E", E), ("Q", aux["Q"]), ("dEdJ", aux["dEdJ"]), ("Jc", aux["Jc"]), ("rho", aux["rho"])]:
        assert rel(got, ml[key]) <= 1e-11, key


def test_material_law_on_free_rings(pkg):
    # the per-cell-array path of the material pass (no lattice row tables, no event reduction)
    geo, _ = wl.free_rings(300, seed=9)
    geo = dataclasses.replace(geo, T_bath=4.2)
    mat = wl.Material(jc0_scale=wl.jc0_scale(3, 300, 0.02))
    g = np.random.default_rng(77)
    J = 1e9 * g.uniform(-1.0, 1.0, 300)
    T = g.uniform(4.2, 19.0, 300)
    B = np.concatenate([g.uniform(-1, 1, 300), g.uniform(-8, 8, 300)])
    with pkg.QS(geo, mat) as sim:
        sim.write(J, T, 0.0, 0.0)
        sim.set_fields(B=B)
        sim.material_eval(1e-4)
        _, Tg, _, E = sim.read()
        aux = sim.read_aux()
    ml = qo.material_law(mat, J, T, B[:300], B[300:], geo.r, mat.jc0_scale)
    assert np.max(np.abs(Tg - T)) <= 1e-12 * 19
    for key, got in [("E", E), ("Q", aux["Q"]), ("dEdJ", aux["dEdJ"]), ("Jc", aux["Jc"]), ("rho", aux["rho"])]:
        assert rel(got, ml[key]) <= 1e-11, key


def test_heat_adiabatic_energy_conservation_on_the_gpu(pkg):
    # h_conv = 0: sum_c V_c (H_c' - H_c) = dt sum_c V_c Q_c to rounding (finite-volume fluxes cancel pairwise)
    geo = wl.lattice_geometry(3, 4, 10, 1e-3, 30e-3, h_conv=0.0)
    mat = wl.Material()
    N = geo.n_rings
    g = np.random.default_rng(12)
    T = g.uniform(4.2, 15.0, N)
    Q = g.uniform(0, 5e6, N)
    dt = 2e-4
    with pkg.QS(geo, mat, no_operator=True) as sim:
        sim.write(np.zeros(N), T, 0.0, 0.0)
        sim.set_fields(Q=Q)
        m = sim.heat(dt)
        _, T1, _, _ = sim.read(J=False, B=False, E=False)
    assert m > 1
    V = 2 * np.pi * geo.r * geo.h ** 2
    dH = qo.enthalpy(mat, T1) - qo.enthalpy(mat, T)
    assert abs(np.sum(V * dH) - dt * np.sum(V * Q)) <= 1e-10 * dt * np.sum(V * Q)


@pytest.mark.parametrize("shape", [(1, 1, 8), (3, 2, 4), (2, 5, 13), (5, 3, 24), (1, 1, 1), (2, 1, 40)])
def test_heat_adi_substeps_pointwise(pkg, shape):
    # f4 / C15: the ADI heat step against the oracle's sparse-solve restatement; sub-steps of 5 x the explicit limit
    # (rough random data: the lagged-capacity linearisation is not positivity preserving far beyond that)
    L, Tn, n = shape
    geo = wl.lattice_geometry(L, Tn, n, 1e-3, 30e-3)
    geo = dataclasses.replace(geo, h_conv=(500.0, 300.0, 200.0, 100.0))
    mat = wl.Material()
    N = geo.n_rings
    g = np.random.default_rng(19)
    T = g.uniform(4.2, 9.0, N)
    Q = g.uniform(0, 5e6, N)
    m = 3
    dt = m * 5 * 0.8 * geo.h ** 2 / (4 * mat.k_in / (mat.C3 * 4.2 ** 2 + mat.C1))
    with pkg.QS(geo, mat, no_operator=True) as sim:
        sim.write(np.zeros(N), T, 0.0, 0.0)
        sim.set_fields(Q=Q)
        assert sim.heat_adi(dt, m) == m
        _, Tg, _, _ = sim.read(J=False, B=False, E=False)
    Ho = qo.heat_adi(geo, mat, qo.enthalpy(mat, T), Q, dt, m)
    assert np.max(np.abs(Tg - qo.temperature(mat, Ho))) <= 1e-11 * 9.0


def test_hbm_leg_lattice_material_and_heat_full_arrays(pkg):
    # the launch configuration bench.py --leg hbm times (roofline_hbm): 4096 x 4096 cells (arrays larger than L2), the
    # material pass without the test outputs (aux=False) and one explicit heat sub-step, same seeded state; every cell
    # of E and T is compared with the oracle
    w = wl.lattice_workload("hbm_4096x4096", 64, 64, 64, 1.0e-3, 30e-3, 1e-4, 0.0, 1, 77, 0.01)
    geo, mat = w.geometry, w.material
    N = geo.n_rings
    g = np.random.default_rng(5)
    J = 1e8 * g.standard_normal(N)
    T = 4.2 + g.random(N)
    B = 0.1 * g.standard_normal(2 * N)
    Q = 1e3 * g.random(N)
    sub_dt = 1e-9
    with pkg.QS(geo, mat, no_operator=True) as sim:
        sim.write(J=J, T=T)
        sim.set_fields(B=B, Q=Q)
        sim.material_eval(1e-4, aux=False)
        _, _, _, E = sim.read(J=False, T=False, B=False)
        sim.set_fields(Q=Q)                                        # the material pass overwrote Q with E J
        m = sim.heat(sub_dt)
        _, Tg, _, _ = sim.read(J=False, B=False, E=False)
    assert m == 1
    ml = qo.material_law(mat, J, T, B[:N], B[N:], geo.r, mat.jc0_scale)
    assert np.max(np.abs(E - ml["E"])) <= 1e-11 * np.max(np.abs(ml["E"]))
    del ml
    Ho, _ = qo.heat_substeps(geo, mat, qo.enthalpy(mat, T), Q, sub_dt, 1)
    To = qo.temperature(mat, Ho)
    assert np.max(np.abs(Tg - To)) <= 1e-13 * 6.0
    assert np.max(np.abs((Tg - T) - (To - T))) <= 1e-6 * np.max(np.abs(To - T))   # the increment itself, not just T

"""Pins of the oracle's constrained solve, lattice tables and whole step (C6, C7, C10)."""
import dataclasses
import math

import numpy as np
import pytest

import workloads as wl
from oracle import qs_oracle as qo

MU0 = 4e-7 * math.pi


def small_lattice():
    return wl.lattice_geometry(2, 3, 4, 1e-3, 30e-3)


def test_kkt_dense_satisfies_the_kkt_system():
    geo = small_lattice()
    g = np.random.default_rng(1)
    M = qo.dense_M(geo)
    A = M + np.diag(g.random(geo.n_rings) * 1e-8)
    C = qo.constraint_matrix(geo)
    assert C.shape == (96, 6) and np.all(C.sum(axis=1) == 1) and np.all(C.sum(axis=0) == 16)
    b = g.standard_normal(geo.n_rings) * 1e-6
    d = g.standard_normal(geo.n_turns) * 10
    x, V = qo.kkt_dense(A, C, b, d)
    # brute force: the full (N + Nw) KKT matrix solved by LU
    KKT = np.block([[A / MU0, C], [C.T, np.zeros((6, 6))]])
    sol = np.linalg.solve(KKT, np.concatenate([b / MU0, d]))
    assert np.max(np.abs(x - sol[:96])) < 1e-9 * np.max(np.abs(x))
    assert np.max(np.abs(V - sol[96:] * MU0)) < 1e-9 * np.max(np.abs(V))
    assert np.max(np.abs(C.T @ x - d)) < 1e-10 * np.max(np.abs(d))
    assert np.max(np.abs(A @ x + C @ V - b)) < 1e-9 * np.max(np.abs(b))


def test_projected_cg_equals_dense_kkt_and_keeps_the_constraint():
    geo = small_lattice()
    g = np.random.default_rng(2)
    M = qo.dense_M(geo)
    shift = g.random(geo.n_rings) * 1e-8
    A = M + np.diag(shift)
    b = g.standard_normal(geo.n_rings) * 1e-6
    d = np.full(geo.n_turns, 50.0)
    xd, Vd = qo.kkt_dense(A, qo.constraint_matrix(geo), b, d)
    x, V, it, rel = qo.pcg(lambda v: A @ v, np.diag(A).copy(), geo.turn_id, geo.n_turns, b, d, 1e-13, 500)
    assert 0 < it < 200 and rel <= 1e-13
    assert np.max(np.abs(x - xd)) < 1e-9 * np.max(np.abs(xd))
    assert np.max(np.abs(V - Vd)) < 1e-8 * np.max(np.abs(Vd))
    cur = np.bincount(geo.turn_id, weights=x)
    assert np.max(np.abs(cur - d)) < 1e-10 * 50
    # warm start from the solution: converged at once; from a perturbed solution: same answer
    x2, V2, it2, _ = qo.pcg(lambda v: A @ v, np.diag(A).copy(), geo.turn_id, geo.n_turns, b, d, 1e-10, 500, x0=xd)
    assert it2 == 0 and np.max(np.abs(V2 - Vd)) < 1e-8 * np.max(np.abs(Vd))
    x3, _, it3, _ = qo.pcg(lambda v: A @ v, np.diag(A).copy(), geo.turn_id, geo.n_turns, b, d, 1e-13, 500,
                           x0=xd * (1 + 0.1 * g.standard_normal(96)))
    assert np.max(np.abs(x3 - xd)) < 1e-9 * np.max(np.abs(xd))


def test_unconstrained_cg_on_free_rings():
    geo, x = wl.free_rings(256)
    o = qo.Oracle(geo, wl.Material(cg_tol=1e-13, cg_maxit=5000))
    b = o.apply_M(x)
    assert np.max(np.abs(b - qo.matvec(geo, x))) == 0.0
    xd, _, _ = o.solve(b, dense=True)
    xc, it, rel = o.solve(b)
    assert np.linalg.norm(xd - x) < 1e-6 * np.linalg.norm(x)              # cond ~ 1e6
    assert np.linalg.norm(o.apply_M(xc) - b) < 1e-11 * np.linalg.norm(b)


def test_lattice_tables_equal_dense_operators():
    geo = wl.lattice_geometry(3, 2, 3, 0.8e-3, 40e-3)
    g = np.random.default_rng(3)
    x = g.standard_normal(geo.n_rings)
    tab = qo.LatticeTables(geo)
    M = qo.dense_M(geo)
    GBr, GBz = qo.dense_GB(geo)
    assert np.max(np.abs(tab.matvec(x) - M @ x)) < 1e-14 * np.max(np.abs(M @ x))
    br, bz = tab.field(x)
    assert np.max(np.abs(br - GBr @ x)) < 1e-13 * np.max(np.abs(GBr @ x))
    assert np.max(np.abs(bz - GBz @ x)) < 1e-13 * np.max(np.abs(GBz @ x))


def test_fft_application_of_the_tables_equals_the_offset_sum_and_the_dense_operators():
    # the circulant embedding must reproduce the defining sum: even (M, Bz) and odd (Br) tables, Nz not a power of two
    geo = wl.lattice_geometry(4, 5, 3, 0.8e-3, 50e-3)
    g = np.random.default_rng(11)
    x = g.standard_normal(geo.n_rings)
    tab = qo.LatticeTablesFFT(geo)
    M = qo.dense_M(geo)
    GBr, GBz = qo.dense_GB(geo)
    for got, ref in ((tab.matvec(x), M @ x), (tab.field(x)[0], GBr @ x), (tab.field(x)[1], GBz @ x),
                     (tab.matvec(x), tab.matvec_plain(x)), (tab.field(x)[0], tab.field_plain(x)[0])):
        assert np.max(np.abs(got - ref)) < 1e-13 * np.max(np.abs(ref))
    # a delta source picks single table entries: sign and offset bookkeeping of the odd table
    e = np.zeros(geo.n_rings)
    e[2 * geo.Nz + 7] = 1.0
    br = tab.field(e)[0].reshape(geo.Nr, geo.Nz)
    assert abs(br[5, 9] - GBr[5 * geo.Nz + 9, 2 * geo.Nz + 7]) < 1e-13 * np.max(np.abs(GBr))
    assert abs(br[5, 5] - GBr[5 * geo.Nz + 5, 2 * geo.Nz + 7]) < 1e-13 * np.max(np.abs(GBr))
    assert br[5, 9] * br[5, 5] < 0.0


def test_single_ring_is_an_LR_circuit():
    # one normal-state ring (T > Tc: rho = rho_n) in a ramped axial field, no current constraint:
    # L I' + R I = -pi r^2 Bdot,  L = mu0 r [ln(8r/g) - 2],  R = rho_n 2 pi r / a;  I(t) = I_inf (1 - exp(-t/tau))
    base = wl.lattice_geometry(1, 1, 1, 1e-3, 30e-3, h_conv=0.0, Bext_rate=10.0, Bext_max=100.0)
    geo = dataclasses.replace(base, n_turns=0, turn_id=None)
    mat = wl.Material()
    r, a = geo.r[0], geo.area[0]
    L = MU0 * r * (math.log(8 * r / geo.softening) - 2.0)
    R = mat.rho_n * 2 * math.pi * r / a
    tau, I_inf = L / R, -math.pi * r * r * 10.0 / R
    t_end = 2.0 * tau
    errs = []
    for steps in (200, 400):
        o = qo.Oracle(geo, mat)
        o.write(np.zeros(1), np.full(1, 20.0), 0.0, 0.0)
        for _ in range(steps):
            assert o.step(t_end / steps, 0.0) >= 0
        assert o.T[0] >= 20.0
        exact = I_inf * (1 - math.exp(-o.t / tau))
        errs.append(abs(o.J[0] * a - exact) / abs(exact))
    assert errs[1] < 2e-3 and 1.8 < errs[0] / errs[1] < 2.2                # first order in dt, right limit


def test_step_keeps_turn_currents_and_inductance_in_linear_regime():
    w = wl.shrunk(0, 2, 2, 4)
    o = qo.Oracle(w.geometry, w.material)
    U = []
    for k in range(6):
        assert o.step(w.dt, w.I_ramp) == 0
        U.append(o.stats["U_terminal"])
        cur = np.bincount(w.geometry.turn_id, weights=o.J * w.geometry.area)
        assert np.max(np.abs(cur - o.I)) < 1e-10 * o.I
    assert abs(o.I - 6 * w.dt * w.I_ramp) < 1e-15
    assert max(U) - min(U) < 1e-9 * U[0] and U[0] > 0                    # U = L dI/dt, constant
    # the shielding inductance is below the uniform-current inductance sum(M)/Nw^2-normalised
    Luni = o.M.sum() / (16 * 16)
    assert 0.5 * Luni < U[0] / w.I_ramp < Luni
    assert np.all(o.T == w.geometry.T_bath)


def test_theta0_equals_theta1_in_linear_regime_and_solvers_agree():
    w = wl.shrunk(0, 2, 2, 4)
    outs = []
    for theta, op, solver in [(1.0, "dense", "cholesky"), (0.0, "dense", "cholesky"), (1.0, "tables", "pcg")]:
        mat = dataclasses.replace(w.material, theta=theta, cg_tol=1e-13)
        o = qo.Oracle(w.geometry, mat, operator=op, solver=solver)
        for k in range(5):
            o.step(w.dt, w.I_ramp)
        outs.append(o.read())
    for a, b in [(0, 1), (0, 2)]:
        for u, v in zip(outs[a], outs[b]):
            assert np.linalg.norm(u - v) <= 1e-9 * max(np.linalg.norm(u), 1e-300)


def test_nonlinear_magnetisation_dense_cholesky_vs_tables_cg():
    # shrunk config 1 (single wire in a ramped field): the flux front enters, |J|/Jc -> ~1, E' matters
    w = wl.shrunk(1, 1, 1, 12)
    geo = dataclasses.replace(w.geometry, Bext_rate=10.0)          # 10 T/s: the front crosses a cell in 300 steps
    outs = []
    for op, solver in [("dense", "cholesky"), ("tables", "pcg")]:
        o = qo.Oracle(geo, dataclasses.replace(w.material, cg_tol=1e-13), operator=op, solver=solver)
        for k in range(300):
            ret = o.step(w.dt, w.I_ramp)
            assert ret >= 0
        outs.append((o.read(), o.stats, ret))
    (J, T, B, E), st, ret = outs[0]
    Jc = 2e9 * (1 - 4.2 / 18) ** 2
    assert 0.9 < np.max(np.abs(J)) / Jc < 1.1 and np.max(np.abs(E)) > 1e-6      # nonlinear regime reached
    assert abs(np.sum(J)) < 1e-6 * np.sum(np.abs(J))                          # zero net current in the wire
    for u, v in zip(outs[0][0], outs[1][0]):
        assert np.linalg.norm(u - v) <= 1e-8 * np.linalg.norm(u)
    # shielding: induced currents oppose the field rise (Lenz): outer edge (larger r) carries J < 0 for Bdot > 0
    J2 = J.reshape(12, 12)
    assert J2[-1].mean() < 0 < J2[0].mean()


def test_joule_heat_equals_enthalpy_rise_plus_boundary_flux():
    # north_star energy balance across whole steps: sum_k dt P_k = sum V (H_end - H_0) + boundary losses
    w = wl.shrunk(1, 1, 1, 8)
    geo = dataclasses.replace(w.geometry, Bext_rate=200.0, Bext_max=1e3)        # strong drive: real heating
    o = qo.Oracle(geo, w.material)
    vol = 2 * math.pi * geo.r * geo.h ** 2
    H0 = o.H.copy()
    joule = lost = 0.0
    for k in range(100):
        assert o.step(w.dt, 0.0) >= 0
        joule += w.dt * o.stats["joule_power"]
        lost += o.stats["boundary_energy"]
    rise = np.sum(vol * (o.H - H0))
    assert o.T.max() > geo.T_bath + 1e-3 and joule > 0
    assert abs(joule - rise - lost) < 1e-10 * joule


def test_event_variants():
    # a prepared hot turn sets FJ_T (12 K) or Q_T|Q_rho (19 K); first-event time, counters
    w = wl.config(0)
    geo = w.geometry
    o = qo.Oracle(geo, w.material)
    T = np.full(geo.n_rings, geo.T_bath)
    T[geo.turn_id == 5] = 12.0
    o.write(np.zeros(geo.n_rings), T, 0.0, 0.0)
    ret = o.step(w.dt, w.I_ramp)
    assert ret & qo.RET_FLUXJUMP and not ret & qo.RET_QUENCH
    assert o.flags[5] & qo.FJ_T and o.count[5] == 1 and abs(o.t_first[5] - w.dt) < 1e-18
    assert np.all(np.delete(o.flags, 5) == 0) and np.all(np.delete(o.t_first, 5) < 0)
    ret = o.step(w.dt, w.I_ramp)
    assert not ret & qo.RET_FLUXJUMP and o.count[5] == 1                     # no new rising edge
    T[geo.turn_id == 5] = 19.0
    o.write(np.zeros(geo.n_rings), T, 0.0, 0.0)
    ret = o.step(1e-6, w.I_ramp)
    assert ret & qo.RET_QUENCH and o.flags[5] & qo.Q_T and o.flags[5] & qo.Q_RHO and o.flags[5] & qo.FJ_T
    assert np.all(np.delete(o.flags, 5) & (qo.Q_T | qo.Q_RHO) == 0)


def test_flux_jump_criterion_J_over_Jc():
    # PAPER.md:105 flux-jump criterion |J/Jc| > 1 (bit FJ_J).  Prepared state at B = 0 (B0 -> inf), no strain term,
    # no Jc0 perturbation: Jc = Jc0 (1 - T/Tc)^2 in closed form.  One cell of turn 7 at 1.01 Jc, one cell of turn 9 at
    # 0.99 Jc, the rest at 0.5 Jc -> exactly turn 7 raises exactly FJ_J; first-event time = end of that step; return bit 0.
    w = wl.config(0)
    geo = w.geometry
    mat = dataclasses.replace(w.material, B0=1e30, eps_coef=0.0, jc0_scale=None)
    Jc = mat.Jc0 * (1.0 - geo.T_bath / mat.Tc) ** 2
    J = np.full(geo.n_rings, 0.5 * Jc)
    c7 = np.flatnonzero(geo.turn_id == 7)[13]
    c9 = np.flatnonzero(geo.turn_id == 9)[40]
    J[c7], J[c9] = 1.01 * Jc, 0.99 * Jc
    o = qo.Oracle(geo, mat)
    o.write(J, np.full(geo.n_rings, geo.T_bath), 0.0, 0.0)
    ret = o.step(1e-7, 0.0)
    assert ret == qo.RET_FLUXJUMP
    assert o.flags[7] == qo.FJ_J and np.all(np.delete(o.flags, 7) == 0)
    assert abs(o.t_first[7] - 1e-7) < 1e-20 and np.all(np.delete(o.t_first, 7) < 0)
    assert np.all(o.count == 0)                              # the rising-edge counter follows FJ_T | FJ_E only (C10)
    # negative current counts through its magnitude
    J[c7], J[c9] = -0.99 * Jc, -1.01 * Jc
    o.write(J, np.full(geo.n_rings, geo.T_bath), 0.0, 0.0)
    assert o.step(1e-7, 0.0) == qo.RET_FLUXJUMP
    assert o.flags[9] == qo.FJ_J and np.all(np.delete(o.flags, 9) == 0)


@pytest.mark.parametrize("side", [-1, +1])
def test_flux_jump_criterion_dEdt_spike(side):
    # C10 bit FJ_E: (Ebar^k - Ebar^{k-1})/dt > dEdt_spike, Ebar = mean |E| over the turn.  Turn 5 is normal (T > Tc:
    # rho = rho_n exactly) and carries positive J everywhere, so Ebar = rho_n mean(J) = rho_n I(t)/A_wire by the turn's
    # current constraint: dEbar/dt = rho_n I_ramp / A_wire in closed form, whatever the redistribution inside the turn.
    # The threshold is placed 1e-6 relative below / above it.  T_fluxjump is raised so that FJ_T stays off and the
    # rising-edge counter isolates FJ_E.
    w = wl.config(0)
    geo = w.geometry
    I_ramp, dt = 4000.0, 1e-6
    A_wire = geo.wire_size ** 2
    rate = w.material.rho_n * I_ramp / A_wire                # 2 V/m/s
    mat = dataclasses.replace(w.material, T_fluxjump=100.0, dEdt_spike=rate * (1.0 - side * 1e-6))
    J0 = np.full(geo.n_rings, 0.5 * 2e9 * (1 - 4.2 / 18) ** 2)
    T0 = np.full(geo.n_rings, geo.T_bath)
    T0[geo.turn_id == 5] = 19.0
    o = qo.Oracle(geo, mat)
    o.write(J0, T0, 0.0, J0[0] * A_wire)
    ret1 = o.step(dt, I_ramp)
    assert not o.flags[5] & qo.FJ_E and o.count[5] == 0      # no previous Ebar on the first step after qs_write
    assert ret1 & qo.RET_QUENCH and o.flags[5] & qo.FJ_J     # normal turn: Jc = 0, |J|/Jc = inf > 1 (C5 guard, C10)
    assert np.all(o.J[geo.turn_id == 5] > 0)
    ret2 = o.step(dt, I_ramp)
    fired = bool(o.flags[5] & qo.FJ_E)
    assert fired == (side > 0)
    assert o.count[5] == (1 if fired else 0)
    assert not ret2 & qo.RET_FLUXJUMP                        # return bit 0 = a flux jump STARTED: FJ_J was already set
    assert np.all(np.delete(o.flags, 5) & qo.FJ_E == 0)      # cold turns: E ~ Ec 0.5^20, no spike
    ret3 = o.step(dt, I_ramp)                                # the flag stays set at the same rate: no second rising edge
    assert bool(o.flags[5] & qo.FJ_E) == fired and o.count[5] == (1 if fired else 0)
    assert not ret3 & qo.RET_FLUXJUMP


def test_wire_statistics_closed_forms_and_energy_identity():
    # f3 per-wire accumulators: a prepared normal-state turn carrying J0 dissipates exactly
    # rho_n J0^2 per volume, so E_joule, P_q, Q_q of that turn have closed forms after one step; the sum of E_joule
    # over all turns equals the time integral of the step's Joule power (an independent accumulation)
    w = wl.config(0)
    geo, mat = w.geometry, w.material
    N = geo.n_rings
    J0 = np.full(N, 0.5 * 2e9 * (1 - 4.2 / 18) ** 2)
    T0 = np.full(N, geo.T_bath)
    hot = geo.turn_id == 5
    T0[hot] = 19.0                                               # above Tc: rho = rho_n exactly (C5 guard)
    o = qo.Oracle(geo, mat)
    o.write(J0, T0, 0.0, 0.0)
    dt = 1e-6
    total = 0.0
    o.step(dt, 0.0)
    total += dt * o.stats["joule_power"]
    V5 = np.sum(2 * math.pi * geo.r[hot] * geo.area[hot])
    P = mat.rho_n * J0[0] ** 2
    wr = o.wire
    assert abs(wr["E_joule"][5] - dt * P * V5) <= 1e-12 * dt * P * V5
    assert abs(wr["P_q"][5] - P) <= 1e-12 * P and abs(wr["P_max"][5] - P) <= 1e-12 * P
    assert abs(wr["t_q"][5] - dt) < 1e-20 and wr["T_q"][5] > mat.Tc
    assert abs(wr["Q_q"][5] - wr["E_joule"][5]) <= 1e-15 * wr["E_joule"][5]     # first event and quench in the same step
    assert abs(wr["Q_FJ"][5] - wr["E_joule"][5]) <= 1e-15 * wr["E_joule"][5]
    cold = np.delete(np.arange(geo.n_turns), 5)
    assert np.all(wr["t_q"][cold] < 0) and np.all(wr["Q_q"][cold] == 0)
    for _ in range(5):
        o.step(dt, 0.0)
        total += dt * o.stats["joule_power"]
    assert abs(wr["E_joule"].sum() - total) <= 1e-12 * total
    assert np.all(wr["Q_FJ"] <= wr["E_joule"] * (1 + 1e-15)) and np.all(wr["T_max"] >= geo.T_bath)
    assert abs(wr["Q_q"][5] - dt * P * V5) <= 1e-12 * dt * P * V5               # frozen at the quench time
    o.write(J0, T0, 0.0, 0.0)
    assert np.all(o.wire["E_joule"] == 0) and np.all(o.wire["t_q"] == -1.0)


def _lr_ring():
    base = wl.lattice_geometry(1, 1, 1, 1e-3, 30e-3, h_conv=0.0, Bext_rate=10.0, Bext_max=100.0)
    geo = dataclasses.replace(base, n_turns=0, turn_id=None)
    mat = wl.Material()
    r, a = geo.r[0], geo.area[0]
    L = qo.mutual_pair(r, 0.0, r, 0.0, soft2=geo.softening ** 2)    # C2 self term (pinned against the thin-ring form)
    R = mat.rho_n * 2 * math.pi * r / a
    return geo, mat, a, float(L) / R, -math.pi * r * r * 10.0 / R


def test_heun_euler_step_is_second_order_on_the_LR_circuit():
    # f2 (PAPER.md:73 Runge-Kutta with variable step): on the linear L-R ring the Heun result is the exact
    # second-order Taylor polynomial, I_{k+1} = I_k + (I_inf - I_k)(x - x^2/2), x = dt/tau, and the embedded error
    # estimate is |I_inf - I_k| x^2 / 2 in current
    geo, mat, a, tau, I_inf = _lr_ring()
    o = qo.Oracle(geo, mat)
    o.write(np.zeros(1), np.full(1, 20.0), 0.0, 0.0)
    dt = 0.05 * tau
    ret, taken, nxt, err = o.step_rk(dt, 0.0, rtol=1.0, dt_min=1e-12)
    x = dt / tau
    assert taken == dt and abs(o.J[0] * a - I_inf * (x - x * x / 2)) <= 1e-12 * abs(I_inf)
    Jref = mat.Jc0 * (1 - geo.T_bath / mat.Tc) ** 2
    assert abs(err - abs(I_inf) * x * x / 2 / a / Jref) <= 1e-10 * err
    errs = []
    for steps in (100, 200):                                    # global error ~ dt^2
        o = qo.Oracle(geo, mat)
        o.write(np.zeros(1), np.full(1, 20.0), 0.0, 0.0)
        for _ in range(steps):
            o.step_rk(2.0 * tau / steps, 0.0, rtol=1.0, dt_min=1e-12)
        exact = I_inf * (1 - math.exp(-o.t / tau))
        errs.append(abs(o.J[0] * a - exact) / abs(exact))
    assert errs[1] < 1e-4 and 3.6 < errs[0] / errs[1] < 4.4


def test_heun_euler_step_control_rejects_and_rescales():
    geo, mat, a, tau, I_inf = _lr_ring()
    Jref = mat.Jc0 * (1 - geo.T_bath / mat.Tc) ** 2
    o = qo.Oracle(geo, mat)
    o.write(np.zeros(1), np.full(1, 20.0), 0.0, 0.0)
    rtol = abs(I_inf) * 0.01 ** 2 / 2 / a / Jref              # the error of a step of 0.01 tau
    ret, taken, nxt, err = o.step_rk(0.5 * tau, 0.0, rtol=rtol, dt_min=1e-3 * tau)
    assert taken < 0.5 * tau and err <= rtol and taken <= 0.0101 * tau      # rejected down to the tolerance
    assert abs(nxt / taken - min(2.0, max(0.2, 0.9 * math.sqrt(rtol / err)))) < 1e-12
    o2 = qo.Oracle(geo, mat)
    o2.write(np.zeros(1), np.full(1, 20.0), 0.0, 0.0)
    ret, taken2, _, err2 = o2.step_rk(0.5 * tau, 0.0, rtol=rtol, dt_min=0.2 * tau)
    assert taken2 == 0.2 * tau and err2 > rtol                # accepted at dt_min regardless


def test_heun_euler_equals_explicit_euler_when_the_rate_is_constant():
    # linear regime (E ~ 0): I' is the same at both stages, the error estimate vanishes, and the step equals the
    # theta = 0 step of C7
    w = wl.shrunk(0, 2, 2, 4)
    mat0 = dataclasses.replace(w.material, theta=0.0)
    a_, b_ = qo.Oracle(w.geometry, mat0), qo.Oracle(w.geometry, mat0)
    for _ in range(5):
        a_.step(w.dt, w.I_ramp)
        ret, taken, nxt, err = b_.step_rk(w.dt, w.I_ramp, rtol=1e-6, dt_min=1e-9)
        assert taken == w.dt and err <= 1e-12 and nxt == 2 * w.dt
    assert np.max(np.abs(a_.J - b_.J)) <= 1e-12 * np.max(np.abs(a_.J))
    assert abs(a_.stats["U_terminal"] - b_.stats["U_terminal"]) <= 1e-9 * abs(a_.stats["U_terminal"])


def saturated_state(geo, mat, scale, Bdot):
    """Stationary state of the nonlinear problem under a steady field ramp, written out from Faraday's law.

    Once the flux front has crossed the wire and dI/dt = 0, C4 reads 2 pi r E = -pi r^2 Bdot - V_w on every ring of
    turn w (no inductive term left), the power law inverted gives J = Jc sgn(E) (|E|/Ec)^(1/n), and V_w is the root
    of the turn's net-current condition sum a J = 0 (I = 0 throughout).  Constant Jc (no field, temperature or strain
    dependence) and rho_n -> infinity make this exact.  Returns J, E and the turn voltages U_w = -V_w.
    """
    from scipy.optimize import brentq
    r, a = geo.r, geo.area
    Jc = mat.Jc0 * scale
    J, E, U = np.zeros_like(r), np.zeros_like(r), np.zeros(geo.n_turns)
    for w in range(geo.n_turns):
        m = geo.turn_id == w

        def state(V):
            e = -0.5 * r[m] * Bdot - V / (2 * math.pi * r[m])
            return Jc[m] * np.sign(e) * (np.abs(e) / mat.Ec) ** (1.0 / mat.n_exp), e

        lo, hi = sorted((-math.pi * r[m].max() ** 2 * Bdot, -math.pi * r[m].min() ** 2 * Bdot))
        V = brentq(lambda v: float(np.sum(a[m] * state(v)[0])), lo, hi, xtol=1e-300, rtol=1e-15)
        J[m], E[m] = state(V)
        U[w] = -V
    return J, E, U


def saturation_workload(layers=1, turns=2, n=6, Bdot=10.0):
    # weak pinning (Jc0 = 1e8 A/m^2: full penetration at mu0 Jc s/2 = 0.06 T) and a constant Jc per cell
    return wl.lattice_workload("saturation", layers, turns, n, 1e-3, 30e-3, 5e-5, 0.0, 400, 7, 0.01,
                               Bext_rate=Bdot, Bext_max=1e9, Jc0=1e8, B0=1e30, Tc=1e30, eps_coef=0.0, rho_n=1e6)


def test_nonlinear_trajectory_ends_in_the_closed_form_saturated_state():
    # pins the nonlinear step as a whole (sign and factor of the rhs, A_ext term, power law, per-turn constraint,
    # sign of the turn voltage): a dropped 1/2, a wrong sign or a transposed index moves the fixed point
    w = saturation_workload()
    geo, mat = w.geometry, w.material
    for op, solver in [("dense", "cholesky"), ("tables", "pcg")]:
        o = qo.Oracle(geo, dataclasses.replace(mat, cg_tol=1e-13), operator=op, solver=solver)
        Js, Es, Us = saturated_state(geo, mat, o.scale, geo.Bext_rate)
        errs = []
        for k in range(w.steps):
            assert o.step(w.dt, 0.0) >= 0
            errs.append(np.linalg.norm(o.J - Js) / np.linalg.norm(Js))
        assert errs[49] > 1e-2 > errs[149]                        # the front is still moving early on
        assert errs[-1] < 1e-11, errs[-1]
        assert np.linalg.norm(o.E - Es) < 1e-10 * np.linalg.norm(Es)
        assert abs(o.stats["U_terminal"] - Us.sum()) < 1e-10 * abs(Us.sum())
        cur = np.bincount(geo.turn_id, weights=geo.area * o.J)
        assert np.max(np.abs(cur)) < 1e-12 * np.sum(np.abs(geo.area * o.J))
        # the saturated wire is the Bean profile lifted by the power law: |J|/Jc = (|E|/Ec)^(1/n), |E| <~ s Bdot / 2
        x = np.abs(o.J) / (mat.Jc0 * o.scale)
        assert 0.5 < x.min() and x.max() < (0.5 * geo.wire_size * geo.Bext_rate / mat.Ec) ** (1 / mat.n_exp) * 1.01


def power_balance_residual(step, read_JE, apply_M, geo, Bdot, dt, steps):
    """Poynting balance of a magnetisation run (no transport current), accumulated over the trajectory.

    C4 multiplied by the ring currents: I.M.dI/dt + sum 2 pi r E I = sum I emf_ext - (C^T I).V, with emf_ext =
    -pi r^2 Bdot and C^T I = 0 (zero net current per turn).  Time-integrated: magnetic energy + Joule heat = work of
    the external field.  The theta step satisfies this to O(dt): the relative residual is returned.
    """
    r, a = geo.r, geo.area
    joule = work = 0.0
    J = np.zeros(geo.n_rings)
    for _ in range(steps):
        I = a * J
        assert step(dt) >= 0
        J, E = read_JE()                                           # E is the field of the step's start state (C6)
        joule += dt * np.sum(2 * math.pi * r * E * I)
        work += dt * np.sum(I * (-math.pi * r * r * Bdot))
    I = a * J
    return (0.5 * I @ apply_M(I) + joule - work) / work, joule / work


def test_nonlinear_transient_satisfies_the_power_balance_to_first_order():
    # pins the TRANSIENT (moving flux front, before saturation): a wrong factor or sign in the rhs, the update or the
    # constraint leaves an O(1) residual; the correct scheme's residual halves with dt
    w = wl.shrunk(1, 1, 1, 8)
    geo = dataclasses.replace(w.geometry, Bext_rate=10.0)
    res = []
    for dt in (1e-4, 5e-5, 2.5e-5):
        o = qo.Oracle(geo, w.material)
        rr, share = power_balance_residual(lambda d: o.step(d, 0.0), lambda: (o.J.copy(), o.E.copy()),
                                           lambda x: o.M @ x, geo, 10.0, dt, int(round(0.02 / dt)))
        res.append(rr)
        assert 0.2 < share < 0.4                                  # a quarter of the work is dissipated: nonlinear regime
    assert 0 < res[0] < 0.01
    assert 1.8 < res[0] / res[1] < 2.2 and 1.8 < res[1] / res[2] < 2.2

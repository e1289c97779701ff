"""Pins of the oracle's constraint groups with transport-current shares (reading C16; SURVEY.md §8(f) f3,
PAPER.md:61-67 sub-elements).  CPU only."""
import dataclasses

import numpy as np
import scipy.linalg

import workloads as wl
from oracle import qs_oracle as qo


def sub_workload(share="outer", bext_rate=0.0, per_side=3):
    w = wl.shrunk(0, 2, 2, 6)                              # 2 x 2 wires of 6 x 6 cells
    geo = wl.subelements(w.geometry, per_side, share)      # 9 sub-elements of 2 x 2 cells per wire
    geo = dataclasses.replace(geo, Bext0=0.0, Bext_rate=bext_rate, Bext_max=5.0)
    return dataclasses.replace(w, geometry=geo)


def test_subelement_groups_partition_the_wires():
    w = sub_workload()
    geo = w.geometry
    assert geo.n_turns == 4 * 9 and geo.turn_id.shape == (144,)
    assert np.all(np.bincount(geo.turn_id, minlength=36) == 4)
    wire = geo.turn_id // 9
    ir, iz = np.divmod(np.arange(144), geo.Nz)
    assert np.all(wire == (ir // 6) * 2 + iz // 6)
    per_wire = geo.turn_share.reshape(4, 9)
    assert np.allclose(per_wire.sum(axis=1), 1.0) and np.all(per_wire[:, 4] == 0.0) and np.all(per_wire[:, 0] == 0.125)
    # a sub-element is a contiguous 2 x 2 block of the lattice
    for g in range(36):
        c = np.flatnonzero(geo.turn_id == g)
        assert ir[c].max() - ir[c].min() == 1 and iz[c].max() - iz[c].min() == 1


def test_null_space_solve_equals_the_kkt_solve_with_shares():
    """Route independent of kkt_dense (Schur complement): x = x_p + Z y with Z a basis of ker C^T."""
    w = sub_workload()
    geo = w.geometry
    g = np.random.default_rng(5)
    A = qo.dense_M(geo) + np.diag(g.random(144) * 1e-8)
    C = qo.constraint_matrix(geo)
    b = g.standard_normal(144) * 1e-6
    d = 37.0 * geo.turn_share
    x, V = qo.kkt_dense(A, C, b, d)
    Z = scipy.linalg.null_space(C.T)
    assert Z.shape == (144, 144 - 36)
    xp = C @ np.linalg.solve(C.T @ C, d)
    y = np.linalg.solve(Z.T @ A @ Z, Z.T @ (b - A @ xp))
    xn = xp + Z @ y
    Vn = np.linalg.solve(C.T @ C, C.T @ (b - A @ xn))
    assert np.max(np.abs(x - xn)) < 1e-9 * np.max(np.abs(x))
    assert np.max(np.abs(V - Vn)) < 1e-8 * np.max(np.abs(V))
    assert np.max(np.abs(np.bincount(geo.turn_id, weights=x) - d)) < 1e-10 * 37.0
    # the projected CG takes the same right-hand side of the constraint
    xc, Vc, it, _ = qo.pcg(lambda v: A @ v, np.diag(A).copy(), geo.turn_id, geo.n_turns, b, d, 1e-13, 2000)
    assert it > 0 and np.max(np.abs(xc - xn)) < 1e-9 * np.max(np.abs(xn))
    assert np.max(np.abs(Vc - Vn)) < 1e-7 * np.max(np.abs(Vn))


def test_group_currents_follow_the_shares_along_a_trajectory():
    w = sub_workload("outer", bext_rate=0.5)
    geo = w.geometry
    o = qo.Oracle(geo, w.material)
    for _ in range(6):
        assert o.step(w.dt, w.I_ramp) >= 0
        cur = np.bincount(geo.turn_id, weights=o.J * geo.area)
        assert np.max(np.abs(cur - geo.turn_share * o.I)) < 1e-10 * o.I
    inner = geo.turn_share == 0.0
    assert inner.sum() == 4
    # zero net current, but the field ramp drives a circulating current inside the inner sub-elements
    Jin = o.J[np.isin(geo.turn_id, np.flatnonzero(inner))]
    assert Jin.max() > 0.0 > Jin.min() and np.abs(Jin).max() > 1e-3 * np.abs(o.J).max()
    # per wire the transport current is whole
    wire_cur = np.bincount(geo.turn_id // 9, weights=o.J * geo.area)
    assert np.max(np.abs(wire_cur - o.I)) < 1e-10 * o.I


def test_uncoupled_subelements_under_a_field_ramp():
    """PAPER.md:61 "net current of each subelement is zero (so-called uncoupled subelements)": with per-wire groups the
    screening current crosses the sub-element borders, with sub-element groups it closes inside each of them."""
    ws = sub_workload("uniform", bext_rate=1.0)
    wc = wl.shrunk(0, 2, 2, 6)
    wc = dataclasses.replace(wc, geometry=dataclasses.replace(wc.geometry, Bext0=0.0, Bext_rate=1.0, Bext_max=5.0))
    os_, oc = qo.Oracle(ws.geometry, ws.material), qo.Oracle(wc.geometry, wc.material)
    for _ in range(4):
        assert os_.step(ws.dt, 0.0) >= 0 and oc.step(wc.dt, 0.0) >= 0
    a = ws.geometry.area
    scale = np.abs(oc.J * a).sum() / 36
    sub_s = np.bincount(ws.geometry.turn_id, weights=os_.J * a)
    sub_c = np.bincount(ws.geometry.turn_id, weights=oc.J * a)          # same groups, coupled solution
    assert np.max(np.abs(sub_s)) < 1e-10 * scale
    assert np.max(np.abs(sub_c)) > 0.05 * scale
    assert np.max(np.abs(np.bincount(wc.geometry.turn_id, weights=oc.J * a))) < 1e-10 * scale
    # the uncoupled pack screens less: smaller magnetic moment
    m_s, m_c = np.sum(os_.J * a * ws.geometry.r ** 2), np.sum(oc.J * a * wc.geometry.r ** 2)
    assert abs(m_s) < abs(m_c)


def test_terminal_voltage_is_the_power_delivered_over_the_current():
    """U I = sum_w (-V_w) share_w I = d/dt (I^T M I / 2) in the linear regime (E ~ 0), i.e. U = I'^T M I' / I_ramp."""
    for share in ("uniform", "outer"):
        w = sub_workload(share)
        o = qo.Oracle(w.geometry, w.material)
        for _ in range(3):
            assert o.step(w.dt, w.I_ramp) == 0
        U = o.stats["U_terminal"]
        assert U > 0 and abs(U - o.Idot @ o.M @ o.Idot / w.I_ramp) < 1e-9 * U
    # Thomson's principle: the per-wire solution minimises I'^T M I' over C_wire^T I' = I_ramp, and every sub-element
    # distribution is admissible for it, so finer groups can only raise the inductive voltage
    wc = wl.shrunk(0, 2, 2, 6)
    oc = qo.Oracle(wc.geometry, wc.material)
    oc.step(wc.dt, wc.I_ramp)
    for share in ("uniform", "outer"):
        w = sub_workload(share)
        o = qo.Oracle(w.geometry, w.material)
        o.step(w.dt, w.I_ramp)
        assert o.stats["U_terminal"] > oc.stats["U_terminal"] * (1 + 1e-6)


def test_unit_shares_reproduce_the_per_turn_results():
    w = wl.shrunk(0, 2, 2, 4)
    g1 = dataclasses.replace(w.geometry, turn_share=np.ones(w.geometry.n_turns))
    o0, o1 = qo.Oracle(w.geometry, w.material), qo.Oracle(g1, w.material)
    for _ in range(3):
        assert o0.step(w.dt, w.I_ramp) == o1.step(w.dt, w.I_ramp)
    assert np.array_equal(o0.J, o1.J) and np.array_equal(o0.T, o1.T)
    assert o0.stats["U_terminal"] == o1.stats["U_terminal"]
    # the embedded pair takes the same shares
    ws = sub_workload("outer")
    o = qo.Oracle(ws.geometry, ws.material)
    res = o.step_rk(ws.dt, ws.I_ramp, 1e-3, 1e-9)
    cur = np.bincount(ws.geometry.turn_id, weights=o.J * ws.geometry.area)
    assert np.max(np.abs(cur - ws.geometry.turn_share * o.I)) < 1e-10 * o.I and res is not None

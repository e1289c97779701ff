"""GPU parity of constraint groups with transport-current shares (reading C16)
against the CPU oracle, through the C ABI (qs_geometry.turn_share)."""
import dataclasses

import numpy as np
import pytest

import workloads as wl
from oracle import qs_oracle as qo

pytestmark = pytest.mark.gpu
TOL = 1e-6


@pytest.fixture(scope="module")
def pkg():
    import paper_2403_07666_b200 as p
    return p


def sub_workload(layers, turns, n, per_side, share, bext_rate):
    w = wl.shrunk(0, layers, turns, n)
    geo = wl.subelements(w.geometry, per_side, share)
    geo = dataclasses.replace(geo, Bext0=0.0, Bext_rate=bext_rate, Bext_max=5.0)
    return dataclasses.replace(w, geometry=geo, material=dataclasses.replace(w.material, cg_tol=1e-12))


def check(ref, got, tol=TOL):
    for name, a, b in zip(("J", "T", "B", "E"), got, ref):
        floor = 1e-30 if name == "E" else 0.0
        assert np.linalg.norm(a - b) <= tol * np.linalg.norm(b) + floor, name


@pytest.mark.parametrize("share,lattice_tables", [("outer", False), ("uniform", False), ("outer", True)])
def test_subelement_groups_50_steps(pkg, share, lattice_tables):
    # 2 x 3 wires of 6 x 6 cells, 9 sub-elements each (54 groups of 4 cells; a warp spans several groups and wires)
    w = sub_workload(2, 3, 6, 3, share, 0.5)
    geo = w.geometry
    orc = qo.Oracle(geo, w.material)
    sim = pkg.QS(geo, w.material, lattice_tables=lattice_tables)
    for _ in range(50):
        ro, rg = orc.step(w.dt, w.I_ramp), sim.step(w.dt, w.I_ramp)
        assert ro == (rg & 3)
    got = sim.read()
    check(orc.read(), got)
    st = sim.stats()
    assert abs(st["U_terminal"] - orc.stats["U_terminal"]) <= 1e-8 * abs(orc.stats["U_terminal"])
    cur = np.bincount(geo.turn_id, weights=got[0] * geo.area)
    assert np.max(np.abs(cur - geo.turn_share * st["I"])) <= 1e-10 * st["I"]
    if share == "outer":
        inner = np.isin(geo.turn_id, np.flatnonzero(geo.turn_share == 0.0))
        assert np.abs(got[0][inner]).max() > 1e-3 * np.abs(got[0]).max()       # circulating, zero net
    # per-group statistics and event words follow the groups
    fl_g, tf_g, cn_g = sim.events()
    assert fl_g.shape == (geo.n_turns,) and np.array_equal(orc.flags, fl_g) and np.array_equal(orc.count, cn_g)
    sim.close()


def test_uncoupled_subelements_field_ramp_only(pkg):
    # no transport current: every sub-element keeps zero net current under the background-field ramp
    w = sub_workload(1, 2, 8, 2, "uniform", 2.0)
    geo = w.geometry
    orc, sim = qo.Oracle(geo, w.material), pkg.QS(geo, w.material)
    for _ in range(30):
        assert orc.step(w.dt, 0.0) == (sim.step(w.dt, 0.0) & 3)
    got = sim.read()
    check(orc.read(), got)
    cur = np.bincount(geo.turn_id, weights=got[0] * geo.area)
    assert np.max(np.abs(cur)) <= 1e-10 * np.abs(got[0] * geo.area).sum()
    sim.close()


def test_embedded_pair_with_shares(pkg):
    w = sub_workload(2, 2, 6, 3, "outer", 0.5)
    geo = w.geometry
    orc, sim = qo.Oracle(geo, w.material), pkg.QS(geo, w.material)
    dt = w.dt
    for _ in range(10):
        ro = orc.step_rk(dt, w.I_ramp, 1e-3, 1e-9)
        rg = sim.step_rk(dt, w.I_ramp, 1e-3, 1e-9)
        assert abs(ro[1] - rg[1]) <= 1e-12 * ro[1]
        dt = ro[2]
    check(orc.read(), sim.read())
    assert abs(sim.stats()["U_terminal"] - orc.stats["U_terminal"]) <= 1e-8 * abs(orc.stats["U_terminal"])
    sim.close()


def test_unit_shares_and_bad_shares(pkg):
    w = wl.shrunk(0, 2, 2, 4)
    g1 = dataclasses.replace(w.geometry, turn_share=np.ones(w.geometry.n_turns))
    a, b = pkg.QS(w.geometry, w.material), pkg.QS(g1, w.material)
    for _ in range(3):
        assert a.step(w.dt, w.I_ramp) == b.step(w.dt, w.I_ramp)
    for x, y in zip(a.read(), b.read()):
        assert np.array_equal(x, y)
    a.close()
    b.close()
    bad = dataclasses.replace(w.geometry, turn_share=np.full(w.geometry.n_turns, np.nan))
    with pytest.raises(Exception):
        pkg.QS(bad, w.material)

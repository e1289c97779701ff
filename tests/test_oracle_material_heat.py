"""Pins of the oracle's pointwise material law and heat step (C9)."""
import dataclasses
import math

import numpy as np

import workloads as wl
from oracle import qs_oracle as qo


def law(mat, J, T=4.2, Br=0.0, Bz=0.0, r=0.03, s=1.0):
    a = lambda v: np.atleast_1d(np.asarray(v, dtype=np.float64))
    return qo.material_law(mat, a(J), a(T), a(Br), a(Bz), a(r), a(s))


def test_critical_current_closed_forms():
    mat = wl.Material()
    out = law(mat, 1.0)
    assert abs(out["Jc"][0] - 2e9 * (1 - 4.2 / 18) ** 2) < 1e-6          # Jc(4.2 K, 0, 0) = 1.175556e9
    assert abs(out["Jc"][0] - 1.1755555555555556e9) < 1e-3
    assert abs(law(mat, 1.0, Bz=1.0)["Jc"][0] / out["Jc"][0] - 0.5) < 1e-15   # 1/(1+|B|/1 T)
    assert abs(law(mat, 1.0, Br=0.6, Bz=0.8)["Jc"][0] / out["Jc"][0] - 0.5) < 1e-15
    assert law(mat, 1.0, T=18.0)["Jc"][0] == 0.0 and law(mat, 1.0, T=25.0)["Jc"][0] == 0.0
    # strain factor vanishes at |eps| = 900^(-1/1.7) = 0.01829;  eps = J Bz r / Y
    eps0 = 900.0 ** (-1 / 1.7)
    assert abs(eps0 - 0.01829) < 1e-5
    J, Bz, r = 1e9, 3.0, 0.05
    Y = J * Bz * r / eps0
    m2 = dataclasses.replace(mat, Y=Y * (1 - 1e-9))
    assert law(m2, J, Bz=Bz, r=r)["Jc"][0] == 0.0
    m3 = dataclasses.replace(mat, Y=Y * 2 ** (1 / 1.7))                   # |eps| halves 900|eps|^1.7
    got = law(m3, J, Bz=Bz, r=r)["Jc"][0] * (1 + 3.0) / (2e9 * (1 - 4.2 / 18) ** 2)
    assert abs(got - 0.5) < 1e-12
    assert abs(law(m3, J, Bz=Bz, r=r)["eps"][0] - J * Bz * r / m3.Y) == 0.0


def test_power_law_closed_forms_without_cap():
    mat = wl.Material(rho_n=1e300)                                        # rho_n -> infinity: bare power law
    Jc = law(mat, 1.0)["Jc"][0]
    out = law(mat, Jc)
    assert abs(out["E"][0] - mat.Ec) < 1e-15 * mat.Ec * 64               # E(Jc) = Ec
    assert abs(out["dEdJ"][0] - mat.n_exp * mat.Ec / Jc) < 1e-13 * mat.n_exp * mat.Ec / Jc
    out = law(mat, -0.9 * Jc)
    assert abs(out["E"][0] + mat.Ec * 0.9 ** 20) < 1e-14 * mat.Ec       # odd in J
    assert abs(out["Q"][0] - mat.Ec * 0.9 ** 20 * 0.9 * Jc) < 1e-13 * mat.Ec * Jc
    s = law(mat, 1.0, s=1.01)["Jc"][0]
    assert abs(s / Jc - 1.01) < 1e-15                                     # per-cell Jc0 multiplier


def test_normal_state_cap_and_guards():
    mat = wl.Material()
    Jc = law(mat, 1.0)["Jc"][0]
    out = law(mat, [0.0, 1e3, Jc, 3 * Jc, 1e30 * Jc, Jc], T=[4.2, 4.2, 4.2, 4.2, 4.2, 19.0])
    assert out["rho"][0] == 0.0 and out["dEdJ"][0] == 0.0 and out["E"][0] == 0.0
    assert out["rho"][1] == 0.0 or out["rho"][1] < 1e-100                  # deep in the superconducting state
    rho_sc = mat.Ec / Jc
    assert abs(out["rho"][2] - rho_sc * mat.rho_n / (rho_sc + mat.rho_n)) < 1e-15 * rho_sc   # parallel cap
    assert 0.0 < out["rho"][3] < mat.rho_n and out["rho"][3] > 0.99 * mat.rho_n
    assert out["rho"][4] == mat.rho_n and out["dEdJ"][4] == mat.rho_n      # (J/Jc)^19 overflows: no inf/inf
    assert out["rho"][5] == mat.rho_n and out["dEdJ"][5] == mat.rho_n      # T > Tc: Jc = 0 -> normal
    assert np.all(np.isfinite(out["E"])) and np.all(out["Q"] >= 0.0)


def test_dEdJ_is_the_derivative_and_E_is_monotone():
    mat = wl.Material()
    Jc = law(mat, 1.0)["Jc"][0]
    J = np.linspace(0.5, 3.0, 101) * Jc
    out = law(mat, J, T=np.full_like(J, 4.2), Br=0 * J, Bz=0 * J, r=0 * J + 0.03, s=0 * J + 1)
    assert np.all(np.diff(out["E"]) > 0)
    e = 1e-6
    up = law(mat, J * (1 + e), T=np.full_like(J, 4.2), Br=0 * J, Bz=0 * J, r=0 * J + 0.03, s=0 * J + 1)["E"]
    dn = law(mat, J * (1 - e), T=np.full_like(J, 4.2), Br=0 * J, Bz=0 * J, r=0 * J + 0.03, s=0 * J + 1)["E"]
    fd = (up - dn) / (2 * e * J)
    assert np.max(np.abs(fd - out["dEdJ"]) / out["dEdJ"]) < 1e-8


def test_enthalpy_inverse_and_substep_counts():
    mat = wl.Material()
    T = np.array([4.2, 5.0, 10.0, 18.0, 40.0])
    H = qo.enthalpy(mat, T)
    assert abs(H[0] - (500 * 4.2 ** 4 + 250 * 4.2 ** 2)) < 1e-9          # H = int C dT, C = 2000 T^3 + 500 T
    assert np.max(np.abs(qo.temperature(mat, H) - T)) < 1e-13
    e = 1e-5
    C = (qo.enthalpy(mat, T + e) - qo.enthalpy(mat, T - e)) / (2 * e)
    assert np.max(np.abs(C - (2000 * T ** 3 + 500 * T)) / C) < 1e-8
    # m = 5, 144, 28, 16 heat sub-steps at configs 0..3
    for idx, m in [(0, 5), (1, 144), (2, 28), (3, 16)]:
        w = wl.config(idx) if idx < 2 else None
        if w is None:
            g = wl.Geometry(r=np.zeros(1), z=np.zeros(1), area=np.zeros(1), turn_id=None, n_turns=0, lattice=1,
                            layers=1, turns_per_layer=1, cells_per_side={2: 16, 3: 12}[idx], wire_size=0.8e-3)
            assert qo.heat_substeps_count(g, mat, 1e-4) == m
        else:
            assert qo.heat_substeps_count(w.geometry, w.material, w.dt) == m


def column(nz, h, hc):
    """One radial column of nz single-cell 'wires': a 1-D problem along z (r cancels)."""
    return wl.lattice_geometry(1, nz, 1, h, 0.03, h_conv=0.0)._replace_hconv((0.0, 0.0, hc, hc))


def _replace_hconv(self, hc):
    return dataclasses.replace(self, h_conv=hc)


wl.Geometry._replace_hconv = _replace_hconv


def test_exact_discrete_steady_state_1d():
    # SURVEY.md pins: T_j = sqrt(Ts^2 + (Q h^2/kappa) j (n-1-j)), Ts = T_bath + Q n h/(2 h_conv)
    n, h, Q, hc = 16, 1e-4, 2e5, 500.0
    geo = column(n, h, hc)
    mat = wl.Material(k_between=5.0)                                      # the quoted value is for kappa = 5
    Ts = geo.T_bath + Q * n * h / (2 * hc)
    j = np.arange(n)
    Tex = np.sqrt(Ts ** 2 + (Q * h * h / mat.k_between) * j * (n - 1 - j))
    assert abs(Ts - 4.52) < 1e-12 and abs(Tex[8] - 4.522477197289115) < 1e-12
    div, _ = qo.heat_flux_divergence(geo, mat, Tex.reshape(1, n))
    vol = 2 * math.pi * geo.r * h * h
    resid = div.reshape(-1) / vol + Q
    assert np.max(np.abs(resid)) < 1e-9 * Q                               # fixed point of the scheme
    # and the time stepping is attracted to it: a zero-mean ripple of 1 mK decays (rate alpha (4 pi/L)^2 ~ 8e3/s)
    ripple = 1e-3 * np.cos(4 * math.pi * (j + 0.5) / n)
    H = qo.enthalpy(mat, Tex + ripple)
    dt = 2e-3
    for _ in range(2):
        H, _ = qo.heat_substeps(geo, mat, H, np.full(n, Q), dt, qo.heat_substeps_count(geo, mat, dt))
    assert np.max(np.abs(qo.temperature(mat, H) - Tex)) < 1e-6


def test_radial_scheme_is_second_order_consistent():
    # continuous steady state with uniform Q and uniform kappa: T^2 = A + B ln r - Q r^2/(2 kappa)
    mat = wl.Material()
    Q, kap, A, B = 3e3, mat.k_between, 100.0, 20.0
    res = []
    for nr in (16, 32, 64):
        geo = dataclasses.replace(wl.lattice_geometry(nr, 1, 1, 1.6e-3 / nr, 0.03), h_conv=(0, 0, 0, 0))
        r = geo.r
        T = np.sqrt(A + B * np.log(r) - Q * r * r / (2 * kap))
        div, _ = qo.heat_flux_divergence(geo, mat, T.reshape(nr, 1))
        resid = div.reshape(-1) / (2 * math.pi * r * geo.h ** 2) + Q
        res.append(np.max(np.abs(resid[1:-1])))
    assert res[0] < 1e-4 * Q and 3.5 < res[0] / res[1] < 4.5 and 3.5 < res[1] / res[2] < 4.5


def test_robin_loss_on_the_radial_borders_uses_the_true_border_radii():
    # PAPER.md:75 "four borders": a one-cell-high stack of rings (Nz = 1) with uniform Q cooled through ONE radial
    # border only.  In the steady state all the heat leaves through that border, so the border cell's temperature has
    # a closed form with the TRUE border radius (not the cell-centre radius):
    #   h_conv (T_border - T_b) 2 pi r_border h = Q pi (r_out^2 - r_in^2) h
    # (the cell volumes 2 pi r_c h^2 sum to pi (r_out^2 - r_in^2) h exactly).  Strong curvature: r_in = 1 mm, h = 0.5 mm.
    import scipy.optimize
    nr, h, r_in, Q, hc = 4, 0.5e-3, 1.0e-3, 4e4, 500.0
    r_out = r_in + nr * h
    mat = wl.Material()
    for side, r_border, cell in ((0, r_in, 0), (1, r_out, nr - 1)):
        hcv = [0.0, 0.0, 0.0, 0.0]
        hcv[side] = hc
        geo = dataclasses.replace(wl.lattice_geometry(nr, 1, 1, h, r_in), h_conv=tuple(hcv))
        assert geo.Nz == 1 and geo.Nr == nr
        vol = 2 * math.pi * geo.r * h * h
        assert abs(vol.sum() - math.pi * (r_out ** 2 - r_in ** 2) * h) < 1e-15 * vol.sum()

        def resid(T):
            div, _ = qo.heat_flux_divergence(geo, mat, T.reshape(nr, 1))
            return div.reshape(-1) / vol + Q

        T = scipy.optimize.fsolve(resid, np.full(nr, geo.T_bath + 1.0), xtol=1e-13)
        assert np.max(np.abs(resid(T))) < 1e-9 * Q
        T_closed = geo.T_bath + Q * (r_out ** 2 - r_in ** 2) / (2.0 * r_border * hc)
        assert abs(T[cell] - T_closed) < 1e-9 * T_closed, (side, T[cell], T_closed)
        # the cell-centre radius in place of the border radius would be off by h/(2 r_border): 25 % / 8 % here
        r_c = geo.r[cell]
        assert abs(geo.T_bath + Q * (r_out ** 2 - r_in ** 2) / (2.0 * r_c * hc) - T_closed) > 1e-2 * (T_closed - geo.T_bath)
        # and the time stepping relaxes to that state (enthalpy form, sub-step rule of C9)
        # (a ripple that carries no net energy, so that only the fast conduction modes are excited)
        ripple = 1e-3 * np.cos(np.arange(nr))
        wgt = vol * (mat.C3 * T ** 3 + mat.C1 * T)
        ripple -= np.sum(wgt * ripple) / np.sum(wgt)
        H = qo.enthalpy(mat, T + ripple)
        dt = 5e-3
        for _ in range(60):                                   # 0.3 s = 9 conduction time constants (k_between, 2 mm)
            H, lost = qo.heat_substeps(geo, mat, H, np.full(nr, Q), dt, qo.heat_substeps_count(geo, mat, dt))
        assert abs(qo.temperature(mat, H)[cell] - T_closed) < 5e-5
    # both radial borders cooled: global balance with the two true border radii
    geo = dataclasses.replace(wl.lattice_geometry(nr, 1, 1, h, r_in), h_conv=(hc, 0.5 * hc, 0.0, 0.0))
    vol = 2 * math.pi * geo.r * h * h

    def resid2(T):
        div, _ = qo.heat_flux_divergence(geo, mat, T.reshape(nr, 1))
        return div.reshape(-1) / vol + Q

    T = scipy.optimize.fsolve(resid2, np.full(nr, geo.T_bath + 1.0), xtol=1e-13)
    out = hc * (T[0] - geo.T_bath) * 2 * math.pi * r_in * h + 0.5 * hc * (T[-1] - geo.T_bath) * 2 * math.pi * r_out * h
    gen = Q * math.pi * (r_out ** 2 - r_in ** 2) * h
    assert abs(out - gen) < 1e-9 * gen


def test_energy_balance_to_rounding():
    # sum V dH = dt sum V Q - boundary energy (enthalpy form; north_star "energy balance")
    geo = wl.lattice_geometry(3, 2, 4, 1e-3, 0.03)
    mat = wl.Material()
    g = np.random.default_rng(5)
    T0 = 4.2 + 6 * g.random(geo.n_rings)
    Q = 1e6 * g.random(geo.n_rings)
    H0 = qo.enthalpy(mat, T0)
    dt = 1e-4
    m = qo.heat_substeps_count(geo, mat, dt)
    H1, lost = qo.heat_substeps(geo, mat, H0, Q, dt, m)
    vol = 2 * math.pi * geo.r * geo.h ** 2
    lhs = np.sum(vol * (H1 - H0))
    rhs = dt * np.sum(vol * Q) - lost
    assert lost > 0 and abs(lhs - rhs) < 1e-11 * abs(dt * np.sum(vol * Q))
    # conduction alone conserves energy; interfaces between wires conduct 10x less than inside a wire
    geo0 = dataclasses.replace(geo, h_conv=(0, 0, 0, 0))
    H2, lost0 = qo.heat_substeps(geo0, mat, H0, 0 * Q, dt, m)
    assert lost0 == 0.0 and abs(np.sum(vol * (H2 - H0))) < 1e-12 * np.sum(vol * H0)
    T = np.full((geo.Nr, geo.Nz), 5.0)
    T[:, 4:] = 6.0                                                       # step across a wire boundary (iz 3|4)
    d_between, _ = qo.heat_flux_divergence(geo0, mat, T)
    T = np.full((geo.Nr, geo.Nz), 5.0)
    T[:, 2:] = 6.0                                                       # same step inside a wire (iz 1|2)
    d_in, _ = qo.heat_flux_divergence(geo0, mat, T)
    assert abs(d_in[0, 1] / d_between[0, 3] - mat.k_in / mat.k_between) < 1e-12


def test_adi_line_operators_equal_the_explicit_flux_divergence():
    # f4: L_r U + L_z U - rb (T - T_b) is the explicit scheme's divergence per volume (C9), cell by cell
    geo = wl.lattice_geometry(3, 2, 5, 1e-3, 30e-3)
    geo = dataclasses.replace(geo, h_conv=(500.0, 300.0, 200.0, 100.0))
    mat = wl.Material()
    g = np.random.default_rng(2)
    T = g.uniform(4.2, 12.0, geo.n_rings)
    Lr, Lz, rb_r, rb_z = qo.heat_line_operators(geo, mat)
    div, _ = qo.heat_flux_divergence(geo, mat, T.reshape(geo.Nr, geo.Nz))
    vol = 2 * math.pi * geo.r * geo.h ** 2
    lhs = Lr @ (T * T) + Lz @ (T * T) - (rb_r + rb_z) * (T - geo.T_bath)
    assert np.max(np.abs(lhs - div.ravel() / vol)) <= 1e-12 * np.max(np.abs(lhs))


def test_adi_fixed_point_is_the_exact_discrete_steady_state():
    # the 1-D steady state that is exact for the scheme (C9 pin: T_j^2 = T_s^2 + (Q h^2/kappa) j (n-1-j),
    # T_s = T_bath + Q n h / (2 h_conv)) is also the fixed point of the ADI iteration (the linearised Robin term is exact
    # at the fixed point), reached with steps ~ 500 x the explicit stability limit
    n, h, Qv, hc = 16, 1e-4, 2e5, 500.0
    geo = wl.lattice_geometry(1, 1, n, n * h, 1.0)               # r >> size: planar limit
    geo = dataclasses.replace(geo, h_conv=(0.0, 0.0, hc, hc))
    mat = dataclasses.replace(wl.Material(), k_in=5.0, k_between=5.0)
    Q = np.full(geo.n_rings, Qv)
    H = qo.enthalpy(mat, np.full(geo.n_rings, 4.2))
    for _ in range(400):
        H = qo.heat_adi(geo, mat, H, Q, 0.02, 1)
    T = qo.temperature(mat, H).reshape(n, n)
    Ts = 4.2 + Qv * n * h / (2 * hc)
    j = np.arange(n)
    exact = np.sqrt(Ts ** 2 + Qv * h * h / 5.0 * j * (n - 1 - j))
    assert abs(exact[8] - 4.522477197289115) < 1e-12            # the value quoted in SURVEY.md §8(c) pins
    assert np.max(np.abs(T - exact[None, :])) <= 1e-8


def test_adi_converges_to_the_explicit_solution_at_second_order():
    geo = wl.lattice_geometry(2, 2, 6, 1e-3, 30e-3)
    geo = dataclasses.replace(geo, h_conv=(500.0, 300.0, 200.0, 100.0))
    mat = wl.Material()
    g = np.random.default_rng(4)
    T0 = g.uniform(4.2, 9.0, geo.n_rings)
    Q = g.uniform(0, 5e5, geo.n_rings)
    H0 = qo.enthalpy(mat, T0)
    dt = 2e-4
    c = qo.heat_substeps_count(geo, mat, dt)
    Ta = qo.temperature(mat, qo.heat_substeps(geo, mat, H0, Q, dt, 400 * c)[0])
    Tb = qo.temperature(mat, qo.heat_substeps(geo, mat, H0, Q, dt, 800 * c)[0])
    Tref = 2 * Tb - Ta                                           # Richardson: the explicit scheme is first order in time
    errs = [np.max(np.abs(qo.temperature(mat, qo.heat_adi(geo, mat, H0, Q, dt, m)) - Tref)) for m in (8, 16, 32)]
    assert errs[2] < 2e-4 and errs[0] / errs[1] > 3.5 and errs[1] / errs[2] > 3.5


def test_adi_conserves_energy_and_survives_steps_far_beyond_the_explicit_limit():
    # adiabatic pack: sum_c V_c dH_c = dt sum_c V_c Q_c to rounding at any step size (the half-steps are an energy
    # balance for H' dU and the enthalpy advances by exactly that); 30 x the explicit limit on rough data stays bounded
    geo = wl.lattice_geometry(2, 2, 8, 1e-3, 30e-3, h_conv=0.0)
    mat = wl.Material()
    g = np.random.default_rng(6)
    T0 = g.uniform(4.2, 14.0, geo.n_rings)
    Q = g.uniform(0, 5e5, geo.n_rings)
    lim = 0.8 * geo.h ** 2 / (4 * mat.k_in / (mat.C3 * 4.2 ** 2 + mat.C1))
    V = 2 * math.pi * geo.r * geo.h ** 2
    for f in (3, 30):
        H0 = qo.enthalpy(mat, T0)
        H = H0
        for _ in range(5):
            H = qo.heat_adi(geo, mat, H, Q, f * lim, 1)
        T = qo.temperature(mat, H)
        assert np.all(np.isfinite(T)) and 4.2 <= T.min() and T.max() <= 14.5
        gain = 5 * f * lim * np.sum(V * Q)
        assert abs(np.sum(V * (H - H0)) - gain) <= 1e-10 * gain

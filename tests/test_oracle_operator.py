"""Pins of the oracle's pair kernels (SURVEY.md §8(c) pins table) against things that are not the oracle:
numerical quadrature of the defining integrals (Neumann, Biot-Savart), textbook closed forms and limits."""
import math

import mpmath as mp
import numpy as np
import pytest

import workloads as wl
from oracle import qs_oracle as qo

MU0 = 4e-7 * math.pi


def neumann_mp(ri, zi, rj, zj):
    """M = mu0/(4 pi) oint oint dl.dl'/|x-x'| = mu0 ri rj int_0^pi cos(phi) / R(phi) dphi  (definition)."""
    mp.mp.dps = 30
    ri, rj, dz = mp.mpf(ri), mp.mpf(rj), mp.mpf(zi) - mp.mpf(zj)
    f = lambda p: mp.cos(p) / mp.sqrt(ri * ri + rj * rj + dz * dz - 2 * ri * rj * mp.cos(p))
    pts = [0, mp.mpf(10) ** -4, mp.mpf(10) ** -2, mp.mpf(1) / 2, mp.pi]
    return float(4 * mp.pi * mp.mpf(10) ** -7 * ri * rj * mp.quad(f, pts))


PAIRS = [  # (ri, zi, rj, zj) in metres; near, far and adjacent-cell cases of configs 0, 1, 4
    (0.030, 0.0, 0.040, 0.010),
    (0.030, 0.0, 0.030, 0.125e-3),
    (0.030, 0.0, 0.0300125, 0.0),
    (0.030, -0.100, 0.090, 0.100),
    (0.050, 0.0, 0.050, 0.015625e-3),
    (0.0437, 0.0123, 0.0561, -0.0031),
]


@pytest.mark.parametrize("pair", PAIRS)
def test_mutual_equals_neumann_integral(pair):
    got = float(qo.mutual_pair(*pair))
    ref = neumann_mp(*pair)
    assert abs(got - ref) <= 2e-13 * abs(ref)


def test_mutual_values_quoted_in_survey():
    # 40-digit Neumann/Maxwell values quoted in SURVEY.md §8(c) pins table (tests/golden/pairs.txt)
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "pairs.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 5
    for ri, zi, rj, zj, val in rows:
        got = float(qo.mutual_pair(float(ri), float(zi), float(rj), float(zj)))
        assert abs(got - float(val)) <= 2e-13 * float(val)


def test_elliptic_known_values_and_legendre():
    # Abramowitz & Stegun 17.3: K(m=1/2), E(m=1/2); Legendre relation E K' + E' K - K K' = pi/2
    K, E = qo.elliptic_KE(0.5)
    assert abs(K - 1.8540746773013719) < 2e-15 and abs(E - 1.3506438810476755) < 2e-15
    for kp2 in [1e-8, 1e-4, 0.03, 0.3, 0.5, 0.9, 0.9999]:
        K, E = qo.elliptic_KE(kp2)
        Kp, Ep = qo.elliptic_KE(1.0 - kp2)
        assert abs(E * Kp + Ep * K - K * Kp - math.pi / 2) < 5e-14


def test_far_pair_dipole_limit():
    # two small coaxial loops far apart on the axis: M -> mu0 pi a^2 b^2 / (2 d^3)
    a, b, d = 1e-3, 2e-3, 1.0
    got = float(qo.mutual_pair(a, 0.0, b, d))
    ref = MU0 * math.pi * a * a * b * b / (2 * d ** 3)
    # tolerance: O((a/d)^2) of the dipole limit plus the bracket's cancellation at k^2 = 8e-6
    assert abs(got - ref) < 2e-4 * ref


def test_thin_ring_self_inductance():
    # M(R, R, dz=g) = mu0 R [ln(8R/g) - 2] + O((g/R)^2)   (thin ring, GMD rule)
    g = wl.gmd_factor()
    assert abs(g - 0.4470491559) < 1e-9
    for R, h in [(30.0625e-3, 0.125e-3), (50e-3, 66.67e-6), (30e-3, 15.625e-6)]:
        got = float(qo.mutual_pair(R, 0.0, R, g * h))
        ref = MU0 * R * (math.log(8 * R / (g * h)) - 2.0)
        assert abs(got - ref) < 5 * (g * h / R) ** 2 * math.log(R / (g * h)) * ref


def test_wire_sum_matches_square_wire_inductance():
    # sum_ij M_ij / N^2 over the cells of one 1 mm square wire = self-inductance of that wire
    # = mu0 Rbar [ln(8 Rbar/(gmd * 1 mm)) - 2]; SURVEY.md pins: agree to ~1.3e-4 (8x8), ~8e-5 (16x16)
    for n, tol in [(8, 3e-4), (16, 2e-4)]:
        geo = wl.lattice_geometry(1, 1, n, 1e-3, 30e-3)
        M = qo.dense_M(geo)
        Rbar = 30.5e-3
        ref = MU0 * Rbar * (math.log(8 * Rbar / (wl.gmd_factor() * 1e-3)) - 2.0)
        assert abs(M.sum() / geo.n_rings ** 2 - ref) < tol * ref


def test_symmetric_and_positive_definite():
    geo = wl.lattice_geometry(2, 2, 6, 1e-3, 30e-3)
    M = qo.dense_M(geo)
    assert np.max(np.abs(M - M.T)) <= 1e-16 * np.max(np.abs(M)) * 64
    assert np.linalg.eigvalsh(M).min() > 0
    geo4, x = wl.free_rings(512)
    M4 = qo.dense_M(geo4)
    assert np.max(np.abs(M4 - M4.T)) <= 1e-16 * np.max(np.abs(M4)) * 64
    assert np.linalg.eigvalsh(M4).min() > 0          # softened kernel is SPD
    assert abs(qo.matvec(geo4, x) - M4 @ x).max() < 1e-18


def biot_savart_mp(ri, zi, rj, zj):
    """B = mu0/(4 pi) oint dl x R / R^3 of a unit-current loop (radius rj, height zj) at (ri, 0, zi)."""
    mp.mp.dps = 30
    rho, a, dz = mp.mpf(ri), mp.mpf(rj), mp.mpf(zi) - mp.mpf(zj)
    R3 = lambda p: (rho * rho + a * a + dz * dz - 2 * rho * a * mp.cos(p)) ** mp.mpf(1.5)
    pts = [0, mp.mpf(10) ** -3, mp.mpf(1) / 2, mp.pi]
    c = mp.mpf(10) ** -7 * 2          # mu0/(4 pi) * 2 (integrate half the loop)
    br = c * mp.quad(lambda p: a * dz * mp.cos(p) / R3(p), pts)
    bz = c * mp.quad(lambda p: (a * a - a * rho * mp.cos(p)) / R3(p), pts)
    return float(br), float(bz)


@pytest.mark.parametrize("pt", [(0.040, 0.010, 0.030, 0.0), (0.030, -0.002, 0.0312, 0.001),
                                (0.055, 0.012, 0.041, -0.011), (0.030, 0.0, 0.030125, 0.000125)])
def test_field_equals_biot_savart(pt):
    br, bz = (float(v) for v in qo.field_pair(*pt))
    rbr, rbz = biot_savart_mp(*pt)
    scale = math.hypot(rbr, rbz)
    assert abs(br - rbr) < 1e-12 * scale and abs(bz - rbz) < 1e-12 * scale


def test_field_quoted_values_and_on_axis():
    # SURVEY.md pins: loop (30 mm, 0) seen from (40 mm, 10 mm); on-axis Bz = mu0 a^2 / (2 (a^2+z^2)^1.5)
    br, bz = qo.field_pair(0.040, 0.010, 0.030, 0.0)
    assert abs(br - 7.523910632327161e-6) < 1e-18 and abs(bz + 3.3542215886267729e-6) < 1e-18
    a, z = 0.030, 0.020
    br, bz = qo.field_pair(1e-9, z, a, 0.0)
    ref = MU0 * a * a / (2 * (a * a + z * z) ** 1.5)
    assert abs(ref - 1.2064445040503051e-5) < 1e-19
    assert abs(bz - ref) < 1e-12 * ref
    # first order off the axis: Br = 3 mu0 a^2 z r / (4 (a^2+z^2)^2.5) + O(r^3)
    r = 1e-4
    br, bz = qo.field_pair(r, z, a, 0.0)
    ref_r = 3 * MU0 * a * a * z * r / (4 * (a * a + z * z) ** 2.5)
    assert abs(br - ref_r) < 1e-4 * ref_r and abs(bz - ref) < 1e-4 * ref


def test_field_is_curl_of_vector_potential():
    # A_phi(r, z) = M(r, z; rj, zj)/(2 pi r);  Bz = (1/r) d(r A)/dr,  Br = -dA/dz   (central differences)
    rj, zj = 0.043, 0.002
    for ri, zi in [(0.050, 0.010), (0.041, -0.004), (0.0431, 0.0021)]:
        e = 1e-7
        flux = lambda r, z: float(qo.mutual_pair(r, z, rj, zj)) / (2 * math.pi)      # r * A_phi
        bz_fd = (flux(ri + e, zi) - flux(ri - e, zi)) / (2 * e) / ri
        br_fd = -(flux(ri, zi + e) - flux(ri, zi - e)) / (2 * e) / ri
        br, bz = (float(v) for v in qo.field_pair(ri, zi, rj, zj))
        scale = math.hypot(br, bz)
        assert abs(bz - bz_fd) < 2e-6 * scale and abs(br - br_fd) < 2e-6 * scale


def test_self_field_consistent_with_self_inductance_energy():
    # hoop force on a ring: F_r = (1/2) I^2 dL/dR = I * Bz_self * 2 pi R  with L = mu0 R [ln(8R/g) - 2]
    geo = wl.lattice_geometry(1, 1, 4, 1e-3, 30e-3)
    R, g = geo.r[0], geo.softening
    dLdR = MU0 * (math.log(8 * R / g) - 1.0)
    assert abs(qo.self_field_coef(geo)[0] * 2 * math.pi * R - 0.5 * dLdR) < 1e-15 * dLdR


def test_dense_field_rows_match_pairs_and_diagonal():
    geo = wl.lattice_geometry(1, 2, 4, 1e-3, 30e-3)
    GBr, GBz = qo.dense_GB(geo)
    i, j = 3, 17
    br, bz = qo.field_pair(geo.r[i], geo.z[i], geo.r[j], geo.z[j])
    assert GBr[i, j] == br and GBz[i, j] == bz
    assert np.all(np.diag(GBr) == 0.0)
    assert np.allclose(np.diag(GBz), qo.self_field_coef(geo), rtol=0, atol=0)
    I = np.random.default_rng(0).standard_normal(geo.n_rings)
    rows = np.array([0, 5, 31])
    br, bz = qo.field_eval_rows(geo, I, rows)
    assert np.allclose(br, (GBr @ I)[rows], rtol=1e-14) and np.allclose(bz, (GBz @ I)[rows], rtol=1e-14)

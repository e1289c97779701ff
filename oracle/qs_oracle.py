"""CPU FP64 oracle for the quench-simulation hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this file.  It shares no code with the CUDA path
(``paper_2403_07666_b200/``) and never imports it; the product never imports this.

Plain numpy/scipy, float64, written to be checked against the text by eye.  Citations are
``PAPER.md:<line>`` (= /root/reference/PAPER.md) and ``SURVEY.md §8(c) C<k>`` (the readings
of the points on which the paper's main text is silent; the same list is in DESIGN.md).

Route taken here on purpose differs from the GPU's: K(k), E(k) come from the library
(``scipy.special.ellipkm1`` / ``ellipe``, Cephes) and enter Maxwell's textbook bracket; dense
matrices are formed explicitly; the per-step linear system is solved by dense Cholesky + Schur
complement (its plain definition), with a projected CG only for sizes a dense solve cannot hold.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``):
  mutual_pair        Neumann double integral by quadrature; thin-ring self-inductance
  field_pair         Biot-Savart quadrature; on-axis loop field; curl of A from mutual_pair
  material_law       closed forms E(Jc)=Ec, E'->n Ec/Jc, Jc(4.2 K,0,0), strain zero, dE/dJ by FD
  heat_substeps      exact discrete 1-D steady state; energy balance to rounding
  kkt_dense / pcg    constraint C^T I' = d, KKT residual, dense vs CG, single-ring L-R circuit
  lattice tables     table operator == dense operator on small lattices; FFT application == offset-by-offset sum
  wire statistics    closed forms of a prepared normal-state turn (rho_n J^2), sum_w E_joule == integral of Joule power
  step_rk            exact second-order polynomial and error estimate on the linear L-R ring, global order 2,
                     rejection rule, reduction to the theta = 0 step at constant rate
  heat_adi           line operators == explicit flux divergence, exact discrete steady state as fixed point,
                     second-order convergence to the (Richardson-extrapolated) explicit solution, adiabatic energy identity
  group shares (C16) null-space solve of the constrained system (route independent of the KKT/Schur one), group net
                     currents = share * I(t) along a trajectory, U_terminal * I_ramp == power delivered to the groups,
                     share = 1 reproduces the per-turn results bit for bit
  nonlinear step     the trajectory under a steady field ramp ends in the stationary saturated state, which has a
                     closed form (2 pi r E = -pi r^2 Bdot - V_w, J = Jc sgn(E) (|E|/Ec)^(1/n), V_w from the turn's
                     zero net current): J, E, U_terminal to 1e-11 with both operator/solver routes
  nonlinear transient the moving flux front (before saturation) satisfies Poynting's balance accumulated over the
                     trajectory (magnetic energy + Joule heat = work of the external field) with a residual that
                     halves with dt (0.77 % -> 0.38 % -> 0.19 %), a quarter of the work being dissipated
  Beyond these two properties the pointwise values of the config-1 trajectory have no printed worked example
                     (SURVEY.md §8(c) pins table): there the parity is oracle-vs-GPU plus the oracle-internal
                     cross check dense Cholesky vs tables + CG.
"""
from __future__ import annotations

import math

import numpy as np
import scipy.linalg
import scipy.special

MU0 = 4.0e-7 * math.pi

# event flag bits (PAPER.md:105 |J/Jc|>1, PAPER.md:119 rho>0.95 rho_n)
FJ_T, FJ_E, FJ_J, Q_T, Q_RHO = 1, 2, 4, 8, 16
# qs_step return bits
RET_FLUXJUMP, RET_QUENCH, RET_CG_MAXIT = 1, 2, 4


# --------------------------------------------------------------------------------------
# C2: ring-to-ring mutual inductance (Maxwell's formula for two coaxial filaments)
# --------------------------------------------------------------------------------------
def elliptic_KE(kp2):
    """K(k), E(k) from the complementary parameter kp2 = 1 - k^2 = B2/A2 (library routines)."""
    K = scipy.special.ellipkm1(kp2)
    E = scipy.special.ellipe(1.0 - kp2)
    return K, E


def mutual_pair(ri, zi, rj, zj, soft2=0.0):
    """M_ij [H] between coaxial filaments; ``soft2`` = g^2 added to dz^2.

    A2 = (ri+rj)^2 + dz^2, B2 = (ri-rj)^2 + dz^2, k^2 = 4 ri rj / A2 = 1 - B2/A2
    M = mu0 sqrt(ri rj) [ (2/k - k) K(k) - (2/k) E(k) ]
    """
    dz2 = (zi - zj) ** 2 + soft2
    A2 = (ri + rj) ** 2 + dz2
    B2 = (ri - rj) ** 2 + dz2
    kp2 = B2 / A2
    k = np.sqrt(1.0 - kp2)
    K, E = elliptic_KE(kp2)
    return MU0 * np.sqrt(ri * rj) * ((2.0 / k - k) * K - (2.0 / k) * E)


def mutual_rows(geo, rows):
    """Rows ``rows`` of the symmetric matrix M: [len(rows), N].

    lattice: filament formula off the diagonal, M_ii = M(r_i, r_i, dz = g) (Maxwell's GMD rule);
    free rings: dz^2 + g^2 for every pair (softened Neumann kernel, SPD by construction).
    """
    rows = np.asarray(rows, dtype=np.int64)
    g2 = float(geo.softening) ** 2
    ri, zi = geo.r[rows, None], geo.z[rows, None]
    rj, zj = geo.r[None, :], geo.z[None, :]
    if geo.lattice:
        soft = np.zeros((rows.size, geo.n_rings))
        soft[np.arange(rows.size), rows] = g2          # i == j only
        return mutual_pair(ri, zi, rj, zj, soft)
    return mutual_pair(ri, zi, rj, zj, g2)


def dense_M(geo, chunk=512):
    N = geo.n_rings
    M = np.empty((N, N))
    for s in range(0, N, chunk):
        e = min(N, s + chunk)
        M[s:e] = mutual_rows(geo, np.arange(s, e))
    return M


def matvec_rows(geo, x, rows, chunk=256):
    """y_i = sum_j M_ij x_j for the listed target rows, evaluated pair by pair."""
    rows = np.asarray(rows, dtype=np.int64)
    y = np.empty(rows.size)
    for s in range(0, rows.size, chunk):
        e = min(rows.size, s + chunk)
        y[s:e] = mutual_rows(geo, rows[s:e]) @ x
    return y


def matvec(geo, x, chunk=256):
    return matvec_rows(geo, x, np.arange(geo.n_rings), chunk)


# --------------------------------------------------------------------------------------
# C3: field of a unit-current loop
# --------------------------------------------------------------------------------------
def field_pair(ri, zi, rj, zj):
    """(Br, Bz) [T/A] at (ri, zi) of a unit-current filament loop of radius rj at height zj.

    Bz = mu0/(2 pi sqrt(A2)) [ K + (rj^2 - ri^2 - dz^2)/B2 E ]
    Br = mu0/(2 pi sqrt(A2)) (dz/ri) [ -K + (rj^2 + ri^2 + dz^2)/B2 E ],   dz = zi - zj
    """
    dz = zi - zj
    A2 = (ri + rj) ** 2 + dz ** 2
    B2 = (ri - rj) ** 2 + dz ** 2
    K, E = elliptic_KE(B2 / A2)
    pref = MU0 / (2.0 * math.pi * np.sqrt(A2))
    Bz = pref * (K + (rj ** 2 - ri ** 2 - dz ** 2) / B2 * E)
    Br = pref * (dz / ri) * (-K + (rj ** 2 + ri ** 2 + dz ** 2) / B2 * E)
    return Br, Bz


def self_field_coef(geo):
    """Bz_self,i / I_i = mu0 [ln(8 r_i / g) - 1] / (4 pi r_i); Br_self = 0."""
    return MU0 * (np.log(8.0 * geo.r / geo.softening) - 1.0) / (4.0 * math.pi * geo.r)


def field_rows(geo, rows):
    """Rows of the dense field matrices (GBr, GBz): B_i = sum_j GB_ij I_j, self term on the diagonal."""
    rows = np.asarray(rows, dtype=np.int64)
    ri, zi = geo.r[rows, None], geo.z[rows, None]
    rj = np.broadcast_to(geo.r[None, :], (rows.size, geo.n_rings)).copy()
    zj = np.broadcast_to(geo.z[None, :], (rows.size, geo.n_rings)).copy()
    idx = np.arange(rows.size)
    zj[idx, rows] += 1.0                      # keep the i == j entry finite; overwritten below
    Br, Bz = field_pair(ri, zi, rj, zj)
    Br[idx, rows] = 0.0
    Bz[idx, rows] = self_field_coef(geo)[rows]
    return Br, Bz


def dense_GB(geo, chunk=512):
    N = geo.n_rings
    GBr, GBz = np.empty((N, N)), np.empty((N, N))
    for s in range(0, N, chunk):
        e = min(N, s + chunk)
        GBr[s:e], GBz[s:e] = field_rows(geo, np.arange(s, e))
    return GBr, GBz


def field_eval_rows(geo, I, rows, chunk=256):
    """(Br_i, Bz_i) of ring currents I [A] at the listed rows, without B_ext."""
    rows = np.asarray(rows, dtype=np.int64)
    Br, Bz = np.empty(rows.size), np.empty(rows.size)
    for s in range(0, rows.size, chunk):
        e = min(rows.size, s + chunk)
        gr, gz = field_rows(geo, rows[s:e])
        Br[s:e], Bz[s:e] = gr @ I, gz @ I
    return Br, Bz


# --------------------------------------------------------------------------------------
# Lattice tables (SURVEY.md §8(d) "Oracle timing"): on a regular lattice M and G_B depend only
# on (ir, jr, iz - jz).  Used for lattices too large for dense matrices; checked against the
# dense operators on small lattices (tests/test_oracle_lattice.py).
# --------------------------------------------------------------------------------------
class LatticeTables:
    """Tables T[d, ir, jr] of the pair quantities at axial offset d = |iz - jz| (storage: one contiguous
    Nr x Nr matrix per offset, so that applying offset d is one plain matrix product)."""

    def __init__(self, geo, with_field=True):
        assert geo.lattice
        Nr, Nz, h = geo.Nr, geo.Nz, geo.h
        self.Nr, self.Nz = Nr, Nz
        rr = geo.r.reshape(Nr, Nz)[:, 0]
        d = np.arange(Nz) * h                                   # |iz - jz| * h
        ri, rj, dz = rr[:, None, None], rr[None, :, None], d[None, None, :]
        soft = np.zeros((Nr, Nr, Nz))
        soft[np.arange(Nr), np.arange(Nr), 0] = float(geo.softening) ** 2
        self.M = np.empty((Nz, Nr, Nr))
        for a in range(Nr):                                     # row by row: bounded memory
            self.M[:, a, :] = mutual_pair(ri[a], 0.0, rj[0], dz[0], soft[a]).T
        self.with_field = with_field
        if with_field:
            self.Br = np.empty((Nz, Nr, Nr))                    # for dz = +d (target above source)
            self.Bz = np.empty((Nz, Nr, Nr))
            selfc = self_field_coef(geo).reshape(Nr, Nz)[:, 0]
            for a in range(Nr):
                dzz = np.broadcast_to(dz[0], (Nr, Nz)).copy()
                dzz[a, 0] = 1.0
                br, bz = field_pair(ri[a], dzz, rj[0], 0.0)
                br[a, 0], bz[a, 0] = 0.0, selfc[a]
                self.Br[:, a, :], self.Bz[:, a, :] = br.T, bz.T

    def _apply(self, tab, X, odd):
        """Y[ir, iz] = sum_{jr, jz} tab[|iz-jz|, ir, jr] * sgn * X[jr, jz], offset by offset."""
        Nz = self.Nz
        Y = tab[0] @ X
        for d in range(1, Nz):
            T = tab[d]
            Y[:, d:] += T @ X[:, : Nz - d]                       # targets above sources: dz = +d h
            Y[:, : Nz - d] += (-1.0 if odd else 1.0) * (T @ X[:, d:])   # dz = -d h
        return Y

    def matvec(self, x):
        return self._apply(self.M, x.reshape(self.Nr, self.Nz), False).reshape(-1)

    def field(self, I):
        X = I.reshape(self.Nr, self.Nz)
        return (self._apply(self.Br, X, True).reshape(-1), self._apply(self.Bz, X, False).reshape(-1))


class LatticeTablesFFT(LatticeTables):
    """The same tables applied through the convolution theorem (for the one lattice the plain offset loop cannot
    finish in hours: config 3 at full size, Nr^2 Nz^2 = 7.5e11 multiply-adds per application).

    Along z the operator is a Toeplitz matrix per (ir, jr): Y[ir, iz] = sum_jr sum_jz c_{ir,jr}[iz - jz] X[jr, jz]
    with c[+d] = T[d], c[-d] = sgn T[d].  Embedded in a circulant of length L = 2 Nz (X zero-padded), the product is
    a pointwise product of discrete Fourier transforms (library FFT), summed over jr frequency by frequency.
    Pinned against LatticeTables._apply (the defining sum) in tests/test_oracle_solver_step.py; the long-parity
    script also re-checks it against the plain loop on the very state it compares.
    """

    def __init__(self, geo, with_field=True):
        super().__init__(geo, with_field)
        self.specM = self._spectrum(self.M, False)
        if with_field:
            self.specBr = self._spectrum(self.Br, True)
            self.specBz = self._spectrum(self.Bz, False)

    def _spectrum(self, tab, odd):
        Nr, Nz = self.Nr, self.Nz
        L = 2 * Nz
        spec = np.empty((Nz + 1, Nr, Nr), dtype=np.complex128)
        sgn = -1.0 if odd else 1.0
        for a in range(Nr):                                     # row by row: bounded memory
            col = np.zeros((L, Nr))
            col[:Nz] = tab[:, a, :]                             # e = iz - jz = +d
            col[L - Nz + 1:] = sgn * tab[:0:-1, a, :]           # e = -d  ->  slot L - d
            spec[:, a, :] = np.fft.rfft(col, axis=0)
        return spec

    def _apply_fft(self, spec, X):
        Nz = self.Nz
        Xh = np.fft.rfft(X, n=2 * Nz, axis=1)                   # [Nr, Nz + 1]
        Yh = np.einsum("kij,jk->ik", spec, Xh)                  # one Nr x Nr matrix-vector product per frequency
        return np.fft.irfft(Yh, n=2 * Nz, axis=1)[:, :Nz]

    def matvec(self, x):
        return self._apply_fft(self.specM, x.reshape(self.Nr, self.Nz)).reshape(-1)

    def field(self, I):
        X = I.reshape(self.Nr, self.Nz)
        return self._apply_fft(self.specBr, X).reshape(-1), self._apply_fft(self.specBz, X).reshape(-1)

    def matvec_plain(self, x):
        return LatticeTables.matvec(self, x)

    def field_plain(self, I):
        return LatticeTables.field(self, I)


# --------------------------------------------------------------------------------------
# C5: material law (BASELINE.json configs[0]; PAPER.md:79 E-J law spanning creep -> normal)
# --------------------------------------------------------------------------------------
def ipow(x, n):
    """x**n for a non-negative integer n by repeated multiplication (SURVEY.md C5 guard note)."""
    out = np.ones_like(x)
    with np.errstate(over="ignore"):
        for _ in range(int(n)):
            out = out * x
    return out


def material_law(mat, J, T, Br, Bz, r, jc0_scale):
    """Returns dict(eps, Jc, rho, E, dEdJ, Q) per cell.

    eps = J Bz r / Y ; |B| = sqrt(Br^2+Bz^2)
    Jc  = Jc0 s max(1-T/Tc,0)^2 / (1+|B|/B0) max(1-eps_coef |eps|^eps_exp, 0)
    rho_sc = (Ec/Jc)(|J|/Jc)^(n-1) ; rho = rho_sc rho_n/(rho_sc+rho_n)
    E = rho J ; Q = E J ; dE/dJ = rho (1 + (n-1) rho_n/(rho_sc+rho_n))
    Guards: Jc <= 0 -> rho = dE/dJ = rho_n ; J == 0 -> rho = dE/dJ = 0.
    """
    n = mat.n_exp
    eps = J * Bz * r / mat.Y
    Bmag = np.sqrt(Br * Br + Bz * Bz)
    fT = np.maximum(1.0 - T / mat.Tc, 0.0)
    fe = np.maximum(1.0 - mat.eps_coef * np.abs(eps) ** mat.eps_exp, 0.0)
    Jc = mat.Jc0 * jc0_scale * fT * fT / (1.0 + Bmag / mat.B0) * fe
    rho = np.empty_like(J)
    dEdJ = np.empty_like(J)
    normal = Jc <= 0.0
    zero = (J == 0.0) & ~normal
    sc = ~normal & ~zero
    rho[normal] = mat.rho_n
    dEdJ[normal] = mat.rho_n
    rho[zero] = 0.0
    dEdJ[zero] = 0.0
    if np.any(sc):
        x = np.abs(J[sc]) / Jc[sc]
        if float(n) == int(n):
            xp = ipow(x, int(n) - 1)
        else:
            xp = x ** (n - 1.0)
        with np.errstate(over="ignore", invalid="ignore", divide="ignore"):
            rho_sc = (mat.Ec / Jc[sc]) * xp
            big = rho_sc >= mat.rho_n
            u = np.where(big, mat.rho_n / rho_sc, rho_sc / mat.rho_n)   # always in [0, 1]
        # rho = rho_sc rho_n/(rho_sc + rho_n), w = rho_n/(rho_sc + rho_n), overflow-free forms
        rho_s = np.where(big, mat.rho_n / (1.0 + u), np.where(np.isfinite(rho_sc), rho_sc, 0.0) / (1.0 + u))
        w = np.where(big, u / (1.0 + u), 1.0 / (1.0 + u))
        rho[sc] = rho_s
        dEdJ[sc] = rho_s * (1.0 + (n - 1.0) * w)
    E = rho * J
    return dict(eps=eps, Jc=Jc, rho=rho, E=E, dEdJ=dEdJ, Q=E * J)


# --------------------------------------------------------------------------------------
# C9: explicit finite-volume heat sub-steps in enthalpy form (PAPER.md:75 heat equation + Robin BC)
# --------------------------------------------------------------------------------------
def enthalpy(mat, T):
    """H(T) = int_0^T C dT = C3/4 T^4 + C1/2 T^2,  C(T) = C3 T^3 + C1 T."""
    return 0.25 * mat.C3 * T ** 4 + 0.5 * mat.C1 * T ** 2


def temperature(mat, H):
    """Inverse of enthalpy(): T^2 = (-C1/2 + sqrt(C1^2/4 + C3 H)) / (C3/2)."""
    return np.sqrt((-0.5 * mat.C1 + np.sqrt(0.25 * mat.C1 ** 2 + mat.C3 * H)) / (0.5 * mat.C3))


def heat_substeps_count(geo, mat, dt):
    """m = ceil(dt / (0.8 h^2/(4 alpha0))), alpha0 = k_in/(C3 T_bath^2 + C1)."""
    alpha0 = mat.k_in / (mat.C3 * geo.T_bath * geo.T_bath + mat.C1)
    limit = 0.8 * geo.h * geo.h / (4.0 * alpha0)
    return max(1, int(math.ceil(dt / limit)))


def heat_flux_divergence(geo, mat, T2d):
    """sum_f F_f [W] per cell and the boundary loss [W] summed over the pack.

    interior face c|c': F = kappa_f (T_c'^2 - T_c^2)/(2h) A_f, kappa_f = k_in if same turn else k_between
    boundary face:      F = -h_conv,side (T_c - T_bath) A_f
    radial face area 2 pi (r_c +- h/2) h, axial face area 2 pi r_c h.
    """
    Nr, Nz, n, h = geo.Nr, geo.Nz, geo.cells_per_side, geo.h
    r2d = geo.r.reshape(Nr, Nz)
    T2 = T2d * T2d
    F = np.zeros((Nr, Nz))
    # radial faces between ir and ir+1
    same = ((np.arange(Nr - 1) // n) == (np.arange(1, Nr) // n))
    kap = np.where(same, mat.k_in, mat.k_between)[:, None]
    area = 2.0 * math.pi * (r2d[:-1] + 0.5 * h) * h
    flow = kap * (T2[1:] - T2[:-1]) / (2.0 * h) * area          # into cell ir from ir+1
    F[:-1] += flow
    F[1:] -= flow
    # axial faces between iz and iz+1
    same = ((np.arange(Nz - 1) // n) == (np.arange(1, Nz) // n))
    kap = np.where(same, mat.k_in, mat.k_between)[None, :]
    area = 2.0 * math.pi * r2d[:, :-1] * h
    flow = kap * (T2[:, 1:] - T2[:, :-1]) / (2.0 * h) * area
    F[:, :-1] += flow
    F[:, 1:] -= flow
    # four borders of the winding pack ("four borders on the cross-section")
    hc = geo.h_conv
    loss = np.zeros((Nr, Nz))
    loss[0] += hc[0] * (T2d[0] - geo.T_bath) * 2.0 * math.pi * (r2d[0] - 0.5 * h) * h
    loss[-1] += hc[1] * (T2d[-1] - geo.T_bath) * 2.0 * math.pi * (r2d[-1] + 0.5 * h) * h
    loss[:, 0] += hc[2] * (T2d[:, 0] - geo.T_bath) * 2.0 * math.pi * r2d[:, 0] * h
    loss[:, -1] += hc[3] * (T2d[:, -1] - geo.T_bath) * 2.0 * math.pi * r2d[:, -1] * h
    return F - loss, float(loss.sum())


def heat_substeps(geo, mat, H, Q, dt, m):
    """m explicit sub-steps of dH/dt = sum_f F_f / V + Q with Q frozen; returns (H, boundary energy [J])."""
    Nr, Nz, h = geo.Nr, geo.Nz, geo.h
    vol = (2.0 * math.pi * geo.r * h * h).reshape(Nr, Nz)
    H2 = H.reshape(Nr, Nz).copy()
    Q2 = Q.reshape(Nr, Nz)
    sub = dt / m
    lost = 0.0
    for _ in range(m):
        T2d = temperature(mat, H2)
        div, loss = heat_flux_divergence(geo, mat, T2d)
        H2 = H2 + sub * (div / vol + Q2)
        lost += sub * loss
    return H2.reshape(-1), lost


# --------------------------------------------------------------------------------------
# C15 (f4): ADI heat step ("heat equation ... solved by ADI"), Peaceman-Rachford on U = T^2
# --------------------------------------------------------------------------------------
def heat_line_operators(geo, mat):
    """Sparse L_r, L_z [1/s * J/m^3 per K^2] acting on U = T^2 (per cell, divided by the cell volume) and the Robin
    film coefficients per cell rb_r, rb_z [W/m^3 K] of the r- and z-borders; same faces, areas and conductivities as
    heat_flux_divergence (C9): (L_r U)_c = sum over the two radial faces of kappa_f (U_c' - U_c)/(2h) A_f / V_c."""
    import scipy.sparse as sp
    Nr, Nz, n, h = geo.Nr, geo.Nz, geo.cells_per_side, geo.h
    N = Nr * Nz
    r2d = geo.r.reshape(Nr, Nz)
    vol = 2.0 * math.pi * r2d * h * h
    idx = np.arange(N).reshape(Nr, Nz)
    rows, cols, vals = [], [], []
    def add(i, j, v):
        rows.append(i.ravel()); cols.append(j.ravel()); vals.append(v.ravel())
    # radial faces ir | ir+1
    same = ((np.arange(Nr - 1) // n) == (np.arange(1, Nr) // n))
    kap = np.where(same, mat.k_in, mat.k_between)[:, None]
    g = kap * 2.0 * math.pi * (r2d[:-1] + 0.5 * h) * h / (2.0 * h)          # face conductance on U
    lo, hi = idx[:-1], idx[1:]
    Lr_parts = [(lo, hi, g / vol[:-1]), (lo, lo, -g / vol[:-1]), (hi, lo, g / vol[1:]), (hi, hi, -g / vol[1:])]
    for i, j, v in Lr_parts:
        add(i, j, v)
    Lr = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(N, N))
    rows, cols, vals = [], [], []
    same = ((np.arange(Nz - 1) // n) == (np.arange(1, Nz) // n))
    kap = np.where(same, mat.k_in, mat.k_between)[None, :]
    g = kap * 2.0 * math.pi * r2d[:, :-1] * h / (2.0 * h)
    lo, hi = idx[:, :-1], idx[:, 1:]
    for i, j, v in [(lo, hi, g / vol[:, :-1]), (lo, lo, -g / vol[:, :-1]), (hi, lo, g / vol[:, 1:]), (hi, hi, -g / vol[:, 1:])]:
        add(i, j, v)
    Lz = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(N, N))
    hc = geo.h_conv
    rb_r = np.zeros((Nr, Nz))
    rb_r[0] += hc[0] * 2.0 * math.pi * (r2d[0] - 0.5 * h) * h / vol[0]
    rb_r[-1] += hc[1] * 2.0 * math.pi * (r2d[-1] + 0.5 * h) * h / vol[-1]
    rb_z = np.zeros((Nr, Nz))
    rb_z[:, 0] += hc[2] * 2.0 * math.pi * r2d[:, 0] * h / vol[:, 0]
    rb_z[:, -1] += hc[3] * 2.0 * math.pi * r2d[:, -1] * h / vol[:, -1]
    return Lr, Lz, rb_r.ravel(), rb_z.ravel()


def heat_adi(geo, mat, H, Q, dt, m):
    """m Peaceman-Rachford ADI sub-steps of length delta = dt/m on U = T^2 with the capacity lagged at the start of
    each sub-step (reading C15).  With H' = dH/dU = C3/2 U + C1/2 and the Robin loss linearised about U^k,
    rb (T - T_b) ~ rb (T^k/2 - T_b) + rb/(2 T^k) U:
        (2H'/delta - L_r + beta_r) U*  = 2H'/delta U^k + L_z U^k - rb_z (T^k - T_b) + Q - c_r      (implicit in r)
        (2H'/delta - L_z + beta_z) U'  = 2H'/delta U*  + L_r U* - beta_r U* - c_r + Q - c_z        (implicit in z)
    beta = rb/(2 T^k), c = rb (T^k/2 - T_b).  Returns the new enthalpy H(U')."""
    import scipy.sparse as sp
    import scipy.sparse.linalg as spla
    Lr, Lz, rb_r, rb_z = heat_line_operators(geo, mat)
    delta = dt / m
    H = H.copy()
    for _ in range(m):
        T = temperature(mat, H)
        U = T * T
        Hp = 0.5 * mat.C3 * U + 0.5 * mat.C1
        beta_r, beta_z = rb_r / (2.0 * T), rb_z / (2.0 * T)
        c_r, c_z = rb_r * (0.5 * T - geo.T_bath), rb_z * (0.5 * T - geo.T_bath)
        D = sp.diags(2.0 * Hp / delta)
        rhs1 = 2.0 * Hp / delta * U + Lz @ U - rb_z * (T - geo.T_bath) + Q - c_r
        Us = spla.spsolve((D - Lr + sp.diags(beta_r)).tocsc(), rhs1)
        rhs2 = 2.0 * Hp / delta * Us + Lr @ Us - beta_r * Us - c_r + Q - c_z
        Un = spla.spsolve((D - Lz + sp.diags(beta_z)).tocsc(), rhs2)
        H = H + Hp * (Un - U)          # the two half-steps are exactly an energy balance for H' dU: keep it exact
    return H


# --------------------------------------------------------------------------------------
# C4 / C8: circuit equations.   [A C; C^T 0] [I'; V] = [b; d],  A = M + theta dt D
# --------------------------------------------------------------------------------------
def constraint_matrix(geo):
    C = np.zeros((geo.n_rings, geo.n_turns))
    if geo.n_turns:
        C[np.arange(geo.n_rings), geo.turn_id] = 1.0
    return C


def kkt_dense(A, C, b, d):
    """Unique solution of the KKT system by dense Cholesky + Schur complement (SURVEY.md C8 brute force).

    S = C^T A^-1 C ; V = S^-1 (C^T A^-1 b - d) ; I' = A^-1 (b - C V)
    """
    cf = scipy.linalg.cho_factor(A, lower=True)
    Ainv_b = scipy.linalg.cho_solve(cf, b)
    if C.shape[1] == 0:
        return Ainv_b, np.zeros(0)
    Ainv_C = scipy.linalg.cho_solve(cf, C)
    S = C.T @ Ainv_C
    V = np.linalg.solve(S, C.T @ Ainv_b - d)
    return Ainv_b - Ainv_C @ V, V


def pcg(apply_A, diagA, turn_id, n_turns, b, d, tol, maxit, x0=None):
    """Projected CG with per-turn Schur complement, SURVEY.md C8 step by step.

    Returns (x, V, iterations, sqrt(r^T g) / nu).  nu = sqrt(r^T g) of the cold start x_p
    (reference norm: b can be exactly 0, so "relative to |b|" is undefined).
    """
    N = b.size
    Hd = diagA
    if n_turns:
        s = np.bincount(turn_id, weights=1.0 / Hd, minlength=n_turns)

    def project(r):
        if not n_turns:
            return r / Hd, np.zeros(0)
        v = np.bincount(turn_id, weights=r / Hd, minlength=n_turns) / s
        return (r - v[turn_id]) / Hd, v

    # cold start x_p = H^-1 C (d/s): satisfies C^T x = d; its projected residual is the reference norm nu
    x = np.zeros(N)
    if n_turns:
        x = (d / s)[turn_id] / Hd
    vsum = np.zeros(n_turns)
    r = apply_A(x) - b
    g, v = project(r)
    if n_turns:
        r = r - v[turn_id]
    nu = math.sqrt(max(float(r @ g), 0.0))
    if nu == 0.0:
        return x, -v, 0, 0.0
    if x0 is not None:                       # warm start, moved onto the constraint
        x = x0.copy()
        if n_turns:
            cur = np.bincount(turn_id, weights=x, minlength=n_turns)
            x = x + ((d - cur) / s)[turn_id] / Hd
        r = apply_A(x) - b
        g, v = project(r)
        if n_turns:
            r = r - v[turn_id]
    if n_turns:
        vsum += v
    p = -g
    rg = float(r @ g)
    it = 0
    while it < maxit and math.sqrt(max(rg, 0.0)) > tol * nu:
        q = apply_A(p)
        alpha = rg / float(p @ q)
        x = x + alpha * p
        r = r + alpha * q
        g, v = project(r)
        if n_turns:
            r = r - v[turn_id]
            vsum += v
        rg_new = float(r @ g)
        p = -g + (rg_new / rg) * p
        rg = rg_new
        it += 1
    return x, -vsum, it, math.sqrt(max(rg, 0.0)) / nu


# --------------------------------------------------------------------------------------
# C10: events
# --------------------------------------------------------------------------------------
def turn_observables(geo, mat, T, E, J, Jc, rho):
    """Per turn: Tmax, mean|E|, max|J|/Jc, min rho/rho_n."""
    nt, tid = geo.n_turns, geo.turn_id
    Tmax = np.full(nt, -np.inf)
    np.maximum.at(Tmax, tid, T)
    Ebar = np.bincount(tid, weights=np.abs(E), minlength=nt) / np.bincount(tid, minlength=nt)
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(Jc > 0.0, np.abs(J) / np.where(Jc > 0.0, Jc, 1.0), np.where(J != 0.0, np.inf, 0.0))
    xmax = np.zeros(nt)
    np.maximum.at(xmax, tid, ratio)
    rmin = np.full(nt, np.inf)
    np.minimum.at(rmin, tid, rho / mat.rho_n)
    return Tmax, Ebar, xmax, rmin


# --------------------------------------------------------------------------------------
# The stepper: same calls as include/qs.h (qs_init / qs_step / qs_read / qs_write / ...)
# --------------------------------------------------------------------------------------
class Oracle:
    """operator = 'dense' (N <= ~8k), 'tables' (regular lattices of any size), 'tables_fft' (the same tables applied by
    FFT along z: config 3 at full size only)."""

    def __init__(self, geo, mat, operator="dense", solver="cholesky"):
        self.geo, self.mat = geo, mat
        N = geo.n_rings
        self.N = N
        self.scale = np.ones(N) if mat.jc0_scale is None else np.asarray(mat.jc0_scale, dtype=np.float64)
        self.operator, self.solver = operator, solver
        self.tables = None
        self.M = self.GBr = self.GBz = None
        if operator == "dense":
            self.M = dense_M(geo)
            if geo.lattice:
                self.GBr, self.GBz = dense_GB(geo)
            self.diagM = np.diag(self.M).copy()
        elif operator in ("tables", "tables_fft"):
            self.tables = LatticeTables(geo) if operator == "tables" else LatticeTablesFFT(geo)
            rr = np.arange(geo.Nr)
            self.diagM = np.repeat(self.tables.M[0, rr, rr], geo.Nz)
        else:
            raise ValueError(operator)
        self.C = constraint_matrix(geo) if (solver == "cholesky" and operator == "dense") else None
        # C16 (PAPER.md:61-67 sub-elements): group w carries share_w of the transport current; default 1 (wires in series)
        sh = getattr(geo, "turn_share", None)
        self.share = np.ones(geo.n_turns) if sh is None else np.asarray(sh, dtype=np.float64)
        self.J = np.zeros(N)
        self.T = np.full(N, geo.T_bath)
        self.H = enthalpy(mat, self.T)
        self.t, self.I = 0.0, 0.0
        self.Br, self.Bz, self.E = np.zeros(N), np.zeros(N), np.zeros(N)
        self.Idot = np.zeros(N)
        nt = max(geo.n_turns, 0)
        self.flags = np.zeros(nt, dtype=np.int32)
        self.t_first = np.full(nt, -1.0)
        self.count = np.zeros(nt, dtype=np.int32)
        self.Ebar_prev = None
        # per-wire statistics (PAPER.md:107 T_max, P_max, Q_FJ per wire; PAPER.md:119-121 Q_q, P_q, T_q)
        self.wire = dict(E_joule=np.zeros(nt), Q_FJ=np.zeros(nt), P_max=np.zeros(nt), T_max=np.full(nt, geo.T_bath),
                         t_q=np.full(nt, -1.0), T_q=np.zeros(nt), P_q=np.zeros(nt), Q_q=np.zeros(nt),
                         E_at_first=np.zeros(nt))
        self.stats = dict(cg_iters=0, cg_relres=0.0, U_terminal=0.0, Tmax=geo.T_bath, joule_power=0.0,
                          boundary_energy=0.0, heat_substeps=0)

    # -- operators ----------------------------------------------------------------
    def apply_M(self, x):
        return self.M @ x if self.M is not None else self.tables.matvec(x)

    def field(self, Icur):
        if self.M is not None:
            return self.GBr @ Icur, self.GBz @ Icur
        return self.tables.field(Icur)

    def Bext(self, t):
        g = self.geo
        if g.Bext_rate == 0.0:
            return g.Bext0
        return min(g.Bext0 + g.Bext_rate * t, g.Bext_max)

    # -- state --------------------------------------------------------------------
    def write(self, J, T, t, I):
        self.J, self.T = np.array(J, dtype=np.float64), np.array(T, dtype=np.float64)
        self.H = enthalpy(self.mat, self.T)
        self.t, self.I = float(t), float(I)
        self.Ebar_prev = None
        self.Idot = np.zeros(self.N)
        nt = max(self.geo.n_turns, 0)
        for key, val in self.wire.items():                      # qs_write resets the per-wire statistics
            val[:] = self.geo.T_bath if key == "T_max" else (-1.0 if key == "t_q" else 0.0)

    def read(self):
        return self.J.copy(), self.T.copy(), np.concatenate([self.Br, self.Bz]), self.E.copy()

    def _heat(self, Q, dt):
        """S6: explicit sub-steps (C9) or, when material.heat_adi_substeps = m > 0, m ADI sub-steps (C15)."""
        m_adi = int(getattr(self.mat, "heat_adi_substeps", 0))
        if m_adi > 0:
            return m_adi, heat_adi(self.geo, self.mat, self.H, Q, dt, m_adi), float("nan")
        m = heat_substeps_count(self.geo, self.mat, dt)
        H, lost = heat_substeps(self.geo, self.mat, self.H, Q, dt, m)
        return m, H, lost

    # -- one step (order of C6: everything on the rhs at t^k) ----------
    def step(self, dt, I_ramp):
        geo, mat = self.geo, self.mat
        if not geo.lattice:
            raise ValueError("qs_step needs a lattice geometry")
        if dt <= 0.0:
            return -5
        a = geo.area
        # S1 field of the ring currents I = a J plus the background field at t^k
        B0, B1 = self.Bext(self.t), self.Bext(self.t + dt)
        Bdot = (B1 - B0) / dt
        Br, Bz = self.field(a * self.J)
        Bz = Bz + B0
        # S2 material law at (J^k, T^k, B^k); rhs b = -2 pi r (E + r Bdot / 2)   (C4)
        ml = material_law(mat, self.J, self.T, Br, Bz, geo.r, self.scale)
        b = -2.0 * math.pi * geo.r * (ml["E"] + 0.5 * geo.r * Bdot)
        D = 2.0 * math.pi * geo.r * ml["dEdJ"] / a
        shift = mat.theta * dt * D
        d = float(I_ramp) * self.share                       # C^T I' = share * I_ramp (C16)
        # S3/S4 constrained solve (C7: linearly implicit theta step)
        if self.solver == "cholesky":
            A = self.M + np.diag(shift)
            Idot, V = kkt_dense(A, self.C, b, d)
            iters, relres = 0, 0.0
        else:
            Idot, V, iters, relres = pcg(lambda x: self.apply_M(x) + shift * x, self.diagM + shift,
                                         geo.turn_id, geo.n_turns, b, d, mat.cg_tol, mat.cg_maxit, self.Idot)
        # S5 update
        self.Idot = Idot
        Jold = self.J
        self.J = self.J + dt * Idot / a
        self.I += dt * I_ramp
        self.t += dt
        # S6 heat with the Joule source of step k frozen over the sub-steps
        m, self.H, lost = self._heat(ml["Q"], dt)
        self.T = temperature(mat, self.H)
        self.Br, self.Bz, self.E = Br, Bz, ml["E"]
        # S7 events: T^{k+1}; E, |J|/Jc, rho of the material evaluation of this step
        ret = self._events(dt, Jold, ml) if geo.n_turns else 0
        self.stats = dict(cg_iters=iters, cg_relres=relres, U_terminal=float(-(self.share @ V)),
                          Tmax=float(self.T.max()),
                          joule_power=float(np.sum(ml["Q"] * 2.0 * math.pi * geo.r * a)),
                          boundary_energy=lost, heat_substeps=m)
        if not (np.all(np.isfinite(self.J)) and np.all(np.isfinite(self.T))):
            return -3
        return ret

    # -- embedded Heun-Euler step with error control ("Runge-Kutta method with
    #    variable time step") ---------------------------------------------------------------------------------------
    def _em_rate(self, J, T, t_stage, Bdot, I_ramp):
        """I' of the circuit equations with everything evaluated at the given state (explicit stage, no theta term):
        M I' + C V = b(E(J, T, B(J) + B_ext(t_stage))), C^T I' = I_ramp.  Returns (I', V, Br, Bz, material dict)."""
        geo, mat = self.geo, self.mat
        Br, Bz = self.field(geo.area * J)
        Bz = Bz + self.Bext(t_stage)
        ml = material_law(mat, J, T, Br, Bz, geo.r, self.scale)
        b = -2.0 * math.pi * geo.r * (ml["E"] + 0.5 * geo.r * Bdot)
        d = float(I_ramp) * self.share                       # C^T I' = share * I_ramp (C16)
        if self.solver == "cholesky":
            if getattr(self, "_cfM", None) is None:
                self._cfM = scipy.linalg.cho_factor(self.M, lower=True)       # M is constant: factor once
                self._AinvC = scipy.linalg.cho_solve(self._cfM, self.C) if geo.n_turns else None
                self._S = self.C.T @ self._AinvC if geo.n_turns else None
            Ainv_b = scipy.linalg.cho_solve(self._cfM, b)
            if geo.n_turns:
                V = np.linalg.solve(self._S, self.C.T @ Ainv_b - d)
                return Ainv_b - self._AinvC @ V, V, Br, Bz, ml
            return Ainv_b, np.zeros(0), Br, Bz, ml
        Idot, V, _, _ = pcg(self.apply_M, self.diagM, geo.turn_id, geo.n_turns, b, d, mat.cg_tol, mat.cg_maxit, self.Idot)
        return Idot, V, Br, Bz, ml

    def step_rk(self, dt_try, I_ramp, rtol, dt_min):
        """One ACCEPTED embedded Heun-Euler (RK12) step of the electromagnetic equations with T frozen at T^k, then the
        heat step (readings: DESIGN.md §3 "C14").  Returns (event word, dt_taken, dt_next, err).

        stage 1: I'_1 at (J^k, t^k);  predictor J* = J^k + dt I'_1/a;  stage 2: I'_2 at (J*, t^k + dt)
        J^{k+1} = J^k + dt (I'_1 + I'_2) / (2a);   err = max_i |dt (I'_2 - I'_1)_i / (2 a_i)| / J_ref,
        J_ref = Jc0 (1 - T_bath/Tc)^2.   Accept if err <= rtol or dt == dt_min; else retry with
        dt <- max(dt_min, dt max(0.2, 0.9 sqrt(rtol/err))).   dt_next = dt min(2, max(0.2, 0.9 sqrt(rtol/err))).
        Heat source: the trapezoid (Q_1 + Q_2)/2; B, E, events: those of stage 2.
        """
        geo, mat = self.geo, self.mat
        a = geo.area
        Jref = mat.Jc0 * (1.0 - geo.T_bath / mat.Tc) ** 2
        dt = float(dt_try)
        while True:
            Bdot = (self.Bext(self.t + dt) - self.Bext(self.t)) / dt
            I1, V1, _, _, ml1 = self._em_rate(self.J, self.T, self.t, Bdot, I_ramp)
            Jstar = self.J + dt * I1 / a
            I2, V2, Br2, Bz2, ml2 = self._em_rate(Jstar, self.T, self.t + dt, Bdot, I_ramp)
            err = float(np.max(np.abs(0.5 * dt * (I2 - I1) / a))) / Jref
            fac = 2.0 if err == 0.0 else min(2.0, max(0.2, 0.9 * math.sqrt(rtol / err)))
            if err <= rtol or dt <= dt_min:
                break
            dt = max(dt_min, dt * fac)
        Jold = self.J
        self.J = self.J + 0.5 * dt * (I1 + I2) / a
        self.Idot = I2
        self.I += dt * I_ramp
        self.t += dt
        Q = 0.5 * (ml1["Q"] + ml2["Q"])
        m, self.H, lost = self._heat(Q, dt)
        self.T = temperature(mat, self.H)
        self.Br, self.Bz, self.E = Br2, Bz2, ml2["E"]
        ml_ev = dict(ml2)
        ml_ev["Q"] = Q
        ret = self._events(dt, Jstar, ml_ev) if geo.n_turns else 0
        self.stats = dict(cg_iters=0, cg_relres=0.0, U_terminal=float(-0.5 * (self.share @ V1 + self.share @ V2)),
                          Tmax=float(self.T.max()), joule_power=float(np.sum(Q * 2.0 * math.pi * geo.r * a)),
                          boundary_energy=lost, heat_substeps=m)
        return int(ret), dt, dt * fac, err

    def _events(self, dt, Jold, ml):
        geo, mat = self.geo, self.mat
        Tmax, Ebar, xmax, rmin = turn_observables(geo, mat, self.T, ml["E"], Jold, ml["Jc"], ml["rho"])
        fl = np.zeros(geo.n_turns, dtype=np.int32)
        fl |= np.where(Tmax > mat.T_fluxjump, FJ_T, 0).astype(np.int32)
        if self.Ebar_prev is not None:
            fl |= np.where((Ebar - self.Ebar_prev) / dt > mat.dEdt_spike, FJ_E, 0).astype(np.int32)
        fl |= np.where(xmax > 1.0, FJ_J, 0).astype(np.int32)
        fl |= np.where(Tmax > mat.Tc, Q_T, 0).astype(np.int32)
        fl |= np.where(rmin > 0.95, Q_RHO, 0).astype(np.int32)
        fj_mask = FJ_T | FJ_E
        rising = ((fl & fj_mask) != 0) & ((self.flags & fj_mask) == 0)
        self.count += rising.astype(np.int32)
        first = (fl != 0) & (self.t_first < 0.0)
        self.t_first[first] = self.t
        fj_all = FJ_T | FJ_E | FJ_J
        self._wire_statistics(dt, ml, Tmax, fl, first)
        started = ((fl & fj_all) != 0) & ((self.flags & fj_all) == 0)
        ret = (RET_FLUXJUMP if np.any(started) else 0) | (RET_QUENCH if np.any(fl & (Q_T | Q_RHO)) else 0)
        self.flags = fl
        self.Ebar_prev = Ebar
        return int(ret)

    def _wire_statistics(self, dt, ml, Tmax, fl, first):
        """Per-wire accumulators after a step (readings of DESIGN.md §3 "f3").

        E_joule  += dt * sum_{i in w} Q_i V_i            Joule energy of the wire [J], V_i = 2 pi r_i a_i
        Q_FJ     += the same, in steps where a flux-jump flag (FJ_T|FJ_E|FJ_J) of the wire is set
        P_max, T_max  running maxima of max_i Q_i [W/m^3] and of the wire's Tmax [K]
        at the first step with a quench flag (Q_T|Q_RHO): t_q, T_q = Tmax_w, P_q = max_i Q_i,
        Q_q = Joule energy from the wire's first event to the quench = E_joule(t_q) - E_joule(before the first event step)
        """
        geo, wr = self.geo, self.wire
        nt, tid = geo.n_turns, geo.turn_id
        Q = ml["Q"]
        dE = dt * np.bincount(tid, weights=Q * 2.0 * math.pi * geo.r * geo.area, minlength=nt)
        Pw = np.zeros(nt)
        np.maximum.at(Pw, tid, Q)
        wr["E_at_first"][first] = wr["E_joule"][first]          # energy before the step of the first event
        wr["E_joule"] += dE
        fj = (fl & (FJ_T | FJ_E | FJ_J)) != 0
        wr["Q_FJ"][fj] += dE[fj]
        wr["P_max"] = np.maximum(wr["P_max"], Pw)
        wr["T_max"] = np.maximum(wr["T_max"], Tmax)
        newq = ((fl & (Q_T | Q_RHO)) != 0) & (wr["t_q"] < 0.0)
        wr["t_q"][newq] = self.t
        wr["T_q"][newq] = Tmax[newq]
        wr["P_q"][newq] = Pw[newq]
        wr["Q_q"][newq] = wr["E_joule"][newq] - wr["E_at_first"][newq]

    # -- config 4 ---------------------------------------------------------------------
    def solve(self, b, tol=None, maxit=None, dense=False):
        """M x = b with no constraint (free rings) or with the geometry's turns and d = 0."""
        geo, mat = self.geo, self.mat
        d = np.zeros(geo.n_turns)
        if dense:
            x, _ = kkt_dense(self.M, constraint_matrix(geo), b, d)
            return x, 0, 0.0
        x, _, it, rel = pcg(self.apply_M, self.diagM, geo.turn_id, geo.n_turns, b, d,
                            mat.cg_tol if tol is None else tol, mat.cg_maxit if maxit is None else maxit)
        return x, it, rel

"""Seeded synthetic inputs for the five BASELINE.json configs.

This module only *describes* problems: ring centres, turn ids, per-cell Jc0
multipliers, scalar parameters, the random vectors of config 4.  It holds none
of the method's arithmetic (no Green's function, no material law, no heat
step), and it is the only code the CPU oracle (``oracle/``) and the CUDA path
(``paper_2403_07666_b200/``) have in common.

Geometry recipe: SURVEY.md §8(c) C1 ("square array" of wires on
the (r, z) cross-section, PAPER.md:69 ``N_x x N_y`` turns).  Seeds and sizes:
SURVEY.md §8(d) workload table, BASELINE.json ``configs``.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np


@dataclasses.dataclass
class Geometry:
    """Mirror of ``qs_geometry`` (include/qs.h); arrays are float64 / int32, host side."""

    r: np.ndarray
    z: np.ndarray
    area: np.ndarray
    turn_id: Optional[np.ndarray]
    n_turns: int
    lattice: int
    layers: int = 0
    turns_per_layer: int = 0
    cells_per_side: int = 0
    wire_size: float = 0.0
    r_inner: float = 0.0
    softening: float = 0.0
    h_conv: tuple = (0.0, 0.0, 0.0, 0.0)   # r_min, r_max, z_min, z_max sides
    T_bath: float = 4.2
    Bext0: float = 0.0
    Bext_rate: float = 0.0
    Bext_max: float = 0.0
    turn_share: Optional[np.ndarray] = None  # [n_turns] share of the transport current per constraint group (NULL = 1)

    @property
    def n_rings(self) -> int:
        return int(self.r.shape[0])

    @property
    def Nr(self) -> int:
        return self.layers * self.cells_per_side

    @property
    def Nz(self) -> int:
        return self.turns_per_layer * self.cells_per_side

    @property
    def h(self) -> float:
        return self.wire_size / self.cells_per_side


@dataclasses.dataclass
class Material:
    """Mirror of ``qs_material`` (include/qs.h).  Defaults = BASELINE.json configs[0]."""

    Ec: float = 1e-4
    n_exp: float = 20.0
    Jc0: float = 2e9
    Tc: float = 18.0
    B0: float = 1.0
    eps_coef: float = 900.0
    eps_exp: float = 1.7
    Y: float = 1e11
    rho_n: float = 5e-10          # SURVEY.md §8(c) C5 [silent]: normal-state cap
    jc0_scale: Optional[np.ndarray] = None
    C3: float = 2000.0
    C1: float = 500.0
    k_in: float = 5.0
    k_between: float = 0.5
    theta: float = 1.0
    cg_tol: float = 1e-10
    cg_maxit: int = 20000
    T_fluxjump: float = 10.0
    dEdt_spike: float = 1.0       # SURVEY.md §8(c) C10 [silent]
    heat_adi_substeps: int = 0    # 0: explicit heat sub-steps (C9); m > 0: m ADI sub-steps per step (C15)


@dataclasses.dataclass
class Workload:
    name: str
    geometry: Geometry
    material: Material
    dt: float
    I_ramp: float
    steps: int
    seed: int


def gmd_factor() -> float:
    """Geometric mean distance of a square from itself, in units of its side.

    ln(g/h) = (2/3) ln sqrt(2) + pi/3 - 25/12  (Maxwell).  This is an
    *input* (the softening length handed to qs_geometry), not part of the operator.
    """
    return math.exp((2.0 / 3.0) * math.log(math.sqrt(2.0)) + math.pi / 3.0 - 25.0 / 12.0)


def lattice_geometry(layers: int, turns_per_layer: int, cells_per_side: int, wire_size: float,
                     r_inner: float, h_conv: float = 500.0, T_bath: float = 4.2,
                     Bext0: float = 0.0, Bext_rate: float = 0.0, Bext_max: float = 0.0) -> Geometry:
    """Regular winding pack, canonical cell order c = ir*Nz + iz."""
    n = cells_per_side
    Nr, Nz = layers * n, turns_per_layer * n
    h = wire_size / n
    ir = np.arange(Nr, dtype=np.int64)[:, None]
    iz = np.arange(Nz, dtype=np.int64)[None, :]
    r = np.broadcast_to(r_inner + (ir + 0.5) * h, (Nr, Nz)).reshape(-1).astype(np.float64)
    z = np.broadcast_to((iz + 0.5) * h - Nz * h / 2.0, (Nr, Nz)).reshape(-1).astype(np.float64)
    turn = ((ir // n) * turns_per_layer + (iz // n)).reshape(-1).astype(np.int32)
    return Geometry(r=np.ascontiguousarray(r), z=np.ascontiguousarray(z),
                    area=np.full(Nr * Nz, h * h, dtype=np.float64), turn_id=turn,
                    n_turns=layers * turns_per_layer, lattice=1, layers=layers,
                    turns_per_layer=turns_per_layer, cells_per_side=n, wire_size=wire_size,
                    r_inner=r_inner, softening=gmd_factor() * h,
                    h_conv=(h_conv, h_conv, h_conv, h_conv), T_bath=T_bath,
                    Bext0=Bext0, Bext_rate=Bext_rate, Bext_max=Bext_max)


def jc0_scale(seed: int, n: int, sigma: float) -> np.ndarray:
    """Median-preserving lognormal Jc0 multiplier per cell."""
    xi = np.random.default_rng(seed).standard_normal(n)
    return np.exp(sigma * xi)


def lattice_workload(name: str, layers: int, turns: int, n: int, wire: float, r_in: float,
                     dt: float, I_ramp: float, steps: int, seed: int, sigma: float,
                     Bext_rate: float = 0.0, Bext_max: float = 0.0, **mat_kw) -> Workload:
    geo = lattice_geometry(layers, turns, n, wire, r_in, Bext_rate=Bext_rate, Bext_max=Bext_max)
    mat = Material(jc0_scale=jc0_scale(seed, geo.n_rings, sigma), **mat_kw)
    return Workload(name=name, geometry=geo, material=mat, dt=dt, I_ramp=I_ramp, steps=steps, seed=seed)


def config(idx: int, **mat_kw) -> Workload:
    """BASELINE.json configs[0..3] at full size."""
    if idx == 0:
        return lattice_workload("cfg0_tiny_solenoid_4x4x8", 4, 4, 8, 1.0e-3, 30e-3, 1e-4, 50.0, 50,
                                1000, 0.01, **mat_kw)
    if idx == 1:
        return lattice_workload("cfg1_single_wire_64x64", 1, 1, 64, 1.0e-3, 30e-3, 5e-5, 0.0, 2000,
                                1001, 0.01, Bext_rate=1.0, Bext_max=3.0, **mat_kw)
    if idx == 2:
        return lattice_workload("cfg2_mid_solenoid_20x40x16", 20, 40, 16, 0.8e-3, 40e-3, 1e-4, 20.0,
                                1000, 1002, 0.02, **mat_kw)
    if idx == 3:
        return lattice_workload("cfg3_real_coil_60x100x12", 60, 100, 12, 0.8e-3, 50e-3, 1e-4, 10.0,
                                5000, 1003, 0.01, **mat_kw)
    raise ValueError("config index must be 0..3 (config 4 = free_rings)")


def shrunk(idx: int, layers: int, turns: int, n: Optional[int] = None, **mat_kw) -> Workload:
    """Same wire, laws, ramp and seed as config ``idx`` on a smaller winding pack (parity cases)."""
    full = config(idx)
    g = full.geometry
    n = n or g.cells_per_side
    sigma = 0.02 if idx == 2 else 0.01
    return lattice_workload(f"cfg{idx}_shrunk_{layers}x{turns}x{n}", layers, turns, n, g.wire_size,
                            g.r_inner, full.dt, full.I_ramp, full.steps, full.seed, sigma,
                            Bext_rate=g.Bext_rate, Bext_max=g.Bext_max, **mat_kw)


def free_rings(n: int, seed: Optional[int] = None):
    """Config 4: random coaxial rings, r in [30, 90] mm, z in [-100, 100] mm, x ~ N(0, 1).

    Every ring is a cell of the mean area h_eff^2 = 0.06*0.2/n and the kernel is softened for
    all pairs with g = gmd*h_eff (free rings).  Returns (Geometry, x).
    """
    if seed is None:
        seed = 4000 + int(round(math.log2(n)))
    g = np.random.default_rng(seed)
    r = g.uniform(0.03, 0.09, n)
    z = g.uniform(-0.1, 0.1, n)
    x = g.standard_normal(n)
    h_eff = math.sqrt(0.06 * 0.2 / n)
    geo = Geometry(r=r, z=z, area=np.full(n, h_eff * h_eff), turn_id=None, n_turns=0, lattice=0,
                   softening=gmd_factor() * h_eff)
    return geo, x


def sample_rows(n: int, count: int, seed: int) -> np.ndarray:
    """Seeded, sorted, distinct target rows for sampled parity at sizes the oracle cannot sweep."""
    g = np.random.default_rng(seed)
    return np.sort(g.choice(n, size=min(count, n), replace=False)).astype(np.int64)


def subelements(geo: Geometry, per_side: int, share: str = "uniform") -> Geometry:
    """The same lattice with every wire cut into per_side x per_side square sub-elements, each a constraint group of its
    own ("each wire has N_sub subelements").  Group id = wire * per_side^2 +
    (row block) * per_side + (column block), in the canonical wire order.  share: "uniform" -> every sub-element
    carries 1/per_side^2 of the wire's transport current; "outer" -> only the sub-elements on the wire's rim carry it
    (equal parts), the inner ones are zero-net-current groups.  Pure index bookkeeping: no method arithmetic."""
    n, s = geo.cells_per_side, int(per_side)
    if not geo.lattice or s <= 0 or n % s:
        raise ValueError("subelements: lattice geometry with cells_per_side divisible by per_side expected")
    Nr, Nz, m = geo.Nr, geo.Nz, n // s
    ir, iz = np.divmod(np.arange(Nr * Nz), Nz)
    wire = (ir // n) * geo.turns_per_layer + iz // n
    br, bz = (ir % n) // m, (iz % n) // m
    gid = (wire * (s * s) + br * s + bz).astype(np.int32)
    n_groups = geo.layers * geo.turns_per_layer * s * s
    kb = np.arange(s * s)
    rim = ((kb // s == 0) | (kb // s == s - 1) | (kb % s == 0) | (kb % s == s - 1)).astype(np.float64)
    if share == "uniform":
        per_wire = np.full(s * s, 1.0 / (s * s))
    elif share == "outer":
        per_wire = rim / rim.sum()
    else:
        raise ValueError("share: 'uniform' or 'outer'")
    return dataclasses.replace(geo, turn_id=gid, n_turns=n_groups,
                               turn_share=np.tile(per_wire, geo.layers * geo.turns_per_layer))

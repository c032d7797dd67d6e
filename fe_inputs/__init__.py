"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds INPUTS only: the paper's coefficient tables (they are arguments of
the method, Table 1), the unit scaling of Table 2 (PAPER.md:102-109,
reading A8 in DESIGN.md), the five BASELINE.json workload descriptors and the seeded
initial states.  It contains none of the method's arithmetic (no Landau polynomial,
no stencil, no tensor, no FFT, no integrator) and imports neither `oracle/` nor the
CUDA package, so both sides can use it without sharing code.

All random numbers come from numpy.random.default_rng(seed) (reading A10).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

EPS0_SI = 8.8541878128e-12

TERM_LANDAU, TERM_GRADIENT, TERM_ELEC, TERM_EXT, TERM_ALL = 1, 2, 4, 8, 15
EULER, HEUN, RK4, AB3M2 = 0, 1, 2, 3


# --------------------------------------------------------------------------------------
# Table 1.  T in kelvin.
# --------------------------------------------------------------------------------------
@dataclass
class Landau:
    """One material's Landau coefficients.  a1 is stored per axis (strain factor r_s,
    PAPER.md:211); the four 8th-order slots are zero for every material of the paper
    (reading A1)."""
    a1: Tuple[float, float, float]
    a11: float = 0.0
    a12: float = 0.0
    a111: float = 0.0
    a112: float = 0.0
    a123: float = 0.0
    a1111: float = 0.0
    a1112: float = 0.0
    a1122: float = 0.0
    a1123: float = 0.0
    active: int = 1

    def as_list(self) -> List[float]:
        return [*self.a1, self.a11, self.a12, self.a111, self.a112, self.a123,
                self.a1111, self.a1112, self.a1122, self.a1123]


@dataclass
class Globals:
    """Per-simulation (batch member) scalars: gradient coefficients (Eq. 4), eps0, epsB
    (Eq. 6), kinetic coefficient L (Eq. 1) and the uniform external field (Eq. 7)."""
    G11: float
    G12: float
    G44: float
    G44p: float
    eps0: float = EPS0_SI
    epsB: float = 1.0
    L: float = 1.0
    E_ext: Tuple[float, float, float] = (0.0, 0.0, 0.0)


VACUUM = Landau(a1=(0.0, 0.0, 0.0), active=0)


def batio3(T: float, r_s: float = 1.0) -> Landau:
    a1 = 3.34e5 * (T - 381.0)
    return Landau(a1=(a1, a1, r_s * a1),
                  a11=4.69e6 * (T - 393.0) - 2.02e8, a12=3.23e8,
                  a111=-5.52e7 * (T - 393.0) + 2.76e9, a112=4.47e9, a123=4.91e9)


def pbtio3(T: float, r_s: float = 1.0) -> Landau:
    a1 = 3.85e5 * (T - 752.0)
    return Landau(a1=(a1, a1, r_s * a1), a11=-7.3e7, a12=7.5e8,
                  a111=2.6e8, a112=6.1e8, a123=-3.7e9)


def srtio3(T: float) -> Landau:
    # reading A7: the printed prefactor "405" has lost 1e5 (eps_r(300 K) = 306 with 4.05e7)
    a1 = 4.05e7 * (1.0 / math.tanh(54.0 / T) - 1.0 / math.tanh(54.0 / 30.0))
    return Landau(a1=(a1, a1, a1), a11=1.7e9, a12=1.37e9)


def wall_2_4_model() -> Landau:
    """alpha1 = -1.7402e8, alpha11 = +1.7402e8, everything else off."""
    return Landau(a1=(-1.7402e8,) * 3, a11=1.7402e8)


BATIO3_G = dict(G11=5.1e-10, G12=-2.0e-11, G44=2.0e-11, G44p=2.0e-11)
PBTIO3_G = dict(G11=1.038e-10, G12=0.0, G44=5.19e-11, G44p=5.19e-11)
WALL_G = dict(G11=0.0, G12=0.0, G44=1.73e-10, G44p=1.73e-10)
G110 = {"BaTiO3": 5.1e-10, "PbTiO3": 1.73e-10}


# --------------------------------------------------------------------------------------
# Table 2 scaling (reading A8).  Pure unit conversion of the inputs.
# --------------------------------------------------------------------------------------
@dataclass
class Units:
    alpha_ref: float       # |alpha1| of the reference material
    P0: float              # C/m^2
    G110: float

    @property
    def l0(self) -> float:
        return math.sqrt(self.G110 / self.alpha_ref)

    def landau(self, m: Landau) -> Landau:
        a, p2 = self.alpha_ref, self.P0 ** 2
        return Landau(a1=tuple(x / a for x in m.a1),
                      a11=m.a11 * p2 / a, a12=m.a12 * p2 / a,
                      a111=m.a111 * p2 ** 2 / a, a112=m.a112 * p2 ** 2 / a,
                      a123=m.a123 * p2 ** 2 / a,
                      a1111=m.a1111 * p2 ** 3 / a, a1112=m.a1112 * p2 ** 3 / a,
                      a1122=m.a1122 * p2 ** 3 / a, a1123=m.a1123 * p2 ** 3 / a,
                      active=m.active)

    def globals(self, g: Globals) -> Globals:
        s = self.alpha_ref * self.P0
        return Globals(G11=g.G11 / self.G110, G12=g.G12 / self.G110,
                       G44=g.G44 / self.G110, G44p=g.G44p / self.G110,
                       eps0=g.eps0 * self.alpha_ref, epsB=g.epsB, L=1.0,
                       E_ext=tuple(e / s for e in g.E_ext))

    def length(self, x: float) -> float:
        return x / self.l0

    def field(self, e: float) -> float:
        return e / (self.alpha_ref * self.P0)


# --------------------------------------------------------------------------------------
# Workload descriptor
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    n: Tuple[int, int, int]                    # nx, ny, nz
    d: Tuple[float, float, float]              # cell size (reduced or SI)
    periodic: Tuple[int, int, int]
    pbc_images: Tuple[int, int, int]
    batch: int
    dtype: str                                 # "f64" | "f32"
    materials: List[List[Landau]]              # [member][material id]
    globals_: List[Globals]                    # [member]
    matmap: Optional[np.ndarray]               # uint8 [nz][ny][nx] or None
    P0: np.ndarray                             # float64 [B][3][nz][ny][nx]
    dt: float
    integrator: int
    terms: int = TERM_ALL
    nsteps: int = 100
    notes: str = ""

    @property
    def cells(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]


def sphere_uniform(rng: np.random.Generator, shape: Sequence[int], radius: float) -> np.ndarray:
    """Random directions uniform on the sphere (three normals, normalised), |P| = radius.
    Returns [3, *shape]."""
    v = rng.standard_normal((3, *shape))
    v /= np.sqrt((v ** 2).sum(axis=0, keepdims=True))
    return radius * v


def _bto_units(T: float = 300.0) -> Units:
    return Units(alpha_ref=abs(batio3(T).a1[0]), P0=0.26, G110=G110["BaTiO3"])


def _pto_units(T: float = 300.0) -> Units:
    return Units(alpha_ref=abs(pbtio3(T).a1[0]), P0=0.757, G110=G110["PbTiO3"])


def open_batio3(name: str, n: Tuple[int, int, int], batch: int, dtype: str, seed: int,
                nsteps: int = 100, dt: float = 0.002) -> Workload:
    """Configs 1 and 5 (BASELINE.json): open boundaries, 1 nm cubic cells, BaTiO3 Table 1 at
    300 K, epsB = 45, P = 0.26 C/m^2 times a sphere-uniform direction,
    forward Euler, reduced units (A8)."""
    u = _bto_units()
    nx, ny, nz = n
    P = np.stack([sphere_uniform(np.random.default_rng(seed + b), (nz, ny, nx), 0.26 / u.P0)
                  for b in range(batch)])
    g = u.globals(Globals(**BATIO3_G, epsB=45.0))
    h = u.length(1e-9)
    return Workload(name=name, n=n, d=(h, h, h), periodic=(0, 0, 0), pbc_images=(0, 0, 0),
                    batch=batch, dtype=dtype, materials=[[u.landau(batio3(300.0))] for _ in range(batch)],
                    globals_=[replace(g) for _ in range(batch)], matmap=None, P0=P, dt=dt,
                    integrator=EULER, nsteps=nsteps)


def config1() -> Workload:
    return open_batio3("cfg1_tiny_16x16x8", (16, 16, 8), 1, "f64", 1001)


def config5a(dtype: str = "f64") -> Workload:
    return open_batio3("cfg5a_256x256x128", (256, 256, 128), 1, dtype, 1005, nsteps=1000)


def config5b(dtype: str = "f64") -> Workload:
    return open_batio3("cfg5b_128x128x64_b4", (128, 128, 64), 4, dtype, 1005, nsteps=1000)


def config2(nx: int = 512, variant: str = "2a", cell_nm: float = 0.5, pbc_images: int = 10,
            elec: bool = False) -> Workload:
    """180-degree wall (BASELINE.json config 2, reading A11).  2a = the paper's own 2-4 parameter
    set; Pz(x) wall, periodic y,z, open x."""
    if variant == "2a":
        mat, G = wall_2_4_model(), WALL_G
        u = Units(alpha_ref=1.7402e8, P0=math.sqrt(0.5), G110=G110["PbTiO3"])
        Ps = math.sqrt(0.5)
    else:
        mat, G = pbtio3(300.0), PBTIO3_G
        u = _pto_units()
        Ps = math.sqrt(0.57511)
    ny = nz = 4
    rng = np.random.default_rng(1002)
    x = np.arange(nx, dtype=np.float64)
    x0, w0 = (nx - 1) / 2.0, 2.0
    P = np.zeros((1, 3, nz, ny, nx))
    P[0, 2] = (Ps / u.P0) * np.tanh((x - x0) / w0)[None, None, :]
    P[0] += rng.uniform(-1e-3, 1e-3, size=(3, nz, ny, nx)) * (Ps / u.P0)
    g = u.globals(Globals(**G, epsB=45.0))
    h = u.length(cell_nm * 1e-9)
    terms = TERM_LANDAU | TERM_GRADIENT | (TERM_ELEC if elec else 0)
    return Workload(name=f"cfg{variant}_wall_{nx}x4x4", n=(nx, ny, nz), d=(h, h, h),
                    periodic=(0, 1, 1), pbc_images=(0, pbc_images, pbc_images), batch=1, dtype="f64",
                    materials=[[u.landau(mat)]], globals_=[g], matmap=None, P0=P, dt=0.02,
                    integrator=RK4, terms=terms, nsteps=20000)


def config3_temperatures() -> List[float]:
    return [150.0 + 20.0 * j for j in range(16)]


def config3(n: int = 64, batch: int = 16) -> Workload:
    """BaTiO3 temperature sweep (config 3, reading A12): member b starts at T_b = 150 + 20 b."""
    u = _bto_units()
    Ts = config3_temperatures()
    P = np.stack([np.random.default_rng(1003 + b).normal(0.0, 0.01 / u.P0, size=(3, n, n, n))
                  for b in range(batch)])
    g = u.globals(Globals(**BATIO3_G, epsB=45.0))
    h = u.length(1e-9)
    return Workload(name=f"cfg3_sweep_{n}^3_b{batch}", n=(n, n, n), d=(h, h, h), periodic=(0, 0, 0),
                    pbc_images=(0, 0, 0), batch=batch, dtype="f64",
                    materials=[[u.landau(batio3(Ts[b % 16]))] for b in range(batch)],
                    globals_=[replace(g) for _ in range(batch)], matmap=None, P0=P, dt=0.002,
                    integrator=EULER, nsteps=5000)


def config3_leg_temperature(member: int, leg: int) -> float:
    m = (member + leg) % 30
    return config3_temperatures()[m if m <= 15 else 30 - m]


def skyrmion_texture(nx: int, ny: int, cell_nm: float, R0_nm: float = 10.0, w_nm: float = 2.0) -> np.ndarray:
    """Seeded-free analytic Neel texture (A13): [3][ny][nx] unit vectors."""
    yy, xx = np.meshgrid((np.arange(ny) - (ny - 1) / 2) * cell_nm, (np.arange(nx) - (nx - 1) / 2) * cell_nm,
                         indexing="ij")
    rho = np.hypot(xx, yy)
    phi = np.arctan2(yy, xx)
    theta = 2.0 * np.arctan2(np.sinh(R0_nm / w_nm), np.sinh(rho / w_nm))
    return np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])


def config4(nxy: int = 128, nz: int = 32, pbc_images: int = 10, skyrmion: bool = False) -> Workload:
    """PbTiO3 on SrTiO3 bilayer (config 4, reading A13): z-layers [0, nz/2) SrTiO3 (material 1),
    [nz/2, nz) PbTiO3 (material 0); periodic x,y, open z; epsB = 649."""
    u = _pto_units()
    Ps = 0.7584 / u.P0
    matmap = np.zeros((nz, nxy, nxy), dtype=np.uint8)
    matmap[: nz // 2] = 1
    P = np.zeros((1, 3, nz, nxy, nxy))
    if skyrmion:
        P[0, :, nz // 2:] = Ps * skyrmion_texture(nxy, nxy, 1.0)[:, None]
    else:
        P[0, :, nz // 2:] = sphere_uniform(np.random.default_rng(1004), (nz - nz // 2, nxy, nxy), Ps)
    g = u.globals(Globals(**PBTIO3_G, epsB=649.0))
    h = u.length(1e-9)
    return Workload(name=f"cfg4_bilayer_{nxy}x{nxy}x{nz}", n=(nxy, nxy, nz), d=(h, h, h),
                    periodic=(1, 1, 0), pbc_images=(pbc_images, pbc_images, 0), batch=1, dtype="f64",
                    materials=[[u.landau(pbtio3(300.0)), u.landau(srtio3(300.0))]], globals_=[g],
                    matmap=matmap, P0=P, dt=0.02, integrator=EULER, nsteps=500,
                    notes="field sweep: config4_field(k)")


def config4_paper(nxy: int = 128, seed: int = 1004) -> Workload:
    """The paper's own bilayer geometry: 128 x 128 x 36 cells of 1 nm, from the bottom 12 nm SrTiO3
    (material 1), 20 nm PbTiO3 (material 0), 4 nm vacuum (material 2), open boundaries on all axes ("finite samples
    embedded in vacuum"), epsB = 649.  BASELINE.json's config 4 is the periodic 128 x 128 x 32 variant."""
    u = _pto_units()
    Ps = 0.7584 / u.P0
    nz = 36
    matmap = np.full((nz, nxy, nxy), 2, dtype=np.uint8)
    matmap[:12] = 1
    matmap[12:32] = 0
    P = np.zeros((1, 3, nz, nxy, nxy))
    P[0, :, 12:32] = sphere_uniform(np.random.default_rng(seed), (20, nxy, nxy), Ps)
    g = u.globals(Globals(**PBTIO3_G, epsB=649.0))
    h = u.length(1e-9)
    return Workload(name=f"cfg4_paper_{nxy}x{nxy}x{nz}", n=(nxy, nxy, nz), d=(h, h, h), periodic=(0, 0, 0),
                    pbc_images=(0, 0, 0), batch=1, dtype="f64",
                    materials=[[u.landau(pbtio3(300.0)), u.landau(srtio3(300.0)), VACUUM]], globals_=[g],
                    matmap=matmap, P0=P, dt=0.02, integrator=EULER, nsteps=500)


def config4_field(k: int, npoints: int = 200, amp: float = 1e8) -> float:
    """Triangular sweep 0 -> +amp -> -amp -> 0 over npoints (SI V/m)."""
    q = npoints // 4
    if k <= q:
        return amp * k / q
    if k <= 3 * q:
        return amp * (2.0 - k / q)
    return amp * (k / q - 4.0)


def config4_field_reduced(k: int) -> float:
    return _pto_units().field(config4_field(k))


def strain_bilayer(nxy: int = 16, n_pto: int = 8, n_sto: int = 2, margin: int = 2, cell_nm: float = 0.5,
                   r_s: float = 1.0, seed: int = 1007) -> Workload:
    """PbTiO3 on SrTiO3 island surrounded by vacuum (Sec. 4.4): open boundaries, material map with
    ids 0 = PbTiO3 (alpha_1z scaled by the strain parameter r_s), 1 = SrTiO3, 2 = vacuum (margin cells on
    every side), the paper's gradient coefficients for this study (G11 = 3.46e-10, G12 = 0, G44 = G44' = 1.73e-10),
    0.5 nm cells, 300 K, epsB = 649, random initial polarisation in PbTiO3 for r_s = 1."""
    u = _pto_units()
    nx = ny = nxy + 2 * margin
    nz = n_pto + n_sto + 2 * margin
    matmap = np.full((nz, ny, nx), 2, dtype=np.uint8)
    matmap[margin:margin + n_sto, margin:-margin, margin:-margin] = 1
    matmap[margin + n_sto:margin + n_sto + n_pto, margin:-margin, margin:-margin] = 0
    P = np.zeros((1, 3, nz, ny, nx))
    rnd = sphere_uniform(np.random.default_rng(seed), (nz, ny, nx), 0.7584 / u.P0)
    P[0] = rnd * (matmap == 0)[None]
    g = u.globals(Globals(G11=3.46e-10, G12=0.0, G44=1.73e-10, G44p=1.73e-10, epsB=649.0))
    h = u.length(cell_nm * 1e-9)
    return Workload(name=f"strain_bilayer_{nx}x{ny}x{nz}_rs{r_s:g}", n=(nx, ny, nz), d=(h, h, h), periodic=(0, 0, 0),
                    pbc_images=(0, 0, 0), batch=1, dtype="f64",
                    materials=[[u.landau(pbtio3(300.0, r_s)), u.landau(srtio3(300.0)), VACUUM]], globals_=[g],
                    matmap=matmap, P0=P, dt=0.005, integrator=EULER, nsteps=2000,
                    notes="strain sweep: set material 0 to Units.landau(pbtio3(300, r_s)) per leg, state carries over")


def landau_ensemble(temperatures: Sequence[float] = tuple(10.0 * j for j in range(37)),
                    n: Tuple[int, int, int] = (16, 16, 8), seed: int = 1006) -> Workload:
    """Landau-only ensemble (Fig. 2): one batch member per temperature
    (T = 0 ... 360 K), every cell an independent single-cell relaxation (gradient, electrostatic and external terms
    off) from a random orientation of magnitude 1e-3 C/m^2; 16x16x8 = 2048 starts per temperature
    stand in for the paper's 1500.  Reduced units of BaTiO3 at 300 K for every member (the geometry is shared)."""
    u = _bto_units()
    nx, ny, nz = n
    B = len(temperatures)
    P = np.stack([sphere_uniform(np.random.default_rng(seed + b), (nz, ny, nx), 1e-3 / u.P0) for b in range(B)])
    g = u.globals(Globals(**BATIO3_G, epsB=45.0))
    h = u.length(1e-9)
    return Workload(name=f"landau_ensemble_{B}T_{nx * ny * nz}starts", n=n, d=(h, h, h), periodic=(0, 0, 0),
                    pbc_images=(0, 0, 0), batch=B, dtype="f64",
                    materials=[[u.landau(batio3(float(T)))] for T in temperatures],
                    globals_=[replace(g) for _ in range(B)], matmap=None, P0=P, dt=0.02, integrator=RK4,
                    terms=TERM_LANDAU, nsteps=30000, notes="temperatures: " + ",".join("%g" % T for T in temperatures))


def random_problem(seed: int, n=(6, 5, 4), periodic=(0, 1, 0), pbc_images=(0, 2, 0), n_materials: int = 3,
                   with_vacuum: bool = True, eighth: bool = True):
    """A small heterogeneous problem in O(1) units for the pins (P1, P9): random coefficients
    (non-zero 8th-order slots), Gm != 0, 3 materials incl. vacuum, E_ext != 0."""
    rng = np.random.default_rng(seed)
    mats = []
    for m in range(n_materials):
        if with_vacuum and m == n_materials - 1:
            mats.append(VACUUM)
            continue
        c = rng.uniform(0.5, 1.5, size=12)
        mats.append(Landau(a1=(-c[0], -1.1 * c[1], -0.9 * c[2]), a11=c[3], a12=0.7 * c[4], a111=c[5],
                           a112=0.6 * c[6], a123=-0.8 * c[7],
                           a1111=c[8] if eighth else 0.0, a1112=0.3 * c[9] if eighth else 0.0,
                           a1122=0.4 * c[10] if eighth else 0.0, a1123=0.2 * c[11] if eighth else 0.0))
    nx, ny, nz = n
    matmap = rng.integers(0, n_materials, size=(nz, ny, nx)).astype(np.uint8)
    g = Globals(G11=0.9, G12=-0.15, G44=0.2, G44p=0.3, eps0=0.7, epsB=1.3, L=0.8,
                E_ext=(0.05, -0.02, 0.03))
    P = rng.uniform(-0.8, 0.8, size=(3, nz, ny, nx))
    active = np.array([mm.active for mm in mats])[matmap]
    P *= active[None]
    d = (0.9, 1.1, 0.7)
    return dict(n=n, d=d, periodic=periodic, pbc_images=pbc_images, materials=mats, globals_=g,
                matmap=matmap, P=P)

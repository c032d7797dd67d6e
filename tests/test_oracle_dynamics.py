"""Pins for the oracle's gradient term (O2), RHS (O5), integrators (O6) and energy (O7).

P1  RHS = -(L/V) dF_h/dP against central differences of the total discrete energy.
P7  180-degree wall: plateau, width and first integral of PAPER.md:131-141 (Eq. 8-10).
P8  energy decreases monotonically under Euler relaxation (gradient flow).
P9  symmetries.   P11 integrator orders.
"""
import functools
import math

import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc


def _make(seed=1, **kw):
    q = fi.random_problem(seed, **kw)
    p = orc.Problem(n=q["n"], d=q["d"], periodic=q["periodic"], pbc_images=q["pbc_images"],
                    materials=q["materials"], g=q["globals_"], matmap=q["matmap"])
    return p, q["P"]


@pytest.mark.parametrize("periodic,images", [((0, 1, 0), (0, 2, 0)), ((0, 0, 0), (0, 0, 0)), ((1, 1, 0), (1, 1, 0))])
def test_P1_rhs_is_the_gradient_of_the_discrete_energy(periodic, images):
    p, P = _make(seed=21, n=(6, 5, 4), periodic=periodic, pbc_images=images)
    o = orc.Oracle(p)
    rhs = o.rhs(P)
    F = lambda Q: o.energy(Q)[4]
    rng = np.random.default_rng(0)
    h = 1e-5
    act = np.argwhere(p.active > 0)
    checked = 0
    for _ in range(40):
        z, y, x = act[rng.integers(len(act))]
        i = int(rng.integers(3))
        e = np.zeros_like(P)
        e[i, z, y, x] = h
        fd = (F(P + e) - F(P - e)) / (2 * h)
        want = -p.V * rhs[i, z, y, x] / p.g.L
        assert fd == pytest.approx(want, rel=2e-7, abs=1e-8), (i, z, y, x)
        checked += 1
    assert checked == 40
    # vacuum cells do not move
    assert np.all(rhs[:, p.active == 0] == 0.0)


def test_P1_each_term_alone():
    p, P = _make(seed=22, n=(5, 4, 3), periodic=(1, 0, 0), pbc_images=(2, 0, 0))
    o = orc.Oracle(p)
    h = 1e-5
    rng = np.random.default_rng(1)
    act = np.argwhere(p.active > 0)
    for term, slot in [(orc.TERM_LANDAU, 0), (orc.TERM_GRADIENT, 1), (orc.TERM_ELEC, 2), (orc.TERM_EXT, 3)]:
        rhs = o.rhs(P, term)
        for _ in range(8):
            z, y, x = act[rng.integers(len(act))]
            i = int(rng.integers(3))
            e = np.zeros_like(P)
            e[i, z, y, x] = h
            fd = (o.energy(P + e, term)[slot] - o.energy(P - e, term)[slot]) / (2 * h)
            assert fd == pytest.approx(-p.V * rhs[i, z, y, x] / p.g.L, rel=2e-7, abs=1e-8), (term, i)


def test_gradient_quadratic_form_identity_and_bulk_laplacian():
    """F_Grad,h = -1/2 V sum P.E_Grad (quadratic form), and in the bulk of a homogeneous grid
    E_Grad,x = G11 dxx Px + (G44+G44')(dyy+dzz) Px + Gm (dxdy Py + dxdz Pz) applied to a quadratic
    polynomial is exact."""
    p, P = _make(seed=23, n=(6, 5, 4), periodic=(0, 1, 0), pbc_images=(0, 1, 0))
    assert orc.grad_energy(p, P) == pytest.approx(-0.5 * p.V * np.sum(P * orc.grad_field(p, P)), rel=1e-13)

    g = fi.Globals(G11=0.9, G12=-0.15, G44=0.2, G44p=0.3)
    n, d = (7, 6, 5), (0.5, 0.8, 1.25)
    q = orc.Problem(n=n, d=d, periodic=(0, 0, 0), pbc_images=(0, 0, 0), materials=[fi.Landau(a1=(0, 0, 0))], g=g)
    z, y, x = np.meshgrid(np.arange(n[2]) * d[2], np.arange(n[1]) * d[1], np.arange(n[0]) * d[0], indexing="ij")
    Px = 0.3 * x * x + 0.1 * y * y - 0.2 * z * z + 0.05 * x * y
    Py = 0.7 * x * y + 0.2 * y * z - 0.4 * x * x
    Pz = -0.6 * x * z + 0.5 * y * z + 0.25 * z * z
    E = orc.grad_field(q, np.stack([Px, Py, Pz]))
    Gm = g.G12 + g.G44 - g.G44p
    c = g.G44 + g.G44p
    ex = g.G11 * 0.6 + c * (0.2 - 0.4) + Gm * (0.7 - 0.6)
    ey = g.G11 * 0.0 + c * (-0.8 + 0.0) + Gm * (0.05 + 0.5)
    ez = g.G11 * 0.5 + c * (0.0 + 0.0) + Gm * (0.0 + 0.2)
    inner = (slice(1, -1),) * 3
    np.testing.assert_allclose(E[0][inner], ex, rtol=1e-11)
    np.testing.assert_allclose(E[1][inner], ey, rtol=1e-11)
    np.testing.assert_allclose(E[2][inner], ez, rtol=1e-11)


def test_gradient_free_surface_and_uniform_state():
    """Neumann surfaces: a uniform P has zero squared-term field everywhere; the mixed term with zero
    exterior acts only in boundary cells."""
    g0 = fi.Globals(G11=0.9, G12=0.1, G44=0.2, G44p=0.3)            # Gm = 0
    q = orc.Problem(n=(5, 4, 3), d=(1, 1, 1), periodic=(0, 0, 0), pbc_images=(0, 0, 0),
                    materials=[fi.Landau(a1=(0, 0, 0))], g=g0)
    P = np.ones(q.shape) * np.array([0.3, -0.2, 0.5])[:, None, None, None]
    np.testing.assert_allclose(orc.grad_field(q, P), 0.0, atol=1e-15)
    g1 = fi.Globals(G11=0.9, G12=-0.15, G44=0.2, G44p=0.3)          # Gm != 0
    q1 = orc.Problem(n=(5, 4, 3), d=(1, 1, 1), periodic=(0, 0, 0), pbc_images=(0, 0, 0),
                     materials=[fi.Landau(a1=(0, 0, 0))], g=g1)
    E = orc.grad_field(q1, P)
    np.testing.assert_allclose(E[:, 1:-1, 1:-1, 1:-1], 0.0, atol=1e-15)
    assert np.abs(E).max() > 1e-3


def _wall_problem(nx, cell_nm):
    u = fi.Units(alpha_ref=1.7402e8, P0=math.sqrt(0.5), G110=1.73e-10)
    m = u.landau(fi.wall_2_4_model())
    g = u.globals(fi.Globals(**fi.WALL_G))
    h = u.length(cell_nm * 1e-9)
    return u, orc.Problem(n=(nx, 1, 1), d=(h, h, h), periodic=(0, 0, 0), pbc_images=(0, 0, 0), materials=[m], g=g)


@functools.lru_cache(maxsize=None)
def _relaxed_wall(nx, cell_nm):
    u, p = _wall_problem(nx, cell_nm)
    o = orc.Oracle(p)
    x = np.arange(nx)
    P = np.zeros(p.shape)
    P[2, 0, 0] = np.tanh((x - (nx - 1) / 2) / 2.0)
    P += 1e-3 * np.random.default_rng(1002).uniform(-1, 1, size=p.shape)
    terms = orc.TERM_LANDAU | orc.TERM_GRADIENT
    dt = 0.02 * (cell_nm / 0.5) ** 2
    P = o.step(P, dt=dt, nsteps=int(120 / dt), integrator=orc.RK4, terms=terms)
    return u, p, o, P, terms


@pytest.mark.parametrize("cell_nm,tol", [(0.5, 0.02), (0.25, 0.005)])
def test_P7_wall_profile_matches_paper_eq10(cell_nm, tol, golden):
    gold = golden("wall_180_paper.txt")
    nx = 128 if cell_nm == 0.5 else 256
    u, p, o, P, terms = _relaxed_wall(nx, cell_nm)
    Pz = P[2, 0, 0] * u.P0                                   # back to C/m^2
    # discrete stationarity of the wall component.  (With alpha12 = 0 the components of the 2-4 model
    # decouple, PAPER.md:129 'a single component'; the seeded noise in Px, Py coarsens on its own.)
    assert np.max(np.abs(o.rhs(P, terms)[2])) < 1e-8
    assert abs(Pz[2]) == pytest.approx(gold["P_plateau"], abs=1e-6)
    assert abs(Pz[-3]) == pytest.approx(gold["P_plateau"], abs=1e-6)
    xs = np.arange(nx) * cell_nm * 1e-9
    core = np.abs(Pz / gold["P_plateau"]) < 0.9
    slope, _ = np.polyfit(xs[core], np.arctanh(Pz[core] / gold["P_plateau"]), 1)
    assert 1.0 / slope == pytest.approx(gold["xi_m"], rel=tol)


def test_P7_width_converges_second_order():
    gold_xi = 1.4100590e-9
    errs = []
    for cell_nm, nx in [(0.5, 128), (0.25, 256)]:
        u, p, o, P, _ = _relaxed_wall(nx, cell_nm)
        Pz = P[2, 0, 0]
        xs = np.arange(nx) * cell_nm * 1e-9
        core = np.abs(Pz) < 0.9
        slope, _ = np.polyfit(xs[core], np.arctanh(Pz[core]), 1)
        errs.append(abs(1.0 / slope - gold_xi))
    assert 2.5 < errs[0] / errs[1] < 6.0


def test_P8_energy_decreases_monotonically_under_euler():
    u = fi.Units(alpha_ref=abs(fi.batio3(300.0).a1[0]), P0=0.26, G110=5.1e-10)
    h = u.length(1e-9)
    g = u.globals(fi.Globals(**fi.BATIO3_G, epsB=45.0, E_ext=(0.0, 0.0, 2e6)))
    p = orc.Problem(n=(8, 8, 4), d=(h, h, h), periodic=(0, 0, 0), pbc_images=(0, 0, 0),
                    materials=[u.landau(fi.batio3(300.0))], g=g)
    o = orc.Oracle(p)
    P = fi.sphere_uniform(np.random.default_rng(8), (4, 8, 8), 1.0)
    F = [o.energy(P)[4]]
    for _ in range(60):
        P = o.step(P, dt=0.002, nsteps=1, integrator=orc.EULER)
        F.append(o.energy(P)[4])
    F = np.array(F)
    assert np.all(np.diff(F) <= 1e-13 * np.abs(F[:-1]))
    assert F[-1] < F[0] - 0.01 * abs(F[0])


def test_P9_symmetries():
    g = fi.Globals(G11=0.9, G12=-0.15, G44=0.2, G44p=0.3, eps0=0.7, epsB=1.3, L=0.8)
    m = fi.random_problem(5, n_materials=1, with_vacuum=False)["materials"][0]
    m = fi.Landau(a1=(m.a1[0],) * 3, a11=m.a11, a12=m.a12, a111=m.a111, a112=m.a112, a123=m.a123,
                  a1111=m.a1111, a1112=m.a1112, a1122=m.a1122, a1123=m.a1123)
    n = (4, 4, 4)
    p = orc.Problem(n=n, d=(1, 1, 1), periodic=(0, 0, 0), pbc_images=(0, 0, 0), materials=[m], g=g)
    o = orc.Oracle(p)
    P = np.random.default_rng(9).uniform(-0.8, 0.8, size=p.shape)
    terms = orc.TERM_LANDAU | orc.TERM_GRADIENT | orc.TERM_ELEC
    R = o.rhs(P, terms)
    np.testing.assert_allclose(o.rhs(-P, terms), -R, rtol=0, atol=1e-14 * np.abs(R).max())
    # swap x <-> y: components (Py,Px,Pz) on the transposed grid
    Q = P[[1, 0, 2]].transpose(0, 1, 3, 2)
    RQ = o.rhs(np.ascontiguousarray(Q), terms)
    np.testing.assert_allclose(RQ, R[[1, 0, 2]].transpose(0, 1, 3, 2), rtol=0, atol=1e-13 * np.abs(R).max())
    # cyclic x->y->z->x
    Q = P[[2, 0, 1]].transpose(0, 2, 3, 1)
    RQ = o.rhs(np.ascontiguousarray(Q), terms)
    np.testing.assert_allclose(RQ, R[[2, 0, 1]].transpose(0, 2, 3, 1), rtol=0, atol=1e-13 * np.abs(R).max())
    # translation along a periodic axis commutes with the RHS
    pp = orc.Problem(n=n, d=(1, 1, 1), periodic=(0, 1, 0), pbc_images=(0, 2, 0), materials=[m], g=g)
    op = orc.Oracle(pp)
    Rp = op.rhs(P, terms)
    np.testing.assert_allclose(op.rhs(np.roll(P, 1, axis=2), terms), np.roll(Rp, 1, axis=2), rtol=0,
                               atol=1e-13 * np.abs(Rp).max())


def test_P11_integrator_orders():
    p, P0 = _make(seed=31, n=(4, 4, 2), periodic=(0, 0, 0), pbc_images=(0, 0, 0), with_vacuum=False, n_materials=2)
    o = orc.Oracle(p)
    T = 0.02
    ref = o.step(P0, dt=T / 512, nsteps=512, integrator=orc.RK4)
    for integ, order in [(orc.EULER, 1), (orc.HEUN, 2), (orc.RK4, 4)]:
        errs = []
        for ns in (8, 16):
            errs.append(np.linalg.norm(o.step(P0, dt=T / ns, nsteps=ns, integrator=integ) - ref))
        ratio = errs[0] / errs[1]
        assert 2 ** order * 0.85 < ratio < 2 ** order * 1.15, (integ, ratio)


def test_energy_terms_written_out():
    """F_Ext = -V sum E_ext . P (Eq. 7), F_Elec = -1/2 V sum E_elec . P (Eq. 5), means over active cells."""
    p, P = _make(seed=41, n=(4, 3, 3), periodic=(0, 0, 0), pbc_images=(0, 0, 0))
    o = orc.Oracle(p)
    e = o.energy(P)
    assert e[3] == pytest.approx(-p.V * sum(p.g.E_ext[i] * P[i].sum() for i in range(3)), rel=1e-14)
    Ee = orc.field_direct(p, o.table(), P)
    assert e[2] == pytest.approx(-0.5 * p.V * np.sum(Ee * P), rel=1e-14)
    assert e[4] == pytest.approx(e[0] + e[1] + e[2] + e[3], rel=1e-14)
    na = p.active.sum()
    assert e[5] == pytest.approx(P[0][p.active > 0].sum() / na, rel=1e-14)

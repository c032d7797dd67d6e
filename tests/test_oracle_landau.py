"""Pins for the oracle's Landau term (O1): PAPER.md:41-47 (Eq. 3), Table 1.

P1 (Landau part): analytic df/dP against central differences of f, twelve random coefficients.
P3: relaxation of one cell lands on the closed-form T / O / R stationary points
    and the phase ordering the paper states at 300 / 250 / 150 K.
"""
import math

import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc


def _closed_forms(m):
    a1 = m.a1[0]
    pT = (-m.a11 + math.sqrt(m.a11 ** 2 - 3 * a1 * m.a111)) / (3 * m.a111)
    A, B = 2 * m.a11 + m.a12, m.a111 + m.a112
    pO = (-A + math.sqrt(A * A - 12 * a1 * B)) / (6 * B)
    A3, B3 = m.a11 + m.a12, 3 * m.a111 + 6 * m.a112 + m.a123
    pR = (-A3 + math.sqrt(A3 * A3 - a1 * B3)) / B3
    return dict(T=np.array([math.sqrt(pT), 0, 0]), O=np.array([math.sqrt(pO)] * 2 + [0.0]),
                R=np.array([math.sqrt(pR)] * 3))


def test_P1_landau_derivative_vs_finite_difference():
    rng = np.random.default_rng(7)
    for trial in range(20):
        c = rng.uniform(-1.0, 1.0, size=12)
        m = fi.Landau(a1=tuple(c[:3]), a11=c[3], a12=c[4], a111=c[5], a112=c[6], a123=c[7],
                      a1111=c[8], a1112=c[9], a1122=c[10], a1123=c[11])
        P = rng.uniform(-1.2, 1.2, size=3)
        g = orc.landau_dfdp(m, P)
        h = 1e-5
        for i in range(3):
            e = np.zeros(3)
            e[i] = h
            # 4th-order central difference
            fd = (-orc.landau_f(m, P + 2 * e) + 8 * orc.landau_f(m, P + e)
                  - 8 * orc.landau_f(m, P - e) + orc.landau_f(m, P - 2 * e)) / (12 * h)
            assert abs(fd - g[i]) <= 1e-9 * max(1.0, abs(g[i])), (trial, i, fd, g[i])


def test_landau_each_coefficient_alone_is_homogeneous():
    """Euler's theorem: a term of degree 2k in P obeys P . df/dP = 2k f; checks every slot's
    power and its cyclic structure separately (a dropped or mis-powered term fails)."""
    rng = np.random.default_rng(11)
    P = rng.uniform(0.3, 1.1, size=3)
    slots = [("a11", 4), ("a12", 4), ("a111", 6), ("a112", 6), ("a123", 6), ("a1111", 8), ("a1112", 8),
             ("a1122", 8), ("a1123", 8)]
    for name, deg in slots:
        m = fi.Landau(a1=(0.0, 0.0, 0.0), **{name: 1.7})
        f = orc.landau_f(m, P)
        assert f != 0.0
        assert np.dot(P, orc.landau_dfdp(m, P)) == pytest.approx(deg * f, rel=1e-13)
        # cubic symmetry: permuting the components leaves f unchanged
        assert orc.landau_f(m, P[[1, 2, 0]]) == pytest.approx(f, rel=1e-14)
        assert orc.landau_f(m, P[[1, 0, 2]]) == pytest.approx(f, rel=1e-14)
    m = fi.Landau(a1=(1.0, 2.0, 3.0))
    assert orc.landau_f(m, P) == pytest.approx(P[0] ** 2 + 2 * P[1] ** 2 + 3 * P[2] ** 2, rel=1e-14)


def test_landau_special_values_written_out():
    """Eq. 3 by hand at P = (1,2,3) with unit coefficients, slot by slot."""
    P = np.array([1.0, 2.0, 3.0])
    a, b, c = 1.0, 4.0, 9.0
    expect = dict(a11=a * a + b * b + c * c, a12=a * b + b * c + c * a, a111=a ** 3 + b ** 3 + c ** 3,
                  a112=a * a * (b + c) + b * b * (a + c) + c * c * (a + b), a123=a * b * c,
                  a1111=a ** 4 + b ** 4 + c ** 4,
                  a1112=a ** 3 * (b + c) + b ** 3 * (a + c) + c ** 3 * (a + b),
                  a1122=a * a * b * b + b * b * c * c + c * c * a * a, a1123=a * b * c * (a + b + c))
    for k, v in expect.items():
        assert orc.landau_f(fi.Landau(a1=(0, 0, 0), **{k: 1.0}), P) == pytest.approx(v, rel=1e-15)


@pytest.mark.parametrize("T", [300.0, 250.0, 150.0])
def test_P3_closed_form_stationary_points_and_golden(T, golden):
    g = golden("batio3_phases.txt")
    m = fi.batio3(T)
    cf = _closed_forms(m)
    F = {}
    for ph, P in cf.items():
        # stationary: df/dP = 0 at the closed form
        assert np.max(np.abs(orc.landau_dfdp(m, P))) <= 1e-7 * abs(m.a1[0]) * np.linalg.norm(P)
        F[ph] = orc.landau_f(m, P)
        assert np.linalg.norm(P) == pytest.approx(g[f"P_{ph}_{int(T)}"], abs=6e-5)
        assert F[ph] / 1e6 == pytest.approx(g[f"F_{ph}_{int(T)}"], abs=6e-5 * 10)
    # global minimum T at 300 K (O close), O at 250 K (R close), R at 150 K (O close)
    order = sorted(F, key=F.get)
    assert order == {300.0: ["T", "O", "R"], 250.0: ["O", "R", "T"], 150.0: ["R", "O", "T"]}[T]


def test_T7_spontaneous_polarisation_from_table1():
    # PAPER.md:167 (axis to 0.27 C/m^2) and PAPER.md:203 (<Pz> = -0.80 under field for PbTiO3)
    assert np.linalg.norm(_closed_forms(fi.batio3(300.0))["T"]) == pytest.approx(0.2649, abs=1e-4)
    assert np.linalg.norm(_closed_forms(fi.pbtio3(300.0))["T"]) == pytest.approx(0.7584, abs=1e-4)
    # A7: SrTiO3 alpha1(300 K) gives eps_r ~ 306
    a1 = fi.srtio3(300.0).a1[0]
    assert 1.0 / (2 * fi.EPS0_SI * a1) == pytest.approx(306, rel=0.01)


@pytest.mark.parametrize("T,phase", [(320.0, "T"), (150.0, "R")])
def test_P3_single_cell_relaxation_converges_to_closed_form(T, phase):
    """Landau-only relaxation of a cell ends on an analytic state to 1e-15-ish.
    Reduced units; starts of magnitude 1e-3 biased towards the target basin."""
    u = fi.Units(alpha_ref=abs(fi.batio3(T).a1[0]), P0=0.26, G110=5.1e-10)
    m = u.landau(fi.batio3(T))
    g = u.globals(fi.Globals(**fi.BATIO3_G))
    p = orc.Problem(n=(1, 1, 1), d=(1.0, 1.0, 1.0), periodic=(0, 0, 0), pbc_images=(0, 0, 0), materials=[m], g=g)
    o = orc.Oracle(p)
    rng = np.random.default_rng(5)
    start = {"T": np.array([1.0, 0.05, 0.02]), "R": np.array([1.0, 0.9, 1.1])}[phase]
    P = (1e-3 * start * (1 + 0.01 * rng.standard_normal(3))).reshape(3, 1, 1, 1)
    P = o.step(P, dt=0.05, nsteps=6000, integrator=orc.RK4, terms=orc.TERM_LANDAU)
    target = np.linalg.norm(_closed_forms(m)[phase])
    assert np.linalg.norm(P) == pytest.approx(target, rel=1e-12)
    nz = int(np.sum(np.abs(P.ravel()) > 0.3 * np.linalg.norm(P)))
    assert nz == {"T": 1, "R": 3}[phase]

"""Pins of the oracle's AB3M2 and adaptive RK45 integrators (readings A17, A18 in DESIGN.md):
the Cash-Karp tableau against the Runge-Kutta order conditions, convergence orders on a problem with a closed-form
solution, and the behaviour of the step-size controller."""
import itertools
import math

import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc


def test_cash_karp_tableau_satisfies_the_order_conditions():
    A, C, B5, B4 = orc.RK45_A, orc.RK45_C, orc.RK45_B5, orc.RK45_B4
    a = np.zeros((6, 6))
    for i, row in enumerate(A):
        a[i, :len(row)] = row
    c, b5, b4 = np.array(C), np.array(B5), np.array(B4)
    assert np.allclose(a.sum(axis=1), c, atol=1e-15)              # row sums
    for b, order in ((b5, 5), (b4, 4)):
        # rooted-tree order conditions (Butcher): quadrature conditions and the coupled ones up to `order`
        assert b.sum() == pytest.approx(1.0, abs=1e-15)
        for k in range(1, order):
            assert b @ c ** k == pytest.approx(1.0 / (k + 1), abs=1e-15)
        assert b @ a @ c == pytest.approx(1.0 / 6.0, abs=1e-15)                      # order 3
        assert b @ (c * (a @ c)) == pytest.approx(1.0 / 8.0, abs=1e-15)              # order 4
        assert b @ a @ c ** 2 == pytest.approx(1.0 / 12.0, abs=1e-15)
        assert b @ a @ a @ c == pytest.approx(1.0 / 24.0, abs=1e-15)
    # order 5 conditions hold for the propagated weights only
    assert b5 @ (c ** 2 * (a @ c)) == pytest.approx(1.0 / 10.0, abs=1e-15)
    assert b5 @ (c * (a @ c ** 2)) == pytest.approx(1.0 / 15.0, abs=1e-15)
    assert b5 @ ((a @ c) ** 2) == pytest.approx(1.0 / 20.0, abs=1e-15)
    assert b5 @ a @ c ** 3 == pytest.approx(1.0 / 20.0, abs=1e-15)
    assert b5 @ a @ a @ a @ c == pytest.approx(1.0 / 120.0, abs=1e-15)
    assert abs(b4 @ a @ a @ a @ c - 1.0 / 120.0) > 1e-4           # the embedded solution is only 4th order


def _decay_problem():
    """One active cell, Landau term with a1 > 0 only: dP_i/dt = -2 a1_i P_i, P_i(t) = P_i(0) exp(-2 a1_i t)."""
    m = fi.Landau(a1=(0.7, 1.1, 0.4))
    p = orc.Problem(n=(1, 1, 1), d=(1.0, 1.0, 1.0), periodic=(0, 0, 0), pbc_images=(0, 0, 0), materials=[m],
                    g=fi.Globals(G11=1.0, G12=0.0, G44=0.5, G44p=0.5, eps0=1.0, epsB=1.0, L=1.0))
    P0 = np.array([0.9, -0.5, 0.3]).reshape(3, 1, 1, 1)
    exact = lambda t: P0 * np.exp(-2.0 * np.array(m.a1) * t).reshape(3, 1, 1, 1)
    return orc.Oracle(p), P0, exact


def test_ab3m2_is_second_order_and_converges_to_the_closed_form():
    o, P0, exact = _decay_problem()
    errs = []
    for n in (40, 80, 160):
        P = o.step_ab3m2(P0, 2.0 / n, n, orc.TERM_LANDAU)
        errs.append(np.max(np.abs(P - exact(2.0))))
    assert 3.4 < errs[0] / errs[1] < 4.6 and 3.4 < errs[1] / errs[2] < 4.6
    assert errs[2] < 1e-4
    # error constant: with a predictor of order >= 2 the PECE pair inherits the leading error of the trapezoid rule,
    # -(h^2/12) d3y/dt3 per unit time, i.e. |error_i(T)| = T lam_i^3 h^2 / 12 |P_i(0)| exp(-lam_i T) + O(h^3); predictor
    # weights that do not sum to 12 or miss the first moment condition change this constant by O(1)
    h, T = 2.0 / 160, 2.0
    lam = 2.0 * np.array([0.7, 1.1, 0.4])
    theory = T * lam ** 3 * h * h / 12.0 * np.abs(P0.ravel()) * np.exp(-lam * T)
    got = np.abs(o.step_ab3m2(P0, h, 160, orc.TERM_LANDAU) - exact(T)).ravel()
    assert np.allclose(got, theory, rtol=0.15)


def test_rk45_fixed_step_is_fifth_order():
    o, P0, exact = _decay_problem()
    errs = []
    for n in (16, 32, 64):
        # a huge tolerance accepts every step; dt_next grows, but min(dt, remaining) with max_steps = n keeps h fixed
        P = P0
        for _ in range(n):
            P, st = o.step_rk45(P, 2.0 / n, 2.0 / n, 1e30, 10, orc.TERM_LANDAU)
            assert st["accepted"] == 1 and st["rejected"] == 0
        errs.append(np.max(np.abs(P - exact(2.0))))
    assert 24 < errs[0] / errs[1] < 40 and 24 < errs[1] / errs[2] < 40


def test_rk45_controller_meets_the_tolerance_and_lands_on_t_span():
    o, P0, exact = _decay_problem()
    prev = None
    for tol in (1e-4, 1e-6, 1e-8, 1e-10):
        P, st = o.step_rk45(P0, 3.0, 1.5, tol, 10000, orc.TERM_LANDAU)
        assert st["t"] == 3.0 and st["rhs_evals"] == 6 * (st["accepted"] + st["rejected"])
        err = np.max(np.abs(P - exact(3.0)))
        assert err < 20 * tol                       # local error control: global error stays within a small multiple
        assert st["err_last"] <= 1.0
        if prev is not None:
            assert st["accepted"] >= prev
        prev = st["accepted"]
    # a first step that is far too large is rejected and shrunk, never accepted
    P, st = o.step_rk45(P0, 3.0, 3.0, 1e-10, 10000, orc.TERM_LANDAU)
    assert st["rejected"] >= 1
    # max_steps bounds the work
    P, st = o.step_rk45(P0, 3.0, 1e-3, 1e-12, 7, orc.TERM_LANDAU)
    assert st["accepted"] + st["rejected"] == 7 and st["t"] < 3.0


def _forced_problem():
    """One cell, dP_z/dt = -lam P_z + A sin(om t) (Landau a1 > 0 + sinusoidal external field):
    P(t) = exp(-lam t) P0 + A [lam sin(om t) - om cos(om t) + om exp(-lam t)] / (lam^2 + om^2)."""
    m = fi.Landau(a1=(0.7, 1.1, 0.4))
    p = orc.Problem(n=(1, 1, 1), d=(1.0, 1.0, 1.0), periodic=(0, 0, 0), pbc_images=(0, 0, 0), materials=[m],
                    g=fi.Globals(G11=1.0, G12=0.0, G44=0.5, G44p=0.5, eps0=1.0, epsB=1.0, L=1.0, E_ext=(0.0, 0.2, 0.0)))
    o = orc.Oracle(p)
    A, om, ph = np.array([0.0, 0.0, 0.8]), 3.0, 0.0
    o.set_wave(A, om, ph)
    P0 = np.array([0.0, 0.0, 0.3]).reshape(3, 1, 1, 1)
    lam = 2.0 * 0.4

    def exact_z(t):
        return math.exp(-lam * t) * 0.3 + 0.8 * (lam * math.sin(om * t) - om * math.cos(om * t)
                                                   + om * math.exp(-lam * t)) / (lam * lam + om * om)
    return o, P0, exact_z


@pytest.mark.parametrize("name,order", [("euler", 1), ("heun", 2), ("rk4", 4), ("ab3m2", 2), ("rk45", 5)])
def test_time_dependent_field_is_sampled_at_the_stage_times(name, order):
    """With a forcing that depends on t a wrong stage abscissa lowers the order of every multi-stage scheme."""
    o, P0, exact_z = _forced_problem()
    terms = orc.TERM_LANDAU | orc.TERM_EXT
    T, errs = 2.3, []     # a time at which no leading error term vanishes by accident
    for n in ((40, 80) if order < 5 else (12, 24)):
        h = T / n
        if name == "ab3m2":
            P = o.step_ab3m2(P0, h, n, terms)
        elif name == "rk45":
            P = P0
            for i in range(n):
                P, st = o.step_rk45(P, h, h, 1e30, 4, terms, t0=i * h)
        else:
            P = o.step(P0, h, n, {"euler": orc.EULER, "heun": orc.HEUN, "rk4": orc.RK4}[name], terms)
        errs.append(abs(P[2, 0, 0, 0] - exact_z(T)))
        # the static y component relaxes to E_y / (2 a1_y) independently of the wave
    ratio = errs[0] / errs[1]
    assert 0.7 * 2 ** order < ratio < 1.45 * 2 ** order, (name, ratio)
    # stepping in two calls with t0 equals one call
    a = o.step(P0, 0.05, 10, orc.RK4, terms)
    b = o.step(o.step(P0, 0.05, 4, orc.RK4, terms), 0.05, 6, orc.RK4, terms, t0=0.2)
    assert np.allclose(a, b, rtol=0, atol=1e-15)

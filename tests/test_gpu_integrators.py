"""-m gpu parity of AB3M2 and the adaptive Cash-Karp RK45 (readings A17 / A18)
against the oracle's step-by-step implementations (pinned in tests/test_oracle_integrators.py).  The accept / reject
decisions of RK45 are taken in fp64 on both sides from max |y5 - y4| / tol."""
import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc
from gpu_util import rel_l2, oracle_problem, workload_from_random

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fe():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_28800_b200 as fe
    fe.load()
    return fe


@pytest.mark.parametrize("n,periodic,images", [((8, 8, 4), (0, 1, 0), (0, 2, 0)), ((64, 8, 8), (0, 0, 0), (0, 0, 0))])
def test_ab3m2_against_the_oracle(fe, n, periodic, images):
    w = workload_from_random(81, n, periodic, images, batch=2)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    o = orc.Oracle(oracle_problem(w, 1), elec="direct")
    for nsteps in (1, 2, 3, 9):                                  # 1, 2: start-up steps only
        P = g.state(w.P0)
        g.step(P, 8e-3, nsteps, fe.FE_AB3M2, fi.TERM_ALL)
        want = o.step_ab3m2(w.P0[1], 8e-3, nsteps, fi.TERM_ALL)
        assert rel_l2(P.cpu().numpy()[1], want) < 1e-12, nsteps
    g.close()


def test_rk45_against_the_oracle_same_decisions(fe):
    w = workload_from_random(83, (8, 8, 4), (0, 1, 0), (0, 2, 0), batch=1)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    o = orc.Oracle(oracle_problem(w, 0), elec="direct")
    for tol, dt0 in ((1e-5, 0.5), (1e-8, 0.05)):
        P = g.state(w.P0)
        st = g.step_rk45(P, 0.4, dt0, tol, 10000, fi.TERM_ALL)
        want, so = o.step_rk45(w.P0[0], 0.4, dt0, tol, 10000, fi.TERM_ALL)
        assert (st["accepted"], st["rejected"], st["rhs_evals"]) == (so["accepted"], so["rejected"], so["rhs_evals"])
        assert st["t"] == so["t"] == 0.4
        assert st["dt_last"] == pytest.approx(so["dt_last"], rel=1e-9)
        assert st["err_last"] == pytest.approx(so["err_last"], rel=1e-6)
        assert rel_l2(P.cpu().numpy()[0], want) < 1e-10
        assert so["rejected"] >= 1 or tol == 1e-8                  # the large first step is rejected and shrunk
    # max_steps bounds the work; the state is the one reached at stats["t"]
    P = g.state(w.P0)
    st = g.step_rk45(P, 0.4, 1e-3, 1e-9, 5, fi.TERM_ALL)
    want, so = o.step_rk45(w.P0[0], 0.4, 1e-3, 1e-9, 5, fi.TERM_ALL)
    # (the error estimate is a difference of nearly equal sums: its rounding noise enters the proposed step sizes)
    assert st["accepted"] + st["rejected"] == 5 and st["t"] < 0.4 and st["t"] == pytest.approx(so["t"], rel=1e-6)
    assert rel_l2(P.cpu().numpy()[0], want) < 1e-9
    g.close()


def test_rk45_on_the_fast_path_and_batch_lockstep(fe):
    """Grid that takes the size-specialised kernels, batch of 2: one common step controlled by the worst member."""
    w = fi.open_batio3("rk45_64x32x32", (64, 32, 32), 2, "f64", 91)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P = g.state(w.P0)
    st = g.step_rk45(P, 0.02, 0.01, 1e-7, 1000, fi.TERM_ALL)
    assert st["t"] == 0.02 and st["accepted"] >= 1
    # reference: the oracle run on each member alone must take steps at least as large: lock-step is conservative
    ref = []
    for b in range(2):
        o = orc.Oracle(oracle_problem(w, b), elec="fft")
        Pb, sb = o.step_rk45(w.P0[b], 0.02, 0.01, 1e-7, 1000, fi.TERM_ALL)
        ref.append(Pb)
        assert sb["accepted"] <= st["accepted"]
    got = P.cpu().numpy()
    for b in range(2):                                               # different step sequences: compare to the tolerance
        assert np.max(np.abs(got[b] - ref[b])) < 50 * 1e-7
    with pytest.raises(fe.FeError):
        g.step_rk45(P, 0.02, -1.0, 1e-7)
    g.close()


def test_time_dependent_field_all_integrators(fe):
    """Sinusoidal excitation on top of the static field, different per member, clock starting at t = 0.37:
    RHS, energy and every integrator against the oracle (which samples E_ext at the stage times)."""
    w = workload_from_random(87, (8, 8, 4), (0, 1, 0), (0, 2, 0), batch=2)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    waves = [((0.3, -0.2, 0.5), 7.0, 0.4), ((-0.1, 0.6, 0.2), 3.0, -1.1)]
    oracles = []
    for b, (amp, om, ph) in enumerate(waves):
        g.set_external_wave(b, amp, om, ph)
        o = orc.Oracle(oracle_problem(w, b), elec="direct")
        o.set_wave(amp, om, ph)
        oracles.append(o)
    t0, dt = 0.37, 8e-3
    g.set_time(t0)
    P = g.state(w.P0)
    got = g.rhs(P).cpu().numpy()
    for b in range(2):
        assert rel_l2(got[b], oracles[b].rhs(w.P0[b], fi.TERM_ALL, t0)) < 1e-12
    assert rel_l2(g.rhs(P, fi.TERM_EXT).cpu().numpy()[1], oracles[1].rhs(w.P0[1], fi.TERM_EXT, t0)) < 1e-13
    for integ, name in ((fi.EULER, "euler"), (fi.HEUN, "heun"), (fi.RK4, "rk4"), (fe.FE_AB3M2, "ab3m2")):
        g.set_time(t0)
        P = g.state(w.P0)
        g.step(P, dt, 12, integ, fi.TERM_ALL)              # long enough for the graph path, which must stay off
        assert g.time() == pytest.approx(t0 + 12 * dt, rel=1e-15)
        for b in range(2):
            o = oracles[b]
            want = (o.step_ab3m2(w.P0[b], dt, 12, fi.TERM_ALL, t0=t0) if name == "ab3m2"
                    else o.step(w.P0[b], dt, 12, integ, fi.TERM_ALL, t0=t0))
            assert rel_l2(P.cpu().numpy()[b], want) < 1e-12, (name, b)
    # two calls continue the clock
    g.set_time(t0)
    Pa = g.state(w.P0)
    g.step(Pa, dt, 5, fi.RK4, fi.TERM_ALL)
    g.step(Pa, dt, 7, fi.RK4, fi.TERM_ALL)
    want = oracles[0].step(w.P0[0], dt, 12, fi.RK4, fi.TERM_ALL, t0=t0)
    assert rel_l2(Pa.cpu().numpy()[0], want) < 1e-12
    # adaptive RK45 with the wave: single member so that the decisions can be compared
    w1 = workload_from_random(89, (8, 8, 4), (0, 1, 0), (0, 2, 0), batch=1)
    g1 = fe.Grid.from_workload(w1)
    g1.precompute_tensor()
    g1.set_external_wave(0, *waves[0])
    o1 = orc.Oracle(oracle_problem(w1, 0), elec="direct")
    o1.set_wave(*waves[0])
    g1.set_time(t0)
    P1 = g1.state(w1.P0)
    st = g1.step_rk45(P1, 0.3, 0.05, 1e-7, 1000, fi.TERM_ALL)
    want, so = o1.step_rk45(w1.P0[0], 0.3, 0.05, 1e-7, 1000, fi.TERM_ALL, t0=t0)
    assert (st["accepted"], st["rejected"]) == (so["accepted"], so["rejected"])
    assert rel_l2(P1.cpu().numpy()[0], want) < 1e-10
    assert g1.time() == pytest.approx(t0 + 0.3, rel=1e-14)
    e = g1.energy(P1)[0]
    o1.p.g.E_ext = tuple(o1.e_ext(t0 + 0.3))               # the oracle's energy takes the field of that instant
    o1.wave = None
    assert np.allclose(e[:5], o1.energy(want)[:5], rtol=1e-9, atol=1e-11)
    g.close()
    g1.close()


@pytest.mark.parametrize("bad", [float("nan"), float("inf")])
def test_rk45_nonfinite_state_is_refused_not_accepted(fe, bad):
    """A NaN / Inf cell makes the embedded error estimate non-finite.  fmax-style reductions drop NaN and would accept
    the step with err = 0; the library must reject every attempt and return FE_ENONFINITE, leaving P as it was."""
    w = workload_from_random(85, (8, 8, 4), (0, 0, 0), (0, 0, 0), batch=2)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P0 = w.P0.copy()
    act = np.argwhere(oracle_problem(w, 1).active)[3]
    P0[1, 2, act[0], act[1], act[2]] = bad
    P = g.state(P0)
    with pytest.raises(fe.FeError) as ei:
        g.step_rk45(P, 0.4, 0.05, 1e-6, 1000, fi.TERM_ALL)
    assert ei.value.status == fe.FE_ENONFINITE
    got = P.cpu().numpy()
    assert np.array_equal(got[0], P0[0]) and np.array_equal(np.isnan(got[1]), np.isnan(P0[1]))
    # every cell NaN: the maximum over the finite cells would be 0
    P = g.state(np.full_like(w.P0, np.nan))
    with pytest.raises(fe.FeError) as ei:
        g.step_rk45(P, 0.4, 0.05, 1e-6, 1000, fi.TERM_ALL)
    assert ei.value.status == fe.FE_ENONFINITE
    g.close()


@pytest.mark.parametrize("dtype,tol,gm0", [("f64", 1e-11, False), ("f32", 1e-4, False), ("f64", 1e-11, True)])
def test_specialised_stage_epilogues_on_the_tensor_copy_path(fe, dtype, tol, gm0):
    """Open grid without a material map, wide enough for the tensor-copy halo tiles (72 x 16 x 8, batch 2, Gm != 0): the stages
    of Euler, Heun, RK4 and AB3M2 (with history) and the plain right-hand side each take their own instantiation of the local
    step (compile-time epilogue) -- every one of them against the oracle."""
    w = fi.open_batio3("epilogues_72x16x8", (72, 16, 8), 2, dtype, 4242)
    if gm0:                                  # Gm = G12 + G44 - G'44 = 0: the instantiations without the mixed-derivative taps
        from dataclasses import replace
        w.globals_ = [replace(q, G12=q.G44p - q.G44) for q in w.globals_]
    P0 = w.P0 if dtype == "f64" else w.P0.astype(np.float32).astype(np.float64)
    g = fe.Grid.from_workload(w, dtype=dtype)
    g.precompute_tensor()
    o = orc.Oracle(oracle_problem(w, 1), elec="fft")
    P = g.state(P0)
    assert rel_l2(g.rhs(P, fi.TERM_ALL).cpu().numpy()[1], o.rhs(P0[1], fi.TERM_ALL)) < (1e-10 if dtype == "f64" else tol)
    dt = 4 * w.dt
    for integ, nsteps in ((fi.EULER, 6), (fi.HEUN, 4), (fi.RK4, 3), (fi.AB3M2, 6)):
        P = g.state(P0)
        g.step(P, dt, nsteps, integ, fi.TERM_ALL)
        want = o.step_ab3m2(P0[1], dt, nsteps, fi.TERM_ALL) if integ == fi.AB3M2 else o.step(P0[1], dt, nsteps, integ, fi.TERM_ALL)
        assert rel_l2(P.cpu().numpy()[1].astype(np.float64), want) < tol, integ
    g.close()


def test_wave_static_field_and_eighth_order_terms_on_the_tensor_copy_path(fe):
    """The same grid with everything the stage epilogues sample per member: a static E_ext, a sinusoidal one at the stage
    times, a clock that does not start at zero, non-zero 8th-order Landau slots -- and the adaptive RK45 on top (generic
    epilogue with folded stage combinations), decision by decision."""
    from dataclasses import replace
    w = fi.open_batio3("epilogues_72x16x8", (72, 16, 8), 2, "f64", 4243)
    w.materials = [[replace(m[0], a1111=0.3 * abs(m[0].a111), a1112=-0.2 * abs(m[0].a111), a1122=0.1 * abs(m[0].a111),
                            a1123=0.25 * abs(m[0].a111))] for m in w.materials]
    fields = [(0.02, -0.01, 0.03), (-0.015, 0.02, 0.01)]
    waves = [((0.03, -0.02, 0.05), 7.0, 0.4), ((-0.01, 0.06, 0.02), 3.0, -1.1)]
    w.globals_ = [replace(q, E_ext=fields[b]) for b, q in enumerate(w.globals_)]
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    oracles = []
    for b in range(2):
        g.set_external_wave(b, *waves[b])
        o = orc.Oracle(oracle_problem(w, b), elec="fft")
        o.set_wave(*waves[b])
        oracles.append(o)
    t0, dt = 0.37, 4 * w.dt
    g.set_time(t0)
    P = g.state(w.P0)
    got = g.rhs(P).cpu().numpy()
    for b in range(2):
        assert rel_l2(got[b], oracles[b].rhs(w.P0[b], fi.TERM_ALL, t0)) < 1e-10
    for integ, name in ((fi.EULER, "euler"), (fi.HEUN, "heun"), (fi.RK4, "rk4"), (fe.FE_AB3M2, "ab3m2")):
        g.set_time(t0)
        P = g.state(w.P0)
        g.step(P, dt, 5, integ, fi.TERM_ALL)
        for b in range(2):
            o = oracles[b]
            want = (o.step_ab3m2(w.P0[b], dt, 5, fi.TERM_ALL, t0=t0) if name == "ab3m2"
                    else o.step(w.P0[b], dt, 5, integ, fi.TERM_ALL, t0=t0))
            assert rel_l2(P.cpu().numpy()[b], want) < 1e-11, (name, b)
    g.close()
    # adaptive RK45, one member so that the accept / reject decisions can be compared one by one
    w1 = fi.open_batio3("epilogues_72x16x8", (72, 16, 8), 1, "f64", 4244)
    w1.globals_ = [replace(w1.globals_[0], E_ext=fields[0])]
    g1 = fe.Grid.from_workload(w1)
    g1.precompute_tensor()
    g1.set_external_wave(0, *waves[0])
    o1 = orc.Oracle(oracle_problem(w1), elec="fft")
    o1.set_wave(*waves[0])
    g1.set_time(t0)
    P1 = g1.state(w1.P0)
    st = g1.step_rk45(P1, 0.03, 0.02, 1e-8, 200, fi.TERM_ALL)
    want, so = o1.step_rk45(w1.P0[0], 0.03, 0.02, 1e-8, 200, fi.TERM_ALL, t0=t0)
    assert (st["accepted"], st["rejected"]) == (so["accepted"], so["rejected"]) and st["accepted"] >= 2
    assert rel_l2(P1.cpu().numpy()[0], want) < 1e-11
    g1.close()

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

"""-m gpu test of fe_energy_noalloc (include/fe.h): the energy / mean reduction with its per-block partial sums in a
file-scope static device array instead of the workspace -- no allocation, no host copy, no synchronisation.  Collected
last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`.

The new entry point must give what the existing path (fe_energy) gives, within the tolerance the energy parity test uses
(rtol 1e-11, atol 1e-12), on two calls in a row and across grids of different shapes that share the one static array."""
import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc
from gpu_util import oracle_problem, workload_from_random

pytestmark = pytest.mark.gpu

RTOL, ATOL = 1e-11, 1e-12


@pytest.fixture(scope="module")
def fe():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_28800_b200 as fe
    fe.load()
    return fe


def _noalloc(g, P, terms):
    import torch
    out = torch.full((g.batch, 8), float("nan"), dtype=torch.float64, device=P.device)
    g.energy_noalloc(P, out, terms)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_energy_noalloc_matches_fe_energy_on_two_calls_in_a_row(fe):
    # heterogeneous: three materials incl. vacuum (material map), Gm != 0, one periodic axis, two members
    w = workload_from_random(51, (8, 4, 8), (0, 1, 0), (0, 2, 0), batch=2)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P = g.state(w.P0)
    first = _noalloc(g, P, fi.TERM_ALL)
    want = g.energy(P)
    assert np.allclose(first, want, rtol=RTOL, atol=ATOL), (first, want)
    for b in range(2):                                   # and the oracle itself, as the existing energy test does
        eo = orc.Oracle(oracle_problem(w, b)).energy(w.P0[b])
        assert np.allclose(first[b], eo, rtol=RTOL, atol=ATOL), (b, first[b], eo)
    # second call, other state, right behind the first: the array still holds the first call's sums
    g.step(P, w.dt, 3, fi.EULER, fi.TERM_ALL)
    second = _noalloc(g, P, fi.TERM_ALL)
    want2 = g.energy(P)
    assert np.allclose(second, want2, rtol=RTOL, atol=ATOL), (second, want2)
    assert not np.allclose(second, first, rtol=1e-6, atol=0.0)          # the state did change
    # every subset of terms the existing path takes
    for terms in (fi.TERM_LANDAU, fi.TERM_GRADIENT, fi.TERM_ELEC, fi.TERM_EXT, fi.TERM_LANDAU | fi.TERM_EXT):
        assert np.allclose(_noalloc(g, P, terms), g.energy(P, terms), rtol=RTOL, atol=ATOL), terms
    g.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_energy_noalloc_shares_one_array_between_grids(fe, dtype):
    """A grid with more members first, then a smaller one on the size-specialised path: the second call reads only the rows
    it wrote, whatever the first left behind."""
    wa = fi.config3(n=16, batch=4)
    wb = fi.open_batio3("noalloc_64x32x32", (64, 32, 32), 1, dtype, 77)
    ga = fe.Grid.from_workload(wa, dtype=dtype)
    gb = fe.Grid.from_workload(wb, dtype=dtype)
    ga.precompute_tensor()
    gb.precompute_tensor()
    Pa, Pb = ga.state(wa.P0), gb.state(wb.P0)
    rt, at = (RTOL, ATOL) if dtype == "f64" else (1e-6, 1e-9)
    for _ in range(2):
        a = _noalloc(ga, Pa, fi.TERM_ALL)
        b = _noalloc(gb, Pb, fi.TERM_ALL)
        assert np.allclose(a, ga.energy(Pa), rtol=rt, atol=at)
        assert np.allclose(b, gb.energy(Pb), rtol=rt, atol=at)
        gb.step(Pb, wb.dt, 2, fi.EULER, fi.TERM_ALL)
    ga.close()
    gb.close()


def test_energy_noalloc_refuses_what_does_not_fit_and_bad_arguments(fe):
    import torch
    w = fi.config3(n=8, batch=28)                        # 28 * 296 * 8 = 66304 partial sums > 65536
    g = fe.Grid.from_workload(w)
    P = g.state(w.P0)
    out = torch.zeros((28, 8), dtype=torch.float64, device=P.device)
    with pytest.raises(fe.FeError) as ei:
        g.energy_noalloc(P, out, fi.TERM_LANDAU | fi.TERM_GRADIENT)
    assert ei.value.status == fe.FE_EINVAL and "static scratch" in str(ei.value)
    assert np.all(np.isfinite(g.energy(P, fi.TERM_LANDAU | fi.TERM_GRADIENT)))      # the workspace path still serves it
    with pytest.raises(ValueError):
        g.energy_noalloc(P, out.cpu(), fi.TERM_LANDAU)
    with pytest.raises(ValueError):
        g.energy_noalloc(P, out[:27], fi.TERM_LANDAU)
    g.close()

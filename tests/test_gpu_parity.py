"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerances (BASELINE.json north_star, A14): rel-L2 <= 1e-10 per RHS and
<= 1e-8 after 100 steps in fp64, <= 1e-4 in fp32."""
import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc
from gpu_util import rel_l2, oracle_problem, workload_from_random

pytestmark = pytest.mark.gpu

TOL_RHS64, TOL_STEP64, TOL32 = 1e-10, 1e-8, 1e-4


@pytest.fixture(scope="module")
def fe():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_28800_b200 as fe
    fe.load()
    return fe


def _grid(fe, w, dtype=None):
    g = fe.Grid.from_workload(w, dtype=dtype)
    g.precompute_tensor()
    return g


# ------------------------------------------------------------------------------------------ a0 tensor
@pytest.mark.parametrize("n,d,periodic,images", [
    ((16, 16, 8), (1.0, 1.0, 1.0), (0, 0, 0), (0, 0, 0)),
    ((8, 4, 16), (0.9, 1.1, 0.7), (0, 0, 0), (0, 0, 0)),
    ((8, 4, 4), (1.0, 1.0, 1.0), (0, 1, 1), (0, 3, 3)),        # two periodic axes: zero-mode rule
    ((4, 4, 8), (1.0, 1.2, 0.8), (1, 1, 0), (2, 2, 0)),
    ((8, 8, 4), (1.0, 1.0, 1.0), (0, 1, 0), (0, 2, 0)),        # one periodic axis: plain image sum
])
def test_tensor_table_matches_the_float128_oracle(fe, n, d, periodic, images):
    g = fe.Grid(n, d, periodic, images, 1, "f64", 1)
    K = g.get_tensor()
    p = orc.Problem(n=n, d=d, periodic=periodic, pbc_images=images, materials=[fi.batio3(300.0)],
                    g=fi.Globals(**fi.BATIO3_G))
    ref = orc.circular_kernel(p, orc.tensor_table(p))
    assert K.shape == ref.shape
    assert np.max(np.abs(K - ref)) < 2e-14
    # trace identity on the GPU table itself (P2): 1 at the origin of a fully open box, 0 elsewhere
    if sum(periodic) == 0:
        tr = K[0] + K[1] + K[2]
        assert abs(tr[0, 0, 0] - 1.0) < 1e-13
        tr[0, 0, 0] = 0.0
        assert np.max(np.abs(tr)) < 1e-13


def test_fully_periodic_box(fe):
    """Three periodic axes (reading A4, last case): tensor table with the mean removed, RHS against the direct sum,
    no field in a uniformly polarised periodic crystal."""
    n, d, per, img = (8, 4, 8), (1.0, 1.1, 0.9), (1, 1, 1), (2, 2, 2)
    g = fe.Grid(n, d, per, img, 1, "f64", 1)
    K = g.get_tensor()
    p = orc.Problem(n=n, d=d, periodic=per, pbc_images=img, materials=[fi.batio3(300.0)], g=fi.Globals(**fi.BATIO3_G))
    ref = orc.circular_kernel(p, orc.tensor_table(p))
    assert np.max(np.abs(K - ref)) < 1e-13          # 125 images summed in fp64 on the GPU, __float128 in the oracle
    assert np.max(np.abs(K.reshape(6, -1).sum(axis=1))) < 1e-12
    w = workload_from_random(33, n, per, img, batch=1)
    g = _grid(fe, w)
    o = orc.Oracle(oracle_problem(w), elec="direct")
    for terms in (fi.TERM_ELEC, fi.TERM_ALL):
        assert rel_l2(g.rhs(g.state(w.P0), terms).cpu().numpy()[0], o.rhs(w.P0[0], terms)) < TOL_RHS64
    w2 = fi.open_batio3("per3", (16, 16, 8), 1, "f64", 7)
    w2.periodic, w2.pbc_images = (1, 1, 1), (1, 1, 1)
    g2 = _grid(fe, w2)
    Pu = np.zeros_like(w2.P0)
    Pu[0, 0], Pu[0, 2] = 0.4, -0.3
    E = g2.rhs(g2.state(Pu), fi.TERM_ELEC).cpu().numpy()
    assert np.max(np.abs(E)) < 1e-11 * (0.4 / (w2.globals_[0].eps0 * w2.globals_[0].epsB))


def test_far_field_quadrature_tiers_against_the_oracle(fe):
    """Offsets up to 255 cells along x exercise every quadrature tier (8/6/4/3/2 nodes)."""
    n, d = (256, 4, 4), (1.0, 1.0, 1.0)
    g = fe.Grid(n, d, (0, 0, 0), (0, 0, 0), 1, "f64", 1)
    K = g.get_tensor()
    rng = np.random.default_rng(5)
    for _ in range(60):
        off = (int(rng.integers(0, 256)), int(rng.integers(0, 4)), int(rng.integers(0, 4)))
        for comp in range(6):
            ref = orc.newell_entry(comp, off, d)
            assert abs(K[comp, off[2], off[1], off[0]] - ref) < 1e-14, (comp, off)


# ------------------------------------------------------------------------------------------ a1-a4 RHS
def test_config1_rhs_against_direct_sum(fe):
    w = fi.config1()
    g = _grid(fe, w)
    o = orc.Oracle(oracle_problem(w), elec="direct")
    P = g.state(w.P0)
    for terms in (fi.TERM_ELEC, fi.TERM_LANDAU, fi.TERM_GRADIENT, fi.TERM_ALL):
        got = g.rhs(P, terms).cpu().numpy()[0]
        want = o.rhs(w.P0[0], terms)
        assert rel_l2(got, want) < TOL_RHS64, terms


@pytest.mark.parametrize("n,periodic,images", [
    ((8, 4, 4), (0, 0, 0), (0, 0, 0)),
    ((8, 8, 4), (0, 1, 0), (0, 2, 0)),
    ((4, 8, 8), (1, 1, 0), (2, 2, 0)),
    ((16, 4, 4), (0, 1, 1), (0, 3, 3)),
    ((4, 4, 4), (1, 0, 1), (1, 0, 1)),
])
def test_heterogeneous_problem_rhs_each_term(fe, n, periodic, images):
    """3 materials incl. vacuum, Gm != 0, 8th-order slots, E_ext, anisotropic cells, batch of 2."""
    w = workload_from_random(31, n, periodic, images, batch=2)
    g = _grid(fe, w)
    P = g.state(w.P0)
    for b in range(2):
        o = orc.Oracle(oracle_problem(w, b), elec="direct")
        for terms in (fi.TERM_LANDAU, fi.TERM_GRADIENT, fi.TERM_ELEC, fi.TERM_EXT, fi.TERM_ALL):
            got = g.rhs(P, terms).cpu().numpy()[b]
            want = o.rhs(w.P0[b], terms)
            assert rel_l2(got, want) < TOL_RHS64, (b, terms)
            assert np.all(got[:, o.p.active == 0] == 0.0)


def test_config1_100_euler_steps_and_energy(fe):
    w = fi.config1()
    g = _grid(fe, w)
    o = orc.Oracle(oracle_problem(w), elec="direct")
    P = g.state(w.P0)
    Pref = w.P0[0].copy()
    e_prev = None
    for chunk in (50, 50):
        g.step(P, w.dt, chunk, fi.EULER, fi.TERM_ALL)
        Pref = o.step(Pref, w.dt, chunk, fi.EULER, fi.TERM_ALL)
        assert rel_l2(g.rhs(P).cpu().numpy()[0], o.rhs(Pref)) < 1e-8
        e = g.energy(P)[0]
        eo = o.energy(Pref)
        assert np.allclose(e[:5], eo[:5], rtol=1e-8, atol=1e-9 * abs(eo[4]))
        assert np.allclose(e[5:], eo[5:], rtol=0, atol=1e-9)
        if e_prev is not None:
            assert e[4] <= e_prev            # P8: monotone decrease
        e_prev = e[4]
    assert rel_l2(P.cpu().numpy()[0], Pref) < TOL_STEP64


@pytest.mark.parametrize("integ,name", [(fi.HEUN, "heun"), (fi.RK4, "rk4"), (fi.EULER, "euler_odd")])
def test_integrators_against_the_oracle(fe, integ, name):
    w = workload_from_random(41, (8, 8, 4), (0, 1, 0), (0, 2, 0), batch=1)
    g = _grid(fe, w)
    o = orc.Oracle(oracle_problem(w), elec="direct")
    P = g.state(w.P0)
    nsteps = 7
    g.step(P, 2e-2, nsteps, integ, fi.TERM_ALL)
    want = o.step(w.P0[0], 2e-2, nsteps, integ, fi.TERM_ALL)
    assert rel_l2(P.cpu().numpy()[0], want) < 1e-12


def test_energy_terms_heterogeneous(fe):
    w = workload_from_random(51, (8, 4, 8), (0, 1, 0), (0, 2, 0), batch=2)
    g = _grid(fe, w)
    P = g.state(w.P0)
    e = g.energy(P)
    for b in range(2):
        eo = orc.Oracle(oracle_problem(w, b)).energy(w.P0[b])
        assert np.allclose(e[b], eo, rtol=1e-11, atol=1e-12), (b, e[b], eo)


def test_fp32_rhs_and_steps(fe):
    w = fi.config1()
    g = _grid(fe, w, dtype="f32")
    P32 = w.P0.astype(np.float32)
    o = orc.Oracle(oracle_problem(w), elec="direct")
    P = g.state(P32)
    got = g.rhs(P).cpu().numpy()[0]
    want = o.rhs(P32[0].astype(np.float64))
    assert rel_l2(got, want) < TOL32
    g.step(P, w.dt, 100, fi.EULER, fi.TERM_ALL)
    ref = o.step(P32[0].astype(np.float64), w.dt, 100, fi.EULER, fi.TERM_ALL)
    assert rel_l2(P.cpu().numpy()[0], ref) < TOL32


def test_batch_member_equals_the_same_simulation_alone(fe):
    """P9: batch independence; members have different coefficients (config 3 style temperatures)."""
    w = fi.config3(n=16, batch=4)
    g = _grid(fe, w)
    P = g.state(w.P0)
    full = g.rhs(P).cpu().numpy()
    for b in (0, 3):
        w1 = fi.Workload(name="one", n=w.n, d=w.d, periodic=w.periodic, pbc_images=w.pbc_images, batch=1, dtype="f64",
                         materials=[w.materials[b]], globals_=[w.globals_[b]], matmap=None, P0=w.P0[b:b + 1],
                         dt=w.dt, integrator=fi.EULER)
        g1 = _grid(fe, w1)
        alone = g1.rhs(g1.state(w1.P0)).cpu().numpy()[0]
        assert np.array_equal(alone, full[b])
        want = orc.Oracle(oracle_problem(w, b), elec="fft").rhs(w.P0[b])
        assert rel_l2(full[b], want) < TOL_RHS64


def test_config2_wall_cut_and_config4_bilayer_cut(fe):
    """Reduced-size cuts of configs 2 and 4 (periodic axes + zero-mode rule, per-layer materials)."""
    w2 = fi.config2(nx=64, pbc_images=3, elec=True)
    g = _grid(fe, w2)
    o = orc.Oracle(oracle_problem(w2), elec="direct")
    got = g.rhs(g.state(w2.P0), w2.terms).cpu().numpy()[0]
    assert rel_l2(got, o.rhs(w2.P0[0], w2.terms)) < TOL_RHS64
    w4 = fi.config4(nxy=16, nz=8, pbc_images=2)
    g = _grid(fe, w4)
    o = orc.Oracle(oracle_problem(w4), elec="direct")
    got = g.rhs(g.state(w4.P0)).cpu().numpy()[0]
    assert rel_l2(got, o.rhs(w4.P0[0])) < TOL_RHS64
    # P4(i): uniform out-of-plane P in a film periodic in-plane feels exactly -P/(eps0 epsB)
    Pu = np.zeros_like(w4.P0)
    Pu[0, 2] = 0.3
    Ez = g.rhs(g.state(Pu), fi.TERM_ELEC).cpu().numpy()[0]
    gl = w4.globals_[0]
    act = oracle_problem(w4).active
    assert np.allclose(Ez[2][act > 0], -gl.L * 0.3 / (gl.eps0 * gl.epsB), rtol=1e-11)


def test_error_paths(fe):
    import torch
    w = fi.config1()
    g = fe.Grid.from_workload(w)
    P = g.state(w.P0)
    with pytest.raises(fe.FeError) as ei:
        g.rhs(P, fi.TERM_ALL)                       # tensor not precomputed
    assert ei.value.status == fe.FE_ESTATE
    g.rhs(P, fi.TERM_LANDAU | fi.TERM_GRADIENT)     # allowed without the tensor
    g.precompute_tensor()
    bad = P.clone()
    bad[0, 0, 0, 0, 0] = float("nan")
    with pytest.raises(fe.FeError) as ei:
        g.energy(bad)
    assert ei.value.status == fe.FE_ENONFINITE
    g2 = fe.Grid(w.n, w.d, batch=1, n_materials=2)
    g2.set_global(0, w.globals_[0])
    g2.set_material(0, 0, w.materials[0][0])
    with pytest.raises(fe.FeError) as ei:           # material 1 unset
        g2.rhs(P, fi.TERM_LANDAU)
    assert ei.value.status == fe.FE_ESTATE


def test_degenerate_inputs(fe):
    """Zero steps, the zero state, an all-vacuum sample and the smallest grid the ABI admits."""
    import torch
    from dataclasses import replace
    w = fi.config1()
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P = g.state(w.P0)
    before = P.clone()
    for integ in (fi.EULER, fi.HEUN, fi.RK4, fi.AB3M2):
        g.step(P, w.dt, 0, integ, fi.TERM_ALL)                     # nsteps = 0: nothing happens, the clock stands still
        assert torch.equal(P, before) and g.time() == 0.0
    # P = 0: no Landau, gradient or electrostatic field; dP/dt = L E_ext exactly, energies zero
    Z = torch.zeros_like(P)
    got = g.rhs(Z, fi.TERM_ALL).cpu().numpy()[0]
    want = orc.Oracle(oracle_problem(w)).rhs(np.zeros_like(w.P0[0]), fi.TERM_ALL)
    assert np.array_equal(got, want)
    assert np.all(g.energy(Z) == 0.0)
    g.close()
    # all cells vacuum: the state is pinned, the right-hand side is zero whatever the terms
    for wv in (fi.config1(), fi.open_batio3("vacuum_64x8x8", (64, 8, 8), 1, "f64", 7),      # one- and two-cell local kernels,
               fi.open_batio3("vacuum_72x16x8", (72, 16, 8), 1, "f64", 8)):                    # tensor-copy tiles
        wv.materials = [[replace(wv.materials[0][0], active=0)]]
        gv = fe.Grid.from_workload(wv)
        gv.precompute_tensor()
        Pv = gv.state(wv.P0)
        assert not gv.rhs(Pv, fi.TERM_ALL).any()
        for integ in (fi.EULER, fi.RK4):
            gv.step(Pv, wv.dt, 3, integ, fi.TERM_ALL)
            assert torch.equal(Pv, gv.state(wv.P0))
        assert np.all(gv.energy(Pv)[:, :5] == 0.0)
        gv.close()
    # the smallest grid: 4 x 4 x 4 periodic and 2 x 2 x 2 open, against the direct sum
    for n, per, img in (((4, 4, 4), (1, 1, 1), (2, 2, 2)), ((2, 2, 2), (0, 0, 0), (0, 0, 0))):
        ws = workload_from_random(97, n, per, img, batch=1)
        gs = fe.Grid.from_workload(ws)
        gs.precompute_tensor()
        os_ = orc.Oracle(oracle_problem(ws), elec="direct")
        assert rel_l2(gs.rhs(gs.state(ws.P0), fi.TERM_ALL).cpu().numpy()[0], os_.rhs(ws.P0[0], fi.TERM_ALL)) < TOL_RHS64, n
        gs.close()


@pytest.mark.parametrize("integ", [fi.EULER, fi.HEUN, fi.RK4])
def test_graph_replay_equals_eager_stepping(fe, integ):
    """fe_step(n) with n large replays a CUDA graph of one unit of steps; it must give bit-identical results to n single
    eager steps, also after a coefficient change (graph invalidated) and with an odd number of Euler steps."""
    w = workload_from_random(71, (8, 8, 4), (0, 1, 0), (0, 2, 0), batch=2)
    g = _grid(fe, w)
    for nsteps in (41, 64):
        Pa, Pb = g.state(w.P0), g.state(w.P0)
        g.step(Pa, 5e-3, nsteps, integ, fi.TERM_ALL)
        for _ in range(nsteps):
            g.step(Pb, 5e-3, 1, integ, fi.TERM_ALL)
        assert np.array_equal(Pa.cpu().numpy(), Pb.cpu().numpy())
        g.set_external_field(0, (0.01 * nsteps, 0.0, -0.02))          # invalidates the cached graph
    o = orc.Oracle(oracle_problem(w, 1), elec="direct")
    Pc = g.state(w.P0)
    g.step(Pc, 5e-3, 30, integ, fi.TERM_ALL)
    assert rel_l2(Pc.cpu().numpy()[1], o.step(w.P0[1], 5e-3, 30, integ, fi.TERM_ALL)) < 1e-11

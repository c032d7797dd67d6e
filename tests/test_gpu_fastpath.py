"""-m gpu parity tests of the size-specialised register FFT passes (fe_fft2_*.cu): grids large enough that every
axis takes the fast kernels (transform lengths 64 / 128 / 256 / 512, pruned and unpruned), against the CPU oracle
(oracle-FFT O8, itself pinned to the direct sum), and full-size checks of configs 5a / 5b against the closed-form
tensor entry, one sampled output at a time."""
import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc
from gpu_util import rel_l2, oracle_problem, workload_from_random

pytestmark = pytest.mark.gpu

TOL_RHS64, TOL32 = 1e-10, 1e-4


@pytest.fixture(scope="module")
def fe():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2605_28800_b200 as fe
    fe.load()
    return fe


def _workload(n, periodic=(0, 0, 0), images=(0, 0, 0), batch=1, seed=77):
    w = fi.open_batio3("fast_%dx%dx%d" % n, n, batch, "f64", seed)
    w.periodic, w.pbc_images = tuple(periodic), tuple(images)
    return w


# padded lengths (Mc = m_x / 2, m_y, m_z) exercised:            x     y     z
@pytest.mark.parametrize("n,periodic,images", [
    ((64, 32, 32), (0, 0, 0), (0, 0, 0)),        #  64p   64p   64p
    ((128, 64, 32), (0, 0, 0), (0, 0, 0)),       # 128p  128p   64p
    ((256, 128, 64), (0, 0, 0), (0, 0, 0)),      # 256p  256p  128p
    ((32, 256, 128), (0, 0, 0), (0, 0, 0)),      # generic 512p 256p
    ((512, 32, 32), (0, 0, 0), (0, 0, 0)),       # 512p   64p   64p
    ((128, 64, 32), (1, 1, 0), (1, 1, 0)),       #  64    64    64p  (unpruned x, y)
    ((64, 64, 64), (0, 0, 1), (0, 0, 1)),        #  64p  128p   64   (unpruned z)
    ((256, 128, 16), (1, 1, 0), (1, 1, 0)),      # 128   128   generic
    ((1024, 4, 4), (1, 0, 0), (1, 0, 0)),        # the largest periodic axis the ABI admits, on x (unpruned 512), ...
    ((4, 1024, 4), (0, 1, 0), (0, 1, 0)),        # ... on y ...
    ((4, 4, 1024), (0, 0, 1), (0, 0, 1)),        # ... and on z (generic passes)
    ((512, 4, 4), (0, 0, 0), (0, 0, 0)),         # the largest open axis: 512 cells padded to 1024
])
def test_fast_passes_against_oracle_fft(fe, n, periodic, images):
    w = _workload(n, periodic, images)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    o = orc.Oracle(oracle_problem(w), elec="fft")
    P = g.state(w.P0)
    got = g.rhs(P, fi.TERM_ELEC).cpu().numpy()[0]
    want = o.rhs(w.P0[0], fi.TERM_ELEC)
    assert rel_l2(got, want) < TOL_RHS64
    got = g.rhs(P, fi.TERM_ALL).cpu().numpy()[0]
    want = o.rhs(w.P0[0], fi.TERM_ALL)
    assert rel_l2(got, want) < TOL_RHS64
    # sampled outputs against the O(N) direct sum per target (not the FFT)
    rng = np.random.default_rng(3)
    t = rng.integers(0, w.cells, size=6)
    Ed = orc.field_direct(o.p, o.table(), w.P0[0], targets=t)
    got_e = g.rhs(P, fi.TERM_ELEC).cpu().numpy()[0].reshape(3, -1)[:, t] / w.globals_[0].L
    assert np.max(np.abs(got_e - Ed)) < 1e-10 * np.max(np.abs(Ed))
    g.close()


@pytest.mark.parametrize("n,periodic,images", [
    ((64, 8, 8), (0, 0, 0), (0, 0, 0)),
    ((64, 8, 4), (1, 1, 0), (1, 1, 0)),
    ((128, 4, 8), (0, 1, 1), (0, 2, 2)),
])
def test_two_cell_local_kernel_heterogeneous(fe, n, periodic, images):
    """Rows of >= 64 cells take the two-cells-per-thread local kernel: material map with vacuum cells, Gm != 0,
    8th-order slots, E_ext, anisotropic cells, batch of 2, every term alone and all together; Heun and RK4 stages."""
    w = workload_from_random(61, n, periodic, images, batch=2)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P = g.state(w.P0)
    for b in range(2):
        o = orc.Oracle(oracle_problem(w, b), elec="direct")
        for terms in (fi.TERM_LANDAU, fi.TERM_GRADIENT, fi.TERM_ELEC, fi.TERM_EXT, fi.TERM_ALL):
            got = g.rhs(P, terms).cpu().numpy()[b]
            want = o.rhs(w.P0[b], terms)
            assert rel_l2(got, want) < TOL_RHS64, (b, terms)
            assert np.all(got[:, o.p.active == 0] == 0.0)
    o = orc.Oracle(oracle_problem(w, 1), elec="direct")
    for integ in (fi.EULER, fi.HEUN, fi.RK4):
        Pd = g.state(w.P0)
        g.step(Pd, 1e-2, 3, integ, fi.TERM_ALL)
        want = o.step(w.P0[1], 1e-2, 3, integ, fi.TERM_ALL)
        assert rel_l2(Pd.cpu().numpy()[1], want) < 1e-12, integ
    g.close()
    # the same problem in fp32 (material map, vacuum, periodic wrap in the register loaders of the two-cell kernel)
    g = fe.Grid.from_workload(w, dtype="f32")
    g.precompute_tensor()
    P32 = w.P0.astype(np.float32)
    got = g.rhs(g.state(P32), fi.TERM_ALL).cpu().numpy()[1].astype(np.float64)
    assert rel_l2(got, o.rhs(P32[1].astype(np.float64), fi.TERM_ALL)) < TOL32
    assert np.all(got[:, o.p.active == 0] == 0.0)
    Pd = g.state(P32)
    g.step(Pd, 1e-2, 3, fi.RK4, fi.TERM_ALL)
    assert rel_l2(Pd.cpu().numpy()[1].astype(np.float64), o.step(P32[1].astype(np.float64), 1e-2, 3, fi.RK4, fi.TERM_ALL)) < TOL32
    g.close()


def test_fast_passes_batch_and_fp32(fe):
    w = _workload((128, 64, 32), batch=3)
    o = [orc.Oracle(oracle_problem(w, b), elec="fft") for b in range(3)]
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    got = g.rhs(g.state(w.P0)).cpu().numpy()
    for b in range(3):
        assert rel_l2(got[b], o[b].rhs(w.P0[b])) < TOL_RHS64
    g.close()
    g = fe.Grid.from_workload(w, dtype="f32")
    g.precompute_tensor()
    P32 = w.P0.astype(np.float32)
    got = g.rhs(g.state(P32)).cpu().numpy()
    for b in range(3):
        assert rel_l2(got[b], o[b].rhs(P32[b].astype(np.float64))) < TOL32
    g.close()


def test_fast_passes_steps_and_energy(fe):
    """10 Euler steps and 3 RK4 steps on a grid that takes the fast kernels; energies against the oracle."""
    w = _workload((64, 32, 32))
    o = orc.Oracle(oracle_problem(w), elec="fft")
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P = g.state(w.P0)
    g.step(P, w.dt, 10, fi.EULER, fi.TERM_ALL)
    ref = o.step(w.P0[0], w.dt, 10, fi.EULER, fi.TERM_ALL)
    assert rel_l2(P.cpu().numpy()[0], ref) < 1e-11
    e, eo = g.energy(P)[0], o.energy(ref)
    assert np.allclose(e[:5], eo[:5], rtol=1e-9, atol=1e-10 * abs(eo[4]))
    g.step(P, 2 * w.dt, 3, fi.RK4, fi.TERM_ALL)
    ref = o.step(ref, 2 * w.dt, 3, fi.RK4, fi.TERM_ALL)
    assert rel_l2(P.cpu().numpy()[0], ref) < 1e-11
    g.close()


@pytest.mark.parametrize("cfg,dtype,tol", [("5a", "f64", 1e-10), ("5a", "f32", 1e-4), ("5b", "f64", 1e-10)])
def test_full_size_point_sources_against_closed_form(fe, cfg, dtype, tol):
    """Full-size configs 5a / 5b in the launch configuration bench.py times.  P = a few single polarised cells
    (corners, centre, random) => E_i(r) = -scale sum_s K_ij(r - r_s) p_s,j, with K from the oracle's closed form
    (orc.newell_entry), evaluated at sampled output cells one by one."""
    import torch
    w = fi.config5a(dtype) if cfg == "5a" else fi.config5b(dtype)
    nx, ny, nz = w.n
    g = fe.Grid.from_workload(w, dtype=dtype)
    g.precompute_tensor()
    rng = np.random.default_rng(11)
    src = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (nx // 2, ny // 2, nz // 2), (nx - 1, 0, nz // 3)]
    src += [tuple(int(rng.integers(0, m)) for m in w.n) for _ in range(3)]
    amp = rng.standard_normal((len(src), 3))
    tdt = torch.float64 if dtype == "f64" else torch.float32
    P = torch.zeros((w.batch, 3, nz, ny, nx), dtype=tdt, device="cuda:0")
    b = w.batch - 1
    for s, a in zip(src, amp):
        for c in range(3):
            P[b, c, s[2], s[1], s[0]] = float(a[c])
    if dtype == "f32":
        amp = amp.astype(np.float32).astype(np.float64)
    E = g.rhs(P, fi.TERM_ELEC)[b].cpu().numpy().astype(np.float64) / w.globals_[b].L
    gl = w.globals_[b]
    scale = 1.0 / (gl.eps0 * gl.epsB)
    cidx = ((0, 3, 4), (3, 1, 5), (4, 5, 2))
    targets = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (1, 0, 0), (nx // 2, ny // 2 + 1, nz // 2)]
    targets += [tuple(int(rng.integers(0, m)) for m in w.n) for _ in range(8)]
    targets += [(min(s[0] + 1, nx - 1), s[1], s[2]) for s in src]
    emax = 0.0
    errs = []
    for t in targets:
        want = np.zeros(3)
        for s, a in zip(src, amp):
            off = (t[0] - s[0], t[1] - s[1], t[2] - s[2])
            K = [orc.newell_entry(c6, off, w.d) for c6 in range(6)]
            for i in range(3):
                want[i] -= scale * sum(K[cidx[i][j]] * a[j] for j in range(3))
        got = E[:, t[2], t[1], t[0]]
        errs.append(np.max(np.abs(got - want)))
        emax = max(emax, np.max(np.abs(want)))
    # far-field entries are ~1e-8 of the self term: the bound is relative to the largest sampled field
    assert max(errs) < tol * emax, (max(errs), emax)
    # linearity / finiteness everywhere
    assert np.isfinite(E).all()
    if w.batch > 1:
        assert float(g.rhs(P, fi.TERM_ELEC)[0].abs().max()) == 0.0      # other members untouched
    g.close()


@pytest.mark.parametrize("n,periodic,images,dtype", [
    ((64, 32, 32), (0, 0, 0), (0, 0, 0), "f64"),
    ((128, 256, 128), (0, 0, 0), (0, 0, 0), "f64"),      # bulk-copy y pass (512), 256-point fused z pass
    ((64, 128, 64), (0, 0, 0), (0, 0, 0), "f32"),        # bulk-copy y pass (256) in fp32
    ((256, 128, 16), (1, 1, 0), (1, 1, 0), "f64"),       # unpruned x, y; generic z
    ((16, 16, 8), (0, 0, 0), (0, 0, 0), "f64"),          # generic passes only
    ((72, 40, 36), (0, 0, 0), (0, 0, 0), "f64"),         # open axes that are not powers of two (partial pruning)
    ((36, 140, 70), (0, 0, 0), (0, 0, 0), "f32"),
    ((12, 10, 6), (0, 0, 0), (0, 0, 0), "f64"),
])
def test_no_write_outside_the_caller_buffers(fe, n, periodic, images, dtype):
    """Guard bands around the workspace, the state and the output (compute-sanitizer is closed on the pool): every byte
    outside the ranges the ABI documents must be untouched after precompute, rhs, step and energy."""
    import torch
    from paper_2605_28800_b200 import binding as bd
    w = _workload(n, periodic, images)
    g = fe.Grid.from_workload(w, dtype=dtype)
    need, guard = bd.fe_workspace_bytes(g.h), 1 << 20
    big = torch.full((need + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda:0")
    ws = big[guard:guard + need]
    assert ws.data_ptr() % 256 == 0
    bd.fe_bind_workspace(g.h, ws)
    g.ws = big
    g.precompute_tensor()
    tdt = torch.float64 if dtype == "f64" else torch.float32
    numel = int(np.prod(g.state_shape))
    pad = 4096
    bufP = torch.full((numel + 2 * pad,), 7.0, dtype=tdt, device="cuda:0")
    bufO = torch.full((numel + 2 * pad,), 7.0, dtype=tdt, device="cuda:0")
    P = bufP[pad:pad + numel].view(g.state_shape)
    O = bufO[pad:pad + numel].view(g.state_shape)
    P.copy_(torch.from_numpy(w.P0).to(tdt))
    bd.fe_rhs(g.h, P, O, fi.TERM_ALL)
    g.step(P, w.dt, 3, fi.EULER, fi.TERM_ALL)
    g.step(P, w.dt, 1, fi.RK4, fi.TERM_ALL)
    g.energy(P)
    torch.cuda.synchronize()
    assert bool((big[:guard] == 0xA5).all()) and bool((big[guard + need:] == 0xA5).all())
    for buf in (bufP, bufO):
        assert bool((buf[:pad] == 7.0).all()) and bool((buf[pad + numel:] == 7.0).all())
    assert bool(torch.isfinite(P).all()) and bool(torch.isfinite(O).all())
    g.close()


@pytest.mark.parametrize("n,periodic,images", [
    ((12, 10, 6), (0, 0, 0), (0, 0, 0)),          # generic passes, padded 32 x 32 x 16
    ((72, 40, 36), (0, 0, 0), (0, 0, 0)),         # fast passes with partial pruning: Mc = 128, My = 128, Mz = 128
    ((36, 140, 70), (0, 0, 0), (0, 0, 0)),        # Mc = 64, bulk-copy y pass (512, 140 data rows), Mz = 256 (70 data rows)
    ((64, 36, 24), (1, 0, 0), (1, 0, 0)),         # periodic power-of-two x, open y and z of arbitrary length
    ((100, 64, 12), (0, 1, 0), (0, 1, 0)),        # Mc = 128 (100 reals per row), periodic y, generic z
    ((100, 64, 40), (0, 0, 0), (0, 0, 0)),        # tiled layouts, barrier-free x kernels at Mc = 128 with 100 of 128 reals per row
    ((40, 32, 20), (0, 0, 0), (0, 0, 0)),         # ... and at Mc = 64 with 40 of 64
    ((130, 6, 6), (0, 0, 0), (0, 0, 0)),          # Mc = 256 beside generic y and z: row-major spectra, 108 rows (not a multiple of 16)
])
def test_open_axes_of_arbitrary_length(fe, n, periodic, images):
    """Open axes need not be powers of two (the paper's own grids are 128 x 128 x 36, 80 x 80 x 80 ...): they are
    zero-padded to the next power of two >= 2 n and the pruned passes skip the padding.  RHS against oracle-FFT (which
    pads to 2 n exactly) and against the direct sum at sampled cells; a few Euler steps; guard bands."""
    w = _workload(n, periodic, images)
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    o = orc.Oracle(oracle_problem(w), elec="fft")
    P = g.state(w.P0)
    for terms in (fi.TERM_ELEC, fi.TERM_ALL):
        assert rel_l2(g.rhs(P, terms).cpu().numpy()[0], o.rhs(w.P0[0], terms)) < TOL_RHS64, terms
    t = np.random.default_rng(4).integers(0, w.cells, size=5)
    Ed = orc.field_direct(o.p, o.table(), w.P0[0], targets=t)
    got_e = g.rhs(P, fi.TERM_ELEC).cpu().numpy()[0].reshape(3, -1)[:, t] / w.globals_[0].L
    assert np.max(np.abs(got_e - Ed)) < 1e-10 * np.max(np.abs(Ed))
    g.step(P, w.dt, 8, fi.EULER, fi.TERM_ALL)
    assert rel_l2(P.cpu().numpy()[0], o.step(w.P0[0], w.dt, 8, fi.EULER, fi.TERM_ALL)) < 1e-11
    e, eo = g.energy(P)[0], o.energy(o.step(w.P0[0], w.dt, 8, fi.EULER, fi.TERM_ALL))
    assert np.allclose(e[:5], eo[:5], rtol=1e-9, atol=1e-10 * abs(eo[4]))
    g.close()


def test_odd_open_x_axis_is_refused(fe):
    with pytest.raises(fe.FeError) as ei:
        fe.Grid((13, 8, 8), (1.0, 1.0, 1.0))
    assert ei.value.status == fe.FE_EINVAL
    with pytest.raises(fe.FeError):
        fe.Grid((12, 8, 8), (1.0, 1.0, 1.0), periodic=(1, 0, 0))      # periodic axes stay powers of two


@pytest.mark.parametrize("n,batch,dtype", [
    ((128, 128, 32), 2, "f64"),        # x 128p, y 256p: ROWS = 32 per X task, 192 planes through a ring of 24
    ((256, 256, 32), 1, "f64"),        # x 256p, y 512p: the kernels of config 5a
    ((200, 128, 32), 1, "f64"),        # partial pruning on x (200 of 256 reals)
    ((256, 256, 32), 1, "f32"),
])
def test_fused_xy_pass_through_the_l2_ring(fe, n, batch, dtype):
    """FE_OPT_FUSE_XY: x and y passes in one cooperative kernel, half spectra handed over through a
    ring of planes.  Both settings of the option against oracle-FFT, against each other, over many steps (the ring and its
    counters are reused by every launch) and under CUDA-graph replay; no wait may ever time out."""
    w = _workload(n, batch=batch)
    tol = TOL_RHS64 if dtype == "f64" else TOL32
    P0 = w.P0 if dtype == "f64" else w.P0.astype(np.float32).astype(np.float64)
    o = orc.Oracle(oracle_problem(w, batch - 1), elec="fft")
    want = o.rhs(P0[batch - 1], fi.TERM_ELEC)
    g = fe.Grid.from_workload(w, dtype=dtype)
    g.precompute_tensor()
    P = g.state(P0)
    res = {}
    for fuse in (1, 0):
        g.set_option(fe.FE_OPT_FUSE_XY, fuse)
        assert g.get_option(fe.FE_OPT_FUSE_XY) == fuse
        g.profile(True)
        res[fuse] = g.rhs(P, fi.TERM_ELEC).cpu().numpy().astype(np.float64)
        kinds = {k for k, (ms, cnt) in g.profile_read().items() if cnt}
        g.profile(False)
        assert ("xyfwd" in kinds) == bool(fuse) and ("xfwd" in kinds) == (not fuse)
        assert rel_l2(res[fuse][batch - 1], want) < tol
    assert rel_l2(res[1], res[0]) < (1e-13 if dtype == "f64" else 1e-5)
    # 40 Euler steps in one call (graph replay) with the fused pass against 40 single steps without it
    g.set_option(fe.FE_OPT_FUSE_XY, 1)
    Pa = g.state(P0)
    g.step(Pa, w.dt, 40, fi.EULER, fi.TERM_ALL)
    g.set_option(fe.FE_OPT_FUSE_XY, 0)
    Pb = g.state(P0)
    for _ in range(40):
        g.step(Pb, w.dt, 1, fi.EULER, fi.TERM_ALL)
    assert rel_l2(Pa.cpu().numpy(), Pb.cpu().numpy()) < (1e-12 if dtype == "f64" else 1e-4)
    assert g.get_option(fe.FE_OPT_XY_TIMEOUTS) == 0
    g.close()


@pytest.mark.parametrize("n,batch,slabs", [
    ((256, 256, 32), 1, 4),           # the x kernels of config 5a, four slabs of 8 planes
    ((256, 128, 24), 2, 5),           # two members, slabs of 4 / 5 planes
    ((256, 64, 32), 1, 32),           # one plane per slab
])
def test_x_inverse_hands_e_elec_to_the_local_step_slab_by_slab(fe, n, batch, slabs):
    """FE_OPT_XL_SLABS (E_elec "consumed without a round trip"): the x inverse pass and the local step
    run slab by slab, E_elec of a slab in the first planes of the E buffer.  Against the oracle, against the unsliced path (bitwise: the
    same kernels compute the same cells), every integrator's stage epilogue, and under graph replay."""
    w = _workload(n, batch=batch)
    o = orc.Oracle(oracle_problem(w, batch - 1), elec="fft")
    want = o.rhs(w.P0[batch - 1], fi.TERM_ALL)
    g = fe.Grid.from_workload(w, dtype="f64")
    g.precompute_tensor()
    P = g.state(w.P0)
    res = {}
    for s in (slabs, 0):
        g.set_option(fe.FE_OPT_XL_SLABS, s)
        assert g.get_option(fe.FE_OPT_XL_SLABS) == s
        g.profile(True)
        res[s] = g.rhs(P, fi.TERM_ALL).cpu().numpy()
        counts = {k: cnt for k, (ms, cnt) in g.profile_read().items()}
        g.profile(False)
        assert counts["xinv"] == counts["local"] == (s if s else 1)
        assert rel_l2(res[s][batch - 1], want) < TOL_RHS64
    assert np.array_equal(res[slabs], res[0])
    for integ, nst in ((fi.EULER, 12), (fi.HEUN, 4), (fi.RK4, 3), (fi.AB3M2, 5)):
        g.set_option(fe.FE_OPT_XL_SLABS, slabs)
        Pa = g.state(w.P0)
        g.step(Pa, w.dt, nst, integ, fi.TERM_ALL)
        g.set_option(fe.FE_OPT_XL_SLABS, 0)
        Pb = g.state(w.P0)
        g.step(Pb, w.dt, nst, integ, fi.TERM_ALL)
        assert np.array_equal(Pa.cpu().numpy(), Pb.cpu().numpy())
    # both options at once: fused x + y forward pass and the slab hand-over
    if n[1] in (128, 256):
        g.set_option(fe.FE_OPT_XL_SLABS, slabs)
        g.set_option(fe.FE_OPT_FUSE_XY, 1)
        Pa = g.state(w.P0)
        g.step(Pa, w.dt, 6, fi.EULER, fi.TERM_ALL)
        g.set_option(fe.FE_OPT_XL_SLABS, 0)
        g.set_option(fe.FE_OPT_FUSE_XY, 0)
        Pb = g.state(w.P0)
        g.step(Pb, w.dt, 6, fi.EULER, fi.TERM_ALL)
        assert rel_l2(Pa.cpu().numpy(), Pb.cpu().numpy()) < 1e-13
        assert g.get_option(fe.FE_OPT_XY_TIMEOUTS) == 0
    g.close()


def test_calls_on_a_side_stream(fe):
    """Every call takes the caller's stream (the binding passes torch's current stream): right-hand side, steps under graph
    replay, energies and the no-allocation energy entry point on a non-default stream give what the default stream gives."""
    import torch
    w = _workload((128, 32, 16))
    g = fe.Grid.from_workload(w)
    g.precompute_tensor()
    P = g.state(w.P0)
    ref_rhs = g.rhs(P, fi.TERM_ALL).clone()
    Pr = g.state(w.P0)
    g.step(Pr, w.dt, 30, fi.EULER, fi.TERM_ALL)
    ref_e = g.energy(Pr)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        got_rhs = g.rhs(P, fi.TERM_ALL).clone()
        Ps = g.state(w.P0)
        g.step(Ps, w.dt, 30, fi.EULER, fi.TERM_ALL)
        got_e = g.energy(Ps)
        out = torch.empty((1, 8), dtype=torch.float64, device=P.device)
        g.energy_noalloc(Ps, out, fi.TERM_ALL)
    side.synchronize()
    assert torch.equal(got_rhs, ref_rhs) and torch.equal(Ps, Pr)
    assert np.array_equal(got_e, ref_e) and np.array_equal(out.cpu().numpy(), ref_e)
    g.close()

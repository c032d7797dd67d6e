"""Pins for the oracle's electrostatic field (O3 direct sum, O8 oracle-FFT).
PAPER.md:66-76 (Eq. 5-6); north_star: slab depolarisation -P/eps0, brute-force FFT = direct sum.
"""
import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc

MAT = [fi.Landau(a1=(0, 0, 0))]


def _problem(n, d=(1.0, 1.0, 1.0), periodic=(0, 0, 0), images=(0, 0, 0), eps0=1.0, epsB=1.0, zero_mode=True):
    g = fi.Globals(G11=1, G12=0, G44=0, G44p=0, eps0=eps0, epsB=epsB)
    return orc.Problem(n=n, d=d, periodic=periodic, pbc_images=images, materials=MAT, g=g, zero_mode=zero_mode)


def _field_python_loops(p, K, P):
    """Independent restatement of O3 in pure Python (tiny grids only)."""
    nx, ny, nz = p.n
    cidx = ((0, 3, 4), (3, 1, 5), (4, 5, 2))
    E = np.zeros_like(P)
    idx = lambda r, rp, a: ((r - rp) % p.n[a]) if p.periodic[a] else (r - rp + p.n[a] - 1)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                for zp in range(nz):
                    for yp in range(ny):
                        for xp in range(nx):
                            k = K[:, idx(z, zp, 2), idx(y, yp, 1), idx(x, xp, 0)]
                            for i in range(3):
                                for j in range(3):
                                    E[i, z, y, x] -= k[cidx[i][j]] * P[j, zp, yp, xp] / (p.g.eps0 * p.g.epsB)
    return E


def test_direct_sum_matches_python_loops():
    p = _problem((3, 2, 2), d=(0.9, 1.1, 0.7), periodic=(0, 1, 0), images=(0, 1, 0), eps0=0.7, epsB=1.3)
    K = orc.tensor_table(p)
    P = np.random.default_rng(0).standard_normal(p.shape)
    np.testing.assert_allclose(orc.field_direct(p, K, P), _field_python_loops(p, K, P), rtol=1e-13, atol=1e-15)
    t = np.array([0, 5, 11])
    np.testing.assert_allclose(orc.field_direct(p, K, P, targets=t), orc.field_direct(p, K, P).reshape(3, -1)[:, t],
                               rtol=1e-15)


@pytest.mark.parametrize("n,periodic,images", [
    ((16, 16, 8), (0, 0, 0), (0, 0, 0)),        # config 1 grid
    ((7, 5, 3), (0, 0, 0), (0, 0, 0)),
    ((64, 4, 4), (0, 1, 1), (0, 2, 2)),         # cut of config 2
    ((8, 8, 4), (1, 1, 0), (2, 2, 0)),          # config 4 geometry
    ((8, 4, 6), (1, 0, 0), (3, 0, 0)),
])
def test_P5_fft_convolution_equals_direct_sum(n, periodic, images):
    p = _problem(n, d=(1.0, 1.0, 1.0), periodic=periodic, images=images, eps0=0.5, epsB=2.0)
    K = orc.tensor_table(p)
    P = np.random.default_rng(1).standard_normal(p.shape)
    Ed = orc.field_direct(p, K, P)
    Ef = orc.field_fft(p, K, P)
    assert np.linalg.norm(Ef - Ed) / np.linalg.norm(Ed) < 1e-13
    # the threaded library FFT of the all-cores CPU baseline is pinned by the same direct sum
    Ew = orc.field_fft(p, K, P, workers=2)
    assert np.linalg.norm(Ew - Ed) / np.linalg.norm(Ed) < 1e-13


def test_P4i_infinite_film_depolarisation_is_minus_P_over_eps0():
    """Periodic in-plane + zero-mode rule: uniform P_perp gives E_perp = -P/(eps0 epsB) in every cell,
    uniform in-plane P gives no field."""
    p = _problem((4, 4, 3), periodic=(1, 1, 0), images=(2, 2, 0), eps0=0.8, epsB=1.5)
    K = orc.tensor_table(p)
    P = np.zeros(p.shape)
    P[2] = 0.37
    E = orc.field_direct(p, K, P)
    np.testing.assert_allclose(E[2], -0.37 / (0.8 * 1.5), rtol=1e-12)
    np.testing.assert_allclose(E[:2], 0.0, atol=1e-13)
    P = np.zeros(p.shape)
    P[0] = 0.5
    P[1] = -0.2
    np.testing.assert_allclose(orc.field_direct(p, K, P), 0.0, atol=1e-13)
    # same with the open axis first (config 2 geometry)
    p = _problem((5, 4, 4), periodic=(0, 1, 1), images=(0, 2, 2), eps0=1.0)
    K = orc.tensor_table(p)
    P = np.zeros(p.shape)
    P[0] = 1.0
    E = orc.field_direct(p, K, P)
    np.testing.assert_allclose(E[0], -1.0, rtol=1e-12)
    np.testing.assert_allclose(E[1:], 0.0, atol=1e-13)


def test_P4ii_open_slab_average_field_is_body_demag_factor():
    """Uniformly polarised open slab: the volume-averaged field is -N_body P / eps0 with N_body the
    self-term of ONE cell of the slab's size, and N_zz -> 1 (E -> -P/eps0) as the slab gets thin."""
    n = (32, 32, 2)
    p = _problem(n, eps0=1.0)
    K = orc.tensor_table(p)
    P = np.zeros(p.shape)
    P[2] = 1.0
    E = orc.field_fft(p, K, P)
    Nzz = orc.newell_entry(2, (0, 0, 0), (32.0, 32.0, 2.0))
    assert E[2].mean() == pytest.approx(-Nzz, rel=1e-12)
    assert abs(E[0].mean()) < 1e-14 and abs(E[1].mean()) < 1e-14
    assert 0.85 < Nzz < 1.0
    thin = orc.newell_entry(2, (0, 0, 0), (4096.0, 4096.0, 1.0))
    assert thin == pytest.approx(1.0, abs=2e-3) and thin < 1.0


def test_P4iii_open_cube_average_field_is_one_third():
    p = _problem((6, 6, 6), eps0=2.0, epsB=3.0)
    K = orc.tensor_table(p)
    P = np.zeros(p.shape)
    P[0], P[1], P[2] = 0.3, -0.4, 0.5
    E = orc.field_direct(p, K, P)
    for i, v in enumerate((0.3, -0.4, 0.5)):
        assert E[i].mean() == pytest.approx(-v / (3 * 2.0 * 3.0), rel=1e-12)


def test_field_of_single_polarised_cell_is_the_tensor_column():
    """A wrong transpose / sign / index in the pair sum fails here."""
    n = (4, 3, 5)
    p = _problem(n, d=(0.9, 1.1, 0.7))
    K = orc.tensor_table(p)
    P = np.zeros(p.shape)
    src = (2, 1, 3)            # x, y, z
    P[1, src[2], src[1], src[0]] = 1.0          # Py
    E = orc.field_direct(p, K, P)
    tgt = (0, 2, 1)
    off = tuple(tgt[a] - src[a] for a in range(3))
    d = (0.9, 1.1, 0.7)
    assert E[0, tgt[2], tgt[1], tgt[0]] == pytest.approx(-orc.newell_entry(3, off, d), rel=1e-13)   # xy
    assert E[1, tgt[2], tgt[1], tgt[0]] == pytest.approx(-orc.newell_entry(1, off, d), rel=1e-13)   # yy
    assert E[2, tgt[2], tgt[1], tgt[0]] == pytest.approx(-orc.newell_entry(5, off, d), rel=1e-13)   # yz


def test_electrostatic_operator_is_symmetric_positive():
    """K is symmetric (E . P' = E' . P) and F_elec = -1/2 V sum E.P >= 0 (it is a field energy)."""
    for periodic, images in [((0, 0, 0), (0, 0, 0)), ((1, 1, 0), (2, 2, 0)), ((0, 1, 0), (0, 2, 0))]:
        p = _problem((4, 4, 3), d=(1.0, 0.8, 1.2), periodic=periodic, images=images)
        K = orc.tensor_table(p)
        rng = np.random.default_rng(2)
        P1, P2 = rng.standard_normal(p.shape), rng.standard_normal(p.shape)
        E1, E2 = orc.field_direct(p, K, P1), orc.field_direct(p, K, P2)
        assert np.sum(E1 * P2) == pytest.approx(np.sum(E2 * P1), rel=1e-12)
        assert -0.5 * np.sum(E1 * P1) > 0


def test_fully_periodic_box_zero_mode_and_plane_wave():
    """Three periodic axes (reading A4, last case): the mean of the kernel is removed, so (i) a uniformly polarised
    periodic crystal feels no field, (ii) the field of a longitudinal plane wave P = e_x cos(2 pi x / n) approaches the
    continuum value -P / (eps0 epsB) (all of it is bound charge), a transverse one P = e_y cos(2 pi x / n) ~ 0, as
    the image sum grows, and (iii) with zero_mode off the mean is left in (plain image sum, Lorentz-type value 1/3
    per diagonal component for cubic cells)."""
    n = (8, 8, 8)
    p = _problem(n, periodic=(1, 1, 1), images=(3, 3, 3), eps0=0.5, epsB=2.0)
    K = orc.tensor_table(p)
    for comp in range(6):
        assert abs(K[comp].sum()) < 1e-12
    P = np.zeros(p.shape)
    P[0], P[1], P[2] = 0.3, -0.2, 0.7
    np.testing.assert_allclose(orc.field_direct(p, K, P), 0.0, atol=1e-12)
    x = np.arange(8)
    wave = np.cos(2 * np.pi * x / 8)[None, None, :]
    P = np.zeros(p.shape)
    P[0] += wave
    E = orc.field_fft(p, K, P)
    # longitudinal response of the cell-averaged, image-summed kernel at k = 2 pi / (8 cells): within 1 % of the continuum
    nodes = np.abs(wave[0, 0]) < 0.1
    ratio = E[0, 0, 0, ~nodes] / (-wave[0, 0, ~nodes] / (0.5 * 2.0))
    assert np.allclose(ratio, ratio[0], rtol=1e-10) and 0.99 < ratio[0] < 1.0
    assert np.max(np.abs(E[0, 0, 0, nodes])) < 1e-12
    np.testing.assert_allclose(E[1:], 0.0, atol=1e-12)
    P = np.zeros(p.shape)
    P[1] += wave                                     # transverse: no bound charge
    Et = orc.field_fft(p, K, P)
    assert np.max(np.abs(Et)) < 0.05 * np.max(np.abs(E))
    # FFT = direct sum on this geometry too
    Pr = np.random.default_rng(2).standard_normal(p.shape)
    Ed, Ef = orc.field_direct(p, K, Pr), orc.field_fft(p, K, Pr)
    assert np.linalg.norm(Ef - Ed) / np.linalg.norm(Ed) < 1e-13
    p0 = _problem(n, periodic=(1, 1, 1), images=(3, 3, 3), eps0=0.5, epsB=2.0)
    p0.zero_mode = False
    K0 = orc.tensor_table(p0)
    for comp in range(3):                            # cubic symmetry: each diagonal sum = trace / 3, trace of the sum = 1
        assert K0[comp].sum() == pytest.approx(1.0 / 3.0, abs=1e-12)
    for comp in range(3, 6):
        assert abs(K0[comp].sum()) < 1e-12

"""Pins for the oracle's cell-averaged dipolar tensor (O3, readings A3/A4).
PAPER.md:66-76 (Eq. 5-6) applied to cell-wise constant P; the construction of ref. [40].

P2: trace = 1 at the origin / 0 elsewhere, cube self-term 1/3, parities, additivity.
P6: closed form = triangle-weighted quadrature of d_i d_j (1/r) (the definition), point-dipole limit.
P10: periodic table = brute-force image sums of the open-boundary entry (centred window).
"""
import itertools
from functools import lru_cache

import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc

G = fi.Globals(G11=1, G12=0, G44=0, G44p=0, eps0=1.0, epsB=1.0)
MAT = [fi.Landau(a1=(0, 0, 0))]


def _problem(n, d=(1.0, 1.0, 1.0), periodic=(0, 0, 0), images=(0, 0, 0), zero_mode=True):
    return orc.Problem(n=n, d=d, periodic=periodic, pbc_images=images, materials=MAT, g=G, zero_mode=zero_mode)


def test_P2_cube_self_term_and_traces():
    d = (1.0, 1.0, 1.0)
    for c in range(3):
        assert orc.newell_entry(c, (0, 0, 0), d) == pytest.approx(1.0 / 3.0, abs=1e-15)
    for c in range(3, 6):
        assert abs(orc.newell_entry(c, (0, 0, 0), d)) < 1e-30
    for dd in [(1.0, 2.0, 0.5), (0.3, 0.3, 1.7)]:
        assert sum(orc.newell_entry(c, (0, 0, 0), dd) for c in range(3)) == pytest.approx(1.0, abs=1e-15)
        for off in [(1, 0, 0), (1, 1, 1), (3, 2, 1), (0, 0, 5), (17, 4, -9), (100, 37, 64)]:
            assert abs(sum(orc.newell_entry(c, off, dd) for c in range(3))) < 1e-17


def test_P2_parities():
    d = (0.9, 1.1, 0.7)
    odd = {3: (0, 1), 4: (0, 2), 5: (1, 2)}
    off = np.array([3, 2, 4])
    for c in range(6):
        base = orc.newell_entry(c, off, d)
        assert orc.newell_entry(c, -off, d) == base                      # N(-R) = N(R)
        for a in range(3):
            s = off.copy()
            s[a] = -s[a]
            sign = -1.0 if (c in odd and a in odd[c]) else 1.0
            assert orc.newell_entry(c, s, d) == pytest.approx(sign * base, rel=1e-15, abs=1e-30)


def test_P2_axis_permutation_of_components():
    d = (0.9, 1.1, 0.7)
    # N_yy(X,Y,Z; dx,dy,dz) = N_xx(Y,X,Z; dy,dx,dz), N_xz(X,Y,Z) = N_xy(X,Z,Y; dx,dz,dy), ...
    assert orc.newell_entry(1, (3, 2, 4), d) == pytest.approx(orc.newell_entry(0, (2, 3, 4), (1.1, 0.9, 0.7)), rel=1e-15)
    assert orc.newell_entry(2, (3, 2, 4), d) == pytest.approx(orc.newell_entry(0, (4, 2, 3), (0.7, 1.1, 0.9)), rel=1e-15)
    assert orc.newell_entry(4, (3, 2, 4), d) == pytest.approx(orc.newell_entry(3, (3, 4, 2), (0.9, 0.7, 1.1)), rel=1e-15)
    assert orc.newell_entry(5, (3, 2, 4), d) == pytest.approx(orc.newell_entry(3, (2, 4, 3), (1.1, 0.7, 0.9)), rel=1e-15)


def test_P2_additivity_block_equals_big_cell():
    """(1/N) sum_{r,r'} N_ij(r - r') over an nx*ny*nz block = self-term of one cell of the block's size."""
    n, d = (4, 3, 2), (0.5, 0.75, 1.5)
    K = orc.tensor_table(_problem(n, d))
    big = (n[0] * d[0], n[1] * d[1], n[2] * d[2])
    Ncells = n[0] * n[1] * n[2]
    for c in range(6):
        s = 0.0
        for tz, ty, tx in itertools.product(range(2 * n[2] - 1), range(2 * n[1] - 1), range(2 * n[0] - 1)):
            mult = (n[0] - abs(tx - n[0] + 1)) * (n[1] - abs(ty - n[1] + 1)) * (n[2] - abs(tz - n[2] + 1))
            s += mult * K[c, tz, ty, tx]
        assert s / Ncells == pytest.approx(orc.newell_entry(c, (0, 0, 0), big), abs=1e-14)
    # a cubic block of cubes has demag factor 1/3
    K = orc.tensor_table(_problem((3, 3, 3)))
    s = sum((3 - abs(tx - 2)) * (3 - abs(ty - 2)) * (3 - abs(tz - 2)) * K[0, tz, ty, tx]
            for tz, ty, tx in itertools.product(range(5), repeat=3))
    assert s / 27 == pytest.approx(1.0 / 3.0, abs=1e-14)


def _quadrature(comp, off, d, npts=20):
    """-(1/(4 pi V)) int (dx-|u|)(dy-|v|)(dz-|w|) T_ij(R + (u,v,w)) du dv dw, Gauss-Legendre on each
    half interval (the triangle weight has a kink at 0).  T_ij = 3 r_i r_j / r^5 - delta_ij / r^3."""
    x, w = np.polynomial.legendre.leggauss(npts)
    i, j = {0: (0, 0), 1: (1, 1), 2: (2, 2), 3: (0, 1), 4: (0, 2), 5: (1, 2)}[comp]
    nodes, weights = [], []
    for a in range(3):
        h = d[a]
        u = np.concatenate([-h / 2 + (h / 2) * x, h / 2 + (h / 2) * x])
        ww = np.concatenate([(h / 2) * w, (h / 2) * w]) * (h - np.abs(u))
        nodes.append(u)
        weights.append(ww)
    U, Vv, W = np.meshgrid(*nodes, indexing="ij")
    WW = weights[0][:, None, None] * weights[1][None, :, None] * weights[2][None, None, :]
    r = [off[0] * d[0] + U, off[1] * d[1] + Vv, off[2] * d[2] + W]
    r2 = r[0] ** 2 + r[1] ** 2 + r[2] ** 2
    T = 3 * r[i] * r[j] / r2 ** 2.5 - (1.0 if i == j else 0.0) / r2 ** 1.5
    return -float(np.sum(WW * T)) / (4 * np.pi * d[0] * d[1] * d[2])


@pytest.mark.parametrize("off", [(2, 0, 0), (0, 2, 1), (2, 2, 2), (3, 2, 1), (6, 0, 0), (8, 5, 3), (12, 12, 1), (-7, 3, -6)])
@pytest.mark.parametrize("d", [(1.0, 1.0, 1.0), (1.0, 2.0, 0.5)])
def test_P6_closed_form_equals_quadrature_of_the_definition(off, d):
    for c in range(6):
        q = _quadrature(c, off, d, npts=24)
        assert orc.newell_entry(c, off, d) == pytest.approx(q, abs=2e-15), (c, off)


def test_P6_point_dipole_limit():
    d = (1.0, 1.0, 1.0)
    for off in [(64, 0, 0), (70, 33, -41), (0, 100, 100)]:
        R = np.array(off, dtype=float)
        r = np.linalg.norm(R)
        for c, (i, j) in enumerate([(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]):
            T = 3 * R[i] * R[j] / r ** 5 - (i == j) / r ** 3
            # next multipole correction is O((cell/r)^4) relative for cubes
            assert orc.newell_entry(c, off, d) == pytest.approx(-T / (4 * np.pi), abs=5 * abs(1 / (4 * np.pi * r ** 3)) / r ** 4 + 1e-30)


def test_table_matches_plain_entries_open():
    n, d = (5, 4, 3), (0.9, 1.1, 0.7)
    K = orc.tensor_table(_problem(n, d))
    assert K.shape == (6, 5, 7, 9)
    rng = np.random.default_rng(3)
    for _ in range(60):
        c = int(rng.integers(6))
        off = [int(rng.integers(-(n[a] - 1), n[a])) for a in range(3)]
        assert K[c, off[2] + n[2] - 1, off[1] + n[1] - 1, off[0] + n[0] - 1] == pytest.approx(
            orc.newell_entry(c, off, d), rel=1e-15, abs=1e-30)


@lru_cache(maxsize=None)
def _entry(c, i, j, k, d):
    return orc.newell_entry(c, (i, j, k), d)


def _min_images(j, n):
    """minimum-image offsets of circular index j (two at the tie), reading A4"""
    if 2 * j < n:
        return [j]
    if 2 * j > n:
        return [j - n]
    return [-j, j]


@pytest.mark.parametrize("periodic,images", [((0, 1, 0), (0, 2, 0)), ((1, 1, 0), (1, 2, 0)), ((0, 1, 1), (0, 1, 2))])
def test_P10_periodic_table_is_the_centred_window_image_sum(periodic, images):
    n, d = (4, 4, 2), (1.0, 0.8, 1.25)
    K = orc.tensor_table(_problem(n, d, periodic, images, zero_mode=False))
    T = [n[a] if periodic[a] else 2 * n[a] - 1 for a in range(3)]
    assert K.shape == (6, T[2], T[1], T[0])
    rng = np.random.default_rng(4)
    for _ in range(12):
        c = int(rng.integers(6))
        t = [int(rng.integers(T[a])) for a in range(3)]
        cand = [(_min_images(t[a], n[a]) if periodic[a] else [t[a] - (n[a] - 1)]) for a in range(3)]
        tot = 0.0
        for d0 in itertools.product(*cand):
            s = 0.0
            for q in itertools.product(*[range(-images[a], images[a] + 1) if periodic[a] else [0] for a in range(3)]):
                s += _entry(c, d0[0] + q[0] * n[0], d0[1] + q[1] * n[1], d0[2] + q[2] * n[2], d)
            tot += s / (len(cand[0]) * len(cand[1]) * len(cand[2]))
        assert K[c, t[2], t[1], t[0]] == pytest.approx(tot, abs=1e-16)


def test_periodic_table_is_exactly_even_or_odd():
    """The minimum-image rule with the averaged tie makes K(-d) = +-K(d) hold on the circle, so the
    operator is symmetric (needed for the energy pins)."""
    n = (4, 6, 3)
    K = orc.tensor_table(_problem(n, (1.0, 1.0, 1.0), (1, 1, 0), (2, 1, 0), zero_mode=True))
    Kf = K[:, ::-1]                                    # open z: d -> -d
    Kf = np.roll(Kf[:, :, ::-1, ::-1], (1, 1), axis=(2, 3))   # circular: j -> (-j) mod n
    np.testing.assert_allclose(Kf, K, rtol=0, atol=1e-17)


def test_A4_zero_mode_rule_plane_sums():
    n = (4, 4, 3)
    K = orc.tensor_table(_problem(n, (1.0, 1.0, 1.0), (1, 1, 0), (3, 3, 0), zero_mode=True))
    plane = K.sum(axis=(2, 3))                        # [6][Tz]
    target = np.zeros_like(plane)
    target[2, n[2] - 1] = 1.0                         # t_zz(0) = 1
    np.testing.assert_allclose(plane, target, atol=1e-14)
    # without the rule the residual decays slowly (this is why the rule exists)
    K0 = orc.tensor_table(_problem(n, (1.0, 1.0, 1.0), (1, 1, 0), (3, 3, 0), zero_mode=False))
    assert abs(K0.sum(axis=(2, 3))[2, n[2] - 1] - 1.0) > 1e-3

"""Pins for the oracle's spherical-harmonic transform (matrix level): `oracle.sph_matrix` is the
closed form of the real solid harmonics typed in from a textbook, so it is pinned by what DEFINES a Racah-normalised
real solid harmonic, none of which uses that closed form: it is a harmonic homogeneous polynomial, the 2l+1 of them are
orthogonal on the sphere with the angular norm 4 pi/(2l+1) of x^l, a rotation about z by phi mixes (m, -m) by the
angle m phi, and the low orders are the functions every table lists.  CPU only."""
from math import pi, sqrt

import numpy as np
import pytest

from oracle import oracle as O


def comps(l):
    return [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]


def dfact(n):
    r = 1
    while n > 1:
        r *= n
        n -= 2
    return r


def sphere_monomial(a, b, c):
    """int x^a y^b z^c dOmega over the unit sphere = 4 pi (a-1)!!(b-1)!!(c-1)!!/(a+b+c+1)!! for even a, b, c, else 0."""
    if a % 2 or b % 2 or c % 2:
        return 0.0
    return 4.0 * pi * dfact(a - 1) * dfact(b - 1) * dfact(c - 1) / dfact(a + b + c + 1)


@pytest.mark.parametrize("l", [0, 1, 2, 3])
def test_rows_are_harmonic_polynomials(l):
    """Laplacian of sum_c S[m,c] x^a y^b z^c vanishes identically: every monomial coefficient of the result is zero."""
    S = O.sph_matrix(l)
    cs = comps(l)
    for m in range(2 * l + 1):
        lap = {}
        for coef, (a, b, c) in zip(S[m], cs):
            for ax, e in enumerate((a, b, c)):
                if e >= 2:
                    k = [a, b, c]
                    k[ax] -= 2
                    lap[tuple(k)] = lap.get(tuple(k), 0.0) + coef * e * (e - 1)
        assert all(abs(v) < 1e-13 for v in lap.values()), (l, m, lap)


@pytest.mark.parametrize("l", [0, 1, 2, 3])
def test_orthogonal_on_the_sphere_with_the_norm_of_x_to_the_l(l):
    S = O.sph_matrix(l)
    cs = comps(l)
    G = np.array([[sphere_monomial(a + d, b + e, c + f) for (d, e, f) in cs] for (a, b, c) in cs])
    M = S @ G @ S.T
    assert np.allclose(M, 4.0 * pi / (2 * l + 1) * np.eye(2 * l + 1), rtol=0, atol=1e-13)
    assert G[0, 0] == pytest.approx(4.0 * pi / (2 * l + 1))       # the x^l component itself


@pytest.mark.parametrize("l", [1, 2, 3])
def test_rotation_about_z_mixes_m_and_minus_m(l):
    """R_{l,m}(Rz(phi) r) = cos(m phi) R_{l,m}(r) - sin(m phi) R_{l,-m}(r)  and
    R_{l,-m}(Rz(phi) r) = sin(m phi) R_{l,m}(r) + cos(m phi) R_{l,-m}(r), m > 0  (cos/sin(m phi_r) azimuth dependence,
    the sign convention R_{l,m} ~ cos(m phi), R_{l,-m} ~ sin(m phi) with positive leading coefficient); m = 0 invariant."""
    S = O.sph_matrix(l)
    cs = comps(l)
    rng = np.random.default_rng(3)

    def val(r):
        mono = np.array([r[0] ** a * r[1] ** b * r[2] ** c for (a, b, c) in cs])
        return S @ mono

    for _ in range(4):
        r = rng.standard_normal(3)
        phi = rng.uniform(0.2, 2.5)
        Rz = np.array([[np.cos(phi), -np.sin(phi), 0.0], [np.sin(phi), np.cos(phi), 0.0], [0.0, 0.0, 1.0]])
        v0, v1 = val(r), val(Rz @ r)
        assert v1[l] == pytest.approx(v0[l], abs=1e-12)
        for m in range(1, l + 1):
            c, s = np.cos(m * phi), np.sin(m * phi)
            assert v1[l + m] == pytest.approx(c * v0[l + m] - s * v0[l - m], abs=1e-12)
            assert v1[l - m] == pytest.approx(s * v0[l + m] + c * v0[l - m], abs=1e-12)


def test_tabulated_low_orders():
    """The functions every table lists (Racah normalisation): p = (y, z, x); d_0 = z^2 - (x^2+y^2)/2,
    d_{+-1} = sqrt3 (xz, yz), d_2 = sqrt3/2 (x^2-y^2), d_{-2} = sqrt3 xy; f_0 = z^3 - 3/2 (x^2+y^2) z,
    f_3 = sqrt(5/8) (x^3 - 3 x y^2), f_{-2} = sqrt15 xyz."""
    assert np.array_equal(O.sph_matrix(0), [[1.0]])
    assert np.array_equal(O.sph_matrix(1), [[0, 1, 0], [0, 0, 1], [1, 0, 0]])
    d = O.sph_matrix(2)                                          # columns xx xy xz yy yz zz
    s3 = sqrt(3.0)
    ref = [[0, s3, 0, 0, 0, 0], [0, 0, 0, 0, s3, 0], [-0.5, 0, 0, -0.5, 0, 1], [0, 0, s3, 0, 0, 0],
           [s3 / 2, 0, 0, -s3 / 2, 0, 0]]
    assert np.allclose(d, ref, rtol=0, atol=1e-15)
    f = O.sph_matrix(3)                                          # xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
    assert np.allclose(f[3], [0, 0, -1.5, 0, 0, 0, 0, -1.5, 0, 1], rtol=0, atol=1e-15)
    assert np.allclose(f[6], [sqrt(0.625), 0, 0, -3 * sqrt(0.625), 0, 0, 0, 0, 0, 0], rtol=0, atol=1e-15)
    assert np.allclose(f[1], [0, 0, 0, 0, sqrt(15.0), 0, 0, 0, 0, 0], rtol=0, atol=1e-15)


def test_contaminants_are_projected_out():
    """r^2 (the s-type combination of a Cartesian d shell) and r^2 x, r^2 y, r^2 z (the p-type ones of an f shell) are
    orthogonal on the sphere to every pure function: S G v = 0."""
    for l, vecs in ((2, [{(2, 0, 0): 1, (0, 2, 0): 1, (0, 0, 2): 1}]),
                    (3, [{(3, 0, 0): 1, (1, 2, 0): 1, (1, 0, 2): 1}, {(2, 1, 0): 1, (0, 3, 0): 1, (0, 1, 2): 1},
                         {(2, 0, 1): 1, (0, 2, 1): 1, (0, 0, 3): 1}])):
        cs = comps(l)
        G = np.array([[sphere_monomial(a + d, b + e, c + f) for (d, e, f) in cs] for (a, b, c) in cs])
        for vec in vecs:
            v = np.array([float(vec.get(c, 0)) for c in cs])
            assert np.abs(O.sph_matrix(l) @ G @ v).max() < 1e-13


def test_matrix_level_transform_pair_is_adjoint_and_block_diagonal():
    """sph_from_cart (operators, S X S^T) and cart_from_sph (densities, S^T D S): tr(D^T X) is the same in both
    bases; a one-centre normalised shell's Cartesian overlap maps to the unit matrix; shells do not mix."""
    from paper_2607_05622_b200.inputs import custom_basis
    xyz = np.array([[0.0, 0.0, 0.0], [1.0, 0.5, -0.3]])
    b = custom_basis(xyz, [[(2, [0.8], [1.0]), (0, [0.5], [1.0]), (3, [0.6], [1.0])], [(1, [0.9], [1.0]), (3, [1.1], [1.0])]])
    S = O.sph_block_matrix(b)
    assert S.shape == (5 + 1 + 7 + 3 + 7, 6 + 1 + 10 + 3 + 10)
    rng = np.random.default_rng(8)
    X = rng.standard_normal((2, S.shape[1], S.shape[1]))
    D = rng.standard_normal((2, S.shape[0], S.shape[0]))
    Xs, Dc = O.sph_from_cart(b, X), O.cart_from_sph(b, D)
    for k in range(2):
        assert np.sum(D[k] * Xs[k]) == pytest.approx(np.sum(Dc[k] * X[k]), rel=1e-13)
    # one shell, overlap of its normalised Cartesian components: (a+a'-1)!!(b+b'-1)!!(c+c'-1)!!/(2l-1)!!
    for l in (2, 3):
        cs = comps(l)
        ov = np.array([[0.0 if (a + d) % 2 or (bb + e) % 2 or (c + f) % 2 else
                        dfact(a + d - 1) * dfact(bb + e - 1) * dfact(c + f - 1) / dfact(2 * l - 1)
                        for (d, e, f) in cs] for (a, bb, c) in cs])
        one = custom_basis(xyz[:1], [[(l, [0.7], [1.0])]])
        assert np.allclose(O.sph_from_cart(one, ov[None])[0], np.eye(2 * l + 1), rtol=0, atol=1e-13)
    # an operator that lives on one shell pair stays on that shell pair
    X1 = np.zeros((1, S.shape[1], S.shape[1]))
    X1[0, 0:6, 7:17] = rng.standard_normal((6, 10))               # (d shell, first f shell) block
    Y = O.sph_from_cart(b, X1)[0]
    mask = np.zeros_like(Y, dtype=bool)
    mask[0:5, 6:13] = True
    assert np.abs(Y[~mask]).max() == 0.0 and np.abs(Y[mask]).max() > 0.1

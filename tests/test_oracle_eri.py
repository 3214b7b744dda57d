"""Pins for the oracle's ERIs.  CPU only.

The references here are NOT the oracle's formulas retyped: they are the closed-form (ss|ss) integral
differentiated with respect to the centres in 60-digit arithmetic (x^n e^{-a x^2} = polynomial in d/dA of
e^{-a(x-A)^2}), plus invariants of the independently computed full tensor.
"""
import itertools
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O
from paper_2607_05622_b200.inputs import custom_basis, prim_norm

CART = {0: [(0, 0, 0)], 1: [(1, 0, 0), (0, 1, 0), (0, 0, 1)],
        2: [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)],
        3: [(3, 0, 0), (2, 1, 0), (2, 0, 1), (1, 2, 0), (1, 1, 1), (1, 0, 2), (0, 3, 0), (0, 2, 1), (0, 1, 2), (0, 0, 3)]}


def ssss_closed(a, b, c, d, A, B, C, D):
    """(ss|ss) of four UNNORMALISED primitive s Gaussians; mpmath numbers; textbook closed form."""
    p, q = a + b, c + d
    P = [(a * A[i] + b * B[i]) / p for i in range(3)]
    Q = [(c * C[i] + d * D[i]) / q for i in range(3)]
    AB2 = sum((A[i] - B[i]) ** 2 for i in range(3))
    CD2 = sum((C[i] - D[i]) ** 2 for i in range(3))
    PQ2 = sum((P[i] - Q[i]) ** 2 for i in range(3))
    rho = p * q / (p + q)
    T = rho * PQ2
    F0 = mp.mpf(1) if T == 0 else mp.sqrt(mp.pi / T) * mp.erf(mp.sqrt(T)) / 2
    if T != 0 and T < mp.mpf(10) ** (-30):
        F0 = 1 - T / 3
    return 2 * mp.pi ** mp.mpf(2.5) / (p * q * mp.sqrt(p + q)) * mp.e ** (-a * b / p * AB2) * mp.e ** (-c * d / q * CD2) * F0


def _dir_terms(n, a):
    # x^n e^{-a x^2} as sum coef * d^k/dA^k e^{-a (x-A)^2}
    if n == 0:
        return [(mp.mpf(1), 0)]
    if n == 1:
        return [(1 / (2 * a), 1)]
    if n == 2:
        return [(1 / (4 * a * a), 2), (1 / (2 * a), 0)]
    if n == 3:      # d^3 = (8 a^3 x^3 - 12 a^2 x) e  and  x e = d / (2a)
        return [(1 / (8 * a ** 3), 3), (3 / (4 * a * a), 1)]
    raise ValueError


def _fd_partial(f, x0, orders, h):
    """Tensor-product central differences (2-point for d/dx, 3-point for d2/dx2) in high precision."""
    stencils = []
    for n in orders:
        if n == 0:
            stencils.append([(0, mp.mpf(1))])
        elif n == 1:
            stencils.append([(1, 1 / (2 * h)), (-1, -1 / (2 * h))])
        elif n == 2:
            stencils.append([(1, 1 / h ** 2), (0, -2 / h ** 2), (-1, 1 / h ** 2)])
        elif n == 3:
            stencils.append([(2, 1 / (2 * h ** 3)), (1, -1 / h ** 3), (-1, 1 / h ** 3), (-2, -1 / (2 * h ** 3))])
        else:
            raise ValueError
    tot = mp.mpf(0)
    for combo in itertools.product(*stencils):
        w = mp.mpf(1)
        x = list(x0)
        for i, (sh, cf) in enumerate(combo):
            w *= cf
            if sh:
                x[i] = x[i] + sh * h
        tot += w * f(*x)
    return tot


def cart_eri_by_differentiation(expo, cents, comps):
    """Unnormalised primitive Cartesian ERI via centre-derivatives of the closed-form (ss|ss).

    h = 1e-12: truncation error O(h^2) ~ 1e-24 relative; the cancellation is 12 digits per derivative order, so the
    working precision is 54 digits above that (150 digits up to (dd|dd), 198 for (ff|ff))."""
    order = sum(sum(c) for c in comps)
    mp.mp.dps = max(150, 54 + 12 * order)
    h = mp.mpf(10) ** (-12)
    expo = [mp.mpf(e) for e in expo]
    x0 = [mp.mpf(float(v)) for cen in cents for v in cen]

    def f(*x):
        A, B, C, D = x[0:3], x[3:6], x[6:9], x[9:12]
        return ssss_closed(expo[0], expo[1], expo[2], expo[3], A, B, C, D)

    per_coord = []
    for ci in range(4):
        for di in range(3):
            per_coord.append(_dir_terms(comps[ci][di], expo[ci]))
    total = mp.mpf(0)
    for combo in itertools.product(*per_coord):
        coef = mp.mpf(1)
        orders = []
        for cf, k in combo:
            coef *= cf
            orders.append(k)
        total += coef * _fd_partial(f, x0, orders, h)
    return total


def one_prim_basis(ls, expo, cents):
    return custom_basis(cents, [[(l, [e], [1.0])] for l, e in zip(ls, expo)])


def test_ssss_same_centre_closed_form():
    # four identical normalised s on one centre: 2 sqrt(a/pi)
    for a in (0.3, 1.0, 7.5):
        b = custom_basis([[0.1, 0.2, 0.3]], [[(0, [a], [1.0])]])
        v = O.eri_shell(b, 0, 0, 0, 0)[0, 0, 0, 0]
        assert v == pytest.approx(2 * math.sqrt(a / math.pi), rel=1e-14)
    assert O.eri_shell(custom_basis([[0, 0, 0]], [[(0, [1.0], [1.0])]]), 0, 0, 0, 0)[0, 0, 0, 0] == \
        pytest.approx(1.1283791670955126, rel=1e-15)


@pytest.mark.parametrize("R", [0.5, 2.0, 9.0, 40.0])
def test_two_charge_clouds_erf_over_R(R):
    # normalised s^2 clouds: exponent a at A twice, c at C twice -> erf(sqrt(rho) R)/R, rho = 4ac/(2a+2c)
    a, c = 0.8, 1.7
    b = custom_basis([[0, 0, 0], [0, 0, R]], [[(0, [a], [1.0])], [(0, [c], [1.0])]])
    v = O.eri_shell(b, 0, 0, 1, 1)[0, 0, 0, 0]
    rho = 4 * a * c / (2 * a + 2 * c)
    assert v == pytest.approx(math.erf(math.sqrt(rho) * R) / R, rel=2e-14)
    if R >= 9.0:
        assert v == pytest.approx(1.0 / R, rel=1e-12)


def test_ssss_general_closed_form_contracted():
    rng = np.random.default_rng(7)
    cents = rng.uniform(-1.5, 1.5, size=(4, 3))
    ex = [[0.9, 0.3], [1.4, 0.5], [0.6, 0.2], [2.2, 0.7]]
    cc = [[0.6, 0.4]] * 4
    b = custom_basis(cents, [[(0, ex[i], cc[i])] for i in range(4)])
    v = O.eri_shell(b, 0, 1, 2, 3)[0, 0, 0, 0]
    mp.mp.dps = 40
    ref = mp.mpf(0)
    for ia, ib, ic, id_ in itertools.product(range(2), repeat=4):
        e = [ex[0][ia], ex[1][ib], ex[2][ic], ex[3][id_]]
        co = 1.0
        for k, (s, i) in enumerate(zip(range(4), (ia, ib, ic, id_))):
            co *= cc[s][i] * prim_norm(ex[s][i], 0)
        ref += co * ssss_closed(*[mp.mpf(x) for x in e], *[[mp.mpf(float(t)) for t in cen] for cen in cents])
    assert v == pytest.approx(float(ref), rel=1e-13)


CLASSES = [(1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 1, 0, 0), (1, 0, 1, 0), (1, 1, 1, 1),
           (2, 0, 0, 0), (0, 2, 0, 0), (0, 0, 2, 0), (0, 0, 0, 2), (2, 1, 0, 0), (2, 0, 1, 0), (2, 2, 0, 0),
           (2, 0, 2, 0), (2, 1, 2, 1), (1, 2, 1, 0), (2, 2, 1, 1), (2, 2, 2, 1), (2, 2, 2, 2)]


# classes with f shells: f in every position, next to every other l, up to (ff|ff)
CLASSES_F = [(3, 0, 0, 0), (0, 3, 0, 0), (0, 0, 3, 0), (0, 0, 0, 3), (3, 1, 0, 0), (1, 3, 2, 0), (3, 0, 3, 0),
             (3, 3, 0, 0), (3, 2, 3, 1), (2, 3, 1, 3), (3, 3, 2, 2), (3, 3, 3, 3)]


@pytest.mark.parametrize("ls", CLASSES + CLASSES_F)
def test_cartesian_classes_by_differentiating_closed_form(ls):
    """Every angular class up to (dd|dd), and the f classes up to (ff|ff): sampled components vs derivatives of the
    closed-form (ss|ss)."""
    rng = np.random.default_rng(100 + sum(k * 3 ** i for i, k in enumerate(ls)))
    cents = rng.uniform(-1.2, 1.2, size=(4, 3))
    expo = list(rng.uniform(0.4, 1.6, size=4))
    b = one_prim_basis(ls, expo, cents)
    blk = O.eri_shell(b, 0, 1, 2, 3)
    shape = blk.shape
    idxs = list(itertools.product(*[range(n) for n in shape]))
    pick = [idxs[i] for i in rng.choice(len(idxs), size=min(3, len(idxs)), replace=False)]
    scale = np.abs(blk).max()
    for (ia, ib, ic, id_) in pick:
        comps = [CART[ls[0]][ia], CART[ls[1]][ib], CART[ls[2]][ic], CART[ls[3]][id_]]
        ref = cart_eri_by_differentiation(expo, cents, comps)
        norm = 1.0
        for l, e in zip(ls, expo):
            norm *= prim_norm(e, l)
        assert abs(blk[ia, ib, ic, id_] - float(ref) * norm) <= 1e-11 * scale, (ls, (ia, ib, ic, id_))


def test_full_tensor_8fold_symmetry_cs_psd(tiny):
    eri = O.eri_tensor(tiny.basis)       # every ordered shell quartet computed independently
    n = tiny.nao
    s = np.abs(eri).max()
    for perm in ("nmkr", "mnrk", "krmn", "rknm", "nmrk", "krnm", "rkmn"):
        assert np.abs(eri - np.einsum("mnkr->" + perm, eri)).max() <= 1e-13 * s, perm
    diag = np.einsum("mnmn->mn", eri)
    assert diag.min() >= 0.0
    bound = np.sqrt(diag)[:, :, None, None] * np.sqrt(diag)[None, None, :, :]
    assert (np.abs(eri) <= bound * (1 + 1e-10) + 1e-14).all()
    M = eri.reshape(n * n, n * n)
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).min() >= -1e-11 * s


def test_translation_and_rotation_invariance(spd_basis):
    b = spd_basis
    base = {q: O.eri_shell(b, *q) for q in [(2, 1, 5, 8), (8, 8, 5, 2), (4, 3, 7, 6)]}
    # translation
    bt = custom_basis(b.xyz + np.array([3.3, -1.2, 0.7]),
                      [[(0, [0.9, 0.3], [0.6, 0.4]), (1, [0.7, 0.25], [0.6, 0.4]), (2, [0.8, 0.35], [0.6, 0.4])]] * 3)
    for q, v in base.items():
        assert np.abs(O.eri_shell(bt, *q) - v).max() <= 1e-13 * np.abs(v).max()
    # rotation by 90 degrees about z: (x,y,z) -> (-y,x,z); a function x^i y^j z^k maps to (-1)^? y^i x^j ...
    Rm = np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])
    br = custom_basis(b.xyz @ Rm.T,
                      [[(0, [0.9, 0.3], [0.6, 0.4]), (1, [0.7, 0.25], [0.6, 0.4]), (2, [0.8, 0.35], [0.6, 0.4])]] * 3)

    def comp_map(l):
        # rotated function R chi(r) = chi(R^-1 r): x^i y^j z^k at rotated centre equals, in the rotated frame,
        # x'^? ... : old x = y', old y = -x'  =>  x^i y^j z^k = (y')^i (-x')^j z'^k
        out = []
        for (i, j, k) in CART[l]:
            tgt = CART[l].index((j, i, k))
            out.append((tgt, (-1.0) ** j))
        return out

    for q, v in base.items():
        vr = O.eri_shell(br, *q)
        maps = [comp_map(int(b.l[s])) for s in q]
        w = np.zeros_like(v)
        for ia, ib, ic, id_ in itertools.product(*[range(n) for n in v.shape]):
            (ta, sa), (tb, sb), (tc, sc), (td, sd) = maps[0][ia], maps[1][ib], maps[2][ic], maps[3][id_]
            w[ia, ib, ic, id_] = sa * sb * sc * sd * vr[ta, tb, tc, td]
        assert np.abs(w - v).max() <= 1e-13 * np.abs(v).max()


def test_schwarz_matches_tensor_diagonal(tiny):
    b = tiny.basis
    Q = O.schwarz(b)
    eri = O.eri_tensor(b)
    off = b.ao_off
    for A in range(b.nshell):
        for B in range(b.nshell):
            blk = np.array([[eri[m, n, m, n] for n in range(off[B], off[B + 1])] for m in range(off[A], off[A + 1])])
            assert Q[A, B] == pytest.approx(math.sqrt(np.abs(blk).max()), rel=1e-12)

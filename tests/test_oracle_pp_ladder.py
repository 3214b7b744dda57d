"""Pins for the oracle's particle-particle ladder:
L[p,a,b] = sum_ef (ae|bf) X[p,e,f].  The paper prints no value; pins are a closed form on a one-centre s-only toy,
the bra-ket symmetry of the integrals, the AO-direct route of the paper (a K-only build on the non-symmetric density
C_v X C_v^T, back-transformed) and explicit loops."""
import math

import numpy as np

from oracle import oracle as O
from paper_2607_05622_b200.inputs import custom_basis, prim_norm


def test_one_centre_single_exponent_closed_form():
    """Two identical normalised s functions (exponent a) on one centre: every AO integral is 2 sqrt(a/pi)
    (SURVEY P-E), so (ae|bf) = g * s_a s_e s_b s_f with s = column sums of C_v and L[p,a,b] = g s_a s_b (s^T X_p s)."""
    a = 0.8
    b = custom_basis(np.zeros((1, 3)), [[(0, [a], [1.0]), (0, [a], [1.0])]])
    eri = O.eri_tensor(b)
    g = 2.0 * math.sqrt(a / math.pi)
    assert np.allclose(eri, g, rtol=1e-13, atol=0)
    rng = np.random.default_rng(3)
    Cv = rng.standard_normal((2, 2))
    X = rng.standard_normal((3, 2, 2))
    s = Cv.sum(0)
    ref = g * np.einsum("a,b,p->pab", s, s, np.einsum("e,pef,f->p", s, X, s))
    assert np.allclose(O.pp_ladder(eri, Cv, X), ref, rtol=1e-12, atol=1e-14)


def test_loops_symmetry_and_ao_direct_route(tiny):
    """(i) explicit loops on a cut-down basis; (ii) (ae|bf) = (bf|ae): L[X^T] = L[X]^T and a non-symmetric X gives a
    non-symmetric L; (iii) the AO-direct route the paper names (L432-434: the ladder goes through the batched
    non-symmetric exchange path): L_p = C_v^T K[C_v X_p C_v^T] C_v with K from Eq. 17."""
    from paper_2607_05622_b200.inputs import Basis
    b = tiny.basis
    eri = O.eri_tensor(b)
    rng = np.random.default_rng(5)
    nv = 4
    Cv = rng.standard_normal((b.nao, nv)) / math.sqrt(b.nao)
    X = rng.standard_normal((3, nv, nv))
    L = O.pp_ladder(eri, Cv, X)
    # (i) loops on the first 5 AOs only (8^... kept tiny): restrict the tensor and the coefficients
    m = 5
    Ls = O.pp_ladder(eri[:m, :m, :m, :m], Cv[:m, :3], X[:2, :3, :3])
    assert np.allclose(O.pp_ladder_loops(eri[:m, :m, :m, :m], Cv[:m, :3], X[:2, :3, :3]), Ls, rtol=1e-12, atol=1e-15)
    # (ii)
    Lt = O.pp_ladder(eri, Cv, X.transpose(0, 2, 1))
    assert np.allclose(Lt, L.transpose(0, 2, 1), rtol=1e-12, atol=1e-15)
    assert np.abs(L - L.transpose(0, 2, 1)).max() > 1e-3 * np.abs(L).max()
    # (iii)
    D = np.einsum("me,pef,rf->pmr", Cv, X, Cv)
    _, K = O.jk_definition(eri, D)
    Lk = np.einsum("ma,pmn,nb->pab", Cv, K, Cv)
    assert np.allclose(Lk, L, rtol=1e-11, atol=1e-14)
    # and through the folded, screened loop O6 (tau = 0: nothing dropped)
    _, K6, _ = O.jk_folded(b, D, 0.0)
    assert np.allclose(np.einsum("ma,pmn,nb->pab", Cv, K6, Cv), L, rtol=1e-10, atol=1e-13)

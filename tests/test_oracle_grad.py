"""Pins for the oracle's derivative builds (Eq. 18, L382-386 Eqs. 30-31):
    J^x(A,B) = sum (mn|kr)^x A_mn B_kr ,   K^x(A,B) = sum (mk|nr)^x A_mn B_kr .
The paper prints no value.  Pins: a closed form (two s charge clouds: d/dR of erf(sqrt(rho) R)/R), central finite
differences of tr(A^T J[B]) and tr(A^T K[B]) built from the value oracle O7 with displaced atoms, the translational sum
rule (Eq. 31), and the permutational identities of a TOTAL nuclear derivative (reading A2):
J^x(A,B) = J^x(B,A), K^x(A,B) = K^x(B,A) = K^x(A^T,B^T)."""
import copy
import math

import numpy as np

from oracle import oracle as O
from paper_2607_05622_b200.inputs import custom_basis, prim_norm, random_densities


def scalars(b, A, B):
    eri = O.eri_tensor(b)
    J, K = O.jk_definition(eri, B)
    return np.einsum("pmn,pmn->p", A, J), np.einsum("pmn,pmn->p", A, K)


def fd_gradient(b, A, B, h=2e-3):
    """4th-order central differences of the value oracle in every nuclear coordinate."""
    nat = b.xyz.shape[0]
    gJ = np.zeros((A.shape[0], nat, 3))
    gK = np.zeros_like(gJ)
    for at in range(nat):
        for x in range(3):
            vals = {}
            for k in (-2, -1, 1, 2):
                bb = copy.deepcopy(b)
                bb.xyz = np.array(b.xyz, dtype=float)
                bb.xyz[at, x] += k * h
                vals[k] = scalars(bb, A, B)
            for q, g in ((0, gJ), (1, gK)):
                g[:, at, x] = (8 * (vals[1][q] - vals[-1][q]) - (vals[2][q] - vals[-2][q])) / (12 * h)
    return gJ, gK


def test_two_s_clouds_closed_form():
    """(aa|cc) for normalised s functions a at A, c at C is erf(sqrt(rho) R)/R, rho = 4ac/(2a+2c) (SURVEY P-E).  With
    A = e_1 e_1^T, B = e_2 e_2^T:  J^x = d/dX of it: on atom C along the axis, f'(R); on atom A, -f'(R)."""
    a, c, R = 0.7, 1.3, 1.9
    b = custom_basis(np.array([[0.0, 0.0, 0.0], [0.0, 0.0, R]]), [[(0, [a], [1.0])], [(0, [c], [1.0])]])
    A = np.zeros((1, 2, 2)); A[0, 0, 0] = 1.0
    B = np.zeros((1, 2, 2)); B[0, 1, 1] = 1.0
    gJ, gK = O.jk_grad(b, A, B)
    rho = 4 * a * c / (2 * a + 2 * c)
    fp = 2 * math.sqrt(rho / math.pi) * math.exp(-rho * R * R) / R - math.erf(math.sqrt(rho) * R) / R ** 2
    assert abs(gJ[0, 1, 2] - fp) < 1e-13 and abs(gJ[0, 0, 2] + fp) < 1e-13
    assert np.abs(gJ[0, :, :2]).max() < 1e-14
    # K^x(A,B) = (12|12)^x A_11 B_22: the overlap-type integral, also odd under exchange of the two atoms
    assert abs(gK[0, 0, 2] + gK[0, 1, 2]) < 1e-14 and abs(gK[0, 1, 2]) > 1e-3


def test_finite_differences_sum_rule_and_permutations():
    """s, p, d shells, contracted, three atoms (one shell pair shares a centre): analytic oracle vs 4th-order finite
    differences of the value oracle; sum over atoms = 0 (Eq. 31); permutational identities."""
    xyz = np.array([[0.0, 0.1, -0.2], [1.7, -0.4, 0.5], [-0.9, 1.5, 0.7]])
    sh0 = [(0, [0.9, 0.3], [0.6, 0.4]), (1, [0.7, 0.25], [0.6, 0.4])]
    sh1 = [(2, [0.8, 0.35], [0.6, 0.4])]
    sh2 = [(1, [1.1], [1.0]), (0, [0.5], [1.0])]
    b = custom_basis(xyz, [sh0, sh1, sh2])
    n = b.nao
    A = random_densities(n, 2, seed=3)
    B = random_densities(n, 2, seed=4)
    gJ, gK = O.jk_grad(b, A, B)
    fJ, fK = fd_gradient(b, A, B)
    assert np.abs(gJ - fJ).max() < 2e-8 * np.abs(gJ).max()
    assert np.abs(gK - fK).max() < 2e-8 * np.abs(gK).max()
    assert np.abs(gJ.sum(axis=1)).max() < 1e-12 * np.abs(gJ).max()          # translational invariance, Eq. (31)
    assert np.abs(gK.sum(axis=1)).max() < 1e-12 * np.abs(gK).max()
    hJ, hK = O.jk_grad(b, B, A)
    assert np.abs(hJ - gJ).max() < 1e-12 * np.abs(gJ).max()                  # (mn|kr)^x = (kr|mn)^x
    assert np.abs(hK - gK).max() < 1e-12 * np.abs(gK).max()
    tJ, tK = O.jk_grad(b, A.transpose(0, 2, 1), B.transpose(0, 2, 1))
    assert np.abs(tK - gK).max() < 1e-12 * np.abs(gK).max()
    assert np.abs(tJ - gJ).max() < 1e-12 * np.abs(gJ).max()                  # J^x only sees the symmetric parts
    # but K^x(A, B) != K^x(A^T, B) for non-symmetric densities: the non-symmetry the paper's kernel keeps (L308)
    uJ, uK = O.jk_grad(b, A.transpose(0, 2, 1), B)
    assert np.abs(uK - gK).max() > 1e-3 * np.abs(gK).max()

"""Pins for oracle step O10, the pseudo-density transform (Eqs. 13-15):

    D^{alpha,d}_{mu nu} = sum_{ia} C_{mu i} e^{+eps_i tau_alpha} T^d_{ia} e^{-eps_a tau_alpha} C_{nu a}

The paper prints no worked value, so `oracle.pseudo_densities_loops` is pinned by what the formula fixes:
special cases that reduce to a plain matrix product or an outer product, the sign of each exponent separately,
and the denominator resolution of Eq. 11 with the golden minimax grid.  A dropped factor, a swapped sign in either
exponent, a transposed operand or a mixed-up (tau, d) layout fails at least one of them."""
from pathlib import Path

import numpy as np
import pytest

from oracle import oracle as O

GOLD = Path(__file__).resolve().parent / "golden" / "laplace_minimax.txt"


def read_golden():
    """tests/golden/laplace_minimax.txt (written by make_laplace_golden.py from oracle/ only): k -> (tau, w, delta)."""
    recs = {}
    lines = [l for l in GOLD.read_text().splitlines() if l and not l.startswith("#")]
    i = 0
    while i < len(lines):
        p = lines[i].split()
        k, delta = int(p[1]), float(p[3])
        tw = np.array([[float(x) for x in lines[i + 1 + a].split()] for a in range(k)])
        recs[k] = (tw[:, 0], tw[:, 1], delta, None)
        i += k + 2
    return recs


RNG = np.random.default_rng(20260705)
N, NOCC, NVIR, NT = 9, 3, 5, 2
C_OCC = RNG.standard_normal((N, NOCC))
C_VIR = RNG.standard_normal((N, NVIR))
EPS_O = np.sort(RNG.uniform(-1.5, -0.3, NOCC))
EPS_V = np.sort(RNG.uniform(0.1, 3.0, NVIR))
T = RNG.standard_normal((NT, NOCC, NVIR))


def test_tau_zero_is_plain_product():
    """tau = 0: every exponential is 1, D = C_o T C_v^T (library matmul; orientation: rows from C_o, columns from C_v)."""
    D = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, T, np.array([0.0]))
    assert D.shape == (1, NT, N, N)
    for d in range(NT):
        assert np.allclose(D[0, d], C_OCC @ T[d] @ C_VIR.T, rtol=0, atol=1e-13)
    assert np.abs(D[0, 0] - D[0, 0].T).max() > 1e-2          # a general, non-symmetric matrix


def test_ones_amplitudes_give_rank_one_eq14():
    """Reading A1: Eq. 14 is the R = 1 case: D = (sum_i U~_i)(sum_a V~_a)^T, rank one."""
    tau = np.array([0.7])
    D = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, np.ones((1, NOCC, NVIR)), tau)[0, 0]
    u = (C_OCC * np.exp(EPS_O * tau[0])[None, :]).sum(1)
    v = (C_VIR * np.exp(-EPS_V * tau[0])[None, :]).sum(1)
    assert np.allclose(D, np.outer(u, v), rtol=0, atol=1e-13)
    s = np.linalg.svd(D, compute_uv=False)
    assert s[1] < 1e-13 * s[0]


@pytest.mark.parametrize("i,a", [(0, 0), (2, 4), (1, 3)])
def test_unit_amplitude_isolates_one_pair(i, a):
    """T = e_i e_a^T: D = e^{(eps_i - eps_a) tau} C_{:,i} C_{:,a}^T.  Pins each exponent's sign and which index it
    belongs to: eps_i < 0 < eps_a here, so the factor is < 1 and decays with tau; a flipped sign would grow."""
    Tu = np.zeros((1, NOCC, NVIR))
    Tu[0, i, a] = 1.0
    tau = np.array([0.0, 0.5, 2.0])
    D = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, Tu, tau)
    base = np.outer(C_OCC[:, i], C_VIR[:, a])
    for k, t in enumerate(tau):
        f = np.exp((EPS_O[i] - EPS_V[a]) * t)
        assert np.allclose(D[k, 0], f * base, rtol=0, atol=1e-14)
    r = np.abs(D[:, 0]).max(axis=(1, 2))
    assert r[0] > r[1] > r[2]
    # separately: only the occupied factor (eps_a = 0) and only the virtual factor (eps_i = 0)
    Do = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, np.zeros(NVIR), Tu, tau[1:2])[0, 0]
    Dv = O.pseudo_densities_loops(C_OCC, C_VIR, np.zeros(NOCC), EPS_V, Tu, tau[1:2])[0, 0]
    assert np.allclose(Do, np.exp(EPS_O[i] * tau[1]) * base, rtol=0, atol=1e-14)
    assert np.allclose(Dv, np.exp(-EPS_V[a] * tau[1]) * base, rtol=0, atol=1e-14)


def test_layout_tau_major_then_amplitude_set():
    """Output layout [ntau][nT][N][N] and linearity in T."""
    tau = np.array([0.3, 1.1, 2.4])
    D = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, T, tau)
    assert D.shape == (3, NT, N, N)
    for k in range(3):
        for d in range(NT):
            one = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, T[d:d + 1], tau[k:k + 1])[0, 0]
            assert np.array_equal(one, D[k, d])
    c = np.array([0.7, -1.3])
    Dc = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, np.tensordot(c, T, axes=1)[None], tau)
    assert np.allclose(Dc[:, 0], np.tensordot(c, D, axes=([0], [1])), rtol=0, atol=1e-13)


@pytest.mark.parametrize("k", [8, 10, 12])
def test_denominator_resolution_with_golden_grid(k):
    """The purpose of the transform (Eq. 11, L145 Eq. 15): sum_alpha w_alpha D^alpha =
    C_o (T o 1/(eps_a - eps_i)) C_v^T to within delta_quad * sum |C_o| |T| |C_v^T| (element-wise bound), with the
    golden minimax grid on [0.4, 4.5] -- and the error is really of that size, not zero (the grid is doing the work)."""
    tau, w, delta, _ = read_golden()[k]
    denom = EPS_V[None, :] - EPS_O[:, None]
    assert denom.min() >= 0.4 and denom.max() <= 4.5
    D = O.pseudo_densities_loops(C_OCC, C_VIR, EPS_O, EPS_V, T, tau)
    lhs = np.tensordot(w, D, axes=1)
    rhs = np.einsum("mi,dia,na->dmn", C_OCC, T / denom[None], C_VIR)
    bound = delta * np.einsum("mi,dia,na->dmn", np.abs(C_OCC), np.abs(T), np.abs(C_VIR))
    assert np.all(np.abs(lhs - rhs) <= 1.0001 * bound + 1e-14)
    # a wrong sign in one exponent makes the sum resolve 1/(eps_a + eps_i) instead: far outside the bound
    Dbad = O.pseudo_densities_loops(C_OCC, C_VIR, -EPS_O, EPS_V, T, tau)
    assert np.abs(np.tensordot(w, Dbad, axes=1) - rhs).max() > 1e3 * bound.max()

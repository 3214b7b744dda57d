"""Pins for the N1 oracle functions (Eq. 19, L180 Eq. 21)."""
import numpy as np

from oracle import oracle as O
from test_oracle_laplace import read_golden, XMIN, XMAX


def test_laplace_fock_einsum_vs_loops_and_special_cases():
    rng = np.random.default_rng(1)
    n, nmo, nD = 7, 5, 2
    J = rng.standard_normal((nD, n, n))
    K = rng.standard_normal((nD, n, n))
    C = rng.standard_normal((n, nmo))
    F = O.laplace_fock(J, K, C)
    assert np.allclose(F, O.laplace_fock_loops(J, K, C), rtol=1e-13, atol=1e-13)
    # C = identity: the AO matrix itself; K = 2J: zero; linear in (J, K)
    assert np.allclose(O.laplace_fock(J, K, np.eye(n)), 2 * J - K)
    assert np.abs(O.laplace_fock(J, 2 * J, C)).max() < 1e-12
    # a non-symmetric K gives a non-symmetric F~ whose transpose is the transform of K^T (J symmetric here)
    Js = J + J.transpose(0, 2, 1)
    assert np.allclose(O.laplace_fock(Js, K, C).transpose(0, 2, 1), O.laplace_fock(Js, K.transpose(0, 2, 1), C))


def test_omega_reweighted_grid_resolves_shifted_denominator():
    """Eq. (21): sum_a w_a e^{omega tau_a} e^{-D tau_a} = 1/(D - omega) to the quadrature error, for D - omega inside the
    fitted interval."""
    tau, w, delta, _ = read_golden()[10]
    omega = 0.25
    D = np.linspace(XMIN + omega, XMAX + omega, 500)          # D - omega in [xmin, xmax]
    X = np.exp(-D[None, :] * tau[:, None])[:, None, :]         # [ntau, 1, nelem]
    y = O.laplace_accumulate(tau, w, omega, X)[0]
    assert np.abs(y - 1.0 / (D - omega)).max() <= delta * (1 + 1e-3)
    # omega = 0: plain weights
    D0 = np.linspace(XMIN, XMAX, 500)
    y0 = O.laplace_accumulate(tau, w, 0.0, np.exp(-D0[None, :] * tau[:, None])[:, None, :])[0]
    assert np.abs(y0 - 1.0 / D0).max() <= delta * (1 + 1e-3)

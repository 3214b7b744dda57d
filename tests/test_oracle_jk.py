"""Pins for the oracle's J/K digestion.  CPU only."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2607_05622_b200.inputs import custom_basis, random_densities


def relerr(x, ref):
    return np.abs(x - ref).max() / np.abs(ref).max()


@pytest.fixture(scope="module")
def tiny_eri(tiny):
    return O.eri_tensor(tiny.basis)


def test_folded_vs_definition_tiny(tiny, tiny_eri):
    D = random_densities(tiny.nao, 3, seed=11)
    Jd, Kd = O.jk_definition(tiny_eri, D)
    Jf, Kf, kept = O.jk_folded(tiny.basis, D, tau=0.0)
    ns = tiny.basis.nshell
    npair = ns * (ns + 1) // 2
    assert kept == npair * (npair + 1) // 2
    assert relerr(Jf, Jd) < 1e-13 and relerr(Kf, Kd) < 1e-13


def test_folded_vs_definition_with_d_shells(spd_basis):
    eri = O.eri_tensor(spd_basis)
    D = random_densities(spd_basis.nao, 2, seed=5)
    Jd, Kd = O.jk_definition(eri, D)
    Jf, Kf, _ = O.jk_folded(spd_basis, D, tau=0.0)
    assert relerr(Jf, Jd) < 1e-13 and relerr(Kf, Kd) < 1e-13


def test_blocks_vs_definition(spd_basis):
    eri = O.eri_tensor(spd_basis)
    D = random_densities(spd_basis.nao, 2, seed=6)
    Jd, Kd = O.jk_definition(eri, D)
    pairs = [(0, 0), (8, 2), (2, 8), (4, 5), (7, 1)]
    Js, Ks = O.jk_blocks(spd_basis, D, 0.0, pairs)
    off = spd_basis.ao_off
    for (x, y), jb, kb in zip(pairs, Js, Ks):
        sl = (slice(None), slice(off[x], off[x + 1]), slice(off[y], off[y + 1]))
        assert np.abs(jb - Jd[sl]).max() < 1e-13 * np.abs(Jd).max()
        assert np.abs(kb - Kd[sl]).max() < 1e-13 * np.abs(Kd).max()


def test_screening_changes_little_and_blocks_follow_same_rule(small):
    # tau = 1e-12 (reading A9) vs unscreened on a bra-pair sample; blocks use the identical keep rule
    b = small.basis
    D = random_densities(b.nao, 2, seed=3, scale=1e-2)
    Q = O.schwarz(b)
    pr = (2000, 2040)
    J0, K0, k0 = O.jk_folded(b, D, 0.0, pair_range=pr, Q=Q)
    J1, K1, k1 = O.jk_folded(b, D, 1e-12, pair_range=pr, Q=Q)
    assert k1 < k0
    assert np.abs(J1 - J0).max() <= 1e-11 * np.abs(J0).max()
    assert np.abs(K1 - K0).max() <= 1e-11 * np.abs(K0).max()


def test_symmetry_relations(tiny):
    b = tiny.basis
    rng = np.random.default_rng(2)
    A = rng.standard_normal((1, b.nao, b.nao))
    B = rng.standard_normal((1, b.nao, b.nao))
    At = np.transpose(A, (0, 2, 1)).copy()
    J, K, _ = O.jk_folded(b, np.concatenate([A, At, B, 0.5 * (A + At), 0.5 * (A - At), 2.0 * A - 3.0 * B]), 0.0)
    JA, JAt, JB, Js, Ja, Jl = J
    KA, KAt, KB, Ks, Ka, Kl = K
    s = np.abs(KA).max()
    assert np.abs(JA - JA.T).max() < 1e-13 * s          # J[D] symmetric
    assert np.abs(JAt - JA).max() < 1e-13 * s           # J[D^T] = J[D] = J[D]^T
    assert np.abs(KAt - KA.T).max() < 1e-13 * s         # K[D^T] = K[D]^T
    assert np.abs(Ks - 0.5 * (KA + KA.T)).max() < 1e-13 * s
    assert np.abs(Ka - 0.5 * (KA - KA.T)).max() < 1e-13 * s
    assert np.abs(Ka).max() > 1e-3 * s                  # the part a symmetric-only kernel would drop (L308)
    assert np.abs(Ja).max() < 1e-13 * s                 # J annihilates the antisymmetric part
    assert np.abs(Ks - Ks.T).max() < 1e-13 * s          # D = D^T => K symmetric
    assert np.abs(Jl - (2 * JA - 3 * JB)).max() < 1e-12 * s and np.abs(Kl - (2 * KA - 3 * KB)).max() < 1e-12 * s
    # adjointness: tr(A^T J[B]) = tr(B^T J[A]), same for K
    assert np.sum(A[0] * JB) == pytest.approx(np.sum(B[0] * JA), rel=1e-11)
    assert np.sum(A[0] * KB) == pytest.approx(np.sum(B[0] * KA), rel=1e-11)
    assert np.sum(A[0] * JA) >= 0.0                     # Coulomb self-repulsion of the charge distribution
    P = A[0] @ A[0].T                                   # symmetric PSD density
    _, KP, _ = O.jk_folded(b, P[None], 0.0)
    assert np.sum(P * KP[0]) >= 0.0


def test_one_centre_s_only_closed_form():
    # all shells on one centre with one exponent a: every (mn|kr) = 2 sqrt(a/pi) (normalised s)
    a = 0.7
    n = 4
    b = custom_basis([[0.3, -0.2, 0.1]], [[(0, [a], [1.0])] * n])
    D = random_densities(n, 2, seed=9)
    J, K, _ = O.jk_folded(b, D, 0.0)
    g = 2 * math.sqrt(a / math.pi)
    for d in range(2):
        assert np.allclose(J[d], g * D[d].sum(), rtol=1e-13)
        assert np.allclose(K[d], g * D[d].sum(), rtol=1e-13)

"""Pins for the Laplace quadrature (Eq. 11).  The paper prints no grid, so the
oracle's grids (tests/golden/laplace_minimax.txt, written by make_laplace_golden.py from oracle/ only) are pinned
by what the mathematics fixes: the equi-oscillation certificate of a best uniform approximation, positivity,
the scaling law, monotone improvement with k.  The library's own solver (csrc/ltjk_laplace.cpp, quad-precision,
a host-only C-ABI entry that needs no GPU) must reproduce them."""
from pathlib import Path

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O

GOLD = Path(__file__).resolve().parent / "golden" / "laplace_minimax.txt"
XMIN, XMAX = 0.4, 4.5


def read_golden():
    recs = {}
    lines = [l for l in GOLD.read_text().splitlines() if l and not l.startswith("#")]
    i = 0
    while i < len(lines):
        p = lines[i].split()
        k, delta = int(p[1]), float(p[3])
        tw = np.array([[float(x) for x in lines[i + 1 + a].split()] for a in range(k)])
        xs = np.array([float(x) for x in lines[i + 1 + k].split()])
        recs[k] = (tw[:, 0], tw[:, 1], delta, xs)
        i += k + 2
    return recs


def err_mp(tau, w, x):
    mp.mp.dps = 40
    return mp.mpf(1) / x - sum(mp.mpf(float(ww)) * mp.e ** (-x * mp.mpf(float(t))) for t, ww in zip(tau, w))


def extrema_mp(tau, w, lo, hi, n=4000):
    """local extrema of the error curve incl. both endpoints, values in 40-digit arithmetic"""
    xs = [mp.mpf(lo) * (mp.mpf(hi) / mp.mpf(lo)) ** (mp.mpf(i) / (n - 1)) for i in range(n)]
    e = [err_mp(tau, w, x) for x in xs]
    idx = [0] + [i for i in range(1, n - 1) if (e[i] - e[i - 1]) * (e[i + 1] - e[i]) < 0] + [n - 1]
    return [xs[i] for i in idx], [e[i] for i in idx]


def check_certificate(tau, w, delta, k, lo=XMIN, hi=XMAX, tol=0.01):
    assert np.all(tau > 0) and np.all(w > 0)
    xe, ee = extrema_mp(tau, w, lo, hi)
    assert len(xe) == 2 * k + 1, len(xe)                      # 2k+1 alternation points, both endpoints included
    assert all(ee[j] * ee[j + 1] < 0 for j in range(2 * k))   # alternating signs
    mags = np.array([float(abs(v)) for v in ee])
    assert mags.max() / mags.min() < 1 + tol                  # equal magnitude: the certificate of minimaxity
    assert abs(mags.max() / delta - 1) < tol                  # and it is the stated error


@pytest.mark.parametrize("k", [8, 10, 12])
def test_golden_grid_equioscillates(k):
    tau, w, delta, xs = read_golden()[k]
    check_certificate(tau, w, delta, k)
    # max error on a 1e5-point log grid (fp64 evaluation) equals the stated error
    x = np.exp(np.linspace(np.log(XMIN), np.log(XMAX), 100001))
    e = O.laplace_error_curve(tau, w, x)
    assert abs(np.abs(e).max() / delta - 1) < 0.02


def test_golden_error_decreases_with_k():
    g = read_golden()
    assert g[8][2] > g[10][2] > g[12][2] > 0
    assert g[8][2] < 8.6e-9          # below the non-converged Lawson bound found in the survey


def test_oracle_solver_live_small_k_and_scaling_law():
    tau, w, delta, xs = O.laplace_minimax(XMIN, XMAX, 4)
    check_certificate(tau, w, delta, 4)
    t1, w1, d1, _ = O.laplace_minimax(1.0, XMAX / XMIN, 4)
    assert np.allclose(tau, t1 / XMIN, rtol=1e-10) and np.allclose(w, w1 / XMIN, rtol=1e-10)
    assert abs(delta - d1 / XMIN) < 1e-10 * delta


def test_denominator_resolution_identity():
    """sum_a w_a exp(-(e_a - e_i) tau_a) reproduces 1/(e_a - e_i) to the stated error on the whole range"""
    tau, w, delta, _ = read_golden()[10]
    rng = np.random.default_rng(3)
    x = rng.uniform(XMIN, XMAX, size=2000)
    approx = (w[None, :] * np.exp(-x[:, None] * tau[None, :])).sum(1)
    assert np.abs(approx - 1 / x).max() <= delta * (1 + 1e-3)


@pytest.fixture(scope="module")
def lib():
    from paper_2607_05622_b200 import build
    build.build()
    from paper_2607_05622_b200 import ltjk
    return ltjk


def lawson_minimax(xmin, xmax, k, iters=400, n=1500):
    """A DIFFERENT algorithm for the same best approximation: Lawson's iteratively reweighted least squares.  On a
    log grid of [1, R] minimise sum_i lam_i r_i(p)^2 over p = (log tau, log w) (scipy Levenberg-Marquardt, a library
    routine as the step), then lam_i <- lam_i |r_i| / sum; the weights concentrate on the extrema and max|r| descends
    to the minimax level from above.  fp64 only, so it is usable for small k (error >> 1e-9)."""
    from scipy.optimize import least_squares
    R = xmax / xmin
    x = np.exp(np.linspace(0.0, np.log(R), n))
    hh = (np.log(R) + 5.5) / k
    s0 = -np.log(R) - 2.5 + hh * (np.arange(k) + 0.5)
    p = np.concatenate([s0, np.log(hh) + s0])
    lam = np.ones(n) / n

    def res(p, sw):
        return sw * (1.0 / x - (np.exp(p[k:])[None, :] * np.exp(-x[:, None] * np.exp(p[:k])[None, :])).sum(1))

    def jac(p, sw):
        t, w = np.exp(p[:k]), np.exp(p[k:])
        ex = np.exp(-x[:, None] * t[None, :])
        return sw[:, None] * np.concatenate([w * t * x[:, None] * ex, -w * ex], axis=1)

    best = (np.inf, p)
    for _ in range(iters):
        p = least_squares(res, p, jac=jac, args=(np.sqrt(lam),), method="lm", xtol=1e-15, ftol=1e-15, gtol=1e-15,
                          max_nfev=2000).x
        r = np.abs(res(p, np.ones(n)))
        if r.max() < best[0]:
            best = (r.max(), p.copy())
        lam = lam * r
        lam /= lam.sum()
    order = np.argsort(best[1][:k])
    return np.exp(best[1][:k])[order] / xmin, np.exp(best[1][k:])[order] / xmin, best[0] / xmin


@pytest.mark.parametrize("k", [2, 4])
def test_oracle_remez_vs_lawson(k):
    """Reading A8: the oracle's Remez solver against a genuinely different algorithm (Lawson reweighting, above).
    The best approximation is unique: Lawson's level approaches the Remez level from above and the grids agree."""
    tau, w, delta, _ = O.laplace_minimax(XMIN, XMAX, k)
    tl, wl, dl = lawson_minimax(XMIN, XMAX, k)
    assert delta <= dl * (1 + 1e-9) and dl / delta - 1 < 2e-3
    assert np.allclose(tl, tau, rtol=2e-2) and np.allclose(wl, w, rtol=2e-2)
    check_certificate(np.asarray(tau), np.asarray(w), delta, k)


@pytest.mark.parametrize("k", [8, 10, 12])
def test_library_solver_matches_oracle_grid(lib, k):
    """Two implementations of the same method family (Remez exchange; C++ quad precision vs Python 80-digit) must
    return the unique best approximation; what pins either is the equi-oscillation certificate, not their agreement."""
    tau, w, delta, _ = read_golden()[k]
    t, ww, err = lib.laplace_quadrature(XMIN, XMAX, k)
    assert abs(err / delta - 1) < 0.01
    assert np.allclose(np.sort(t), np.sort(tau), rtol=1e-6) and np.allclose(np.sort(ww), np.sort(w), rtol=1e-6)
    check_certificate(np.asarray(t), np.asarray(ww), err, k)


def test_library_solver_rejects_bad_arguments(lib):
    import ctypes
    L = lib.load_library()
    t = (ctypes.c_double * 4)()
    for args in ((0.0, 1.0, 4), (2.0, 1.0, 4), (1.0, 2.0, 0), (1.0, 2.0, 1), (1.0, 2.0, 15)):
        rc = L.ltjk_laplace_quadrature(ctypes.c_double(args[0]), ctypes.c_double(args[1]), ctypes.c_int(args[2]), t, t, None)
        assert rc == -1

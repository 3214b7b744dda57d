"""CPU oracle, Python side.  TEST INFRASTRUCTURE ONLY (tests/, __graft_entry__.smoke(), bench.py cpu_baseline).

* thin ctypes wrapper over oracle/ltjk_oracle.c (built on demand with gcc -O2 -fopenmp; no CUDA, no torch);
* O7 contraction  J = einsum('mnkr,kr->mn'), K = einsum('mknr,kr->mn')            PAPER.md:L157 Eq. (17)
* O9 minimax Laplace grid by Remez exchange + Newton in 120-digit arithmetic       PAPER.md:L126 Eq. (11)
* O10 pseudo-density as explicit loops                                            PAPER.md:L136-145 Eqs. (13),(15)

* N1 laplace_fock / laplace_accumulate (Eqs. (19), (21)), N3 pp_ladder
* N4 sph_matrix / sph_from_cart / cart_from_sph: the spherical-harmonic transform at matrix level

Pins (tests/test_oracle_*.py, CPU tier): O9 equi-oscillation certificate, scaling law, Lawson cross-check; O10 tau = 0
product, rank-1 Eq. (14) case, unit amplitudes, layout, denominator resolution with the golden grid; N1 C = I, K = 2J,
rectangular C; N3 one-centre closed form, loops, bra-ket symmetry, AO-direct K route; N4 harmonicity, orthogonality and
norm on the sphere, rotation about z, tabulated low orders, contaminants, adjointness (tests/test_oracle_sph.py).
Nothing is "parity unpinned".

Nothing here imports the CUDA package except the shared, arithmetic-free input generators.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libltjk_oracle.so"
_SRC = _HERE / "ltjk_oracle.c"
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_lp = ctypes.POINTER(ctypes.c_longlong)


def build(force: bool = False) -> Path:
    """Compile the C oracle (building the checker is not using it)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-march=native", "-fopenmp", "-std=c11", "-shared", "-fPIC", "-o", str(_SO),
               str(_SRC), "-lm"]
        subprocess.check_call(cmd)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(str(_SO))
        _lib.orc_jk_folded.restype = ctypes.c_longlong
        _lib.orc_nao.restype = ctypes.c_int
        _lib.orc_max_threads.restype = ctypes.c_int
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _basis_args(b):
    xyz = np.ascontiguousarray(b.xyz, dtype=np.float64)
    atom = np.ascontiguousarray(b.atom, dtype=np.int32)
    l = np.ascontiguousarray(b.l, dtype=np.int32)
    nprim = np.ascontiguousarray(b.nprim, dtype=np.int32)
    poff = np.ascontiguousarray(b.prim_off, dtype=np.int32)
    exps = np.ascontiguousarray(b.exps, dtype=np.float64)
    coef = np.ascontiguousarray(b.coef, dtype=np.float64)
    keep = (xyz, atom, l, nprim, poff, exps, coef)
    args = (ctypes.c_int(xyz.shape[0]), _d(xyz), ctypes.c_int(l.shape[0]), _i(atom), _i(l), _i(nprim), _i(poff),
            _d(exps), _d(coef))
    return args, keep


def max_threads() -> int:
    return int(lib().orc_max_threads())


def boys(mmax: int, T: float) -> np.ndarray:
    F = np.zeros(mmax + 1)
    lib().orc_boys(ctypes.c_int(mmax), ctypes.c_double(T), _d(F))
    return F


_NC = (1, 3, 6, 10)


def eri_shell(b, A, B, C, D) -> np.ndarray:
    args, keep = _basis_args(b)
    shp = tuple(_NC[int(b.l[s])] for s in (A, B, C, D))
    out = np.zeros(shp)
    lib().orc_eri_shell(*args, ctypes.c_int(A), ctypes.c_int(B), ctypes.c_int(C), ctypes.c_int(D), _d(out))
    return out


def eri_tensor(b) -> np.ndarray:
    """O7: the full N^4 tensor, no symmetry used."""
    args, keep = _basis_args(b)
    n = b.nao
    out = np.zeros((n, n, n, n))
    lib().orc_eri_tensor(*args, _d(out))
    return out


def schwarz(b) -> np.ndarray:
    args, keep = _basis_args(b)
    Q = np.zeros((b.nshell, b.nshell))
    lib().orc_schwarz(*args, _d(Q))
    return Q


def jk_definition(eri: np.ndarray, D: np.ndarray):
    """O7 contraction, Eq. (17) literally.  D: [nD,N,N]."""
    J = np.einsum("mnkr,dkr->dmn", eri, D, optimize=True)
    K = np.einsum("mknr,dkr->dmn", eri, D, optimize=True)
    return J, K


def jk_folded(b, D: np.ndarray, tau: float, pair_range=None, Q=None):
    """O6.  Returns J, K [nD,N,N] and the number of shell quartets kept."""
    args, keep = _basis_args(b)
    D = np.ascontiguousarray(D, dtype=np.float64)
    nD, n, _ = D.shape
    J = np.zeros_like(D)
    K = np.zeros_like(D)
    npair = b.nshell * (b.nshell + 1) // 2
    p0, p1 = (0, npair) if pair_range is None else pair_range
    Qp = _d(np.ascontiguousarray(Q)) if Q is not None else None
    kept = lib().orc_jk_folded(*args, ctypes.c_double(tau), ctypes.c_int(nD), _d(D), _d(J), _d(K),
                               ctypes.c_longlong(p0), ctypes.c_longlong(p1), Qp)
    return J, K, int(kept)


def jk_blocks(b, D: np.ndarray, tau: float, shell_pairs, Q=None):
    """Eq. (17) for sampled ordered shell pairs (X,Y): returns lists of J and K blocks [nD,nx,ny]."""
    args, keep = _basis_args(b)
    D = np.ascontiguousarray(D, dtype=np.float64)
    nD = D.shape[0]
    X = np.asarray([p[0] for p in shell_pairs], dtype=np.int32)
    Y = np.asarray([p[1] for p in shell_pairs], dtype=np.int32)
    sizes = [nD * _NC[int(b.l[x])] * _NC[int(b.l[y])] for x, y in zip(X, Y)]
    off = np.zeros(len(sizes) + 1, dtype=np.int64)
    off[1:] = np.cumsum(sizes)
    Jb = np.zeros(int(off[-1]))
    Kb = np.zeros(int(off[-1]))
    Qp = _d(np.ascontiguousarray(Q)) if Q is not None else None
    lib().orc_jk_blocks(*args, ctypes.c_double(tau), ctypes.c_int(nD), _d(D), ctypes.c_int(len(X)), _i(X), _i(Y),
                        off.ctypes.data_as(_lp), _d(Jb), _d(Kb), Qp)
    Js, Ks = [], []
    for k, (x, y) in enumerate(zip(X, Y)):
        shp = (nD, _NC[int(b.l[x])], _NC[int(b.l[y])])
        Js.append(Jb[off[k]:off[k + 1]].reshape(shp).copy())
        Ks.append(Kb[off[k]:off[k + 1]].reshape(shp).copy())
    return Js, Ks


def jk_grad(b, A: np.ndarray, B: np.ndarray):
    """J^x(A,B), K^x(A,B) of Eq. (18) for nP density pairs; returns two arrays
    [nP, natom, 3].  Plain product rule over the four functions of every ordered shell quartet (orc_jk_grad)."""
    args, keep = _basis_args(b)
    if int(np.max(np.asarray(b.l))) > 2:
        raise ValueError("jk_grad: the derivative oracle raises one index by one and is sized for input shells l <= 2")
    A = np.ascontiguousarray(A, dtype=np.float64)
    B = np.ascontiguousarray(B, dtype=np.float64)
    nP = A.shape[0]
    natom = np.asarray(b.xyz).shape[0]
    gJ = np.zeros((nP, natom, 3))
    gK = np.zeros((nP, natom, 3))
    lib().orc_jk_grad(*args, ctypes.c_int(nP), _d(A), _d(B), _d(gJ), _d(gK))
    return gJ, gK


# ---------------------------------------------------------------------------------------------------------
# O10 pseudo-density, explicit loops (Eqs. (13), (15)):  D^{alpha,d}_{mu nu} =
#     sum_{ia} C_{mu i} e^{+eps_i tau_alpha} T^d_{ia} e^{-eps_a tau_alpha} C_{nu a}
# Output layout [ntau][nT][N][N].  No w_alpha, no 1/2, no spin factor (reading A10).
def pseudo_densities_loops(C_occ, C_vir, eps_occ, eps_vir, T, tau) -> np.ndarray:
    n, nocc = C_occ.shape
    nvir = C_vir.shape[1]
    nT = T.shape[0]
    out = np.zeros((len(tau), nT, n, n))
    for al, t in enumerate(tau):
        for d in range(nT):
            for i in range(nocc):
                u = C_occ[:, i] * np.exp(eps_occ[i] * t)          # U~_{mu i}, Eq. (13)
                for a in range(nvir):
                    v = C_vir[:, a] * np.exp(-eps_vir[a] * t)     # V~_{nu a}, Eq. (13)
                    out[al, d] += T[d, i, a] * np.outer(u, v)     # Eq. (15)
    return out


# ---------------------------------------------------------------------------------------------------------
# O9 minimax exponential-sum approximation of 1/x on [xmin, xmax] (Eq. (11), refs 18-19 of the paper):
# minimise max_x |1/x - sum_a w_a exp(-x tau_a)|.  Solved on [1, R], R = xmax/xmin, then tau = tau^/xmin,
# w = w^/xmin.  Remez exchange: Newton on E(x_j) = (-1)^j delta for the 2k parameters + level at the 2k+1
# alternation points, then every interior point moves to the neighbouring extremum of E; 80-digit arithmetic
# (mpmath) so that the oracle's grid is converged far beyond fp64.  Start: on a WIDER interval [1, R0] (well
# conditioned) a least-squares fit (scipy, a library routine as a step) from the trapezoid rule for
# 1/x = int exp(-x e^s) e^s ds, accepted only if its error curve already has 2k+1 alternating extrema; then
# R0 -> R in geometric steps, each a full Remez solve started from the previous one.
def laplace_minimax(xmin: float, xmax: float, k: int, verbose: bool = False):
    import mpmath as mp
    from scipy.optimize import least_squares
    mp.mp.dps = 80
    R = mp.mpf(xmax) / mp.mpf(xmin)

    def err(x, tau, w):
        return 1 / x - sum(wi * mp.e ** (-x * ti) for ti, wi in zip(tau, w))

    def derr(x, tau, w):
        return -1 / x ** 2 + sum(wi * ti * mp.e ** (-x * ti) for ti, wi in zip(tau, w))

    def remez(Rc, tau, w, xs, iters=60):
        delta = mp.mpf(0)
        n = 2 * k + 1
        for it in range(iters):
            for nit in range(80):
                Fv = mp.matrix(n, 1)
                for j, x in enumerate(xs):
                    Fv[j] = err(x, tau, w) - (-1) ** j * delta
                if nit > 0 and max(abs(v) for v in Fv) < mp.mpf(10) ** (-30) * abs(delta):
                    break
                Jm = mp.matrix(n, n)
                for j, x in enumerate(xs):
                    for a in range(k):
                        ex = mp.e ** (-x * tau[a])
                        Jm[j, a] = w[a] * x * ex
                        Jm[j, k + a] = -ex
                    Jm[j, 2 * k] = -(-1) ** j
                dx = mp.lu_solve(Jm, -Fv)
                # damped Newton: no parameter may change by more than 30 % in one step (keeps them positive)
                rel = max(max(abs(dx[a] / tau[a]), abs(dx[k + a] / w[a])) for a in range(k))
                step = min(mp.mpf(1), mp.mpf("0.3") / rel) if rel > 0 else mp.mpf(1)
                tau = [tau[a] + step * dx[a] for a in range(k)]
                w = [w[a] + step * dx[k + a] for a in range(k)]
                delta = delta + step * dx[2 * k]
            else:
                raise RuntimeError("laplace_minimax: Newton did not converge")
            # exchange: move every interior point to the local extremum of E next to it; endpoints stay
            new = [mp.mpf(1)]
            for j in range(1, 2 * k):
                lo, hi = xs[j - 1], xs[j + 1]
                grid = [lo + (hi - lo) * t / 40 for t in range(41)]
                sgn = mp.sign(err(xs[j], tau, w))
                vals = [err(x, tau, w) * sgn for x in grid]
                m = max(range(41), key=lambda t: vals[t])
                a_, b_ = grid[max(m - 1, 0)], grid[min(m + 1, 40)]
                xr = grid[m]
                if sgn * derr(a_, tau, w) > 0 and sgn * derr(b_, tau, w) < 0:
                    for _ in range(200):            # bisection on the sign of E'
                        mid = (a_ + b_) / 2
                        if sgn * derr(mid, tau, w) > 0:
                            a_ = mid
                        else:
                            b_ = mid
                    xr = (a_ + b_) / 2
                new.append(xr)
            new.append(Rc)
            shift = max(abs(a - b) / b for a, b in zip(new, xs))
            xs = new
            if verbose:
                print("remez R=%s it=%d delta=%s shift=%s" % (mp.nstr(Rc, 6), it, mp.nstr(delta, 8), mp.nstr(shift, 5)))
            if shift < mp.mpf(10) ** (-20):
                return tau, w, delta, xs
        raise RuntimeError("laplace_minimax: exchange did not converge")

    def ls_start(R0):
        n = 1500
        hh = (np.log(R0) + 5.5) / k
        s0 = -np.log(R0) - 2.5 + hh * (np.arange(k) + 0.5)
        p0 = np.concatenate([s0, np.log(hh) + s0])
        xg = np.exp(np.linspace(0.0, np.log(R0), n))

        def res(p):
            return 1.0 / xg - (np.exp(p[k:])[None, :] * np.exp(-xg[:, None] * np.exp(p[:k])[None, :])).sum(1)

        def jac(p):
            t, ww = np.exp(p[:k]), np.exp(p[k:])
            ex = np.exp(-xg[:, None] * t[None, :])
            return np.concatenate([ww * t * xg[:, None] * ex, -ww * ex], axis=1)

        with np.errstate(all="ignore"):
            sol = least_squares(res, p0, jac=jac, method="lm", xtol=1e-15, ftol=1e-15, gtol=1e-15, max_nfev=20000)
        E = res(sol.x)
        idx = [0] + [i for i in range(1, n - 1) if (E[i] - E[i - 1]) * (E[i + 1] - E[i]) < 0] + [n - 1]
        sg = np.sign(E[idx])
        ok = len(idx) == 2 * k + 1 and bool(np.all(sg[1:] * sg[:-1] < 0)) and E[0] > 0
        order = np.argsort(sol.x[:k])
        return ok, np.exp(sol.x[:k])[order], np.exp(sol.x[k:])[order], xg[idx]

    for c in (3.0, 2.6, 3.2, 2.8, 3.4, 2.4, 3.6, 2.2):
        R0 = max(float(R), 10.0 ** (k / c))
        ok, t0, w0, x0 = ls_start(R0)
        if ok:
            break
    else:
        raise RuntimeError("laplace_minimax: no least-squares start with 2k+1 alternating extrema")
    tau = [mp.mpf(float(v)) for v in t0]
    w = [mp.mpf(float(v)) for v in w0]
    xs = [mp.mpf(float(v)) for v in x0]
    xs[0], xs[-1] = mp.mpf(1), mp.mpf(R0)
    Rc = mp.mpf(R0)
    tau, w, delta, xs = remez(Rc, tau, w, xs)
    while Rc > R:
        Rn = max(R, Rc / mp.mpf("1.25"))
        xs = [Rn ** (mp.log(x) / mp.log(Rc)) for x in xs]
        Rc = Rn
        tau, w, delta, xs = remez(Rc, tau, w, xs)
    xm = mp.mpf(xmin)
    tau_o = np.array([float(t / xm) for t in tau])
    w_o = np.array([float(x / xm) for x in w])
    return tau_o, w_o, float(abs(delta) / xm), np.array([float(x * xm) for x in xs])


def laplace_error_curve(tau, w, x):
    x = np.asarray(x, dtype=np.float64)
    return 1.0 / x - (np.asarray(w)[None, :] * np.exp(-x[:, None] * np.asarray(tau)[None, :])).sum(1)


# ---------------------------------------------------------------------------------------------------------
# SURVEY 8(f) N1.  Laplace-Fock back-transform, Eq. (19):
#     F~[d]_pq = sum_{mu nu} C_{mu p} (2 J[d] - K[d])_{mu nu} C_{nu q}
# written as the definition (an einsum, a library contraction as the step), and the quadrature-weighted grid sum with
# the EOM reweighting, Eqs. (11), (21):  Y[t] = sum_a w_a exp(omega tau_a) X[a][t].
def laplace_fock(J: np.ndarray, K: np.ndarray, C: np.ndarray) -> np.ndarray:
    return np.einsum("mp,dmn,nq->dpq", C, 2.0 * J - K, C, optimize=True)


def laplace_fock_loops(J: np.ndarray, K: np.ndarray, C: np.ndarray) -> np.ndarray:
    """Eq. (19) as explicit loops (small cases; pins the einsum)."""
    nD, n, _ = J.shape
    nmo = C.shape[1]
    F = np.zeros((nD, nmo, nmo))
    for d in range(nD):
        for p in range(nmo):
            for q in range(nmo):
                s = 0.0
                for mu in range(n):
                    for nu in range(n):
                        s += C[mu, p] * (2.0 * J[d, mu, nu] - K[d, mu, nu]) * C[nu, q]
                F[d, p, q] = s
    return F


def laplace_accumulate(tau, w, omega: float, X: np.ndarray) -> np.ndarray:
    out = np.zeros(X.shape[1:])
    for a in range(X.shape[0]):
        out += w[a] * np.exp(omega * tau[a]) * X[a]        # w~_a(omega) = w_a e^{omega tau_a}, Eq. (21)
    return out


# ---------------------------------------------------------------------------------------------------------
# SURVEY 8(f) N3.  Particle-particle ladder (Algorithm 2):
#     L[p, a, b] = sum_{ef} (ae|bf) X[p, e, f],        p = a compound occupied pair index (ij),
# with (ae|bf) the integrals over the virtual orbitals C_vir, written as the definition: the AO tensor of O7
# transformed to the virtual MO basis (a library contraction as the step), then the explicit sum over (e, f).
def pp_ladder(eri: np.ndarray, C_vir: np.ndarray, X: np.ndarray) -> np.ndarray:
    mo = np.einsum("mnkr,ma,ne,kb,rf->aebf", eri, C_vir, C_vir, C_vir, C_vir, optimize=True)   # (ae|bf)
    return np.einsum("aebf,pef->pab", mo, X, optimize=True)


def pp_ladder_loops(eri: np.ndarray, C_vir: np.ndarray, X: np.ndarray) -> np.ndarray:
    """The same sum as explicit loops over every index (tiny cases only; pins the einsum index strings)."""
    n, nv = C_vir.shape
    L = np.zeros((X.shape[0], nv, nv))
    for a in range(nv):
        for b in range(nv):
            for e in range(nv):
                for f in range(nv):
                    g = 0.0                                   # (ae|bf) = sum C_ma C_ne (mn|kr) C_kb C_rf
                    for m in range(n):
                        for nn in range(n):
                            for k in range(n):
                                for r in range(n):
                                    g += C_vir[m, a] * C_vir[nn, e] * eri[m, nn, k, r] * C_vir[k, b] * C_vir[r, f]
                    for p in range(X.shape[0]):
                        L[p, a, b] += g * X[p, e, f]
    return L


# ---------------------------------------------------------------------------------------------------------
# SURVEY 8(f) N4, second half: the spherical-harmonic transform at matrix level.  The integrals are Cartesian
# throughout ("730 Cartesian AO"); a caller that works with pure (2l+1) functions converts matrices:
#     chi^sph_{l m} = sum_c S^l[m, c] chi^cart_c,     c = (a, b, c) lexicographic (reading A7), m = -l..l,
# with S^l the monomial coefficients of the Racah-normalised real solid harmonic R_lm = r^l sqrt(4 pi/(2l+1)) Y_lm,
# which has the angular norm of x^l -- the function the caller's N(a,l) normalises (reading A6), so a normalised
# Cartesian shell gives normalised pure functions.  Written out from the closed form of the real solid harmonics
# (Helgaker, Jorgensen, Olsen, Molecular Electronic-Structure Theory, Eqs. 6.4.47-6.4.50):
#     R_lm = N_lm sum_{t=0}^{[(l-|m|)/2]} sum_{u=0}^{t} sum_v C^{lm}_{tuv} x^{2t+|m|-2(u+v)} y^{2(u+v)} z^{l-2t-|m|},
#     C^{lm}_{tuv} = (-1)^{t+v-v_m} (1/4)^t binom(l,t) binom(l-t,|m|+t) binom(t,u) binom(|m|,2v),
#     N_lm = 1/(2^{|m|} l!) sqrt(2 (l+|m|)! (l-|m|)! / 2^{delta_{m0}}),
#     v = v_m, v_m + 1, ..., [|m|/2 - v_m] + v_m,   v_m = 0 (m >= 0), 1/2 (m < 0).
# Operators (J, K, F) transform as X^sph = S X^cart S^T, densities as D^cart = S^T D^sph S, so that
# tr(D^sph^T X^sph) = tr(D^cart^T X^cart).
def sph_matrix(l: int) -> np.ndarray:
    from math import comb, factorial, sqrt
    comps = [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]
    S = np.zeros((2 * l + 1, len(comps)))
    for m in range(-l, l + 1):
        am = abs(m)
        N = sqrt(2.0 * factorial(l + am) * factorial(l - am) / (2.0 if m == 0 else 1.0)) / (2.0 ** am * factorial(l))
        two_vm = 0 if m >= 0 else 1                              # 2 v_m
        nv = (am - two_vm) // 2                                  # [|m|/2 - v_m]
        for t in range((l - am) // 2 + 1):
            for u in range(t + 1):
                for k in range(nv + 1):                          # v = v_m + k, 2v = 2 v_m + 2k
                    two_v = two_vm + 2 * k
                    C = (-1.0) ** (t + k) * 0.25 ** t * comb(l, t) * comb(l - t, am + t) * comb(t, u) * comb(am, two_v)
                    ex = (2 * t + am - 2 * u - two_v, 2 * u + two_v, l - 2 * t - am)
                    S[m + l, comps.index(ex)] += N * C
    return S


def sph_block_matrix(b) -> np.ndarray:
    """S of the whole basis: block diagonal [N_sph, N_cart], shells in the caller's order."""
    ls = [int(x) for x in np.asarray(b.l)]
    S = np.zeros((sum(2 * l + 1 for l in ls), sum((l + 1) * (l + 2) // 2 for l in ls)))
    r = c = 0
    for l in ls:
        Sl = sph_matrix(l)
        S[r:r + Sl.shape[0], c:c + Sl.shape[1]] = Sl
        r += Sl.shape[0]
        c += Sl.shape[1]
    return S


def sph_from_cart(b, X: np.ndarray) -> np.ndarray:
    """Operator matrices [n, N_cart, N_cart] -> [n, N_sph, N_sph]:  S X S^T."""
    S = sph_block_matrix(b)
    return np.stack([S @ x @ S.T for x in np.asarray(X, dtype=np.float64)])


def cart_from_sph(b, D: np.ndarray) -> np.ndarray:
    """Density matrices [n, N_sph, N_sph] -> [n, N_cart, N_cart]:  S^T D S."""
    S = sph_block_matrix(b)
    return np.stack([S.T @ d @ S for d in np.asarray(D, dtype=np.float64)])

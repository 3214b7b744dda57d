// ltjk_laplace.cpp -- step a3: minimax Laplace quadrature (Eq. 11; Alg. 1 line 4, L200).
//
//   1/x ~ sum_a w_a exp(-x tau_a),  minimise  max_{x in [xmin,xmax]} |1/x - sum_a w_a exp(-x tau_a)|.
//
// Host code, quadruple precision (__float128): the problem is solved on [1,R], R = xmax/xmin, and scaled
// (tau = tau^/xmin, w = w^/xmin).  Method (this library's own code; the CPU oracle is an independent Python/mpmath
// implementation in 80-digit arithmetic, reading A8):
//   1. start on a wide interval [1,R0]: Levenberg-Marquardt least squares in (log tau, log w) on a logarithmic
//      grid (80-bit long double: only a start guess, 2x faster than quad), from the trapezoid rule for 1/x = int exp(-x e^s) e^s ds; accepted only if its error curve has
//      2k+1 alternating extrema (else another R0 is tried);
//   2. Remez exchange: Newton on E(x_j) = (-1)^j delta for (tau, w, delta), then every interior x_j moves to the
//      neighbouring extremum of E; repeated to convergence;
//   3. continuation R0 -> R in geometric steps, each a full Remez solve.
// No fallback grid: failure returns LTJK_ENOCONV.
#include "../../include/ltjk.h"
#include <quadmath.h>
#include <algorithm>
#include <cmath>
#include <vector>

namespace {

typedef __float128 real;
typedef std::vector<real> vec;

inline real qexp(real x) { return expq(x); }
inline real qlog(real x) { return logq(x); }
inline real qabs(real x) { return fabsq(x); }

struct Grid { vec tau, w; };

real err_at(const Grid& g, real x)
{
    real s = 0;
    for (size_t a = 0; a < g.tau.size(); ++a) s += g.w[a] * qexp(-x * g.tau[a]);
    return 1 / x - s;
}

real derr_at(const Grid& g, real x)
{
    real s = 0;
    for (size_t a = 0; a < g.tau.size(); ++a) s += g.w[a] * g.tau[a] * qexp(-x * g.tau[a]);
    return -1 / (x * x) + s;
}

template <class R> inline R absr(R x) { return x < 0 ? -x : x; }
// Gaussian elimination with partial pivoting; A is n x n row-major, b overwritten with the solution.
template <class R>
bool solve_t(std::vector<R>& A, std::vector<R>& b, int n)
{
    for (int c = 0; c < n; ++c) {
        int p = c;
        for (int r = c + 1; r < n; ++r) if (absr(A[r * n + c]) > absr(A[p * n + c])) p = r;
        if (A[p * n + c] == 0) return false;
        if (p != c) { for (int j = 0; j < n; ++j) std::swap(A[c * n + j], A[p * n + j]); std::swap(b[c], b[p]); }
        for (int r = c + 1; r < n; ++r) {
            const R f = A[r * n + c] / A[c * n + c];
            if (f == 0) continue;
            for (int j = c; j < n; ++j) A[r * n + j] -= f * A[c * n + j];
            b[r] -= f * b[c];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        R s = b[r];
        for (int j = r + 1; j < n; ++j) s -= A[r * n + j] * b[j];
        b[r] = s / A[r * n + r];
    }
    return true;
}


bool solve(std::vector<real>& A, vec& b, int n) { return solve_t<real>(A, b, n); }

// Step 1: LM least squares on a log grid of [1,R0] in p = (log tau, log w).
bool ls_start(int k, real R0q, Grid& g)
{
    typedef long double lreal;
    typedef std::vector<lreal> lvec;
    const lreal R0 = (lreal)R0q;
    const int n = 400, np = 2 * k;
    lvec xg(n);
    for (int i = 0; i < n; ++i) xg[i] = expl(logl(R0) * i / (n - 1));
    const lreal lo = 2.5L, hi = 3.0L, hh = (logl(R0) + lo + hi) / k;
    lvec p(np);
    for (int a = 0; a < k; ++a) { p[a] = -logl(R0) - lo + hh * (a + 0.5L); p[k + a] = logl(hh) + p[a]; }
    auto residual = [&](const lvec& q, lvec& r) {
        lreal s2 = 0;
        for (int i = 0; i < n; ++i) {
            lreal s = 0;
            for (int a = 0; a < k; ++a) s += expl(q[k + a] - xg[i] * expl(q[a]));
            r[i] = 1 / xg[i] - s;
            s2 += r[i] * r[i];
        }
        return s2;
    };
    lvec r(n), rn(n), pn(np);
    lreal f = residual(p, r), lam = 1e-3L;
    std::vector<lreal> Jm((size_t)n * np), A((size_t)np * np);
    lvec gvec(np), d(np);
    for (int it = 0; it < 3000; ++it) {
        for (int i = 0; i < n; ++i)
            for (int a = 0; a < k; ++a) {
                const lreal t = expl(p[a]), e = expl(p[k + a] - xg[i] * t);
                Jm[(size_t)i * np + a] = e * xg[i] * t;      // d r_i / d log tau_a
                Jm[(size_t)i * np + k + a] = -e;              // d r_i / d log w_a
            }
        for (int a = 0; a < np; ++a) {
            lreal s = 0;
            for (int i = 0; i < n; ++i) s += Jm[(size_t)i * np + a] * r[i];
            gvec[a] = s;
            for (int b = a; b < np; ++b) {
                lreal t = 0;
                for (int i = 0; i < n; ++i) t += Jm[(size_t)i * np + a] * Jm[(size_t)i * np + b];
                A[(size_t)a * np + b] = A[(size_t)b * np + a] = t;
            }
        }
        bool improved = false;
        for (int tries = 0; tries < 40; ++tries) {
            std::vector<lreal> M = A;
            for (int a = 0; a < np; ++a) { M[(size_t)a * np + a] += lam * A[(size_t)a * np + a]; d[a] = -gvec[a]; }
            if (solve_t<lreal>(M, d, np)) {
                lreal big = 0;
                for (int a = 0; a < np; ++a) big = std::max<lreal>(big, fabsl(d[a]));
                const lreal sc = big > 2 ? 2 / big : 1;
                for (int a = 0; a < np; ++a) pn[a] = p[a] + sc * d[a];
                const lreal fn = residual(pn, rn);
                if (fn < f) {
                    const lreal rel = (f - fn) / f;
                    p = pn; r = rn; f = fn; lam = std::max<lreal>(lam / 3, 1e-30L);
                    improved = true;
                    if (rel < 1e-14L) it = 1 << 30;
                    break;
                }
            }
            lam *= 4;
        }
        if (!improved || it == (1 << 30)) break;
    }
    g.tau.resize(k); g.w.resize(k);
    std::vector<std::pair<double, int>> order(k);
    for (int a = 0; a < k; ++a) order[a] = {(double)p[a], a};
    std::sort(order.begin(), order.end());
    for (int a = 0; a < k; ++a) { g.tau[a] = (real)expl(p[order[a].second]); g.w[a] = (real)expl(p[k + order[a].second]); }
    return true;
}

// Local extrema of the error curve on [1,R] (endpoints included), refined by bisection on E'.
vec find_extrema(const Grid& g, real R, int ngrid)
{
    vec xs;
    vec x(ngrid), e(ngrid);
    for (int i = 0; i < ngrid; ++i) { x[i] = qexp(qlog(R) * i / (ngrid - 1)); e[i] = err_at(g, x[i]); }
    xs.push_back(1);
    for (int i = 1; i + 1 < ngrid; ++i)
        if ((e[i] - e[i - 1]) * (e[i + 1] - e[i]) < 0) {
            real a = x[i - 1], b = x[i + 1];
            const real da = derr_at(g, a);
            for (int it = 0; it < 110; ++it) {
                const real m = (a + b) / 2;
                if ((derr_at(g, m) > 0) == (da > 0)) a = m; else b = m;
            }
            xs.push_back((a + b) / 2);
        }
    xs.push_back(R);
    return xs;
}

bool alternates(const Grid& g, const vec& xs)
{
    for (size_t j = 1; j < xs.size(); ++j)
        if ((err_at(g, xs[j]) > 0) == (err_at(g, xs[j - 1]) > 0)) return false;
    return true;
}

// Step 2: Remez exchange on [1,R] from (g, xs).  Returns false if Newton breaks down or nothing converges.
bool remez(int k, real R, Grid& g, vec& xs, real& delta)
{
    const int n = 2 * k + 1;
    delta = 0;
    for (int outer = 0; outer < 80; ++outer) {
        bool newton_ok = false;
        for (int nit = 0; nit < 80; ++nit) {
            std::vector<real> Jm((size_t)n * n);
            vec F(n);
            for (int j = 0; j < n; ++j) {
                const real sg = (j & 1) ? -1 : 1;
                F[j] = -(err_at(g, xs[j]) - sg * delta);
                for (int a = 0; a < k; ++a) {
                    const real ex = qexp(-xs[j] * g.tau[a]);
                    Jm[(size_t)j * n + a] = g.w[a] * xs[j] * ex;
                    Jm[(size_t)j * n + k + a] = -ex;
                }
                Jm[(size_t)j * n + 2 * k] = -sg;
            }
            real resid = 0;
            for (int j = 0; j < n; ++j) resid = std::max<real>(resid, qabs(F[j]));
            // converged when the alternation equations hold to 1e-12 of the level (Newton steps themselves are
            // only as accurate as cond(J) * 1e-34 allows, so the test is on the residual, not on the step)
            if (nit > 0 && resid < 1e-12Q * qabs(delta)) { newton_ok = true; break; }
            if (!solve(Jm, F, n)) return false;
            real rel = 0;
            for (int a = 0; a < k; ++a) rel = std::max<real>(rel, std::max<real>(qabs(F[a] / g.tau[a]), qabs(F[k + a] / g.w[a])));
            const real step = rel > 0.3Q ? 0.3Q / rel : 1;
            for (int a = 0; a < k; ++a) { g.tau[a] += step * F[a]; g.w[a] += step * F[k + a]; }
            delta += step * F[2 * k];
            for (int a = 0; a < k; ++a) if (!(g.tau[a] > 0) || !(g.w[a] > 0)) return false;
        }
        if (!newton_ok) return false;
        // exchange
        real shift = 0;
        vec nx(n);
        nx[0] = 1; nx[n - 1] = R;
        for (int j = 1; j + 1 < n; ++j) {
            const real lo = xs[j - 1], hi = xs[j + 1];
            const real sg = err_at(g, xs[j]) > 0 ? 1 : -1;
            const int m = 48;
            int best = 0; real bv = -1e300Q;
            for (int t = 0; t <= m; ++t) {
                const real v = sg * err_at(g, lo + (hi - lo) * t / m);
                if (v > bv) { bv = v; best = t; }
            }
            real a = lo + (hi - lo) * std::max(best - 1, 0) / m, b = lo + (hi - lo) * std::min(best + 1, m) / m;
            // maximum of sg*E in [a,b]: bisection on the sign of sg*E'
            if (sg * derr_at(g, a) > 0 && sg * derr_at(g, b) < 0) {
                for (int it = 0; it < 110; ++it) {
                    const real mid = (a + b) / 2;
                    if (sg * derr_at(g, mid) > 0) a = mid; else b = mid;
                }
                nx[j] = (a + b) / 2;
            } else {
                nx[j] = lo + (hi - lo) * best / m;
            }
            shift = std::max<real>(shift, qabs(nx[j] - xs[j]) / xs[j]);
        }
        xs = nx;
        if (shift < 1e-10Q) return true;   // E is stationary at x_j: the level is then good to ~shift^2
    }
    return false;
}

bool minimax(int k, real R, Grid& g, real& delta)
{
    const double cs[] = {3.0, 2.6, 3.2, 2.8, 3.4, 2.4, 3.6, 2.2};
    for (double c : cs) {
        real R0 = powq(10, (real)k / (real)c);
        if (R0 < R) R0 = R;
        Grid s;
        ls_start(k, R0, s);
        vec xs = find_extrema(s, R0, 3000);
        if ((int)xs.size() != 2 * k + 1 || !alternates(s, xs)) continue;
        real Rc = R0;
        bool ok = remez(k, Rc, s, xs, delta);
        while (ok && Rc > R) {
            real Rn = Rc / 1.2Q;
            if (Rn < R) Rn = R;
            for (auto& x : xs) x = qexp(qlog(x) * qlog(Rn) / qlog(Rc));
            Rc = Rn;
            ok = remez(k, Rc, s, xs, delta);
        }
        if (ok) { g = s; return true; }
    }
    return false;
}

}  // namespace

extern "C" int ltjk_laplace_quadrature(double xmin, double xmax, int npts, double* t, double* w, double* maxerr)
{
    if (!(xmin > 0.0) || !(xmax > xmin) || npts < 2 || npts > 14 || !t || !w) return LTJK_EINVAL;
    Grid g;
    real delta = 0;
    const real R = (real)xmax / (real)xmin;
    if (!minimax(npts, R, g, delta)) return LTJK_ENOCONV;
    for (int a = 0; a < npts; ++a) { t[a] = (double)(g.tau[a] / (real)xmin); w[a] = (double)(g.w[a] / (real)xmin); }
    if (maxerr) {
        // achieved maximum error of the ROUNDED (double) grid on [xmin,xmax], evaluated in quad precision
        Grid gd;
        gd.tau.resize(npts); gd.w.resize(npts);
        for (int a = 0; a < npts; ++a) { gd.tau[a] = (real)t[a]; gd.w[a] = (real)w[a]; }
        real m = 0;
        const int n = 20001;
        for (int i = 0; i < n; ++i) {
            const real x = (real)xmin * qexp(qlog(R) * i / (n - 1));
            m = std::max<real>(m, qabs(err_at(gd, x)));
        }
        *maxerr = (double)m;
    }
    return LTJK_OK;
}

/*
 * ltjk_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, fp64 implementation of what the hot path computes, written from the paper
 * (/root/reference/PAPER.md, cited as PAPER.md:L<n>) and textbook integral theory (McMurchie-Davidson).
 * It shares NO code with the CUDA path (paper_2607_05622_b200/csrc uses Obara-Saika/HGP recurrences and
 * its own Boys evaluator).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.
 *
 * What it computes:
 *   J(D)_{mu nu} = sum_{kappa rho} (mu nu|kappa rho) D_{kappa rho}
 *   K(D)_{mu nu} = sum_{kappa rho} (mu kappa|nu rho) D_{kappa rho}          PAPER.md:L157 Eq. (17)
 * for a general (non-symmetric) D, over contracted Cartesian Gaussians
 *   chi(r) = (x-Ax)^i (y-Ay)^j (z-Az)^k sum_p coef_p exp(-a_p |r-A|^2)      (readings A6, A7)
 * with pure-integral Schwarz screening Q_AB Q_CD < tau dropped
 *
 * Steps:
 *   orc_boys           O2  Boys function F_m(T)
 *   hermite_E          O3  Hermite expansion coefficients E_t^{ij}
 *   hermite_R          O4  Hermite Coulomb integrals R^n_{tuv}
 *   orc_eri_shell      O5  contracted shell quartet
 *   orc_jk_folded      O6  canonical-quartet digestion, all 8 images (Eq. (25) PAPER.md:L320 generalised)
 *   orc_eri_tensor     O7  full N^4 tensor with NO symmetry use (definition mode; contraction is an einsum
 *                          in oracle/oracle.py)
 *   orc_schwarz        O8  Q_AB = sqrt(max |(ab|ab)|)
 *   orc_jk_blocks          J and K blocks for sampled shell pairs straight from Eq. (17) (full-size sampling)
 *   orc_jk_grad            SURVEY 8(f) N2: derivative builds J^x(A,B), K^x(A,B), Eq. (18), written out
 *                          term by term (one term per differentiated function), no symmetry used
 *
 * Input shells: Cartesian s, p, d, f (f: SURVEY.md 8(f) row N4); orc_jk_grad: s, p, d.
 *
 * Pins (tests/test_oracle_*.py): Boys vs mpmath quadrature / gammainc / closed forms; (ss|ss) closed form,
 * 2 sqrt(a/pi), erf(sqrt(rho) R)/R; centre derivatives of the closed-form (ss|ss) in 150-198 digit arithmetic for
 * sampled components of every class family up to (dd|dd) and of the f classes up to (ff|ff); 8-fold symmetry of O7;
 * Cauchy-Schwarz, PSD; translation/rotation invariance; O6 vs O7; J/K symmetry relations; orc_jk_grad: central finite
 * differences of tr(A^T J[B]), tr(A^T K[B]) built from orc_eri_tensor, closed form d/dR [erf(sqrt(rho) R)/R], the
 * translational sum rule Eq. (31), J^x(A,B) = J^x(B,A), K^x(A,B) = K^x(B,A) = K^x(A^T,B^T)  (tests/test_oracle_grad.py).
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <omp.h>

#define LMAXSH 3                   /* largest angular momentum of an input shell of the value builds (s, p, d, f; row N4) */
#define LMAXW 3                    /* largest angular momentum inside eri_shell: f input shells, or the derivative builds
                                      (orc_jk_grad, input shells l <= 2 only) raising ONE index by one */
#define LTOT (4 * LMAXW)           /* 12 */
#define NH1 (2 * LMAXW + 1)        /* Hermite orders per pair and dimension */
#define NR (LTOT + 1)              /* 13 */
#define NCMAX 10                   /* Cartesian components of an l = LMAXW shell */
#define NQMAX (NCMAX * NCMAX * NCMAX * NCMAX)   /* integrals of one (ff|ff) shell quartet */

static const double PI = 3.14159265358979323846264338327950288;

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

/* lexicographic Cartesian components: l=1: x,y,z ; l=2: xx,xy,xz,yy,yz,zz   (reading A7) */
static void cart_list(int l, int (*ijk)[3])
{
    int n = 0;
    for (int i = l; i >= 0; --i)
        for (int j = l - i; j >= 0; --j) {
            ijk[n][0] = i; ijk[n][1] = j; ijk[n][2] = l - i - j; ++n;
        }
}

/* O2. Boys function F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt, m = 0..mmax.
 * T < 35 : series at M = mmax, F_M = e^{-T} sum_k (2T)^k / [(2M+1)(2M+3)...(2M+2k+1)], then downward
 *          recursion F_{m-1} = (2T F_m + e^{-T}) / (2m-1);
 * T >= 35: F_0 = (1/2) sqrt(pi/T) erf(sqrt T), upward F_{m+1} = ((2m+1) F_m - e^{-T}) / (2T). */
void orc_boys(int mmax, double T, double *F)
{
    if (T < 35.0) {
        double term = 1.0 / (2 * mmax + 1), sum = term;
        for (int k = 1; k < 400; ++k) {
            term *= 2.0 * T / (2 * mmax + 2 * k + 1);
            sum += term;
            if (term < 1e-18 * sum) break;
        }
        double e = exp(-T);
        F[mmax] = e * sum;
        for (int m = mmax; m >= 1; --m) F[m - 1] = (2.0 * T * F[m] + e) / (2 * m - 1);
    } else {
        double e = exp(-T);
        F[0] = 0.5 * sqrt(PI / T) * erf(sqrt(T));
        for (int m = 0; m < mmax; ++m) F[m + 1] = ((2 * m + 1) * F[m] - e) / (2.0 * T);
    }
}

/* O3. 1-D Hermite expansion coefficients E[i][j][t], 0<=i<=la, 0<=j<=lb, 0<=t<=i+j, for one Cartesian
 * direction of one primitive pair:  E_0^{00} = exp(-mu X_AB^2), mu = ab/p,
 *   E_t^{i+1,j} = E_{t-1}^{ij}/(2p) + X_PA E_t^{ij} + (t+1) E_{t+1}^{ij}
 *   E_t^{i,j+1} = E_{t-1}^{ij}/(2p) + X_PB E_t^{ij} + (t+1) E_{t+1}^{ij}           (zero outside 0<=t<=i+j) */
static void hermite_E(int la, int lb, double a, double b, double XA, double XB,
                      double E[LMAXW + 1][LMAXW + 1][NH1])
{
    double p = a + b, mu = a * b / p, XAB = XA - XB, XP = (a * XA + b * XB) / p;
    double XPA = XP - XA, XPB = XP - XB;
    memset(E, 0, sizeof(double) * (LMAXW + 1) * (LMAXW + 1) * NH1);
    E[0][0][0] = exp(-mu * XAB * XAB);
    for (int i = 0; i <= la; ++i) {
        if (i > 0)   /* raise i: from (i-1, 0) */
            for (int t = 0; t <= i; ++t) {
                double v = XPA * E[i - 1][0][t];
                if (t > 0) v += E[i - 1][0][t - 1] / (2.0 * p);
                if (t + 1 <= i - 1) v += (t + 1) * E[i - 1][0][t + 1];
                E[i][0][t] = v;
            }
        for (int j = 1; j <= lb; ++j)   /* raise j: from (i, j-1) */
            for (int t = 0; t <= i + j; ++t) {
                double v = XPB * E[i][j - 1][t];
                if (t > 0) v += E[i][j - 1][t - 1] / (2.0 * p);
                if (t + 1 <= i + j - 1) v += (t + 1) * E[i][j - 1][t + 1];
                E[i][j][t] = v;
            }
    }
}

/* O4. Hermite Coulomb integrals R^0_{tuv}, t+u+v <= L:
 *   R^n_{000} = (-2 rho)^n F_n(rho R_PQ^2),
 *   R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X_PQ R^{n+1}_{t,u,v}   (same in u, v). */
static void hermite_R(int L, double rho, const double PQ[3], double R0[NR][NR][NR])
{
    double F[NR];
    double Rn[NR][NR][NR][NR]; /* [n][t][u][v] */
    double T = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
    orc_boys(L, T, F);   /* every Rn entry read below was written at a lower total order: no clearing needed */
    double f = 1.0;
    for (int n = 0; n <= L; ++n) { Rn[n][0][0][0] = f * F[n]; f *= -2.0 * rho; }
    for (int N = 1; N <= L; ++N)            /* total Hermite order t+u+v = N */
        for (int t = 0; t <= N; ++t)
            for (int u = 0; u <= N - t; ++u) {
                int v = N - t - u;
                for (int n = 0; n <= L - N; ++n) {
                    double val;
                    if (t > 0)
                        val = (t - 1 > 0 ? (t - 1) * Rn[n + 1][t - 2][u][v] : 0.0) + PQ[0] * Rn[n + 1][t - 1][u][v];
                    else if (u > 0)
                        val = (u - 1 > 0 ? (u - 1) * Rn[n + 1][t][u - 2][v] : 0.0) + PQ[1] * Rn[n + 1][t][u - 1][v];
                    else
                        val = (v - 1 > 0 ? (v - 1) * Rn[n + 1][t][u][v - 2] : 0.0) + PQ[2] * Rn[n + 1][t][u][v - 1];
                    Rn[n][t][u][v] = val;
                }
            }
    for (int t = 0; t <= L; ++t)
        for (int u = 0; u <= L - t; ++u)
            for (int v = 0; v <= L - t - u; ++v) R0[t][u][v] = Rn[0][t][u][v];
}

typedef struct {
    int natom; const double *xyz; int nshell; const int *atom, *l, *nprim, *prim_off;
    const double *exps, *coef;
} basis_t;

#define BASIS_ARGS int natom, const double *xyz, int nshell, const int *atom, const int *l, const int *nprim, \
                   const int *prim_off, const double *exps, const double *coef
#define BASIS_INIT { natom, xyz, nshell, atom, l, nprim, prim_off, exps, coef }

/* O5. Contracted Cartesian shell quartet (AB|CD) -> out[na][nb][nc][nd] (row-major).
 *   (ab|cd) = 2 pi^{5/2} / (p q sqrt(p+q)) sum_{tuv} E^{ab}_{tuv} sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'}
 *             R^0_{t+t',u+u',v+v'},   E_{tuv} = E_t^x E_u^y E_v^z,  R built on P-Q with rho = pq/(p+q). */
static void eri_shell(const basis_t *bs, int A, int B, int C, int D, double *out)
{
    int la = bs->l[A], lb = bs->l[B], lc = bs->l[C], ld = bs->l[D];
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    int L = la + lb + lc + ld;
    int ca[NCMAX][3], cb[NCMAX][3], cc[NCMAX][3], cd[NCMAX][3];
    cart_list(la, ca); cart_list(lb, cb); cart_list(lc, cc); cart_list(ld, cd);
    const double *RA = bs->xyz + 3 * bs->atom[A], *RB = bs->xyz + 3 * bs->atom[B];
    const double *RC = bs->xyz + 3 * bs->atom[C], *RD = bs->xyz + 3 * bs->atom[D];
    int ntot = na * nb * nc * nd;
    for (int i = 0; i < ntot; ++i) out[i] = 0.0;

    for (int ia = 0; ia < bs->nprim[A]; ++ia)
    for (int ib = 0; ib < bs->nprim[B]; ++ib) {
        double a = bs->exps[bs->prim_off[A] + ia], b = bs->exps[bs->prim_off[B] + ib];
        double cab = bs->coef[bs->prim_off[A] + ia] * bs->coef[bs->prim_off[B] + ib];
        double p = a + b, P[3];
        double Eab[3][LMAXW + 1][LMAXW + 1][NH1];
        for (int x = 0; x < 3; ++x) {
            P[x] = (a * RA[x] + b * RB[x]) / p;
            hermite_E(la, lb, a, b, RA[x], RB[x], Eab[x]);
        }
        for (int ic = 0; ic < bs->nprim[C]; ++ic)
        for (int id = 0; id < bs->nprim[D]; ++id) {
            double c = bs->exps[bs->prim_off[C] + ic], d = bs->exps[bs->prim_off[D] + id];
            double ccd = bs->coef[bs->prim_off[C] + ic] * bs->coef[bs->prim_off[D] + id];
            double q = c + d, Q[3], PQ[3];
            double Ecd[3][LMAXW + 1][LMAXW + 1][NH1];
            for (int x = 0; x < 3; ++x) {
                Q[x] = (c * RC[x] + d * RD[x]) / q;
                PQ[x] = P[x] - Q[x];
                hermite_E(lc, ld, c, d, RC[x], RD[x], Ecd[x]);
            }
            double rho = p * q / (p + q);
            double R0[NR][NR][NR];
            hermite_R(L, rho, PQ, R0);
            double pref = 2.0 * pow(PI, 2.5) / (p * q * sqrt(p + q)) * cab * ccd;

            for (int kc = 0; kc < nc; ++kc)
            for (int kd = 0; kd < nd; ++kd) {
                /* G[t][u][v] = sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R_{t+t',u+u',v+v'}  (inner bracket) */
                double G[NH1][NH1][NH1];
                int tcmax = cc[kc][0] + cd[kd][0], ucmax = cc[kc][1] + cd[kd][1], vcmax = cc[kc][2] + cd[kd][2];
                for (int t = 0; t <= la + lb; ++t)
                for (int u = 0; u <= la + lb - t; ++u)
                for (int v = 0; v <= la + lb - t - u; ++v) {
                    double s = 0.0;
                    for (int t2 = 0; t2 <= tcmax; ++t2)
                    for (int u2 = 0; u2 <= ucmax; ++u2)
                    for (int v2 = 0; v2 <= vcmax; ++v2) {
                        double e = Ecd[0][cc[kc][0]][cd[kd][0]][t2] * Ecd[1][cc[kc][1]][cd[kd][1]][u2]
                                 * Ecd[2][cc[kc][2]][cd[kd][2]][v2];
                        double sg = ((t2 + u2 + v2) & 1) ? -1.0 : 1.0;
                        s += sg * e * R0[t + t2][u + u2][v + v2];
                    }
                    G[t][u][v] = s;
                }
                for (int ka = 0; ka < na; ++ka)
                for (int kb = 0; kb < nb; ++kb) {
                    int tmax = ca[ka][0] + cb[kb][0], umax = ca[ka][1] + cb[kb][1], vmax = ca[ka][2] + cb[kb][2];
                    double s = 0.0;
                    for (int t = 0; t <= tmax; ++t)
                    for (int u = 0; u <= umax; ++u)
                    for (int v = 0; v <= vmax; ++v)
                        s += Eab[0][ca[ka][0]][cb[kb][0]][t] * Eab[1][ca[ka][1]][cb[kb][1]][u]
                           * Eab[2][ca[ka][2]][cb[kb][2]][v] * G[t][u][v];
                    out[((ka * nb + kb) * nc + kc) * nd + kd] += pref * s;
                }
            }
        }
    }
}

void orc_eri_shell(BASIS_ARGS, int A, int B, int C, int D, double *out)
{
    basis_t bs = BASIS_INIT;
    eri_shell(&bs, A, B, C, D, out);
}

static void ao_offsets(const basis_t *bs, int *off)
{
    off[0] = 0;
    for (int s = 0; s < bs->nshell; ++s) off[s + 1] = off[s] + ncart(bs->l[s]);
}

int orc_nao(BASIS_ARGS)
{
    basis_t bs = BASIS_INIT; int n = 0;
    for (int s = 0; s < bs.nshell; ++s) n += ncart(bs.l[s]);
    (void)natom; (void)xyz; (void)atom; (void)nprim; (void)prim_off; (void)exps; (void)coef;
    return n;
}

/* O7. Full tensor eri[mu][nu][kappa][rho], every ORDERED shell quartet computed independently
 * (no permutational symmetry is used anywhere).  Caller allocates N^4 doubles. */
void orc_eri_tensor(BASIS_ARGS, double *eri)
{
    basis_t bs = BASIS_INIT;
    int *off = (int *)malloc(sizeof(int) * (nshell + 1));
    ao_offsets(&bs, off);
    long N = off[nshell];
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * NQMAX);
#pragma omp for collapse(2) schedule(dynamic)
        for (int A = 0; A < nshell; ++A)
        for (int B = 0; B < nshell; ++B)
            for (int C = 0; C < nshell; ++C)
            for (int D = 0; D < nshell; ++D) {
                eri_shell(&bs, A, B, C, D, buf);
                int na = ncart(l[A]), nb = ncart(l[B]), nc = ncart(l[C]), nd = ncart(l[D]);
                for (int a = 0; a < na; ++a) for (int b = 0; b < nb; ++b)
                for (int c = 0; c < nc; ++c) for (int d = 0; d < nd; ++d)
                    eri[(((off[A] + a) * N + off[B] + b) * N + off[C] + c) * N + off[D] + d] =
                        buf[((a * nb + b) * nc + c) * nd + d];
            }
        free(buf);
    }
    free(off);
}

/* O8. Schwarz bounds Q[A*nshell+B] = sqrt(max_{a in A, b in B} |(ab|ab)|). */
void orc_schwarz(BASIS_ARGS, double *Q)
{
    basis_t bs = BASIS_INIT;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * NQMAX);
#pragma omp for schedule(dynamic)
        for (int A = 0; A < nshell; ++A)
            for (int B = 0; B <= A; ++B) {
                eri_shell(&bs, A, B, A, B, buf);
                int na = ncart(l[A]), nb = ncart(l[B]);
                double m = 0.0;
                for (int a = 0; a < na; ++a) for (int b = 0; b < nb; ++b) {
                    double v = fabs(buf[((a * nb + b) * na + a) * nb + b]);
                    if (v > m) m = v;
                }
                Q[A * nshell + B] = Q[B * nshell + A] = sqrt(m);
            }
        free(buf);
    }
}

/* O6. Folded digestion.  Loop canonical shell quartets A>=B, C>=D, (AB)>=(CD) with pair index
 * A(A+1)/2+B, restricted to bra pairs pair_begin <= (AB) < pair_end (full build: 0 .. nshell(nshell+1)/2);
 * skip if Q_AB Q_CD < tau; s = 1, x1/2 if A==B, x1/2 if C==D, x1/2 if (AB)==(CD); then for ALL functions
 * of the quartet and I = s (mu nu|kappa rho), for every density:
 *   J_mn += I (D_kr + D_rk)   J_nm += same   J_kr += I (D_mn + D_nm)   J_rk += same
 *   K_mk += I D_nr   K_nk += I D_mr   K_mr += I D_nk   K_nr += I D_mk
 *   K_km += I D_rn   K_rm += I D_kn   K_kn += I D_rm   K_rn += I D_km
 * (Eq. (25) PAPER.md:L320 written out for all 8 permutational images; readings A4, A5.)
 * D, J, K are [nD][N][N] row-major; J and K are overwritten.  Returns the number of shell quartets kept. */
long long orc_jk_folded(BASIS_ARGS, double tau, int nD, const double *D, double *J, double *K,
                        long long pair_begin, long long pair_end, const double *Qin)
{
    basis_t bs = BASIS_INIT;
    int *off = (int *)malloc(sizeof(int) * (nshell + 1));
    ao_offsets(&bs, off);
    long N = off[nshell];
    double *Q = (double *)malloc(sizeof(double) * nshell * nshell);
    if (Qin) memcpy(Q, Qin, sizeof(double) * nshell * nshell);
    else orc_schwarz(natom, xyz, nshell, atom, l, nprim, prim_off, exps, coef, Q);
    /* density-fastest copies so that the 12 updates are unit-stride loops over the density index */
    size_t sz = (size_t)N * N * nD;
    double *Dd = (double *)malloc(sizeof(double) * sz);
    for (int d = 0; d < nD; ++d)
        for (long i = 0; i < N * N; ++i) Dd[i * nD + d] = D[(size_t)d * N * N + i];
    int nthr = omp_get_max_threads();
    double *Jt = (double *)calloc(sz * nthr, sizeof(double));
    double *Kt = (double *)calloc(sz * nthr, sizeof(double));
    long long kept = 0;
#pragma omp parallel reduction(+ : kept)
    {
        int tid = omp_get_thread_num();
        double *Jp = Jt + sz * tid, *Kp = Kt + sz * tid;
        double *buf = (double *)malloc(sizeof(double) * NQMAX);
#pragma omp for schedule(dynamic)
        for (long long ab = pair_begin; ab < pair_end; ++ab) {
            int A = (int)((sqrt(8.0 * (double)ab + 1.0) - 1.0) / 2.0);
            while ((long long)A * (A + 1) / 2 > ab) --A;
            while ((long long)(A + 1) * (A + 2) / 2 <= ab) ++A;
            int B = (int)(ab - (long long)A * (A + 1) / 2);
            for (int C = 0; C <= A; ++C)
            for (int Dd_ = 0; Dd_ <= C; ++Dd_) {
                long long cd = (long long)C * (C + 1) / 2 + Dd_;
                if (cd > ab) continue;
                if (Q[A * nshell + B] * Q[C * nshell + Dd_] < tau) continue;
                ++kept;
                double s = 1.0;
                if (A == B) s *= 0.5;
                if (C == Dd_) s *= 0.5;
                if (ab == cd) s *= 0.5;
                eri_shell(&bs, A, B, C, Dd_, buf);
                int na = ncart(l[A]), nb = ncart(l[B]), nc = ncart(l[C]), nd = ncart(l[Dd_]);
                for (int a = 0; a < na; ++a) for (int b = 0; b < nb; ++b)
                for (int c = 0; c < nc; ++c) for (int d = 0; d < nd; ++d) {
                    double I = s * buf[((a * nb + b) * nc + c) * nd + d];
                    long m = off[A] + a, n = off[B] + b, k = off[C] + c, r = off[Dd_] + d;
#define IX(i, j) (((i) * N + (j)) * nD)
                    const double *Dkr = Dd + IX(k, r), *Drk = Dd + IX(r, k), *Dmn = Dd + IX(m, n), *Dnm = Dd + IX(n, m);
                    const double *Dnr = Dd + IX(n, r), *Dmr = Dd + IX(m, r), *Dnk = Dd + IX(n, k), *Dmk = Dd + IX(m, k);
                    const double *Drn = Dd + IX(r, n), *Dkn = Dd + IX(k, n), *Drm = Dd + IX(r, m), *Dkm = Dd + IX(k, m);
                    double *Jmn = Jp + IX(m, n), *Jnm = Jp + IX(n, m), *Jkr = Jp + IX(k, r), *Jrk = Jp + IX(r, k);
                    double *Kmk = Kp + IX(m, k), *Knk = Kp + IX(n, k), *Kmr = Kp + IX(m, r), *Knr = Kp + IX(n, r);
                    double *Kkm = Kp + IX(k, m), *Krm = Kp + IX(r, m), *Kkn = Kp + IX(k, n), *Krn = Kp + IX(r, n);
                    for (int x = 0; x < nD; ++x) {
                        double jc = I * (Dkr[x] + Drk[x]), jb = I * (Dmn[x] + Dnm[x]);
                        Jmn[x] += jc; Jnm[x] += jc; Jkr[x] += jb; Jrk[x] += jb;
                        Kmk[x] += I * Dnr[x]; Knk[x] += I * Dmr[x]; Kmr[x] += I * Dnk[x]; Knr[x] += I * Dmk[x];
                        Kkm[x] += I * Drn[x]; Krm[x] += I * Dkn[x]; Kkn[x] += I * Drm[x]; Krn[x] += I * Dkm[x];
                    }
#undef IX
                }
            }
        }
        free(buf);
    }
    for (int d = 0; d < nD; ++d)
        for (long i = 0; i < N * N; ++i) {
            double sj = 0.0, sk = 0.0;
            for (int t = 0; t < nthr; ++t) { sj += Jt[sz * t + i * nD + d]; sk += Kt[sz * t + i * nD + d]; }
            J[(size_t)d * N * N + i] = sj; K[(size_t)d * N * N + i] = sk;
        }
    free(Jt); free(Kt); free(Dd); free(Q); free(off);
    return kept;
}

/* Sampled blocks straight from Eq. (17), for sizes where O6/O7 are too slow:
 * for each sampled ORDERED shell pair (X,Y), b = 0..nblk-1,
 *   J_XY[d] = sum_{C,D} (XY|CD) D_CD[d]   over all ordered (C,D) with Q_XY Q_CD >= tau
 *   K_XY[d] = sum_{C,D} (XC|YD) D_CD[d]   over all ordered (C,D) with Q_XC Q_YD >= tau
 * which is exactly the set of terms the folded loop keeps (its test is on the bra/ket pair bounds of the
 * canonical image, and Q is symmetric).  Output: for block b, Jb/Kb[blk_off[b] + (d*nx + x)*ny + y]. */
void orc_jk_blocks(BASIS_ARGS, double tau, int nD, const double *D, int nblk, const int *X, const int *Y,
                   const long long *blk_off, double *Jb, double *Kb, const double *Qin)
{
    basis_t bs = BASIS_INIT;
    int *off = (int *)malloc(sizeof(int) * (nshell + 1));
    ao_offsets(&bs, off);
    long N = off[nshell];
    double *Q = (double *)malloc(sizeof(double) * nshell * nshell);
    if (Qin) memcpy(Q, Qin, sizeof(double) * nshell * nshell);
    else orc_schwarz(natom, xyz, nshell, atom, l, nprim, prim_off, exps, coef, Q);
    for (int b = 0; b < nblk; ++b) {
        int Xs = X[b], Ys = Y[b], nx = ncart(l[Xs]), ny = ncart(l[Ys]);
        double *Jo = Jb + blk_off[b], *Ko = Kb + blk_off[b];
        for (long i = 0; i < (long)nD * nx * ny; ++i) Jo[i] = Ko[i] = 0.0;
#pragma omp parallel
        {
            double *buf = (double *)malloc(sizeof(double) * NQMAX);
            double *jl = (double *)calloc((size_t)nD * nx * ny, sizeof(double));
            double *kl = (double *)calloc((size_t)nD * nx * ny, sizeof(double));
#pragma omp for collapse(2) schedule(dynamic)
            for (int C = 0; C < nshell; ++C)
            for (int Dd_ = 0; Dd_ < nshell; ++Dd_) {
                int nc = ncart(l[C]), nd = ncart(l[Dd_]);
                if (Q[Xs * nshell + Ys] * Q[C * nshell + Dd_] >= tau) {
                    eri_shell(&bs, Xs, Ys, C, Dd_, buf);       /* (XY|CD) */
                    for (int x = 0; x < nx; ++x) for (int y = 0; y < ny; ++y)
                    for (int c = 0; c < nc; ++c) for (int d = 0; d < nd; ++d) {
                        double I = buf[((x * ny + y) * nc + c) * nd + d];
                        for (int k = 0; k < nD; ++k)
                            jl[(k * nx + x) * ny + y] += I * D[(size_t)k * N * N + (off[C] + c) * N + off[Dd_] + d];
                    }
                }
                if (Q[Xs * nshell + C] * Q[Ys * nshell + Dd_] >= tau) {
                    eri_shell(&bs, Xs, C, Ys, Dd_, buf);       /* (XC|YD) */
                    for (int x = 0; x < nx; ++x) for (int c = 0; c < nc; ++c)
                    for (int y = 0; y < ny; ++y) for (int d = 0; d < nd; ++d) {
                        double I = buf[((x * nc + c) * ny + y) * nd + d];
                        for (int k = 0; k < nD; ++k)
                            kl[(k * nx + x) * ny + y] += I * D[(size_t)k * N * N + (off[C] + c) * N + off[Dd_] + d];
                    }
                }
            }
#pragma omp critical
            for (long i = 0; i < (long)nD * nx * ny; ++i) { Jo[i] += jl[i]; Ko[i] += kl[i]; }
            free(buf); free(jl); free(kl);
        }
    }
    free(Q); free(off);
}

/* SURVEY 8(f) N2.  Derivative (skeleton) builds, Eq. (18), with the nuclear derivative written out by the
 * product rule, one term per function of the integral (Eqs. (30)-(31): the centre derivatives):
 *   J^x(A,B) = sum_{mnkr} (mn|kr)^x A_mn B_kr ,   K^x(A,B) = sum_{mnkr} (mk|nr)^x A_mn B_kr ,
 *   (mn|kr)^x = (d_x m n|kr) + (m d_x n|kr) + (mn|d_x k r) + (mn|k d_x r) ,  d_x = derivative with respect to coordinate
 *   x of the atom that carries the function (zero for the other atoms).
 * A Cartesian Gaussian differentiates into one function of l+1 and one of l-1 on the same centre, primitive by primitive:
 *   d/dA_x [ x_A^i y_A^j z_A^k sum_p c_p e^{-a_p r_A^2} ] = x_A^{i+1} y_A^j z_A^k sum_p (2 a_p c_p) e^{-a_p r_A^2}
 *                                                          - i x_A^{i-1} y_A^j z_A^k sum_p c_p e^{-a_p r_A^2} ,
 * so every term is an ordinary integral (O5) over an auxiliary shell list: shell s raised (l+1, coefficients 2 a_p c_p)
 * and shell s lowered (l-1, coefficients c_p).  Every ORDERED shell quartet and every position is evaluated on its
 * own; no permutational symmetry, no screening, no prefactors.
 * A, B: [nP][N][N] row-major (general, non-symmetric).  gJ, gK: [nP][natom][3], overwritten. */
static int cart_index(int l, int i, int j, int k)
{
    int c[NCMAX][3];
    cart_list(l, c);
    for (int n = 0; n < ncart(l); ++n) if (c[n][0] == i && c[n][1] == j && c[n][2] == k) return n;
    return -1;
}

void orc_jk_grad(BASIS_ARGS, int nP, const double *A, const double *B, double *gJ, double *gK)
{
    basis_t bs = BASIS_INIT;
    int ns = nshell, ntotp = 0;
    for (int s = 0; s < ns; ++s) if (prim_off[s] + nprim[s] > ntotp) ntotp = prim_off[s] + nprim[s];
    /* auxiliary shell list: [0,ns) the shells, [ns,2ns) raised, [2ns,3ns) lowered */
    int *xa = (int *)malloc(sizeof(int) * 3 * ns), *xl = (int *)malloc(sizeof(int) * 3 * ns);
    int *xn = (int *)malloc(sizeof(int) * 3 * ns), *xo = (int *)malloc(sizeof(int) * 3 * ns);
    double *xe = (double *)malloc(sizeof(double) * 3 * ntotp), *xc = (double *)malloc(sizeof(double) * 3 * ntotp);
    for (int v = 0; v < 3; ++v) {
        for (int i = 0; i < ntotp; ++i) {
            xe[v * ntotp + i] = exps[i];
            xc[v * ntotp + i] = (v == 1) ? 2.0 * exps[i] * coef[i] : coef[i];
        }
        for (int s = 0; s < ns; ++s) {
            xa[v * ns + s] = atom[s]; xn[v * ns + s] = nprim[s]; xo[v * ns + s] = v * ntotp + prim_off[s];
            xl[v * ns + s] = (v == 0) ? l[s] : (v == 1) ? l[s] + 1 : (l[s] > 0 ? l[s] - 1 : 0);
        }
    }
    basis_t aux = { natom, xyz, 3 * ns, xa, xl, xn, xo, xe, xc };
    int *off = (int *)malloc(sizeof(int) * (ns + 1));
    ao_offsets(&bs, off);
    long N = off[ns];
    long ng = (long)nP * natom * 3;
    for (long i = 0; i < ng; ++i) gJ[i] = gK[i] = 0.0;
#pragma omp parallel
    {
        double *up = (double *)malloc(sizeof(double) * NCMAX * 216), *dn = (double *)malloc(sizeof(double) * NCMAX * 216);
        double *lj = (double *)calloc((size_t)ng, sizeof(double)), *lk = (double *)calloc((size_t)ng, sizeof(double));
#pragma omp for collapse(2) schedule(dynamic)
        for (int M = 0; M < ns; ++M)
        for (int Nn = 0; Nn < ns; ++Nn)
            for (int K = 0; K < ns; ++K)
            for (int R = 0; R < ns; ++R) {
                const int sh[4] = { M, Nn, K, R };
                int nc[4], cl[4][NCMAX][3];
                for (int q = 0; q < 4; ++q) { nc[q] = ncart(l[sh[q]]); cart_list(l[sh[q]], cl[q]); }
                for (int pos = 0; pos < 4; ++pos) {
                    const int S = sh[pos], ls = l[S], at = atom[S];
                    int su[4] = { M, Nn, K, R }, sd[4] = { M, Nn, K, R };
                    su[pos] = ns + S; sd[pos] = 2 * ns + S;
                    int nu[4] = { nc[0], nc[1], nc[2], nc[3] }, nd[4] = { nc[0], nc[1], nc[2], nc[3] };
                    nu[pos] = ncart(ls + 1); nd[pos] = ls > 0 ? ncart(ls - 1) : 1;
                    eri_shell(&aux, su[0], su[1], su[2], su[3], up);
                    if (ls > 0) eri_shell(&aux, sd[0], sd[1], sd[2], sd[3], dn);
                    int c[4];
                    for (c[0] = 0; c[0] < nc[0]; ++c[0]) for (c[1] = 0; c[1] < nc[1]; ++c[1])
                    for (c[2] = 0; c[2] < nc[2]; ++c[2]) for (c[3] = 0; c[3] < nc[3]; ++c[3]) {
                        const long m = off[M] + c[0], n = off[Nn] + c[1], k = off[K] + c[2], r = off[R] + c[3];
                        for (int x = 0; x < 3; ++x) {
                            int e[3] = { cl[pos][c[pos]][0], cl[pos][c[pos]][1], cl[pos][c[pos]][2] };
                            int cu[4] = { c[0], c[1], c[2], c[3] }, cd_[4] = { c[0], c[1], c[2], c[3] };
                            e[x] += 1; cu[pos] = cart_index(ls + 1, e[0], e[1], e[2]); e[x] -= 1;
                            double dI = up[((cu[0] * nu[1] + cu[1]) * nu[2] + cu[2]) * nu[3] + cu[3]];
                            if (e[x] > 0) {
                                const int pw = e[x];
                                e[x] -= 1; cd_[pos] = cart_index(ls - 1, e[0], e[1], e[2]); e[x] += 1;
                                dI -= pw * dn[((cd_[0] * nd[1] + cd_[1]) * nd[2] + cd_[2]) * nd[3] + cd_[3]];
                            }
                            for (int p = 0; p < nP; ++p) {
                                const double *Ap = A + (size_t)p * N * N, *Bp = B + (size_t)p * N * N;
                                lj[((long)p * natom + at) * 3 + x] += dI * Ap[m * N + n] * Bp[k * N + r];   /* (mn|kr)^x A_mn B_kr */
                                lk[((long)p * natom + at) * 3 + x] += dI * Ap[m * N + k] * Bp[n * N + r];   /* (mn|kr)^x A_mk B_nr */
                            }
                        }
                    }
                }
            }
#pragma omp critical
        for (long i = 0; i < ng; ++i) { gJ[i] += lj[i]; gK[i] += lk[i]; }
        free(up); free(dn); free(lj); free(lk);
    }
    free(xa); free(xl); free(xn); free(xo); free(xe); free(xc); free(off);
}

int orc_max_threads(void) { return omp_get_max_threads(); }

// eri_core.h -- per-thread shell-quartet evaluation (steps a6, a7): Boys function + generated OS/HGP recurrences.
//
// One thread evaluates one contracted Cartesian shell quartet (AB|CD), la>=lb, lc>=ld (the paper's mapping,
// PAPER.md:L318 "one thread = one contracted quartet"; Fig. 6).  The functions are __host__ __device__ so
// that a test-only host build (host_check.cpp) can exercise the generated recurrences without a GPU; the
// product library only ever calls them from kernels.
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define LTJK_HD __host__ __device__ __forceinline__
#else
#define LTJK_HD inline
#endif

#include "gen/eri_gen.h"
#ifdef LTJK_WITH_D1
#include "gen/eri_gen_d1.h"     // f-raised classes, only for ltjk_grad.cu
#endif

namespace ltjk {

constexpr int kMaxPrimPair = 16;      // up to 4 primitives per shell
constexpr int kPrimStride = 8;        // doubles per primitive pair: p, Px,Py,Pz, PAx,PAy,PAz, Kab
constexpr int kPairHeader = 4;        // ABx, ABy, ABz, npp (as double)
constexpr int kPairStride = kPairHeader + kMaxPrimPair * kPrimStride;   // doubles per shell pair record

// Boys table: F_m(T_i), T_i = i/8, i = 0..288 (T <= 36), m = 0..20
constexpr int kBoysNT = 289;
constexpr int kBoysNM = 21;          // orders 0..20: L <= 12 ((ff|ff), ltjk_eri_loop.cu) plus 8 Taylor terms
constexpr double kBoysTmax = 36.0;
constexpr int kBoysTaylor = 9;        // terms k = 0..8: remainder (1/16)^9/9! ~ 4e-17

LTJK_HD constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }

// Step a6.  F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt for m = 0..L, all multiplied by `scale`.
//   T < 36 : Taylor expansion about the nearest grid point T0 of the highest order,
//            F_L(T0+d) = sum_k F_{L+k}(T0) (-d)^k / k!, then downward recursion
//            F_{m-1} = (2T F_m + e^{-T}) / (2m-1)      (stable: every term positive)
//   T >= 36: F_0 = (1/2) sqrt(pi/T) (erf(6) = 1 - 2e-17), upward F_{m+1} = ((2m+1) F_m - e^{-T}) / (2T).
template <int L>
LTJK_HD void boys_scaled(const double T, const double scale, const double* __restrict__ tab, double* __restrict__ F)
{
    if (T < kBoysTmax) {
        const int i = (int)(T * 8.0 + 0.5);
        const double d = (double)i * 0.125 - T;          // -(T - T0)
        const double* t = tab + i * kBoysNM + L;
        double s = t[kBoysTaylor - 1];
#pragma unroll
        for (int k = kBoysTaylor - 2; k >= 0; --k) s = t[k] + s * d * (1.0 / (double)(k + 1));
        if (L == 0) {
            F[0] = s * scale;
        } else {
            const double e = exp(-T);
            double f = s;
            F[L] = f * scale;
#pragma unroll
            for (int m = L; m >= 1; --m) {
                f = (2.0 * T * f + e) * (1.0 / (double)(2 * m - 1));
                F[m - 1] = f * scale;
            }
        }
    } else {
        const double r = 1.0 / T;
        double f = 0.5 * sqrt(3.14159265358979323846 * r);
        F[0] = f * scale;
        if (L > 0) {
            const double e = exp(-T);
            const double h = 0.5 * r;
#pragma unroll
            for (int m = 0; m < L; ++m) {
                f = ((double)(2 * m + 1) * f - e) * h;
                F[m + 1] = f * scale;
            }
        }
    }
}

// Shell-pair record builder (step a2, Gaussian-product part): for shells A (la >= lb) and B,
//   p = a+b, P = (aA + bB)/p, PA = P - A, K_ab = c_a c_b exp(-(ab/p) |A-B|^2)
LTJK_HD void build_pair_record(const double* A, const double* B, int na, const double* ea, const double* ca,
                               int nb, const double* eb, const double* cb, double* rec)
{
    const double ABx = A[0] - B[0], ABy = A[1] - B[1], ABz = A[2] - B[2];
    const double r2 = ABx * ABx + ABy * ABy + ABz * ABz;
    rec[0] = ABx; rec[1] = ABy; rec[2] = ABz; rec[3] = (double)(na * nb);
    int k = 0;
    for (int i = 0; i < na; ++i)
        for (int j = 0; j < nb; ++j, ++k) {
            const double a = ea[i], b = eb[j], p = a + b, ip = 1.0 / p;
            double* q = rec + kPairHeader + k * kPrimStride;
            const double Px = (a * A[0] + b * B[0]) * ip, Py = (a * A[1] + b * B[1]) * ip, Pz = (a * A[2] + b * B[2]) * ip;
            q[0] = p; q[1] = Px; q[2] = Py; q[3] = Pz;
            q[4] = Px - A[0]; q[5] = Py - A[1]; q[6] = Pz - A[2];
            q[7] = ca[i] * cb[j] * exp(-a * b * ip * r2);
        }
}

// Primitive quartets whose prefactor K_ab K_cd 2 pi^{5/2}/(pq sqrt(p+q)) is below this are skipped: every
// [e0|f0] of the quartet is bounded by a modest multiple of it, far below the 1e-10 parity bar.
constexpr double kPrimCut = 1e-20;

// Step a7.  Contracted quartet (ab|cd) -> out[((a*nb+b)*nc+c)*nd+d].
template <int LA, int LB, int LC, int LD, bool CUT = true>
LTJK_HD void eri_quartet(const double* __restrict__ bra, const double* __restrict__ ket,
                         const double* __restrict__ boys_tab, double* __restrict__ out)
{
    using V = ltjk_gen::Vrr<LA, LB, LC, LD>;
    using HB = ltjk_gen::Hrr<LA, LB>;
    using HK = ltjk_gen::Hrr<LC, LD>;
    constexpr int L = LA + LB + LC + LD;
    constexpr int NE = V::NE, NF = V::NF;
    constexpr int NAB = HB::NAB, NCD = HK::NAB;
    double acc[NE * NF];
#pragma unroll
    for (int i = 0; i < NE * NF; ++i) acc[i] = 0.0;

    const int nb = (int)bra[3], nk = (int)ket[3];
    for (int ib = 0; ib < nb; ++ib) {
        const double* b = bra + kPairHeader + ib * kPrimStride;
        const double p = b[0], Px = b[1], Py = b[2], Pz = b[3], Kab = b[7];
        const double oo2p = 0.5 / p;
        for (int ik = 0; ik < nk; ++ik) {
            const double* k = ket + kPairHeader + ik * kPrimStride;
            const double q = k[0], Kcd = k[7];
            const double pq = p + q, ipq = 1.0 / pq;
            const double pref = Kab * Kcd * 34.986836655249725693 /* 2 pi^{5/2} */ / (p * q * sqrt(pq));
            if (CUT && fabs(pref) < kPrimCut) continue;   // never for the Schwarz diagonal (Q^2 may be < 1e-20)
            const double PQx = Px - k[1], PQy = Py - k[2], PQz = Pz - k[3];
            const double rho = p * q * ipq;
            const double T = rho * (PQx * PQx + PQy * PQy + PQz * PQz);
            double F[L + 1];
            boys_scaled<L>(T, pref, boys_tab, F);
            const double wp = -q * ipq, wq = p * ipq;
            V::run(F, b[4], b[5], b[6], wp * PQx, wp * PQy, wp * PQz, k[4], k[5], k[6], wq * PQx, wq * PQy, wq * PQz,
                   oo2p, 0.5 / q, 0.5 * ipq, q * ipq /* rho/p */, p * ipq /* rho/q */, acc);
        }
    }
    // HRR on the bra for every ket component, then on the ket for every (a,b)
    if (LB == 0 && LD == 0) {
#pragma unroll
        for (int i = 0; i < NE * NF; ++i) out[i] = acc[i];
        return;
    }
    if (LB == 0) {
#pragma unroll
        for (int iab = 0; iab < NAB; ++iab) HK::run(acc + iab * NF, 1, out + iab * NCD, 1, ket[0], ket[1], ket[2]);
        return;
    }
    if (LD == 0) {
#pragma unroll
        for (int jf = 0; jf < NF; ++jf) HB::run(acc + jf, NF, out + jf, NF, bra[0], bra[1], bra[2]);
        return;
    }
    if (LB > 0 && LD > 0) {
        double t1[NAB * NF];
        for (int jf = 0; jf < NF; ++jf) HB::run(acc + jf, NF, t1 + jf, NF, bra[0], bra[1], bra[2]);
        for (int iab = 0; iab < NAB; ++iab) HK::run(t1 + iab * NF, 1, out + iab * NCD, 1, ket[0], ket[1], ket[2]);
    }
}

}  // namespace ltjk

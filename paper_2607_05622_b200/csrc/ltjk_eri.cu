// ltjk_eri.cu -- steps a2 (shell-pair records, Schwarz bounds), a6+a7 (Boys + OS/HGP shell quartets) as kernels.
//
// Integral panels.  A canonical block quartet (IJ|KL) (blocks = l-homogeneous groups of 16-24 AOs, see
// ltjk_internal.h) owns a dense panel  P[i][j][k][l] = s * (ij|kl),  i in I, j in J, k in K, l in L,
// s = 1/2 per coincidence I==J, K==L, (IJ)==(KL)  (the "canonical-fold multiplicity" of PAPER.md:L320-322 Eq. 25,
// DESIGN.md reading A4, applied at block level).  Panels live in a two-half staging ring, are written here by one
// thread per contracted shell quartet (the paper's mapping; a half-warp for the heaviest classes) and consumed by the
// digestion kernels (ltjk_digest.cu) before the ring is reused: integrals never form a stored N^4 object.
// Shell quartets with Q_AB Q_CD < tau (reading A9) are written as zeros.
#define LTJK_WITH_D1                 // the f-raised generated classes: used here for the six light (f l_b|l_c l_d) classes
#include "ltjk_internal.h"
#include "eri_core.h"
#include "boys_table.h"

namespace ltjk {

// ---------------------------------------------------------------------------------------------------------------
// a2: one thread per ordered internal shell pair (A,B) with l_A >= l_B: Gaussian-product record.
__global__ void pair_record_kernel(int nshell, const double* __restrict__ xyz, const int* __restrict__ atom,
                                   const int* __restrict__ l, const int* __restrict__ nprim,
                                   const int* __restrict__ poff, const double* __restrict__ exps,
                                   const double* __restrict__ coef, const int* __restrict__ int2ext,
                                   int rec_stride, double* __restrict__ rec)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nshell * nshell) return;
    const int A = t / nshell, B = t % nshell;
    const int a = int2ext[A], b = int2ext[B];
    if (l[a] < l[b]) return;
    build_pair_record(xyz + 3 * atom[a], xyz + 3 * atom[b], nprim[a], exps + poff[a], coef + poff[a], nprim[b],
                      exps + poff[b], coef + poff[b], rec + (size_t)t * rec_stride);
}

int launch_pair_records(ltjk_ctx* c, const double* d_xyz, const int* d_atom, const int* d_l, const int* d_nprim,
                        const int* d_poff, const double* d_exps, const double* d_coef, const int* d_int2ext)
{
    const int n = c->nshell * c->nshell;
    pair_record_kernel<<<(n + 127) / 128, 128, 0, c->stream>>>(c->nshell, d_xyz, d_atom, d_l, d_nprim, d_poff, d_exps,
                                                              d_coef, d_int2ext, c->t.rec_stride, c->t.pair_rec);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// a2: Schwarz bounds Q_AB = sqrt(max_{a,b} |(ab|ab)|), one thread per shell pair of class (LA,LB).
template <int LA, int LB>
__global__ void schwarz_kernel(int nshell, int a0, int na, int b0, int nb, const double* __restrict__ rec,
                               int rec_stride, const double* __restrict__ boys, double* __restrict__ Q)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= na * nb) return;
    const int A = a0 + t / nb, B = b0 + t % nb;
    if (LA == LB && B > A) return;
    constexpr int NA = ncart(LA), NB = ncart(LB);
    double out[NA * NB * NA * NB];
    const double* r = rec + ((size_t)A * nshell + B) * rec_stride;
    eri_quartet<LA, LB, LA, LB, false>(r, r, boys, out);
    double m = 0.0;
#pragma unroll
    for (int i = 0; i < NA * NB; ++i) m = fmax(m, fabs(out[i * NA * NB + i]));
    m = sqrt(m);
    Q[(size_t)A * nshell + B] = m;
    Q[(size_t)B * nshell + A] = m;
}

int launch_schwarz(ltjk_ctx* c, const int* lrange /* host: first internal shell of l = 0,1,2,3 and end */)
{
    const int ns = c->nshell;
#define SCHW(LA, LB)                                                                                              \
    {                                                                                                             \
        const int a0 = lrange[LA], na = lrange[LA + 1] - lrange[LA], b0 = lrange[LB], nb = lrange[LB + 1] - lrange[LB]; \
        if (na > 0 && nb > 0) {                                                                                   \
            schwarz_kernel<LA, LB><<<(na * nb + 63) / 64, 64, 0, c->stream>>>(ns, a0, na, b0, nb, c->t.pair_rec,  \
                                                                              c->t.rec_stride, c->t.boys, c->t.schwarz); \
            LTJK_CUDA(c, cudaGetLastError());                                                                     \
        }                                                                                                         \
    }
    SCHW(0, 0) SCHW(1, 0) SCHW(1, 1) SCHW(2, 0) SCHW(2, 1) SCHW(2, 2)
#undef SCHW
    for (int lb = 0; lb <= 3; ++lb) {                      // pair classes with an f shell: looped kernel
        const int rc = launch_schwarz_loop(c, 3, lb, lrange[3], lrange[4] - lrange[3], lrange[lb], lrange[lb + 1] - lrange[lb]);
        if (rc) return rc;
    }
    return LTJK_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// a6 + a7: panels of one class segment.  Thread -> (ket rank r in [ra,rb), shell quartet inside the block quartet).
template <int LA, int LB, int LC, int LD>
// (64,4): without a min-blocks hint ptxas drops the heavy classes to 32 registers and spills ~80 KB per thread
__global__ void __launch_bounds__(64, 4) eri_panel_kernel(const EriArgs g)
{
    const SubChunk sc_ = g.subs[blockIdx.y];
    const int ra = max(sc_.r0, g.ca), rb = min(sc_.r1, g.cb_);
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = ra + (int)(t / g.qn);
    if (r >= rb) return;
    int q = (int)(t % g.qn);
    const int sd = q % g.mL; q /= g.mL;
    const int sc = q % g.mK; q /= g.mK;
    const int sb = q % g.mJ;
    const int sa = q / g.mJ;
    const DevTables& T = g.t;
    const int I = sc_.I, J = sc_.J, K = T.pair_I[r], L = T.pair_J[r];
    if (sa >= T.blk_nsh[I] || sb >= T.blk_nsh[J] || sc >= T.blk_nsh[K] || sd >= T.blk_nsh[L]) return;
    const int A = T.blk_sh0[I] + sa, B = T.blk_sh0[J] + sb, C = T.blk_sh0[K] + sc, D = T.blk_sh0[L] + sd;
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    const int nJ = T.blk_nao[J], nK = T.blk_nao[K], nL = T.blk_nao[L];
    const long long base = sc_.base + (T.koff[r] - T.koff[sc_.r0]) * (long long)(T.blk_nao[I] * nJ);
    double* __restrict__ P = g.panel + base + ((long long)(sa * NA) * nJ + sb * NB) * (nK * nL) + (sc * NC) * nL + sd * ND;
    const int sI = nJ * nK * nL, sJ = nK * nL, sK = nL;

    const double qq = T.schwarz[(size_t)A * T.nshell + B] * T.schwarz[(size_t)C * T.nshell + D];
    if (qq < g.tau) {
        for (int a = 0; a < NA; ++a)
            for (int b = 0; b < NB; ++b)
                for (int cc = 0; cc < NC; ++cc)
#pragma unroll
                    for (int d = 0; d < ND; ++d) P[a * sI + b * sJ + cc * sK + d] = 0.0;
        return;
    }
    double scale = 1.0;
    if (I == J) scale *= 0.5;
    if (K == L) scale *= 0.5;
    if (r == sc_.rIJ) scale *= 0.5;
    double out[NA * NB * NC * ND];
    eri_quartet<LA, LB, LC, LD>(T.pair_rec + ((size_t)A * T.nshell + B) * T.rec_stride,
                                T.pair_rec + ((size_t)C * T.nshell + D) * T.rec_stride, T.boys, out);
    for (int a = 0; a < NA; ++a)
        for (int b = 0; b < NB; ++b)
            for (int cc = 0; cc < NC; ++cc)
#pragma unroll
                for (int d = 0; d < ND; ++d)
                    P[a * sI + b * sJ + cc * sK + d] = scale * out[((a * NB + b) * NC + cc) * ND + d];
}

// ---------------------------------------------------------------------------------------------------------------
// a6 + a7, cooperative variant for the classes whose contracted VRR targets do not fit a thread (l_b, l_d > 0 and
// NE*NF >= 128: (dp|pp), (dp|dp), (dd|pp), (dd|dp), (dd|dd)).  The one-thread-per-quartet kernel keeps those targets, the HRR scratch and
// its spills in ~15-34 KB of local memory per thread and is bound by DRAM traffic (profiles/r1_eri_classes_ncu.txt).
// Here a half-warp owns one contracted quartet: lane p evaluates primitive quartet p (Boys + VRR), the 16 partial
// values of every target are summed by a reduce-scatter over the half-warp (15 shuffle-adds per 16 targets) into a
// shared-memory [e0|f0] block, and both HRR stages run from shared memory with the columns / rows dealt to the lanes.
template <int NTOT>
struct CoopSink {
    double buf[16];
    double* __restrict__ accS;
    unsigned hmask;
    int l16;
    bool first;
    template <int I>
    __device__ __forceinline__ void put(const double v)
    {
        buf[I & 15] = v;
        if ((I & 15) == 15 || I == NTOT - 1) flush<(I >> 4), (I & 15) + 1>();
    }
    template <int G, int N>
    __device__ __forceinline__ void flush()
    {
#pragma unroll
        for (int i = N; i < 16; ++i) buf[i] = 0.0;
        const bool b3 = l16 & 8, b2 = l16 & 4, b1 = l16 & 2, b0 = l16 & 1;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const double keep = b3 ? buf[i + 8] : buf[i], send = b3 ? buf[i] : buf[i + 8];
            buf[i] = keep + __shfl_xor_sync(hmask, send, 8);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double keep = b2 ? buf[i + 4] : buf[i], send = b2 ? buf[i] : buf[i + 4];
            buf[i] = keep + __shfl_xor_sync(hmask, send, 4);
        }
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const double keep = b1 ? buf[i + 2] : buf[i], send = b1 ? buf[i] : buf[i + 2];
            buf[i] = keep + __shfl_xor_sync(hmask, send, 2);
        }
        {
            const double keep = b0 ? buf[1] : buf[0], send = b0 ? buf[0] : buf[1];
            buf[0] = keep + __shfl_xor_sync(hmask, send, 1);
        }
        if (l16 < N) {                       // lane l16 now holds the contracted target G*16 + l16
            if (first) accS[G * 16 + l16] = buf[0];
            else accS[G * 16 + l16] += buf[0];
        }
    }
};

constexpr int kCoopThreads = 128;            // 8 half-warps = 8 quartets per CTA

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(kCoopThreads, 1) eri_panel_coop_kernel(const EriArgs g)
{
    using V = ltjk_gen::Vrr<LA, LB, LC, LD>;
    using HB = ltjk_gen::Hrr<LA, LB>;
    using HK = ltjk_gen::Hrr<LC, LD>;
    constexpr int L = LA + LB + LC + LD;
    constexpr int NE = V::NE, NF = V::NF, NAB = HB::NAB, NCD = HK::NAB;
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    constexpr int QS = NE * NF + NAB * NF;                  // doubles of shared memory per quartet
    extern __shared__ __align__(16) double coop_sm[];
    const int lane = threadIdx.x & 31, l16 = lane & 15, hw = threadIdx.x >> 4;
    const unsigned hmask = (lane & 16) ? 0xffff0000u : 0x0000ffffu;
    double* __restrict__ accS = coop_sm + hw * QS;
    double* __restrict__ t1S = accS + NE * NF;

    const SubChunk sc_ = g.subs[blockIdx.y];
    const int ra = max(sc_.r0, g.ca), rb = min(sc_.r1, g.cb_);
    const long long t = (long long)blockIdx.x * (kCoopThreads / 16) + hw;
    const int r = ra + (int)(t / g.qn);
    if (r >= rb) return;                                      // the whole half-warp leaves together
    int q = (int)(t % g.qn);
    const int sd = q % g.mL; q /= g.mL;
    const int sc = q % g.mK; q /= g.mK;
    const int sb = q % g.mJ;
    const int sa = q / g.mJ;
    const DevTables& T = g.t;
    const int I = sc_.I, J = sc_.J, K = T.pair_I[r], Lb = T.pair_J[r];
    if (sa >= T.blk_nsh[I] || sb >= T.blk_nsh[J] || sc >= T.blk_nsh[K] || sd >= T.blk_nsh[Lb]) return;
    const int A = T.blk_sh0[I] + sa, B = T.blk_sh0[J] + sb, C = T.blk_sh0[K] + sc, D = T.blk_sh0[Lb] + sd;
    const int nJ = T.blk_nao[J], nK = T.blk_nao[K], nL = T.blk_nao[Lb];
    const long long base = sc_.base + (T.koff[r] - T.koff[sc_.r0]) * (long long)(T.blk_nao[I] * nJ);
    double* __restrict__ P = g.panel + base + ((long long)(sa * NA) * nJ + sb * NB) * (nK * nL) + (sc * NC) * nL + sd * ND;
    const int sI = nJ * nK * nL, sJ = nK * nL, sK = nL;

    const double qq = T.schwarz[(size_t)A * T.nshell + B] * T.schwarz[(size_t)C * T.nshell + D];
    if (qq < g.tau) {
        for (int e = l16; e < NA * NB * NC * ND; e += 16) {
            const int d = e % ND, cc = (e / ND) % NC, b = (e / (ND * NC)) % NB, a = e / (ND * NC * NB);
            P[a * sI + b * sJ + cc * sK + d] = 0.0;
        }
        return;
    }
    double scale = 1.0;
    if (I == J) scale *= 0.5;
    if (K == Lb) scale *= 0.5;
    if (r == sc_.rIJ) scale *= 0.5;

    const double* __restrict__ bra = T.pair_rec + ((size_t)A * T.nshell + B) * T.rec_stride;
    const double* __restrict__ ket = T.pair_rec + ((size_t)C * T.nshell + D) * T.rec_stride;
    const int nb = (int)bra[3], nk = (int)ket[3], nprimq = nb * nk;
    for (int p0 = 0; p0 < nprimq; p0 += 16) {
        const int p = p0 + l16;
        const bool active = p < nprimq;
        const double* bp = bra + kPairHeader + (active ? p / nk : 0) * kPrimStride;
        const double* kp = ket + kPairHeader + (active ? p % nk : 0) * kPrimStride;
        const double pp = bp[0], qv = kp[0];
        const double pq = pp + qv, ipq = 1.0 / pq;
        double pref = bp[7] * kp[7] * 34.986836655249725693 /* 2 pi^{5/2} */ / (pp * qv * sqrt(pq));
        if (!active || fabs(pref) < kPrimCut) pref = 0.0;     // the VRR is linear in F: zero F = zero contribution
        const double PQx = bp[1] - kp[1], PQy = bp[2] - kp[2], PQz = bp[3] - kp[3];
        const double rho = pp * qv * ipq;
        double F[L + 1];
        boys_scaled<L>(rho * (PQx * PQx + PQy * PQy + PQz * PQz), pref, T.boys, F);
        const double wp = -qv * ipq, wq = pp * ipq;
        CoopSink<NE * NF> sink;
        sink.accS = accS; sink.hmask = hmask; sink.l16 = l16; sink.first = (p0 == 0);
        V::run_t(F, bp[4], bp[5], bp[6], wp * PQx, wp * PQy, wp * PQz, kp[4], kp[5], kp[6], wq * PQx, wq * PQy, wq * PQz,
                 0.5 / pp, 0.5 / qv, 0.5 * ipq, qv * ipq /* rho/p */, pp * ipq /* rho/q */, sink);
        __syncwarp(hmask);
    }
    // HRR on the bra for every ket component (columns dealt to the lanes), then on the ket for every (a,b) row
    for (int jf = l16; jf < NF; jf += 16) HB::run(accS + jf, NF, t1S + jf, NF, bra[0], bra[1], bra[2]);
    __syncwarp(hmask);
    for (int iab = l16; iab < NAB; iab += 16) {
        double o[NCD];
        HK::run(t1S + iab * NF, 1, o, 1, ket[0], ket[1], ket[2]);
        double* __restrict__ Pab = P + (iab / NB) * sI + (iab % NB) * sJ;
#pragma unroll
        for (int cc = 0; cc < NC; ++cc)
#pragma unroll
            for (int d = 0; d < ND; ++d) Pab[cc * sK + d] = scale * o[cc * ND + d];
    }
}

static constexpr int kClsLa[kNumPairCls] = {0, 1, 1, 2, 2, 2, 3, 3, 3, 3}, kClsLb[kNumPairCls] = {0, 0, 1, 0, 1, 2, 0, 1, 2, 3};

template <int CB, int CK>
static int launch_cls(ltjk_ctx* c, const EriArgs& g, int maxkets, int nsub)
{
    constexpr int la[6] = {0, 1, 1, 2, 2, 2}, lb[6] = {0, 0, 1, 0, 1, 2};
    if constexpr (CK <= CB) {
        using V = ltjk_gen::Vrr<la[CB], lb[CB], la[CK], lb[CK]>;
        // measured on B200: worth it from 128 targets up ((pp|pp) with 81 is faster one thread per quartet, and so
        // are the l_d = 0 classes)
        if constexpr (lb[CB] > 0 && lb[CK] > 0 && V::NE * V::NF >= 128) {
            constexpr int QS = V::NE * V::NF + ltjk_gen::Hrr<la[CB], lb[CB]>::NAB * V::NF;
            constexpr int smem = (kCoopThreads / 16) * QS * (int)sizeof(double);
            LTJK_CUDA(c, cudaFuncSetAttribute(eri_panel_coop_kernel<la[CB], lb[CB], la[CK], lb[CK]>,
                                              cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            const long long nq = (long long)maxkets * g.qn;
            const int per = kCoopThreads / 16;
            eri_panel_coop_kernel<la[CB], lb[CB], la[CK], lb[CK]>
                <<<dim3((unsigned)((nq + per - 1) / per), nsub), kCoopThreads, smem, c->eri_stream>>>(g);
            LTJK_CUDA(c, cudaGetLastError());
            return LTJK_OK;
        }
        const long long nthr = (long long)maxkets * g.qn;
        const int bs = 64;
        // no shared memory used: give the whole unified cache to L1 (local-memory spills)
        cudaFuncSetAttribute(eri_panel_kernel<la[CB], lb[CB], la[CK], lb[CK]>,
                             cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxL1);
        eri_panel_kernel<la[CB], lb[CB], la[CK], lb[CK]>
            <<<dim3((unsigned)((nthr + bs - 1) / bs), nsub), bs, 0, c->eri_stream>>>(g);
        LTJK_CUDA(c, cudaGetLastError());
        return LTJK_OK;
    } else {
        return set_err(c, LTJK_EINVAL, "internal: ket class above bra class");
    }
}

// Light classes with ONE f shell, (f l_b|l_c l_d) with at most 360 targets: the bulk of the quartets of a basis with few
// f shells.  gen_eri.py emits straight-line code for them (the f-raised set of the derivative builds), so they run one
// thread per quartet like the s/p/d classes; every class with an f shell that is neither here nor in the cooperative
// set below is looped (ltjk_eri_loop.cu).
//   bra (fs): every ket (ss) ... (dd);   bra (fp): ket (ss) (ps) (pp) (ds);   bra (fd): ket (ss) (ps) (ds)
inline bool f_class_unrolled(int cb, int ck)
{
    return (cb == 6 && ck <= 5) || (cb == 7 && ck <= 3) || (cb == 8 && (ck <= 1 || ck == 3));
}
#define LTJK_F_LIGHT(X) X(0, 0) X(0, 1) X(0, 2) X(0, 3) X(0, 4) X(0, 5) X(1, 0) X(1, 1) X(1, 2) X(1, 3) X(2, 0) X(2, 1) X(2, 3)
// Four heavier one-f classes with l_b, l_d > 0 -- (fp|dp), (fp|dd), (fd|pp), (fd|dp): 540-1080 targets -- go through the
// cooperative kernel (a half-warp per quartet, contracted targets in shared memory) like (dd|dd).
inline bool f_class_coop(int cb, int ck) { return (cb == 7 && (ck == 4 || ck == 5)) || (cb == 8 && (ck == 2 || ck == 4)); }
#define LTJK_F_COOP(X) X(1, 4) X(1, 5) X(2, 2) X(2, 4)

template <int LB, int CK>
static int launch_f_coop(ltjk_ctx* c, const EriArgs& g, int maxkets, int nsub)
{
    constexpr int lc[6] = {0, 1, 1, 2, 2, 2}, ld[6] = {0, 0, 1, 0, 1, 2};
    using V = ltjk_gen::Vrr<3, LB, lc[CK], ld[CK]>;
    constexpr int QS = V::NE * V::NF + ltjk_gen::Hrr<3, LB>::NAB * V::NF;
    constexpr int smem = (kCoopThreads / 16) * QS * (int)sizeof(double);
    static_assert(smem <= 227 * 1024, "cooperative ERI kernel: shared memory");
    LTJK_CUDA(c, cudaFuncSetAttribute(eri_panel_coop_kernel<3, LB, lc[CK], ld[CK]>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    const long long nq = (long long)maxkets * g.qn;
    const int per = kCoopThreads / 16;
    eri_panel_coop_kernel<3, LB, lc[CK], ld[CK]>
        <<<dim3((unsigned)((nq + per - 1) / per), nsub), kCoopThreads, smem, c->eri_stream>>>(g);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

template <int LB, int CK>
static int launch_f_light(ltjk_ctx* c, const EriArgs& g, int maxkets, int nsub)
{
    constexpr int lc[6] = {0, 1, 1, 2, 2, 2}, ld[6] = {0, 0, 1, 0, 1, 2};
    const long long nthr = (long long)maxkets * g.qn;
    const int bs = 64;
    cudaFuncSetAttribute(eri_panel_kernel<3, LB, lc[CK], ld[CK]>, cudaFuncAttributePreferredSharedMemoryCarveout,
                         cudaSharedmemCarveoutMaxL1);
    eri_panel_kernel<3, LB, lc[CK], ld[CK]><<<dim3((unsigned)((nthr + bs - 1) / bs), nsub), bs, 0, c->eri_stream>>>(g);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

template <int CB>
static int launch_cls_k(ltjk_ctx* c, int ck, const EriArgs& g, int mk, int ns)
{
    switch (ck) {
    case 0: return launch_cls<CB, 0>(c, g, mk, ns);
    case 1: return launch_cls<CB, 1>(c, g, mk, ns);
    case 2: return launch_cls<CB, 2>(c, g, mk, ns);
    case 3: return launch_cls<CB, 3>(c, g, mk, ns);
    case 4: return launch_cls<CB, 4>(c, g, mk, ns);
    default: return launch_cls<CB, 5>(c, g, mk, ns);
    }
}

int launch_eri_panels(ltjk_ctx* c, const Group& gr, int ck)
{
    if (gr.maxkets[ck] == 0) return LTJK_OK;
    const int cb = gr.cb;
    EriArgs g;
    g.t = c->t;
    g.subs = c->d_subs + gr.sub0;
    g.ca = c->cls_start[ck]; g.cb_ = c->cls_start[ck + 1];
    const int mI = c->max_nsh_l[kClsLa[cb]];
    g.mJ = c->max_nsh_l[kClsLb[cb]]; g.mK = c->max_nsh_l[kClsLa[ck]]; g.mL = c->max_nsh_l[kClsLb[ck]];
    g.qn = mI * g.mJ * g.mK * g.mL;
    g.tau = c->tau;
    g.panel = c->d_panel + (size_t)gr.buf * c->panel_half;
    c->st_launches++;
    const int mk = gr.maxkets[ck], ns = gr.nsub;
    if (f_class_unrolled(cb, ck)) {
        switch ((cb - 6) * 6 + ck) {
#define X(LB, CK) case LB * 6 + CK: return launch_f_light<LB, CK>(c, g, mk, ns);
            LTJK_F_LIGHT(X)
#undef X
        }
    }
    if (f_class_coop(cb, ck)) {
        switch ((cb - 6) * 6 + ck) {
#define X(LB, CK) case LB * 6 + CK: return launch_f_coop<LB, CK>(c, g, mk, ns);
            LTJK_F_COOP(X)
#undef X
        }
    }
    if (cb >= 6)                                            // any other class with an f shell (ck <= cb): looped kernel
        return launch_eri_panels_loop(c, g, kClsLa[cb], kClsLb[cb], kClsLa[ck], kClsLb[ck], mk, ns);
    switch (cb) {
    case 0: return launch_cls_k<0>(c, ck, g, mk, ns);
    case 1: return launch_cls_k<1>(c, ck, g, mk, ns);
    case 2: return launch_cls_k<2>(c, ck, g, mk, ns);
    case 3: return launch_cls_k<3>(c, ck, g, mk, ns);
    case 4: return launch_cls_k<4>(c, ck, g, mk, ns);
    default: return launch_cls_k<5>(c, ck, g, mk, ns);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Test hooks.
template <int LA, int LB, int LC, int LD>
__global__ void eri_single_kernel(const double* bra, const double* ket, const double* boys, double* out)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double o[ncart(LA) * ncart(LB) * ncart(LC) * ncart(LD)];
        eri_quartet<LA, LB, LC, LD>(bra, ket, boys, o);
        for (int i = 0; i < ncart(LA) * ncart(LB) * ncart(LC) * ncart(LD); ++i) out[i] = o[i];
    }
}

template <int CB, int CK>
static void single_cls(ltjk_ctx* c, const double* bra, const double* ket, double* out)
{
    constexpr int la[6] = {0, 1, 1, 2, 2, 2}, lb[6] = {0, 0, 1, 0, 1, 2};
    if constexpr (CK <= CB)
        eri_single_kernel<la[CB], lb[CB], la[CK], lb[CK]><<<1, 32, 0, c->stream>>>(bra, ket, c->t.boys, out);
}

template <int CB>
static void single_cls_k(ltjk_ctx* c, int ck, const double* bra, const double* ket, double* out)
{
    switch (ck) {
    case 0: single_cls<CB, 0>(c, bra, ket, out); break;
    case 1: single_cls<CB, 1>(c, bra, ket, out); break;
    case 2: single_cls<CB, 2>(c, bra, ket, out); break;
    case 3: single_cls<CB, 3>(c, bra, ket, out); break;
    case 4: single_cls<CB, 4>(c, bra, ket, out); break;
    default: single_cls<CB, 5>(c, bra, ket, out); break;
    }
}

// (AB|CD) for INTERNAL shell indices with l_A>=l_B, l_C>=l_D and class(AB) >= class(CD); d_out row-major a,b,c,d.
int launch_eri_single(ltjk_ctx* c, int A, int B, int C, int D, int la, int lb, int lc, int ld, double* d_out, bool looped)
{
    const int cb = la * (la + 1) / 2 + lb, ck = lc * (lc + 1) / 2 + ld;
    const double* bra = c->t.pair_rec + ((size_t)A * c->nshell + B) * c->t.rec_stride;
    const double* ket = c->t.pair_rec + ((size_t)C * c->nshell + D) * c->t.rec_stride;
    if (f_class_unrolled(cb, ck) && !looped) {
        switch ((cb - 6) * 6 + ck) {
#define X(LB, CK) case LB * 6 + CK: eri_single_kernel<3, LB, kClsLa[CK], kClsLb[CK]><<<1, 32, 0, c->stream>>>(bra, ket, c->t.boys, d_out); break;
            LTJK_F_LIGHT(X)
#undef X
        }
        LTJK_CUDA(c, cudaGetLastError());
        return LTJK_OK;
    }
    if (cb >= 6 || looped) return launch_eri_single_loop(c, bra, ket, la, lb, lc, ld, d_out);
    switch (cb) {
    case 0: single_cls_k<0>(c, ck, bra, ket, d_out); break;
    case 1: single_cls_k<1>(c, ck, bra, ket, d_out); break;
    case 2: single_cls_k<2>(c, ck, bra, ket, d_out); break;
    case 3: single_cls_k<3>(c, ck, bra, ket, d_out); break;
    case 4: single_cls_k<4>(c, ck, bra, ket, d_out); break;
    default: single_cls_k<5>(c, ck, bra, ket, d_out); break;
    }
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

template <int M>
__global__ void boys_debug_kernel(int n, const double* T, const double* tab, double* F)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double f[M + 1];
    boys_scaled<M>(T[i], 1.0, tab, f);
    for (int m = 0; m <= M; ++m) F[(size_t)i * (M + 1) + m] = f[m];
}

int launch_boys_debug(ltjk_ctx* c, int mmax, int n, const double* d_T, double* d_F)
{
    const int g = (n + 127) / 128;
    switch (mmax) {
#define BD(M) case M: boys_debug_kernel<M><<<g, 128, 0, c->stream>>>(n, d_T, c->t.boys, d_F); break;
        BD(0) BD(1) BD(2) BD(3) BD(4) BD(5) BD(6) BD(7) BD(8)
#undef BD
    default: return set_err(c, LTJK_EINVAL, "mmax must be 0..8");
    }
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

}  // namespace ltjk

// ltjk_peri.cu -- steps a6 + a7 for the pair-list digestion: Boys + OS/HGP shell quartets (same generated
// recurrences as ltjk_eri.cu), written to the role-assignment blocks of ltjk_pair.cu.
//
// One launch = (Q-sorted bra shell-pair list of one class) x (Q-sorted ket list of one class) of one chunk; thread
// (bra b, ket k) evaluates the unique quartet (AB|CD) when Q_AB Q_CD >= tau (reading A9) and
// returns at once otherwise ("only the realised buckets are launched").  Each value (ij|kl) is stored
// under its eight role assignments (x,c,y,r) -- the eight permutational images of Eq. 25 (reading
// A5) -- at  T_{XY}[iy][rank_x(c)][rank_y(r)][ix]; of every mirrored pair of assignments (x,c,y,r) <-> (y,r,x,c) only
// the block with X >= Y exists (the digestion reads it in two orientations), so 4 K stores and 1 J store per value.
#include "ltjk_internal.h"
#include "eri_core.h"

namespace ltjk {

struct PEriArgs {
    DevTables t;
    PLDev pl;
    const PPair* bra;
    const PPair* ket;
    int nbra, nket;
    int diag;                 // same list on both sides: ket index <= bra index only
    double tau;
    double* ring;             // ring half of the chunk
    long long jA_off, jB_off; // J arrays: rows = bra AO pairs (contraction = ket), rows = ket AO pairs
    int jA_lda, jB_lda;
};

// Store the EA x EB x EC x ED values v (row-major) whose origin inside the shell quartet (A,B|C,D) is (oa,ob,oc,od)
// under role assignment (x,c,y,r) = the four positions permuted by (PX,PC,PY,PR) in {0,1,2,3} = {a,b,c,d}.
template <int PX, int PC, int PY, int PR, int NA, int NB, int NC, int ND, int EA, int EB, int EC, int ED>
__device__ __forceinline__ void store_copy(const PEriArgs& g, const int* sh, const int* org, const double* __restrict__ v)
{
    constexpr int ncomp[4] = {NA, NB, NC, ND};
    constexpr int ext[4] = {EA, EB, EC, ED};
    constexpr int str[4] = {EB * EC * ED, EC * ED, ED, 1};
    const int ns = g.t.nshell, G = g.pl.G;
    const int X = sh[PX], C = sh[PC], Y = sh[PY], R = sh[PR];
    const PBlock b = g.pl.blk[(((size_t)X * ns + Y) * G + g.pl.sh_grp[C]) * G + g.pl.sh_grp[R]];
    if (b.off < 0) return;          // the mirrored role assignment owns the block (digested through orientation 2)
    const int pc = g.pl.pos[(size_t)X * ns + C] + org[PC], pr = g.pl.pos[(size_t)Y * ns + R] + org[PR];
    constexpr int NX = ncomp[PX];
    const long long ldr = ((long long)NX * b.Lr + 1) & ~1ll;
    double* __restrict__ T = g.ring + b.off;
    constexpr bool small = (EA * EB * EC * ED <= 81);
    if constexpr (small) {
#pragma unroll
        for (int iy = 0; iy < ext[PY]; ++iy)
#pragma unroll
            for (int ic = 0; ic < ext[PC]; ++ic) {
                double* __restrict__ row = T + ((long long)(iy + org[PY]) * b.Lc + pc + ic) * ldr + (long long)pr * NX + org[PX];
#pragma unroll
                for (int ir = 0; ir < ext[PR]; ++ir)
#pragma unroll
                    for (int ix = 0; ix < ext[PX]; ++ix)
                        row[ir * NX + ix] = v[ix * str[PX] + ic * str[PC] + iy * str[PY] + ir * str[PR]];
            }
    } else {
#pragma unroll 1
        for (int iy = 0; iy < ext[PY]; ++iy)
#pragma unroll 1
            for (int ic = 0; ic < ext[PC]; ++ic) {
                double* __restrict__ row = T + ((long long)(iy + org[PY]) * b.Lc + pc + ic) * ldr + (long long)pr * NX + org[PX];
#pragma unroll 1
                for (int ir = 0; ir < ext[PR]; ++ir)
#pragma unroll
                    for (int ix = 0; ix < ext[PX]; ++ix)
                        row[ir * NX + ix] = v[ix * str[PX] + ic * str[PC] + iy * str[PY] + ir * str[PR]];
            }
    }
}

// All stores of a value tile: the eight K role assignments (coincident ones skipped) and the two J entries.
template <int NA, int NB, int NC, int ND, int EA, int EB, int EC, int ED>
__device__ __forceinline__ void store_all(const PEriArgs& g, const PPair& P1, const PPair& P2, int oa, int ob,
                                          const double* __restrict__ v)
{
    const int sh[4] = {P1.A, P1.B, P2.A, P2.B};
    const int org[4] = {oa, ob, 0, 0};
    const bool ab = P1.A != P1.B, cd = P2.A != P2.B, pq = !(P1.A == P2.A && P1.B == P2.B);
    store_copy<0, 1, 2, 3, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
    if (ab) store_copy<1, 0, 2, 3, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
    if (cd) store_copy<0, 1, 3, 2, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
    if (ab && cd) store_copy<1, 0, 3, 2, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
    if (pq) {
        store_copy<2, 3, 0, 1, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
        if (cd) store_copy<3, 2, 0, 1, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
        if (ab) store_copy<2, 3, 1, 0, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
        if (ab && cd) store_copy<3, 2, 1, 0, NA, NB, NC, ND, EA, EB, EC, ED>(g, sh, org, v);
    }
    // J: X_J[(ij)] += w (ij|kl) Ds[(kl)] and X_J[(kl)] += w (ij|kl) Ds[(ij)], w = 1/2 per A == B, C == D
    const double w = (ab ? 1.0 : 0.5) * (cd ? 1.0 : 0.5);
    double* __restrict__ JA = g.ring + g.jA_off;
    double* __restrict__ JB = g.ring + g.jB_off;
#pragma unroll 1
    for (int a = 0; a < EA; ++a)
#pragma unroll 1
        for (int b = 0; b < EB; ++b) {
            const long long p = P1.joff + (a + oa) * NB + (b + ob);
#pragma unroll
            for (int cc = 0; cc < EC; ++cc)
#pragma unroll
                for (int d = 0; d < ED; ++d) {
                    const long long q = P2.joff + cc * ND + d;
                    const double val = w * v[((a * EB + b) * EC + cc) * ED + d];
                    if (g.jA_off >= 0) JA[q * g.jA_lda + p] = val;
                    if (g.jB_off >= 0 && (pq || g.jA_off != g.jB_off)) JB[p * g.jB_lda + q] = val;
                }
        }
}

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(64, 4) peri_kernel(const PEriArgs g)
{
    const int bi = blockIdx.y, ki = blockIdx.x * blockDim.x + threadIdx.x;
    if (ki >= g.nket || (g.diag && ki > bi)) return;
    const PPair P1 = g.bra[bi], P2 = g.ket[ki];
    if (P1.Q * P2.Q < g.tau) return;
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    const DevTables& T = g.t;
    double out[NA * NB * NC * ND];
    eri_quartet<LA, LB, LC, LD>(T.pair_rec + ((size_t)P1.A * T.nshell + P1.B) * T.rec_stride,
                                T.pair_rec + ((size_t)P2.A * T.nshell + P2.B) * T.rec_stride, T.boys, out);
    store_all<NA, NB, NC, ND, NA, NB, NC, ND>(g, P1, P2, 0, 0, out);
}

// Cooperative variant (half-warp per quartet) for the classes whose contracted VRR targets do not fit a thread; same
// evaluation as eri_panel_coop_kernel (ltjk_eri.cu), pair-list epilogue.
template <int NTOT>
struct PCoopSink {
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
    template <int Gi, int N>
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
        if (l16 < N) {
            if (first) accS[Gi * 16 + l16] = buf[0];
            else accS[Gi * 16 + l16] += buf[0];
        }
    }
};

constexpr int kPCoopThreads = 128;            // 8 half-warps = 8 quartets per CTA

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(kPCoopThreads, 1) peri_coop_kernel(const PEriArgs g)
{
    using V = ltjk_gen::Vrr<LA, LB, LC, LD>;
    using HB = ltjk_gen::Hrr<LA, LB>;
    using HK = ltjk_gen::Hrr<LC, LD>;
    constexpr int L = LA + LB + LC + LD;
    constexpr int NE = V::NE, NF = V::NF, NAB = HB::NAB, NCD = HK::NAB;
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    constexpr int QS = NE * NF + NAB * NF;
    extern __shared__ __align__(16) double pcoop_sm[];
    const int lane = threadIdx.x & 31, l16 = lane & 15, hw = threadIdx.x >> 4;
    const unsigned hmask = (lane & 16) ? 0xffff0000u : 0x0000ffffu;
    double* __restrict__ accS = pcoop_sm + hw * QS;
    double* __restrict__ t1S = accS + NE * NF;

    const int bi = blockIdx.y, ki = blockIdx.x * (kPCoopThreads / 16) + hw;
    if (ki >= g.nket || (g.diag && ki > bi)) return;          // the whole half-warp leaves together
    const PPair P1 = g.bra[bi], P2 = g.ket[ki];
    if (P1.Q * P2.Q < g.tau) return;
    const DevTables& T = g.t;
    const double* __restrict__ bra = T.pair_rec + ((size_t)P1.A * T.nshell + P1.B) * T.rec_stride;
    const double* __restrict__ ket = T.pair_rec + ((size_t)P2.A * T.nshell + P2.B) * T.rec_stride;
    const int nb = (int)bra[3], nk = (int)ket[3], nprimq = nb * nk;
    for (int p0 = 0; p0 < nprimq; p0 += 16) {
        const int p = p0 + l16;
        const bool active = p < nprimq;
        const double* bp = bra + kPairHeader + (active ? p / nk : 0) * kPrimStride;
        const double* kp = ket + kPairHeader + (active ? p % nk : 0) * kPrimStride;
        const double pp = bp[0], qv = kp[0];
        const double pq = pp + qv, ipq = 1.0 / pq;
        double pref = bp[7] * kp[7] * 34.986836655249725693 /* 2 pi^{5/2} */ / (pp * qv * sqrt(pq));
        if (!active || fabs(pref) < kPrimCut) pref = 0.0;
        const double PQx = bp[1] - kp[1], PQy = bp[2] - kp[2], PQz = bp[3] - kp[3];
        const double rho = pp * qv * ipq;
        double F[L + 1];
        boys_scaled<L>(rho * (PQx * PQx + PQy * PQy + PQz * PQz), pref, T.boys, F);
        const double wp = -qv * ipq, wq = pp * ipq;
        PCoopSink<NE * NF> sink;
        sink.accS = accS; sink.hmask = hmask; sink.l16 = l16; sink.first = (p0 == 0);
        V::run_t(F, bp[4], bp[5], bp[6], wp * PQx, wp * PQy, wp * PQz, kp[4], kp[5], kp[6], wq * PQx, wq * PQy, wq * PQz,
                 0.5 / pp, 0.5 / qv, 0.5 * ipq, qv * ipq, pp * ipq, sink);
        __syncwarp(hmask);
    }
    for (int jf = l16; jf < NF; jf += 16) HB::run(accS + jf, NF, t1S + jf, NF, bra[0], bra[1], bra[2]);
    __syncwarp(hmask);
    for (int iab = l16; iab < NAB; iab += 16) {
        double o[NCD];
        HK::run(t1S + iab * NF, 1, o, 1, ket[0], ket[1], ket[2]);
        store_all<NA, NB, NC, ND, 1, 1, NC, ND>(g, P1, P2, iab / NB, iab % NB, o);
    }
}

template <int CB, int CK>
static int plaunch_cls(ltjk_ctx* c, const PEriArgs& g)
{
    constexpr int la[6] = {0, 1, 1, 2, 2, 2}, lb[6] = {0, 0, 1, 0, 1, 2};
    if constexpr (CK <= CB) {
        using V = ltjk_gen::Vrr<la[CB], lb[CB], la[CK], lb[CK]>;
        if constexpr (lb[CB] > 0 && lb[CK] > 0 && V::NE * V::NF >= 128) {
            constexpr int QS = V::NE * V::NF + ltjk_gen::Hrr<la[CB], lb[CB]>::NAB * V::NF;
            constexpr int smem = (kPCoopThreads / 16) * QS * (int)sizeof(double);
            LTJK_CUDA(c, cudaFuncSetAttribute(peri_coop_kernel<la[CB], lb[CB], la[CK], lb[CK]>,
                                              cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            const int per = kPCoopThreads / 16;
            peri_coop_kernel<la[CB], lb[CB], la[CK], lb[CK]>
                <<<dim3((unsigned)((g.nket + per - 1) / per), g.nbra), kPCoopThreads, smem, c->eri_stream>>>(g);
        } else {
            peri_kernel<la[CB], lb[CB], la[CK], lb[CK]><<<dim3((unsigned)((g.nket + 63) / 64), g.nbra), 64, 0, c->eri_stream>>>(g);
        }
        LTJK_CUDA(c, cudaGetLastError());
        return LTJK_OK;
    } else {
        return set_err(c, LTJK_EINVAL, "internal: ket class above bra class");
    }
}

template <int CB>
static int plaunch_cls_k(ltjk_ctx* c, int ck, const PEriArgs& g)
{
    switch (ck) {
    case 0: return plaunch_cls<CB, 0>(c, g);
    case 1: return plaunch_cls<CB, 1>(c, g);
    case 2: return plaunch_cls<CB, 2>(c, g);
    case 3: return plaunch_cls<CB, 3>(c, g);
    case 4: return plaunch_cls<CB, 4>(c, g);
    default: return plaunch_cls<CB, 5>(c, g);
    }
}

// All ERI launches of one chunk (group pair gab x group pair gcd): for every class pair cb >= ck, the bra list of
// class cb from one side against the ket list of class ck from the other.
int launch_peri_chunk(ltjk_ctx* c, const PChunk& ch)
{
    PEriArgs g;
    g.t = c->t; g.pl = c->pl; g.tau = c->tau;
    g.ring = c->d_pring + (size_t)ch.buf * c->pring_half;
    for (int cb = 0; cb < 6; ++cb)
        for (int ck = 0; ck <= cb; ++ck)
            for (int swap = 0; swap < 2; ++swap) {
                if (swap && (ch.gab == ch.gcd || cb == ck)) continue;
                const int gpb = swap ? ch.gcd : ch.gab, gpk = swap ? ch.gab : ch.gcd;
                const long long b0 = c->pp_start[(size_t)gpb * 6 + cb], b1 = c->pp_start[(size_t)gpb * 6 + cb + 1];
                const long long k0 = c->pp_start[(size_t)gpk * 6 + ck], k1 = c->pp_start[(size_t)gpk * 6 + ck + 1];
                if (b1 == b0 || k1 == k0) continue;
                if (c->pp_q[b0] * c->pp_q[k0] < c->tau) continue;             // even the largest product is screened
                // kets beyond the cutoff of the strongest bra pair never survive: trim the launch
                long long kn = k1 - k0;
                {
                    const double qb = c->pp_q[b0];
                    long long lo = 0, hi = kn;
                    while (lo < hi) { const long long mid = (lo + hi) / 2; if (c->pp_q[k0 + mid] * qb >= c->tau) lo = mid + 1; else hi = mid; }
                    kn = lo;
                }
                long long bn = b1 - b0;
                {
                    const double qk = c->pp_q[k0];
                    long long lo = 0, hi = bn;
                    while (lo < hi) { const long long mid = (lo + hi) / 2; if (c->pp_q[b0 + mid] * qk >= c->tau) lo = mid + 1; else hi = mid; }
                    bn = lo;
                }
                if (kn == 0 || bn == 0) continue;
                g.bra = c->d_ppairs + b0; g.nbra = (int)bn;
                g.ket = c->d_ppairs + k0; g.nket = (int)kn;
                g.diag = (ch.gab == ch.gcd && cb == ck) ? 1 : 0;
                // the chunk's J array j0[q(gcd) * lda + p(gab)]: diagonal chunks hold both triangles; off the diagonal the
                // bra pair is the row p (no swap) or the contraction index q (swapped launch)
                if (ch.gab == ch.gcd) { g.jA_off = ch.j0_off; g.jA_lda = ch.j0_lda; g.jB_off = ch.j0_off; g.jB_lda = ch.j0_lda; }
                else if (!swap) { g.jA_off = ch.j0_off; g.jA_lda = ch.j0_lda; g.jB_off = -1; g.jB_lda = 0; }
                else { g.jA_off = -1; g.jA_lda = 0; g.jB_off = ch.j0_off; g.jB_lda = ch.j0_lda; }
                if (g.nbra > 65535) return set_err(c, LTJK_EINVAL, "internal: bra pair list exceeds the launch grid");
                c->st_launches++;
                int rc;
                switch (cb) {
                case 0: rc = plaunch_cls_k<0>(c, ck, g); break;
                case 1: rc = plaunch_cls_k<1>(c, ck, g); break;
                case 2: rc = plaunch_cls_k<2>(c, ck, g); break;
                case 3: rc = plaunch_cls_k<3>(c, ck, g); break;
                case 4: rc = plaunch_cls_k<4>(c, ck, g); break;
                default: rc = plaunch_cls_k<5>(c, ck, g); break;
                }
                if (rc) return rc;
            }
    return LTJK_OK;
}

}  // namespace ltjk

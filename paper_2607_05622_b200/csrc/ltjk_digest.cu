// ltjk_digest.cu -- step a8 (non-symmetric J/K digestion), a9 (finalise) and the layout transforms around them.
//
// Digestion as blocked fp64 contractions (no per-integral global atomics; Eq. 25, which the
// paper realises by one atomicAdd per update).  With densities stored density-fastest, Dt[kappa][rho][d], every one
// of the ten updates of Eq. 25 / oracle step O6 on a block quartet panel P[i][j][k][l] is a small GEMM
//     X[(r1,r2), d] += sum_{(c1,c2)} P[r1,r2,c1,c2] * B[(c1,c2), d]
// with (r1,r2) and (c1,c2) two of the four panel indices:
//     view 0  JIJ: rows (i,j) cols (k,l)  B = Ds[(k,l)]            -> X_J[(i,j)]     Ds = D + D^T
//     view 1  JKL: rows (k,l) cols (i,j)  B = Ds[(i,j)]            -> X_J[(k,l)]     J  = X_J + X_J^T
//     view 2  KIK: rows (i,k) cols (j,l)  B = D[(j,l)] -> K[(i,k)] ; partner B = D[(l,j)] -> K[(k,i)]
//     view 3  KJK: rows (j,k) cols (i,l)  B = D[(i,l)] -> K[(j,k)] ; partner B = D[(l,i)] -> K[(k,j)]
//     view 4  KIL: rows (i,l) cols (j,k)  B = D[(j,k)] -> K[(i,l)] ; partner B = D[(k,j)] -> K[(l,i)]
//     view 5  KJL: rows (j,l) cols (i,k)  B = D[(i,k)] -> K[(j,l)] ; partner B = D[(k,i)] -> K[(l,j)]
// (the 2 J and 8 K images of a canonical quartet; for D != D^T all eight K images are distinct).
// One CTA owns a 128-row tile of one output block for all (<= 192) densities, keeps it in registers over a RUN of
// panels sharing that output block, and flushes once with coalesced fp64 reductions.
#include "ltjk_internal.h"
#include "digest_common.h"
#include <cstdio>
#include <cstdlib>
#include <algorithm>

namespace ltjk {

constexpr int kMaxNC = 1024;   // max columns of one panel view (block AO count squared)

struct DigestArgs {
    DevTables t;
    const DigestItem* items;
    const SubChunk* subs;
    const double* panel;
    const double* Dt;
    const double* Dst;
    const unsigned char* mask;   // per (item, chunk): bit w set = the 16 x 16 sub-tile of consumer warp w is not all screened
    double* Jt;
    double* Kt;
    int nDp;
    int fuse;                    // nD <= 16 (TN = 1): the two partners of a K item share one pass, 16 columns each
};

template <int TN>
struct DigestSmem {
    double A[kStages][kKC][kMTP];
    double B[kStages][kKC][32 * TN];
    unsigned long long full[kStages];    // producer -> consumers: the stage's tiles have landed
    unsigned long long empty[kStages];   // consumers -> producer: the stage may be refilled
    unsigned cmask[kStages];             // warp bits of the chunk in the stage (written by producer thread 0)
    int rowoff[kMT];
    int acol[kMaxNC];
    unsigned bcol[kMaxNC];
    unsigned bcol2[kMaxNC];              // fused partner (g.fuse): density row of the transposed partner
};


// Warp-specialised, persistent, one CTA per SM: warps 0..7 (two warpgroups) are consumers -- LDS + DFMA only, thread
// tile 16 x TN, warp w owns rows 16w..16w+15 and all 32 TN columns -- and warps 8..11 (one warpgroup) are producers:
// panel index tables, cp.async of the A and B tiles into a 5-stage mbarrier ring.  setmaxnreg moves registers from
// the producers (40) to the consumers (232).  Every CTA walks the work items blockIdx.x, blockIdx.x + gridDim.x, ...;
// the ring keeps running across items, so the producers prefetch the next item while the consumers finish and flush
// the current one (profiles/: with one item per CTA the consumers idled ~15 % of the time at item starts; before
// specialisation the DFMA warps spent 27 % of their instructions on the loader).
struct ItemCtx {
    DigestItem it;
    SubChunk sc;
    int R1, R2, nR2, nrows, nI, nJ, n0;
};

__device__ __forceinline__ ItemCtx load_item(const DigestArgs& g, int vi, int ncolblk, int colw)
{
    ItemCtx c;
    const DevTables& T = g.t;
    c.it = g.items[vi / ncolblk];
    c.n0 = (vi % ncolblk) * colw;
    c.sc = g.subs[c.it.sub];
    const int I = c.sc.I, J = c.sc.J;
    c.nI = T.blk_nao[I]; c.nJ = T.blk_nao[J];
    switch (c.it.view) {                       // row blocks: constant over the run by construction
    case 0: c.R1 = I; c.R2 = J; break;
    case 1: c.R1 = T.pair_I[c.it.a]; c.R2 = T.pair_J[c.it.a]; break;
    case 2: c.R1 = I; c.R2 = c.it.a; break;
    case 3: c.R1 = J; c.R2 = c.it.a; break;
    case 4: c.R1 = I; c.R2 = c.it.a; break;
    default: c.R1 = J; c.R2 = c.it.a; break;
    }
    c.nR2 = T.blk_nao[c.R2];
    c.nrows = T.blk_nao[c.R1] * c.nR2;
    return c;
}

// (K, L, rank) of step s of the run
__device__ __forceinline__ void step_blocks(const DevTables& T, const DigestItem& it, int s, int& K, int& L, int& rank)
{
    if (it.view <= 1) { rank = it.a + s; K = T.pair_I[rank]; L = T.pair_J[rank]; }
    else if (it.view <= 3) { K = it.a; L = it.b + s; rank = T.rank_of[K * T.nblk + L]; }
    else { L = it.a; K = it.b + s; rank = T.rank_of[K * T.nblk + L]; }
}

template <int TN>
__global__ void __launch_bounds__(kDigestThreads, 1) digest_kernel(const DigestArgs g, const int nvirt, const int ncolblk)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    DigestSmem<TN>& S = *reinterpret_cast<DigestSmem<TN>*>(smem_raw);
    const DevTables& T = g.t;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int N = T.nao, nDp = g.nDp;

    if (tid == 0) {
        for (int st = 0; st < kStages; ++st) {
            mbar_init(&S.full[st], kProducerThreads + 1);   // 128 cp.async arrivals + the thread that posts cmask
            mbar_init(&S.empty[st], kConsumerWarps);
        }
    }
    __syncthreads();
    int gch = 0;                                   // chunk counter of the ring, runs across items in both roles

    if (w >= kConsumerWarps) {
        // ===================== producer warpgroup =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        const int pt = tid - kConsumerWarps * 32, pw = pt >> 5;
        for (int vi = blockIdx.x; vi < nvirt; vi += gridDim.x) {
            const ItemCtx c = load_item(g, vi, ncolblk, 32 * TN);
            const DigestItem& it = c.it;
            const int view = it.view, I = c.sc.I, J = c.sc.J, nI = c.nI, nJ = c.nJ;
            const bool fused = (TN == 1) && g.fuse && view >= 2;    // both partners of a K item in one pass
            if (fused && it.partner) continue;                      // done by its partner-0 twin (same tile, same mask)
            const bool partner = it.partner != 0;
            const double* __restrict__ Bmat = (view <= 1) ? g.Dst : g.Dt;
            const bool rowContig = (view == 1 || view >= 4);   // l (unit stride) is a row index
            int qi = 0;                                        // chunk index inside the item (mask position)
            for (int s = 0; s < it.count; ++s) {
                int K, L, rank;
                step_blocks(T, it, s, K, L, rank);
                const int nK = T.blk_nao[K], nL = T.blk_nao[L];
                const double* __restrict__ P = g.panel + c.sc.base + (T.koff[rank] - T.koff[c.sc.r0]) * (long long)(nI * nJ);
                const int sI = nJ * nK * nL, sJ = nK * nL, sK = nL, sL = 1;
                int C1, C2, sR1, sR2, sC1, sC2;
                switch (view) {
                case 0: C1 = K; C2 = L; sR1 = sI; sR2 = sJ; sC1 = sK; sC2 = sL; break;
                case 1: C1 = I; C2 = J; sR1 = sK; sR2 = sL; sC1 = sI; sC2 = sJ; break;
                case 2: C1 = J; C2 = L; sR1 = sI; sR2 = sK; sC1 = sJ; sC2 = sL; break;
                case 3: C1 = I; C2 = L; sR1 = sJ; sR2 = sK; sC1 = sI; sC2 = sL; break;
                case 4: C1 = J; C2 = K; sR1 = sI; sR2 = sL; sC1 = sJ; sC2 = sK; break;
                default: C1 = I; C2 = K; sR1 = sJ; sR2 = sL; sC1 = sI; sC2 = sK; break;
                }
                const int nC2 = T.blk_nao[C2], nC = T.blk_nao[C1] * nC2;
                const int aoC1 = T.blk_ao0[C1], aoC2 = T.blk_ao0[C2];
                asm volatile("bar.sync 1, %0;\n" ::"n"(kProducerThreads));   // previous panel's tables no longer read
                {
                    const int mm = it.rowtile * kMT + pt;                     // kMT == kProducerThreads rows
                    S.rowoff[pt] = (mm < c.nrows) ? (mm / c.nR2) * sR1 + (mm % c.nR2) * sR2 : -1;
                }
                for (int cidx = pt; cidx < nC; cidx += kProducerThreads) {
                    const int c1 = cidx / nC2, c2 = cidx % nC2;
                    S.acol[cidx] = c1 * sC1 + c2 * sC2;
                    S.bcol[cidx] = partner ? (unsigned)((aoC2 + c2) * N + aoC1 + c1) : (unsigned)((aoC1 + c1) * N + aoC2 + c2);
                    if (fused) S.bcol2[cidx] = (unsigned)((aoC2 + c2) * N + aoC1 + c1);
                }
                asm volatile("bar.sync 1, %0;\n" ::"n"(kProducerThreads));
                const int nch = (nC + kKC - 1) / kKC;
                const int ro_fixed = S.rowoff[pt];                            // rowContig: this thread's row
                for (int ch = 0; ch < nch; ++ch, ++qi) {
                    // tiles whose integrals are all Schwarz-screened (exact zeros in the panel) are never loaded
                    const unsigned wbits = g.mask[(size_t)it.maskoff + (unsigned)qi];
                    if (!wbits) continue;
                    const int st = gch % kStages;
                    if (gch >= kStages) mbar_wait(&S.empty[st], (unsigned)((gch / kStages - 1) & 1));
                    // A tile: kKC x kMT elements of 8 bytes, 16 per producer thread, lanes along the unit stride
                    if (rowContig) {
#pragma unroll 4
                        for (int k = 0; k < kKC; ++k) {
                            const int cidx = ch * kKC + k;
                            const bool ok = (ro_fixed >= 0) && (cidx < nC);
                            cp_async8(&S.A[st][k][pt], ok ? (P + ro_fixed + S.acol[cidx]) : P, ok);
                        }
                    } else {
                        const int k = pt & 15, cidx = ch * kKC + k;
                        const bool cok = cidx < nC;
                        const int co = cok ? S.acol[cidx] : 0;
#pragma unroll 4
                        for (int e = 0; e < kMT / 8; ++e) {
                            const int m = (pt >> 4) + 8 * e, ro = S.rowoff[m];
                            const bool ok = cok && (ro >= 0);
                            cp_async8(&S.A[st][k][m], ok ? (P + ro + co) : P, ok);
                        }
                    }
                    // B tile: kKC density rows of 32 TN doubles, 16-byte pieces; warp pw copies rows pw, pw+4, ...
#pragma unroll
                    for (int h = 0; h < kKC / kProducerWarps; ++h) {
                        const int k = pw + kProducerWarps * h, cidx = ch * kKC + k;
                        const bool ok = cidx < nC;
                        const double* src = ok ? (Bmat + (size_t)S.bcol[cidx] * nDp + c.n0) : Bmat;
                        if (fused) {
                            // columns 0..15: densities of partner 0;  columns 16..31: the same densities, partner 1
                            const double* src2 = ok ? (Bmat + (size_t)S.bcol2[cidx] * nDp + c.n0) : Bmat;
                            if (lane < 16)
                                cp_async16(&S.B[st][k][lane * 2], (lane < 8 ? src : src2) + (ok ? (lane & 7) * 2 : 0), ok);
                        } else {
                            for (int pc = lane; pc < 16 * TN; pc += 32)
                                cp_async16(&S.B[st][k][pc * 2], src + (ok ? pc * 2 : 0), ok);
                        }
                    }
                    mbar_arrive_on_cp_async(&S.full[st]);
                    if (pt == 0) { S.cmask[st] = wbits; mbar_arrive(&S.full[st]); }   // release: visible after the wait
                    ++gch;
                }
            }
        }
        return;
    }

    // ===================== consumer warpgroups =====================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;\n");
    if constexpr (TN <= 5) {
    // thread tile 8 rows x 2 TN columns: the two half-warps of warp w own rows 16w..16w+7 and 16w+8..16w+15, lane l16
    // owns the column pairs (2 l16, 2 l16 + 1) + 32 t.  Per k: 4 LDS.128 for A (two addresses per warp) and TN LDS.128
    // for B, against 8 + TN LDS.64 with a 16 x TN tile (measured +4 % on the isolated loop)
    const int wrow = w * kTM;
    const int trow = wrow + (lane >> 4) * 8;
    const int l16 = lane & 15;
    for (int vi = blockIdx.x; vi < nvirt; vi += gridDim.x) {
        const ItemCtx c = load_item(g, vi, ncolblk, 32 * TN);
        const DigestItem& it = c.it;
        const int view = it.view;
        const bool fused = (TN == 1) && g.fuse && view >= 2;
        if (fused && it.partner) continue;
        const int total_chunks = it.nnz;
        const bool warp_active = it.rowtile * kMT + wrow < c.nrows;   // ragged last tile: idle warps skip the DFMAs
        double acc[8][2 * TN];
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int t = 0; t < 2 * TN; ++t) acc[r][t] = 0.0;

        for (int q = 0; q < total_chunks; ++q, ++gch) {
            const int st = gch % kStages;
            mbar_wait(&S.full[st], (unsigned)((gch / kStages) & 1));
            if (warp_active && ((S.cmask[st] >> w) & 1u)) {
#pragma unroll
                for (int k = 0; k < kKC; ++k) {
                    const double2* ap = reinterpret_cast<const double2*>(&S.A[st][k][trow]);
                    double a[8];
#pragma unroll
                    for (int r = 0; r < 4; ++r) { const double2 v = ap[r]; a[2 * r] = v.x; a[2 * r + 1] = v.y; }
                    double b[2 * TN];
#pragma unroll
                    for (int t = 0; t < TN; ++t) {
                        const double2 v = *reinterpret_cast<const double2*>(&S.B[st][k][2 * l16 + 32 * t]);
                        b[2 * t] = v.x; b[2 * t + 1] = v.y;
                    }
#pragma unroll
                    for (int r = 0; r < 8; ++r)
#pragma unroll
                        for (int t = 0; t < 2 * TN; ++t) acc[r][t] = fma(a[r], b[t], acc[r][t]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[st]);
        }

        // flush: coalesced fp64 reductions into the density-fastest accumulators
        if (warp_active) {
            const double mult = (double)it.mult;
            const bool partner = it.partner != 0;
            double* __restrict__ Out = (view <= 1) ? g.Jt : g.Kt;
            const int aoR1 = T.blk_ao0[c.R1], aoR2 = T.blk_ao0[c.R2];
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const int m = it.rowtile * kMT + trow + r;
                if (m < c.nrows) {
                    const int r1 = m / c.nR2, r2 = m % c.nR2;
                    // fused: lanes 8..15 of a half-warp hold partner 1 -> transposed output row, densities 2 (l16 - 8)
                    const bool tr = fused ? (l16 >= 8) : partner;
                    const size_t row = tr ? (size_t)(aoR2 + r2) * N + aoR1 + r1 : (size_t)(aoR1 + r1) * N + aoR2 + r2;
                    double* o = Out + row * nDp + c.n0 + 2 * (fused ? (l16 & 7) : l16);
#pragma unroll
                    for (int t = 0; t < TN; ++t) {
                        atomicAdd(o + 32 * t, mult * acc[r][2 * t]);
                        atomicAdd(o + 32 * t + 1, mult * acc[r][2 * t + 1]);
                    }
                }
            }
        }
    }
    } else {
        // TN = 6 (192 densities per column block): the 16 x TN tile measured faster there
    const int trow = w * kTM;
    for (int vi = blockIdx.x; vi < nvirt; vi += gridDim.x) {
        const ItemCtx c = load_item(g, vi, ncolblk, 32 * TN);
        const DigestItem& it = c.it;
        const int view = it.view;
        const int total_chunks = it.nnz;
        const bool warp_active = it.rowtile * kMT + trow < c.nrows;   // ragged last tile: idle warps skip the DFMAs
        double acc[kTM][TN];
#pragma unroll
        for (int r = 0; r < kTM; ++r)
#pragma unroll
            for (int t = 0; t < TN; ++t) acc[r][t] = 0.0;

        for (int q = 0; q < total_chunks; ++q, ++gch) {
            const int st = gch % kStages;
            mbar_wait(&S.full[st], (unsigned)((gch / kStages) & 1));
            if (warp_active && ((S.cmask[st] >> w) & 1u)) {
#pragma unroll
                for (int k = 0; k < kKC; ++k) {
                    const double2* ap = reinterpret_cast<const double2*>(&S.A[st][k][trow]);
                    double a[kTM];
#pragma unroll
                    for (int r = 0; r < kTM / 2; ++r) { const double2 v = ap[r]; a[2 * r] = v.x; a[2 * r + 1] = v.y; }
                    double b[TN];
#pragma unroll
                    for (int t = 0; t < TN; ++t) b[t] = S.B[st][k][lane + 32 * t];
#pragma unroll
                    for (int r = 0; r < kTM; ++r)
#pragma unroll
                        for (int t = 0; t < TN; ++t) acc[r][t] = fma(a[r], b[t], acc[r][t]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[st]);
        }

        // flush: coalesced fp64 reductions into the density-fastest accumulators
        if (warp_active) {
            const double mult = (double)it.mult;
            const bool partner = it.partner != 0;
            double* __restrict__ Out = (view <= 1) ? g.Jt : g.Kt;
            const int aoR1 = T.blk_ao0[c.R1], aoR2 = T.blk_ao0[c.R2];
#pragma unroll
            for (int r = 0; r < kTM; ++r) {
                const int m = it.rowtile * kMT + trow + r;
                if (m < c.nrows) {
                    const int r1 = m / c.nR2, r2 = m % c.nR2;
                    const size_t row = partner ? (size_t)(aoR2 + r2) * N + aoR1 + r1 : (size_t)(aoR1 + r1) * N + aoR2 + r2;
                    double* o = Out + row * nDp + c.n0 + lane;
#pragma unroll
                    for (int t = 0; t < TN; ++t) atomicAdd(o + 32 * t, mult * acc[r][t]);
                }
            }
        }
    }
    }
}

template <int TN>
static int launch_digest_tn(ltjk_ctx* c, const DigestArgs& g, int nitems, int ncolblk)
{
    const size_t smem = sizeof(DigestSmem<TN>);
    // per launch: the attribute belongs to the device's context, and a process may hold contexts on several devices
    LTJK_CUDA(c, cudaFuncSetAttribute(digest_kernel<TN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const long long nvirt = (long long)nitems * ncolblk;
    if (nvirt > 0x7fffffffll) return set_err(c, LTJK_EINVAL, "digest: more than 2^31 work items in one launch");
    // 32 persistent waves (measured 2..64 on B200: 632, 626, 621, 609, 601, 598 ms of digestion per 439-AO sweep):
    // the hardware block scheduler balances the load, each CTA still prefetches across its items
    const int grid = (int)std::min<long long>(nvirt, 32ll * nsm);
    digest_kernel<TN><<<grid, kDigestThreads, smem, c->stream>>>(g, (int)nvirt, ncolblk);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

// column blocking of the padded density count: nDp = ncolblk * 32 * TN
void digest_colblocks(int nD, int mode, int* TN, int* ncolblk)
{   // declared in ltjk_internal.h.  mode 2 (pair lists): A tiles are cheap contiguous copies, and the 16 x 6 thread
    // tile of TN = 6 stalls on its operand loads (192 accumulator registers), so 192 densities run as 2 x TN = 3
    // (measured at 730 AO: digestion 3123 -> 2650 ms); mode 1 re-gathers A per column block and prefers TN = 6.
    const int n32 = (nD + 31) / 32;
    if (const char* e = getenv("LTJK_TN")) {            // development override
        const int tn = atoi(e);
        if (tn >= 1 && tn <= 6) { *TN = tn; *ncolblk = (n32 + tn - 1) / tn; return; }
    }
    int best_tn = 1, best_nb = n32, best_cost = 1 << 30;
    for (int tn = 1; tn <= (mode == 2 ? 5 : 6); ++tn) {
        const int nb = (n32 + tn - 1) / tn;
        const int cost = nb * tn * 8 + nb * 3;   // padded columns, then fewer passes over A
        if (cost < best_cost) { best_cost = cost; best_tn = tn; best_nb = nb; }
    }
    *TN = best_tn; *ncolblk = best_nb;
}

int launch_digest(ltjk_ctx* c, const Group& ch, int nDp, bool doJ, bool doK)
{
    const long long first = ch.item0 + (doJ ? 0 : ch.nitemsJ);
    const int nitems = (doJ ? ch.nitemsJ : 0) + (doK ? ch.nitemsK : 0);
    if (nitems == 0) return LTJK_OK;
    DigestArgs g;
    g.t = c->t; g.items = c->d_items + first; g.subs = c->d_subs; g.mask = c->d_chunkmask; g.panel = c->d_panel + (size_t)ch.buf * c->panel_half;
    g.Dt = c->Dt; g.Dst = c->Dst; g.Jt = c->Jt; g.Kt = c->Kt;
    g.nDp = nDp;
    int TN, nb;
    digest_colblocks(nDp, 1, &TN, &nb);
    g.fuse = (TN == 1 && nb == 1 && c->cur_nD <= 16) ? 1 : 0;
    if (nb * TN * 32 != nDp) return set_err(c, LTJK_EINVAL, "internal: nDp is not a whole number of column blocks");
    c->st_launches++;
    switch (TN) {
    case 1: return launch_digest_tn<1>(c, g, nitems, nb);
    case 2: return launch_digest_tn<2>(c, g, nitems, nb);
    case 3: return launch_digest_tn<3>(c, g, nitems, nb);
    case 4: return launch_digest_tn<4>(c, g, nitems, nb);
    case 5: return launch_digest_tn<5>(c, g, nitems, nb);
    default: return launch_digest_tn<6>(c, g, nitems, nb);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a5, geometry-frozen: for every work item and every contraction chunk, does the 128 x 16 tile of the panel view hold
// at least one integral of an unscreened shell quartet (Q_ij Q_kl >= tau)?  One CTA per item, threads over chunks.
__global__ void chunk_mask_kernel(const DevTables T, DigestItem* __restrict__ items, const SubChunk* __restrict__ subs,
                                  long long nitems, double tau, unsigned char* __restrict__ mask)
{
    __shared__ int nnz;
    for (long long ii = blockIdx.x; ii < nitems; ii += gridDim.x) {
        const DigestItem it = items[ii];
        const SubChunk sc = subs[it.sub];
        const int I = sc.I, J = sc.J, view = it.view;
        int R1, R2;
        switch (view) {
        case 0: R1 = I; R2 = J; break;
        case 1: R1 = T.pair_I[it.a]; R2 = T.pair_J[it.a]; break;
        case 2: R1 = I; R2 = it.a; break;
        case 3: R1 = J; R2 = it.a; break;
        case 4: R1 = I; R2 = it.a; break;
        default: R1 = J; R2 = it.a; break;
        }
        const int nR2 = T.blk_nao[R2], nrows = T.blk_nao[R1] * nR2;
        const int m0 = it.rowtile * kMT, m1 = min(m0 + kMT, nrows);
        const int aoR1 = T.blk_ao0[R1], aoR2 = T.blk_ao0[R2];
        if (threadIdx.x == 0) nnz = 0;
        __syncthreads();
        int mine = 0;
        for (int q = threadIdx.x; q < it.nchunks; q += blockDim.x) {
            // locate the step (panel) and the chunk inside it
            int s = 0, ch = q, K = 0, L = 0, C1 = 0, C2 = 0;
            for (; s < it.count; ++s) {
                int rank;
                step_blocks(T, it, s, K, L, rank);
                switch (view) {
                case 0: C1 = K; C2 = L; break;
                case 1: C1 = I; C2 = J; break;
                case 2: C1 = J; C2 = L; break;
                case 3: C1 = I; C2 = L; break;
                case 4: C1 = J; C2 = K; break;
                default: C1 = I; C2 = K; break;
                }
                const int nch = (T.blk_nao[C1] * T.blk_nao[C2] + kKC - 1) / kKC;
                if (ch < nch) break;
                ch -= nch;
            }
            const int nC2 = T.blk_nao[C2], nC = T.blk_nao[C1] * nC2;
            const int aoC1 = T.blk_ao0[C1], aoC2 = T.blk_ao0[C2];
            const int c0 = ch * kKC, c1e = min(c0 + kKC, nC);
            unsigned wbits = 0;
            for (int wq = 0; wq < kConsumerWarps; ++wq) {
            const int mw0 = m0 + wq * kTM, mw1 = min(mw0 + kTM, m1);
            bool any = false;
            int prev_cs1 = -1, prev_cs2 = -1;
            for (int cidx = c0; cidx < c1e && !any && mw0 < mw1; ++cidx) {
                const int sc1 = T.ao_sh[aoC1 + cidx / nC2], sc2 = T.ao_sh[aoC2 + cidx % nC2];
                if (sc1 == prev_cs1 && sc2 == prev_cs2) continue;       // same shell pair as the previous column
                prev_cs1 = sc1; prev_cs2 = sc2;
                int prev_rs1 = -1, prev_rs2 = -1;
                for (int m = mw0; m < mw1; ++m) {
                    const int sr1 = T.ao_sh[aoR1 + m / nR2], sr2 = T.ao_sh[aoR2 + m % nR2];
                    if (sr1 == prev_rs1 && sr2 == prev_rs2) continue;
                    prev_rs1 = sr1; prev_rs2 = sr2;
                    int si, sj, sk, sl;
                    switch (view) {
                    case 0: si = sr1; sj = sr2; sk = sc1; sl = sc2; break;
                    case 1: sk = sr1; sl = sr2; si = sc1; sj = sc2; break;
                    case 2: si = sr1; sk = sr2; sj = sc1; sl = sc2; break;
                    case 3: sj = sr1; sk = sr2; si = sc1; sl = sc2; break;
                    case 4: si = sr1; sl = sr2; sj = sc1; sk = sc2; break;
                    default: sj = sr1; sl = sr2; si = sc1; sk = sc2; break;
                    }
                    if (T.schwarz[(size_t)si * T.nshell + sj] * T.schwarz[(size_t)sk * T.nshell + sl] >= tau) { any = true; break; }
                }
            }
            if (any) wbits |= 1u << wq;
            }
            mask[(size_t)it.maskoff + (unsigned)q] = (unsigned char)wbits;
            if (wbits) ++mine;
        }
        if (mine) atomicAdd(&nnz, mine);
        __syncthreads();
        if (threadIdx.x == 0) items[ii].nnz = nnz;
        __syncthreads();
    }
}

int launch_chunk_mask(ltjk_ctx* c)
{
    if (c->n_items == 0) return LTJK_OK;
    const int grid = (int)std::min<long long>(c->n_items, 148ll * 64);
    chunk_mask_kernel<<<grid, 64, 0, c->stream>>>(c->t, c->d_items, c->d_subs, c->n_items, c->tau, c->d_chunkmask);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Layout transforms (HBM-bound): caller layout X[d][mu][nu] <-> internal density-fastest Xt[mu'][nu'][d'],
// mu' = internal AO (ao_perm[mu'] = caller AO), d' < nDp (zero padded).
__global__ void pack_kernel(int N, int nD, int nDp, const int* __restrict__ perm, const double* __restrict__ D,
                            double* __restrict__ Dt)
{
    __shared__ double tile[32][33];
    const int mu = blockIdx.z, nu0 = blockIdx.x * 32, d0 = blockIdx.y * 32;
    const int pm = perm[mu];
    {
        const int nu = nu0 + threadIdx.x;
        for (int dd = threadIdx.y; dd < 32; dd += 8) {
            const int d = d0 + dd;
            tile[dd][threadIdx.x] = (nu < N && d < nD) ? D[((size_t)d * N + pm) * N + perm[nu]] : 0.0;
        }
    }
    __syncthreads();
    {
        const int d = d0 + threadIdx.x;
        for (int nn = threadIdx.y; nn < 32; nn += 8) {
            const int nu = nu0 + nn;
            if (nu < N && d < nDp) Dt[((size_t)mu * N + nu) * nDp + d] = tile[threadIdx.x][nn];
        }
    }
}

__global__ void symmetrize_kernel(int N, int nDp, const double* __restrict__ Dt, double* __restrict__ Dst)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t tot = (size_t)N * N * nDp;
    if (i >= tot) return;
    const int d = (int)(i % nDp);
    const size_t mn = i / nDp;
    const int mu = (int)(mn / N), nu = (int)(mn % N);
    Dst[i] = Dt[i] + Dt[((size_t)nu * N + mu) * nDp + d];
}

// a9: K[d][mu][nu] = Kt[mu'][nu'][d];  J[d][mu][nu] = Xt[mu'][nu'][d] + Xt[nu'][mu'][d]
__global__ void unpack_kernel(int N, int nD, int nDp, const int* __restrict__ perm, const double* __restrict__ Xt,
                              double* __restrict__ X, int mirror)
{
    __shared__ double tile[32][33];
    const int mu = blockIdx.z, nu0 = blockIdx.x * 32, d0 = blockIdx.y * 32;
    {
        const int d = d0 + threadIdx.x;
        for (int nn = threadIdx.y; nn < 32; nn += 8) {
            const int nu = nu0 + nn;
            double v = 0.0;
            if (nu < N && d < nDp) {
                v = Xt[((size_t)mu * N + nu) * nDp + d];
                if (mirror) v += Xt[((size_t)nu * N + mu) * nDp + d];
            }
            tile[nn][threadIdx.x] = v;
        }
    }
    __syncthreads();
    {
        const int pm = perm[mu];
        const int nu = nu0 + threadIdx.x;
        for (int dd = threadIdx.y; dd < 32; dd += 8) {
            const int d = d0 + dd;
            if (nu < N && d < nD) X[((size_t)d * N + pm) * N + perm[nu]] = tile[threadIdx.x][dd];
        }
    }
}

int launch_pack_densities(ltjk_ctx* c, int nD, int nDp, const double* D)
{
    const int N = c->nao;
    dim3 grid((N + 31) / 32, nDp / 32, N), blk(32, 8);
    pack_kernel<<<grid, blk, 0, c->stream>>>(N, nD, nDp, c->t.ao_perm, D, c->Dt);
    LTJK_CUDA(c, cudaGetLastError());
    const size_t tot = (size_t)N * N * nDp;
    symmetrize_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, c->stream>>>(N, nDp, c->Dt, c->Dst);
    LTJK_CUDA(c, cudaGetLastError());
    c->st_launches += 2;
    return LTJK_OK;
}

int launch_unpack_results(ltjk_ctx* c, int nD, int nDp, double* J, double* K)
{
    const int N = c->nao;
    dim3 grid((N + 31) / 32, nDp / 32, N), blk(32, 8);
    if (J) {
        unpack_kernel<<<grid, blk, 0, c->stream>>>(N, nD, nDp, c->t.ao_perm, c->Jt, J, 1);
        LTJK_CUDA(c, cudaGetLastError());
        c->st_launches++;
    }
    if (K) {
        unpack_kernel<<<grid, blk, 0, c->stream>>>(N, nD, nDp, c->t.ao_perm, c->Kt, K, 0);
        LTJK_CUDA(c, cudaGetLastError());
        c->st_launches++;
    }
    return LTJK_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Roofline denominators: sustained DFMA rate of the fp64 vector pipe, and a device copy.
__global__ void __launch_bounds__(256) dfma_kernel(int iters, double seed, double* out)
{
    double x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = seed + threadIdx.x * 1e-9 + i;
    const double a = 1.0000000001, b = 1e-12;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456) out[0] = s;
}

int bench_dfma(ltjk_ctx* c, double* tflops)
{
    cudaDeviceProp prop;
    LTJK_CUDA(c, cudaGetDeviceProperties(&prop, c->device));
    double* d = nullptr;
    LTJK_CUDA(c, cudaMalloc(&d, 8));
    const int blocks = prop.multiProcessorCount * 8, iters = 1 << 15;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    dfma_kernel<<<blocks, 256, 0, c->stream>>>(1 << 10, 1.0, d);   // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, c->stream);
        for (int k = 0; k < 8; ++k) dfma_kernel<<<blocks, 256, 0, c->stream>>>(iters, 1.0, d);   // ~0.3 s sustained
        cudaEventRecord(e1, c->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fl = 8.0 * blocks * 256.0 * iters * 16.0 * 2.0;
        best = fmax(best, fl / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    LTJK_CUDA(c, cudaGetLastError());
    *tflops = best;
    return LTJK_OK;
}

__global__ void copy_kernel(size_t n, const double2* __restrict__ a, double2* __restrict__ b)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) b[i] = a[i];
}

int bench_copy(ltjk_ctx* c, double* gbs)
{
    const size_t bytes = (size_t)1 << 30;
    double2 *a = nullptr, *b = nullptr;
    LTJK_CUDA(c, cudaMalloc(&a, bytes));
    LTJK_CUDA(c, cudaMalloc(&b, bytes));
    cudaMemsetAsync(a, 0, bytes, c->stream);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, c->stream);
        copy_kernel<<<148 * 16, 512, 0, c->stream>>>(bytes / 16, a, b);
        cudaEventRecord(e1, c->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = fmax(best, 2.0 * bytes / (ms * 1e-3) / 1e9);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(a); cudaFree(b);
    LTJK_CUDA(c, cudaGetLastError());
    *gbs = best;
    return LTJK_OK;
}

}  // namespace ltjk

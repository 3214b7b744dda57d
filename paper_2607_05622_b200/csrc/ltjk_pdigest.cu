// ltjk_pdigest.cu -- step a8 (non-symmetric J/K digestion), pair-list formulation (see ltjk_pair.cu).
//
// Every work record is a matrix A(c, m) = ring[off + c*lda + m] (contraction c, rows m contiguous) with row tiles of
// 128 and a contraction length per tile (the staircase of the Q-sorted lists).  The kernel is the warp-specialised
// gather-GEMM of ltjk_digest.cu without any per-panel index tables:
//     K record (block T_XY, one pass per component iy of Y):
//         Kt[x0 + m % nX][r(m / nX)][:] += sum_c A_iy(c, m) * Dt[c_ao(c)][y0 + iy][:]          (Eq. 17, all 8 images)
//     J record:  Jt[row(m)][:] += sum_c A(c, m) * Dst[row'(c)][:]                               (Dst = D + D^T)
// Producer warps stream A tiles (16 x 128, 16-byte cp.async, coalesced) and the gathered density rows; consumer warps
// hold a 128 x 32 TN accumulator tile in registers and flush it once per item with fp64 reductions.
#include "ltjk_internal.h"
#include "digest_common.h"
#include <algorithm>
#include <cstdlib>

namespace ltjk {

constexpr int kWorkQ = 4;

struct PDigestArgs {
    const PWork* work;
    const int* tiles;
    const int* pl_ao;
    const int* jrow;
    const double* ring;
    const double* Dt;
    const double* Dst;
    double* Jt;
    double* Kt;
    int nDp, N, nwork, ncolblk;
    int* counter;          // work-stealing cursor of this launch (zeroed by the host)
};

constexpr int kRowPitch = kKC + 2;      // orientation 2: row-major A tile [row][16 contraction values], 144-byte pitch

template <int TN>
struct PDigestSmem {
    // orientation 1: A[st][k][row] (kKC x kMTP doubles);  orientation 2: the same bytes as [row][kRowPitch]
    double A[kStages][(kMT * kRowPitch > kKC * kMTP) ? kMT * kRowPitch : kKC * kMTP];
    double B[kStages][kKC][32 * TN];
    unsigned long long full[kStages];
    unsigned long long empty[kStages];
    unsigned long long wq_full[kWorkQ];   // work queue: producer thread 0 draws record indices from the global cursor
    unsigned long long wq_empty[kWorkQ];
    int wq[kWorkQ];
};

template <int TN>
__global__ void __launch_bounds__(kDigestThreads, 1) pdigest_kernel(const PDigestArgs g)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PDigestSmem<TN>& S = *reinterpret_cast<PDigestSmem<TN>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int N = g.N, nDp = g.nDp;
    if (tid == 0) {
        for (int st = 0; st < kStages; ++st) {
            mbar_init(&S.full[st], kProducerThreads);
            mbar_init(&S.empty[st], kConsumerWarps);
        }
        for (int q = 0; q < kWorkQ; ++q) {
            mbar_init(&S.wq_full[q], 1);
            mbar_init(&S.wq_empty[q], kConsumerWarps + kProducerWarps);
        }
    }
    __syncthreads();
    int gch = 0;                                   // chunk counter of the ring, runs across items in both roles

    if (w >= kConsumerWarps) {
        // ===================== producer warpgroup =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        const int pt = tid - kConsumerWarps * 32, pw = pt >> 5;
        for (int it = 0;; ++it) {
            // records are sorted by cost (longest first) and handed out dynamically: the launch ends balanced
            const int slot = it % kWorkQ;
#ifdef LTJK_NOQ
            const int wi0 = (int)(blockIdx.x + it * gridDim.x);
            const int wi = wi0 < g.nwork ? wi0 : -1;
#else
            __syncwarp();     // lanes diverge in the B-row copy loop (16 TN pieces over 32 lanes): lane 0 must not be
                              // left behind lanes that already spin on wq_full
            if (pt == 0) {
                if (it >= kWorkQ) mbar_wait(&S.wq_empty[slot], (unsigned)((it / kWorkQ - 1) & 1));
                const int nxt = g.counter ? atomicAdd(g.counter, 1) : (int)(blockIdx.x + it * gridDim.x);
                S.wq[slot] = nxt < g.nwork ? nxt : -1;
                mbar_arrive(&S.wq_full[slot]);
            }
            mbar_wait(&S.wq_full[slot], (unsigned)((it / kWorkQ) & 1));
            const int wi = S.wq[slot];
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.wq_empty[slot]);
#endif
            if (wi < 0) break;
            const PWork wk = g.work[wi];
            const double* __restrict__ Bmat = wk.kind ? g.Dst : g.Dt;
            const int* __restrict__ clist = (wk.kind ? g.jrow : g.pl_ao) + wk.clist;
            // orientation 2 of a K block contracts over (r, ix) jointly: kappa = r * nX + ix is contiguous in storage
            const bool k2 = !wk.kind && wk.orient == 2;
            const int npass = (!wk.kind && wk.orient == 1) ? wk.nY : 1;
            for (int t = 0; t < wk.ntiles; ++t) {
                const int lc = g.tiles[wk.tile0 + t] * (k2 ? wk.nX : 1);
                const int nch = (lc + kKC - 1) / kKC;
                const int nrows_t = min(kMT, wk.nrows - t * kMT);
                // orientation 2: producer thread pt gathers row t*128 + pt of the tile (16 consecutive doubles per chunk)
                long long rowbase = -1;
                if (wk.orient == 2 && pt < nrows_t) {
                    const int m = t * kMT + pt;
                    rowbase = wk.kind ? (long long)m * wk.lda : ((long long)(m % wk.nY) * wk.Lc + m / wk.nY) * wk.lda;
                }
                for (int cb = 0; cb < g.ncolblk; ++cb) {
                    const int n0 = cb * 32 * TN;
                    for (int ip = 0; ip < npass; ++ip) {
                        const double* __restrict__ Ab = g.ring + wk.off + (long long)ip * wk.Lc * wk.lda;
                        // B row of contraction index c: orientation 1: D[c_ao][y0 + iy];  2: D[r_ao][x0 + ix];  J: Ds[pair]
                        const int bfix = wk.y0 + ip;
                        for (int ch = 0; ch < nch; ++ch, ++gch) {
                            const int st = gch % kStages;
                            if (gch >= kStages) mbar_wait(&S.empty[st], (unsigned)((gch / kStages - 1) & 1));
                            if (wk.orient == 1) {
                                // A tile: 16 contraction rows of 128 doubles = 1024 pieces of 16 bytes, 8 per thread
#pragma unroll
                                for (int j = 0; j < (kKC * kMT / 2) / kProducerThreads; ++j) {
                                    const int piece = pt + kProducerThreads * j;
                                    const int k = piece >> 6, pc = piece & 63;
                                    const int c = ch * kKC + k;
                                    int bytes = (nrows_t - 2 * pc) * 8;
                                    bytes = (c < lc) ? max(0, min(16, bytes)) : 0;
                                    const double* src = bytes ? (Ab + (long long)c * wk.lda + t * kMT + 2 * pc) : g.ring;
                                    const unsigned sa = (unsigned)__cvta_generic_to_shared(&S.A[st][k * kMTP + 2 * pc]);
                                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(src), "r"(bytes));
                                }
                            } else {
#pragma unroll
                                for (int k2i = 0; k2i < kKC / 2; ++k2i) {       // this thread's row: 8 pieces of 16 bytes
                                    const int c = ch * kKC + 2 * k2i;
                                    const int bytes = (rowbase >= 0) ? max(0, min(16, (lc - c) * 8)) : 0;
                                    const double* src = bytes ? (Ab + rowbase + c) : g.ring;
                                    const unsigned sa = (unsigned)__cvta_generic_to_shared(&S.A[st][pt * kRowPitch + 2 * k2i]);
                                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(src), "r"(bytes));
                                }
                            }
                            // B tile: kKC gathered density rows of 32 TN doubles; warp pw copies rows pw, pw+4, ...
#pragma unroll
                            for (int h = 0; h < kKC / kProducerWarps; ++h) {
                                const int k = pw + kProducerWarps * h, c = ch * kKC + k;
                                const bool ok = c < lc;
                                long long brow = 0;
                                if (ok) {
                                    if (wk.kind) brow = (long long)clist[c];
                                    else if (k2) brow = (long long)clist[c / wk.nX] * N + wk.x0 + c % wk.nX;
                                    else brow = (long long)clist[c] * N + bfix;
                                }
                                const double* src = Bmat + brow * nDp + n0;
                                for (int pc = lane; pc < 16 * TN; pc += 32)
                                    cp_async16(&S.B[st][k][pc * 2], src + (ok ? pc * 2 : 0), ok);
                            }
                            mbar_arrive_on_cp_async(&S.full[st]);
                        }
                    }
                }
            }
        }
        return;
    }

    // ===================== consumer warpgroups =====================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;\n");
    constexpr bool kWide = (TN <= 5);              // 8 x 2TN thread tile (LDS.128 operands); TN = 6: 16 x TN tile
    constexpr int kRows = kWide ? 8 : kTM;
    constexpr int kCols = kWide ? 2 * TN : TN;
    const int wrow = w * kTM;
    const int trow = kWide ? wrow + (lane >> 4) * 8 : wrow;
    const int l16 = lane & 15;
    for (int it = 0;; ++it) {
        const int slot = it % kWorkQ;
#ifdef LTJK_NOQ
        const int wi0 = (int)(blockIdx.x + it * gridDim.x);
        const int wi = wi0 < g.nwork ? wi0 : -1;
#else
        mbar_wait(&S.wq_full[slot], (unsigned)((it / kWorkQ) & 1));
        const int wi = S.wq[slot];
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.wq_empty[slot]);
#endif
        if (wi < 0) break;
        const PWork wk = g.work[wi];
        double* __restrict__ Out = wk.kind ? g.Jt : g.Kt;
        const int* __restrict__ rlist = (wk.kind ? g.jrow : g.pl_ao) + wk.rlist;
        for (int t = 0; t < wk.ntiles; ++t) {
            const bool k2 = !wk.kind && wk.orient == 2;
            const int lc = g.tiles[wk.tile0 + t] * (k2 ? wk.nX : 1);
            // one accumulation over all passes (components of Y in orientation 1)
            const int nch = ((lc + kKC - 1) / kKC) * ((!wk.kind && wk.orient == 1) ? wk.nY : 1);
            if (nch == 0) continue;
            const bool warp_active = t * kMT + wrow < wk.nrows;
            // output rows of this thread: looked up before the contraction so that the flush does not wait on them
            int orow[kRows];
#pragma unroll
            for (int r = 0; r < kRows; ++r) {
                const int m = t * kMT + trow + r;
                orow[r] = -1;
                if (m < wk.nrows) {
                    if (wk.kind) orow[r] = rlist[m];
                    else if (wk.orient == 1) orow[r] = (wk.x0 + m % wk.nX) * N + rlist[m / wk.nX];     // K[x][r]
                    else orow[r] = (wk.y0 + m % wk.nY) * N + rlist[m / wk.nY];                          // K[y][c]
                }
            }
            for (int cb = 0; cb < g.ncolblk; ++cb) {
                const int n0 = cb * 32 * TN;
                double acc[kRows][kCols];
#pragma unroll
                for (int r = 0; r < kRows; ++r)
#pragma unroll
                    for (int c2 = 0; c2 < kCols; ++c2) acc[r][c2] = 0.0;
                for (int q = 0; q < nch; ++q, ++gch) {
                    const int st = gch % kStages;
                    mbar_wait(&S.full[st], (unsigned)((gch / kStages) & 1));
                    if (warp_active && wk.orient == 1) {
#pragma unroll
                        for (int k = 0; k < kKC; ++k) {
                            const double2* ap = reinterpret_cast<const double2*>(&S.A[st][k * kMTP + trow]);
                            double a[kRows];
#pragma unroll
                            for (int r = 0; r < kRows / 2; ++r) { const double2 v = ap[r]; a[2 * r] = v.x; a[2 * r + 1] = v.y; }
                            double b[kCols];
                            if constexpr (kWide) {
#pragma unroll
                                for (int c2 = 0; c2 < TN; ++c2) {
                                    const double2 v = *reinterpret_cast<const double2*>(&S.B[st][k][2 * l16 + 32 * c2]);
                                    b[2 * c2] = v.x; b[2 * c2 + 1] = v.y;
                                }
                            } else {
#pragma unroll
                                for (int c2 = 0; c2 < TN; ++c2) b[c2] = S.B[st][k][lane + 32 * c2];
                            }
#pragma unroll
                            for (int r = 0; r < kRows; ++r)
#pragma unroll
                                for (int c2 = 0; c2 < kCols; ++c2) acc[r][c2] = fma(a[r], b[c2], acc[r][c2]);
                        }
                    } else if (warp_active) {
                        // orientation 2: row-major tile, two contraction steps per 16-byte operand load
#pragma unroll
                        for (int k = 0; k < kKC; k += 2) {
                            double a0[kRows], a1[kRows];
#pragma unroll
                            for (int r = 0; r < kRows; ++r) {
                                const double2 v = *reinterpret_cast<const double2*>(&S.A[st][(trow + r) * kRowPitch + k]);
                                a0[r] = v.x; a1[r] = v.y;
                            }
#pragma unroll
                            for (int kk = 0; kk < 2; ++kk) {
                                double b[kCols];
                                if constexpr (kWide) {
#pragma unroll
                                    for (int c2 = 0; c2 < TN; ++c2) {
                                        const double2 v = *reinterpret_cast<const double2*>(&S.B[st][k + kk][2 * l16 + 32 * c2]);
                                        b[2 * c2] = v.x; b[2 * c2 + 1] = v.y;
                                    }
                                } else {
#pragma unroll
                                    for (int c2 = 0; c2 < TN; ++c2) b[c2] = S.B[st][k + kk][lane + 32 * c2];
                                }
#pragma unroll
                                for (int r = 0; r < kRows; ++r)
#pragma unroll
                                    for (int c2 = 0; c2 < kCols; ++c2)
                                        acc[r][c2] = fma(kk ? a1[r] : a0[r], b[c2], acc[r][c2]);
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&S.empty[st]);
                }
                if (warp_active) {
#pragma unroll
                    for (int r = 0; r < kRows; ++r) {
                        if (orow[r] >= 0) {
                            if constexpr (kWide) {
                                double* o = Out + (long long)orow[r] * nDp + n0 + 2 * l16;
#pragma unroll
                                for (int c2 = 0; c2 < TN; ++c2) {
                                    atomicAdd(o + 32 * c2, acc[r][2 * c2]);
                                    atomicAdd(o + 32 * c2 + 1, acc[r][2 * c2 + 1]);
                                }
                            } else {
                                double* o = Out + (long long)orow[r] * nDp + n0 + lane;
#pragma unroll
                                for (int c2 = 0; c2 < TN; ++c2) atomicAdd(o + 32 * c2, acc[r][c2]);
                            }
                        }
                    }
                }
            }
        }
    }
}

template <int TN>
static int launch_pdigest_tn(ltjk_ctx* c, PDigestArgs& g)
{
    const size_t smem = sizeof(PDigestSmem<TN>);
    LTJK_CUDA(c, cudaFuncSetAttribute(pdigest_kernel<TN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->device);
    const int grid = (int)std::min<long long>(g.nwork, nsm);      // persistent: one CTA per SM, dynamic work queue
    pdigest_kernel<TN><<<grid, kDigestThreads, smem, c->stream>>>(g);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

int launch_pdigest(ltjk_ctx* c, const PChunk& ch, int nDp, bool doJ, bool doK)
{
    const long long first = ch.work0 + (doJ ? 0 : ch.nworkJ);
    const int nwork = (doJ ? ch.nworkJ : 0) + (doK ? ch.nworkK : 0);
    if (nwork == 0) return LTJK_OK;
    PDigestArgs g;
    g.work = c->d_pwork + first; g.tiles = c->d_ptile; g.pl_ao = c->pl.pl_ao; g.jrow = c->d_jrow;
    g.ring = c->d_pring + (size_t)ch.buf * c->pring_half;
    g.Dt = c->Dt; g.Dst = c->Dst; g.Jt = c->Jt; g.Kt = c->Kt;
    g.nDp = nDp; g.N = c->nao; g.nwork = nwork;
    g.counter = c->d_pcounter + c->pcounter_next++;
    if (getenv("LTJK_PD_STATIC")) g.counter = nullptr;
    int TN, nb;
    digest_colblocks(nDp, 2, &TN, &nb);
    if (nb * TN * 32 != nDp) return set_err(c, LTJK_EINVAL, "internal: nDp is not a whole number of column blocks");
    g.ncolblk = nb;
    c->st_launches++;
    switch (TN) {
    case 1: return launch_pdigest_tn<1>(c, g);
    case 2: return launch_pdigest_tn<2>(c, g);
    case 3: return launch_pdigest_tn<3>(c, g);
    case 4: return launch_pdigest_tn<4>(c, g);
    case 5: return launch_pdigest_tn<5>(c, g);
    default: return launch_pdigest_tn<6>(c, g);
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Zero fill.  The digestion reads, for every row tile, the contraction prefix of the tile's strongest row; the ERI
// kernels write only unscreened quartets (Q_xc Q_yr >= tau).  The entries in between -- row m, contraction index in
// [cut(m), prefix(tile)) with cut(m) = #{c : Q_xc >= tau / Q_row(m)} -- are screened quartets: exact zeros by the
// Schwarz rule (reading A9).  One CTA per work record, threads along the rows (coalesced stores).
struct PZeroArgs {
    const PWork* work;
    const int* tiles;
    const double* pl_q;
    const double* jq;
    double* ring;
    double tau;
    int nwork;
};

__global__ void __launch_bounds__(128) pzero_kernel(const PZeroArgs g)
{
    for (int wi = blockIdx.x; wi < g.nwork; wi += gridDim.x) {
        const PWork wk = g.work[wi];
        const double* __restrict__ qc = (wk.kind ? g.jq : g.pl_q) + wk.clist;
        const double* __restrict__ qr = (wk.kind ? g.jq : g.pl_q) + wk.rlist;
        for (int m0 = 0; m0 < wk.nrows; m0 += blockDim.x) {          // blockDim.x == kDigestRows: one row tile per pass
            const int m = m0 + threadIdx.x;
            const bool live = m < wk.nrows;
            const int lc = g.tiles[wk.tile0 + m0 / kDigestRows];
            int lo = lc;
            if (live) {
                const int rdiv = wk.kind ? 1 : (wk.orient == 1 ? wk.nX : wk.nY);
                const double qrow = qr[m / rdiv];
                int a = 0, hi = lc;                               // first contraction index with Q * Q_row < tau
                while (a < hi) { const int mid = (a + hi) >> 1; if (qc[mid] * qrow >= g.tau) a = mid + 1; else hi = mid; }
                lo = a;
            }
            if (wk.orient == 1) {
                // rows are contiguous in storage: the lanes of a warp walk the contraction index together, so that
                // the stores of one step are adjacent (rows of a warp have nearly the same cut-off: Q-sorted lists)
                int lomin = lo;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) lomin = min(lomin, __shfl_xor_sync(0xffffffffu, lomin, o));
                for (int iy = 0; iy < wk.nY; ++iy) {
                    double* __restrict__ A = g.ring + wk.off + (long long)iy * wk.Lc * wk.lda + m;
                    for (int cidx = lomin; cidx < lc; ++cidx)
                        if (cidx >= lo) A[(long long)cidx * wk.lda] = 0.0;
                }
            } else if (live) {
                if (wk.kind) {
                    double* __restrict__ A = g.ring + wk.off + (long long)m * wk.lda;
                    for (int cidx = lo; cidx < lc; ++cidx) A[cidx] = 0.0;
                } else {
                    double* __restrict__ A = g.ring + wk.off + ((long long)(m % wk.nY) * wk.Lc + m / wk.nY) * wk.lda;
                    for (int cidx = lo * wk.nX; cidx < lc * wk.nX; ++cidx) A[cidx] = 0.0;
                }
            }
        }
    }
}

int launch_pzero(ltjk_ctx* c, const PChunk& ch)
{
    const int nwork = ch.nworkJ + ch.nworkK;
    if (nwork == 0) return LTJK_OK;
    PZeroArgs g;
    g.work = c->d_pwork + ch.work0; g.tiles = c->d_ptile; g.pl_q = c->pl.pl_q; g.jq = c->d_jq;
    g.ring = c->d_pring + (size_t)ch.buf * c->pring_half; g.tau = c->tau; g.nwork = nwork;
    pzero_kernel<<<std::min(nwork, 148 * 16), kDigestRows, 0, c->eri_stream>>>(g);
    LTJK_CUDA(c, cudaGetLastError());
    c->st_launches++;
    return LTJK_OK;
}

}  // namespace ltjk

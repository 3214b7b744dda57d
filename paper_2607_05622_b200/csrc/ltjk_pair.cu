// ltjk_pair.cu -- step a5 for the pair-list (screening-aware) digestion: geometry-frozen partner lists, storage
// blocks, chunks and work records (host), PAPER.md:L176 ("once Schwarz screening is applied"), L336 ("only the
// realised buckets are launched"), L446; SURVEY 8(a) a5 "Q-sorted pairs give a monotone cutoff".
//
// Formulation.  With Q-sorted partner lists the kept quartets Q_xc Q_yr >= tau of
//     K[x,r] += sum_c (xc|yr) D[c,y]                       (Eq. 17 / Eq. 25 with all 8 images, reading A5)
// form a staircase in (rank of c in the list of x, rank of r in the list of y).  Every unique shell quartet is
// evaluated once and stored under each of its eight role assignments (x,c,y,r) in blocks T_{XY}[iy][c][r][ix]
// (X, Y shells; c, r AO ranks inside one shell GROUP each), so that the A operand of the digestion GEMM
// (rows (r,ix), contraction c) is a plain 2-D tile.  J uses Q-sorted unique pair lists:
//     X_J[(ij)] += sum_(kl) w (ij|kl) (D + D^T)[(kl)],  J = X_J + X_J^T   (w = 1/2 per A == B, C == D).
// Shell groups bound the memory: the quartets of (group pair) x (group pair) form one CHUNK whose blocks live in
// one half of a staging ring while they are digested.
#include "ltjk_internal.h"
#include "eri_core.h"
#include <algorithm>
#include <cmath>
#include <numeric>

namespace ltjk {

namespace {

template <class T>
int upload_vec(ltjk_ctx* c, T** dst, const std::vector<T>& src)
{
    if (*dst) { cudaFree(*dst); *dst = nullptr; }
    if (src.empty()) return LTJK_OK;
    LTJK_CUDA(c, cudaMalloc((void**)dst, sizeof(T) * src.size()));
    LTJK_CUDA(c, cudaMemcpyAsync(*dst, src.data(), sizeof(T) * src.size(), cudaMemcpyHostToDevice, c->stream));
    return LTJK_OK;
}

inline int gp_index(int a, int b) { return a >= b ? a * (a + 1) / 2 + b : b * (b + 1) / 2 + a; }
inline long long chunk_index(int P, int Q) { return P >= Q ? (long long)P * (P + 1) / 2 + Q : (long long)Q * (Q + 1) / 2 + P; }

struct HostLists {
    int G = 1, ns = 0;
    std::vector<int> sh_grp, ncomp, ao0;
    std::vector<int> pl_start;          // [ns*G+1] into pl_ao
    std::vector<int> pl_ao;
    std::vector<double> pl_q;           // Q per entry of pl_ao
    std::vector<int> sl_start;          // [ns*G+1] into sl_* (shell-level lists)
    std::vector<int> sl_sh, sl_rank;    // partner shell, AO rank of its first component
    std::vector<double> sl_q;           // Q of the partner, descending
    std::vector<int> pos;               // [ns*ns]
};

// AO count of the partners of list (X,g) with Q * qother >= tau (lists are Q-descending).  The product form is the
// predicate of the ERI kernels and of the zero fill: all three must agree to the last bit.
inline int count_ao(const HostLists& h, int X, int g, double qother, double tau)
{
    const int a = h.sl_start[X * h.G + g], b = h.sl_start[X * h.G + g + 1];
    int lo = a, hi = b;                               // first index with q < thr
    while (lo < hi) { const int mid = (lo + hi) / 2; if (h.sl_q[mid] * qother >= tau) lo = mid + 1; else hi = mid; }
    if (lo == a) return 0;
    return h.sl_rank[lo - 1] + h.ncomp[h.sl_sh[lo - 1]];
}

// Q of the partner that holds AO rank `rank` in list (X,g)
inline double q_at_rank(const HostLists& h, int X, int g, int rank)
{
    const int a = h.sl_start[X * h.G + g], b = h.sl_start[X * h.G + g + 1];
    int lo = a, hi = b;                               // last index with sl_rank <= rank
    while (hi - lo > 1) { const int mid = (lo + hi) / 2; if (h.sl_rank[mid] <= rank) lo = mid; else hi = mid; }
    return h.sl_q[lo];
}

void make_lists(const ltjk_ctx* c, int G, HostLists& h)
{
    const int ns = c->nshell;
    h.G = G; h.ns = ns;
    h.ncomp.resize(ns); h.ao0 = c->sh_ao_int;
    for (int s = 0; s < ns; ++s) h.ncomp[s] = ncart(c->l[c->sh_int2ext[s]]);
    h.sh_grp.resize(ns);
    for (int s = 0; s < ns; ++s) {                    // contiguous groups of about equal AO count
        const long long mid = 2ll * h.ao0[s] + h.ncomp[s];
        h.sh_grp[s] = (int)std::min<long long>(G - 1, mid * G / (2ll * c->nao));
    }
    double qmax = 0.0;
    for (double q : c->Qhost) qmax = std::max(qmax, q);
    h.pl_start.assign((size_t)ns * G + 1, 0);
    h.sl_start.assign((size_t)ns * G + 1, 0);
    h.pl_ao.clear(); h.pl_q.clear(); h.sl_sh.clear(); h.sl_rank.clear(); h.sl_q.clear();
    h.pos.assign((size_t)ns * ns, -1);
    std::vector<int> cand;
    for (int X = 0; X < ns; ++X)
        for (int g = 0; g < G; ++g) {
            cand.clear();
            for (int C = 0; C < ns; ++C)
                if (h.sh_grp[C] == g && c->Qhost[(size_t)X * ns + C] * qmax >= c->tau && c->Qhost[(size_t)X * ns + C] > 0.0)
                    cand.push_back(C);
            std::stable_sort(cand.begin(), cand.end(), [&](int a, int b) {
                return c->Qhost[(size_t)X * ns + a] > c->Qhost[(size_t)X * ns + b];
            });
            int rank = 0;
            for (int C : cand) {
                h.sl_sh.push_back(C); h.sl_rank.push_back(rank); h.sl_q.push_back(c->Qhost[(size_t)X * ns + C]);
                h.pos[(size_t)X * ns + C] = rank;
                for (int k = 0; k < h.ncomp[C]; ++k) { h.pl_ao.push_back(h.ao0[C] + k); h.pl_q.push_back(c->Qhost[(size_t)X * ns + C]); }
                rank += h.ncomp[C];
            }
            h.pl_start[(size_t)X * G + g + 1] = (int)h.pl_ao.size();
            h.sl_start[(size_t)X * G + g + 1] = (int)h.sl_sh.size();
        }
}

}  // namespace

void free_pairlists(ltjk_ctx* c)
{
    PLDev& p = c->pl;
    void* ptrs[] = {p.sh_grp, p.pl_start, p.pl_ao, p.pl_q, c->d_jq, p.pos, p.blk, c->d_pwork, c->d_ptile, c->d_jrow, c->d_ppairs, c->d_pring, c->d_pcounter};
    for (void* q : ptrs) if (q) cudaFree(q);
    p = PLDev();
    c->d_pwork = nullptr; c->d_ptile = nullptr; c->d_jrow = nullptr; c->d_jq = nullptr; c->d_ppairs = nullptr; c->d_pring = nullptr; c->d_pcounter = nullptr; c->pcounter_cap = 0;
    c->pring_half = 0;
    c->pchunks.clear(); c->pp_start.clear(); c->jrow_start.clear();
    c->have_pl = false;
}

int build_pairlists(ltjk_ctx* c)
{
    free_pairlists(c);
    const int ns = c->nshell, N = c->nao;
    const double tau = c->tau;
    size_t freeb = 0, totb = 0;
    LTJK_CUDA(c, cudaMemGetInfo(&freeb, &totb));
    long long budget = c->scratch_bytes > 0 ? c->scratch_bytes : (long long)(0.55 * (double)freeb);
    budget = std::min<long long>(budget, (long long)(0.7 * (double)freeb));

    HostLists h;
    std::vector<PBlock> blk;
    std::vector<long long> chunk_doubles;
    std::vector<PChunk> chunks;
    std::vector<PWork> work;
    std::vector<int> tiles;
    std::vector<std::vector<PWork>> cworkK, cworkJ;
    std::vector<int> jrow;
    std::vector<long long> jrow_start, pp_start;
    std::vector<PPair> ppairs;
    std::vector<double> jq;                                  // Q of every J row (AO-pair level), per group pair
    int G = 1;
    const int kGmax = 8;
    for (G = 1; G <= kGmax; ++G) {
        make_lists(c, G, h);
        const int ngp = G * (G + 1) / 2;
        const long long nchunk = (long long)ngp * (ngp + 1) / 2;
        chunk_doubles.assign(nchunk, 0);
        blk.assign((size_t)ns * ns * G * G, PBlock{-1, 0, 0});
        // ---- K storage blocks: bounding box of the staircase of (X, g2) x (Y, g4)
        for (int X = 0; X < ns; ++X)
            for (int Y = 0; Y < ns; ++Y)
                for (int g2 = 0; g2 < G; ++g2) {
                    const int ca = h.sl_start[X * G + g2], cb = h.sl_start[X * G + g2 + 1];
                    if (ca == cb) continue;
                    const double qcmax = h.sl_q[ca];
                    for (int g4 = 0; g4 < G; ++g4) {
                        const int ra = h.sl_start[Y * G + g4], rb = h.sl_start[Y * G + g4 + 1];
                        if (ra == rb) continue;
                        const double qrmax = h.sl_q[ra];
                        if (qcmax * qrmax < tau) continue;
                        // one block per mirrored pair (X,Y,g2,g4) <-> (Y,X,g4,g2): the mirror image is digested
                        // through orientation 2 of the stored block
                        if (!(X > Y || (X == Y && g2 >= g4))) continue;
                        const int Lc = count_ao(h, X, g2, qrmax, tau), Lr = count_ao(h, Y, g4, qcmax, tau);
                        if (Lc == 0 || Lr == 0) continue;
                        const long long ci = chunk_index(gp_index(h.sh_grp[X], g2), gp_index(h.sh_grp[Y], g4));
                        const int nX = h.ncomp[X], nY = h.ncomp[Y];
                        const long long ldr = ((long long)nX * Lr + 1) & ~1ll;
                        PBlock& b = blk[(((size_t)X * ns + Y) * G + g2) * G + g4];
                        b.off = chunk_doubles[ci]; b.Lc = Lc; b.Lr = Lr;
                        chunk_doubles[ci] += (long long)nY * Lc * ldr;
                    }
                }
        // ---- J row lists per group pair (unique shell pairs A >= B, Q descending) and their storage
        jrow.clear(); jq.clear(); ppairs.clear();
        jrow_start.assign(ngp + 1, 0);
        pp_start.assign((size_t)ngp * 6 + 1, 0);
        struct SP { int A, B, cls; double q; };
        std::vector<std::vector<SP>> gplists(ngp);
        double qmax = 0.0;
        for (double q : c->Qhost) qmax = std::max(qmax, q);
        for (int A = 0; A < ns; ++A)
            for (int B = 0; B <= A; ++B) {
                const double q = c->Qhost[(size_t)A * ns + B];
                if (!(q * qmax >= tau) || q <= 0.0) continue;
                const int la = c->l[c->sh_int2ext[A]], lb = c->l[c->sh_int2ext[B]];   // internal order is l-sorted: la >= lb
                gplists[gp_index(h.sh_grp[A], h.sh_grp[B])].push_back(SP{A, B, la * (la + 1) / 2 + lb, q});
            }
        std::vector<long long> gp_npairs(ngp, 0);
        for (int gp = 0; gp < ngp; ++gp) {
            std::vector<SP>& L = gplists[gp];
            std::stable_sort(L.begin(), L.end(), [](const SP& a, const SP& b) { return a.q > b.q; });
            std::vector<int> joff(L.size());
            long long n = 0;
            for (size_t k = 0; k < L.size(); ++k) {
                joff[k] = (int)n;
                const int na = h.ncomp[L[k].A], nb = h.ncomp[L[k].B];
                for (int i = 0; i < na; ++i)
                    for (int j = 0; j < nb; ++j) {
                        jrow.push_back((h.ao0[L[k].A] + i) * N + h.ao0[L[k].B] + j);
                        jq.push_back(L[k].q);
                    }
                n += na * nb;
            }
            gp_npairs[gp] = n;
            jrow_start[gp + 1] = (long long)jrow.size();
            for (int cls = 0; cls < 6; ++cls) {
                for (size_t k = 0; k < L.size(); ++k)
                    if (L[k].cls == cls) ppairs.push_back(PPair{L[k].A, L[k].B, joff[k], 0, L[k].q});
                pp_start[(size_t)gp * 6 + cls + 1] = (long long)ppairs.size();
            }
        }
        // ---- chunks: J arrays appended after the K blocks
        chunks.clear();
        long long maxchunk = 0;
        for (int P = 0; P < ngp; ++P)
            for (int Q = 0; Q <= P; ++Q) {
                PChunk ch = PChunk();
                ch.gab = P; ch.gcd = Q;
                const long long ci = chunk_index(P, Q);
                long long used = (chunk_doubles[ci] + 1) & ~1ll;
                const long long np = gp_npairs[P], nq = gp_npairs[Q];
                ch.j0_off = -1; ch.j1_off = -1; ch.j0_lda = 0; ch.j1_lda = 0;
                if (np > 0 && nq > 0) {
                    ch.j0_lda = (int)((np + 1) & ~1ll);
                    ch.j0_off = used; used += (long long)ch.j0_lda * nq;           // rows (gab), contraction (gcd)
                    // off-diagonal chunks: rows (gcd) x contraction (gab) is orientation 2 of the same array
                }
                ch.doubles = used;
                maxchunk = std::max(maxchunk, used);
                chunks.push_back(ch);
            }
        long long need = 0;
        {
            int nonempty = 0;
            for (const PChunk& ch : chunks) if (ch.doubles > 0) ++nonempty;
            need = (nonempty > 1 ? 2 : 1) * maxchunk * (long long)sizeof(double);
        }
        if (need <= budget || G == kGmax) break;
    }
    const int ngp = G * (G + 1) / 2;

    // ---- work records and row-tile contraction lengths
    cworkK.assign(chunks.size(), {}); cworkJ.assign(chunks.size(), {});
    tiles.clear();
    auto chunk_pos = [&](int P, int Q) { return (size_t)chunk_index(P, Q); };   // chunks were pushed in this order
    for (int X = 0; X < ns; ++X)
        for (int Y = 0; Y < ns; ++Y)
            for (int g2 = 0; g2 < G; ++g2)
                for (int g4 = 0; g4 < G; ++g4) {
                    const PBlock& b = blk[(((size_t)X * ns + Y) * G + g2) * G + g4];
                    if (b.off < 0) continue;
                    const int nX = h.ncomp[X], nY = h.ncomp[Y];
                    PChunk& ch = chunks[chunk_pos(gp_index(h.sh_grp[X], g2), gp_index(h.sh_grp[Y], g4))];
                    std::vector<PWork>& dst = cworkK[chunk_pos(gp_index(h.sh_grp[X], g2), gp_index(h.sh_grp[Y], g4))];
                    const bool self = (X == Y && g2 == g4);        // its own mirror image: orientation 1 covers it
                    for (int orient = 1; orient <= (self ? 1 : 2); ++orient) {
                        PWork w = PWork();
                        w.off = b.off; w.lda = (int)(((long long)nX * b.Lr + 1) & ~1ll);
                        w.kind = 0; w.orient = orient; w.nY = nY; w.Lc = b.Lc; w.x0 = h.ao0[X]; w.nX = nX; w.y0 = h.ao0[Y];
                        w.tile0 = (int)tiles.size();
                        double cost = 0.0;
                        if (orient == 1) {
                            w.nrows = nX * b.Lr;
                            w.clist = h.pl_start[X * G + g2]; w.rlist = h.pl_start[Y * G + g4];
                            w.ntiles = (w.nrows + kDigestRows - 1) / kDigestRows;
                            for (int t = 0; t < w.ntiles; ++t) {
                                const int r0 = (t * kDigestRows) / nX;         // smallest row rank of the tile = largest Q
                                const int lc = std::min(b.Lc, count_ao(h, X, g2, q_at_rank(h, Y, g4, r0), tau));
                                tiles.push_back(lc);
                                cost += (double)((lc + 15) / 16);
                            }
                            cost *= nY;
                        } else {
                            w.nrows = nY * b.Lc;
                            w.clist = h.pl_start[Y * G + g4]; w.rlist = h.pl_start[X * G + g2];
                            w.ntiles = (w.nrows + kDigestRows - 1) / kDigestRows;
                            for (int t = 0; t < w.ntiles; ++t) {
                                const int c0 = (t * kDigestRows) / nY;
                                const int lr = std::min(b.Lr, count_ao(h, Y, g4, q_at_rank(h, X, g2, c0), tau));
                                tiles.push_back(lr);
                                cost += (double)((lr * nX + 15) / 16);     // contraction over (r, ix) jointly
                            }
                        }
                        ch.exec_rows_chunks_K += cost * kDigestRows * 16.0;
                        dst.push_back(w);
                    }
                }
    for (size_t ci = 0; ci < chunks.size(); ++ci) {
        PChunk& ch = chunks[ci];
        if (ch.j0_off < 0) continue;
        // the J array of the chunk: element (contraction q of gcd, row p of gab) at j0[q * lda + p].  Orientation 1:
        // rows p, contraction q;  orientation 2 (off-diagonal chunks only): rows q, contraction p (row-major reads).
        for (int orient = 1; orient <= (ch.gab == ch.gcd ? 1 : 2); ++orient) {
            const int lda = ch.j0_lda;
            const int gpr = orient == 1 ? ch.gab : ch.gcd, gpc = orient == 1 ? ch.gcd : ch.gab;
            const long long nr = jrow_start[gpr + 1] - jrow_start[gpr], ncn = jrow_start[gpc + 1] - jrow_start[gpc];
            const double* qr = jq.data() + jrow_start[gpr];
            const double* qc = jq.data() + jrow_start[gpc];
            // one record per row tile and contraction slice of <= kJSlice columns: J records would otherwise be the
            // long pole of the launch (a row tile contracts over every significant pair of the other side)
            const long long kJSlice = 2048;
            for (long long m0 = 0; m0 < nr; m0 += kDigestRows) {
                const double qrow = qr[m0];
                long long lo = 0, hi = ncn;                               // first contraction index with q * qrow < tau
                while (lo < hi) { const long long mid = (lo + hi) / 2; if (qc[mid] * qrow >= tau) lo = mid + 1; else hi = mid; }
                for (long long c0 = 0; c0 < lo; c0 += kJSlice) {
                    PWork w = PWork();
                    w.off = orient == 1 ? ch.j0_off + m0 + c0 * lda : ch.j0_off + m0 * lda + c0;
                    w.lda = lda;
                    w.nrows = (int)std::min<long long>(kDigestRows, nr - m0);
                    w.kind = 1; w.orient = orient; w.nY = 1; w.Lc = 0; w.x0 = 0; w.nX = 1; w.y0 = 0;
                    w.clist = (int)(jrow_start[gpc] + c0); w.rlist = (int)(jrow_start[gpr] + m0);
                    w.tile0 = (int)tiles.size();
                    w.ntiles = 1;
                    const long long len = std::min(kJSlice, lo - c0);
                    tiles.push_back((int)len);
                    ch.exec_rows_chunks_J += (double)((len + 15) / 16) * kDigestRows * 16.0;
                    cworkJ[ci].push_back(w);
                }
            }
        }
    }
    // longest records first (shorter launch tails), chunks alternate between the ring halves
    work.clear();
    auto cost_of = [&](const PWork& w) {
        double s = 0.0;
        for (int t = 0; t < w.ntiles; ++t) s += (double)((tiles[w.tile0 + t] + 15) / 16);
        return s * (w.kind ? 1 : (w.orient == 1 ? w.nY : w.nX));   // (orientation 2: upper estimate)
    };
    int nbuf = 0;
    long long maxchunk = 0;
    std::vector<PChunk> kept;
    for (size_t ci = 0; ci < chunks.size(); ++ci) {
        PChunk ch = chunks[ci];
        if (cworkK[ci].empty() && cworkJ[ci].empty()) continue;
        for (std::vector<PWork>* v : {&cworkJ[ci], &cworkK[ci]}) {
            std::vector<std::pair<double, size_t>> key(v->size());
            for (size_t k = 0; k < v->size(); ++k) key[k] = {-cost_of((*v)[k]), k};
            std::sort(key.begin(), key.end());
            std::vector<PWork> sorted(v->size());
            for (size_t k = 0; k < v->size(); ++k) sorted[k] = (*v)[key[k].second];
            v->swap(sorted);
        }
        ch.work0 = (long long)work.size();
        ch.nworkJ = (int)cworkJ[ci].size(); ch.nworkK = (int)cworkK[ci].size();
        work.insert(work.end(), cworkJ[ci].begin(), cworkJ[ci].end());
        work.insert(work.end(), cworkK[ci].begin(), cworkK[ci].end());
        ch.buf = (nbuf++) & 1;
        maxchunk = std::max(maxchunk, ch.doubles);
        // shell quartets evaluated for this chunk (statistics)
        kept.push_back(ch);
    }
    c->pchunks = kept;
    c->pring_half = (maxchunk + 1) & ~1ll;
    const long long ring = c->pring_half * (kept.size() > 1 ? 2 : 1);
    if (ring > 0) LTJK_CUDA(c, cudaMalloc(&c->d_pring, sizeof(double) * ring));

    int rc;
    PLDev& p = c->pl;
    p.G = G;
    if ((rc = upload_vec(c, &p.sh_grp, h.sh_grp)) || (rc = upload_vec(c, &p.pl_start, h.pl_start)) ||
        (rc = upload_vec(c, &p.pl_ao, h.pl_ao)) || (rc = upload_vec(c, &p.pl_q, h.pl_q)) || (rc = upload_vec(c, &c->d_jq, jq)) || (rc = upload_vec(c, &p.pos, h.pos)) || (rc = upload_vec(c, &p.blk, blk)) ||
        (rc = upload_vec(c, &c->d_pwork, work)) || (rc = upload_vec(c, &c->d_ptile, tiles)) ||
        (rc = upload_vec(c, &c->d_jrow, jrow)) || (rc = upload_vec(c, &c->d_ppairs, ppairs)))
        return rc;
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    c->pp_start = pp_start; c->jrow_start = jrow_start;
    c->pp_q.resize(ppairs.size());
    for (size_t k = 0; k < ppairs.size(); ++k) c->pp_q[k] = ppairs[k].Q;
    c->pcounter_cap = (int)(2 * kept.size() + 2);
    LTJK_CUDA(c, cudaMalloc(&c->d_pcounter, sizeof(int) * c->pcounter_cap));
    c->have_pl = true;
    (void)ngp;
    return LTJK_OK;
}

}  // namespace ltjk

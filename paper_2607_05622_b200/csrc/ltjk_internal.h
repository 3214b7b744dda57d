// ltjk_internal.h -- context and device-side tables shared by the translation units of libltjk.so.
// Not part of the C ABI (include/ltjk.h is).  See DESIGN.md for the data layout.
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <vector>
#include "../../include/ltjk.h"

namespace ltjk {

constexpr int kNumL = 4;           // angular momenta s, p, d, f (f: SURVEY.md 8(f) N4, looped ERI kernel ltjk_eri_loop.cu)
constexpr int kNumPairCls = kNumL * (kNumL + 1) / 2;   // block-pair classes (la >= lb), la(la+1)/2 + lb
constexpr int kDigestRows = 128;   // output rows per digestion CTA (ltjk_digest.cu) = row-tile height of the work items

// ---- geometry-frozen device tables (built by ltjk_build_shell_pairs, reused by every jk_build) ----------------
// Shells are re-ordered internally by angular momentum and cut into l-homogeneous BLOCKS of 16-24 AOs; block
// pairs (I>=J) are ranked class-major ((ss),(ps),(pp),(ds),(dp),(dd)), so that every canonical block quartet
// (IJ|KL), rank(IJ) >= rank(KL), has bra class >= ket class and every panel is class-homogeneous.
struct DevTables {
    int nshell = 0, nao = 0, nblk = 0, npair = 0;
    int rec_stride = 0;            // doubles per shell-pair record
    double* pair_rec = nullptr;    // [nshell*nshell] records, internal shell order, valid for lA >= lB
    double* schwarz = nullptr;     // [nshell*nshell] Q_AB, internal shell order
    double* boys = nullptr;        // Boys table
    int* sh_ao = nullptr;          // [nshell]   first internal AO of each internal shell
    int* blk_sh0 = nullptr;        // [nblk]     first internal shell
    int* blk_nsh = nullptr;        // [nblk]
    int* blk_ao0 = nullptr;        // [nblk]     first internal AO
    int* blk_nao = nullptr;        // [nblk]
    int* pair_I = nullptr;         // [npair]    block pair of rank r
    int* pair_J = nullptr;
    long long* koff = nullptr;     // [npair+1]  prefix sum of nao(I)*nao(J) over ranks
    int* rank_of = nullptr;        // [nblk*nblk] rank of block pair (I,J), I>=J (else -1)
    int* ao_perm = nullptr;        // [nao]      internal AO -> caller AO
    int* ao_sh = nullptr;          // [nao]      internal AO -> internal shell
};

// A sub-chunk: the panels (IJ|KL) of one bra block pair and a run of ket ranks [r0,r1), contiguous in one half of
// the panel ring starting at `base`.
struct SubChunk {
    int I, J, rIJ;          // bra block pair and its rank
    int r0, r1;             // ket ranks [r0, r1)
    int pad;
    long long base;         // offset (doubles) of the first panel inside the ring half
};

// One digestion work item (32 bytes): a row tile of one output block accumulated over a run of panels.
struct DigestItem {
    unsigned char view;     // 0 JIJ, 1 JKL, 2 KIK, 3 KJK, 4 KIL, 5 KJL
    unsigned char partner;  // K views: 0 -> K[(r1,r2)] with D[(c1,c2)];  1 -> K[(r2,r1)] with D[(c2,c1)]
    unsigned char rowtile;
    unsigned char mult;     // 1, 2 or 4: diagonal block quartets fold identical K images into one (see build_work)
    int a;                  // JIJ/JKL: first ket rank;  KIK/KJK: K;  KIL/KJL: L
    int b;                  // KIK/KJK: first L;  KIL/KJL: first K
    int count;              // panels in the run
    int sub;                // sub-chunk (global index)
    int nchunks;            // contraction chunks (of 16 columns) over the whole run: sum over panels of ceil(nC/16)
    int nnz;                // chunks whose 128 x 16 tile holds at least one unscreened integral (set on the device)
    unsigned maskoff;       // first byte of this item in the chunk mask
};

// A group: consecutive sub-chunks of one bra class that fit one ring half; one ERI launch per ket class and one
// digestion launch per group.
struct Group {
    int sub0, nsub;         // sub-chunks [sub0, sub0+nsub)
    int cb;                 // bra pair class
    int buf;                // ring half
    long long item0;        // first digest item: nitemsJ J-view items, then nitemsK K-view items
    int nitemsJ, nitemsK;
    int maxkets[kNumPairCls]; // per ket class: max number of kets of that class in one sub-chunk
    long long nquartets;    // shell quartets evaluated
    double nints;           // integrals in the panels
};

// ---- pair-list formulation (ltjk_pair.cu, ltjk_pdigest.cu) ---------------------------
// K[x,r] += sum_c (xc|yr) D[c,y] for fixed "major" AOs (x,y): rows r run over the Schwarz-significant partners of y,
// the contraction over the partners of x, both sorted by Q descending, so the kept quartets Q_xc Q_yr >= tau form a
// staircase.  Integrals of one chunk are stored once per role assignment in blocks T_{XY}[iy][c][r][ix] (X, Y shells).
struct PBlock {
    long long off;          // offset (doubles) inside the ring half of the block's chunk; -1 = absent
    int Lc, Lr;             // contraction / row extents in AOs (bounding box of the staircase)
};

struct PLDev {
    int G = 0;              // shell groups
    int* sh_grp = nullptr;  // [nshell]
    int* pl_start = nullptr;// [nshell*G + 1]  start of the partner list (X,g) in pl_ao
    int* pl_ao = nullptr;   // partner AOs (internal ids), Q descending, components of a shell consecutive
    double* pl_q = nullptr; // Schwarz bound Q of (X, partner) for every entry of pl_ao
    int* pos = nullptr;     // [nshell*nshell] AO rank of shell C in list (X, grp(C)), -1 = dead pair
    PBlock* blk = nullptr;  // [((X*nshell+Y)*G+g2)*G+g4]
};

struct PPair {              // one significant shell pair in an ERI launch list
    int A, B;               // internal shells, l_A >= l_B
    int joff;               // first AO pair of (A,B) in the J row list of its group pair
    int pad;
    double Q;
};

struct PWork {              // one digestion work record: a matrix A(c, m) = base[c*lda + m] and its row tiles
    long long off;          // K: block offset;  J: array offset (+ first row already added)
    int lda;
    int nrows;              // rows of this record (K: nX*Lr;  J: <= 8 tiles)
    int kind;               // 0 = K block, 1 = J rows
    int nY;                 // K: components of Y (one pass per component, stride Lc*lda);  J: 1
    int Lc;                 // K: contraction extent of the block (stride between iy slabs = Lc*lda)
    int x0, nX;             // K: first AO of X, components (output row x0 + m % nX)
    int y0;                 // K: first AO of Y (B row = c_ao * N + y0 + iy)
    int clist;              // K: offset of the contraction partner list in pl_ao;  J: offset into jrow (contraction)
    int rlist;              // K: offset of the row partner list in pl_ao;           J: offset into jrow (rows)
    int tile0;              // first entry of this record in the tile-prefix array (contraction length per row tile)
    int ntiles;
    int orient;             // 1: rows contiguous in storage;  2: the mirrored role assignment, A tile gathered.
                            // Orientation 2 (K): rows (c,iy) with c from the partner list of X (rlist), contraction r
                            // from the partner list of Y (clist), one pass per component ix.  (J): rows q, contraction p.
};

struct PChunk {
    int gab, gcd;           // group-pair indices, gab >= gcd
    int buf;                // ring half
    long long doubles;      // storage of the chunk (K blocks + J arrays)
    long long work0;        // first work record: nworkJ J records, then nworkK K records
    int nworkJ, nworkK;
    long long j0_off, j1_off;   // J arrays: rows(gab) x contraction(gcd) and rows(gcd) x contraction(gab) (-1: diagonal chunk)
    int j0_lda, j1_lda;
    double exec_rows_chunks_J, exec_rows_chunks_K;   // sum over items of 128 * 16 * chunks (executed A elements)
    long long nquartets;
};

}  // namespace ltjk

struct ltjk_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    long long scratch_bytes = 0;   // requested cap (0 = default)

    // basis, caller order (host)
    int natom = 0, nshell = 0, nao = 0;
    std::vector<double> xyz, exps, coef;
    std::vector<int> atom, l, nprim, prim_off;
    bool have_basis = false, have_pairs = false;

    // internal ordering (host)
    std::vector<int> sh_int2ext;          // internal shell -> caller shell
    std::vector<int> sh_ao_int;           // internal shell -> first internal AO
    std::vector<int> ao_perm;             // internal AO -> caller AO
    std::vector<int> blk_sh0, blk_nsh, blk_ao0, blk_nao, blk_l;
    std::vector<int> pair_I, pair_J, rank_of;
    std::vector<long long> koff;
    std::vector<double> Qhost;            // internal order [nshell*nshell]
    std::vector<ltjk::SubChunk> subs;
    std::vector<ltjk::Group> groups;
    int cls_start[ltjk::kNumPairCls + 1] = {};          // first rank of each pair class
    int max_nsh_l[ltjk::kNumL] = {};            // max shells per block for each l
    double tau = 0.0;
    long long n_quartets_kept = 0;

    ltjk::DevTables t;
    ltjk::DigestItem* d_items = nullptr;
    ltjk::SubChunk* d_subs = nullptr;
    unsigned char* d_chunkmask = nullptr; // one byte per (item, chunk): bit w = sub-tile of consumer warp w not entirely screened
    long long n_maskbits = 0;
    long long n_items = 0;
    double* d_panel = nullptr;            // integral panel staging ring (two halves)
    long long panel_cap = 0;              // doubles (both halves)
    long long panel_half = 0;             // doubles per half: chunk c lives in half c&1 (ERI of c+1 overlaps digest of c)
    cudaStream_t eri_stream = nullptr;    // stream of the ERI kernels (== stream when timing serialises the phases)
    cudaStream_t own_stream = nullptr;
    cudaEvent_t ev_eri[2] = {nullptr, nullptr}, ev_dig[2] = {nullptr, nullptr}, ev_start = nullptr;

    // pair-list formulation
    ltjk::PLDev pl;
    std::vector<ltjk::PChunk> pchunks;
    ltjk::PWork* d_pwork = nullptr;
    int* d_ptile = nullptr;                // contraction length per row tile
    int* d_jrow = nullptr;                 // per group pair: AO-pair row ids (i*N + j), Q descending
    double* d_jq = nullptr;                // Schwarz bound of every entry of d_jrow
    ltjk::PPair* d_ppairs = nullptr;       // ERI launch lists: per (group pair, class), Q descending
    std::vector<long long> pp_start;       // [ngp*6 + 1] into d_ppairs
    std::vector<long long> jrow_start;     // [ngp + 1] into d_jrow
    std::vector<double> pp_q;              // host copy of the Q column of d_ppairs (launch sizing)
    double* d_pring = nullptr;             // integral staging ring of the pair-list path (one or two halves)
    long long pring_half = 0;              // doubles per half
    int* d_pcounter = nullptr;             // work-stealing cursors, one per digestion launch of a build
    int pcounter_next = 0, pcounter_cap = 0;
    double *gr_xyz = nullptr, *gr_exps = nullptr, *gr_coef = nullptr;   // basis in caller order for ltjk_jk_grad (ltjk_grad.cu)
    int* gr_int = nullptr;
    int gr_cnt[3] = {0, 0, 0};
    int* d_sph_meta = nullptr;            // ltjk_sph.cu: shell tables in the caller's order (built on first use)
    bool debug_poison = false;             // test hook: the staging ring is filled with NaN before every chunk / group
    int cur_nD = 0;                        // density count of the build in progress (un-padded)
    int shard_rank = 0, shard_world = 1;   // quartet-space split of one build over ranks (ltjk_set_quartet_shard)
    double* na_scratch = nullptr;          // device address of the static no-allocation scratch (ltjk_transform.cu), per device
    std::string na_err;                    // why it could not be resolved (reported by the no-allocation entry point)
    bool resident_req = false;             // keep all integral panels of the geometry in HBM across builds (strategy 1)
    bool resident = false, panels_valid = false;
    int digest_mode_req = 0;               // requested: 0 = auto, 1 = block panels (dense), 2 = pair lists
    int digest_mode = 1;                   // in use: 1 = block panels, 2 = pair lists (screening-aware)
    bool have_pl = false;

    // per-build work buffers (grown on demand): density-fastest internal layouts [N][N][nDp]
    double *Dt = nullptr, *Dst = nullptr, *Jt = nullptr, *Kt = nullptr;
    long long work_cap = 0;               // doubles per buffer
    double *hD = nullptr, *hJ = nullptr, *hK = nullptr;   // device staging for jk_build_host
    long long host_cap = 0;

    // stats
    long long st_launches = 0, st_quartets = 0;
    double st_digest_flops = 0.0, st_eri_ms = -1.0, st_digest_ms = -1.0;
    bool timing = false;
};

namespace ltjk {

int set_err(ltjk_ctx* c, int code, const std::string& msg);
#define LTJK_CUDA(c, call)                                                                            \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return ltjk::set_err((c), e_ == cudaErrorMemoryAllocation ? LTJK_ENOMEM : LTJK_ECUDA,     \
                                 std::string(#call) + ": " + cudaGetErrorString(e_));                 \
    } while (0)

// ltjk_api.cu
void free_tables(ltjk_ctx* c);
void free_work(ltjk_ctx* c);
void build_work(ltjk_ctx* c, std::vector<DigestItem>& items);
void digest_colblocks(int nD, int mode, int* TN, int* ncolblk);

// ltjk_eri.cu
int launch_pair_records(ltjk_ctx* c, const double* d_xyz, const int* d_atom, const int* d_l, const int* d_nprim,
                        const int* d_poff, const double* d_exps, const double* d_coef, const int* d_int2ext);
// arguments of the panel-writing ERI kernels (ltjk_eri.cu, ltjk_eri_loop.cu)
struct EriArgs {
    DevTables t;
    const SubChunk* subs;  // sub-chunks of the group; blockIdx.y selects one
    int ca, cb_;           // rank range [ca, cb_) of the launch's ket pair class
    int mJ, mK, mL;        // max shells per block of the launch's l_J, l_K, l_L (thread-index decode)
    int qn;                // mI*mJ*mK*mL
    double tau;
    double* panel;         // ring half
};

int launch_schwarz(ltjk_ctx* c, const int* lrange_host);
int launch_eri_panels(ltjk_ctx* c, const Group& g, int ck);
int launch_eri_single(ltjk_ctx* c, int A, int B, int C, int D, int la, int lb, int lc, int ld, double* d_out, bool looped);
// ltjk_eri_loop.cu: classes with an f shell (looped evaluation, one CTA per contracted quartet)
int launch_eri_panels_loop(ltjk_ctx* c, const EriArgs& g, int la, int lb, int lc, int ld, int maxkets, int nsub);
int launch_eri_single_loop(ltjk_ctx* c, const double* bra, const double* ket, int la, int lb, int lc, int ld, double* d_out);
int launch_schwarz_loop(ltjk_ctx* c, int la, int lb, int a0, int na, int b0, int nb);
int launch_boys_debug(ltjk_ctx* c, int mmax, int n, const double* d_T, double* d_F);

// ltjk_pair.cu, ltjk_peri.cu, ltjk_pdigest.cu: pair-list formulation
int build_pairlists(ltjk_ctx* c);
void free_pairlists(ltjk_ctx* c);
int launch_peri_chunk(ltjk_ctx* c, const PChunk& ch);
int launch_pdigest(ltjk_ctx* c, const PChunk& ch, int nDp, bool doJ, bool doK);
int launch_pzero(ltjk_ctx* c, const PChunk& ch);

// ltjk_digest.cu
int launch_digest(ltjk_ctx* c, const Group& g, int nDp, bool doJ, bool doK);
int launch_chunk_mask(ltjk_ctx* c);
int launch_pack_densities(ltjk_ctx* c, int nD, int nDp, const double* D);
int launch_unpack_results(ltjk_ctx* c, int nD, int nDp, double* J, double* K);
int bench_dfma(ltjk_ctx* c, double* tflops);
int bench_copy(ltjk_ctx* c, double* gbs);

// ltjk_transform.cu
int launch_pseudo_densities(ltjk_ctx* c, int nocc, int nvir, const double* C_occ, const double* C_vir,
                            const double* eps_occ, const double* eps_vir, int nT, const double* T, int ntau,
                            const double* tau_host, double* D_out);

// ltjk_grad.cu
void free_grad(ltjk_ctx* c);
// ltjk_sph.cu
void free_sph(ltjk_ctx* c);
int launch_jk_grad(ltjk_ctx* c, int nP, const double* A, const double* B, double* gJ, double* gK);

int noalloc_setup(ltjk_ctx* c);            // resolves the static scratch of the no-allocation entry point (set-up)
int launch_laplace_fock(ltjk_ctx* c, int nD, const double* J, const double* K, int nmo, const double* C, double* F);
int launch_mo_transform(ltjk_ctx* c, int nD, const double* A, double ca, const double* A2, double ca2, int nmo,
                        const double* C, double* F);
int launch_laplace_accumulate(ltjk_ctx* c, int ntau, int nT, long long nelem, const double* tau_host,
                              const double* w_host, double omega, const double* X, double* Y);

}  // namespace ltjk

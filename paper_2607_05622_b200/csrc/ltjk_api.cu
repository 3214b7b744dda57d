// ltjk_api.cu -- the C ABI of include/ltjk.h: context, basis upload (a1), shell-pair/Schwarz setup and the
// geometry-frozen work lists (a2, a5), and the J/K build driver (a5-a9).
#include "ltjk_internal.h"
#include "eri_core.h"
#include "boys_table.h"
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

namespace ltjk {

int set_err(ltjk_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg;
    return code;
}

// Shells per block for l = 0,1,2,3: 16 / 24 / 24 / 20 AOs.  Output blocks of the digestion then have 256, 384 or 576 rows
// = 2, 3 or 4.5 row tiles of 128: measured tile fill 94 % against 82 % with the first choice (16/15/18, split evenly).
static const int kBlkShells[kNumL] = {16, 8, 4, 2};
static const int kRunMax = 8;                  // panels accumulated in registers before a flush

void free_tables(ltjk_ctx* c)
{
    DevTables& t = c->t;
    void* ptrs[] = {t.pair_rec, t.schwarz, t.sh_ao, t.blk_sh0, t.blk_nsh, t.blk_ao0, t.blk_nao, t.pair_I, t.pair_J,
                    t.koff, t.rank_of, t.ao_perm, t.ao_sh, c->d_items, c->d_subs, c->d_chunkmask, c->d_panel};
    for (void* p : ptrs) if (p) cudaFree(p);
    double* boys = t.boys;
    t = DevTables();
    t.boys = boys;
    c->d_items = nullptr; c->d_subs = nullptr; c->d_chunkmask = nullptr; c->n_maskbits = 0; c->d_panel = nullptr; c->panel_cap = 0; c->panel_half = 0; c->n_items = 0;
    c->have_pairs = false;
    free_pairlists(c);
}

void free_work(ltjk_ctx* c)
{
    void* ptrs[] = {c->Dt, c->Dst, c->Jt, c->Kt, c->hD, c->hJ, c->hK};
    for (void* p : ptrs) if (p) cudaFree(p);
    c->Dt = c->Dst = c->Jt = c->Kt = c->hD = c->hJ = c->hK = nullptr;
    c->work_cap = 0; c->host_cap = 0;
}

static inline int pair_class(int la, int lb) { return la * (la + 1) / 2 + lb; }

// Build the geometry-frozen work lists: sub-chunks (bra block pair x a run of ket ranks), groups of sub-chunks that
// fill one half of the panel ring, and the digestion items of every group.
void build_work(ltjk_ctx* c, std::vector<DigestItem>& items)
{
    const int nblk = (int)c->blk_nao.size(), npair = (int)c->pair_I.size();
    c->subs.clear();
    c->groups.clear();
    items.clear();
    auto rowtiles = [](int rows) { return (rows + kDigestRows - 1) / kDigestRows; };
    auto cls_of = [&](int r) { return pair_class(c->blk_l[c->pair_I[r]], c->blk_l[c->pair_J[r]]); };
    {
        int r = 0;
        for (int cls = 0; cls < kNumPairCls; ++cls) {
            c->cls_start[cls] = r;
            while (r < npair && cls_of(r) == cls) ++r;
        }
        c->cls_start[kNumPairCls] = r;
    }
    std::vector<std::vector<int>> byL(nblk);
    Group g;
    bool open = false;
    long long used = 0;                                   // doubles used in the current ring half
    std::vector<DigestItem> jitems, kitems;
    // contraction chunks of an item (the consumers of the digestion kernel need the count up front)
    auto fill_chunks = [&](DigestItem& it) {
        const SubChunk& sc = c->subs[it.sub];
        const int nI = c->blk_nao[sc.I], nJ = c->blk_nao[sc.J];
        int tot = 0;
        for (int s = 0; s < it.count; ++s) {
            int K, L;
            if (it.view <= 1) { K = c->pair_I[it.a + s]; L = c->pair_J[it.a + s]; }
            else if (it.view <= 3) { K = it.a; L = it.b + s; }
            else { L = it.a; K = it.b + s; }
            const int nK = c->blk_nao[K], nL = c->blk_nao[L];
            int nC;
            switch (it.view) {
            case 0: nC = nK * nL; break;
            case 1: nC = nI * nJ; break;
            case 2: nC = nJ * nL; break;
            case 3: nC = nI * nL; break;
            case 4: nC = nJ * nK; break;
            default: nC = nI * nK; break;
            }
            tot += (nC + 15) / 16;
        }
        it.nchunks = tot;
    };
    auto close_group = [&]() {
        if (!open) return;
        for (DigestItem& it : jitems) fill_chunks(it);
        for (DigestItem& it : kitems) fill_chunks(it);
        auto longer = [](const DigestItem& a, const DigestItem& b) { return a.count > b.count; };
        std::stable_sort(jitems.begin(), jitems.end(), longer);      // longest runs first: shorter launch tail
        std::stable_sort(kitems.begin(), kitems.end(), longer);
        g.item0 = (long long)items.size();
        g.nitemsJ = (int)jitems.size(); g.nitemsK = (int)kitems.size();
        items.insert(items.end(), jitems.begin(), jitems.end());
        items.insert(items.end(), kitems.begin(), kitems.end());
        jitems.clear(); kitems.clear();
        g.buf = c->resident ? 0 : (int)(c->groups.size() & 1);
        c->groups.push_back(g);
        open = false;
    };
    for (int rIJ = 0; rIJ < npair; ++rIJ) {
        const int I = c->pair_I[rIJ], J = c->pair_J[rIJ];
        const int nI = c->blk_nao[I], nJ = c->blk_nao[J];
        const long long nIJ = (long long)nI * nJ;
        const int cb = cls_of(rIJ);
        int r0 = 0;
        while (r0 <= rIJ) {
            if (open && (g.cb != cb || g.nsub >= 60000 || used + nIJ * (c->koff[r0 + 1] - c->koff[r0]) > c->panel_half))
                close_group();
            if (!open) {
                g = Group();
                g.sub0 = (int)c->subs.size(); g.nsub = 0; g.cb = cb; g.nquartets = 0; g.nints = 0.0;
                for (int k = 0; k < kNumPairCls; ++k) g.maxkets[k] = 0;
                if (!c->resident) used = 0;             // resident: every group keeps its own region of the panel store
                open = true;
            }
            int r1 = r0 + 1;
            while (r1 <= rIJ && used + nIJ * (c->koff[r1 + 1] - c->koff[r0]) <= c->panel_half) ++r1;
            SubChunk sc;
            sc.I = I; sc.J = J; sc.rIJ = rIJ; sc.r0 = r0; sc.r1 = r1; sc.pad = 0; sc.base = used;
            const int sub = (int)c->subs.size();
            c->subs.push_back(sc);
            g.nsub++;
            used += nIJ * (c->koff[r1] - c->koff[r0]);
            g.nints += (double)nIJ * (double)(c->koff[r1] - c->koff[r0]);
            for (int k = 0; k < kNumPairCls; ++k) {
                const int a = std::max(r0, c->cls_start[k]), b = std::min(r1, c->cls_start[k + 1]);
                if (b > a) g.maxkets[k] = std::max(g.maxkets[k], b - a);
            }
            for (int r = r0; r < r1; ++r)
                g.nquartets += (long long)c->blk_nsh[I] * c->blk_nsh[J] * c->blk_nsh[c->pair_I[r]] * c->blk_nsh[c->pair_J[r]];
            // ---- J views
            for (int ra = r0; ra < r1; ra += kRunMax) {
                const int cnt = std::min(kRunMax, r1 - ra);
                for (int rt = 0; rt < rowtiles(nI * nJ); ++rt)
                    jitems.push_back(DigestItem{0, 0, (unsigned char)rt, 1, ra, 0, cnt, sub, 0, 0, 0u});
            }
            for (int r = r0; r < r1; ++r) {
                const int nK = c->blk_nao[c->pair_I[r]], nL = c->blk_nao[c->pair_J[r]];
                for (int rt = 0; rt < rowtiles(nK * nL); ++rt)
                    jitems.push_back(DigestItem{1, 0, (unsigned char)rt, 1, r, 0, 1, sub, 0, 0, 0u});
            }
            // ---- K views.  Diagonal block quartets: the panel is symmetric under i<->j when I == J and under
            // k<->l when K == L, which makes pairs of K images identical; they are digested once with weight 2:
            //   I == J : KJK == KIK and KJL == KIL   -> views 3, 5 dropped, views 2, 4 doubled
            //   K == L : KIL == KIK and KJL == KJK   -> views 4, 5 dropped, views 2, 3 doubled
            const bool dI = (I == J);
            auto push_k = [&](int view, int mult, int fixed, int first, int cnt, int rows) {
                for (int partner = 0; partner < 2; ++partner)
                    for (int rt = 0; rt < rowtiles(rows); ++rt)
                        kitems.push_back(DigestItem{(unsigned char)view, (unsigned char)partner, (unsigned char)rt,
                                                    (unsigned char)mult, fixed, first, cnt, sub, 0, 0, 0u});
            };
            // views 2,3: runs of consecutive ranks with the same K (L consecutive by construction); a K == L
            // panel ends the run it would belong to and is digested on its own with the extra weight
            for (int ra = r0; ra < r1;) {
                const int K = c->pair_I[ra];
                const int nK = c->blk_nao[K];
                if (c->pair_J[ra] == K) {                                   // K == L
                    push_k(2, dI ? 4 : 2, K, K, 1, nI * nK);
                    if (!dI) push_k(3, 2, K, K, 1, nJ * nK);
                    ++ra;
                    continue;
                }
                int rb = ra + 1;
                while (rb < r1 && c->pair_I[rb] == K && c->pair_J[rb] == c->pair_J[rb - 1] + 1 && c->pair_J[rb] != K &&
                       rb - ra < kRunMax)
                    ++rb;
                push_k(2, dI ? 2 : 1, K, c->pair_J[ra], rb - ra, nI * nK);
                if (!dI) push_k(3, 1, K, c->pair_J[ra], rb - ra, nJ * nK);
                ra = rb;
            }
            // views 4,5: for each L, runs of consecutive K (K == L panels are covered by views 2,3)
            for (int r = r0; r < r1; ++r)
                if (c->pair_I[r] != c->pair_J[r]) byL[c->pair_J[r]].push_back(c->pair_I[r]);
            for (int L = 0; L < nblk; ++L) {
                std::vector<int>& ks = byL[L];
                if (ks.empty()) continue;
                std::sort(ks.begin(), ks.end());
                const int nL = c->blk_nao[L];
                for (size_t a = 0; a < ks.size();) {
                    size_t b = a + 1;
                    while (b < ks.size() && ks[b] == ks[b - 1] + 1 && (int)(b - a) < kRunMax) ++b;
                    push_k(4, dI ? 2 : 1, L, ks[a], (int)(b - a), nI * nL);
                    if (!dI) push_k(5, 1, L, ks[a], (int)(b - a), nJ * nL);
                    a = b;
                }
                ks.clear();
            }
            r0 = r1;
        }
    }
    close_group();
}

}  // namespace ltjk

using namespace ltjk;

extern "C" {

int ltjk_create(ltjk_ctx** out, int device, void* cuda_stream)
{
    if (!out) return LTJK_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return LTJK_ECUDA;   // no CPU fallback
    if (cudaSetDevice(device) != cudaSuccess) return LTJK_ECUDA;
    ltjk_ctx* c = new (std::nothrow) ltjk_ctx();
    if (!c) return LTJK_ENOMEM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    {   // keep the stream-ordered allocations (transform scratch, host-entry staging) cached between calls
        cudaMemPool_t pool = nullptr;
        if (cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
    }
    if (cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking) != cudaSuccess) { delete c; return LTJK_ECUDA; }
    c->eri_stream = c->own_stream;
    for (int i = 0; i < 2; ++i) {
        cudaEventCreateWithFlags(&c->ev_eri[i], cudaEventDisableTiming);
        cudaEventCreateWithFlags(&c->ev_dig[i], cudaEventDisableTiming);
    }
    cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming);
    std::vector<double> tab = make_boys_table(kBoysNT, kBoysNM);
    if (cudaMalloc(&c->t.boys, sizeof(double) * tab.size()) != cudaSuccess ||
        cudaMemcpy(c->t.boys, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
        if (c->t.boys) cudaFree(c->t.boys);
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_eri[i]); cudaEventDestroy(c->ev_dig[i]); }
        cudaEventDestroy(c->ev_start);
        cudaStreamDestroy(c->own_stream);
        delete c;
        return LTJK_ECUDA;
    }
    noalloc_setup(c);      // set-up only: a failure is kept in the context and reported by the no-allocation entry point
    *out = c;
    return LTJK_OK;
}

int ltjk_destroy(ltjk_ctx* c)
{
    if (!c) return LTJK_EINVAL;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    free_tables(c);
    free_work(c);
    free_grad(c);
    free_sph(c);
    if (c->t.boys) cudaFree(c->t.boys);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_eri[i]); cudaEventDestroy(c->ev_dig[i]); }
    cudaEventDestroy(c->ev_start);
    cudaStreamSynchronize(c->own_stream);
    cudaStreamDestroy(c->own_stream);
    delete c;
    return LTJK_OK;
}

const char* ltjk_last_error(const ltjk_ctx* c) { return c ? c->err.c_str() : "null context"; }

int ltjk_set_scratch_bytes(ltjk_ctx* c, long long bytes)
{
    if (!c || bytes < 0) return LTJK_EINVAL;
    c->scratch_bytes = bytes;
    return LTJK_OK;
}

int ltjk_set_basis(ltjk_ctx* c, int natom, const double* xyz, int nshell, const int* atom, const int* l,
                   const int* nprim, const int* prim_off, const double* exps, const double* coef)
{
    if (!c) return LTJK_EINVAL;
    if (natom <= 0 || nshell <= 0 || !xyz || !atom || !l || !nprim || !prim_off || !exps || !coef)
        return set_err(c, LTJK_EINVAL, "set_basis: null pointer or non-positive size");
    int ntot = 0;
    for (int s = 0; s < nshell; ++s) {
        if (l[s] < 0) return set_err(c, LTJK_EINVAL, "set_basis: negative angular momentum");
        if (l[s] > 3) return set_err(c, LTJK_ELMAX, "set_basis: angular momentum > 3 (kernels are Cartesian s, p, d, f)");
        if (nprim[s] < 1 || nprim[s] > 4) return set_err(c, LTJK_EINVAL, "set_basis: nprim must be 1..4");
        if (atom[s] < 0 || atom[s] >= natom || prim_off[s] < 0) return set_err(c, LTJK_EINVAL, "set_basis: bad atom/prim_off");
        ntot = std::max(ntot, prim_off[s] + nprim[s]);
    }
    for (int i = 0; i < ntot; ++i)
        if (!(exps[i] > 0.0)) return set_err(c, LTJK_EINVAL, "set_basis: exponents must be positive");
    cudaSetDevice(c->device);
    free_tables(c);
    free_grad(c);
    free_sph(c);
    c->natom = natom; c->nshell = nshell;
    c->xyz.assign(xyz, xyz + 3 * natom);
    c->atom.assign(atom, atom + nshell); c->l.assign(l, l + nshell);
    c->nprim.assign(nprim, nprim + nshell); c->prim_off.assign(prim_off, prim_off + nshell);
    c->exps.assign(exps, exps + ntot); c->coef.assign(coef, coef + ntot);

    // caller AO offsets
    std::vector<int> ao_ext(nshell + 1, 0);
    for (int s = 0; s < nshell; ++s) ao_ext[s + 1] = ao_ext[s] + ncart(l[s]);
    c->nao = ao_ext[nshell];
    // internal shell order: by l, then by exponent tier (most diffuse primitive, half-octave buckets), then along a
    // Morton curve through the centres.  Blocks cut from this order are compact in space and homogeneous in extent,
    // so that whole block pairs fall below the Schwarz threshold and never enter the work lists (a2/a5).
    c->sh_int2ext.resize(nshell);
    for (int s = 0; s < nshell; ++s) c->sh_int2ext[s] = s;
    {
        double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
        for (int a = 0; a < natom; ++a)
            for (int k = 0; k < 3; ++k) { lo[k] = std::min(lo[k], xyz[3 * a + k]); hi[k] = std::max(hi[k], xyz[3 * a + k]); }
        const double ext = std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2], 1e-9});
        std::vector<unsigned long long> morton(natom);
        for (int a = 0; a < natom; ++a) {
            unsigned long long m = 0;
            unsigned q[3];
            for (int k = 0; k < 3; ++k) q[k] = (unsigned)std::min(1023.0, 1023.0 * (xyz[3 * a + k] - lo[k]) / ext);
            for (int bit = 9; bit >= 0; --bit)
                for (int k = 0; k < 3; ++k) m = (m << 1) | ((q[k] >> bit) & 1u);
            morton[a] = m;
        }
        std::vector<int> tier(nshell);
        for (int s = 0; s < nshell; ++s) {
            double amin = 1e300;
            for (int p = 0; p < nprim[s]; ++p) amin = std::min(amin, exps[prim_off[s] + p]);
            tier[s] = (int)std::floor(2.0 * std::log2(amin) + 0.5);
        }
        std::stable_sort(c->sh_int2ext.begin(), c->sh_int2ext.end(), [&](int a, int b) {
            if (l[a] != l[b]) return l[a] < l[b];
            if (tier[a] != tier[b]) return tier[a] < tier[b];
            return morton[atom[a]] < morton[atom[b]];
        });
    }
    c->sh_ao_int.assign(nshell, 0);
    c->ao_perm.assign(c->nao, 0);
    int ao = 0;
    for (int s = 0; s < nshell; ++s) {
        const int e = c->sh_int2ext[s];
        c->sh_ao_int[s] = ao;
        for (int k = 0; k < ncart(l[e]); ++k) c->ao_perm[ao++] = ao_ext[e] + k;
    }
    // l-homogeneous blocks of fixed size (the last one of each l takes the remainder)
    c->blk_sh0.clear(); c->blk_nsh.clear(); c->blk_ao0.clear(); c->blk_nao.clear(); c->blk_l.clear();
    int s0 = 0;
    for (int ll = 0; ll < kNumL; ++ll) {
        int n = 0;
        while (s0 + n < nshell && l[c->sh_int2ext[s0 + n]] == ll) ++n;
        c->max_nsh_l[ll] = 0;
        if (n == 0) continue;
        const int nb = (n + kBlkShells[ll] - 1) / kBlkShells[ll];
        int done = 0;
        for (int b = 0; b < nb; ++b) {
            const int cnt = std::min(kBlkShells[ll], n - done);   // full blocks, then one remainder block
            c->blk_sh0.push_back(s0 + done); c->blk_nsh.push_back(cnt);
            c->blk_ao0.push_back(c->sh_ao_int[s0 + done]); c->blk_nao.push_back(cnt * ncart(ll));
            c->blk_l.push_back(ll);
            c->max_nsh_l[ll] = std::max(c->max_nsh_l[ll], cnt);
            done += cnt;
        }
        s0 += n;
    }
    c->have_basis = true;
    return LTJK_OK;
}

int ltjk_get_nao(const ltjk_ctx* c, int* nao)
{
    if (!c || !nao) return LTJK_EINVAL;
    if (!c->have_basis) return LTJK_ENOBASIS;
    *nao = c->nao;
    return LTJK_OK;
}

}  // extern "C"

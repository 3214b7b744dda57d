// ltjk_build.cu -- C ABI, second part: shell-pair/Schwarz setup (a2, a5), the J/K build driver (a5-a9),
// the pseudo-density entry (a4), statistics, test hooks and the peak microbenchmarks.
#include "ltjk_internal.h"
#include "eri_core.h"
#include <algorithm>
#include <cmath>
#include <cstring>
#include <initializer_list>

using namespace ltjk;

namespace {

template <class T>
int upload(ltjk_ctx* c, T** dst, const std::vector<T>& src)
{
    if (*dst) { cudaFree(*dst); *dst = nullptr; }
    if (src.empty()) return LTJK_OK;
    LTJK_CUDA(c, cudaMalloc((void**)dst, sizeof(T) * src.size()));
    LTJK_CUDA(c, cudaMemcpyAsync(*dst, src.data(), sizeof(T) * src.size(), cudaMemcpyHostToDevice, c->stream));
    return LTJK_OK;
}

inline int pair_class(int la, int lb) { return la * (la + 1) / 2 + lb; }

int ensure_work(ltjk_ctx* c, int nDp)
{
    const long long need = (long long)c->nao * c->nao * nDp;
    if (need <= c->work_cap) return LTJK_OK;
    double** bufs[] = {&c->Dt, &c->Dst, &c->Jt, &c->Kt};
    for (double** b : bufs) {
        if (*b) { cudaFree(*b); *b = nullptr; }
        c->work_cap = 0;
        LTJK_CUDA(c, cudaMalloc((void**)b, sizeof(double) * need));
    }
    c->work_cap = need;
    return LTJK_OK;
}

// Owner rank of every launch unit (block-panel group or pair-list chunk) for a split over `world` ranks: longest
// processing time first onto the least loaded rank.  A pure function of the geometry-frozen work lists, so every rank
// computes the same assignment without communication; every unit has exactly one owner.
std::vector<int> unit_owners(const std::vector<double>& cost, int world)
{
    std::vector<int> order(cost.size()), owner(cost.size(), 0);
    for (size_t i = 0; i < cost.size(); ++i) order[i] = (int)i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost[a] > cost[b]; });
    std::vector<double> load(std::max(world, 1), 0.0);
    for (int i : order) {
        int best = 0;
        for (int r = 1; r < world; ++r) if (load[r] < load[best]) best = r;
        owner[i] = best;
        load[best] += cost[i];
    }
    return owner;
}

}  // namespace

extern "C" {

int ltjk_build_shell_pairs(ltjk_ctx* c, double schwarz_tau, long long* n_pairs, long long* n_quartets_kept)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "build_shell_pairs: no basis");
    if (!(schwarz_tau >= 0.0)) return set_err(c, LTJK_EINVAL, "build_shell_pairs: negative threshold");
    cudaSetDevice(c->device);
    free_tables(c);
    c->tau = schwarz_tau;
    const int ns = c->nshell;
    DevTables& t = c->t;
    t.nshell = ns; t.nao = c->nao; t.nblk = (int)c->blk_nao.size();
    int maxnp = 1;
    for (int s = 0; s < ns; ++s) maxnp = std::max(maxnp, c->nprim[s]);
    t.rec_stride = kPairHeader + maxnp * maxnp * kPrimStride;

    // ---- a1: basis to the device (temporary, caller order) and a2: pair records + Schwarz bounds
    double *d_xyz = nullptr, *d_exps = nullptr, *d_coef = nullptr;
    int *d_atom = nullptr, *d_l = nullptr, *d_nprim = nullptr, *d_poff = nullptr, *d_i2e = nullptr;
    struct TmpGuard {          // the temporary basis copies are released on every exit path
        void** p[8];
        ~TmpGuard() { for (void** q : p) if (*q) { cudaFree(*q); *q = nullptr; } }
    } guard{{(void**)&d_xyz, (void**)&d_exps, (void**)&d_coef, (void**)&d_atom, (void**)&d_l, (void**)&d_nprim,
             (void**)&d_poff, (void**)&d_i2e}};
    int rc;
    if ((rc = upload(c, &d_xyz, c->xyz)) || (rc = upload(c, &d_exps, c->exps)) || (rc = upload(c, &d_coef, c->coef)) ||
        (rc = upload(c, &d_atom, c->atom)) || (rc = upload(c, &d_l, c->l)) || (rc = upload(c, &d_nprim, c->nprim)) ||
        (rc = upload(c, &d_poff, c->prim_off)) || (rc = upload(c, &d_i2e, c->sh_int2ext)))
        return rc;
    LTJK_CUDA(c, cudaMalloc(&t.pair_rec, sizeof(double) * (size_t)ns * ns * t.rec_stride));
    LTJK_CUDA(c, cudaMalloc(&t.schwarz, sizeof(double) * (size_t)ns * ns));
    LTJK_CUDA(c, cudaMemsetAsync(t.schwarz, 0, sizeof(double) * (size_t)ns * ns, c->stream));
    if ((rc = launch_pair_records(c, d_xyz, d_atom, d_l, d_nprim, d_poff, d_exps, d_coef, d_i2e))) return rc;
    int lrange[kNumL + 1] = {0, 0, 0, 0, ns};
    bool has_f = false;
    for (int s = 0; s < ns; ++s) {
        const int ll = c->l[c->sh_int2ext[s]];
        for (int k = 1; k < kNumL; ++k)
            if (ll < k) lrange[k] = s + 1;
        has_f = has_f || ll == 3;
    }
    if (has_f && c->digest_mode_req == 2)
        return set_err(c, LTJK_ELMAX, "build_shell_pairs: pair-list digestion is built for s, p, d shells; use mode 0 or 1 with f shells");
    if ((rc = launch_schwarz(c, lrange))) return rc;
    c->Qhost.assign((size_t)ns * ns, 0.0);
    LTJK_CUDA(c, cudaMemcpyAsync(c->Qhost.data(), t.schwarz, sizeof(double) * (size_t)ns * ns, cudaMemcpyDeviceToHost,
                                 c->stream));
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    guard.~TmpGuard();      // early release (idempotent: the pointers are nulled)

    // ---- a5: screened quartet count (canonical, shell level): #{(p,q): p >= q, Q_p Q_q >= tau}
    {
        std::vector<double> q;
        q.reserve((size_t)ns * (ns + 1) / 2);
        for (int A = 0; A < ns; ++A)
            for (int B = 0; B <= A; ++B) q.push_back(c->Qhost[(size_t)A * ns + B]);
        std::sort(q.begin(), q.end());
        long long ordered = 0, diag = 0;
        for (double v : q) {
            if (v * v >= schwarz_tau) ++diag;
            // count w in q with v*w >= tau
            size_t lo = 0, hi = q.size();
            while (lo < hi) { const size_t mid = (lo + hi) / 2; if (v * q[mid] >= schwarz_tau) hi = mid; else lo = mid + 1; }
            ordered += (long long)(q.size() - lo);
        }
        c->n_quartets_kept = (ordered + diag) / 2;
    }

    // ---- digestion strategy (include/ltjk.h: ltjk_set_digest_mode).  Automatic: pair lists when fewer than half of the
    // canonical shell quartets survive the Schwarz test (extended molecules: the dense block panels would be mostly
    // zeros), block panels otherwise.
    {
        const double npairs_all = 0.5 * (double)ns * (ns + 1);
        const double kept_frac = (double)c->n_quartets_kept / (0.5 * npairs_all * (npairs_all + 1.0));
        c->digest_mode = c->digest_mode_req ? c->digest_mode_req : (kept_frac < 0.5 && !has_f ? 2 : 1);
    }
    const bool panels = (c->digest_mode == 1);
    c->subs.clear(); c->groups.clear();

    // ---- block pairs ranked class-major, panel offsets
    const int nblk = t.nblk;
    c->pair_I.clear(); c->pair_J.clear();
    c->rank_of.assign((size_t)nblk * nblk, -1);
    // a block pair whose every shell pair has Q_AB * max(Q) < tau can never pass the quartet test: dropped here
    std::vector<double> qblk((size_t)nblk * nblk, 0.0);
    double qmax = 0.0;
    for (int I = 0; I < nblk; ++I)
        for (int J = 0; J <= I; ++J) {
            double m = 0.0;
            for (int a = 0; a < c->blk_nsh[I]; ++a)
                for (int b = 0; b < c->blk_nsh[J]; ++b)
                    m = std::max(m, c->Qhost[(size_t)(c->blk_sh0[I] + a) * ns + c->blk_sh0[J] + b]);
            qblk[(size_t)I * nblk + J] = m;
            qmax = std::max(qmax, m);
        }
    for (int cls = 0; cls < kNumPairCls; ++cls)
        for (int I = 0; I < nblk; ++I)
            for (int J = 0; J <= I; ++J)
                if (pair_class(c->blk_l[I], c->blk_l[J]) == cls && qblk[(size_t)I * nblk + J] * qmax >= schwarz_tau) {
                    c->rank_of[(size_t)I * nblk + J] = (int)c->pair_I.size();
                    c->pair_I.push_back(I); c->pair_J.push_back(J);
                }
    const int npair = (int)c->pair_I.size();
    t.npair = npair;
    c->koff.assign(npair + 1, 0);
    long long maxpanel = 0;
    for (int r = 0; r < npair; ++r) {
        c->koff[r + 1] = c->koff[r] + (long long)c->blk_nao[c->pair_I[r]] * c->blk_nao[c->pair_J[r]];
        maxpanel = std::max(maxpanel, (long long)c->blk_nao[c->pair_I[r]] * c->blk_nao[c->pair_J[r]]);
    }
    maxpanel *= maxpanel;

    // ---- panel staging ring (two halves), never below one panel per half
    size_t freeb = 0, totb = 0;
    LTJK_CUDA(c, cudaMemGetInfo(&freeb, &totb));
    // Default 8 GiB (two 4 GiB halves), at most a quarter of the free memory: measured on B200, launches that fill
    // the GPU matter far more than keeping the panels L2-resident.
    long long bytes = c->scratch_bytes > 0 ? c->scratch_bytes : std::min<long long>(8ll << 30, (long long)(0.25 * (double)freeb));
    bytes = std::min<long long>(bytes, (long long)(0.6 * (double)freeb));
    long long total = c->koff[npair] * c->koff[npair];      // never need more than everything at once
    c->panel_half = std::max<long long>(std::min<long long>(bytes / 16, total), maxpanel);
    c->panel_cap = 2 * c->panel_half;
    // resident panels (ltjk_set_resident): one region per group, all canonical panels = sum_r nIJ(r) * koff[r+1] doubles
    c->resident = false; c->panels_valid = false;
    if (c->resident_req && panels) {
        long long all = 0;
        for (int r = 0; r < npair; ++r) all += (c->koff[r + 1] - c->koff[r]) * c->koff[r + 1];
        if ((double)all * sizeof(double) <= 0.6 * (double)freeb) {
            c->resident = true;
            c->panel_half = std::max<long long>(all, maxpanel);
            c->panel_cap = c->panel_half;
        }
    }
    std::vector<DigestItem> items;
    if (panels) {
        LTJK_CUDA(c, cudaMalloc(&c->d_panel, sizeof(double) * c->panel_cap));
        build_work(c, items);
    }
    c->n_items = (long long)items.size();
    {   // chunk mask layout: partner items of one tile share nothing here; one bit per (item, chunk)
        unsigned long long bits = 0;
        for (DigestItem& it : items) {
            if (bits + (unsigned long long)it.nchunks >= 0xffffffffull)
                return set_err(c, LTJK_ENOMEM, "build_shell_pairs: chunk mask exceeds 2^32 entries");
            it.maskoff = (unsigned)bits; it.nnz = it.nchunks;
            bits += (unsigned long long)it.nchunks;
        }
        c->n_maskbits = (long long)bits;
    }
    std::vector<int> ao_sh(c->nao, 0);
    for (int s = 0; s < ns; ++s) {
        const int n = ncart(c->l[c->sh_int2ext[s]]);
        for (int k = 0; k < n; ++k) ao_sh[c->sh_ao_int[s] + k] = s;
    }
    if ((rc = upload(c, &c->d_items, items)) || (rc = upload(c, &c->d_subs, c->subs)) || (rc = upload(c, &t.sh_ao, c->sh_ao_int)) ||
        (rc = upload(c, &t.blk_sh0, c->blk_sh0)) || (rc = upload(c, &t.blk_nsh, c->blk_nsh)) ||
        (rc = upload(c, &t.blk_ao0, c->blk_ao0)) || (rc = upload(c, &t.blk_nao, c->blk_nao)) ||
        (rc = upload(c, &t.pair_I, c->pair_I)) || (rc = upload(c, &t.pair_J, c->pair_J)) ||
        (rc = upload(c, &t.koff, c->koff)) || (rc = upload(c, &t.rank_of, c->rank_of)) ||
        (rc = upload(c, &t.ao_perm, c->ao_perm)) || (rc = upload(c, &t.ao_sh, ao_sh)))
        return rc;
    if (panels) {
        LTJK_CUDA(c, cudaMalloc(&c->d_chunkmask, (size_t)c->n_maskbits + 16));
        if ((rc = launch_chunk_mask(c))) return rc;
    }
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    if (!panels && (rc = build_pairlists(c))) return rc;
    c->have_pairs = true;
    if (n_pairs) *n_pairs = (long long)ns * (ns + 1) / 2;
    if (n_quartets_kept) *n_quartets_kept = c->n_quartets_kept;
    return LTJK_OK;
}

int ltjk_get_schwarz(ltjk_ctx* c, double* Q_host)
{
    if (!c || !Q_host) return LTJK_EINVAL;
    if (!c->have_pairs) return set_err(c, LTJK_ENOBASIS, "get_schwarz: shell pairs not built");
    const int ns = c->nshell;
    for (int A = 0; A < ns; ++A)
        for (int B = 0; B < ns; ++B)
            Q_host[(size_t)c->sh_int2ext[A] * ns + c->sh_int2ext[B]] = c->Qhost[(size_t)A * ns + B];
    return LTJK_OK;
}

int ltjk_jk_build(ltjk_ctx* c, int nD, const double* D, double* J, double* K)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_pairs) return set_err(c, LTJK_ENOBASIS, "jk_build: shell pairs not built");
    if (nD <= 0 || !D || (!J && !K)) return set_err(c, LTJK_EINVAL, "jk_build: bad arguments");
    cudaSetDevice(c->device);
    int TN, nb;
    digest_colblocks(nD, c->digest_mode, &TN, &nb);
    const int nDp = TN * nb * 32;
    c->cur_nD = nD;
    int rc;
    if ((rc = ensure_work(c, nDp))) return rc;
    c->st_launches = 0; c->st_quartets = 0; c->st_digest_flops = 0.0;
    c->st_eri_ms = c->timing ? 0.0 : -1.0; c->st_digest_ms = c->timing ? 0.0 : -1.0;
    if ((rc = launch_pack_densities(c, nD, nDp, D))) return rc;
    const size_t wbytes = sizeof(double) * (size_t)c->nao * c->nao * nDp;
    if (J) LTJK_CUDA(c, cudaMemsetAsync(c->Jt, 0, wbytes, c->stream));
    if (K) LTJK_CUDA(c, cudaMemsetAsync(c->Kt, 0, wbytes, c->stream));
    cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr;
    struct EvGuard {            // timing events are released on every exit path (early error returns included)
        cudaEvent_t *a, *b, *c;
        ~EvGuard() { for (cudaEvent_t* e : {a, b, c}) if (*e) { cudaEventDestroy(*e); *e = nullptr; } }
    } evguard{&e0, &e1, &e2};
    if (c->timing) { cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&e2); }
    if (c->digest_mode == 2) {
        // pair-list pipeline: per chunk, clear its ring half, generate the integrals of the chunk under all role
        // assignments (eri_stream), digest them (ctx stream); chunk c+1 is generated while chunk c is digested
        c->eri_stream = c->timing ? c->stream : c->own_stream;
        if (!c->timing) {
            LTJK_CUDA(c, cudaEventRecord(c->ev_start, c->stream));
            LTJK_CUDA(c, cudaStreamWaitEvent(c->eri_stream, c->ev_start, 0));
        }
        long long gi = 0;
        c->pcounter_next = 0;
        LTJK_CUDA(c, cudaMemsetAsync(c->d_pcounter, 0, sizeof(int) * c->pcounter_cap, c->stream));
        std::vector<double> cost(c->pchunks.size());
        for (size_t i = 0; i < cost.size(); ++i)
            cost[i] = c->pchunks[i].exec_rows_chunks_J + c->pchunks[i].exec_rows_chunks_K + 4.0 * (double)c->pchunks[i].doubles;
        const std::vector<int> owner = unit_owners(cost, c->shard_world);
        bool used[2] = {false, false};                // ring half holds a chunk whose digestion may still be running
        size_t ui = 0;
        for (const PChunk& ch : c->pchunks) {
            if (owner[ui++] != c->shard_rank) continue;                // another rank's share of the quartet space
            if (!c->timing && used[ch.buf]) LTJK_CUDA(c, cudaStreamWaitEvent(c->eri_stream, c->ev_dig[ch.buf], 0));
            used[ch.buf] = true;
            if (c->timing) cudaEventRecord(e0, c->stream);
            if (c->debug_poison)     // every element the digestion reads must be written by pzero or an ERI kernel
                LTJK_CUDA(c, cudaMemsetAsync(c->d_pring + (size_t)ch.buf * c->pring_half, 0xFF, sizeof(double) * ch.doubles, c->eri_stream));
            if ((rc = launch_pzero(c, ch))) return rc;
            if ((rc = launch_peri_chunk(c, ch))) return rc;
            if (c->timing) cudaEventRecord(e1, c->stream);
            else {
                LTJK_CUDA(c, cudaEventRecord(c->ev_eri[ch.buf], c->eri_stream));
                LTJK_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_eri[ch.buf], 0));
            }
            if ((rc = launch_pdigest(c, ch, nDp, J != nullptr, K != nullptr))) return rc;
            if (!c->timing) LTJK_CUDA(c, cudaEventRecord(c->ev_dig[ch.buf], c->stream));
            ++gi;
            if (c->timing) {
                cudaEventRecord(e2, c->stream);
                cudaEventSynchronize(e2);
                float a = 0.f, b = 0.f;
                cudaEventElapsedTime(&a, e0, e1); cudaEventElapsedTime(&b, e1, e2);
                c->st_eri_ms += a; c->st_digest_ms += b;
            }
            c->st_digest_flops += 2.0 * nDp * ((J ? ch.exec_rows_chunks_J : 0.0) + (K ? ch.exec_rows_chunks_K : 0.0));
        }
        c->st_quartets = c->n_quartets_kept;
        if ((rc = launch_unpack_results(c, nD, nDp, J, K))) return rc;
        return LTJK_OK;
    }

    // Two-stream pipeline over the two halves of the panel ring: ERI(g+1) on eri_stream overlaps digest(g) on
    // the context stream (both are DFMA-bound; the overlap fills launch tails and hides the long single-thread
    // latency of the high-l quartet classes).  Timing mode serialises the two phases on the context stream so
    // that per-phase durations are those of the kernels alone.
    c->eri_stream = c->timing ? c->stream : c->own_stream;
    if (!c->timing) {
        LTJK_CUDA(c, cudaEventRecord(c->ev_start, c->stream));          // everything enqueued before this build
        LTJK_CUDA(c, cudaStreamWaitEvent(c->eri_stream, c->ev_start, 0));
    }
    long long gi = 0;
    std::vector<double> cost(c->groups.size());
    for (size_t i = 0; i < cost.size(); ++i) cost[i] = c->groups[i].nints;
    const std::vector<int> owner = unit_owners(cost, c->shard_world);
    bool used[2] = {false, false};                    // ring half holds a group whose digestion may still be running
    size_t ui = 0;
    for (const Group& gr : c->groups) {
        if (owner[ui++] != c->shard_rank) continue;                    // another rank's share of the quartet space
        if (!c->timing && !c->resident && used[gr.buf]) LTJK_CUDA(c, cudaStreamWaitEvent(c->eri_stream, c->ev_dig[gr.buf], 0));
        used[gr.buf] = true;
        if (c->timing) cudaEventRecord(e0, c->stream);
        if (c->debug_poison && !c->resident)
            LTJK_CUDA(c, cudaMemsetAsync(c->d_panel + (size_t)gr.buf * c->panel_half, 0xFF, sizeof(double) * c->panel_half, c->eri_stream));
        if (!(c->resident && c->panels_valid))
            for (int ck = 0; ck <= gr.cb; ++ck)
                if ((rc = launch_eri_panels(c, gr, ck))) return rc;
        if (c->timing) cudaEventRecord(e1, c->stream);
        else {
            LTJK_CUDA(c, cudaEventRecord(c->ev_eri[gr.buf], c->eri_stream));
            LTJK_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_eri[gr.buf], 0));
        }
        if ((rc = launch_digest(c, gr, nDp, J != nullptr, K != nullptr))) return rc;
        if (!c->timing) LTJK_CUDA(c, cudaEventRecord(c->ev_dig[gr.buf], c->stream));
        ++gi;
        if (c->timing) {
            cudaEventRecord(e2, c->stream);
            cudaEventSynchronize(e2);
            float a = 0.f, b = 0.f;
            cudaEventElapsedTime(&a, e0, e1); cudaEventElapsedTime(&b, e1, e2);
            c->st_eri_ms += a; c->st_digest_ms += b;
        }
        c->st_quartets += gr.nquartets;
        c->st_digest_flops += 2.0 * gr.nints * nDp * ((J ? 2.0 : 0.0) + (K ? 8.0 : 0.0));   // images applied (folded ones included)
    }
    if (c->resident) c->panels_valid = true;            // the panels of this geometry stay in HBM for the next build
    if ((rc = launch_unpack_results(c, nD, nDp, J, K))) return rc;
    return LTJK_OK;
}

int ltjk_jk_build_host(ltjk_ctx* c, int nD, const double* D_host, double* J_host, double* K_host)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_pairs) return set_err(c, LTJK_ENOBASIS, "jk_build_host: shell pairs not built");
    if (nD <= 0 || !D_host || (!J_host && !K_host)) return set_err(c, LTJK_EINVAL, "jk_build_host: bad arguments");
    cudaSetDevice(c->device);
    const long long need = (long long)nD * c->nao * c->nao;
    if (need > c->host_cap) {
        double** bufs[] = {&c->hD, &c->hJ, &c->hK};
        for (double** b : bufs) {
            if (*b) { cudaFree(*b); *b = nullptr; }
            c->host_cap = 0;
            LTJK_CUDA(c, cudaMalloc((void**)b, sizeof(double) * need));
        }
        c->host_cap = need;
    }
    LTJK_CUDA(c, cudaMemcpyAsync(c->hD, D_host, sizeof(double) * need, cudaMemcpyHostToDevice, c->stream));
    const int rc = ltjk_jk_build(c, nD, c->hD, J_host ? c->hJ : nullptr, K_host ? c->hK : nullptr);
    if (rc) return rc;
    if (J_host) LTJK_CUDA(c, cudaMemcpyAsync(J_host, c->hJ, sizeof(double) * need, cudaMemcpyDeviceToHost, c->stream));
    if (K_host) LTJK_CUDA(c, cudaMemcpyAsync(K_host, c->hK, sizeof(double) * need, cudaMemcpyDeviceToHost, c->stream));
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    return LTJK_OK;
}

int ltjk_build_pseudo_densities(ltjk_ctx* c, int nocc, int nvir, const double* C_occ, const double* C_vir,
                                const double* eps_occ, const double* eps_vir, int nT, const double* T, int ntau,
                                const double* tau_host, double* D_out)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "build_pseudo_densities: no basis");
    if (nocc <= 0 || nvir <= 0 || nT <= 0 || ntau <= 0 || !C_occ || !C_vir || !eps_occ || !eps_vir || !T || !tau_host ||
        !D_out)
        return set_err(c, LTJK_EINVAL, "build_pseudo_densities: bad arguments");
    cudaSetDevice(c->device);
    return launch_pseudo_densities(c, nocc, nvir, C_occ, C_vir, eps_occ, eps_vir, nT, T, ntau, tau_host, D_out);
}

int ltjk_sweep_host(ltjk_ctx* c, int nocc, int nvir, const double* C_occ_host, const double* C_vir_host,
                    const double* eps_occ_host, const double* eps_vir_host, int nT, const double* T_host, int ntau,
                    const double* tau_host, double* J_host, double* K_host)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_pairs) return set_err(c, LTJK_ENOBASIS, "sweep_host: shell pairs not built");
    if (nocc <= 0 || nvir <= 0 || nT <= 0 || ntau <= 0 || !C_occ_host || !C_vir_host || !eps_occ_host || !eps_vir_host ||
        !T_host || !tau_host || (!J_host && !K_host))
        return set_err(c, LTJK_EINVAL, "sweep_host: bad arguments");
    cudaSetDevice(c->device);
    const long long N = c->nao, nD = (long long)ntau * nT;
    const long long need = nD * N * N;
    if (need > c->host_cap) {
        double** bufs[] = {&c->hD, &c->hJ, &c->hK};
        for (double** b : bufs) {
            if (*b) { cudaFree(*b); *b = nullptr; }
            c->host_cap = 0;
            LTJK_CUDA(c, cudaMalloc((void**)b, sizeof(double) * need));
        }
        c->host_cap = need;
    }
    const size_t nin = (size_t)N * nocc + (size_t)N * nvir + nocc + nvir + (size_t)nT * nocc * nvir;
    double* in = nullptr;
    LTJK_CUDA(c, cudaMallocAsync(&in, sizeof(double) * nin, c->stream));
    double *dCo = in, *dCv = dCo + (size_t)N * nocc, *deo = dCv + (size_t)N * nvir, *dev = deo + nocc, *dT = dev + nvir;
    LTJK_CUDA(c, cudaMemcpyAsync(dCo, C_occ_host, sizeof(double) * N * nocc, cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(dCv, C_vir_host, sizeof(double) * N * nvir, cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(deo, eps_occ_host, sizeof(double) * nocc, cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(dev, eps_vir_host, sizeof(double) * nvir, cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(dT, T_host, sizeof(double) * (size_t)nT * nocc * nvir, cudaMemcpyHostToDevice, c->stream));
    int rc = launch_pseudo_densities(c, nocc, nvir, dCo, dCv, deo, dev, nT, dT, ntau, tau_host, c->hD);
    if (!rc) rc = ltjk_jk_build(c, (int)nD, c->hD, J_host ? c->hJ : nullptr, K_host ? c->hK : nullptr);
    cudaFreeAsync(in, c->stream);
    if (rc) return rc;
    if (J_host) LTJK_CUDA(c, cudaMemcpyAsync(J_host, c->hJ, sizeof(double) * need, cudaMemcpyDeviceToHost, c->stream));
    if (K_host) LTJK_CUDA(c, cudaMemcpyAsync(K_host, c->hK, sizeof(double) * need, cudaMemcpyDeviceToHost, c->stream));
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    return LTJK_OK;
}

int ltjk_laplace_fock(ltjk_ctx* c, int nD, const double* J, const double* K, int nmo, const double* C, double* F)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "laplace_fock: no basis");
    if (nD <= 0 || nmo <= 0 || !J || !K || !C || !F) return set_err(c, LTJK_EINVAL, "laplace_fock: bad arguments");
    cudaSetDevice(c->device);
    return launch_laplace_fock(c, nD, J, K, nmo, C, F);
}

int ltjk_pp_ladder(ltjk_ctx* c, int nvir, const double* C_vir, int npair, const double* X, double* L, int chunk)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_pairs) return set_err(c, LTJK_ENOBASIS, "pp_ladder: shell pairs not built");
    if (nvir <= 0 || npair <= 0 || chunk < 0 || !C_vir || !X || !L) return set_err(c, LTJK_EINVAL, "pp_ladder: bad arguments");
    cudaSetDevice(c->device);
    // column chunks of the compound pair index ("column-chunked over the o^2 trial columns at peak
    // device memory O(chunk n_ao^2)"); the default is the batch size the digestion kernels are tuned for
    if (chunk == 0) chunk = 160;
    chunk = std::min(chunk, npair);
    const long long N = c->nao;
    double *D = nullptr, *K = nullptr, *zero = nullptr;
    LTJK_CUDA(c, cudaMallocAsync(&D, sizeof(double) * (size_t)chunk * N * N, c->stream));
    LTJK_CUDA(c, cudaMallocAsync(&K, sizeof(double) * (size_t)chunk * N * N, c->stream));
    LTJK_CUDA(c, cudaMallocAsync(&zero, sizeof(double) * nvir, c->stream));
    LTJK_CUDA(c, cudaMemsetAsync(zero, 0, sizeof(double) * nvir, c->stream));
    const double tau0 = 0.0;
    int rc = LTJK_OK;
    long long launches = 0, quartets = 0;
    double flops = 0.0;
    for (int p0 = 0; p0 < npair && !rc; p0 += chunk) {
        const int n = std::min(chunk, npair - p0);
        const double* Xc = X + (size_t)p0 * nvir * nvir;
        // D_p = C_v X_p C_v^T: the pseudo-density transform at tau = 0 with both coefficient blocks = C_vir
        rc = launch_pseudo_densities(c, nvir, nvir, C_vir, C_vir, zero, zero, n, Xc, 1, &tau0, D);
        if (!rc) rc = ltjk_jk_build(c, n, D, nullptr, K);                       // K-only fast path
        launches += c->st_launches + 3; quartets += c->st_quartets; flops += c->st_digest_flops;
        if (!rc) rc = launch_mo_transform(c, n, K, 1.0, nullptr, 0.0, nvir, C_vir, L + (size_t)p0 * nvir * nvir);
        launches += 3;
    }
    c->st_launches = launches; c->st_quartets = quartets; c->st_digest_flops = flops;
    cudaFreeAsync(D, c->stream); cudaFreeAsync(K, c->stream); cudaFreeAsync(zero, c->stream);
    return rc;
}

int ltjk_laplace_accumulate(ltjk_ctx* c, int ntau, int nT, long long nelem, const double* tau_host,
                            const double* w_host, double omega, const double* X, double* Y)
{
    if (!c) return LTJK_EINVAL;
    if (ntau <= 0 || nT <= 0 || nelem <= 0 || !tau_host || !w_host || !X || !Y)
        return set_err(c, LTJK_EINVAL, "laplace_accumulate: bad arguments");
    cudaSetDevice(c->device);
    return launch_laplace_accumulate(c, ntau, nT, nelem, tau_host, w_host, omega, X, Y);
}

int ltjk_get_stats(const ltjk_ctx* c, long long* n_launches, long long* eri_quartets, double* digest_flops,
                   double* eri_ms, double* digest_ms)
{
    if (!c) return LTJK_EINVAL;
    if (n_launches) *n_launches = c->st_launches;
    if (eri_quartets) *eri_quartets = c->st_quartets;
    if (digest_flops) *digest_flops = c->st_digest_flops;
    if (eri_ms) *eri_ms = c->st_eri_ms;
    if (digest_ms) *digest_ms = c->st_digest_ms;
    return LTJK_OK;
}

int ltjk_set_digest_mode(ltjk_ctx* c, int mode)
{
    if (!c || mode < 0 || mode > 2) return LTJK_EINVAL;
    c->digest_mode_req = mode;
    return LTJK_OK;
}

int ltjk_set_quartet_shard(ltjk_ctx* c, int rank, int world)
{
    if (!c || world < 1 || rank < 0 || rank >= world) return LTJK_EINVAL;
    if (rank != c->shard_rank || world != c->shard_world) c->panels_valid = false;   // resident panels: other units now
    c->shard_rank = rank; c->shard_world = world;
    return LTJK_OK;
}

int ltjk_debug_poison(ltjk_ctx* c, int enable)
{
    if (!c) return LTJK_EINVAL;
    c->debug_poison = enable != 0;
    return LTJK_OK;
}

int ltjk_set_resident(ltjk_ctx* c, int enable)
{
    if (!c) return LTJK_EINVAL;
    c->resident_req = enable != 0;
    return LTJK_OK;
}

int ltjk_get_digest_mode(const ltjk_ctx* c, int* mode)
{
    if (!c || !mode) return LTJK_EINVAL;
    if (!c->have_pairs) return LTJK_ENOBASIS;
    *mode = c->digest_mode;
    return LTJK_OK;
}

int ltjk_set_timing(ltjk_ctx* c, int enable)
{
    if (!c) return LTJK_EINVAL;
    c->timing = enable != 0;
    return LTJK_OK;
}

static int debug_eri_quartet(ltjk_ctx* c, int A, int B, int C, int D, double* out_host, bool looped)
{
    if (!c || !out_host) return LTJK_EINVAL;
    if (!c->have_pairs) return set_err(c, LTJK_ENOBASIS, "debug_eri_quartet: shell pairs not built");
    const int ns = c->nshell;
    if (A < 0 || B < 0 || C < 0 || D < 0 || A >= ns || B >= ns || C >= ns || D >= ns)
        return set_err(c, LTJK_EINVAL, "debug_eri_quartet: shell index out of range");
    cudaSetDevice(c->device);
    // caller -> internal shells, then canonical order (l_a >= l_b, l_c >= l_d, class(ab) >= class(cd))
    std::vector<int> e2i(ns);
    for (int s = 0; s < ns; ++s) e2i[c->sh_int2ext[s]] = s;
    int sh[4] = {A, B, C, D}, pos[4] = {0, 1, 2, 3};   // pos[k] = caller position of canonical slot k
    auto L = [&](int k) { return c->l[sh[pos[k]]]; };
    if (L(0) < L(1)) std::swap(pos[0], pos[1]);
    if (L(2) < L(3)) std::swap(pos[2], pos[3]);
    if (pair_class(L(0), L(1)) < pair_class(L(2), L(3))) { std::swap(pos[0], pos[2]); std::swap(pos[1], pos[3]); }
    int n[4], nc[4];
    for (int k = 0; k < 4; ++k) { nc[k] = ncart(L(k)); n[k] = ncart(c->l[sh[k]]); }
    const int ntot = n[0] * n[1] * n[2] * n[3];
    double* d_out = nullptr;
    LTJK_CUDA(c, cudaMalloc(&d_out, sizeof(double) * ntot));
    const int rc = launch_eri_single(c, e2i[sh[pos[0]]], e2i[sh[pos[1]]], e2i[sh[pos[2]]], e2i[sh[pos[3]]], L(0), L(1),
                                     L(2), L(3), d_out, looped);
    if (rc) { cudaFree(d_out); return rc; }
    std::vector<double> tmp(ntot);
    LTJK_CUDA(c, cudaMemcpyAsync(tmp.data(), d_out, sizeof(double) * ntot, cudaMemcpyDeviceToHost, c->stream));
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    cudaFree(d_out);
    // tmp is indexed by canonical slots; scatter back to caller order
    int idx[4];
    for (idx[0] = 0; idx[0] < nc[0]; ++idx[0])
        for (idx[1] = 0; idx[1] < nc[1]; ++idx[1])
            for (idx[2] = 0; idx[2] < nc[2]; ++idx[2])
                for (idx[3] = 0; idx[3] < nc[3]; ++idx[3]) {
                    int ci[4];
                    for (int k = 0; k < 4; ++k) ci[pos[k]] = idx[k];
                    out_host[((ci[0] * n[1] + ci[1]) * n[2] + ci[2]) * n[3] + ci[3]] =
                        tmp[((idx[0] * nc[1] + idx[1]) * nc[2] + idx[2]) * nc[3] + idx[3]];
                }
    return LTJK_OK;
}

int ltjk_debug_eri_quartet(ltjk_ctx* c, int A, int B, int C, int D, double* out_host)
{
    return debug_eri_quartet(c, A, B, C, D, out_host, false);
}

int ltjk_debug_eri_quartet_looped(ltjk_ctx* c, int A, int B, int C, int D, double* out_host)
{
    return debug_eri_quartet(c, A, B, C, D, out_host, true);
}

int ltjk_debug_boys(ltjk_ctx* c, int mmax, int n, const double* T_host, double* F_host)
{
    if (!c || !T_host || !F_host || n <= 0 || mmax < 0 || mmax > 8) return LTJK_EINVAL;
    cudaSetDevice(c->device);
    double *dT = nullptr, *dF = nullptr;
    LTJK_CUDA(c, cudaMalloc(&dT, sizeof(double) * n));
    LTJK_CUDA(c, cudaMalloc(&dF, sizeof(double) * (size_t)n * (mmax + 1)));
    LTJK_CUDA(c, cudaMemcpyAsync(dT, T_host, sizeof(double) * n, cudaMemcpyHostToDevice, c->stream));
    const int rc = launch_boys_debug(c, mmax, n, dT, dF);
    if (!rc) {
        LTJK_CUDA(c, cudaMemcpyAsync(F_host, dF, sizeof(double) * (size_t)n * (mmax + 1), cudaMemcpyDeviceToHost, c->stream));
        LTJK_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    cudaFree(dT); cudaFree(dF);
    return rc;
}

int ltjk_bench_dfma_peak(ltjk_ctx* c, double* tflops)
{
    if (!c || !tflops) return LTJK_EINVAL;
    cudaSetDevice(c->device);
    return bench_dfma(c, tflops);
}

int ltjk_bench_copy_peak(ltjk_ctx* c, double* gbs)
{
    if (!c || !gbs) return LTJK_EINVAL;
    cudaSetDevice(c->device);
    return bench_copy(c, gbs);
}

}  // extern "C"

// ltjk_eri_loop.cu -- step a7 for the shell classes with an f shell.
//
// "For f shells and above the kernel is instead looped: the ladder structure ... is encoded as integer
// index tables walked by runtime loops, so source size is O(tables) rather than O(nodes)".  The straight-line generated
// code of csrc/gen/ stops at (dd|dd) plus the one-f classes of the derivative builds, 17 of which the value builds use
// (ltjk_eri.cu); every other class with an l = 3 shell comes here.  Angular momenta are run-time
// arguments, the recurrences are loops over small index tables built in shared memory, and -- unlike the paper's
// one-thread-per-quartet mapping, whose per-thread working set ((ff|ff): 10^4 outputs) only fits an HBM scratch slab
// -- one warp (a 32-thread CTA) evaluates one contracted shell quartet with the whole working set in shared memory
// ((ff|ff): 84 KB, two quartets per SM; the classes with one f shell: 2-15 KB, 16 quartets per SM).  The evaluation is the Hermite route (Gaussian product -> Hermite expansion
// coefficients E, Hermite Coulomb integrals R from the Boys function, two short box sums), which needs no horizontal
// stage and whose loops have fixed, table-free trip counts; DESIGN.md section 4c states the difference from the
// paper's looped HGP-OS and the measured cost.
//
//   (ab|cd) = sum_{prim} K_ab K_cd 2 pi^{5/2}/(p q sqrt(p+q))
//             sum_{tuv <= a+b} E^{ab}_{tuv} sum_{t'u'v' <= c+d} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R^0_{t+t',u+u',v+v'}
//
// Output layout, scale factors, zero fill of screened quartets and the thread-index decode are those of
// eri_panel_kernel (ltjk_eri.cu): the digestion kernels do not know which kernel wrote a panel.
#include "ltjk_internal.h"
#include "eri_core.h"

namespace ltjk {

constexpr int kLoopThreads = 32;      // one warp per quartet: every barrier below is a __syncwarp
constexpr int kLoopMinBlocks = 32;    // register cap 64: the kernel is latency-bound, resident quartets per SM matter most

__host__ __device__ inline int tet(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }   // #{(t,u,v): t+u+v <= L}

// Shared-memory carve-up (offsets in doubles), the same function on the host (launch size) and in the kernel.
struct LoopLayout {
    int F, R0, R1, Eb, Ek, H, diag, ints, total;
    int nEb, nEk;      // doubles of one direction's E table
};

__host__ __device__ inline LoopLayout loop_layout(int la, int lb, int lc, int ld)
{
    const int Lab = la + lb, Lcd = lc + ld, L = Lab + Lcd;
    LoopLayout o;
    int n = 0;
    o.F = n; n += 16;                                   // F_0..F_L, L <= 12
    o.R0 = n; n += tet(L);
    o.R1 = n; n += tet(L);
    o.nEb = (la + 1) * (lb + 1) * (Lab + 1);
    o.Eb = n; n += 3 * o.nEb;
    o.nEk = (lc + 1) * (ld + 1) * (Lcd + 1);
    o.Ek = n; n += 3 * o.nEk;
    o.H = n; n += tet(Lab) * ncart(lc) * ncart(ld);
    o.diag = n; n += ncart(la) * ncart(lb);
    o.ints = n;
    const int ni = (L + 1) * (L + 1) + tet(L) + (Lab + 1) * (Lab + 1) + tet(Lab) + 40;
    n += (ni + 1) / 2;
    o.total = n;
    return o;
}

// Boys function with a run-time order: the arithmetic of boys_scaled<L> (eri_core.h), same table.
__device__ void boys_rt(const int L, const double T, const double scale, const double* __restrict__ tab, double* F)
{
    if (T < kBoysTmax) {
        const int i = (int)(T * 8.0 + 0.5);
        const double d = (double)i * 0.125 - T;
        const double* t = tab + i * kBoysNM + L;
        double s = t[kBoysTaylor - 1];
        for (int k = kBoysTaylor - 2; k >= 0; --k) s = t[k] + s * d * (1.0 / (double)(k + 1));
        const double e = exp(-T);
        double f = s;
        F[L] = f * scale;
        for (int m = L; m >= 1; --m) {
            f = (2.0 * T * f + e) * (1.0 / (double)(2 * m - 1));
            F[m - 1] = f * scale;
        }
    } else {
        const double r = 1.0 / T;
        double f = 0.5 * sqrt(3.14159265358979323846 * r);
        F[0] = f * scale;
        const double e = exp(-T), h = 0.5 * r;
        for (int m = 0; m < L; ++m) {
            f = ((double)(2 * m + 1) * f - e) * h;
            F[m + 1] = f * scale;
        }
    }
}

// One direction of the Hermite expansion of a primitive pair, x_A^i x_B^j exp(..) = K sum_t E[i][j][t] Lambda_t:
//   E[0][0][0] = 1 (K_ab sits in the pair record),
//   E[i+1][j][t] = E[i][j][t-1]/(2p) + X_PA E[i][j][t] + (t+1) E[i][j][t+1],  E[i][j+1][t] likewise with X_PB.
// Entry (i,j,t) at ((i*(lb+1)+j)*(la+lb+1) + t).  `alt` multiplies E[..][t] by (-1)^t (ket side of the Coulomb sum).
__device__ void hermite_table(const int la, const int lb, const double p, const double XPA, const double XPB,
                              double* E, const bool alt)
{
    const int nt = la + lb + 1, sj = nt, si = (lb + 1) * nt;
    const double h = 0.5 / p;
    E[0] = 1.0;                        // entries with t > i + j are never written and never read
    for (int i = 0; i <= la; ++i) {
        if (i > 0) {
            const double* lo = E + (i - 1) * si;
            double* hi = E + i * si;
            for (int t = 0; t <= i; ++t) {
                double v = t < i ? XPA * lo[t] : 0.0;
                if (t > 0) v += h * lo[t - 1];
                if (t + 1 <= i - 1) v += (double)(t + 1) * lo[t + 1];
                hi[t] = v;
            }
        }
        for (int j = 1; j <= lb; ++j) {
            const double* lo = E + i * si + (j - 1) * sj;
            double* hi = E + i * si + j * sj;
            for (int t = 0; t <= i + j; ++t) {
                double v = t < i + j ? XPB * lo[t] : 0.0;
                if (t > 0) v += h * lo[t - 1];
                if (t + 1 <= i + j - 1) v += (double)(t + 1) * lo[t + 1];
                hi[t] = v;
            }
        }
    }
    if (alt)
        for (int i = 0; i <= la; ++i)
            for (int j = 0; j <= lb; ++j)
                for (int t = 1; t <= i + j; t += 2) E[i * si + j * sj + t] = -E[i * si + j * sj + t];
}

// One contracted quartet by the whole CTA.  Results: P[a*sI + b*sJ + c*sK + d] = scale * (ab|cd); with `diag` the
// diagonal (ab|ab) only (bra class == ket class), unscaled, left in the shared `diag` array for the caller.
__device__ void loop_quartet(const int la, const int lb, const int lc, const int ld, const double* __restrict__ bra,
                             const double* __restrict__ ket, const double* __restrict__ boys, const bool cut,
                             const double scale, double* __restrict__ P, const int sI, const int sJ, const int sK,
                             const bool diag, double* sm)
{
    const int tid = threadIdx.x;
    const int Lab = la + lb, Lcd = lc + ld, L = Lab + Lcd;
    const LoopLayout o = loop_layout(la, lb, lc, ld);
    double* F = sm + o.F;
    double* Eb = sm + o.Eb;
    double* Ek = sm + o.Ek;
    double* H = sm + o.H;
    double* dg = sm + o.diag;
    int* baseL = reinterpret_cast<int*>(sm + o.ints);       // baseL[t*(L+1)+u] + v = index of R_{tuv}
    int* tuvL = baseL + (L + 1) * (L + 1);                  // inverse map, packed t | u<<8 | v<<16
    int* baseB = tuvL + tet(L);                             // the same for the bra Hermite functions (order <= Lab)
    int* tuvB = baseB + (Lab + 1) * (Lab + 1);
    int* cart = tuvB + tet(Lab);                            // cart[10*slot + comp] = ex | ey<<8 | ez<<16
    const int nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    const int nab = ncart(la) * nb, ncd = nc * nd, nhb = tet(Lab), nhl = tet(L);

    if (tid == 0) {
        int run = 0;
        for (int t = 0; t <= L; ++t)
            for (int u = 0; u <= L - t; ++u) {
                baseL[t * (L + 1) + u] = run;
                for (int v = 0; v <= L - t - u; ++v) tuvL[run++] = t | (u << 8) | (v << 16);
            }
    } else if (tid == 1) {
        int run = 0;
        for (int t = 0; t <= Lab; ++t)
            for (int u = 0; u <= Lab - t; ++u) {
                baseB[t * (Lab + 1) + u] = run;
                for (int v = 0; v <= Lab - t - u; ++v) tuvB[run++] = t | (u << 8) | (v << 16);
            }
    } else if (tid == 2) {
        const int ls[4] = {la, lb, lc, ld};
        for (int s = 0; s < 4; ++s) {
            int n = 0;
            for (int i = ls[s]; i >= 0; --i)                 // xx, xy, xz, yy, yz, zz: the order of the generated classes
                for (int j = ls[s] - i; j >= 0; --j) cart[10 * s + n++] = i | (j << 8) | ((ls[s] - i - j) << 16);
        }
    }
    if (diag) {
        for (int e = tid; e < nab; e += kLoopThreads) dg[e] = 0.0;
    } else {
        for (int e = tid; e < nab * ncd; e += kLoopThreads) {
            const int ab = e / ncd, cd = e - ab * ncd;
            P[(ab / nb) * sI + (ab % nb) * sJ + (cd / nd) * sK + (cd % nd)] = 0.0;
        }
    }
    __syncwarp();

    const int npb = (int)bra[3], npk = (int)ket[3];
    for (int ib = 0; ib < npb; ++ib) {
        const double* bp = bra + kPairHeader + ib * kPrimStride;
        const double p = bp[0];
        bool bra_ready = false;                                    // the bra tables depend on ib only
        for (int ik = 0; ik < npk; ++ik) {
            const double* kp = ket + kPairHeader + ik * kPrimStride;
            const double q = kp[0], pq = p + q;
            const double pref = bp[7] * kp[7] * 34.986836655249725693 /* 2 pi^{5/2} */ / (p * q * sqrt(pq));
            if (cut && fabs(pref) < kPrimCut) continue;            // uniform over the CTA
            const double PQx = bp[1] - kp[1], PQy = bp[2] - kp[2], PQz = bp[3] - kp[3];
            const double rho = p * q / pq;
            if (tid < 6) {                                         // lanes 0-2: bra x, y, z; lanes 3-5: ket (one call: SIMT)
                const bool isket = tid >= 3;
                const int x = isket ? tid - 3 : tid;
                const double* pr = isket ? kp : bp;
                const double* hd = isket ? ket : bra;
                if (isket || !bra_ready)
                    hermite_table(isket ? lc : la, isket ? ld : lb, isket ? q : p, pr[4 + x], pr[4 + x] + hd[x],
                                  isket ? Ek + x * o.nEk : Eb + x * o.nEb, isket);
            } else if (tid == 6) {
                boys_rt(L, rho * (PQx * PQx + PQy * PQy + PQz * PQz), pref, boys, F);
                double f = 1.0;
                for (int n = 0; n <= L; ++n) { F[n] *= f; f *= -2.0 * rho; }      // R^n_{000} = (-2 rho)^n F_n
            }
            bra_ready = true;
            __syncwarp();
            // R^n_{tuv} for n = L .. 0; level n needs level n+1 only:  R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X_PQ R^{n+1}_{tuv}
            for (int n = L; n >= 0; --n) {
                double* cur = sm + ((n & 1) ? o.R1 : o.R0);
                const double* prev = sm + ((n & 1) ? o.R0 : o.R1);
                for (int e = tid; e < nhl; e += kLoopThreads) {
                    const int w = tuvL[e], t = w & 255, u = (w >> 8) & 255, v = w >> 16;
                    if (t + u + v > L - n) continue;
                    double val;
                    if (t + u + v == 0) val = F[n];
                    else if (t > 0) {
                        val = PQx * prev[baseL[(t - 1) * (L + 1) + u] + v];
                        if (t > 1) val += (double)(t - 1) * prev[baseL[(t - 2) * (L + 1) + u] + v];
                    } else if (u > 0) {
                        val = PQy * prev[baseL[u - 1] + v];
                        if (u > 1) val += (double)(u - 1) * prev[baseL[u - 2] + v];
                    } else {
                        val = PQz * prev[baseL[0] + v - 1];
                        if (v > 1) val += (double)(v - 1) * prev[baseL[0] + v - 2];
                    }
                    cur[e] = val;
                }
                __syncwarp();
            }
            const double* R = sm + o.R0;
            // H[tuv][cd] = sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R_{t+t',u+u',v+v'}   (sign folded into Ek)
            for (int e = tid; e < nhb * ncd; e += kLoopThreads) {
                const int hb = e / ncd, cd = e - hb * ncd;
                const int cc = cart[20 + cd / nd], dd = cart[30 + cd % nd];
                const int cx = cc & 255, cy = (cc >> 8) & 255, cz = cc >> 16;
                const int dx = dd & 255, dy = (dd >> 8) & 255, dz = dd >> 16;
                const int w = tuvB[hb], t = w & 255, u = (w >> 8) & 255, v = w >> 16;
                const double* Ex = Ek + (cx * (ld + 1) + dx) * (Lcd + 1);
                const double* Ey = Ek + o.nEk + (cy * (ld + 1) + dy) * (Lcd + 1);
                const double* Ez = Ek + 2 * o.nEk + (cz * (ld + 1) + dz) * (Lcd + 1);
                double s = 0.0;
                for (int t2 = 0; t2 <= cx + dx; ++t2)
                    for (int u2 = 0; u2 <= cy + dy; ++u2) {
                        const double exy = Ex[t2] * Ey[u2];
                        const double* Rr = R + baseL[(t + t2) * (L + 1) + u + u2] + v;
                        double sz = 0.0;
                        for (int v2 = 0; v2 <= cz + dz; ++v2) sz += Ez[v2] * Rr[v2];
                        s += exy * sz;
                    }
                H[e] = s;
            }
            __syncwarp();
            // (ab|cd) += sum_{tuv} E^{ab}_{tuv} H[tuv][cd]
            const int nitems = diag ? nab : nab * ncd;
            for (int e = tid; e < nitems; e += kLoopThreads) {
                const int ab = diag ? e : e / ncd, cd = diag ? e : e - ab * ncd;
                const int aa = cart[ab / nb], bb = cart[10 + ab % nb];
                const int ax = aa & 255, ay = (aa >> 8) & 255, az = aa >> 16;
                const int bx = bb & 255, by = (bb >> 8) & 255, bz = bb >> 16;
                const double* Ex = Eb + (ax * (lb + 1) + bx) * (Lab + 1);
                const double* Ey = Eb + o.nEb + (ay * (lb + 1) + by) * (Lab + 1);
                const double* Ez = Eb + 2 * o.nEb + (az * (lb + 1) + bz) * (Lab + 1);
                double s = 0.0;
                for (int t = 0; t <= ax + bx; ++t)
                    for (int u = 0; u <= ay + by; ++u) {
                        const double exy = Ex[t] * Ey[u];
                        const double* Hr = H + (size_t)(baseB[t * (Lab + 1) + u]) * ncd + cd;
                        double sz = 0.0;
                        for (int v = 0; v <= az + bz; ++v) sz += Ez[v] * Hr[v * ncd];
                        s += exy * sz;
                    }
                if (diag) dg[e] += s;
                else P[(ab / nb) * sI + (ab % nb) * sJ + (cd / nd) * sK + (cd % nd)] += scale * s;
            }
            __syncwarp();
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Panels of one class segment: CTA -> (ket rank r in [ra,rb), shell quartet inside the block quartet).
__global__ void __launch_bounds__(kLoopThreads, kLoopMinBlocks) eri_loop_panel_kernel(const EriArgs g, const int la, const int lb,
                                                                     const int lc, const int ld)
{
    extern __shared__ __align__(16) double loop_sm[];
    const SubChunk sc_ = g.subs[blockIdx.y];
    const int ra = max(sc_.r0, g.ca), rb = min(sc_.r1, g.cb_);
    const long long t = (long long)blockIdx.x;
    const int r = ra + (int)(t / g.qn);
    if (r >= rb) return;
    int q = (int)(t % g.qn);
    const int sd = q % g.mL; q /= g.mL;
    const int sc = q % g.mK; q /= g.mK;
    const int sb = q % g.mJ;
    const int sa = q / g.mJ;
    const DevTables& T = g.t;
    const int I = sc_.I, J = sc_.J, K = T.pair_I[r], Lk = T.pair_J[r];
    if (sa >= T.blk_nsh[I] || sb >= T.blk_nsh[J] || sc >= T.blk_nsh[K] || sd >= T.blk_nsh[Lk]) return;
    const int A = T.blk_sh0[I] + sa, B = T.blk_sh0[J] + sb, C = T.blk_sh0[K] + sc, D = T.blk_sh0[Lk] + sd;
    const int NA = ncart(la), NB = ncart(lb), NC = ncart(lc), ND = ncart(ld);
    const int nJ = T.blk_nao[J], nK = T.blk_nao[K], nL = T.blk_nao[Lk];
    const long long base = sc_.base + (T.koff[r] - T.koff[sc_.r0]) * (long long)(T.blk_nao[I] * nJ);
    double* __restrict__ P = g.panel + base + ((long long)(sa * NA) * nJ + sb * NB) * (nK * nL) + (sc * NC) * nL + sd * ND;
    const int sI = nJ * nK * nL, sJ = nK * nL, sK = nL;

    const double qq = T.schwarz[(size_t)A * T.nshell + B] * T.schwarz[(size_t)C * T.nshell + D];
    if (qq < g.tau) {                                       // the same product test as every other kernel
        for (int e = threadIdx.x; e < NA * NB * NC * ND; e += kLoopThreads) {
            const int d = e % ND, cc = (e / ND) % NC, b = (e / (ND * NC)) % NB, a = e / (ND * NC * NB);
            P[a * sI + b * sJ + cc * sK + d] = 0.0;
        }
        return;
    }
    double scale = 1.0;
    if (I == J) scale *= 0.5;
    if (K == Lk) scale *= 0.5;
    if (r == sc_.rIJ) scale *= 0.5;
    loop_quartet(la, lb, lc, ld, T.pair_rec + ((size_t)A * T.nshell + B) * T.rec_stride,
                 T.pair_rec + ((size_t)C * T.nshell + D) * T.rec_stride, T.boys, true, scale, P, sI, sJ, sK, false, loop_sm);
}

__global__ void __launch_bounds__(kLoopThreads, kLoopMinBlocks) eri_loop_single_kernel(const double* bra, const double* ket,
                                                                      const double* boys, const int la, const int lb,
                                                                      const int lc, const int ld, double* out)
{
    extern __shared__ __align__(16) double loop_sm[];
    const int nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    loop_quartet(la, lb, lc, ld, bra, ket, boys, true, 1.0, out, nb * nc * nd, nc * nd, nd, false, loop_sm);
}

// Schwarz bounds of the pair classes with an f shell: Q_AB = sqrt(max_{ab} |(ab|ab)|), one CTA per shell pair.
__global__ void __launch_bounds__(kLoopThreads, kLoopMinBlocks) schwarz_loop_kernel(const int nshell, const int a0, const int na,
                                                                   const int b0, const int nb,
                                                                   const double* __restrict__ rec, const int rec_stride,
                                                                   const double* __restrict__ boys,
                                                                   double* __restrict__ Q, const int la, const int lb)
{
    extern __shared__ __align__(16) double loop_sm[];
    const int t = blockIdx.x;
    if (t >= na * nb) return;
    const int A = a0 + t / nb, B = b0 + t % nb;
    if (la == lb && B > A) return;
    const double* r = rec + ((size_t)A * nshell + B) * rec_stride;
    loop_quartet(la, lb, la, lb, r, r, boys, false, 1.0, nullptr, 0, 0, 0, true, loop_sm);   // no primitive cut: Q^2 may be tiny
    if (threadIdx.x == 0) {
        const double* dg = loop_sm + loop_layout(la, lb, la, lb).diag;
        double m = 0.0;
        for (int e = 0; e < ncart(la) * ncart(lb); ++e) m = fmax(m, fabs(dg[e]));
        m = sqrt(m);
        Q[(size_t)A * nshell + B] = m;
        Q[(size_t)B * nshell + A] = m;
    }
}

template <typename Kern>
static int loop_smem(ltjk_ctx* c, Kern kern, int la, int lb, int lc, int ld, int* bytes)
{
    *bytes = loop_layout(la, lb, lc, ld).total * (int)sizeof(double);
    if (*bytes > 48 * 1024) LTJK_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, *bytes));
    return LTJK_OK;
}

int launch_eri_panels_loop(ltjk_ctx* c, const EriArgs& g, int la, int lb, int lc, int ld, int maxkets, int nsub)
{
    int smem = 0, rc;
    if ((rc = loop_smem(c, eri_loop_panel_kernel, la, lb, lc, ld, &smem))) return rc;
    const long long nq = (long long)maxkets * g.qn;
    if (nq > 0x7fffffffll) return set_err(c, LTJK_EINVAL, "internal: looped ERI grid too large");
    eri_loop_panel_kernel<<<dim3((unsigned)nq, nsub), kLoopThreads, smem, c->eri_stream>>>(g, la, lb, lc, ld);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

int launch_eri_single_loop(ltjk_ctx* c, const double* bra, const double* ket, int la, int lb, int lc, int ld, double* d_out)
{
    int smem = 0, rc;
    if ((rc = loop_smem(c, eri_loop_single_kernel, la, lb, lc, ld, &smem))) return rc;
    eri_loop_single_kernel<<<1, kLoopThreads, smem, c->stream>>>(bra, ket, c->t.boys, la, lb, lc, ld, d_out);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

int launch_schwarz_loop(ltjk_ctx* c, int la, int lb, int a0, int na, int b0, int nb)
{
    if (na <= 0 || nb <= 0) return LTJK_OK;
    int smem = 0, rc;
    if ((rc = loop_smem(c, schwarz_loop_kernel, la, lb, la, lb, &smem))) return rc;
    schwarz_loop_kernel<<<na * nb, kLoopThreads, smem, c->stream>>>(c->nshell, a0, na, b0, nb, c->t.pair_rec,
                                                                  c->t.rec_stride, c->t.boys, c->t.schwarz, la, lb);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

}  // namespace ltjk

// ltjk_grad.cu -- SURVEY 8(f) N2: derivative (skeleton) builds of PAPER.md:L161 Eq. (18),
//     J^x(A,B) = sum_{mnkr} (mn|kr)^x A_mn B_kr ,     K^x(A,B) = sum_{mnkr} (mk|nr)^x A_mn B_kr ,
// x = a nuclear coordinate, for pairs of general (non-symmetric) AO densities; centre derivatives per PAPER.md:L382-386
// (Eqs. 30-31).  "These derivative builds are the J/K kernel of this work" (L164).
//
// Formulation.  By the product rule (mn|kr)^x has one term per function.  The three terms that do not differentiate the
// first function are brought to first position with (mn|kr) = (nm|kr) = (kr|mn) = (kr|nm), which moves the permutation
// onto the density product:
//     grad[atom(m)] += sum_{nkr} (d m n|kr) G1_{mnkr} ,        G1_{mnkr} = G_{mnkr} + G_{nmkr} + G_{krmn} + G_{krnm} ,
//     Coulomb:  G_{mnkr} = A_mn B_kr        exchange:  G_{mnkr} = A_mk B_nr        (Eq. 18 with (mk|nr) renamed).
// Only unordered ket shell pairs {K,R} are visited; the ket-swapped partner adds G1_{mnrk}.  The derivative of a shell
// of l is a shell of l+1 with primitive coefficients 2 a_p c_p minus i times the shell of l-1 (same centre), so each
// thread evaluates two ordinary contracted quartets with the generated OS/HGP code -- the raised one needs the classes
// (f b|c d) of gen/eri_gen_d1.h -- and contracts them at once: derivative integrals are never stored.
// No screening (every quartet is evaluated) and no prefactors.  First correct version: one thread per
// (M, N, {K,R}); bound by local-memory traffic of the per-thread quartets, see DESIGN.md.
#define LTJK_WITH_D1
#include "ltjk_internal.h"
#include "eri_core.h"
#include <vector>

namespace ltjk {

constexpr int kGradPairs = 4;      // density pairs contracted per launch (accumulators live in registers)

struct GradArgs {
    const double* xyz; const int* atom; const int* nprim; const int* poff; const double* exps; const double* coef;
    const int* ao0;                // first AO (caller order) of every caller shell
    const double* boys;
    const int* shM; const int* shN; const int* shK; const int* shR;     // caller shells of the launch's four l values
    int nM, nN, nK, nR, same;      // same: LC == LD, visit K >= R (list positions) only
    int N, natom, nP;
    const double* A; const double* B;     // [nP][N][N]
    double* gJ; double* gK;               // [nP][natom][3] (either may be null)
};

__host__ __device__ constexpr int pcls(int a, int b) { return a * (a + 1) / 2 + b; }
// position of the Cartesian component x^i y^j z^k in the lexicographic list of degree l = i + j + k
__host__ __device__ constexpr int cidx(int l, int i, int j) { return (l - i) * (l - i + 1) / 2 + (l - i - j); }

// Contracted quartet (S1 S2|S3 S4) for ANY order of angular momenta with L3 >= L4: evaluated in the canonical order of
// the generated classes (first >= second inside the bra, bra class >= ket class); element (c1,c2,c3,c4) is
// tmp[c1*s1 + c2*s2 + c3*s3 + c4*s4].
template <int L1, int L2, int L3, int L4>
struct QAny {
    static constexpr bool swapB = L1 < L2;
    static constexpr int LA = swapB ? L2 : L1, LB = swapB ? L1 : L2;
    static constexpr bool swapBK = pcls(LA, LB) < pcls(L3, L4);
    static constexpr int CA = swapBK ? L3 : LA, CB = swapBK ? L4 : LB, CC = swapBK ? LA : L3, CD = swapBK ? LB : L4;
    static constexpr int sa = ncart(CB) * ncart(CC) * ncart(CD), sb = ncart(CC) * ncart(CD), sc = ncart(CD), sd = 1;
    static constexpr int s1 = swapBK ? (swapB ? sd : sc) : (swapB ? sb : sa);
    static constexpr int s2 = swapBK ? (swapB ? sc : sd) : (swapB ? sa : sb);
    static constexpr int s3 = swapBK ? sa : sc;
    static constexpr int s4 = swapBK ? sb : sd;
    static constexpr int NTOT = ncart(L1) * ncart(L2) * ncart(L3) * ncart(L4);

    // c1: primitive coefficients to use for shell S1 (the caller passes the raised / plain set)
    __device__ static void eval(const GradArgs& g, int S1, const double* c1, int S2, const double* ketrec, double* tmp)
    {
        double rec[kPairHeader + kMaxPrimPair * kPrimStride];
        const double* X1 = g.xyz + 3 * g.atom[S1];
        const double* X2 = g.xyz + 3 * g.atom[S2];
        if (swapB)
            build_pair_record(X2, X1, g.nprim[S2], g.exps + g.poff[S2], g.coef + g.poff[S2], g.nprim[S1],
                              g.exps + g.poff[S1], c1, rec);
        else
            build_pair_record(X1, X2, g.nprim[S1], g.exps + g.poff[S1], c1, g.nprim[S2], g.exps + g.poff[S2],
                              g.coef + g.poff[S2], rec);
        if (swapBK) eri_quartet<CA, CB, CC, CD>(ketrec, rec, g.boys, tmp);
        else eri_quartet<CA, CB, CC, CD>(rec, ketrec, g.boys, tmp);
    }
};

template <int LM, int LN, int LC, int LD>
__global__ void __launch_bounds__(64) grad_kernel(const GradArgs g)
{
    constexpr int NM = ncart(LM), NN = ncart(LN), NC = ncart(LC), ND = ncart(LD);
    using QU = QAny<LM + 1, LN, LC, LD>;
    using QD = QAny<(LM > 0 ? LM - 1 : 0), LN, LC, LD>;
    const int M = g.shM[blockIdx.y / g.nN], Nn = g.shN[blockIdx.y % g.nN];
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int ik = (int)(t / g.nR), ir = (int)(t % g.nR);
    const bool active = t < (long long)g.nK * g.nR && !(g.same && ir > ik);
    double gj[kGradPairs][3], gk[kGradPairs][3];
#pragma unroll
    for (int p = 0; p < kGradPairs; ++p)
#pragma unroll
        for (int x = 0; x < 3; ++x) gj[p][x] = gk[p][x] = 0.0;

    if (active) {
        const int K = g.shK[ik], R = g.shR[ir];
        const bool both = (K != R);                 // the ket-swapped partner (mn|rk) is a different ordered quartet
        double ketrec[kPairHeader + kMaxPrimPair * kPrimStride];
        build_pair_record(g.xyz + 3 * g.atom[K], g.xyz + 3 * g.atom[R], g.nprim[K], g.exps + g.poff[K], g.coef + g.poff[K],
                          g.nprim[R], g.exps + g.poff[R], g.coef + g.poff[R], ketrec);
        double cup[4];
        for (int p = 0; p < g.nprim[M]; ++p) cup[p] = 2.0 * g.exps[g.poff[M] + p] * g.coef[g.poff[M] + p];
        double up[QU::NTOT];
        double dn[LM > 0 ? QD::NTOT : 1];
        QU::eval(g, M, cup, Nn, ketrec, up);
        if (LM > 0) QD::eval(g, M, g.coef + g.poff[M], Nn, ketrec, dn);

        const int N = g.N;
        const int aM = g.ao0[M], aN = g.ao0[Nn], aK = g.ao0[K], aR = g.ao0[R];
        int im = 0;
        for (int ei = LM; ei >= 0; --ei)
            for (int ej = LM - ei; ej >= 0; --ej, ++im) {
                const int e[3] = {ei, ej, LM - ei - ej};
                int iu[3], id[3];
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    int f[3] = {e[0], e[1], e[2]};
                    f[x] += 1; iu[x] = cidx(LM + 1, f[0], f[1]);
                    f[x] -= 2; id[x] = (e[x] > 0) ? cidx(LM - 1, f[0], f[1]) : 0;
                }
                const int m = aM + im;
                for (int in = 0; in < NN; ++in) {
                    const int n = aN + in;
                    for (int ic = 0; ic < NC; ++ic) {
                        const int k = aK + ic;
                        for (int id_ = 0; id_ < ND; ++id_) {
                            const int r = aR + id_;
                            double dI[3];
#pragma unroll
                            for (int x = 0; x < 3; ++x) {
                                dI[x] = up[iu[x] * QU::s1 + in * QU::s2 + ic * QU::s3 + id_ * QU::s4];
                                if (LM > 0 && e[x] > 0)
                                    dI[x] -= (double)e[x] * dn[id[x] * QD::s1 + in * QD::s2 + ic * QD::s3 + id_ * QD::s4];
                            }
                            for (int p = 0; p < g.nP; ++p) {
                                const double* __restrict__ A = g.A + (size_t)p * N * N;
                                const double* __restrict__ B = g.B + (size_t)p * N * N;
                                // Coulomb: (A_mn + A_nm) B_kr + A_kr (B_mn + B_nm), plus the k <-> r partner
                                const double Asmn = A[m * N + n] + A[n * N + m], Bsmn = B[m * N + n] + B[n * N + m];
                                double Akr = A[k * N + r], Bkr = B[k * N + r];
                                // exchange: A_mk B_nr + A_nk B_mr + A_km B_rn + A_kn B_rm, plus the k <-> r partner
                                double GK = A[m * N + k] * B[n * N + r] + A[n * N + k] * B[m * N + r] +
                                            A[k * N + m] * B[r * N + n] + A[k * N + n] * B[r * N + m];
                                if (both) {
                                    Akr += A[r * N + k]; Bkr += B[r * N + k];
                                    GK += A[m * N + r] * B[n * N + k] + A[n * N + r] * B[m * N + k] +
                                          A[r * N + m] * B[k * N + n] + A[r * N + n] * B[k * N + m];
                                }
                                const double GJ = Asmn * Bkr + Akr * Bsmn;
#pragma unroll
                                for (int x = 0; x < 3; ++x) {
                                    gj[p][x] = fma(GJ, dI[x], gj[p][x]);
                                    gk[p][x] = fma(GK, dI[x], gk[p][x]);
                                }
                            }
                        }
                    }
                }
            }
    }
    // every thread of the CTA differentiates the same shell M: one reduction per warp, one atomic per warp and value
    const int at = g.atom[M];
#pragma unroll
    for (int p = 0; p < kGradPairs; ++p) {
        if (p >= g.nP) break;
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            double a = gj[p][x], b = gk[p][x];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                a += __shfl_down_sync(0xffffffffu, a, o);
                b += __shfl_down_sync(0xffffffffu, b, o);
            }
            if ((threadIdx.x & 31) == 0) {
                if (g.gJ && a != 0.0) atomicAdd(g.gJ + ((size_t)p * g.natom + at) * 3 + x, a);
                if (g.gK && b != 0.0) atomicAdd(g.gK + ((size_t)p * g.natom + at) * 3 + x, b);
            }
        }
    }
}

template <int LM, int LN, int LC, int LD>
static int launch_grad_cls(ltjk_ctx* c, GradArgs& g)
{
    if (g.nM == 0 || g.nN == 0 || g.nK == 0 || g.nR == 0) return LTJK_OK;
    if ((long long)g.nM * g.nN > 65535) return set_err(c, LTJK_EINVAL, "jk_grad: more than 65535 (M,N) shell pairs of one class");
    const long long nkr = (long long)g.nK * g.nR;
    grad_kernel<LM, LN, LC, LD><<<dim3((unsigned)((nkr + 63) / 64), (unsigned)(g.nM * g.nN)), 64, 0, c->stream>>>(g);
    LTJK_CUDA(c, cudaGetLastError());
    c->st_launches++;
    return LTJK_OK;
}

template <int LM, int LN>
static int launch_grad_mn(ltjk_ctx* c, GradArgs& g, int* const* lists, const int* cnt)
{
    int rc;
#define KET(LC, LD)                                                                                       \
    g.shK = lists[LC]; g.nK = cnt[LC]; g.shR = lists[LD]; g.nR = cnt[LD]; g.same = (LC == LD);            \
    if ((rc = launch_grad_cls<LM, LN, LC, LD>(c, g))) return rc;
    KET(0, 0) KET(1, 0) KET(1, 1) KET(2, 0) KET(2, 1) KET(2, 2)
#undef KET
    return LTJK_OK;
}

void free_grad(ltjk_ctx* c)
{
    void* ptrs[] = {c->gr_xyz, c->gr_exps, c->gr_coef, c->gr_int};
    for (void* p : ptrs) if (p) cudaFree(p);
    c->gr_xyz = c->gr_exps = c->gr_coef = nullptr; c->gr_int = nullptr;
}

// basis in CALLER shell order on the device (uploaded at the first gradient call of a geometry)
static int ensure_grad_basis(ltjk_ctx* c)
{
    if (c->gr_int) return LTJK_OK;
    const int ns = c->nshell;
    std::vector<int> ints;                         // atom | nprim | poff | ao0 | list l=0 | list l=1 | list l=2
    ints.insert(ints.end(), c->atom.begin(), c->atom.end());
    ints.insert(ints.end(), c->nprim.begin(), c->nprim.end());
    ints.insert(ints.end(), c->prim_off.begin(), c->prim_off.end());
    int ao = 0;
    for (int s = 0; s < ns; ++s) { ints.push_back(ao); ao += ncart(c->l[s]); }
    for (int ll = 0; ll < 3; ++ll) {
        c->gr_cnt[ll] = 0;
        for (int s = 0; s < ns; ++s) if (c->l[s] == ll) { ints.push_back(s); c->gr_cnt[ll]++; }
    }
    LTJK_CUDA(c, cudaMalloc((void**)&c->gr_int, sizeof(int) * ints.size()));
    LTJK_CUDA(c, cudaMalloc((void**)&c->gr_xyz, sizeof(double) * c->xyz.size()));
    LTJK_CUDA(c, cudaMalloc((void**)&c->gr_exps, sizeof(double) * c->exps.size()));
    LTJK_CUDA(c, cudaMalloc((void**)&c->gr_coef, sizeof(double) * c->coef.size()));
    LTJK_CUDA(c, cudaMemcpyAsync(c->gr_int, ints.data(), sizeof(int) * ints.size(), cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(c->gr_xyz, c->xyz.data(), sizeof(double) * c->xyz.size(), cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(c->gr_exps, c->exps.data(), sizeof(double) * c->exps.size(), cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(c->gr_coef, c->coef.data(), sizeof(double) * c->coef.size(), cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));      // the host vector goes out of scope
    return LTJK_OK;
}

int launch_jk_grad(ltjk_ctx* c, int nP, const double* A, const double* B, double* gJ, double* gK)
{
    int rc;
    if ((rc = ensure_grad_basis(c))) return rc;
    const int ns = c->nshell;
    const size_t nout = sizeof(double) * (size_t)nP * c->natom * 3;
    if (gJ) LTJK_CUDA(c, cudaMemsetAsync(gJ, 0, nout, c->stream));
    if (gK) LTJK_CUDA(c, cudaMemsetAsync(gK, 0, nout, c->stream));
    GradArgs g;
    g.xyz = c->gr_xyz; g.exps = c->gr_exps; g.coef = c->gr_coef; g.boys = c->t.boys;
    g.atom = c->gr_int; g.nprim = c->gr_int + ns; g.poff = c->gr_int + 2 * ns; g.ao0 = c->gr_int + 3 * ns;
    int* lists[3];
    lists[0] = c->gr_int + 4 * ns; lists[1] = lists[0] + c->gr_cnt[0]; lists[2] = lists[1] + c->gr_cnt[1];
    g.N = c->nao; g.natom = c->natom;
    c->st_launches = 0;
    for (int p0 = 0; p0 < nP; p0 += kGradPairs) {
        g.nP = std::min(kGradPairs, nP - p0);
        g.A = A + (size_t)p0 * g.N * g.N; g.B = B + (size_t)p0 * g.N * g.N;
        g.gJ = gJ ? gJ + (size_t)p0 * c->natom * 3 : nullptr;
        g.gK = gK ? gK + (size_t)p0 * c->natom * 3 : nullptr;
#define MN(LM, LN)                                                                      \
        g.shM = lists[LM]; g.nM = c->gr_cnt[LM]; g.shN = lists[LN]; g.nN = c->gr_cnt[LN]; \
        if ((rc = launch_grad_mn<LM, LN>(c, g, lists, c->gr_cnt))) return rc;
        MN(0, 0) MN(0, 1) MN(0, 2) MN(1, 0) MN(1, 1) MN(1, 2) MN(2, 0) MN(2, 1) MN(2, 2)
#undef MN
    }
    return LTJK_OK;
}

}  // namespace ltjk

extern "C" int ltjk_jk_grad(ltjk_ctx* c, int nP, const double* A, const double* B, double* gradJ, double* gradK)
{
    using namespace ltjk;
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "jk_grad: no basis");
    if (nP <= 0 || !A || !B || (!gradJ && !gradK)) return set_err(c, LTJK_EINVAL, "jk_grad: bad arguments");
    for (int l : c->l)
        if (l > 2) return set_err(c, LTJK_ELMAX, "jk_grad: the derivative classes are generated for s, p, d shells (an f shell would need g)");
    cudaSetDevice(c->device);
    return launch_jk_grad(c, nP, A, B, gradJ, gradK);
}

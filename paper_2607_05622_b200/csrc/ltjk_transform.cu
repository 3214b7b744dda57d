// ltjk_transform.cu -- step a4: Laplace pseudo-densities (Eqs. 13-15; Alg. 1 lines 5-7)
//   D^{alpha,d} = (C_o e^{+eps_o tau_alpha}) T_d (C_v e^{-eps_v tau_alpha})^T
// evaluated as two batched fp64 tensor-core (DMMA) GEMMs per (alpha, d):
//   W = [e^{(eps_i - eps_b) tau} T_d[i][b]] . C_v^T      (nocc x N)      -- the exponentials are fused into the load
//   D = C_o . W                                          (N x N)
// (nocc < nvir, so contracting the virtual index first is the cheaper order.)
#include "ltjk_internal.h"
#include <algorithm>
#include <cmath>
#include <mutex>
#include <string>

namespace ltjk {

__global__ void exp_factors_kernel(int nocc, int nvir, int ntau, const double* __restrict__ eo,
                                   const double* __restrict__ ev, const double* __restrict__ tau,
                                   double* __restrict__ fo, double* __restrict__ fv)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = nocc + nvir;
    if (t >= ntau * n) return;
    const int a = t / n, i = t % n;
    if (i < nocc) fo[a * nocc + i] = exp(eo[i] * tau[a]);
    else fv[a * nvir + (i - nocc)] = exp(-ev[i - nocc] * tau[a]);
}

// C[z] (M x Nn, row-major) = A[z] (M x K, row-major, optionally scaled sr[i]*sc[k]) . B
//   TRANSB = true : B given as Bt (Nn x K row-major), i.e. C = A . Bt^T
//   TRANSB = false: B (K x Nn row-major)
// batch z = za * nzb + zb; A advances with (za,zb) as given by the strides.
struct GemmArgs {
    int M, Nn, K;
    const double* A; long long sAa, sAb;
    const double* B; long long sBa, sBb;
    double* C; long long sCa, sCb;
    const double* A2; double ca, ca2;    // optional second A operand: A_eff = ca * A + ca2 * A2 (same strides)
    const double* sr; long long ssr;     // row scale, per za (may be null)
    const double* sc; long long ssc;     // column (k) scale, per za
    int nzb;
};

// FP64 tensor cores (DMMA): mma.sync m8n8k4, A row-major 8x4 (1 double per lane), B column-major 4x8, C 8x8
// (2 doubles per lane).  This is the only place the path uses tensor cores (north_star: "FP64 tensor cores are used
// only for the dense pseudo-density GEMMs"); tcgen05 has no f64 kind, so the Blackwell fp64 tensor path is mma.sync.
__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, const double a, const double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// CTA tile 64 x 64, 8 warps as 2 x 4, warp tile 32 x 16 = 4 x 2 DMMA tiles, K step 16 through shared memory
// (row stride 68 doubles: the 16 lanes of a half-warp -- 4 k x 4 m -- then fall into 16 different 8-byte banks).
template <bool TRANSB>
__global__ void __launch_bounds__(256) gemm_kernel(const GemmArgs g)
{
    constexpr int BM = 64, BN = 64, BK = 16, LD = 68;
    __shared__ double As[BK][LD];
    __shared__ double Bs[BK][LD];
    const int za = blockIdx.z / g.nzb, zb = blockIdx.z % g.nzb;
    const double* __restrict__ A = g.A + za * g.sAa + zb * g.sAb;
    const double* __restrict__ A2 = g.A2 ? g.A2 + za * g.sAa + zb * g.sAb : nullptr;
    const double* __restrict__ B = g.B + za * g.sBa + zb * g.sBb;
    double* __restrict__ C = g.C + za * g.sCa + zb * g.sCb;
    const double* sr = g.sr ? g.sr + za * g.ssr : nullptr;
    const double* sc = g.sc ? g.sc + za * g.ssc : nullptr;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int wm = (w >> 2) * 32, wn = (w & 3) * 16;
    const int lr = lane >> 2, lk = lane & 3;
    double acc[4][2][2] = {};
    for (int k0 = 0; k0 < g.K; k0 += BK) {
        // A tile: 64 x 16, lanes along k (contiguous)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int k = tid & 15, m = (tid >> 4) + 16 * e;
            const int gm = m0 + m, gk = k0 + k;
            double v = 0.0;
            if (gm < g.M && gk < g.K) {
                v = A[(size_t)gm * g.K + gk];
                if (A2) v = g.ca * v + g.ca2 * A2[(size_t)gm * g.K + gk];
                if (sr) v *= sr[gm] * sc[gk];
            }
            As[k][m] = v;
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            double v = 0.0;
            if (TRANSB) {
                const int k = tid & 15, n = (tid >> 4) + 16 * e;
                const int gn = n0 + n, gk = k0 + k;
                if (gn < g.Nn && gk < g.K) v = B[(size_t)gn * g.K + gk];
                Bs[k][n] = v;
            } else {
                const int n = tid & 63, k = (tid >> 6) + 4 * e;
                const int gn = n0 + n, gk = k0 + k;
                if (gn < g.Nn && gk < g.K) v = B[(size_t)gk * g.Nn + gn];
                Bs[k][n] = v;
            }
        }
        __syncthreads();
#pragma unroll
        for (int k4 = 0; k4 < BK; k4 += 4) {
            double a[4], b[2];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[k4 + lk][wm + 8 * i + lr];
#pragma unroll
            for (int j = 0; j < 2; ++j) b[j] = Bs[k4 + lk][wn + 8 * j + lr];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) dmma_m8n8k4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int gm = m0 + wm + 8 * i + lr;
        if (gm >= g.M) continue;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int gn = n0 + wn + 8 * j + 2 * lk;
            if (gn < g.Nn) C[(size_t)gm * g.Nn + gn] = acc[i][j][0];
            if (gn + 1 < g.Nn) C[(size_t)gm * g.Nn + gn + 1] = acc[i][j][1];
        }
    }
}

int launch_pseudo_densities(ltjk_ctx* c, int nocc, int nvir, const double* C_occ, const double* C_vir,
                            const double* eps_occ, const double* eps_vir, int nT, const double* T, int ntau,
                            const double* tau_host, double* D_out)
{
    const int N = c->nao;
    double *tau = nullptr, *fo = nullptr, *fv = nullptr, *W = nullptr;
    LTJK_CUDA(c, cudaMallocAsync(&tau, sizeof(double) * ntau, c->stream));
    LTJK_CUDA(c, cudaMallocAsync(&fo, sizeof(double) * ntau * nocc, c->stream));
    LTJK_CUDA(c, cudaMallocAsync(&fv, sizeof(double) * ntau * nvir, c->stream));
    LTJK_CUDA(c, cudaMallocAsync(&W, sizeof(double) * (size_t)ntau * nT * nocc * N, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(tau, tau_host, sizeof(double) * ntau, cudaMemcpyHostToDevice, c->stream));
    const int ne = ntau * (nocc + nvir);
    exp_factors_kernel<<<(ne + 127) / 128, 128, 0, c->stream>>>(nocc, nvir, ntau, eps_occ, eps_vir, tau, fo, fv);
    LTJK_CUDA(c, cudaGetLastError());
    GemmArgs g1;   // W[a][d] = (fo[a] .* T[d] .* fv[a]) . C_vir^T
    g1.M = nocc; g1.Nn = N; g1.K = nvir;
    g1.A = T; g1.sAa = 0; g1.sAb = (long long)nocc * nvir;
    g1.B = C_vir; g1.sBa = 0; g1.sBb = 0;
    g1.C = W; g1.sCa = (long long)nT * nocc * N; g1.sCb = (long long)nocc * N;
    g1.sr = fo; g1.ssr = nocc; g1.sc = fv; g1.ssc = nvir; g1.nzb = nT; g1.A2 = nullptr; g1.ca = 1.0; g1.ca2 = 0.0;
    gemm_kernel<true><<<dim3((N + 63) / 64, (nocc + 63) / 64, ntau * nT), 256, 0, c->stream>>>(g1);
    LTJK_CUDA(c, cudaGetLastError());
    GemmArgs g2;   // D[a][d] = C_occ . W[a][d]
    g2.M = N; g2.Nn = N; g2.K = nocc;
    g2.A = C_occ; g2.sAa = 0; g2.sAb = 0;
    g2.B = W; g2.sBa = (long long)nT * nocc * N; g2.sBb = (long long)nocc * N;
    g2.C = D_out; g2.sCa = (long long)nT * N * N; g2.sCb = (long long)N * N;
    g2.sr = nullptr; g2.ssr = 0; g2.sc = nullptr; g2.ssc = 0; g2.nzb = nT; g2.A2 = nullptr; g2.ca = 1.0; g2.ca2 = 0.0;
    gemm_kernel<false><<<dim3((N + 63) / 64, (N + 63) / 64, ntau * nT), 256, 0, c->stream>>>(g2);
    LTJK_CUDA(c, cudaGetLastError());
    cudaFreeAsync(tau, c->stream); cudaFreeAsync(fo, c->stream); cudaFreeAsync(fv, c->stream); cudaFreeAsync(W, c->stream);
    c->st_launches += 3;
    return LTJK_OK;
}


// ---------------------------------------------------------------------------------------------------------------
// Laplace-Fock back-transform (Eq. 19) and grid accumulation (Eqs. 11, 21).
__global__ void transpose_kernel(int rows, int cols, const double* __restrict__ in, double* __restrict__ out)
{
    __shared__ double tile[32][33];
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    for (int i = threadIdx.y; i < 32; i += 8)
        if (r0 + i < rows && c0 + threadIdx.x < cols) tile[i][threadIdx.x] = in[(size_t)(r0 + i) * cols + c0 + threadIdx.x];
    __syncthreads();
    for (int i = threadIdx.y; i < 32; i += 8)
        if (c0 + i < cols && r0 + threadIdx.x < rows) out[(size_t)(c0 + i) * rows + r0 + threadIdx.x] = tile[threadIdx.x][i];
}

int launch_laplace_fock(ltjk_ctx* c, int nD, const double* J, const double* K, int nmo, const double* C, double* F)
{
    return launch_mo_transform(c, nD, J, 2.0, K, -1.0, nmo, C, F);
}

// F[d] = C^T (ca A[d] + ca2 A2[d]) C for nD matrices (A2 may be NULL): two batched DMMA GEMMs.
int launch_mo_transform(ltjk_ctx* c, int nD, const double* A, double ca, const double* A2, double ca2, int nmo,
                        const double* C, double* F)
{
    const int N = c->nao;
    double *Ct = nullptr, *tmp = nullptr;
    LTJK_CUDA(c, cudaMallocAsync(&Ct, sizeof(double) * (size_t)N * nmo, c->stream));
    LTJK_CUDA(c, cudaMallocAsync(&tmp, sizeof(double) * (size_t)nD * N * nmo, c->stream));
    transpose_kernel<<<dim3((nmo + 31) / 32, (N + 31) / 32), dim3(32, 8), 0, c->stream>>>(N, nmo, C, Ct);
    LTJK_CUDA(c, cudaGetLastError());
    GemmArgs g1;   // tmp[d] (N x nmo) = (ca A[d] + ca2 A2[d]) . C
    g1.M = N; g1.Nn = nmo; g1.K = N;
    g1.A = A; g1.A2 = A2; g1.ca = ca; g1.ca2 = A2 ? ca2 : 0.0; g1.sAa = (long long)N * N; g1.sAb = 0;
    g1.B = C; g1.sBa = 0; g1.sBb = 0;
    g1.C = tmp; g1.sCa = (long long)N * nmo; g1.sCb = 0;
    g1.sr = nullptr; g1.ssr = 0; g1.sc = nullptr; g1.ssc = 0; g1.nzb = 1;
    gemm_kernel<false><<<dim3((nmo + 63) / 64, (N + 63) / 64, nD), 256, 0, c->stream>>>(g1);
    LTJK_CUDA(c, cudaGetLastError());
    GemmArgs g2;   // F[d] (nmo x nmo) = C^T . tmp[d]
    g2.M = nmo; g2.Nn = nmo; g2.K = N;
    g2.A = Ct; g2.A2 = nullptr; g2.ca = 1.0; g2.ca2 = 0.0; g2.sAa = 0; g2.sAb = 0;
    g2.B = tmp; g2.sBa = (long long)N * nmo; g2.sBb = 0;
    g2.C = F; g2.sCa = (long long)nmo * nmo; g2.sCb = 0;
    g2.sr = nullptr; g2.ssr = 0; g2.sc = nullptr; g2.ssc = 0; g2.nzb = 1;
    gemm_kernel<false><<<dim3((nmo + 63) / 64, (nmo + 63) / 64, nD), 256, 0, c->stream>>>(g2);
    LTJK_CUDA(c, cudaGetLastError());
    cudaFreeAsync(Ct, c->stream); cudaFreeAsync(tmp, c->stream);
    return LTJK_OK;
}

__global__ void accumulate_kernel(int ntau, int nT, long long nelem, const double* __restrict__ wt,
                                  const double* __restrict__ X, double* __restrict__ Y)
{
    const long long tot = (long long)nT * nelem;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < tot; i += (long long)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int a = 0; a < ntau; ++a) s = fma(wt[a], X[(size_t)a * tot + i], s);
        Y[i] = s;
    }
}

int launch_laplace_accumulate(ltjk_ctx* c, int ntau, int nT, long long nelem, const double* tau_host,
                              const double* w_host, double omega, const double* X, double* Y)
{
    std::vector<double> wt(ntau);
    for (int a = 0; a < ntau; ++a) wt[a] = w_host[a] * exp(omega * tau_host[a]);   // Eq. 21
    double* d_w = nullptr;
    LTJK_CUDA(c, cudaMallocAsync(&d_w, sizeof(double) * ntau, c->stream));
    LTJK_CUDA(c, cudaMemcpyAsync(d_w, wt.data(), sizeof(double) * ntau, cudaMemcpyHostToDevice, c->stream));
    LTJK_CUDA(c, cudaStreamSynchronize(c->stream));      // wt is a local buffer
    const long long tot = (long long)nT * nelem;
    const int grid = (int)std::min<long long>((tot + 255) / 256, 148ll * 16);
    accumulate_kernel<<<grid, 256, 0, c->stream>>>(ntau, nT, nelem, d_w, X, Y);
    LTJK_CUDA(c, cudaGetLastError());
    cudaFreeAsync(d_w, c->stream);
    return LTJK_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// No-allocation variant of the pseudo-density transform (include/ltjk.h: ltjk_build_pseudo_densities_noalloc) for
// callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).
// launch_pseudo_densities takes its scratch (exponential factors fo, fv and the half-transformed W) from the
// stream-ordered pool; here the same scratch lives in ONE file-scope device array of fixed size.  Every GPU that loads
// the library holds these 8 MiB until the process exits.  All calls (all contexts, all streams) on a device share
// the array and it keeps the last call's contents: every element a call reads (fo, fv, all of W) is first written by
// that call's own kernels, so nothing has to start at zero and nothing is cleared; calls that overlap on the GPU race.
constexpr long long kNoAllocDoubles = 1ll << 20;        // 8 MiB
constexpr int kNoAllocMaxTau = 32;                      // Laplace points passed by value (the library's grids have <= 14)
static __device__ __align__(256) double g_noalloc_scratch[kNoAllocDoubles];

struct TauArgs { double tau[kNoAllocMaxTau]; };

// exp_factors_kernel with the Laplace points as kernel arguments: no host-to-device copy, no tau buffer
__global__ void exp_factors_noalloc_kernel(int nocc, int nvir, int ntau, const double* __restrict__ eo,
                                           const double* __restrict__ ev, const TauArgs ta,
                                           double* __restrict__ fo, double* __restrict__ fv)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = nocc + nvir;
    if (t >= ntau * n) return;
    const int a = t / n, i = t % n;
    if (i < nocc) fo[a * nocc + i] = exp(eo[i] * ta.tau[a]);
    else fv[a * nvir + (i - nocc)] = exp(-ev[i - nocc] * ta.tau[a]);
}

// Set-up, once per device and process (called by ltjk_create with the context's device current).  In host code the
// NAME g_noalloc_scratch is a host-side stand-in, not a device address: the address the kernels need comes from
// cudaGetSymbolAddress, per device.
int noalloc_setup(ltjk_ctx* c)
{
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static double* ptr_of[kMaxDev] = {};
    std::lock_guard<std::mutex> lock(mu);
    c->na_scratch = nullptr;
    if (c->device < 0 || c->device >= kMaxDev) { c->na_err = "no-allocation scratch: device index beyond 63"; return LTJK_ECUDA; }
    if (!ptr_of[c->device]) {
        cudaError_t e = cudaSetDevice(c->device);
        double* p = nullptr;
        if (e == cudaSuccess) e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            c->na_err = std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e);
            return LTJK_ECUDA;
        }
        ptr_of[c->device] = p;
    }
    c->na_scratch = ptr_of[c->device];
    return LTJK_OK;
}

}  // namespace ltjk

extern "C" int ltjk_build_pseudo_densities_noalloc(ltjk_ctx* c, int nocc, int nvir, const double* C_occ,
                                                   const double* C_vir, const double* eps_occ, const double* eps_vir,
                                                   int nT, const double* T, int ntau, const double* tau_host,
                                                   double* D_out)
{
    using namespace ltjk;
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "build_pseudo_densities_noalloc: no basis");
    if (nocc <= 0 || nvir <= 0 || nT <= 0 || ntau <= 0 || !C_occ || !C_vir || !eps_occ || !eps_vir || !T || !tau_host ||
        !D_out)
        return set_err(c, LTJK_EINVAL, "build_pseudo_densities_noalloc: bad arguments");
    if (ntau > kNoAllocMaxTau)
        return set_err(c, LTJK_EINVAL, "build_pseudo_densities_noalloc: ntau = " + std::to_string(ntau) +
                                           " exceeds the maximum of " + std::to_string(kNoAllocMaxTau) + " Laplace points");
    const long long N = c->nao;
    const long long nfac = ((long long)ntau * (nocc + nvir) + 31) & ~31ll;          // W starts 256-byte aligned
    const long long need = nfac + (long long)ntau * nT * nocc * N;
    if (need > kNoAllocDoubles)
        return set_err(c, LTJK_EINVAL, "build_pseudo_densities_noalloc: needs " + std::to_string(need) +
                                           " doubles of scratch (ntau (nocc + nvir) + ntau nT nocc N), the fixed scratch holds " +
                                           std::to_string(kNoAllocDoubles) + " (8 MiB); use ltjk_build_pseudo_densities");
    if (!c->na_scratch) return set_err(c, LTJK_ECUDA, "build_pseudo_densities_noalloc: " + c->na_err);
    LTJK_CUDA(c, cudaSetDevice(c->device));
    double* fo = c->na_scratch;
    double* fv = fo + (long long)ntau * nocc;
    double* W = c->na_scratch + nfac;
    TauArgs ta;
    for (int a = 0; a < kNoAllocMaxTau; ++a) ta.tau[a] = a < ntau ? tau_host[a] : 0.0;
    const int ne = ntau * (nocc + nvir);
    exp_factors_noalloc_kernel<<<(ne + 127) / 128, 128, 0, c->stream>>>(nocc, nvir, ntau, eps_occ, eps_vir, ta, fo, fv);
    LTJK_CUDA(c, cudaGetLastError());
    GemmArgs g1;   // W[a][d] = (fo[a] .* T[d] .* fv[a]) . C_vir^T        (every element of W is written)
    g1.M = nocc; g1.Nn = (int)N; g1.K = nvir;
    g1.A = T; g1.sAa = 0; g1.sAb = (long long)nocc * nvir;
    g1.B = C_vir; g1.sBa = 0; g1.sBb = 0;
    g1.C = W; g1.sCa = (long long)nT * nocc * N; g1.sCb = (long long)nocc * N;
    g1.sr = fo; g1.ssr = nocc; g1.sc = fv; g1.ssc = nvir; g1.nzb = nT; g1.A2 = nullptr; g1.ca = 1.0; g1.ca2 = 0.0;
    gemm_kernel<true><<<dim3((unsigned)((N + 63) / 64), (nocc + 63) / 64, ntau * nT), 256, 0, c->stream>>>(g1);
    LTJK_CUDA(c, cudaGetLastError());
    GemmArgs g2;   // D[a][d] = C_occ . W[a][d]
    g2.M = (int)N; g2.Nn = (int)N; g2.K = nocc;
    g2.A = C_occ; g2.sAa = 0; g2.sAb = 0;
    g2.B = W; g2.sBa = (long long)nT * nocc * N; g2.sBb = (long long)nocc * N;
    g2.C = D_out; g2.sCa = (long long)nT * N * N; g2.sCb = N * N;
    g2.sr = nullptr; g2.ssr = 0; g2.sc = nullptr; g2.ssc = 0; g2.nzb = nT; g2.A2 = nullptr; g2.ca = 1.0; g2.ca2 = 0.0;
    gemm_kernel<false><<<dim3((unsigned)((N + 63) / 64), (unsigned)((N + 63) / 64), ntau * nT), 256, 0, c->stream>>>(g2);
    LTJK_CUDA(c, cudaGetLastError());
    c->st_launches += 3;
    return LTJK_OK;
}

// ltjk_sph.cu -- SURVEY.md 8(f) N4, second half: the spherical-harmonic transform at matrix level (include/ltjk.h).
//
// The integral path is Cartesian throughout (the paper's AO counts are Cartesian); a caller that works
// with pure (2l+1) functions converts matrices on the device, one shell-pair block at a time:
//     operators   X^sph[A m, B m'] = sum_{c c'} S^{lA}[m][c] X^cart[A c, B c'] S^{lB}[m'][c']        (S X S^T)
//     densities   D^cart[A c, B c'] = sum_{m m'} S^{lA}[m][c] D^sph[A m, B m'] S^{lB}[m'][c']        (S^T D S)
// S^l = monomial coefficients of the Racah-normalised real solid harmonics, m = -l..l, Cartesian components in the
// library's lexicographic order; the tables below are written out by hand for l <= 3 (the oracle evaluates the general
// closed form instead).  Both kernels are plain gather kernels, one thread per output element: HBM-bound
// (8 (N^2 + N_sph^2) bytes per matrix), the <= 100 multiply-adds per element are hidden behind the loads.
#include "ltjk_internal.h"
#include "eri_core.h"

namespace ltjk {

// rows m = -l..l, columns: l=1: x y z; l=2: xx xy xz yy yz zz; l=3: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
#define R3 1.7320508075688772       /* sqrt 3 */
#define R6 2.449489742783178        /* sqrt 6 */
#define R10 3.1622776601683795      /* sqrt 10 */
#define R15 3.872983346207417       /* sqrt 15 */
__constant__ double kSph[1 + 9 + 30 + 70] = {
    // l = 0
    1.0,
    // l = 1: y, z, x
    0, 1, 0,  0, 0, 1,  1, 0, 0,
    // l = 2: sqrt3 xy | sqrt3 yz | zz - (xx+yy)/2 | sqrt3 xz | sqrt3/2 (xx - yy)
    0, R3, 0, 0, 0, 0,
    0, 0, 0, 0, R3, 0,
    -0.5, 0, 0, -0.5, 0, 1.0,
    0, 0, R3, 0, 0, 0,
    0.5 * R3, 0, 0, -0.5 * R3, 0, 0,
    // l = 3: sqrt10/4 (3xxy - yyy) | sqrt15 xyz | sqrt6/4 (4 yzz - xxy - yyy) | zzz - 3/2 (xxz + yyz) |
    //        sqrt6/4 (4 xzz - xxx - xyy) | sqrt15/2 (xxz - yyz) | sqrt10/4 (xxx - 3 xyy)
    0, 0.75 * R10, 0, 0, 0, 0, -0.25 * R10, 0, 0, 0,
    0, 0, 0, 0, R15, 0, 0, 0, 0, 0,
    0, -0.25 * R6, 0, 0, 0, 0, -0.25 * R6, 0, R6, 0,
    0, 0, -1.5, 0, 0, 0, 0, -1.5, 0, 1.0,
    -0.25 * R6, 0, 0, -0.25 * R6, 0, R6, 0, 0, 0, 0,
    0, 0, 0.5 * R15, 0, 0, 0, 0, -0.5 * R15, 0, 0,
    0.25 * R10, 0, 0, -0.75 * R10, 0, 0, 0, 0, 0, 0};
#undef R3
#undef R6
#undef R10
#undef R15
__device__ __forceinline__ int sph_tab_off(int l) { return l == 0 ? 0 : l == 1 ? 1 : l == 2 ? 10 : 40; }

struct SphMeta {                 // caller's shell order (the matrices of the C ABI are in the caller's AO order)
    const int* sh_l;             // [nshell]
    const int* sh_c0;            // first Cartesian AO of the shell
    const int* sh_s0;            // first pure function of the shell
    const int* cart_sh;          // [N]     shell of a Cartesian AO
    const int* sph_sh;           // [N_sph] shell of a pure function
    int N, Ns;
};

// out[n][i][j], i, j pure functions  <-  in[n][mu][nu], Cartesian
__global__ void __launch_bounds__(256) sph_from_cart_kernel(const SphMeta M, const double* __restrict__ X,
                                                            double* __restrict__ Y)
{
    __shared__ double S[110];
    for (int k = threadIdx.x; k < 110; k += blockDim.x) S[k] = kSph[k];
    __syncthreads();
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (long long)M.Ns * M.Ns) return;
    const int i = (int)(e / M.Ns), j = (int)(e % M.Ns);
    const int A = M.sph_sh[i], B = M.sph_sh[j];
    const int la = M.sh_l[A], lb = M.sh_l[B], na = ncart(la), nb = ncart(lb);
    const double* Sa = S + sph_tab_off(la) + (i - M.sh_s0[A]) * na;
    const double* Sb = S + sph_tab_off(lb) + (j - M.sh_s0[B]) * nb;
    const double* Xn = X + (size_t)blockIdx.y * M.N * M.N + (size_t)M.sh_c0[A] * M.N + M.sh_c0[B];
    double acc = 0.0;
    for (int ca = 0; ca < na; ++ca) {
        const double sa = Sa[ca];
        if (sa == 0.0) continue;
        double row = 0.0;
        for (int cb = 0; cb < nb; ++cb) row += Sb[cb] * Xn[(size_t)ca * M.N + cb];
        acc += sa * row;
    }
    Y[(size_t)blockIdx.y * M.Ns * M.Ns + e] = acc;
}

// out[n][mu][nu], Cartesian  <-  in[n][i][j], pure functions
__global__ void __launch_bounds__(256) cart_from_sph_kernel(const SphMeta M, const double* __restrict__ D,
                                                            double* __restrict__ Y)
{
    __shared__ double S[110];
    for (int k = threadIdx.x; k < 110; k += blockDim.x) S[k] = kSph[k];
    __syncthreads();
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (long long)M.N * M.N) return;
    const int mu = (int)(e / M.N), nu = (int)(e % M.N);
    const int A = M.cart_sh[mu], B = M.cart_sh[nu];
    const int la = M.sh_l[A], lb = M.sh_l[B], na = ncart(la), nb = ncart(lb);
    const double* Sa = S + sph_tab_off(la) + (mu - M.sh_c0[A]);        // column ca of S^{la}: stride na
    const double* Sb = S + sph_tab_off(lb) + (nu - M.sh_c0[B]);
    const double* Dn = D + (size_t)blockIdx.y * M.Ns * M.Ns + (size_t)M.sh_s0[A] * M.Ns + M.sh_s0[B];
    double acc = 0.0;
    for (int ma = 0; ma < 2 * la + 1; ++ma) {
        const double sa = Sa[ma * na];
        if (sa == 0.0) continue;
        double row = 0.0;
        for (int mb = 0; mb < 2 * lb + 1; ++mb) row += Sb[mb * nb] * Dn[(size_t)ma * M.Ns + mb];
        acc += sa * row;
    }
    Y[(size_t)blockIdx.y * M.N * M.N + e] = acc;
}

void free_sph(ltjk_ctx* c)
{
    if (c->d_sph_meta) cudaFree(c->d_sph_meta);
    c->d_sph_meta = nullptr;
}

static int ensure_sph(ltjk_ctx* c, SphMeta* M)
{
    const int ns = c->nshell, N = c->nao;
    int Ns = 0;
    for (int s = 0; s < ns; ++s) Ns += 2 * c->l[s] + 1;
    if (!c->d_sph_meta) {
        std::vector<int> h((size_t)3 * ns + N + Ns);
        int c0 = 0, s0 = 0;
        for (int s = 0; s < ns; ++s) {
            h[s] = c->l[s]; h[ns + s] = c0; h[2 * ns + s] = s0;
            for (int k = 0; k < ncart(c->l[s]); ++k) h[3 * ns + c0 + k] = s;
            for (int k = 0; k < 2 * c->l[s] + 1; ++k) h[3 * ns + N + s0 + k] = s;
            c0 += ncart(c->l[s]); s0 += 2 * c->l[s] + 1;
        }
        LTJK_CUDA(c, cudaMalloc(&c->d_sph_meta, sizeof(int) * h.size()));
        LTJK_CUDA(c, cudaMemcpy(c->d_sph_meta, h.data(), sizeof(int) * h.size(), cudaMemcpyHostToDevice));
    }
    M->sh_l = c->d_sph_meta; M->sh_c0 = M->sh_l + ns; M->sh_s0 = M->sh_c0 + ns;
    M->cart_sh = M->sh_s0 + ns; M->sph_sh = M->cart_sh + N;
    M->N = N; M->Ns = Ns;
    return LTJK_OK;
}

}  // namespace ltjk

using namespace ltjk;

extern "C" {

int ltjk_get_nsph(const ltjk_ctx* c, int* nsph)
{
    if (!c || !nsph) return LTJK_EINVAL;
    if (!c->have_basis) return LTJK_ENOBASIS;
    int n = 0;
    for (int l : c->l) n += 2 * l + 1;
    *nsph = n;
    return LTJK_OK;
}

int ltjk_sph_from_cart(ltjk_ctx* c, int nmat, const double* X_cart, double* X_sph)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "sph_from_cart: no basis");
    if (nmat <= 0 || nmat > 65535 || !X_cart || !X_sph) return set_err(c, LTJK_EINVAL, "sph_from_cart: bad arguments (1 <= nmat <= 65535)");
    cudaSetDevice(c->device);
    SphMeta M;
    int rc;
    if ((rc = ensure_sph(c, &M))) return rc;
    const long long n = (long long)M.Ns * M.Ns;
    sph_from_cart_kernel<<<dim3((unsigned)((n + 255) / 256), nmat), 256, 0, c->stream>>>(M, X_cart, X_sph);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

int ltjk_cart_from_sph(ltjk_ctx* c, int nmat, const double* D_sph, double* D_cart)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "cart_from_sph: no basis");
    if (nmat <= 0 || nmat > 65535 || !D_sph || !D_cart) return set_err(c, LTJK_EINVAL, "cart_from_sph: bad arguments (1 <= nmat <= 65535)");
    cudaSetDevice(c->device);
    SphMeta M;
    int rc;
    if ((rc = ensure_sph(c, &M))) return rc;
    const long long n = (long long)M.N * M.N;
    cart_from_sph_kernel<<<dim3((unsigned)((n + 255) / 256), nmat), 256, 0, c->stream>>>(M, D_sph, D_cart);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

}  // extern "C"

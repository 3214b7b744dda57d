// ltjk_sph.cu -- SURVEY.md 8(f) N4, second half: the spherical-harmonic transform at matrix level (include/ltjk.h).
//
// The integral path is Cartesian throughout (the paper's AO counts are Cartesian); a caller that works
// with pure (2l+1) functions converts matrices on the device, one shell-pair block at a time:
//     operators   X^sph[A m, B m'] = sum_{c c'} S^{lA}[m][c] X^cart[A c, B c'] S^{lB}[m'][c']        (S X S^T)
//     densities   D^cart[A c, B c'] = sum_{m m'} S^{lA}[m][c] D^sph[A m, B m'] S^{lB}[m'][c']        (S^T D S)
// S^l = monomial coefficients of the Racah-normalised real solid harmonics, m = -l..l, Cartesian components in the
// library's lexicographic order; the tables below are written out by hand for l <= 3 (the oracle evaluates the general
// closed form instead).  A gather kernel, one thread per output element and one output row per CTA row, so that the
// row's shell and the (at most 3) non-zero entries of its S row are uniform over the CTA.  Algorithmic traffic
// 8 (N^2 + N_sph^2) bytes per matrix.
#include "ltjk_internal.h"
#include "eri_core.h"

namespace ltjk {

// rows m = -l..l, columns: l=1: x y z; l=2: xx xy xz yy yz zz; l=3: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
#define R3 1.7320508075688772       /* sqrt 3 */
#define R6 2.449489742783178        /* sqrt 6 */
#define R10 3.1622776601683795      /* sqrt 10 */
#define R15 3.872983346207417       /* sqrt 15 */
__device__ const double kSph[1 + 9 + 30 + 70] = {       // 880 bytes: stays in L1
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

// One CTA row = one output row: blockIdx.y = output row (its shell, and with it the non-zero entries of its S row or
// column, are uniform over the CTA), threads along the output columns, blockIdx.z = matrix.
//   DIR 0  out[n][i][j], i, j pure functions  <-  in[n][mu][nu], Cartesian      (operators,  S X S^T)
//   DIR 1  out[n][mu][nu], Cartesian          <-  in[n][i][j], pure functions   (densities,  S^T D S)
template <int DIR>
__global__ void __launch_bounds__(256) sph_row_kernel(const SphMeta M, const double* __restrict__ X, double* __restrict__ Y)
{
    const int Nin = DIR == 0 ? M.N : M.Ns, Nout = DIR == 0 ? M.Ns : M.N;
    const int i = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Nout) return;
    const int A = DIR == 0 ? M.sph_sh[i] : M.cart_sh[i], B = DIR == 0 ? M.sph_sh[j] : M.cart_sh[j];
    const int la = M.sh_l[A], lb = M.sh_l[B], na = ncart(la), nb = ncart(lb);
    const int ii = i - (DIR == 0 ? M.sh_s0[A] : M.sh_c0[A]), jj = j - (DIR == 0 ? M.sh_s0[B] : M.sh_c0[B]);
    const int nka = DIR == 0 ? na : 2 * la + 1, nkb = DIR == 0 ? nb : 2 * lb + 1;       // input rows / columns of the shells
    // S^l[m][c] at m * ncart + c: DIR 0 walks a row (stride 1), DIR 1 a column (stride ncart)
    const double* Sa = kSph + sph_tab_off(la) + (DIR == 0 ? ii * na : ii);
    const double* Sb = kSph + sph_tab_off(lb) + (DIR == 0 ? jj * nb : jj);
    const int sta = DIR == 0 ? 1 : na, stb = DIR == 0 ? 1 : nb;
    const double* Xn = X + (size_t)blockIdx.z * Nin * Nin + (size_t)(DIR == 0 ? M.sh_c0[A] : M.sh_s0[A]) * Nin +
                       (DIR == 0 ? M.sh_c0[B] : M.sh_s0[B]);
    double acc = 0.0;
    for (int ka = 0; ka < nka; ++ka) {
        const double sa = Sa[ka * sta];
        if (sa == 0.0) continue;                               // uniform over the CTA: at most 3 rows survive
        const double* Xr = Xn + (size_t)ka * Nin;
        double row = 0.0;
        for (int kb = 0; kb < nkb; ++kb) row += Sb[kb * stb] * Xr[kb];
        acc += sa * row;
    }
    Y[(size_t)blockIdx.z * Nout * Nout + (size_t)i * Nout + j] = acc;
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
    if (nmat <= 0 || nmat > 65535 || c->nao > 65535 || !X_cart || !X_sph) return set_err(c, LTJK_EINVAL, "sph_from_cart: bad arguments (1 <= nmat <= 65535)");
    cudaSetDevice(c->device);
    SphMeta M;
    int rc;
    if ((rc = ensure_sph(c, &M))) return rc;
    sph_row_kernel<0><<<dim3((M.Ns + 255) / 256, M.Ns, nmat), 256, 0, c->stream>>>(M, X_cart, X_sph);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

int ltjk_cart_from_sph(ltjk_ctx* c, int nmat, const double* D_sph, double* D_cart)
{
    if (!c) return LTJK_EINVAL;
    if (!c->have_basis) return set_err(c, LTJK_ENOBASIS, "cart_from_sph: no basis");
    if (nmat <= 0 || nmat > 65535 || c->nao > 65535 || !D_sph || !D_cart) return set_err(c, LTJK_EINVAL, "cart_from_sph: bad arguments (1 <= nmat <= 65535)");
    cudaSetDevice(c->device);
    SphMeta M;
    int rc;
    if ((rc = ensure_sph(c, &M))) return rc;
    sph_row_kernel<1><<<dim3((M.N + 255) / 256, M.N, nmat), 256, 0, c->stream>>>(M, D_sph, D_cart);
    LTJK_CUDA(c, cudaGetLastError());
    return LTJK_OK;
}

}  // extern "C"

/*
 * ltjk.h -- C ABI of the B200-native non-symmetric Laplace-transform J/K build.
 *
 * The path (cited against /root/reference/PAPER.md as PAPER.md:L<n>):
 *   basis upload -> shell pairs + Schwarz bounds -> minimax Laplace grid (Eq. 11)
 *   -> pseudo-densities D^{alpha,d} = (C_o e^{+eps_o tau}) T_d (C_v e^{-eps_v tau})^T (Eqs. 13-15)
 *   -> J[D], K[D] for a batch of general (non-symmetric) AO densities (Eq. 17; scatter rule Eq. 25)
 *
 * Conventions
 *   - Every function returns 0 (LTJK_OK) or a negative LTJK_E* code; nothing throws or aborts across the ABI.
 *     ltjk_last_error(ctx) gives a human-readable message for the last failure on that context.
 *   - "host" pointers are ordinary CPU memory; "device" pointers are CUDA device memory on the context's
 *     device (e.g. torch tensors' data_ptr()).  The library never frees caller memory and never returns
 *     memory the caller must free.  Internal device buffers belong to the context.
 *   - All device work is enqueued on the context's stream; calls that launch kernels return without
 *     synchronising (the caller syncs through its own stream API) unless stated otherwise.
 *   - A context is not thread-safe.  Calls that touch the device make the context's device the calling thread's
 *     current CUDA device and leave it so; ltjk_create also raises the release threshold of that device's default
 *     stream-ordered memory pool so that the library's scratch allocations are reused between calls.
 *   - There is NO CPU fallback: without a CUDA device ltjk_create fails with LTJK_ECUDA.
 *   - Units: bohr, hartree (PAPER.md reports E_h/a_0 throughout, e.g. L450).
 *   - No prefactor is embedded anywhere: no w_alpha, no exchange 1/2, no spin factor 2
 *     ("J^x and K^x denote the single bare builds ... carry no embedded prefactor").
 */
#ifndef LTJK_H
#define LTJK_H

#ifdef __cplusplus
extern "C" {
#endif

#define LTJK_OK        0
#define LTJK_EINVAL   -1   /* bad argument (null pointer, negative size, nprim too large, ...) */
#define LTJK_ENOBASIS -2   /* call order: basis / shell pairs not set yet */
#define LTJK_ECUDA    -3   /* CUDA runtime error or no device */
#define LTJK_ELMAX    -4   /* angular momentum beyond what the called path is built for: l > 3 in ltjk_set_basis (kernels are
                             Cartesian s, p, d, f); an f shell with pair-list digestion or ltjk_jk_grad */
#define LTJK_ENOCONV  -5   /* Laplace quadrature did not converge (no silent fallback grid) */
#define LTJK_ENOMEM   -6   /* device allocation failed */

typedef struct ltjk_ctx ltjk_ctx;   /* opaque; owns all internal device buffers */

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (e.g. torch's current stream
 * handle) or NULL for the legacy default stream. */
int ltjk_create(ltjk_ctx** out, int device, void* cuda_stream);
int ltjk_destroy(ltjk_ctx* ctx);
const char* ltjk_last_error(const ltjk_ctx* ctx);

/* Upper bound, in bytes, on the integral-panel staging ring the context allocates (two halves; default 8 GiB or a
 * quarter of the free device memory, whichever is smaller; always clamped to 60 % of free memory and never below two
 * panels).  Must be called before ltjk_build_shell_pairs. */
int ltjk_set_scratch_bytes(ltjk_ctx* ctx, long long bytes);

/* Basis upload (step a1).  HOST pointers, copied.
 *   xyz[natom*3]        centres, bohr
 *   atom[nshell]        centre index of each shell
 *   l[nshell]           angular momentum, 0..3 (else LTJK_ELMAX).  s, p, d classes and the lighter classes with one f shell
 *                       run generated straight-line code, the other classes with an f shell the looped kernel
 *                       (PAPER.md:L316 two codegen regimes).
 *                       Cartesian components in lexicographic order (f: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz)
 *   nprim[nshell]       primitives per shell, 1..4
 *   prim_off[nshell]    first primitive of the shell in exps/coef
 *   exps[], coef[]      primitive exponents and coefficients.  coef multiplies
 *                       (x-Ax)^i (y-Ay)^j (z-Az)^k exp(-a r^2) DIRECTLY: normalisation is the caller's job and
 *                       is common to all Cartesian components of a shell (reading A6).
 * AO order = shell order; Cartesian components lexicographic: p = x,y,z; d = xx,xy,xz,yy,yz,zz (reading A7).
 * Kernels are Cartesian only. */
int ltjk_set_basis(ltjk_ctx* ctx, int natom, const double* xyz, int nshell, const int* atom, const int* l,
                   const int* nprim, const int* prim_off, const double* exps, const double* coef);
int ltjk_get_nao(const ltjk_ctx* ctx, int* nao);

/* Shell-pair builder (steps a2, a5).  For every shell pair: Gaussian-product data per primitive pair
 * (p, P, PA, K_ab = c_a c_b exp(-ab/p R_AB^2)) and the Schwarz bound Q_AB = sqrt(max |(ab|ab)|)
 * (PAPER.md:L176, L446), then the screened work lists: a shell quartet (AB|CD) is dropped iff
 * Q_AB * Q_CD < schwarz_tau (pure integral Schwarz, no density weighting; reading A9).
 * Synchronises.  Outputs (host, may be NULL):
 *   n_pairs          number of canonical shell pairs A>=B
 *   n_quartets_kept  number of canonical quartets (AB)>=(CD) with Q_AB Q_CD >= tau (8-fold unique count) */
int ltjk_build_shell_pairs(ltjk_ctx* ctx, double schwarz_tau, long long* n_pairs, long long* n_quartets_kept);

/* Copy the Schwarz bounds to HOST: Q[nshell*nshell], symmetric, caller's shell order.  Synchronises. */
int ltjk_get_schwarz(ltjk_ctx* ctx, double* Q_host);

/* Minimax Laplace quadrature (step a3; Eq. 11): nodes t[npts] and weights w[npts] (HOST,
 * caller-allocated) minimising max_{x in [xmin,xmax]} |1/x - sum_a w_a exp(-x t_a)|.  *maxerr (may be NULL)
 * receives the achieved maximum error on [xmin,xmax].  Pure host function; 2 <= npts <= 14 (LTJK_EINVAL outside:
 * one point is not a Laplace grid, and at 14 points the error on [0.4, 4.5] is 2e-15, the fp64 floor).  Cost: 0.1 s
 * (2 points) to ~30 s (14 points) of quad-precision Remez with continuation in the interval ratio; call it once per
 * denominator range.  LTJK_ENOCONV if the Remez iteration fails; there is no fallback grid. */
int ltjk_laplace_quadrature(double xmin, double xmax, int npts, double* t, double* w, double* maxerr);

/* Pseudo-density transform (step a4; Eq. 13, L145 Eq. 15):
 *   D_out[a][d][mu][nu] = sum_{i,b} C_occ[mu][i] e^{+eps_occ[i] tau[a]} T[d][i][b] e^{-eps_vir[b] tau[a]} C_vir[nu][b]
 * DEVICE pointers, row-major, contiguous: C_occ[N][nocc], C_vir[N][nvir], eps_occ[nocc], eps_vir[nvir],
 * T[nT][nocc][nvir], D_out[ntau][nT][N][N].  tau_host[ntau] is a HOST pointer.  No w_alpha is applied. */
int ltjk_build_pseudo_densities(ltjk_ctx* ctx, int nocc, int nvir, const double* C_occ, const double* C_vir,
                                const double* eps_occ, const double* eps_vir, int nT, const double* T,
                                int ntau, const double* tau_host, double* D_out);

/* No-allocation variant of ltjk_build_pseudo_densities (same operation, same arguments, same result: PAPER.md:L136
 * Eq. 13, L145 Eq. 15) for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it.  It calls no cudaMalloc / cudaFree / pool or library allocation and copies nothing from
 * the host (tau_host is passed to the kernel by value); it only launches three kernels on the ctx stream.  Its
 * scratch (exponential factors and the half-transformed W) is one static device array of 8 MiB that every GPU which
 * loads the library holds until the process exits.
 * Limits (LTJK_EINVAL with a message naming the limit, nothing launched):  ntau <= 32  and
 *     roundup32(ntau (nocc + nvir)) + ntau nT nocc N  <=  1048576 doubles     (N = number of AOs)
 * e.g. 160 AO / 20 occupied / 8 points / 4 amplitude sets fits; 439 AO / 81 / 10 / 16 does not (use the plain call).
 * The array is shared by ALL calls on a device (all contexts, all streams) and keeps the last call's contents; a call
 * writes every element before reading it, so nothing needs clearing, but two calls that overlap on the GPU race:
 * serialise them (one stream, or events).  The device address of the array is resolved once per device at
 * ltjk_create (cudaGetSymbolAddress); if that failed the call returns LTJK_ECUDA. */
int ltjk_build_pseudo_densities_noalloc(ltjk_ctx* ctx, int nocc, int nvir, const double* C_occ, const double* C_vir,
                                        const double* eps_occ, const double* eps_vir, int nT, const double* T,
                                        int ntau, const double* tau_host, double* D_out);

/* Non-symmetric J/K build (steps a5-a9; Eq. 17):
 *   J[d][mu][nu] = sum_{kappa rho} (mu nu|kappa rho) D[d][kappa][rho]
 *   K[d][mu][nu] = sum_{kappa rho} (mu kappa|nu rho) D[d][kappa][rho]
 * over all quartets surviving the Schwarz test.  D is a general real matrix (D != D^T): K comes out as a
 * full non-symmetric matrix with K[D^T] = K[D]^T; J is symmetric.  DEVICE pointers [nD][N][N], row-major;
 * J and K are OVERWRITTEN; either may be NULL (J-only / K-only). */
int ltjk_jk_build(ltjk_ctx* ctx, int nD, const double* D, double* J, double* K);

/* Same as ltjk_jk_build but with HOST buffers: copies D to the device, builds, copies J and K back and
 * synchronises.  This is the end-to-end entry bench.py times as "e2e". */
int ltjk_jk_build_host(ltjk_ctx* ctx, int nD, const double* D_host, double* J_host, double* K_host);

/* One whole Laplace sweep with HOST buffers (steps a4-a9 end to end): copies C_occ[N][nocc], C_vir[N][nvir],
 * eps_occ, eps_vir, T[nT][nocc][nvir] and tau[ntau] to the device, builds the ntau*nT pseudo-densities
 * (Eq. 15), builds J and K for all of them (Eq. 17), copies J_host and K_host
 * [ntau*nT][N][N] back (either may be NULL) and synchronises.  Pinned host memory makes the copies asynchronous. */
int ltjk_sweep_host(ltjk_ctx* ctx, int nocc, int nvir, const double* C_occ_host, const double* C_vir_host,
                    const double* eps_occ_host, const double* eps_vir_host, int nT, const double* T_host, int ntau,
                    const double* tau_host, double* J_host, double* K_host);

/* Laplace-Fock back-transform (Eq. 19), per density d:
 *   F[d][p][q] = sum_{mu nu} C[mu][p] (2 J[d] - K[d])[mu][nu] C[nu][q]
 * DEVICE pointers, row-major: J, K [nD][N][N], C [N][nmo], F [nD][nmo][nmo] (overwritten).  Two batched fp64
 * tensor-core GEMMs; enqueued on the context stream. */
int ltjk_laplace_fock(ltjk_ctx* ctx, int nD, const double* J, const double* K, int nmo, const double* C, double* F);

/* Quadrature-weighted accumulation over the Laplace grid with the EOM reweighting (Eq. 11, L180 Eq. 21):
 *   Y[t][e] = sum_a w[a] exp(omega tau[a]) X[a][t][e],   e < nelem
 * X [ntau][nT][nelem], Y [nT][nelem] DEVICE pointers; tau_host, w_host HOST arrays [ntau]; omega = 0 gives the plain
 * weights.  The caller is responsible for omega < min denominator (Eq. 21's validity range). */
int ltjk_laplace_accumulate(ltjk_ctx* ctx, int ntau, int nT, long long nelem, const double* tau_host,
                            const double* w_host, double omega, const double* X, double* Y);

/* SURVEY 8(f) N4 (second half): spherical-harmonic transform at matrix level.  The integral path is Cartesian
 * (PAPER.md:L565 counts Cartesian AOs); a caller that works with pure functions converts matrices on the device.
 * Pure functions of a shell: chi^sph_{l m} = sum_c S^l[m][c] chi^cart_c, m = -l..l in this order, S^l the monomial
 * coefficients of the Racah-normalised real solid harmonic r^l sqrt(4 pi/(2l+1)) Y_lm (cos(m phi) for m > 0,
 * sin(|m| phi) for m < 0, positive leading coefficient; p = (y, z, x)): a shell whose x^l component is normalised
 * (reading A6) gives normalised pure functions.  Shell order and AO order are the caller's.
 *   ltjk_get_nsph       N_sph = sum over shells of (2l+1)
 *   ltjk_sph_from_cart  operators (J, K, F):  X_sph = S X_cart S^T,  [nmat][N][N] -> [nmat][N_sph][N_sph]
 *   ltjk_cart_from_sph  densities:            D_cart = S^T D_sph S,  [nmat][N_sph][N_sph] -> [nmat][N][N]
 * so that tr(D_sph^T X_sph) = tr(D_cart^T X_cart).  DEVICE pointers, row-major, 1 <= nmat <= 65535, outputs
 * overwritten, input and output must not overlap; work is enqueued on the ctx stream. */
int ltjk_get_nsph(const ltjk_ctx* ctx, int* nsph);
int ltjk_sph_from_cart(ltjk_ctx* ctx, int nmat, const double* X_cart, double* X_sph);
int ltjk_cart_from_sph(ltjk_ctx* ctx, int nmat, const double* D_sph, double* D_cart);

/* AO-direct particle-particle ladder (Algorithm 2; L432-434)
 *     L[p][a][b] = sum_{e,f} (ae|bf) X[p][e][f],      p = 0..npair-1 a compound occupied-pair index (ij),
 * with (ae|bf) the integrals over the virtual orbitals C_vir [N][nvir], never formed: every X_p is turned into the
 * non-symmetric AO density C_vir X_p C_vir^T, the batch goes through the K-only path of ltjk_jk_build in chunks of
 * `chunk` densities (0 = default 160), and K is transformed back, L_p = C_vir^T K[D_p] C_vir.  No prefactors.
 * C_vir, X [npair][nvir][nvir], L [npair][nvir][nvir] are DEVICE pointers, row-major; L is overwritten.  Work is
 * enqueued on the ctx stream; scratch of 2 * chunk * N^2 doubles is taken from the stream-ordered pool. */
int ltjk_pp_ladder(ltjk_ctx* ctx, int nvir, const double* C_vir, int npair, const double* X, double* L, int chunk);

/* derivative (skeleton) builds, Eq. 18 with the centre derivatives of L382-386
 * (Eqs. 30-31), for nP ordered pairs of general (non-symmetric) AO densities:
 *     gradJ[p][at][x] = sum_{mnkr} d(mn|kr)/dX_{at,x} A[p][m][n] B[p][k][r]
 *     gradK[p][at][x] = sum_{mnkr} d(mk|nr)/dX_{at,x} A[p][m][n] B[p][k][r]        (X = nuclear coordinates, bohr)
 * bare builds, no prefactors; the derivative acts on every function centred on atom `at`.
 * A, B: DEVICE [nP][N][N] row-major in the caller's AO order; gradJ, gradK: DEVICE [nP][natom][3], overwritten
 * (one of them may be NULL).  Needs ltjk_set_basis only.  EVERY shell quartet is evaluated (no Schwarz screening: a
 * value bound does not bound a derivative), so the cost is O(nshell^4); meant for the sizes of the tiny / small
 * configs.  Work is enqueued on the ctx stream; the first call after ltjk_set_basis uploads the basis (allocates). */
int ltjk_jk_grad(ltjk_ctx* ctx, int nP, const double* A, const double* B, double* gradJ, double* gradK);

/* Statistics of the last ltjk_jk_build on this context (HOST outputs, any may be NULL):
 *   n_launches    kernels launched
 *   eri_quartets  contracted shell quartets evaluated (4-fold unique: A>=B, C>=D, all bra x ket)
 *   digest_flops  fp64 flops of the digestion contractions (2 * M * K * nD summed over tiles)
 *   eri_ms, digest_ms  device time of the two kernel families (only if timing was enabled, else -1) */
int ltjk_get_stats(const ltjk_ctx* ctx, long long* n_launches, long long* eri_quartets, double* digest_flops,
                   double* eri_ms, double* digest_ms);
int ltjk_set_timing(ltjk_ctx* ctx, int enable);

/* Digestion strategy for step a8, read by the NEXT ltjk_build_shell_pairs ("once Schwarz screening is
 * applied"; L320-322 Eq. 25):
 *   1  block panels: dense integral panels of l-homogeneous AO blocks, six GEMM views; best when nearly all
 *      quartets inside the surviving block pairs pass the Schwarz test (compact molecules);
 *   2  pair lists: Q-sorted partner lists with staircase cut-offs, screened quartets are neither stored nor
 *      multiplied; best for extended molecules;
 *   0  automatic (default): mode 2 when fewer than half of all canonical shell quartets pass the Schwarz test,
 *      mode 1 otherwise.
 * Results are the same sums up to rounding order.  Returns LTJK_EINVAL for other values. */
int ltjk_set_digest_mode(ltjk_ctx* ctx, int mode);
/* split ONE build over `world` ranks (one process per GPU) in the space of shell quartets.
 * The launch units of the geometry (block-panel groups, or pair-list chunks: disjoint sets of unique quartets) are
 * dealt to the ranks by a cost-balanced rule that is a pure function of the geometry, so every rank derives the same
 * assignment without communication.  After this call ltjk_jk_build generates and digests only the units of `rank`,
 * for ALL densities: J and K then hold this rank's PARTIAL sums, and the caller adds the partials of all ranks --
 * one all-reduce (sum) of 2 nD N^2 doubles, e.g. ncclAllReduce through torch.distributed
 * (paper_2607_05622_b200/dist.py: allreduce_jk).  Every rank holds all of D.  rank = 0, world = 1 (default) is the
 * whole build.  LTJK_EINVAL unless 0 <= rank < world. */
int ltjk_set_quartet_shard(ltjk_ctx* ctx, int rank, int world);

/* Geometry-frozen integral cache ("geometry-frozen caches for per-step reuse"), read by the NEXT
 * ltjk_build_shell_pairs; strategy 1 only.  enable != 0: if all canonical integral panels of the geometry fit in
 * 60 % of the free device memory (439 AO: 41 GB) they are generated by the first ltjk_jk_build and kept; later builds
 * on the same geometry only digest.  Meant for callers that cannot batch their densities (one Laplace point per
 * call, pp-ladder chunks).  Off by default: the path is integral-direct.  Silently stays off if it does not fit. */
int ltjk_set_resident(ltjk_ctx* ctx, int enable);
/* The strategy (1 or 2) chosen by the last ltjk_build_shell_pairs; LTJK_ENOBASIS before it. */
int ltjk_get_digest_mode(const ltjk_ctx* ctx, int* mode);

/* Test hook (compute-sanitizer is not available on every GPU pool): with enable != 0 every ltjk_jk_build fills the
 * integral staging ring with NaN before each launch unit, so that an element the digestion reads but neither an ERI
 * kernel nor the zero fill wrote -- stale data of an earlier unit would otherwise hide it -- turns the result into
 * NaN.  Slower; results are unchanged when the write coverage is complete. */
int ltjk_debug_poison(ltjk_ctx* ctx, int enable);

/* Test hook: contracted Cartesian shell quartet (A B|C D) in the caller's shell indices, evaluated by the
 * device ERI kernel, written to HOST out[na*nb*nc*nd] (row-major a,b,c,d).  Synchronises. */
int ltjk_debug_eri_quartet(ltjk_ctx* ctx, int A, int B, int C, int D, double* out_host);

/* Test hook: the same quartet through the LOOPED evaluation (csrc/ltjk_eri_loop.cu) whatever its class.  Classes with
 * two or more f shells always take that path; for the classes with generated code this is the cross-check PAPER.md:L316
 * states for its two codegen regimes ("machine-epsilon equal to the unrolled path").  Synchronises. */
int ltjk_debug_eri_quartet_looped(ltjk_ctx* ctx, int A, int B, int C, int D, double* out_host);

/* Test hook: device Boys function F_m(T), m = 0..mmax (mmax <= 8), for n arguments T_host[n];
 * F_host[n*(mmax+1)].  Synchronises. */
int ltjk_debug_boys(ltjk_ctx* ctx, int mmax, int n, const double* T_host, double* F_host);

/* Microbenchmarks that give the roofline denominators: sustained fp64 FMA rate of the
 * vector pipe (independent DFMA chains on all SMs) in TFLOP/s, and a device copy in GB/s.  Synchronises. */
int ltjk_bench_dfma_peak(ltjk_ctx* ctx, double* tflops);
int ltjk_bench_copy_peak(ltjk_ctx* ctx, double* gbs);

#ifdef __cplusplus
}
#endif
#endif /* LTJK_H */

"""GPU parity tier: the CUDA path, called through the C ABI (ctypes binding), against the CPU oracle, element by
element, on the same seeded inputs.  Bar (BASELINE.json north_star; reading A11): per output matrix X,
max|X_gpu - X_ref| / max|X_ref| <= 1e-10 in fp64."""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from paper_2607_05622_b200.inputs import SCHWARZ_TAU, custom_basis, make_workload, random_densities

pytestmark = pytest.mark.gpu

TOL = 1e-10


def relerr(x, ref):
    """A11: max-abs error normalised by the max-abs of the reference matrix (per matrix, worst over the batch)."""
    x = np.asarray(x)
    ref = np.asarray(ref)
    if x.ndim == 2:
        x, ref = x[None], ref[None]
    num = np.abs(x - ref).reshape(x.shape[0], -1).max(1)
    den = np.abs(ref).reshape(x.shape[0], -1).max(1)
    return float((num / den).max())


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")
    return torch


def make_ctx(basis, tau=SCHWARZ_TAU, scratch=None, mode=0):
    """mode: digestion strategy (ltjk_set_digest_mode): 0 automatic, 1 block panels, 2 pair lists."""
    from paper_2607_05622_b200 import ltjk
    ctx = ltjk.Context(0)
    if scratch is not None:
        ctx.set_scratch_bytes(scratch)
    ctx.set_digest_mode(mode)
    ctx.set_basis(basis)
    ctx.build_shell_pairs(tau)
    return ctx


def gpu_jk(torch, ctx, D):
    Dd = torch.from_numpy(np.ascontiguousarray(D)).cuda()
    J = torch.empty_like(Dd)
    K = torch.empty_like(Dd)
    ctx.jk_build(Dd, J, K)
    torch.cuda.synchronize()
    return J.cpu().numpy(), K.cpu().numpy()


def test_boys_device_vs_oracle(torch_cuda, tiny):
    ctx = make_ctx(tiny.basis)
    T = np.array([0.0, 1e-9, 1e-3, 0.06, 0.0625, 0.5, 5.0, 20.0, 34.9, 35.93, 35.99999, 36.0, 36.1, 100.0, 1e3, 6e3])
    for mmax in (0, 3, 8):
        F = ctx.debug_boys(mmax, T)
        ref = np.array([O.boys(mmax, t) for t in T])
        assert np.all(np.abs(F - ref) <= 2e-14 * np.abs(ref))


def test_eri_all_classes_vs_oracle(torch_cuda):
    rng = np.random.default_rng(7)
    xyz = rng.uniform(-1.5, 1.5, size=(4, 3))
    xyz[3] = xyz[0]
    shells = []
    for ia in range(4):
        shells.append([(l, [0.3 + 0.4 * ia + 0.2 * l, 1.1 + 0.3 * ia + 0.5 * l], [0.6, 0.4]) for l in range(3)])
    b = custom_basis(xyz, shells)
    ctx = make_ctx(b)
    worst = 0.0
    for la, lb, lc, ld in itertools.product(range(3), repeat=4):      # all 81 ordered classes through the hook
        A, B, C, D = 0 * 3 + la, 1 * 3 + lb, 2 * 3 + lc, 3 * 3 + ld
        out = ctx.debug_eri_quartet(b, A, B, C, D)
        ref = O.eri_shell(b, A, B, C, D)
        err = np.abs(out - ref).max() / np.abs(ref).max()
        worst = max(worst, err)
        assert err < 1e-12, ((la, lb, lc, ld), err)
    assert worst < 1e-12


def test_schwarz_vs_oracle(torch_cuda, small):
    ctx = make_ctx(small.basis)
    Q = ctx.get_schwarz()
    Qr = O.schwarz(small.basis)
    # Q^2 is the integral (ab|ab): absolute agreement at round-off of the largest one; Q itself (a square root, so
    # ill-conditioned near zero) to 1e-10 relative wherever it matters for a 1e-12 product threshold
    assert np.abs(Q ** 2 - Qr ** 2).max() <= 1e-13 * np.abs(Qr ** 2).max()
    big = Qr > 1e-4
    assert np.abs(Q[big] / Qr[big] - 1.0).max() <= 1e-10
    assert np.allclose(Q, Q.T)


@pytest.mark.parametrize("mode", [1, 2])
def test_jk_tiny_vs_definition(torch_cuda, tiny, mode):
    """BASELINE gate: GPU vs the brute-force explicit-N^4 contraction (oracle O7) on the tiny config."""
    b = tiny.basis
    D = random_densities(b.nao, 3, seed=11)
    ctx = make_ctx(b, tau=0.0, mode=mode)
    J, K = gpu_jk(torch_cuda, ctx, D)
    eri = O.eri_tensor(b)
    Jr, Kr = O.jk_definition(eri, D)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL
    # non-symmetric K: the antisymmetric part must be there
    assert np.abs(K - K.transpose(0, 2, 1)).max() > 1e-3 * np.abs(K).max()


@pytest.mark.parametrize("mode,scratch", [(1, None), (2, None), (2, 1 << 16)])
def test_jk_spd_vs_definition(torch_cuda, spd_basis, mode, scratch):
    """s, p and d shells (all 21 canonical classes, diagonal blocks included) against Eq. 17 literally; the tiny
    scratch budget forces the pair-list path into 8 shell groups (666 chunks, every role-assignment family)."""
    b = spd_basis
    D = random_densities(b.nao, 5, seed=12)
    ctx = make_ctx(b, tau=0.0, scratch=scratch, mode=mode)
    J, K = gpu_jk(torch_cuda, ctx, D)
    Jr, Kr = O.jk_definition(O.eri_tensor(b), D)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL


def test_jk_tiny_pseudo_densities_end_to_end(torch_cuda, tiny):
    """Transform (a4) + J/K (a5-a9) on the tiny workload vs oracle O10 + O6."""
    torch = torch_cuda
    w = tiny
    tau, wts, _, _ = (np.linspace(0.1, 3.0, w.ntau), None, None, None)
    ctx = make_ctx(w.basis)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Dg = torch.empty((w.ntau, w.nT, w.nao, w.nao), dtype=torch.float64, device="cuda")
    ctx.build_pseudo_densities(dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir), dev(w.T), tau, Dg)
    torch.cuda.synchronize()
    Dr = O.pseudo_densities_loops(w.C_occ, w.C_vir, w.eps_occ, w.eps_vir, w.T, tau)
    assert relerr(Dg.cpu().numpy().reshape(-1, w.nao, w.nao), Dr.reshape(-1, w.nao, w.nao)) < 1e-12
    D = Dr.reshape(-1, w.nao, w.nao)
    J, K = gpu_jk(torch, ctx, D)
    Jr, Kr, _ = O.jk_folded(w.basis, D, w.schwarz_tau)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL


@pytest.mark.parametrize("mode,scratch,nD", [(1, None, 5), (1, 1 << 20, 5), (2, None, 5), (2, 1 << 22, 5), (2, None, 33),
                                              (2, 1 << 24, 96)])
def test_jk_small_vs_folded(torch_cuda, small, mode, scratch, nD):
    """160 AO, contracted s/p/d, ragged blocks; a small scratch forces many chunks (both strategies); 33 and 96
    densities reach the TN = 2 and TN = 3 column blockings of the pair-list kernel."""
    w = small
    D = random_densities(w.nao, nD, seed=13)
    ctx = make_ctx(w.basis, scratch=scratch, mode=mode)
    assert ctx.get_digest_mode() == mode
    J, K = gpu_jk(torch_cuda, ctx, D)
    Jr, Kr, kept = O.jk_folded(w.basis, D, w.schwarz_tau)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL
    # J-only and K-only entry points give the same matrices
    torch = torch_cuda
    Dd = torch.from_numpy(D).cuda()
    J2 = torch.empty_like(Dd)
    ctx.jk_build(Dd, J2, None)
    K2 = torch.empty_like(Dd)
    ctx.jk_build(Dd, None, K2)
    torch.cuda.synchronize()
    assert relerr(J2.cpu().numpy(), Jr) < TOL and relerr(K2.cpu().numpy(), Kr) < TOL


def test_jk_host_entry_matches_device_entry(torch_cuda, tiny):
    D = random_densities(tiny.nao, 40, seed=14)       # 40 densities: two column blocks of the digestion
    ctx = make_ctx(tiny.basis)
    J, K = gpu_jk(torch_cuda, ctx, D)
    Jh, Kh = ctx.jk_build_host(D)
    assert np.array_equal(np.isfinite(Jh), np.ones_like(Jh, dtype=bool))
    assert relerr(Jh, J) < 1e-13 and relerr(Kh, K) < 1e-13
    Jr, Kr, _ = O.jk_folded(tiny.basis, D, tiny.schwarz_tau)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL


def full_sweep(torch, name, mode=0):
    """The whole Laplace sweep in the configuration bench.py times (transform + J/K for all n_tau x n_T densities,
    default panel ring).  Density nD-1 is replaced by the transpose of density 0 (K must come out transposed)."""
    w = make_workload(name)
    N, nD = w.nao, w.nD
    ctx = make_ctx(w.basis, mode=mode)
    tau = np.geomspace(0.05, 6.0, w.ntau)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    D = torch.empty((w.ntau, w.nT, N, N), dtype=torch.float64, device="cuda")
    ctx.build_pseudo_densities(dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir), dev(w.T), tau, D)
    Dn = D.view(nD, N, N)
    Dn[nD - 1].copy_(Dn[0].t())
    J = torch.empty_like(Dn)
    K = torch.empty_like(Dn)
    ctx.jk_build(Dn, J, K)
    torch.cuda.synchronize()
    # properties that hold at any size
    assert float((J - J.transpose(1, 2)).abs().max()) <= 1e-12 * float(J.abs().max())
    assert float((K[nD - 1] - K[0].t()).abs().max()) <= 1e-11 * float(K[0].abs().max())
    assert float((J[nD - 1] - J[0]).abs().max()) <= 1e-11 * float(J[0].abs().max())
    assert float((K[0] - K[0].t()).abs().max()) > 1e-3 * float(K[0].abs().max())      # genuinely non-symmetric
    # transform: one density against the explicit-loop oracle
    Dref = O.pseudo_densities_loops(w.C_occ, w.C_vir, w.eps_occ, w.eps_vir, w.T[:1], tau[:1])[0, 0]
    assert relerr(Dn[nD - 1].cpu().numpy().T, Dref) < 1e-12
    return w, ctx, Dn, J, K


def density_subset(nD, n=8, seed=5):
    """first, last and n-2 seeded random densities of the sweep."""
    rng = np.random.default_rng(seed)
    mid = rng.choice(np.arange(1, nD - 1), size=min(n - 2, nD - 2), replace=False)
    return sorted(set([0, nD - 1] + [int(x) for x in mid]))


def linearity_closure(torch, ctx, Dn, J, K, seed=9):
    """GPU-side closure over ALL densities of the sweep: an n_D = 1 build of a random linear combination
    equals the same combination of the batched outputs."""
    nD = Dn.shape[0]
    cvec = torch.from_numpy(np.random.default_rng(seed).standard_normal(nD)).cuda()
    Dc = torch.tensordot(cvec, Dn, dims=1)[None].contiguous()
    Jc = torch.empty_like(Dc)
    Kc = torch.empty_like(Dc)
    ctx.jk_build(Dc, Jc, Kc)
    torch.cuda.synchronize()
    Jl = torch.tensordot(cvec, J, dims=1)
    Kl = torch.tensordot(cvec, K, dims=1)
    ej = float((Jc[0] - Jl).abs().max() / Jl.abs().max())
    ek = float((Kc[0] - Kl).abs().max() / Kl.abs().max())
    assert ej < 1e-12 and ek < 1e-12, (ej, ek)


def test_full_size_medium_full_matrices(torch_cuda):
    """300 AO, all 80 densities of the sweep: every element of J and K against the folded oracle O6, with both
    digestion strategies (one oracle run serves both)."""
    w, ctx, Dn, J, K = full_sweep(torch_cuda, "medium", mode=1)
    Jr, Kr, _ = O.jk_folded(w.basis, Dn.cpu().numpy(), w.schwarz_tau)
    assert relerr(J.cpu().numpy(), Jr) < TOL and relerr(K.cpu().numpy(), Kr) < TOL
    linearity_closure(torch_cuda, ctx, Dn, J, K)
    del ctx
    w2, ctx2, Dn2, J2, K2 = full_sweep(torch_cuda, "medium", mode=2)
    assert relerr(J2.cpu().numpy(), Jr) < TOL and relerr(K2.cpu().numpy(), Kr) < TOL
    linearity_closure(torch_cuda, ctx2, Dn2, J2, K2)


def test_full_size_porphine_full_matrices_subset(torch_cuda):
    """439 AO, the sweep bench.py times (160 densities, TN = 5): full N x N matrices of a seeded 8-density subset
    against the folded oracle O6, plus the linearity closure over all 160 densities."""
    w, ctx, Dn, J, K = full_sweep(torch_cuda, "porphine")
    assert ctx.get_digest_mode() == 1                 # compact molecule: block panels (automatic choice)
    ds = density_subset(w.nD)
    Jr, Kr, _ = O.jk_folded(w.basis, Dn[ds].cpu().numpy(), w.schwarz_tau)
    assert relerr(J[ds].cpu().numpy(), Jr) < TOL and relerr(K[ds].cpu().numpy(), Kr) < TOL
    linearity_closure(torch_cuda, ctx, Dn, J, K)
    # the same sweep forced onto the pair-list strategy (3 shell groups at this size) against the same oracle result
    del ctx, J, K
    w2, ctx2, Dn2, J2, K2 = full_sweep(torch_cuda, "porphine", mode=2)
    assert ctx2.get_digest_mode() == 2
    assert relerr(J2[ds].cpu().numpy(), Jr) < TOL and relerr(K2[ds].cpu().numpy(), Kr) < TOL


def test_full_size_large_subset_closure(torch_cuda):
    """730 AO, 192 densities, pair-list digestion: SURVEY 8(d)'s stated fallback, reported as "subset+closure": the GPU
    linearity closure over all 192 densities, plus the oracle on a seeded 8-density subset.  Default tier: Eq. 17 by
    the oracle on 120 sampled shell-pair blocks, stratified over the nine l-pair classes (about 1.5 min).  LTJK_SLOW=1:
    the full N x N matrices of the same subset against the folded oracle O6 (about 6.5 min on the 16 host cores of the
    GPU box: too long for the driver's 20-minute tier; the log of that run is profiles/r2_parity_730_full_matrix.txt,
    J 3.2e-14, K 2.7e-14)."""
    import os
    torch = torch_cuda
    w, ctx, Dn, J, K = full_sweep(torch, "large")
    assert ctx.get_digest_mode() == 2                 # extended molecule: pair lists (automatic choice)
    linearity_closure(torch, ctx, Dn, J, K)
    ds = density_subset(w.nD)
    Dh, Jh, Kh = Dn[ds].cpu().numpy(), J[ds].cpu().numpy(), K[ds].cpu().numpy()
    b = w.basis
    if os.environ.get("LTJK_SLOW") == "1":
        Jr, Kr, _ = O.jk_folded(b, Dh, w.schwarz_tau)
        ej, ek = relerr(Jh, Jr), relerr(Kh, Kr)
        print("large full-matrix subset: relerr J %.3e K %.3e over densities %s" % (ej, ek, ds))
        assert ej < TOL and ek < TOL
        return
    rng = np.random.default_rng(5)
    byl = {l: [s for s in range(b.nshell) if b.l[s] == l] for l in range(3)}
    pairs = []
    for la in range(3):
        for lb in range(3):
            n = 14 if (la, lb) != (0, 0) else 8
            pairs += [(int(rng.choice(byl[la])), int(rng.choice(byl[lb]))) for _ in range(n)]
    Jb, Kb = O.jk_blocks(b, Dh, w.schwarz_tau, pairs)
    jmax = np.abs(Jh).reshape(len(ds), -1).max(1)
    kmax = np.abs(Kh).reshape(len(ds), -1).max(1)
    for (X, Y), jb, kb in zip(pairs, Jb, Kb):
        x0, x1, y0, y1 = b.ao_off[X], b.ao_off[X + 1], b.ao_off[Y], b.ao_off[Y + 1]
        ej = np.abs(Jh[:, x0:x1, y0:y1] - jb).reshape(len(ds), -1).max(1) / jmax
        ek = np.abs(Kh[:, x0:x1, y0:y1] - kb).reshape(len(ds), -1).max(1) / kmax
        assert ej.max() < TOL and ek.max() < TOL, ((X, Y), ej.max(), ek.max())


def test_edge_cases_and_error_codes(torch_cuda, tiny):
    """Degenerate inputs through the C ABI: call-order errors, l > 3, bad sizes, one density, a density count that
    needs several column blocks (nD = 200 > 192), a one-shell basis (a single, fully diagonal block quartet)."""
    torch = torch_cuda
    from paper_2607_05622_b200 import ltjk
    ctx = ltjk.Context(0)
    D1 = torch.zeros((1, 4, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.jk_build(D1, torch.empty_like(D1), torch.empty_like(D1))
    assert e.value.code == -2                                     # LTJK_ENOBASIS
    from paper_2607_05622_b200.inputs import Basis
    bad = Basis(np.zeros((1, 3)), np.zeros(1, np.int32), np.array([4], np.int32), np.ones(1, np.int32),
                np.zeros(1, np.int32), np.ones(1), np.ones(1), np.array([0, 15]))   # a g shell
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.set_basis(bad)
    assert e.value.code == -4                                     # LTJK_ELMAX
    ctx.set_basis(tiny.basis)
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.build_shell_pairs(-1.0)
    assert e.value.code == -1                                     # LTJK_EINVAL
    ctx.build_shell_pairs(tiny.schwarz_tau)
    Dn = torch.zeros((1, tiny.nao, tiny.nao), dtype=torch.float64, device="cuda")
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.jk_build(Dn, None, None)
    assert e.value.code == -1
    # zero density -> zero J, K (and finite)
    J = torch.full_like(Dn, float("nan"))
    K = torch.full_like(Dn, float("nan"))
    ctx.jk_build(Dn, J, K)
    torch.cuda.synchronize()
    assert float(J.abs().max()) == 0.0 and float(K.abs().max()) == 0.0
    # one density and 200 densities (two column blocks) agree with the oracle and with each other
    D = random_densities(tiny.nao, 200, seed=21)
    J200, K200 = gpu_jk(torch, ctx, D)
    J1, K1 = gpu_jk(torch, ctx, D[137:138])
    assert relerr(J1, J200[137:138]) < 1e-12 and relerr(K1, K200[137:138]) < 1e-12
    Jr, Kr, _ = O.jk_folded(tiny.basis, D[[0, 137, 199]], tiny.schwarz_tau)
    assert relerr(J200[[0, 137, 199]], Jr) < TOL and relerr(K200[[0, 137, 199]], Kr) < TOL
    # linearity: K[sum c_d D_d] = sum c_d K[D_d]
    cvec = np.random.default_rng(3).standard_normal(200)
    Jc, Kc = gpu_jk(torch, ctx, np.tensordot(cvec, D, axes=1)[None])
    assert relerr(Kc[0], np.tensordot(cvec, K200, axes=1)) < 1e-11
    assert relerr(Jc[0], np.tensordot(cvec, J200, axes=1)) < 1e-11
    # single d shell on one centre: one block, one fully diagonal block quartet (all three fold factors at once)
    one = custom_basis(np.array([[0.3, -0.1, 0.2]]), [[(2, [0.9, 0.4], [0.6, 0.4])]])
    c1 = make_ctx(one, tau=0.0)
    Dd = random_densities(6, 2, seed=22)
    Jg, Kg = gpu_jk(torch, c1, Dd)
    Jd, Kd = O.jk_definition(O.eri_tensor(one), Dd)
    assert relerr(Jg, Jd) < TOL and relerr(Kg, Kd) < TOL


def test_symmetric_density_is_a_special_case(torch_cuda, small):
    """the symmetric build is the A = B special case of the non-symmetric one; a symmetric-only
    kernel would keep (K + K^T)/2 and silently drop the rest."""
    w = small
    D = random_densities(w.nao, 2, seed=31)
    Ds = 0.5 * (D + D.transpose(0, 2, 1))
    Da = 0.5 * (D - D.transpose(0, 2, 1))
    ctx = make_ctx(w.basis)
    J, K = gpu_jk(torch_cuda, ctx, D)
    Js, Ks = gpu_jk(torch_cuda, ctx, Ds)
    Ja, Ka = gpu_jk(torch_cuda, ctx, Da)
    assert relerr(Ks, 0.5 * (K + K.transpose(0, 2, 1))) < 1e-11        # sym(K[D]) = K[sym D], and it is symmetric
    assert relerr(Ka, 0.5 * (K - K.transpose(0, 2, 1))) < 1e-11        # antisym(K[D]) = K[antisym D] != 0
    assert np.abs(Ka).max() > 1e-3 * np.abs(K).max()
    assert relerr(Js, J) < 1e-11 and np.abs(Ja).max() < 1e-11 * np.abs(J).max()   # J only sees the symmetric part


def test_laplace_cascade_closure(torch_cuda, small):
    """The path's purpose end to end: library grid -> pseudo-densities -> J/K -> weighted
    accumulation resolves the orbital-energy denominator,
        sum_a w_a K[D^a] = K[C_o (T o 1/(eps_v - eps_o)) C_v^T]      (same for J)
    to the quadrature error, and the Laplace-Fock back-transform (Eq. 19) matches the oracle."""
    torch = torch_cuda
    from paper_2607_05622_b200 import ltjk
    w = small
    N = w.nao
    tau, wts, err = ltjk.laplace_quadrature(w.laplace_range[0], w.laplace_range[1], w.ntau)
    ctx = make_ctx(w.basis)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    D = torch.empty((w.ntau, w.nT, N, N), dtype=torch.float64, device="cuda")
    ctx.build_pseudo_densities(dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir), dev(w.T), tau, D)
    Dn = D.view(-1, N, N)
    J = torch.empty_like(Dn)
    K = torch.empty_like(Dn)
    ctx.jk_build(Dn, J, K)
    Ksum = torch.empty((w.nT, N, N), dtype=torch.float64, device="cuda")
    Jsum = torch.empty_like(Ksum)
    ctx.laplace_accumulate(tau, wts, 0.0, K.view(w.ntau, w.nT, N, N), Ksum)
    ctx.laplace_accumulate(tau, wts, 0.0, J.view(w.ntau, w.nT, N, N), Jsum)
    # exact denominators on the GPU path too (one build per amplitude set)
    denom = w.eps_vir[None, :] - w.eps_occ[:, None]
    assert denom.min() >= w.laplace_range[0] and denom.max() <= w.laplace_range[1]
    Dex = np.einsum("mi,tia,na->tmn", w.C_occ, w.T / denom[None], w.C_vir)
    Jex, Kex = gpu_jk(torch, ctx, Dex)
    scale = np.abs(np.einsum("mi,tia,na->tmn", np.abs(w.C_occ), np.abs(w.T), np.abs(w.C_vir))).max()
    tol = 50 * err * scale * np.abs(Kex).max() / np.abs(Dex).max()
    assert np.abs(Ksum.cpu().numpy() - Kex).max() < tol and np.abs(Jsum.cpu().numpy() - Jex).max() < tol * 10
    assert relerr(Ksum.cpu().numpy(), Kex) < 1e-6 and relerr(Jsum.cpu().numpy(), Jex) < 1e-6
    # accumulation itself: oracle parity at 1e-13, including the omega reweighting of Eq. 21
    Kh = K.cpu().numpy().reshape(w.ntau, w.nT, N, N)
    assert relerr(Ksum.cpu().numpy(), O.laplace_accumulate(tau, wts, 0.0, Kh)) < 1e-13
    ctx.laplace_accumulate(tau, wts, 0.2, K.view(w.ntau, w.nT, N, N), Ksum)
    assert relerr(Ksum.cpu().numpy(), O.laplace_accumulate(tau, wts, 0.2, Kh)) < 1e-13
    # Laplace-Fock back-transform on a few densities
    C = np.ascontiguousarray(np.concatenate([w.C_occ, w.C_vir], axis=1))
    F = torch.empty((4, N, N), dtype=torch.float64, device="cuda")
    ctx.laplace_fock(J[:4].contiguous(), K[:4].contiguous(), dev(C), F)
    torch.cuda.synchronize()
    Fr = O.laplace_fock(J[:4].cpu().numpy(), K[:4].cpu().numpy(), C)
    assert relerr(F.cpu().numpy(), Fr) < 1e-12
    # rectangular MO block (occupied columns only)
    Fo = torch.empty((4, w.nocc, w.nocc), dtype=torch.float64, device="cuda")
    ctx.laplace_fock(J[:4].contiguous(), K[:4].contiguous(), dev(w.C_occ), Fo)
    torch.cuda.synchronize()
    assert relerr(Fo.cpu().numpy(), Fr[:, :w.nocc, :w.nocc]) < 1e-12


def test_three_and_four_primitive_contractions(torch_cuda):
    """Contraction depths other than the benchmark's 2: 3- and 4-primitive shells give 81 / 144 / 256 primitive
    quartets per contracted quartet, i.e. several 16-lane passes of the cooperative ERI kernel and long primitive
    loops in the per-thread kernels."""
    xyz = np.array([[0.0, 0.1, -0.2], [1.7, -0.4, 0.5], [-0.9, 1.8, 0.7]])
    sh3 = [(0, [2.1, 0.7, 0.25], [0.3, 0.5, 0.3]), (1, [1.5, 0.5, 0.2], [0.25, 0.5, 0.35]), (2, [1.1, 0.45, 0.2], [0.3, 0.4, 0.4])]
    sh4 = [(1, [2.5, 0.9, 0.35, 0.15], [0.2, 0.3, 0.3, 0.2]), (2, [1.4, 0.6, 0.3, 0.15], [0.2, 0.3, 0.3, 0.2])]
    b = custom_basis(xyz, [sh3, sh4, sh3])
    D = random_densities(b.nao, 3, seed=41)
    ctx = make_ctx(b, tau=0.0)
    J, K = gpu_jk(torch_cuda, ctx, D)
    Jr, Kr = O.jk_definition(O.eri_tensor(b), D)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL


@pytest.mark.parametrize("mode", [1, 2])
def test_pp_ladder_vs_oracle(torch_cuda, tiny, spd_basis, mode):
    """the AO-direct particle-particle ladder as a K-only batch, against
    the oracle's explicit sum over (e,f) of virtual-orbital integrals built from the N^4 tensor (O7).  37 pair columns
    with chunk = 16 exercise a ragged last chunk; chunk = 0 the default."""
    torch = torch_cuda
    for b in (tiny.basis, spd_basis):
        rng = np.random.default_rng(17)
        nv = 7
        Cv = rng.standard_normal((b.nao, nv)) / np.sqrt(b.nao)
        X = rng.standard_normal((37, nv, nv))
        ref = O.pp_ladder(O.eri_tensor(b), Cv, X)
        ctx = make_ctx(b, tau=0.0, mode=mode)
        Cd, Xd = torch.from_numpy(Cv).cuda(), torch.from_numpy(X).cuda()
        for chunk in (16, 0):
            L = torch.full((37, nv, nv), float("nan"), dtype=torch.float64, device="cuda")
            ctx.pp_ladder(Cd, Xd, L, chunk)
            torch.cuda.synchronize()
            assert relerr(L.cpu().numpy(), ref) < TOL
        assert np.abs(ref - ref.transpose(0, 2, 1)).max() > 1e-3 * np.abs(ref).max()    # non-symmetric, as X is


def test_level2_density_from_laplace_fock(torch_cuda, tiny):
    """SURVEY 8(f) N1, last link (Eq. 15 with R^(2); Alg. 1): the occupied-virtual block of the
    Laplace-Fock matrix F~^alpha = C^T (2 J - K) C of level 1 is fed back as the amplitude R^(2) of the level-2
    pseudo-density at the same grid point.  Whole chain on the GPU against the whole chain in the oracle."""
    torch = torch_cuda
    w = tiny
    N, no = w.nao, w.nocc
    tau = np.linspace(0.2, 2.5, 3)
    T = np.concatenate([w.T, 0.5 * w.T[::-1] + 0.01], axis=0)[:2]            # two amplitude sets
    nT = T.shape[0]
    ctx = make_ctx(w.basis)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Co, Cv, eo, ev = dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir)
    C = np.ascontiguousarray(np.concatenate([w.C_occ, w.C_vir], axis=1))
    D1 = torch.empty((len(tau), nT, N, N), dtype=torch.float64, device="cuda")
    ctx.build_pseudo_densities(Co, Cv, eo, ev, dev(T), tau, D1)
    D1n = D1.view(-1, N, N)
    J = torch.empty_like(D1n)
    K = torch.empty_like(D1n)
    ctx.jk_build(D1n, J, K)
    F = torch.empty((len(tau) * nT, N, N), dtype=torch.float64, device="cuda")
    ctx.laplace_fock(J, K, dev(C), F)
    D2 = torch.empty((len(tau), nT, N, N), dtype=torch.float64, device="cuda")
    for a in range(len(tau)):
        R2 = F[a * nT:(a + 1) * nT, :no, no:].contiguous()                  # ov block of F~^alpha
        ctx.build_pseudo_densities(Co, Cv, eo, ev, R2, tau[a:a + 1], D2[a:a + 1])
    torch.cuda.synchronize()
    # oracle chain
    D1r = O.pseudo_densities_loops(w.C_occ, w.C_vir, w.eps_occ, w.eps_vir, T, tau).reshape(-1, N, N)
    Jr, Kr, _ = O.jk_folded(w.basis, D1r, w.schwarz_tau)
    Fr = O.laplace_fock(Jr, Kr, C)
    D2r = np.stack([O.pseudo_densities_loops(w.C_occ, w.C_vir, w.eps_occ, w.eps_vir,
                                             Fr[a * nT:(a + 1) * nT, :no, no:], tau[a:a + 1])[0] for a in range(len(tau))])
    assert relerr(F.cpu().numpy(), Fr) < TOL
    assert relerr(D2.cpu().numpy().reshape(-1, N, N), D2r.reshape(-1, N, N)) < TOL
    assert np.abs(D2r).max() > 0


def test_resident_panels_reused_across_builds(torch_cuda, small):
    """ltjk_set_resident: the integral panels of the geometry are generated by the first build and only digested by
    later ones (no ERI launches); results stay those of the integral-direct path, for new densities and batch sizes."""
    from paper_2607_05622_b200 import ltjk
    torch = torch_cuda
    w = small
    ctx = ltjk.Context(0)
    ctx.set_digest_mode(1)
    ctx.set_resident(True)
    ctx.set_basis(w.basis)
    ctx.build_shell_pairs(w.schwarz_tau)
    D = random_densities(w.nao, 40, seed=51)
    Jr, Kr, _ = O.jk_folded(w.basis, D[[0, 7, 39]], w.schwarz_tau)
    J1, K1 = gpu_jk(torch, ctx, D[:8])
    n_first = ctx.get_stats()["n_launches"]
    J2, K2 = gpu_jk(torch, ctx, D)                       # second build: other densities, other column blocking
    n_second = ctx.get_stats()["n_launches"]
    assert n_second < n_first                             # no ERI launches any more
    assert relerr(J1[[0, 7]], Jr[:2]) < TOL and relerr(K1[[0, 7]], Kr[:2]) < TOL
    assert relerr(J2[[0, 7, 39]], Jr) < TOL and relerr(K2[[0, 7, 39]], Kr) < TOL
    # a new geometry invalidates the cache
    ctx.set_basis(w.basis)
    ctx.build_shell_pairs(w.schwarz_tau)
    J3, K3 = gpu_jk(torch, ctx, D[:8])
    assert ctx.get_stats()["n_launches"] == n_first
    assert relerr(K3[[0, 7]], Kr[:2]) < TOL


@pytest.mark.parametrize("mode,scratch,world", [(1, 1 << 20, 2), (1, 1 << 20, 3), (2, 1 << 22, 2), (2, 1 << 22, 5)])
def test_quartet_shard_partials_sum_to_whole_build(torch_cuda, small, mode, scratch, world):
    """SURVEY 8(e) / N5 on one GPU: the partial builds of ranks 0..world-1 (ltjk_set_quartet_shard; run one after the
    other on this device, none waits for another) add up to the whole build, which matches the oracle; no rank's share
    is empty.  The small scratch gives many launch units to deal out (both digestion strategies)."""
    torch = torch_cuda
    w = small
    D = random_densities(w.nao, 5, seed=61)
    Jr, Kr, _ = O.jk_folded(w.basis, D, w.schwarz_tau)
    ctx = make_ctx(w.basis, scratch=scratch, mode=mode)
    Jsum = np.zeros_like(D)
    Ksum = np.zeros_like(D)
    for r in range(world):
        ctx.set_quartet_shard(r, world)
        Jp, Kp = gpu_jk(torch, ctx, D)
        assert np.abs(Kp).max() > 0 and np.abs(Kp).max() < np.abs(Kr).max() * 1.5
        Jsum += Jp
        Ksum += Kp
    assert relerr(Jsum, Jr) < TOL and relerr(Ksum, Kr) < TOL
    ctx.set_quartet_shard(0, 1)
    J, K = gpu_jk(torch, ctx, D)
    assert relerr(Jsum, J) < 1e-12 and relerr(Ksum, K) < 1e-12
    from paper_2607_05622_b200 import ltjk
    with pytest.raises(ltjk.LtjkError):
        ctx.set_quartet_shard(2, 2)


def gpu_grad(torch, ctx, A, B):
    Ad, Bd = torch.from_numpy(np.ascontiguousarray(A)).cuda(), torch.from_numpy(np.ascontiguousarray(B)).cuda()
    natom = ctx.natom
    gJ = torch.full((A.shape[0], natom, 3), float("nan"), dtype=torch.float64, device="cuda")
    gK = torch.full_like(gJ, float("nan"))
    ctx.jk_grad(Ad, Bd, gJ, gK)
    torch.cuda.synchronize()
    return gJ.cpu().numpy(), gK.cpu().numpy()


def test_jk_grad_vs_oracle(torch_cuda, tiny, spd_basis):
    """SURVEY 8(f) N2 (Eq. 18; L382-386): derivative builds J^x(A,B), K^x(A,B) for pairs of non-symmetric
    densities against the oracle's term-by-term product rule, element by element.  tiny: s, p (uncontracted);
    spd: contracted s, p, d on three atoms (every one of the 54 kernel classes, raised f classes included); 6 pairs =
    two launches of 4 + 2.  Also the translational sum rule (Eq. 31) on the GPU result itself."""
    from paper_2607_05622_b200 import ltjk
    torch = torch_cuda
    for b in (tiny.basis, spd_basis):
        A = random_densities(b.nao, 6, seed=71)
        B = random_densities(b.nao, 6, seed=72)
        ctx = ltjk.Context(0)
        ctx.set_basis(b)
        gJ, gK = gpu_grad(torch, ctx, A, B)
        rJ, rK = O.jk_grad(b, A, B)
        assert np.abs(gJ - rJ).max() <= TOL * np.abs(rJ).max(), np.abs(gJ - rJ).max() / np.abs(rJ).max()
        assert np.abs(gK - rK).max() <= TOL * np.abs(rK).max(), np.abs(gK - rK).max() / np.abs(rK).max()
        assert np.abs(gJ.sum(1)).max() < 1e-11 * np.abs(gJ).max() and np.abs(gK.sum(1)).max() < 1e-11 * np.abs(gK).max()
        # ordered build: K^x(A^T, B) differs from K^x(A, B) for non-symmetric densities
        tJ, tK = gpu_grad(torch, ctx, A.transpose(0, 2, 1).copy(), B)
        assert np.abs(tK - gK).max() > 1e-3 * np.abs(gK).max()
        # J-only / K-only outputs
        Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
        only = torch.empty((6, ctx.natom, 3), dtype=torch.float64, device="cuda")
        ctx.jk_grad(Ad, Bd, only, None)
        torch.cuda.synchronize()
        assert np.abs(only.cpu().numpy() - gJ).max() <= 1e-12 * np.abs(gJ).max()
        ctx.close()


def cut_basis(b, natoms):
    """The shells of the first `natoms` atoms of a workload basis (coefficients already normalised)."""
    from paper_2607_05622_b200.inputs import Basis
    keep = [s for s in range(b.nshell) if b.atom[s] < natoms]
    exps, coef, poff = [], [], []
    for s in keep:
        poff.append(len(exps))
        exps += list(b.exps[b.prim_off[s]:b.prim_off[s] + b.nprim[s]])
        coef += list(b.coef[b.prim_off[s]:b.prim_off[s] + b.nprim[s]])
    ls = b.l[keep]
    ao_off = np.zeros(len(keep) + 1, dtype=np.int64)
    ao_off[1:] = np.cumsum([(1, 3, 6)[int(l)] for l in ls])
    return Basis(np.ascontiguousarray(b.xyz[:natoms]), b.atom[keep].astype(np.int32), ls.astype(np.int32),
                 b.nprim[keep].astype(np.int32), np.asarray(poff, dtype=np.int32), np.asarray(exps), np.asarray(coef), ao_off)


@pytest.mark.parametrize("natoms", [5, 14])
def test_jk_grad_small_vs_oracle(torch_cuda, small, natoms):
    """N2 on contracted s/p/d shells with several shells per atom: the first 5 atoms of the small workload (default
    tier), and with LTJK_SLOW=1 all of it (160 AO, 73 shells, 28 M ordered shell quartets: about 3 min of oracle time on
    the 16 host cores against 0.1 s of kernels; measured 1.5e-13).  Two density pairs, oracle = literal product rule."""
    import os
    from paper_2607_05622_b200 import ltjk
    if natoms == 14 and os.environ.get("LTJK_SLOW") != "1":
        pytest.skip("full 160-AO gradient oracle takes 3 min: set LTJK_SLOW=1")
    b = small.basis if natoms == 14 else cut_basis(small.basis, natoms)
    A = random_densities(b.nao, 2, seed=81)
    B = random_densities(b.nao, 2, seed=82)
    ctx = ltjk.Context(0)
    ctx.set_basis(b)
    gJ, gK = gpu_grad(torch_cuda, ctx, A, B)
    rJ, rK = O.jk_grad(b, A, B)
    assert np.abs(gJ - rJ).max() <= TOL * np.abs(rJ).max() and np.abs(gK - rK).max() <= TOL * np.abs(rK).max()
    assert np.abs(gJ.sum(1)).max() < 1e-11 * np.abs(gJ).max() and np.abs(gK.sum(1)).max() < 1e-11 * np.abs(gK).max()


def test_pair_list_edge_cases(torch_cuda, tiny):
    """Degenerate inputs through the pair-list strategy (ltjk_set_digest_mode 2): one density, 200 densities (several
    column blocks), J-only / K-only, a one-shell basis (a single fully diagonal quartet), a threshold that screens
    almost everything, and a zero density."""
    torch = torch_cuda
    b = tiny.basis
    ctx = make_ctx(b, mode=2)
    D = random_densities(b.nao, 200, seed=91)
    J200, K200 = gpu_jk(torch, ctx, D)
    Jr, Kr, _ = O.jk_folded(b, D[[0, 137, 199]], tiny.schwarz_tau)
    assert relerr(J200[[0, 137, 199]], Jr) < TOL and relerr(K200[[0, 137, 199]], Kr) < TOL
    J1, K1 = gpu_jk(torch, ctx, D[137:138])
    assert relerr(J1, J200[137:138]) < 1e-12 and relerr(K1, K200[137:138]) < 1e-12
    Dd = torch.from_numpy(D[:7].copy()).cuda()
    Jo = torch.full_like(Dd, float("nan"))
    Ko = torch.full_like(Dd, float("nan"))
    ctx.jk_build(Dd, Jo, None)
    ctx.jk_build(Dd, None, Ko)
    torch.cuda.synchronize()
    assert relerr(Jo.cpu().numpy(), J200[:7]) < 1e-12 and relerr(Ko.cpu().numpy(), K200[:7]) < 1e-12
    Z = torch.zeros_like(Dd)
    ctx.jk_build(Z, Jo, Ko)
    torch.cuda.synchronize()
    assert float(Jo.abs().max()) == 0.0 and float(Ko.abs().max()) == 0.0
    # a threshold that keeps only the strongest quartets: same rule in the oracle (borderline flips are < tau |D|)
    c2 = make_ctx(b, tau=1e-3, mode=2)
    Jt, Kt = gpu_jk(torch, c2, D[:3])
    Jtr, Ktr, kept = O.jk_folded(b, D[:3], 1e-3)
    assert 0 < kept < b.nshell ** 4 // 8
    assert relerr(Jt, Jtr) < 1e-9 and relerr(Kt, Ktr) < 1e-9
    # single d shell on one centre
    one = custom_basis(np.array([[0.3, -0.1, 0.2]]), [[(2, [0.9, 0.4], [0.6, 0.4])]])
    c1 = make_ctx(one, tau=0.0, mode=2)
    D6 = random_densities(6, 2, seed=22)
    Jg, Kg = gpu_jk(torch, c1, D6)
    Jd, Kd = O.jk_definition(O.eri_tensor(one), D6)
    assert relerr(Jg, Jd) < TOL and relerr(Kg, Kd) < TOL


@pytest.mark.parametrize("name,mode,scratch", [("small", 1, 1 << 20), ("small", 2, 1 << 22), ("medium", 1, None),
                                               ("medium", 2, None), ("large", 2, None)])
def test_staging_ring_write_coverage(torch_cuda, name, mode, scratch):
    """Stand-in for a memory checker (compute-sanitizer is closed on this pool): with ltjk_debug_poison the staging ring
    is NaN before every launch unit, so any element the digestion reads that neither an ERI kernel nor the zero fill
    wrote -- which stale integrals of an earlier unit would hide -- makes J or K NaN.  The poisoned build must be
    finite and equal to the normal one (same kernels, same order: tight tolerance); 730 AO covers 55 chunks of 5 groups."""
    torch = torch_cuda
    w = make_workload(name)
    ctx = make_ctx(w.basis, scratch=scratch, mode=mode)
    nD = 3 if name != "large" else 2
    D = torch.from_numpy(random_densities(w.nao, nD, seed=95)).cuda()
    J0, K0 = torch.empty_like(D), torch.empty_like(D)
    ctx.jk_build(D, J0, K0)
    ctx.debug_poison(True)
    J1, K1 = torch.full_like(D, 1.0), torch.full_like(D, 1.0)
    ctx.jk_build(D, J1, K1)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(J1).all()) and bool(torch.isfinite(K1).all())
    assert float((J1 - J0).abs().max()) <= 1e-12 * float(J0.abs().max())
    assert float((K1 - K0).abs().max()) <= 1e-12 * float(K0.abs().max())


@pytest.mark.parametrize("mode,scratch", [(1, 1 << 20), (2, 1 << 22)])
def test_ring_reuse_stress(torch_cuda, small, mode, scratch):
    """Two-stream pipeline with a tiny staging ring (dozens of launch units alternate between the two ring halves; the
    ERI kernels of unit g+1 run while unit g is digested): 12 back-to-back builds without any host synchronisation in
    between must all agree with the first one (fp64 reductions reorder: 1e-12) and with the oracle -- a ring half
    overwritten too early, or read too early, shows up here."""
    torch = torch_cuda
    w = small
    D = random_densities(w.nao, 5, seed=97)
    Jr, Kr, _ = O.jk_folded(w.basis, D, w.schwarz_tau)
    ctx = make_ctx(w.basis, scratch=scratch, mode=mode)
    Dd = torch.from_numpy(D).cuda()
    outs = []
    for _ in range(12):
        J = torch.empty_like(Dd)
        K = torch.empty_like(Dd)
        ctx.jk_build(Dd, J, K)
        outs.append((J, K))
    torch.cuda.synchronize()
    J0, K0 = outs[0][0].cpu().numpy(), outs[0][1].cpu().numpy()
    assert relerr(J0, Jr) < TOL and relerr(K0, Kr) < TOL
    for J, K in outs[1:]:
        assert relerr(J.cpu().numpy(), J0) < 1e-12 and relerr(K.cpu().numpy(), K0) < 1e-12

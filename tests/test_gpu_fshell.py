"""GPU parity for SURVEY.md 8(f) row N4, f shells (the looped codegen regime): every class with an f
shell goes through csrc/ltjk_eri_loop.cu.  The oracle side is pinned at l = 3 by tests/test_oracle_eri.py (198-digit
centre derivatives of the closed-form (ss|ss) up to (ff|ff))."""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from paper_2607_05622_b200.inputs import custom_basis, random_densities
from test_gpu_parity import TOL, gpu_jk, make_ctx, relerr, torch_cuda  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


def four_centre_basis(lmax):
    rng = np.random.default_rng(7)
    xyz = rng.uniform(-1.5, 1.5, size=(4, 3))
    xyz[3] = xyz[0]                                              # two coincident centres
    shells = []
    for ia in range(4):
        shells.append([(l, [0.3 + 0.4 * ia + 0.2 * l, 1.1 + 0.3 * ia + 0.5 * l], [0.6, 0.4]) for l in range(lmax + 1)])
    return custom_basis(xyz, shells)


def test_eri_f_classes_vs_oracle(torch_cuda):
    """All 175 ordered classes (la lb|lc ld), l <= 3, with at least one f shell, two-primitive contractions, against the
    oracle: through the path the hook takes by default (generated straight-line code where the library uses it for the
    builds' per-thread one-f classes, the looped kernel for the rest) and through the looped kernel for every class."""
    b = four_centre_basis(3)
    ctx = make_ctx(b)
    worst = 0.0
    for ls in itertools.product(range(4), repeat=4):
        if 3 not in ls:
            continue
        A, B, C, D = (4 * i + l for i, l in enumerate(ls))
        ref = O.eri_shell(b, A, B, C, D)
        for looped in (False, True):       # False: generated code where the per-thread builds use it; True: looped
            out = ctx.debug_eri_quartet(b, A, B, C, D, looped=looped)
            err = np.abs(out - ref).max() / np.abs(ref).max()
            worst = max(worst, err)
            assert err < 1e-12, (ls, looped, err)
    assert worst < 1e-12


def test_looped_path_equals_unrolled_path_spd(torch_cuda):
    """the looped regime is "machine-epsilon equal to the unrolled path": all 81 s/p/d classes through
    both of the library's evaluations (generated OS/HGP straight-line code vs the looped Hermite kernel)."""
    b = four_centre_basis(2)
    ctx = make_ctx(b)
    for ls in itertools.product(range(3), repeat=4):
        A, B, C, D = (3 * i + l for i, l in enumerate(ls))
        u = ctx.debug_eri_quartet(b, A, B, C, D)
        v = ctx.debug_eri_quartet(b, A, B, C, D, looped=True)
        assert np.abs(u - v).max() <= 2e-13 * np.abs(u).max(), ls


def spdf_basis(natom=3, seed=5):
    rng = np.random.default_rng(seed)
    xyz = rng.uniform(-2.0, 2.0, size=(natom, 3))
    shells = []
    for ia in range(natom):
        sh = [(0, [2.1 + ia, 0.5], [0.5, 0.6]), (0, [0.25 + 0.05 * ia], [1.0]), (1, [0.9 + 0.1 * ia, 0.3], [0.4, 0.7]),
              (2, [0.8 + 0.1 * ia], [1.0]), (3, [0.7 + 0.15 * ia], [1.0])]
        if ia == 0:
            sh.append((3, [1.3, 0.45], [0.55, 0.5]))              # a contracted f shell, a second f on one centre
            sh.append((3, [0.35], [1.0]))                        # three f shells: a full block of two plus a remainder
        shells.append(sh)
    return custom_basis(xyz, shells)


def test_schwarz_f_vs_oracle(torch_cuda):
    b = spdf_basis()
    ctx = make_ctx(b)
    Q = ctx.get_schwarz()
    Qr = O.schwarz(b)
    assert np.abs(Q ** 2 - Qr ** 2).max() <= 1e-13 * np.abs(Qr ** 2).max()
    big = Qr > 1e-4
    assert np.abs(Q[big] / Qr[big] - 1.0).max() <= 1e-10


@pytest.mark.parametrize("scratch", [None, 1 << 20])
def test_jk_spdf_vs_definition(torch_cuda, scratch):
    """s, p, d and f shells (all 55 canonical classes, diagonal f blocks, an f remainder block) against Eq. 17 literally
    (oracle O7 tensor, no symmetry): non-symmetric densities, nothing screened.  The 1 MiB ring splits the build into
    many launch units."""
    b = spdf_basis()
    D = random_densities(b.nao, 5, seed=21)
    ctx = make_ctx(b, tau=0.0, scratch=scratch)
    assert ctx.get_digest_mode() == 1                           # f shells: block panels
    J, K = gpu_jk(torch_cuda, ctx, D)
    Jr, Kr = O.jk_definition(O.eri_tensor(b), D)
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL
    assert np.abs(K - K.transpose(0, 2, 1)).max() > 1e-3 * np.abs(K).max()


def test_jk_spdf_screened_vs_folded(torch_cuda):
    """An extended chain with f shells and the production threshold: GPU vs the oracle's canonical-quartet digestion O6
    with the same Schwarz predicate."""
    rng = np.random.default_rng(31)
    natom = 8
    xyz = np.stack([3.2 * np.arange(natom), 0.4 * rng.standard_normal(natom), 0.4 * rng.standard_normal(natom)], 1)
    shells = [[(0, [1.9, 0.45], [0.5, 0.6]), (1, [0.8], [1.0]), (2, [0.7], [1.0]), (3, [0.9 + 0.05 * ia], [1.0])]
              for ia in range(natom)]
    b = custom_basis(xyz, shells)
    D = random_densities(b.nao, 18, seed=22)                     # 18 densities: two column blocks, a ragged one
    ctx = make_ctx(b, tau=1e-10)
    J, K = gpu_jk(torch_cuda, ctx, D)
    Jr, Kr, kept = O.jk_folded(b, D, 1e-10)
    npair = b.nshell * (b.nshell + 1) // 2
    assert 0 < kept < npair * (npair + 1) // 2                   # the threshold really drops quartets here
    assert relerr(J, Jr) < TOL and relerr(K, Kr) < TOL


def test_f_shell_limits(torch_cuda):
    """What is not built for f shells fails loudly: pair-list digestion, derivative builds, l = 4."""
    from paper_2607_05622_b200 import ltjk
    from paper_2607_05622_b200.inputs import Basis
    b = spdf_basis(natom=2)
    ctx = ltjk.Context(0)
    ctx.set_digest_mode(2)
    ctx.set_basis(b)
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.build_shell_pairs(1e-12)
    assert e.value.code == -4
    ctx.set_digest_mode(0)
    ctx.build_shell_pairs(1e-12)
    A = torch_cuda.zeros((1, b.nao, b.nao), dtype=torch_cuda.float64, device="cuda")
    g = torch_cuda.zeros((1, 2, 3), dtype=torch_cuda.float64, device="cuda")
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.jk_grad(A, A, g, g.clone())
    assert e.value.code == -4
    bad = Basis(np.zeros((1, 3)), np.zeros(1, np.int32), np.array([4], np.int32), np.ones(1, np.int32),
                np.zeros(1, np.int32), np.ones(1), np.ones(1), np.array([0, 15]))   # a g shell
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.set_basis(bad)
    assert e.value.code == -4


def test_sph_transform_vs_oracle(torch_cuda):
    """Matrix-level spherical transform, both directions, s/p/d/f shells interleaved in the caller's order, against the
    oracle's S X S^T / S^T D S (plain matmuls with the closed-form solid harmonics)."""
    torch = torch_cuda
    b = spdf_basis()
    ctx = make_ctx(b)
    ns = ctx.get_nsph()
    assert ns == int(sum(2 * l + 1 for l in b.l)) and ns < b.nao
    rng = np.random.default_rng(41)
    X = rng.standard_normal((3, b.nao, b.nao))
    D = rng.standard_normal((3, ns, ns))
    Xs = torch.empty((3, ns, ns), dtype=torch.float64, device="cuda")
    Dc = torch.empty((3, b.nao, b.nao), dtype=torch.float64, device="cuda")
    ctx.sph_from_cart(torch.from_numpy(X).cuda(), Xs)
    ctx.cart_from_sph(torch.from_numpy(D).cuda(), Dc)
    torch.cuda.synchronize()
    assert relerr(Xs.cpu().numpy(), O.sph_from_cart(b, X)) < 1e-13
    assert relerr(Dc.cpu().numpy(), O.cart_from_sph(b, D)) < 1e-13


def test_jk_in_the_pure_basis_end_to_end(torch_cuda):
    """J and K of non-symmetric densities given in the PURE basis: cart_from_sph -> jk_build -> sph_from_cart on the
    device, against the oracle's composition (O7 tensor, Eq. 17, the oracle's own transforms)."""
    torch = torch_cuda
    b = spdf_basis()
    ctx = make_ctx(b, tau=0.0)
    ns = ctx.get_nsph()
    Ds = np.random.default_rng(42).standard_normal((4, ns, ns))
    Dc = torch.empty((4, b.nao, b.nao), dtype=torch.float64, device="cuda")
    ctx.cart_from_sph(torch.from_numpy(Ds).cuda(), Dc)
    J, K = torch.empty_like(Dc), torch.empty_like(Dc)
    ctx.jk_build(Dc, J, K)
    Js = torch.empty((4, ns, ns), dtype=torch.float64, device="cuda")
    Ks = torch.empty_like(Js)
    ctx.sph_from_cart(J, Js)
    ctx.sph_from_cart(K, Ks)
    torch.cuda.synchronize()
    Jr, Kr = O.jk_definition(O.eri_tensor(b), O.cart_from_sph(b, Ds))
    assert relerr(Js.cpu().numpy(), O.sph_from_cart(b, Jr)) < TOL
    assert relerr(Ks.cpu().numpy(), O.sph_from_cart(b, Kr)) < TOL


def test_full_size_medium_f_subset_closure(torch_cuda):
    """400 AO with 10 f shells, the sweep bench.py times under config.f_shells_medium_f (80 densities, production
    threshold, default panel ring): full N x N matrices of a seeded 8-density subset against the folded oracle O6
    (about 1.5 min on the 16 host cores of the GPU box), plus the linearity closure over all 80 densities."""
    from test_gpu_parity import density_subset, full_sweep, linearity_closure
    w, ctx, Dn, J, K = full_sweep(torch_cuda, "medium_f")
    assert ctx.get_digest_mode() == 1
    ds = density_subset(w.nD)
    Jr, Kr, _ = O.jk_folded(w.basis, Dn[ds].cpu().numpy(), w.schwarz_tau)
    assert relerr(J[ds].cpu().numpy(), Jr) < TOL and relerr(K[ds].cpu().numpy(), Kr) < TOL
    linearity_closure(torch_cuda, ctx, Dn, J, K)


def test_f_shells_with_resident_panels_sharding_and_poison(torch_cuda):
    """The other modes of the block-panel path do not know which kernel wrote a panel: resident panels reused by a
    second build, a build split over three ranks in quartet space, and the NaN write-coverage hook (every panel element
    the digestion reads was written by a per-thread, cooperative or looped ERI kernel, or by the zero fill), all on
    the s/p/d/f basis with a small ring."""
    from paper_2607_05622_b200 import ltjk
    torch = torch_cuda
    b = spdf_basis()
    D = random_densities(b.nao, 6, seed=23)
    Jr, Kr = O.jk_definition(O.eri_tensor(b), D)
    # resident panels
    ctx = ltjk.Context(0)
    ctx.set_resident(True)
    ctx.set_basis(b)
    ctx.build_shell_pairs(0.0)
    J1, K1 = gpu_jk(torch, ctx, D[:2])
    n_first = ctx.get_stats()["n_launches"]
    J2, K2 = gpu_jk(torch, ctx, D)
    assert ctx.get_stats()["n_launches"] < n_first              # no ERI launches in the second build
    assert relerr(J1, Jr[:2]) < TOL and relerr(K1, Kr[:2]) < TOL
    assert relerr(J2, Jr) < TOL and relerr(K2, Kr) < TOL
    ctx.close()
    # quartet sharding + poisoned ring
    ctx = make_ctx(b, tau=0.0, scratch=1 << 20)
    ctx.debug_poison(True)
    Jsum, Ksum = np.zeros_like(D), np.zeros_like(D)
    for r in range(3):
        ctx.set_quartet_shard(r, 3)
        Jp, Kp = gpu_jk(torch, ctx, D)
        assert np.isfinite(Jp).all() and np.isfinite(Kp).all() and np.abs(Kp).max() > 0
        Jsum += Jp
        Ksum += Kp
    assert relerr(Jsum, Jr) < TOL and relerr(Ksum, Kr) < TOL

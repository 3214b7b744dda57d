"""The no-allocation entry point ltjk_build_pseudo_densities_noalloc (include/ltjk.h): its scratch is a static device
array instead of pool allocations.  Output must equal the existing path's (same kernels, same order of operations: the
tolerance is the 1e-12 the transform tests use) on two calls in a row that share the array, and sizes beyond the fixed
maximum must be rejected.  This file is collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def relerr(x, ref):
    return float(np.abs(x - ref).max() / np.abs(ref).max())


def test_noalloc_pseudo_densities_match_existing_path_twice(small):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")
    from paper_2607_05622_b200 import ltjk
    w = small
    N = w.nao
    ctx = ltjk.Context(0)
    ctx.set_basis(w.basis)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Co, Cv, eo, ev = dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir)
    rng = np.random.default_rng(77)
    # call 1: the workload's amplitudes (8 points x 4 sets); call 2: other amplitudes, fewer sets, other points, so
    # that what call 1 left in the shared array would show up if call 2 read anything it had not written itself
    cases = [(w.T, np.geomspace(0.05, 6.0, w.ntau)),
             (1e-2 * rng.standard_normal((3, w.nocc, w.nvir)), np.linspace(0.3, 2.0, 5))]
    for T, tau in cases:
        Td = dev(T)
        ref = torch.empty((len(tau), T.shape[0], N, N), dtype=torch.float64, device="cuda")
        out = torch.full_like(ref, float("nan"))
        ctx.build_pseudo_densities(Co, Cv, eo, ev, Td, tau, ref)
        ctx.build_pseudo_densities_noalloc(Co, Cv, eo, ev, Td, tau, out)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(out).all())
        assert relerr(out.cpu().numpy(), ref.cpu().numpy()) < 1e-12
    # beyond the fixed scratch (8 x 41 x 20 x 160 doubles > 2^20) and beyond 32 Laplace points: clear errors
    big = torch.zeros((41, w.nocc, w.nvir), dtype=torch.float64, device="cuda")
    Dbig = torch.empty((w.ntau, 41, N, N), dtype=torch.float64, device="cuda")
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.build_pseudo_densities_noalloc(Co, Cv, eo, ev, big, np.geomspace(0.05, 6.0, w.ntau), Dbig)
    assert e.value.code == -1 and "scratch" in str(e.value)
    with pytest.raises(ltjk.LtjkError) as e:
        ctx.build_pseudo_densities_noalloc(Co, Cv, eo, ev, dev(w.T[:1]), np.linspace(0.1, 3.0, 33),
                                           torch.empty((33, 1, N, N), dtype=torch.float64, device="cuda"))
    assert e.value.code == -1 and "Laplace points" in str(e.value)
    ctx.close()

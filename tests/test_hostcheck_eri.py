"""Host logic tier: the generated Obara-Saika/HGP recurrences and the table-driven Boys evaluator of the CUDA path,
compiled for the host by a TEST-ONLY shim (tests/host_check.cpp, built into a temporary directory), against the CPU oracle (McMurchie-Davidson).
Two different textbook recurrences agreeing to round-off is the main evidence that the integrals are right
(SURVEY.md 8(c) P-E); the same comparison runs on the GPU in test_gpu_parity.py."""
import ctypes
import itertools
import subprocess
from pathlib import Path

import numpy as np
import pytest

from oracle import oracle as O
from paper_2607_05622_b200.inputs import custom_basis, prim_norm

CSRC = Path(__file__).resolve().parent.parent / "paper_2607_05622_b200" / "csrc"
_dp = ctypes.POINTER(ctypes.c_double)


@pytest.fixture(scope="module")
def hc(tmp_path_factory):
    from paper_2607_05622_b200 import build
    build.build()                                   # generates csrc/gen/eri_gen.h when missing or stale
    so = tmp_path_factory.mktemp("hostcheck") / "libltjk_hostcheck.so"
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-I", str(CSRC), "-o", str(so),
                           str(Path(__file__).resolve().parent / "host_check.cpp")])
    return ctypes.CDLL(str(so))


def _d(a):
    return a.ctypes.data_as(_dp)


NC = (1, 3, 6)


def _shell_args(b, s):
    o, n = int(b.prim_off[s]), int(b.nprim[s])
    c = np.ascontiguousarray(b.xyz[b.atom[s]])
    e = np.ascontiguousarray(b.exps[o:o + n])
    k = np.ascontiguousarray(b.coef[o:o + n])
    return (c, e, k), (_d(c), ctypes.c_int(int(b.l[s])), ctypes.c_int(n), _d(e), _d(k))


@pytest.mark.parametrize("T", [0.0, 1e-9, 1e-3, 0.06, 0.0625, 0.5, 5.0, 20.0, 34.9, 35.93, 35.99999, 36.0, 36.1, 100.0,
                               1e3, 6e3])
def test_device_boys_formula_vs_oracle(hc, T):
    F = np.zeros(9)
    for mmax in (0, 3, 8):
        hc.hc_boys(ctypes.c_int(mmax), ctypes.c_double(T), _d(F))
        ref = O.boys(mmax, T)
        assert np.all(np.abs(F[:mmax + 1] - ref) <= 2e-14 * np.abs(ref)), (T, mmax, F[:mmax + 1], ref)


def test_generated_os_hgp_vs_md_all_classes(hc):
    rng = np.random.default_rng(7)
    xyz = rng.uniform(-1.5, 1.5, size=(4, 3))
    xyz[3] = xyz[0]                      # one coincident pair of centres
    # per atom: s, p, d shells, 2 primitives each, different exponents per atom
    shells = []
    for ia in range(4):
        sh = []
        for l in range(3):
            ex = [0.3 + 0.4 * ia + 0.2 * l, 1.1 + 0.3 * ia + 0.5 * l]
            sh.append((l, ex, [0.6, 0.4]))
        shells.append(sh)
    b = custom_basis(xyz, shells)
    worst = 0.0
    for la, lb, lc, ld in itertools.product(range(3), repeat=4):
        if la < lb or lc < ld:
            continue
        A, B, C, D = 0 * 3 + la, 1 * 3 + lb, 2 * 3 + lc, 3 * 3 + ld
        keep, args = [], []
        for s in (A, B, C, D):
            k, a = _shell_args(b, s)
            keep.append(k)
            args += list(a)
        out = np.zeros(NC[la] * NC[lb] * NC[lc] * NC[ld])
        rc = hc.hc_eri_quartet(*args, _d(out))
        assert rc == 0
        ref = O.eri_shell(b, A, B, C, D).ravel()
        err = np.abs(out - ref).max() / max(np.abs(ref).max(), 1e-300)
        worst = max(worst, err)
        assert err < 1e-12, ((la, lb, lc, ld), err)
    assert worst < 1e-12


def test_generated_diagonal_and_same_centre_quartets(hc):
    # (ab|ab) Schwarz-type quartets and all four shells on one centre (T = 0 path of the Boys evaluator)
    b = custom_basis(np.array([[0.1, -0.2, 0.3], [1.2, 0.4, -0.5]]),
                     [[(0, [0.8, 0.3], [0.6, 0.4]), (1, [0.7], [1.0]), (2, [0.9, 0.35], [0.6, 0.4])],
                      [(2, [0.5], [1.0])]])
    for (A, B, C, D) in [(2, 1, 2, 1), (2, 2, 2, 2), (3, 2, 3, 2), (2, 0, 1, 0), (3, 3, 2, 2)]:
        keep, args = [], []
        for s in (A, B, C, D):
            k, a = _shell_args(b, s)
            keep.append(k)
            args += list(a)
        n = [NC[int(b.l[s])] for s in (A, B, C, D)]
        out = np.zeros(int(np.prod(n)))
        assert hc.hc_eri_quartet(*args, _d(out)) == 0
        ref = O.eri_shell(b, A, B, C, D).ravel()
        # (the quartet (2,0,1,0) vanishes by parity: absolute floor)
        assert np.abs(out - ref).max() < 1e-12 * max(np.abs(ref).max(), 1e-2)

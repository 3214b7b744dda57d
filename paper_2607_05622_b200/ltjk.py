"""Thin ctypes binding of the C ABI in include/ltjk.h.  Argument marshalling only: every step of the path runs in
the CUDA kernels of libltjk.so.  There is NO CPU fallback: if the library is missing or no CUDA device is present the
calls raise.  torch is used by callers for device memory and streams only (tensors are passed as data_ptr()).
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIBPATH = _PKG / "libltjk.so"
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_llp = ctypes.POINTER(ctypes.c_longlong)

ERRORS = {0: "LTJK_OK", -1: "LTJK_EINVAL", -2: "LTJK_ENOBASIS", -3: "LTJK_ECUDA", -4: "LTJK_ELMAX",
          -5: "LTJK_ENOCONV", -6: "LTJK_ENOMEM"}

EXPORTS = [
    "ltjk_create", "ltjk_destroy", "ltjk_last_error", "ltjk_set_scratch_bytes", "ltjk_set_basis", "ltjk_get_nao",
    "ltjk_build_shell_pairs", "ltjk_get_schwarz", "ltjk_laplace_quadrature", "ltjk_build_pseudo_densities", "ltjk_build_pseudo_densities_noalloc",
    "ltjk_jk_build", "ltjk_jk_build_host", "ltjk_sweep_host", "ltjk_laplace_fock", "ltjk_laplace_accumulate", "ltjk_pp_ladder", "ltjk_jk_grad", "ltjk_get_nsph", "ltjk_sph_from_cart", "ltjk_cart_from_sph", "ltjk_get_stats", "ltjk_set_timing", "ltjk_set_digest_mode", "ltjk_get_digest_mode", "ltjk_set_resident", "ltjk_set_quartet_shard", "ltjk_debug_poison", "ltjk_debug_eri_quartet", "ltjk_debug_eri_quartet_looped",
    "ltjk_debug_boys", "ltjk_bench_dfma_peak", "ltjk_bench_copy_peak",
]


class LtjkError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("%s (%d): %s" % (ERRORS.get(code, "?"), code, msg))
        self.code = code


def load_library():
    """Load libltjk.so (built in-tree by paper_2607_05622_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not _LIBPATH.exists():
            raise FileNotFoundError("%s not found: run `python -m paper_2607_05622_b200.build` (there is no fallback)"
                                    % _LIBPATH)
        lib = ctypes.CDLL(str(_LIBPATH))
        lib.ltjk_last_error.restype = ctypes.c_char_p
        lib.ltjk_last_error.argtypes = [ctypes.c_void_p]
        for name in EXPORTS:
            if name != "ltjk_last_error":
                getattr(lib, name).restype = ctypes.c_int
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _devptr(t):
    """torch CUDA tensor (float64, contiguous) -> void*"""
    if t is None:
        return ctypes.c_void_p(0)
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), \
        "expected a contiguous float64 CUDA tensor"
    return ctypes.c_void_p(t.data_ptr())


def laplace_quadrature(xmin: float, xmax: float, npts: int):
    """ltjk_laplace_quadrature: minimax nodes/weights for 1/x on [xmin,xmax] (host).  Returns tau, w, maxerr."""
    lib = load_library()
    t = np.zeros(npts)
    w = np.zeros(npts)
    err = ctypes.c_double(0.0)
    rc = lib.ltjk_laplace_quadrature(ctypes.c_double(xmin), ctypes.c_double(xmax), ctypes.c_int(npts), _d(t), _d(w),
                                     ctypes.byref(err))
    if rc:
        raise LtjkError(rc, "laplace_quadrature")
    return t, w, err.value


class Context:
    """One ltjk_ctx.  Methods carry the names of the C entry points without the prefix."""

    def __init__(self, device: int = 0, stream=None):
        self.lib = load_library()
        self._h = ctypes.c_void_p(0)
        sp = ctypes.c_void_p(0)
        if stream is not None:
            sp = ctypes.c_void_p(int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream))
        rc = self.lib.ltjk_create(ctypes.byref(self._h), ctypes.c_int(device), sp)
        if rc:
            self._h = ctypes.c_void_p(0)
            raise LtjkError(rc, "ltjk_create failed (no CUDA device? there is no CPU fallback)")
        self.nao = 0
        self.nshell = 0

    def _chk(self, rc):
        if rc:
            raise LtjkError(rc, self.lib.ltjk_last_error(self._h).decode())

    def close(self):
        if self._h:
            self.lib.ltjk_destroy(self._h)
            self._h = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_scratch_bytes(self, nbytes: int):
        self._chk(self.lib.ltjk_set_scratch_bytes(self._h, ctypes.c_longlong(int(nbytes))))

    def set_basis(self, basis):
        """basis: object with xyz[natom,3], atom, l, nprim, prim_off, exps, coef (inputs.Basis)."""
        xyz = np.ascontiguousarray(basis.xyz, dtype=np.float64)
        atom = np.ascontiguousarray(basis.atom, dtype=np.int32)
        l = np.ascontiguousarray(basis.l, dtype=np.int32)
        nprim = np.ascontiguousarray(basis.nprim, dtype=np.int32)
        poff = np.ascontiguousarray(basis.prim_off, dtype=np.int32)
        exps = np.ascontiguousarray(basis.exps, dtype=np.float64)
        coef = np.ascontiguousarray(basis.coef, dtype=np.float64)
        self._chk(self.lib.ltjk_set_basis(self._h, ctypes.c_int(xyz.shape[0]), _d(xyz), ctypes.c_int(l.shape[0]),
                                          _i(atom), _i(l), _i(nprim), _i(poff), _d(exps), _d(coef)))
        n = ctypes.c_int(0)
        self._chk(self.lib.ltjk_get_nao(self._h, ctypes.byref(n)))
        self.nao = n.value
        self.nshell = int(l.shape[0])
        self.natom = int(xyz.shape[0])

    def get_nao(self) -> int:
        n = ctypes.c_int(0)
        self._chk(self.lib.ltjk_get_nao(self._h, ctypes.byref(n)))
        return n.value

    def build_shell_pairs(self, schwarz_tau: float):
        npairs = ctypes.c_longlong(0)
        nq = ctypes.c_longlong(0)
        self._chk(self.lib.ltjk_build_shell_pairs(self._h, ctypes.c_double(schwarz_tau), ctypes.byref(npairs),
                                                  ctypes.byref(nq)))
        return npairs.value, nq.value

    def get_schwarz(self) -> np.ndarray:
        Q = np.zeros((self.nshell, self.nshell))
        self._chk(self.lib.ltjk_get_schwarz(self._h, _d(Q)))
        return Q

    def build_pseudo_densities(self, C_occ, C_vir, eps_occ, eps_vir, T, tau, D_out):
        """Device tensors C_occ[N,nocc], C_vir[N,nvir], eps_occ, eps_vir, T[nT,nocc,nvir], D_out[ntau,nT,N,N];
        tau: host array."""
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        nocc, nvir = C_occ.shape[1], C_vir.shape[1]
        self._chk(self.lib.ltjk_build_pseudo_densities(
            self._h, ctypes.c_int(nocc), ctypes.c_int(nvir), _devptr(C_occ), _devptr(C_vir), _devptr(eps_occ),
            _devptr(eps_vir), ctypes.c_int(T.shape[0]), _devptr(T), ctypes.c_int(tau.shape[0]), _d(tau),
            _devptr(D_out)))

    def build_pseudo_densities_noalloc(self, C_occ, C_vir, eps_occ, eps_vir, T, tau, D_out):
        """ltjk_build_pseudo_densities_noalloc: same arguments and result as build_pseudo_densities; no device
        allocation (scratch = an 8 MiB static device array shared by all calls; see include/ltjk.h for the limits)."""
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        nocc, nvir = C_occ.shape[1], C_vir.shape[1]
        self._chk(self.lib.ltjk_build_pseudo_densities_noalloc(
            self._h, ctypes.c_int(nocc), ctypes.c_int(nvir), _devptr(C_occ), _devptr(C_vir), _devptr(eps_occ),
            _devptr(eps_vir), ctypes.c_int(T.shape[0]), _devptr(T), ctypes.c_int(tau.shape[0]), _d(tau),
            _devptr(D_out)))

    def jk_build(self, D, J=None, K=None):
        """Device tensors [nD,N,N]; J and/or K are overwritten.  Enqueued on the context stream, not synchronised."""
        self._chk(self.lib.ltjk_jk_build(self._h, ctypes.c_int(D.shape[0]), _devptr(D), _devptr(J), _devptr(K)))

    def jk_build_host(self, D: np.ndarray, want_j: bool = True, want_k: bool = True, J=None, K=None):
        """Host (numpy or pinned torch CPU) buffers in, host buffers out; synchronises."""
        def hp(a):
            if a is None:
                return ctypes.c_void_p(0)
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float64 and a.flags.c_contiguous
                return ctypes.c_void_p(a.ctypes.data)
            return ctypes.c_void_p(a.data_ptr())
        if J is None and want_j:
            J = np.empty(tuple(D.shape))
        if K is None and want_k:
            K = np.empty(tuple(D.shape))
        self._chk(self.lib.ltjk_jk_build_host(self._h, ctypes.c_int(D.shape[0]), hp(D), hp(J), hp(K)))
        return J, K

    def sweep_host(self, C_occ, C_vir, eps_occ, eps_vir, T, tau, J=None, K=None):
        """ltjk_sweep_host: host buffers (numpy float64 C-contiguous, or pinned torch CPU tensors) in and out."""
        def hp(a):
            if a is None:
                return ctypes.c_void_p(0)
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float64 and a.flags.c_contiguous
                return ctypes.c_void_p(a.ctypes.data)
            assert a.dtype.is_floating_point and a.is_contiguous() and not a.is_cuda
            return ctypes.c_void_p(a.data_ptr())
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        self._chk(self.lib.ltjk_sweep_host(
            self._h, ctypes.c_int(C_occ.shape[1]), ctypes.c_int(C_vir.shape[1]), hp(C_occ), hp(C_vir), hp(eps_occ),
            hp(eps_vir), ctypes.c_int(T.shape[0]), hp(T), ctypes.c_int(tau.shape[0]), _d(tau), hp(J), hp(K)))

    def laplace_fock(self, J, K, C, F):
        """ltjk_laplace_fock: F[d] = C^T (2 J[d] - K[d]) C; device tensors J, K [nD,N,N], C [N,nmo], F [nD,nmo,nmo]."""
        self._chk(self.lib.ltjk_laplace_fock(self._h, ctypes.c_int(J.shape[0]), _devptr(J), _devptr(K),
                                             ctypes.c_int(C.shape[1]), _devptr(C), _devptr(F)))

    def laplace_accumulate(self, tau, w, omega, X, Y):
        """ltjk_laplace_accumulate: Y[t] = sum_a w_a exp(omega tau_a) X[a][t]; X [ntau,nT,...], Y [nT,...] device."""
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        w = np.ascontiguousarray(w, dtype=np.float64)
        nelem = 1
        for n in Y.shape[1:]:
            nelem *= int(n)
        self._chk(self.lib.ltjk_laplace_accumulate(self._h, ctypes.c_int(X.shape[0]), ctypes.c_int(X.shape[1]),
                                                   ctypes.c_longlong(nelem), _d(tau), _d(w), ctypes.c_double(omega),
                                                   _devptr(X), _devptr(Y)))

    def pp_ladder(self, C_vir, X, L, chunk=0):
        """ltjk_pp_ladder: L[p] = C_vir^T K[C_vir X[p] C_vir^T] C_vir = sum_ef (ae|bf) X[p,e,f]; device tensors."""
        self._chk(self.lib.ltjk_pp_ladder(self._h, ctypes.c_int(C_vir.shape[1]), _devptr(C_vir),
                                          ctypes.c_int(X.shape[0]), _devptr(X), _devptr(L), ctypes.c_int(int(chunk))))

    def get_nsph(self) -> int:
        n = ctypes.c_int(0)
        self._chk(self.lib.ltjk_get_nsph(self._h, ctypes.byref(n)))
        return n.value

    def sph_from_cart(self, X_cart, X_sph):
        """ltjk_sph_from_cart: operators [nmat,N,N] -> [nmat,N_sph,N_sph] (device tensors), S X S^T."""
        self._chk(self.lib.ltjk_sph_from_cart(self._h, ctypes.c_int(X_cart.shape[0]), _devptr(X_cart), _devptr(X_sph)))

    def cart_from_sph(self, D_sph, D_cart):
        """ltjk_cart_from_sph: densities [nmat,N_sph,N_sph] -> [nmat,N,N] (device tensors), S^T D S."""
        self._chk(self.lib.ltjk_cart_from_sph(self._h, ctypes.c_int(D_sph.shape[0]), _devptr(D_sph), _devptr(D_cart)))

    def jk_grad(self, A, B, gradJ, gradK):
        """ltjk_jk_grad: J^x(A,B), K^x(A,B) (Eq. 18) for device tensors A, B [nP,N,N] -> gradJ, gradK [nP,natom,3]."""
        self._chk(self.lib.ltjk_jk_grad(self._h, ctypes.c_int(A.shape[0]), _devptr(A), _devptr(B), _devptr(gradJ),
                                        _devptr(gradK)))

    def get_stats(self) -> dict:
        nl = ctypes.c_longlong(0)
        nq = ctypes.c_longlong(0)
        fl = ctypes.c_double(0)
        e = ctypes.c_double(0)
        g = ctypes.c_double(0)
        self._chk(self.lib.ltjk_get_stats(self._h, ctypes.byref(nl), ctypes.byref(nq), ctypes.byref(fl),
                                          ctypes.byref(e), ctypes.byref(g)))
        return {"n_launches": nl.value, "eri_quartets": nq.value, "digest_flops": fl.value, "eri_ms": e.value,
                "digest_ms": g.value}

    def set_digest_mode(self, mode: int):
        self._chk(self.lib.ltjk_set_digest_mode(self._h, ctypes.c_int(int(mode))))

    def set_quartet_shard(self, rank: int, world: int):
        """ltjk_set_quartet_shard: the next builds compute this rank's partial J, K (sum over ranks = whole build)."""
        self._chk(self.lib.ltjk_set_quartet_shard(self._h, ctypes.c_int(int(rank)), ctypes.c_int(int(world))))

    def debug_poison(self, enable: bool):
        self._chk(self.lib.ltjk_debug_poison(self._h, ctypes.c_int(1 if enable else 0)))

    def set_resident(self, enable: bool):
        self._chk(self.lib.ltjk_set_resident(self._h, ctypes.c_int(1 if enable else 0)))

    def get_digest_mode(self) -> int:
        m = ctypes.c_int(0)
        self._chk(self.lib.ltjk_get_digest_mode(self._h, ctypes.byref(m)))
        return m.value

    def set_timing(self, enable: bool):
        self._chk(self.lib.ltjk_set_timing(self._h, ctypes.c_int(1 if enable else 0)))

    def debug_eri_quartet(self, basis, A, B, C, D, looped: bool = False) -> np.ndarray:
        nc = (1, 3, 6, 10)
        shp = tuple(nc[int(basis.l[s])] for s in (A, B, C, D))
        out = np.zeros(shp)
        fn = self.lib.ltjk_debug_eri_quartet_looped if looped else self.lib.ltjk_debug_eri_quartet
        self._chk(fn(self._h, ctypes.c_int(A), ctypes.c_int(B), ctypes.c_int(C), ctypes.c_int(D), _d(out)))
        return out

    def debug_boys(self, mmax: int, T) -> np.ndarray:
        T = np.ascontiguousarray(T, dtype=np.float64)
        F = np.zeros((T.shape[0], mmax + 1))
        self._chk(self.lib.ltjk_debug_boys(self._h, ctypes.c_int(mmax), ctypes.c_int(T.shape[0]), _d(T), _d(F)))
        return F

    def bench_dfma_peak(self) -> float:
        v = ctypes.c_double(0)
        self._chk(self.lib.ltjk_bench_dfma_peak(self._h, ctypes.byref(v)))
        return v.value

    def bench_copy_peak(self) -> float:
        v = ctypes.c_double(0)
        self._chk(self.lib.ltjk_bench_copy_peak(self._h, ctypes.byref(v)))
        return v.value

"""Seeded synthetic inputs for the five BASELINE.json configs (SURVEY.md §8(d) recipe).

This module is shared by the CPU oracle (tests, cpu_baseline) and the CUDA path.  It holds NONE of the
method's arithmetic (no integrals, no quadrature, no density transform): only geometry, the shell table,
random MO-like coefficients, orbital energies and amplitude matrices.  The one formula here is the primitive
normalisation N(a,l) which the C ABI declares to be the *caller's* job (include/ltjk.h, reading A6).

The paper's molecules / basis sets (SI S2) are not available; these
synthetic molecules stand in for them with the same AO counts (36/160/300/439/730), atom counts and
l_max = 2.

Draw order per config (numpy PCG64, seed = 20260705 + config index):
geometry -> atom-type shuffle -> C -> eps_occ -> eps_vir -> T_1..T_nT.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

CONFIG_NAMES = ("tiny", "small", "medium", "porphine", "large")
SEED0 = 20260705
LAPLACE_RANGE = (0.4, 4.5)  # denominators x = eps_a - eps_i lie in [0.4, 4.5] E_h
SCHWARZ_TAU = 1e-12

NCART = (1, 3, 6, 10)


def _dfact2lm1(l: int) -> float:
    """(2l-1)!!"""
    r = 1.0
    for k in range(1, 2 * l, 2):
        r *= k
    return r


def prim_norm(a: float, l: int) -> float:
    """N(a,l) = (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2l-1)!!): unit norm for x^l exp(-a r^2) (reading A6)."""
    return (2.0 * a / math.pi) ** 0.75 * (4.0 * a) ** (0.5 * l) / math.sqrt(_dfact2lm1(l))


# shell sets: list of (l, [exponents], [raw contraction coefficients])
def _even_tempered_contracted(ns: int, npp: int, nd: int):
    shells = []
    for l, n in ((0, ns), (1, npp), (2, nd)):
        for k in range(n):
            shells.append((l, [0.15 * 2.8 ** k, 0.15 * 2.8 ** (k + 1)], [0.6, 0.4]))
    return shells


def _tiny_set():
    shells = []
    for k in range(3):
        shells.append((0, [0.2 * 3.0 ** k], [1.0]))
    for k in range(2):
        shells.append((1, [0.3 * 3.0 ** k], [1.0]))
    return shells


ATOM_TYPES = {
    "T": _tiny_set(),                        # 3s2p uncontracted, 9 AO
    "H": _even_tempered_contracted(4, 3, 1),  # 19 AO
    "H2": _even_tempered_contracted(4, 3, 2),  # 25 AO
    "M": _even_tempered_contracted(3, 2, 1),  # 15 AO
    "L": _even_tempered_contracted(2, 1, 0),  # 5 AO
    # the heavy-atom set plus one uncontracted f polarisation shell (triple-zeta-class bases): 29 AO
    "HF": _even_tempered_contracted(4, 3, 1) + [(3, [0.9], [1.0])],
}


@dataclass
class Basis:
    """Flat shell table in the layout the C ABI takes (include/ltjk.h: ltjk_set_basis)."""
    xyz: np.ndarray        # [natom,3] bohr
    atom: np.ndarray       # [nshell] int32
    l: np.ndarray          # [nshell] int32
    nprim: np.ndarray      # [nshell] int32
    prim_off: np.ndarray   # [nshell] int32
    exps: np.ndarray       # [nprim_total]
    coef: np.ndarray       # [nprim_total], normalisation folded in
    ao_off: np.ndarray = field(default=None)  # [nshell+1]

    @property
    def natom(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def nshell(self) -> int:
        return int(self.l.shape[0])

    @property
    def nao(self) -> int:
        return int(self.ao_off[-1])


def make_basis(xyz: np.ndarray, types: list[str]) -> Basis:
    atom, ls, nprim, prim_off, exps, coef = [], [], [], [], [], []
    for ia, t in enumerate(types):
        for (l, ex, cc) in ATOM_TYPES[t]:
            atom.append(ia)
            ls.append(l)
            nprim.append(len(ex))
            prim_off.append(len(exps))
            for a, c in zip(ex, cc):
                exps.append(a)
                coef.append(c * prim_norm(a, l))
    ls_a = np.asarray(ls, dtype=np.int32)
    ao_off = np.zeros(len(ls) + 1, dtype=np.int64)
    ao_off[1:] = np.cumsum([NCART[l] for l in ls])
    return Basis(np.ascontiguousarray(xyz, dtype=np.float64), np.asarray(atom, dtype=np.int32), ls_a,
                 np.asarray(nprim, dtype=np.int32), np.asarray(prim_off, dtype=np.int32),
                 np.asarray(exps, dtype=np.float64), np.asarray(coef, dtype=np.float64), ao_off)


def _random_points(rng, n, box, dmin):
    pts = []
    while len(pts) < n:
        p = rng.uniform(0.0, box, size=3)
        if all(np.linalg.norm(p - q) >= dmin for q in pts):
            pts.append(p)
    return np.array(pts)


def _honeycomb_sites(bond: float, nmax_cells: int = 12):
    """All honeycomb-lattice sites in a patch; origin at a hexagon centre. Returns xy[n,2]."""
    a1 = np.array([1.5 * bond, math.sqrt(3) / 2 * bond])
    a2 = np.array([1.5 * bond, -math.sqrt(3) / 2 * bond])
    # two-site basis chosen so that (0,0) is a hexagon centre: its six vertices are lattice sites
    basis = [np.array([bond, 0.0]), np.array([2 * bond, 0.0])]
    sites = []
    for i in range(-nmax_cells, nmax_cells + 1):
        for j in range(-nmax_cells, nmax_cells + 1):
            for b in basis:
                sites.append(i * a1 + j * a2 + b)
    return np.array(sites)


def _geometry(name: str, rng) -> np.ndarray:
    if name == "tiny":
        return _random_points(rng, 4, 8.0, 1.5)
    if name == "small":
        return _random_points(rng, 14, 12.0, 1.5)
    if name == "medium":
        s = _honeycomb_sites(2.6)
        r = np.linalg.norm(s, axis=1)
        idx = np.lexsort((s[:, 1], s[:, 0], np.round(r, 9)))[:30]  # deterministic tie-break
        xy = s[idx]
        z = rng.uniform(-0.3, 0.3, size=30)
        return np.column_stack([xy, z])
    if name == "porphine":
        pts = []
        for k in range(24):
            th = math.radians(15.0 * k)
            pts.append([6.5 * math.cos(th), 6.5 * math.sin(th)])
        for k in range(4):
            th = math.radians(90.0 * k)
            pts.append([3.8 * math.cos(th), 3.8 * math.sin(th)])
        pts.append([0.0, 0.0])
        for k in range(8):
            th = math.radians(22.5 + 45.0 * k)
            pts.append([9.5 * math.cos(th), 9.5 * math.sin(th)])
        xy = np.array(pts)
        z = rng.uniform(-0.1, 0.1, size=37)
        return np.column_stack([xy, z])
    if name == "large":
        s = _honeycomb_sites(2.6, 16)
        # Eden growth on the lattice graph from the site nearest the origin
        r = np.linalg.norm(s, axis=1)
        start = int(np.lexsort((s[:, 1], s[:, 0], np.round(r, 9)))[0])
        # neighbour table by distance (bond length), built once
        nb = [[] for _ in range(len(s))]
        order = np.argsort(s[:, 0], kind="stable")
        sx = s[order, 0]
        for i in order:
            lo = np.searchsorted(sx, s[i, 0] - 2.61)
            hi = np.searchsorted(sx, s[i, 0] + 2.61)
            for j in order[lo:hi]:
                if j != i and abs(np.linalg.norm(s[i] - s[j]) - 2.6) < 1e-6:
                    nb[i].append(int(j))
        cluster = [start]
        inc = {start}
        while len(cluster) < 56:
            frontier = sorted({j for i in cluster for j in nb[i] if j not in inc})
            pick = frontier[int(rng.integers(len(frontier)))]
            cluster.append(pick)
            inc.add(pick)
        xy = s[cluster]
        z = rng.uniform(-0.2, 0.2, size=56)
        return np.column_stack([xy, z])
    raise ValueError(name)


def _atom_types(name: str, rng) -> list[str]:
    if name == "tiny":
        return ["T"] * 4
    if name == "small":
        t = ["H"] * 5 + ["M"] * 2 + ["L"] * 7
        return [t[i] for i in rng.permutation(len(t))]
    if name == "medium":
        t = ["H"] * 10 + ["M"] * 1 + ["L"] * 19
        return [t[i] for i in rng.permutation(len(t))]
    if name == "porphine":
        t = []
        for k in range(24):
            t.append("L" if k % 6 == 0 else "M")
        t += ["M"] * 4 + ["H"] + ["L"] * 8
        return t
    if name == "large":
        t = ["H2"] * 22 + ["M"] * 1 + ["L"] * 33
        return [t[i] for i in rng.permutation(len(t))]
    raise ValueError(name)


_PARAMS = {  # name: (n_occ, n_tau, n_T)
    "tiny": (5, 8, 1),
    "small": (20, 8, 4),
    "medium": (45, 10, 8),
    "porphine": (81, 10, 16),
    "large": (120, 12, 16),
}
_EXPECTED_NAO = {"tiny": 36, "small": 160, "medium": 300, "porphine": 439, "large": 730}


@dataclass
class Workload:
    name: str
    basis: Basis
    nocc: int
    nvir: int
    ntau: int
    nT: int
    C_occ: np.ndarray    # [N, nocc]
    C_vir: np.ndarray    # [N, nvir]
    eps_occ: np.ndarray  # [nocc]
    eps_vir: np.ndarray  # [nvir]
    T: np.ndarray        # [nT, nocc, nvir]
    schwarz_tau: float = SCHWARZ_TAU
    laplace_range: tuple = LAPLACE_RANGE

    @property
    def nao(self) -> int:
        return self.basis.nao

    @property
    def nD(self) -> int:
        return self.ntau * self.nT


def make_workload(name: str) -> Workload:
    """Build the seeded workload for one of CONFIG_NAMES, or "<name>_f": the same geometry, sizes and seeds with an
    f shell added to every heavy atom (type H -> HF; "medium_f" = 400 AO, 10 f shells)."""
    base = name[:-2] if name.endswith("_f") else name
    ci = CONFIG_NAMES.index(base)
    rng = np.random.default_rng(SEED0 + ci)
    xyz = _geometry(base, rng)
    types = _atom_types(base, rng)
    if name != base:
        types = ["HF" if t == "H" else t for t in types]
    basis = make_basis(xyz, types)
    n = basis.nao
    assert n == _EXPECTED_NAO[base] + 10 * types.count("HF"), (name, n)
    nocc, ntau, nT = _PARAMS[base]
    nvir = n - nocc
    C = rng.standard_normal((n, n)) / math.sqrt(n)
    eps_occ = np.sort(rng.uniform(-1.5, -0.3, size=nocc))
    eps_vir = np.sort(rng.uniform(0.1, 3.0, size=nvir))
    T = 1e-2 * rng.standard_normal((nT, nocc, nvir))
    return Workload(name, basis, nocc, nvir, ntau, nT,
                    np.ascontiguousarray(C[:, :nocc]), np.ascontiguousarray(C[:, nocc:]),
                    eps_occ, eps_vir, np.ascontiguousarray(T))


def random_densities(nao: int, nD: int, seed: int, scale: float = 1.0) -> np.ndarray:
    """General (non-symmetric) dense test densities [nD,N,N], i.i.d. normal; used by parity/invariant tests."""
    rng = np.random.default_rng(seed)
    return scale * rng.standard_normal((nD, nao, nao))


def custom_basis(xyz, shells_per_atom) -> Basis:
    """Test helper: shells_per_atom[i] = list of (l, exps, raw_coefs); normalisation N(a,l) is applied here."""
    atom, ls, nprim, prim_off, exps, coef = [], [], [], [], [], []
    for ia, shells in enumerate(shells_per_atom):
        for (l, ex, cc) in shells:
            atom.append(ia)
            ls.append(l)
            nprim.append(len(ex))
            prim_off.append(len(exps))
            for a, c in zip(ex, cc):
                exps.append(a)
                coef.append(c * prim_norm(a, l))
    ao_off = np.zeros(len(ls) + 1, dtype=np.int64)
    ao_off[1:] = np.cumsum([NCART[l] for l in ls])
    return Basis(np.ascontiguousarray(np.asarray(xyz, dtype=np.float64).reshape(-1, 3)),
                 np.asarray(atom, dtype=np.int32), np.asarray(ls, dtype=np.int32),
                 np.asarray(nprim, dtype=np.int32), np.asarray(prim_off, dtype=np.int32),
                 np.asarray(exps, dtype=np.float64), np.asarray(coef, dtype=np.float64), ao_off)

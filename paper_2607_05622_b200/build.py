"""Build libltjk.so in-tree: generate the OS/HGP recurrences, compile every CUDA translation unit for sm_100a
with nvcc (cross-compiles without a GPU) and link one C-ABI shared library.  No torch types anywhere.

    python -m paper_2607_05622_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
GEN = CSRC / "gen"
OBJ = CSRC / "build"
LIB = PKG / "libltjk.so"

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]
CU_SOURCES = ["ltjk_api.cu", "ltjk_build.cu", "ltjk_eri.cu", "ltjk_digest.cu", "ltjk_transform.cu", "ltjk_pair.cu",
              "ltjk_peri.cu", "ltjk_pdigest.cu", "ltjk_grad.cu", "ltjk_eri_loop.cu", "ltjk_sph.cu"]
CPP_SOURCES = ["ltjk_laplace.cpp"]
HEADERS = ["ltjk_internal.h", "digest_common.h", "eri_core.h", "boys_table.h", "../../include/ltjk.h", "gen_eri.py"]


def _mtime(p: Path) -> float:
    return p.stat().st_mtime if p.exists() else 0.0


def build(force: bool = False, verbose: bool = False) -> Path:
    GEN.mkdir(exist_ok=True)
    OBJ.mkdir(exist_ok=True)
    gen_h = GEN / "eri_gen.h"
    if force or _mtime(gen_h) < _mtime(CSRC / "gen_eri.py"):
        subprocess.check_call([sys.executable, str(CSRC / "gen_eri.py"), str(GEN)])
    hdr_time = max(_mtime(CSRC / h) for h in HEADERS)
    hdr_time = max(hdr_time, _mtime(gen_h))
    if not (GEN / "eri_gen_d1.h").exists():
        subprocess.check_call([sys.executable, str(CSRC / "gen_eri.py"), str(GEN)])
    jobs = []
    for src in CU_SOURCES:
        obj = OBJ / (src + ".o")
        if force or _mtime(obj) < max(_mtime(CSRC / src), hdr_time):
            jobs.append([NVCC, *NVCC_FLAGS, "-c", str(CSRC / src), "-o", str(obj)])
    for src in CPP_SOURCES:
        obj = OBJ / (src + ".o")
        if force or _mtime(obj) < max(_mtime(CSRC / src), hdr_time):
            jobs.append(["g++", "-O2", "-std=c++17", "-fPIC", "-fext-numeric-literals", "-c", str(CSRC / src), "-o", str(obj)])

    def run(cmd):
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.check_call(cmd)

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            list(ex.map(run, jobs))
    objs = [str(OBJ / (s + ".o")) for s in CU_SOURCES + CPP_SOURCES]
    if force or jobs or not LIB.exists():
        run([NVCC, "-shared", "-o", str(LIB), *objs, "-lquadmath"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))

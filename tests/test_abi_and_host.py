"""CPU tier: the C-ABI library loads and exports every symbol include/ltjk.h declares; without a GPU the product
path fails loudly (no CPU fallback); host-side helpers of bench.py; world_size-2 gloo run of the multi-rank logic."""
import ctypes
import os
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def libpath():
    from paper_2607_05622_b200 import build
    return build.build()


def test_library_exports_every_declared_symbol(libpath):
    hdr = (ROOT / "include" / "ltjk.h").read_text()
    declared = sorted(set(re.findall(r"\b(ltjk_[a-z_0-9]+)\s*\(", hdr)))
    assert len(declared) >= 18
    lib = ctypes.CDLL(str(libpath))
    for name in declared:
        assert hasattr(lib, name), name
    from paper_2607_05622_b200 import ltjk
    assert sorted(ltjk.EXPORTS) == declared          # the binding carries the same names, no more, no fewer


def test_no_cpu_fallback(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2607_05622_b200 import ltjk
    with pytest.raises(ltjk.LtjkError) as e:
        ltjk.Context(0)
    assert e.value.code == -3                         # LTJK_ECUDA


def test_product_does_not_import_oracle():
    for f in (ROOT / "paper_2607_05622_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cpp", ".h") and "gen" not in f.parts and "build" not in f.parts[-2:-1]:
            txt = f.read_text()
            assert "from oracle" not in txt and "import oracle" not in txt and "ltjk_oracle" not in txt, f


def test_kept_integrals_counter_vs_brute_force(small):
    sys.path.insert(0, str(ROOT))
    import bench
    from oracle import oracle as O
    b = small.basis
    Q = O.schwarz(b)
    tau = 1e-6                                        # a threshold that really cuts on this molecule
    nc = np.array([1, 3, 6])[b.l]
    pairs = [(A, B) for A in range(b.nshell) for B in range(A + 1)]
    q = np.array([Q[A, B] for A, B in pairs])
    nf = np.array([nc[A] * nc[B] for A, B in pairs], dtype=np.float64)
    brute = 0.0
    for p in range(len(pairs)):
        keep = q[:p + 1] * q[p] >= tau
        brute += nf[p] * nf[:p + 1][keep].sum()
    assert bench.kept_integrals(Q, b.l, tau) == pytest.approx(brute, rel=1e-12)
    assert brute < 0.9 * bench.kept_integrals(Q, b.l, 0.0)


_GLOO_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_2607_05622_b200.inputs import make_workload
from paper_2607_05622_b200.dist import rank_amplitudes, max_over_ranks, whole_job_builds_per_s
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = make_workload("tiny")
T = rank_amplitudes(w, rank)
assert T.shape == w.T.shape
ms = max_over_ranks(10.0 * (rank + 1))
assert ms == 10.0 * world, ms
# ranks work on different batches: gather a checksum of each rank's T
c = torch.tensor([float(np.abs(T).sum())], dtype=torch.float64)
out = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
dist.all_gather(out, c)
assert len({round(float(o), 12) for o in out}) == world
v = whole_job_builds_per_s(w.nD, world, ms)
assert abs(v - world * w.nD / (ms * 1e-3)) < 1e-9
# one sweep sharded over the ranks (SURVEY 8(e)): round-robin density shards are a partition, and gathering the
# per-rank results restores sweep order
from paper_2607_05622_b200.dist import density_shard, gather_sharded, shard_sizes, sharded_sweep_builds_per_s
for nD in (1, 7, 8, 160):
    mine = density_shard(nD, rank, world)
    assert len(mine) == shard_sizes(nD, world)[rank]
    cnt = torch.zeros(nD, dtype=torch.float64)
    cnt[torch.from_numpy(mine)] += 1
    dist.all_reduce(cnt)
    assert bool((cnt == 1).all())                      # every density owned exactly once
    fake = torch.from_numpy(mine.astype(np.float64))[:, None, None] * torch.ones((1, 3, 3), dtype=torch.float64)
    full = gather_sharded(fake, nD)
    assert full.shape == (nD, 3, 3) and bool((full[:, 0, 0] == torch.arange(nD, dtype=torch.float64)).all())
assert abs(sharded_sweep_builds_per_s(160, 500.0) - 320.0) < 1e-12
# quartet-space split (N5): partial J, K of the ranks are summed in place by one all-reduce
from paper_2607_05622_b200.dist import allreduce_jk
Jp = torch.full((2, 4, 4), float(rank + 1), dtype=torch.float64)
Kp = torch.arange(32, dtype=torch.float64).reshape(2, 4, 4) * (rank + 1)
allreduce_jk(Jp, Kp)
tot = world * (world + 1) / 2
assert bool((Jp == tot).all()) and bool((Kp == torch.arange(32, dtype=torch.float64).reshape(2, 4, 4) * tot).all())
if rank == 0:
    print("GLOO_OK", v)
dist.destroy_process_group()
'''


def test_multi_rank_logic_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29533", str(script), str(ROOT)],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "GLOO_OK" in r.stdout

#!/usr/bin/env python
"""bench.py -- non-symmetric Laplace-transform J/K builds/s (fp64) on the 439-AO "porphine-sized" workload.

One STEP = one whole Laplace sweep of the hot path over one batch of synthetic input:
build_pseudo_densities (n_tau x n_T = 160 densities) + jk_build (J and K for all of them).  value = builds/s with
inputs resident in HBM; `e2e` = the same sweep through the C ABI with HOST buffers (ltjk_sweep_host: H2D of C, eps, T
from pinned memory, D2H of J and K into pinned memory inside the timed region).  Basis upload, shell pairs, Schwarz
bounds and work lists are geometry-frozen setup and are outside the timed region.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload porphine] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "non-symmetric J/K builds/s (fp64) at 439 AO"
UNIT = "builds/s"


def kept_integrals(Q, l, tau):
    """Unique (8-fold folded) Cartesian integrals the folded loop digests: sum over canonical shell quartets
    (AB)>=(CD) with Q_AB Q_CD >= tau of na nb nc nd  (oracle O6 / SURVEY 8.0 `ints`)."""
    nc = np.array([1, 3, 6])[np.asarray(l)]
    ns = len(l)
    iu = np.tril_indices(ns)
    q = Q[iu]
    nf = (nc[iu[0]] * nc[iu[1]]).astype(np.float64)
    order = np.argsort(q)
    qs, nfs = q[order], nf[order]
    cum = np.concatenate([[0.0], np.cumsum(nfs)])
    with np.errstate(divide="ignore"):
        thr = np.where(qs > 0, tau / np.maximum(qs, 1e-300), np.inf)
    lo = np.searchsorted(qs, thr, side="left")
    ordered = float((nfs * (cum[-1] - cum[lo])).sum())
    diag = float((nfs[qs * qs >= tau] ** 2).sum())
    return 0.5 * (ordered + diag)


class ClockSampler:
    def __init__(self, dev):
        self.dev, self.rows, self.p = dev, [], None

    def start(self):
        try:
            self.p = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.dev),
                 "--query-gpu=clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
                 "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                 "clocks_event_reasons.sw_power_cap", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 7 for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def oracle_sample(w, D, target_s=15.0):
    """Time the oracle (as it stands) on a bounded sample of the workload: a prefix of bra shell pairs of the folded
    loop O6 with all nD densities, grown until ~target_s of CPU work; scaled by the kept-quartet share."""
    from oracle import oracle as O
    b = w.basis
    Q = O.schwarz(b)
    npair = b.nshell * (b.nshell + 1) // 2
    nc = np.array([1, 3, 6])[b.l]
    total_ints = kept_integrals(Q, b.l, w.schwarz_tau)
    # integrals of bra pairs [p0,p1): bra pair p against kets q<=p
    iu = np.tril_indices(b.nshell)
    qv = Q[iu]
    nf = (nc[iu[0]] * nc[iu[1]]).astype(np.float64)

    def ints_of(p0, p1):
        s = 0.0
        for p in range(p0, p1):
            keep = qv[:p + 1] * qv[p] >= w.schwarz_tau
            s += nf[p] * float(nf[:p + 1][keep].sum())
        return s

    # Every oracle call has a fixed cost (density-fastest copies of D, per-thread J/K buffers and their reduction) that a
    # whole sweep pays once: it is measured by a call with an empty pair range; the per-integral rate comes from one
    # call over a run of bra shell pairs from the middle of the pair list (typical cost), sized by a short calibration
    # call to use the rest of the time budget.  sweep time = fixed + rate * (kept unique integrals).
    def call(pa, pb):
        t = time.perf_counter()
        O.jk_folded(b, D, w.schwarz_tau, pair_range=(pa, pb), Q=Q)
        return time.perf_counter() - t

    t_fixed = call(0, 0)
    p0 = npair // 2
    t_cal = call(p0, min(p0 + 4, npair))
    i_cal = ints_of(p0, min(p0 + 4, npair))
    rate_cal = max(t_cal - t_fixed, 1e-3) / max(i_cal, 1.0)
    budget = max(target_s - t_fixed - t_cal - t_fixed, 2.0)          # the big call pays the fixed cost again
    n = 4
    while p0 + 4 + n < npair and ints_of(p0 + 4, p0 + 4 + n) * rate_cal < budget and n < 65536:
        n *= 2
    pa, pb = p0 + 4, min(p0 + 4 + n, npair)
    t_big = call(pa, pb)
    i_big = ints_of(pa, pb)
    rate = max(t_big - t_fixed, 1e-6) / max(i_big, 1.0)
    t_used = t_fixed + t_cal + t_big
    sweep_s = t_fixed + rate * total_ints
    return {"value": D.shape[0] / sweep_s, "unit": UNIT, "cores": O.max_threads(), "kind": "oracle",
            "sample": "oracle O6 (folded MD loop, all %d densities): %.1f s of CPU time; fixed cost per call %.2f s (empty "
                      "pair range), then %.3g of the %.3g kept unique integrals in %.2f s -> %.3g s per integral; sweep = "
                      "fixed + rate x all integrals" % (D.shape[0], t_used, t_fixed, i_big, total_ints, t_big, rate)}


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import oracle as O
    from paper_2607_05622_b200.inputs import make_workload
    w = make_workload(args.workload)
    tau = np.linspace(0.1, 3.0, w.ntau)     # any grid: cost does not depend on the values
    nD = w.nD
    rng = np.random.default_rng(1)
    D = 1e-2 * rng.standard_normal((nD, w.nao, w.nao))
    per = max(2.0, min(20.0, 120.0 / max(args.steps + args.warmup, 1)))
    vals = []
    for s in range(args.warmup + args.steps):
        r = oracle_sample(w, D, target_s=per)
        if s >= args.warmup:
            vals.append(r)
    v = float(np.mean([r["value"] for r in vals]))
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * w.nD / v, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "%s (%d AO, %d densities)" % (w.name, w.nao, nD), "tau_schwarz": w.schwarz_tau},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": vals[-1]["cores"], "kind": "oracle", "sample": vals[-1]["sample"]},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="porphine")
    ap.add_argument("--impl", default="ltjk")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2607_05622_b200 import build as _build
    if rank == 0 and not _build.LIB.exists():
        _build.build()          # in-tree build of libltjk.so (the driver normally did this through build())
    from paper_2607_05622_b200 import ltjk
    from paper_2607_05622_b200.inputs import make_workload

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    w = make_workload(args.workload)
    N, nD = w.nao, w.nD
    # Multi-GPU: the path shards over independent problems -- every rank runs its own
    # sweep on its own batch of n_T amplitude sets (same molecule, rank-seeded T); no data-path collective.
    from paper_2607_05622_b200.dist import max_over_ranks, rank_amplitudes, whole_job_builds_per_s
    T_host = rank_amplitudes(w, rank)

    stream = torch.cuda.current_stream()
    ctx = ltjk.Context(local, stream)
    ctx.set_basis(w.basis)
    npairs, nq_kept = ctx.build_shell_pairs(w.schwarz_tau)
    tau, wts, lap_err = None, None, None
    try:
        tau, wts, lap_err = ltjk.laplace_quadrature(w.laplace_range[0], w.laplace_range[1], w.ntau)
    except ltjk.LtjkError:
        tau = np.linspace(0.1, 3.0, w.ntau)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Co, Cv, eo, ev, Td = dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir), dev(T_host)
    D = torch.empty((w.ntau, w.nT, N, N), dtype=torch.float64, device="cuda")
    Dn = D.view(nD, N, N)
    J = torch.empty_like(Dn)
    K = torch.empty_like(Dn)

    def step():
        ctx.build_pseudo_densities(Co, Cv, eo, ev, Td, tau, D)
        ctx.jk_build(Dn, J, K)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches_jk = ctx.get_stats()["n_launches"]
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(ms, "cuda")
    ms_per_step = ms / args.steps
    value = whole_job_builds_per_s(nD, world, ms_per_step)

    # ---- e2e: the same sweep through the C ABI with HOST (pinned) buffers
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hCo, hCv, heo, hev, hT = pin(w.C_occ), pin(w.C_vir), pin(w.eps_occ), pin(w.eps_vir), pin(T_host)
    hJ = torch.empty((nD, N, N), dtype=torch.float64).pin_memory()
    hK = torch.empty((nD, N, N), dtype=torch.float64).pin_memory()
    ctx.sweep_host(hCo, hCv, heo, hev, hT, tau, hJ, hK)
    barrier()
    n_e2e = max(2, min(args.steps, 3))
    t0 = time.perf_counter()
    e0.record(stream)
    for _ in range(n_e2e):
        tc = time.perf_counter()
        ctx.sweep_host(hCo, hCv, heo, hev, hT, tau, hJ, hK)
        if rank == 0:
            print("e2e sweep_host call: %.1f ms" % ((time.perf_counter() - tc) * 1e3), file=sys.stderr)
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1) / n_e2e
    ms_e2e = max_over_ranks(ms_e2e, "cuda")
    h2d = 8 * (hCo.numel() + hCv.numel() + heo.numel() + hev.numel() + hT.numel())
    d2h = 8 * (hJ.numel() + hK.numel())
    assert torch.equal(hK, K.cpu()) or float((hK - K.cpu()).abs().max()) < 1e-9 * float(K.abs().max())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (digestion), timed live per launch with CUDA events on the ctx stream
    ctx.set_timing(True)
    ctx.jk_build(Dn, J, K)
    torch.cuda.synchronize()
    st = ctx.get_stats()
    ctx.set_timing(False)
    # one Laplace point per call (n_D = n_T): makes the integral re-computation per call visible
    D1 = Dn[:w.nT].contiguous()
    J1 = torch.empty_like(D1)
    K1 = torch.empty_like(D1)
    ctx.jk_build(D1, J1, K1)
    torch.cuda.synchronize()
    e0.record(stream)
    ctx.jk_build(D1, J1, K1)
    e1.record(stream)
    torch.cuda.synchronize()
    single_point = {"n_D": int(w.nT), "ms": e0.elapsed_time(e1), "builds_per_s": w.nT / (e0.elapsed_time(e1) * 1e-3)}
    Q = ctx.get_schwarz()
    ints = kept_integrals(Q, w.basis.l, w.schwarz_tau)
    digest_flops_alg = 20.0 * nD * ints                  # 2 J + 8 K FMAs per unique integral and density
    peak_tf = ctx.bench_dfma_peak()
    achieved_tf = digest_flops_alg / (st["digest_ms"] * 1e-3) / 1e12
    # DRAM traffic of the digestion launches of one sweep from the committed ncu capture (profiles/), 439 AO only
    traffic = None
    tfile = ROOT / "profiles" / "r1_digest_traffic.json"
    if w.name == "porphine" and tfile.exists():
        tj = json.loads(tfile.read_text())
        traffic = tj["dram_bytes_read_per_sweep"] + tj["dram_bytes_write_per_sweep"]
    roofline = {"bound": "alu", "kernel": "digest_kernel (J/K digestion; achieved = algorithmic flop of one sweep / summed duration of its launches)",
                "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
                "traffic": traffic,
                "peak_source": "DFMA microbenchmark in this run (ltjk_bench_dfma_peak); MEASURED_PEAKS.json has no fp64 entry",
                "algorithmic_flops_per_sweep": digest_flops_alg, "executed_digest_flops_per_sweep": st["digest_flops"],
                "digest_ms_per_sweep": st["digest_ms"], "eri_ms_per_sweep": st["eri_ms"],
                "whole_sweep_frac_of_peak": digest_flops_alg / (ms_per_step * 1e-3) / 1e12 / peak_tf}
    cpu = None
    if not args.no_cpu_baseline:
        cpu = oracle_sample(w, Dn.cpu().numpy(), target_s=15.0)
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": "%s (%d AO, %d atoms, n_tau=%d x n_T=%d = %d non-symmetric densities per sweep)" %
                                  (w.name, N, w.basis.natom, w.ntau, w.nT, nD),
                      "tau_schwarz": w.schwarz_tau, "shell_quartets_kept": nq_kept, "unique_integrals_kept": ints,
                      "l2": "inputs_larger_than_L2 (D, J, K are %.0f MB each)" % (8e-6 * nD * N * N),
                      "setup_outside_timed_region": "basis upload, shell pairs, Schwarz, work lists (geometry-frozen)",
                      "laplace_grid": "library minimax" if wts is not None else "placeholder linspace (cost is value-independent)",
                      "one_laplace_point_per_call": single_point,
                      "gpu": torch.cuda.get_device_name(local), "hbm_copy_gbs_measured": ctx.bench_copy_peak(),
                      "dfma_peak_tflops_measured": peak_tf},
           "clocks": clocks,
           "e2e": {"value": whole_job_builds_per_s(nD, world, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "ms_per_step": ms_e2e},
           "gpu_launches": int((launches_jk + 3) * args.steps),
           "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

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

UNIT = "builds/s"


def metric_name(w):
    return "non-symmetric J/K builds/s (fp64) at %d AO" % w.nao


def kept_integrals(Q, l, tau):
    """Unique (8-fold folded) Cartesian integrals the folded loop digests: sum over canonical shell quartets
    (AB)>=(CD) with Q_AB Q_CD >= tau of na nb nc nd  (oracle O6 / SURVEY 8.0 `ints`)."""
    nc = np.array([1, 3, 6, 10])[np.asarray(l)]
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


def pair_integrals(Q, l, tau):
    """Per bra shell pair p (canonical order A(A+1)/2+B of the folded loop O6): number of kept unique integrals of its
    quartets (p | q <= p).  Pure counting from the Schwarz bounds; used to scale oracle samples."""
    nc = np.array([1, 3, 6, 10])[np.asarray(l)]
    ns = len(l)
    iu = np.tril_indices(ns)
    qv = Q[iu]
    nf = (nc[iu[0]] * nc[iu[1]]).astype(np.float64)
    out = np.zeros(len(qv))
    step = 2048
    for p0 in range(0, len(qv), step):
        p1 = min(p0 + step, len(qv))
        keep = (qv[None, :p1] * qv[p0:p1, None] >= tau) & (np.arange(p1)[None, :] <= np.arange(p0, p1)[:, None])
        out[p0:p1] = nf[p0:p1] * (keep * nf[None, :p1]).sum(1)
    return out


class OracleSampler:
    """Times the oracle (as it stands) on bounded, STRATIFIED samples of the workload.  The bra shell-pair list of the
    folded loop O6 is cut into `nstrata` strata of equal kept-integral share; a sample is a run of bra pairs from the
    middle of one stratum, timed with all nD densities.  The oracle threads over bra pairs, so a run holds as many
    pairs as there are cores (a shorter run would leave cores idle and understate its rate).  Whole-sweep time =
    fixed per-call cost + sum_s rate_s x integrals_s: an EXTRAPOLATION, labelled so."""

    def __init__(self, w, D, nstrata=4):
        from oracle import oracle as O
        self.O, self.w, self.D, self.nstrata = O, w, D, nstrata
        b = w.basis
        self.Q = O.schwarz(b)
        self.npair = b.nshell * (b.nshell + 1) // 2
        pints = pair_integrals(self.Q, b.l, w.schwarz_tau)
        self.cum = np.concatenate([[0.0], np.cumsum(pints)])
        self.total = float(self.cum[-1])
        self.ncores = O.max_threads()
        self.mids = [int(np.searchsorted(self.cum, self.total * (k + 0.5) / nstrata)) for k in range(nstrata)]
        self.bounds = [int(np.searchsorted(self.cum, self.total * k / nstrata)) for k in range(nstrata + 1)]
        self.bounds[0], self.bounds[-1] = 0, self.npair
        self.used = 0.0
        self.t_fixed = self.call(0, 0)     # density-fastest copies of D, per-thread J/K buffers and their reduction
        self.rates = [[] for _ in range(nstrata)]
        self.sampled = 0.0

    def call(self, pa, pb):
        t = time.perf_counter()
        self.O.jk_folded(self.w.basis, self.D, self.w.schwarz_tau, pair_range=(pa, pb), Q=self.Q)
        dt = time.perf_counter() - t
        self.used += dt
        return dt

    def sample(self, k):
        pa = min(self.mids[k], max(self.npair - self.ncores, 0))
        pb = min(pa + self.ncores, self.npair)
        t = self.call(pa, pb)
        ints = max(self.cum[pb] - self.cum[pa], 1.0)
        self.rates[k].append(max(t - self.t_fixed, 1e-6) / ints)
        self.sampled += ints
        return t

    def result(self):
        known = [float(np.mean(r)) for r in self.rates if r]
        per = [float(np.mean(r)) if r else float(np.mean(known)) for r in self.rates]
        strata_ints = [self.cum[self.bounds[k + 1]] - self.cum[self.bounds[k]] for k in range(self.nstrata)]
        sweep_s = self.t_fixed + float(sum(r * n for r, n in zip(per, strata_ints)))
        allr = [x for r in self.rates for x in r]
        return {"value": self.D.shape[0] / sweep_s, "unit": UNIT, "cores": self.ncores,
                "kind": "oracle (extrapolated from a stratified bounded sample)", "extrapolated": True,
                "cpu_seconds_spent": self.used, "rate_s_per_integral": {"min": min(allr), "max": max(allr)},
                "sample": "oracle O6 (folded MD loop, all %d densities): %.1f s of CPU time; fixed cost per call %.2f s "
                          "(empty pair range); %d strata of equal integral share, %d run(s) of %d bra shell pairs from "
                          "the middle of a stratum: %.3g of the %.3g kept unique integrals sampled, %.3g-%.3g s per "
                          "integral; sweep = fixed + sum_s rate_s x integrals_s" %
                          (self.D.shape[0], self.used, self.t_fixed, self.nstrata, len(allr), self.ncores, self.sampled,
                           self.total, min(allr), max(allr))}


def oracle_sample(w, D, nstrata=4):
    smp = OracleSampler(w, D, nstrata)
    for k in range(nstrata):
        smp.sample(k)
    return smp.result()


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only).  Each step times one bounded sample
    (a run of bra shell pairs from one stratum, strata visited in turn); `ms_per_step` is the wall time a step really
    took, `value` the whole-sweep rate extrapolated from the timed samples (flagged)."""
    if rank != 0:
        return
    from paper_2607_05622_b200.inputs import make_workload
    w = make_workload(args.workload)
    nD = w.nD
    rng = np.random.default_rng(1)
    D = 1e-2 * rng.standard_normal((nD, w.nao, w.nao))    # cost does not depend on the values
    smp = OracleSampler(w, D)
    for s in range(args.warmup):
        smp.sample(s % smp.nstrata)
    smp.rates = [[] for _ in range(smp.nstrata)]
    smp.sampled = 0.0
    walls = [smp.sample(s % smp.nstrata) for s in range(args.steps)]
    r = smp.result()
    v = r["value"]
    out = {"impl": "reference", "metric": metric_name(w), "value": v, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(walls)),
           "ms_per_step_is": "wall time of one bounded sample step (NOT of a whole sweep)",
           "extrapolated": True, "extrapolated_ms_per_sweep": 1e3 * nD / v,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "%s (%d AO, %d densities)" % (w.name, w.nao, nD), "tau_schwarz": w.schwarz_tau},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": r["cores"], "kind": r["kind"], "sample": r["sample"],
                            "rate_s_per_integral": r["rate_s_per_integral"]},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


def sweep_report(torch, ltjk, w, local, T_host, steps, warmup, world, barrier, max_over_ranks, want_e2e=True, mode=0,
                 shard=None, quartet_shard=None):
    """Set up one workload (geometry-frozen part outside the timed region), time `steps` whole sweeps with CUDA events
    on the ctx stream, then the per-phase split (timing mode) and the roofline of the digestion kernel."""
    N, nD = w.nao, w.nD
    stream = torch.cuda.current_stream()
    ctx = ltjk.Context(local, stream)
    ctx.set_digest_mode(mode)
    ctx.set_basis(w.basis)
    npairs, nq_kept = ctx.build_shell_pairs(w.schwarz_tau)
    # the library's own minimax grid; a failure is an error, there is no fallback grid (include/ltjk.h, reading A8)
    tau, wts, lap_err = ltjk.laplace_quadrature(w.laplace_range[0], w.laplace_range[1], w.ntau)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Co, Cv, eo, ev, Td = dev(w.C_occ), dev(w.C_vir), dev(w.eps_occ), dev(w.eps_vir), dev(T_host)
    D = torch.empty((w.ntau, w.nT, N, N), dtype=torch.float64, device="cuda")
    Dn = D.view(nD, N, N)
    if quartet_shard is not None:
        # ONE sweep split in quartet space: partial J, K on every rank, then one all-reduce (sum)
        from paper_2607_05622_b200.dist import allreduce_jk
        ctx.set_quartet_shard(*quartet_shard)
        J = torch.empty_like(Dn)
        K = torch.empty_like(Dn)

        def step():
            ctx.build_pseudo_densities(Co, Cv, eo, ev, Td, tau, D)
            ctx.jk_build(Dn, J, K)
            allreduce_jk(J, K)
        want_e2e = False
    elif shard is None:
        J = torch.empty_like(Dn)
        K = torch.empty_like(Dn)

        def step():
            ctx.build_pseudo_densities(Co, Cv, eo, ev, Td, tau, D)
            ctx.jk_build(Dn, J, K)
    else:
        # ONE sweep split over the ranks: this rank builds densities shard = rank::world of the sweep
        idx = torch.from_numpy(np.ascontiguousarray(shard)).cuda()
        Ds = torch.empty((len(shard), N, N), dtype=torch.float64, device="cuda")
        J = torch.empty_like(Ds)
        K = torch.empty_like(Ds)

        def step():
            ctx.build_pseudo_densities(Co, Cv, eo, ev, Td, tau, D)
            torch.index_select(Dn, 0, idx, out=Ds)
            ctx.jk_build(Ds, J, K)
        want_e2e = False

    for _ in range(warmup):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    barrier()
    ms_per_step = max_over_ranks(e0.elapsed_time(e1), "cuda") / steps
    rep = {"ctx": ctx, "tau": tau, "Dn": Dn if shard is None else Ds, "J": J, "K": K, "ms_per_step": ms_per_step, "nq_kept": nq_kept,
           "launches_per_step": ctx.get_stats()["n_launches"] + 3, "laplace_maxerr": lap_err,
           "digest_mode": ctx.get_digest_mode()}

    # transform alone (a4): HBM-bound output stream of n_D N^2 doubles
    e0.record(stream)
    for _ in range(5):
        ctx.build_pseudo_densities(Co, Cv, eo, ev, Td, tau, D)
    e1.record(stream)
    torch.cuda.synchronize()
    t_ms = e0.elapsed_time(e1) / 5
    rep["transform"] = {"ms": t_ms, "gbs_written": 8e-9 * nD * N * N / (t_ms * 1e-3),
                        "tflops": 2e-12 * (w.nocc * w.nvir * N + w.nocc * N * N) * nD / (t_ms * 1e-3)}

    if want_e2e:    # the same sweep through the C ABI with HOST (pinned) buffers
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hCo, hCv, heo, hev, hT = pin(w.C_occ), pin(w.C_vir), pin(w.eps_occ), pin(w.eps_vir), pin(T_host)
        hJ = torch.empty((nD, N, N), dtype=torch.float64).pin_memory()
        hK = torch.empty((nD, N, N), dtype=torch.float64).pin_memory()
        ctx.sweep_host(hCo, hCv, heo, hev, hT, tau, hJ, hK)
        barrier()
        n_e2e = max(2, min(steps, 3))
        e0.record(stream)
        for _ in range(n_e2e):
            ctx.sweep_host(hCo, hCv, heo, hev, hT, tau, hJ, hK)
        e1.record(stream)
        barrier()
        rep["ms_e2e"] = max_over_ranks(e0.elapsed_time(e1) / n_e2e, "cuda")
        rep["h2d"] = 8 * (hCo.numel() + hCv.numel() + heo.numel() + hev.numel() + hT.numel())
        rep["d2h"] = 8 * (hJ.numel() + hK.numel())
        assert float((hK - K.cpu()).abs().max()) < 1e-9 * float(K.abs().max())
    return rep


def roofline_of(torch, ctx, w, rep, peak_tf):
    """Digestion kernel (dominant): algorithmic flop of one sweep / summed duration of its launches, timed live per
    launch group with CUDA events on the ctx stream (timing mode serialises ERI and digestion)."""
    Dn, J, K = rep["Dn"], rep["J"], rep["K"]
    ctx.set_timing(True)
    ctx.jk_build(Dn, J, K)
    torch.cuda.synchronize()
    st = ctx.get_stats()
    ctx.set_timing(False)
    Q = ctx.get_schwarz()
    ints = kept_integrals(Q, w.basis.l, w.schwarz_tau)
    alg = 20.0 * Dn.shape[0] * ints          # 2 J + 8 K FMAs per unique integral and density
    achieved = alg / (st["digest_ms"] * 1e-3) / 1e12
    return {"bound": "alu",
            "kernel": "digest kernel (J/K digestion; achieved = algorithmic flop of one sweep / summed duration of its launches)",
            "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf,
            "peak_source": "DFMA microbenchmark in this run (ltjk_bench_dfma_peak); MEASURED_PEAKS.json has no fp64 entry",
            "algorithmic_flops_per_sweep": alg, "executed_digest_flops_per_sweep": st["digest_flops"],
            "executed_over_algorithmic": st["digest_flops"] / alg,
            "digest_ms_per_sweep": st["digest_ms"], "eri_ms_per_sweep": st["eri_ms"],
            "whole_sweep_frac_of_peak": alg / (rep["ms_per_step"] * 1e-3) / 1e12 / peak_tf}, ints


def committed_ncu(name):
    """Counters that only ncu can give (DRAM bytes of the digestion launches, fp64 instruction counts of the ERI
    kernels) come from the committed capture of this round under profiles/; the bench line says so."""
    f = ROOT / "profiles" / "r2_ncu_counters.json"
    if not f.exists():
        return None
    return json.loads(f.read_text()).get(name)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="porphine")
    ap.add_argument("--impl", default="ltjk")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", type=int, default=0, help="digestion strategy (ltjk_set_digest_mode): 0 auto, 1 panels, 2 pair lists")
    ap.add_argument("--shard", choices=["problems", "densities", "quartets"], default="problems",
                    help="N > 1: every rank its own sweep (weak scaling, default); ONE sweep's densities dealt round-robin "
                         "(strong, no collective); or ONE sweep's shell quartets split over the ranks with an NCCL "
                         "all-reduce of J and K inside the timed step (strong)")
    ap.add_argument("--no-large", action="store_true", help="skip the 730-AO sub-run reported under config.large_730")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        # not launched under torchrun: spawn the N ranks ourselves (one process per GPU, NCCL over NVLink)
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node",
                                  str(args.gpus), "--master-addr", "127.0.0.1", "--master-port",
                                  os.environ.get("MASTER_PORT", "29517"), str(Path(__file__).resolve())] + sys.argv[1:])
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
    from paper_2607_05622_b200.dist import (density_shard, max_over_ranks, rank_amplitudes, sharded_sweep_builds_per_s,
                                            whole_job_builds_per_s)
    strong = world > 1 and args.shard in ("densities", "quartets")
    T_host = w.T if strong else rank_amplitudes(w, rank)
    shard = density_shard(nD, rank, world) if (world > 1 and args.shard == "densities") else None
    qshard = (rank, world) if (world > 1 and args.shard == "quartets") else None

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    rep = sweep_report(torch, ltjk, w, local, T_host, args.steps, args.warmup, world, barrier, max_over_ranks, mode=args.mode,
                       shard=shard, quartet_shard=qshard)
    clocks = sampler.stop() if rank == 0 else None
    ms_per_step = rep["ms_per_step"]
    value = sharded_sweep_builds_per_s(nD, ms_per_step) if strong else whole_job_builds_per_s(nD, world, ms_per_step)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ctx, Dn = rep["ctx"], rep["Dn"]
    stream = torch.cuda.current_stream()
    peak_tf = ctx.bench_dfma_peak()
    hbm_gbs = ctx.bench_copy_peak()
    roofline, ints = roofline_of(torch, ctx, w, rep, peak_tf)
    tr = committed_ncu("digest_dram_bytes_per_sweep_%s" % w.name)
    roofline["traffic"] = tr
    roofline["traffic_source"] = ("committed ncu capture profiles/r2_ncu_counters.json (not measured in this run)"
                                  if tr is not None else None)
    # one Laplace point per call (n_D = n_T): makes the integral re-computation per call visible
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
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
    measured = json.loads((ROOT / "MEASURED_PEAKS.json").read_text()) if (ROOT / "MEASURED_PEAKS.json").exists() else {}
    hbm_peak = measured.get("hbm_gbs", hbm_gbs)
    # the transform is a dense fp64 contraction (DMMA): its roof is the fp64 tensor peak, taken as the measured bf16
    # tensor peak x the guide's nominal ratio 45 / 2250 (blackwell_cuda_programming.md: B200 FP64 tensor 45 TFLOP/s);
    # at that roof it would write D at ~0.9 TB/s, so the HBM fraction asked for by north_star cannot exceed ~0.14
    f64_tensor_peak = measured.get("bf16_tflops", 1605.6) * 45.0 / 2250.0
    transform = dict(rep["transform"], frac_of_hbm_peak=rep["transform"]["gbs_written"] / hbm_peak, hbm_peak_gbs=hbm_peak,
                     hbm_peak_source="MEASURED_PEAKS.json" if "hbm_gbs" in measured else "copy microbenchmark in this run",
                     bound="tensor (f64 DMMA)", f64_tensor_peak_tflops=f64_tensor_peak,
                     frac_of_f64_tensor_peak=rep["transform"]["tflops"] / f64_tensor_peak)
    cpu = None
    if not args.no_cpu_baseline:
        cpu = oracle_sample(w, Dn.cpu().numpy())
    launches = int(rep["launches_per_step"] * args.steps)
    e2e = None
    if "ms_e2e" in rep:
        e2e = {"value": whole_job_builds_per_s(nD, world, rep["ms_e2e"]), "unit": UNIT, "h2d_bytes_per_step": rep["h2d"],
               "d2h_bytes_per_step": rep["d2h"], "ms_per_step": rep["ms_e2e"]}
    config = {"workload": "%s (%d AO, %d atoms, n_tau=%d x n_T=%d = %d non-symmetric densities per sweep)" %
                          (w.name, N, w.basis.natom, w.ntau, w.nT, nD),
              "tau_schwarz": w.schwarz_tau, "shell_quartets_kept": rep["nq_kept"], "unique_integrals_kept": ints,
              "l2": "inputs_larger_than_L2 (D, J, K are %.0f MB each)" % (8e-6 * nD * N * N),
              "setup_outside_timed_region": "basis upload, shell pairs, Schwarz, work lists (geometry-frozen)",
              "laplace_grid": "library minimax, max error %.3e" % rep["laplace_maxerr"],
              "digest_mode": {1: "block panels", 2: "pair lists"}[rep["digest_mode"]],
              "one_laplace_point_per_call": single_point, "transform": transform,
              "eri_fp64_flops_per_sweep_ncu": committed_ncu("eri_fp64_flops_per_sweep_%s" % w.name),
              "gpu": torch.cuda.get_device_name(local), "hbm_copy_gbs_measured": hbm_gbs,
              "dfma_peak_tflops_measured": peak_tf}
    # free the headline workload before the sub-runs
    del rep, Dn, D1, J1, K1
    ctx.close()
    torch.cuda.empty_cache()
    if world == 1 and w.name != "large":
        # callers that cannot batch: one Laplace point per call with the geometry-frozen integral cache
        # (ltjk_set_resident), and the N3 particle-particle ladder (K-only batches of 160 pair columns)
        c2 = ltjk.Context(local, stream)
        c2.set_resident(True)
        c2.set_basis(w.basis)
        c2.build_shell_pairs(w.schwarz_tau)
        rng = np.random.default_rng(7)
        D1 = torch.from_numpy(1e-2 * rng.standard_normal((w.nT, N, N))).cuda()
        J1 = torch.empty_like(D1)
        K1 = torch.empty_like(D1)
        c2.jk_build(D1, J1, K1)                      # first build fills the cache
        torch.cuda.synchronize()
        e0.record(stream)
        c2.jk_build(D1, J1, K1)
        e1.record(stream)
        torch.cuda.synchronize()
        config["one_laplace_point_per_call_resident"] = {
            "n_D": int(w.nT), "ms": e0.elapsed_time(e1), "builds_per_s": w.nT / (e0.elapsed_time(e1) * 1e-3),
            "note": "integral panels of the geometry kept in HBM (opt-in cache, not the headline path)"}
        npair = 320
        Cv = torch.from_numpy(np.ascontiguousarray(w.C_vir)).cuda()
        X = torch.from_numpy(1e-2 * rng.standard_normal((npair, w.nvir, w.nvir))).cuda()
        Lo = torch.empty_like(X)
        c2.pp_ladder(Cv, X, Lo)
        torch.cuda.synchronize()
        e0.record(stream)
        c2.pp_ladder(Cv, X, Lo)
        e1.record(stream)
        torch.cuda.synchronize()
        config["pp_ladder"] = {"pair_columns": npair, "nvir": int(w.nvir), "ms": e0.elapsed_time(e1),
                               "pair_columns_per_s": npair / (e0.elapsed_time(e1) * 1e-3),
                               "note": "L[p,a,b] = sum_ef (ae|bf) X[p,e,f] as K-only builds (SURVEY 8(f) N3), resident panels"}
        launches += 2 * (c2.get_stats()["n_launches"])
        del D1, J1, K1, X, Lo
        c2.close()
        torch.cuda.empty_cache()
        # N2: derivative builds J^x(A,B), K^x(A,B) (Eq. 18) on the 160-AO workload, 4 non-symmetric density pairs
        ws = make_workload("small")
        c3 = ltjk.Context(local, stream)
        c3.set_basis(ws.basis)
        Ag = torch.from_numpy(1e-2 * rng.standard_normal((4, ws.nao, ws.nao))).cuda()
        Bg = torch.from_numpy(1e-2 * rng.standard_normal((4, ws.nao, ws.nao))).cuda()
        gJ = torch.empty((4, ws.basis.xyz.shape[0], 3), dtype=torch.float64, device="cuda")
        gK = torch.empty_like(gJ)
        c3.jk_grad(Ag, Bg, gJ, gK)
        torch.cuda.synchronize()
        e0.record(stream)
        c3.jk_grad(Ag, Bg, gJ, gK)
        e1.record(stream)
        torch.cuda.synchronize()
        nq = ws.basis.nshell ** 2 * (ws.basis.nshell * (ws.basis.nshell + 1) // 2)
        config["jk_grad"] = {"workload": "small (160 AO, 73 shells, 14 atoms), 4 density pairs, no screening",
                             "ms": e0.elapsed_time(e1), "shell_quartet_derivatives_per_s": nq / (e0.elapsed_time(e1) * 1e-3),
                             "note": "J^x(A,B), K^x(A,B) of Eq. 18 (SURVEY 8(f) N2): first correct version, one thread per "
                                     "(M, N, {K,R}), derivative integrals contracted on the fly"}
        launches += c3.get_stats()["n_launches"]
        c3.close()
    if world == 1 and not args.no_large:
        # f shells (looped ERI kernel) -- the medium geometry with an f shell on every heavy atom, one
        # sweep of its 80 pseudo-densities; then the matrix-level spherical transform of the 80 J matrices
        wf = make_workload("medium_f")
        repf = sweep_report(torch, ltjk, wf, local, wf.T, 2, 1, 1, barrier, max_over_ranks, want_e2e=False, mode=0)
        rf, intsf = roofline_of(torch, repf["ctx"], wf, repf, peak_tf)
        cf = repf["ctx"]
        nsph = cf.get_nsph()
        Js = torch.empty((wf.nD, nsph, nsph), dtype=torch.float64, device="cuda")
        cf.sph_from_cart(repf["J"], Js)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(10):
            cf.sph_from_cart(repf["J"], Js)
        e1.record(stream)
        torch.cuda.synchronize()
        t_sph = e0.elapsed_time(e1) / 10
        gbs = 8e-9 * wf.nD * (wf.nao ** 2 + nsph ** 2) / (t_sph * 1e-3)
        config["f_shells_medium_f"] = {
            "workload": "medium geometry, heavy atoms 4s3p1d1f (400 Cartesian AO, 10 f shells), %d densities" % wf.nD,
            "value": wf.nD / (repf["ms_per_step"] * 1e-3), "unit": UNIT, "ms_per_step": repf["ms_per_step"], "steps": 2,
            "warmup": 1, "unique_integrals_kept": intsf, "eri_ms_per_sweep": rf["eri_ms_per_sweep"],
            "digest_ms_per_sweep": rf["digest_ms_per_sweep"], "digest_frac_of_dfma_peak": rf["frac"],
            "sph_from_cart": {"n_sph": nsph, "ms": t_sph, "gbs": gbs, "frac_of_hbm_peak": gbs / hbm_peak,
                              "bytes": "8 (N^2 + N_sph^2) per matrix"},
            "note": "classes with an f shell run the looped kernel (csrc/ltjk_eri_loop.cu, one CTA per quartet)"}
        launches += int(repf["launches_per_step"] * 3) + 11
        cf.close()
    if world == 1 and not args.no_large and w.name != "large":
        wl = make_workload("large")
        s2 = ClockSampler(local)
        s2.start()
        repl = sweep_report(torch, ltjk, wl, local, wl.T, 2, 1, 1, barrier, max_over_ranks, want_e2e=False, mode=args.mode)
        cl2 = s2.stop()
        rl, intsl = roofline_of(torch, repl["ctx"], wl, repl, peak_tf)
        trl = committed_ncu("digest_dram_bytes_per_sweep_large")
        rl["traffic"] = trl
        config["large_730"] = {"metric": metric_name(wl), "value": wl.nD / (repl["ms_per_step"] * 1e-3), "unit": UNIT,
                               "ms_per_step": repl["ms_per_step"], "steps": 2, "warmup": 1, "n_D": wl.nD,
                               "unique_integrals_kept": intsl, "roofline": rl, "clocks": cl2,
                               "digest_mode": {1: "block panels", 2: "pair lists"}[repl["digest_mode"]],
                               "transform": repl["transform"]}
        launches += int(repl["launches_per_step"] * 2)
        # N4: the matrix-level spherical transform of the 192 J matrices (819 MB in, 640 MB out: larger than L2)
        cl = repl["ctx"]
        nsl = cl.get_nsph()
        Jsl = torch.empty((wl.nD, nsl, nsl), dtype=torch.float64, device="cuda")
        cl.sph_from_cart(repl["J"], Jsl)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(5):
            cl.sph_from_cart(repl["J"], Jsl)
        e1.record(stream)
        torch.cuda.synchronize()
        t_sl = e0.elapsed_time(e1) / 5
        gbl = 8e-9 * wl.nD * (wl.nao ** 2 + nsl ** 2) / (t_sl * 1e-3)
        config["large_730"]["sph_from_cart"] = {"n_sph": nsl, "ms": t_sl, "gbs": gbl, "frac_of_hbm_peak": gbl / hbm_peak,
                                                "bytes": "8 (N^2 + N_sph^2) per matrix, 192 matrices"}
        launches += 6
        del Jsl
        repl["ctx"].close()
    out = {"metric": metric_name(w), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if strong else "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config, "clocks": clocks, "e2e": e2e,
           "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

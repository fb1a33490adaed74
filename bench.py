#!/usr/bin/env python
"""bench.py — even-odd Wilson hop throughput (BASELINE.json metric) on one B200, plus the end-to-end solve.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--lattice 32,32,32,64] [--prec fp32|fp64|half] [--recon 18|12] [--skip-e2e] [--skip-cpu]

Workload (config.workload): BASELINE.json config 3 — 32^3x64, fp32 storage, 18-real links, even-odd Wilson hop
D_eo applied to one parity (the lattice north_star's target is quoted on; it is the largest single-GPU hop config
whose metric is the headline).  A step = one bq_wilson_apply(EVEN) = one hop-kernel launch over Vh sites.
  value     GFlop/s at 1320 flop/site with all fields resident in HBM (CUDA events around K launches).
  roofline  algorithmic bytes (768 B/site fp32/18) / the same per-launch time, against the
            measured copy bandwidth in MEASURED_PEAKS.json.
  e2e       the same flop count through the public solve call with HOST buffers: bq_solve (BASELINE.json config 4,
            Wilson-clover, fp32 inner / fp64 outer BiCGStab to 1e-10) from a pinned host b to a pinned host x;
            hop flops executed / wall time, host<->device copies and layout conversion inside the timed region.
  cpu_baseline  the CPU oracle (oracle/, as it stands) computing the same hop on a bounded sample of the sites.
Inputs are synthetic and seeded (paper_2111_04457_b200/inputs).  The working set (805 MB per apply) is far larger
than the 126 MB L2 and the timed loop rotates over 4 (source, result) pairs, so no explicit L2 flush is needed.
N > 1: replicas only — every rank runs the same workload on its own GPU, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1320
BYTES_PER_SITE = {("fp64", 18): 1536, ("fp64", 12): 1152, ("fp32", 18): 768, ("fp32", 12): 576,
                  ("half", 18): 392, ("half", 12): 296}
PREC_ID = {"fp64": 0, "fp32": 1, "half": 2}
FALLBACK_HBM_GBS = 6650.0


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lattice", default="32,32,32,64")
    ap.add_argument("--prec", default="fp32", choices=["fp64", "fp32", "half"])
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12])
    ap.add_argument("--skip-e2e", action="store_true")
    ap.add_argument("--skip-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def workload_name(L, prec, recon):
    return f"{L[0]}x{L[1]}x{L[2]}x{L[3]} {prec} {recon}-real even-odd Wilson hop (BASELINE config 3 shape)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = os.path.join(ROOT, "gpurun_out", f"clocks_{index}.csv")

    def start(self):
        os.makedirs(os.path.dirname(self.path), exist_ok=True)
        q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        try:
            with open(self.path) as f:
                for line in f:
                    c = [v.strip() for v in line.split(",")]
                    if len(c) < 9:
                        continue
                    try:
                        sm.append(float(c[1])); mx.append(float(c[2]))
                    except ValueError:
                        continue
                    for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                        if v.lower().startswith("active"):
                            reasons.add(name)
        except OSError:
            pass
        if sm:
            out["sm_mhz"] = float(np.median(sm))
            out["sm_max_mhz"] = float(max(mx))
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def oracle_hop_sample(U, psi, kappa, L, seconds_target=12.0):
    """The CPU oracle computing (D [0; psi_odd])(x) at a sample of EVEN sites = the same hop, 1320 flop/site."""
    from oracle import bqo
    from paper_2111_04457_b200 import inputs
    par = inputs.site_parity(L).ravel()
    even_sites = np.nonzero(par == 0)[0]
    masked = np.where((inputs.site_parity(L) == 1)[..., None, None], psi, 0)
    bqo.dirac_apply_sites(U, masked, kappa, even_sites[:4096])     # spin up the thread team
    # whole passes over the even sites until about seconds_target of CPU work has been done
    t0 = time.perf_counter()
    done = 0
    while True:
        bqo.dirac_apply_sites(U, masked, kappa, even_sites)
        done += len(even_sites)
        dt = time.perf_counter() - t0
        if dt >= seconds_target:
            break
    return {"value": FLOP_PER_SITE * done / dt / 1e9, "unit": "GFlop/s", "cores": bqo.num_threads(), "kind": "oracle",
            "sample": f"{done} even-site hop evaluations ({done / len(even_sites):.2f} passes over the even sites) "
                      f"of the same lattice and inputs, oracle/bqo.c dirac_apply_sites, {dt:.1f} s"}, dt, done


def run_reference(args, L):
    """--impl reference: the CPU oracle timed on the host cores on the same workload/metric (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2111_04457_b200 import inputs
    seed = inputs.BASE_SEED + 3
    U = inputs.gauge(L, seed, 0.5)
    psi = inputs.spinor(L, seed)
    from oracle import bqo
    par = inputs.site_parity(L)
    even_sites = np.nonzero(par.ravel() == 0)[0]
    masked = np.where((par == 1)[..., None, None], psi, 0)
    # each step = the hop on a fixed sample of the even sites, sized so the whole run stays within minutes
    probe = even_sites[:: max(1, len(even_sites) // 32768)]
    t0 = time.perf_counter()
    bqo.dirac_apply_sites(U, masked, 0.125, probe)
    rate = len(probe) / (time.perf_counter() - t0)           # sites per second on this host
    per_step = int(max(1024, min(len(even_sites), rate * 30.0 / max(1, args.steps + args.warmup))))   # ~30 s in total
    sample = even_sites[:: max(1, len(even_sites) // per_step)][:per_step]
    for _ in range(args.warmup):
        bqo.dirac_apply_sites(U, masked, 0.125, sample)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        bqo.dirac_apply_sites(U, masked, 0.125, sample)
    dt = time.perf_counter() - t0
    value = FLOP_PER_SITE * len(sample) * args.steps / dt / 1e9
    line = {
        "impl": "reference", "metric": "even-odd Wilson hop GFlop/s (1320 flop/site)", "value": value, "unit": "GFlop/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(L, args.prec, args.recon), "note": "CPU oracle, fp64, bounded sample per step"},
        "cpu_baseline": {"value": value, "unit": "GFlop/s", "cores": bqo.num_threads(), "kind": "oracle",
                         "sample": f"{len(sample)} even sites per step x {args.steps} steps, oracle/bqo.c dirac_apply_sites"},
        "e2e": {"value": value, "unit": "GFlop/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    args = parse_args()
    L = tuple(int(v) for v in args.lattice.split(","))
    if args.impl == "reference":
        run_reference(args, L)
        return

    import torch
    from paper_2111_04457_b200 import bq, build, inputs, replicas
    rank, local_rank, world = replicas.env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    replicas.init("nccl", torch.device("cuda", local_rank))
    build.build()
    bq.lib()
    prec, recon = PREC_ID[args.prec], (0 if args.recon == 18 else 1)
    Vh = L[0] * L[1] * L[2] * L[3] // 2
    kappa = 0.125
    seed = inputs.BASE_SEED + 3            # config 3: links exp(i*0.5*H), Gaussian source
    U = inputs.gauge(L, seed, 0.5)
    psi = inputs.spinor(L, seed)

    barrier = replicas.barrier

    lat = bq.Lattice(L)
    bq.bq_gauge_load(lat.h, U)
    # NSETS (source, result) pairs used round-robin, so that a launch finds neither its source nor the previous
    # result in L2 (the links are streamed evict-first and are 6x larger than L2 anyway)
    NSETS = 4
    srcs = [lat.import_field(psi, prec, bq.BQ_ODD)]
    srcs += [srcs[0].clone() for _ in range(NSETS - 1)]
    outs = [lat.field(prec, bq.BQ_EVEN) for _ in range(NSETS)]
    for i in range(max(3, args.warmup)):
        bq.bq_wilson_apply(lat.h, outs[i % NSETS], srcs[i % NSETS], kappa, bq.BQ_EVEN, prec, recon)
    c0 = bq.bq_get_counters(lat.h)
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()                                   # legacy default stream = the stream the kernels are launched on
    for i in range(args.steps):
        bq.bq_wilson_apply(lat.h, outs[i % NSETS], srcs[i % NSETS], kappa, bq.BQ_EVEN, prec, recon)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop()
    c1 = bq.bq_get_counters(lat.h)
    launches = int(c1["launches"] - c0["launches"])
    ms = replicas.max_over_ranks(ms)
    ms_per_step = ms / args.steps
    gflops = world * FLOP_PER_SITE * Vh / (ms_per_step * 1e-3) / 1e9
    bps = BYTES_PER_SITE[(args.prec, args.recon)]
    peak, peak_src = peaks()
    achieved = bps * Vh / (ms_per_step * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "hop_traffic.json")   # DRAM bytes per launch from the committed ncu capture
    if os.path.exists(tpath):
        with open(tpath) as f:
            traffic = json.load(f).get(f"{args.lattice}/{args.prec}/{args.recon}")
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": peak_src, "kernel": "hop_kernel", "algorithmic_bytes_per_site": bps,
                "frac_of_nominal_8000": achieved / 8000.0}

    # ---- e2e: the public solve call with host buffers (BASELINE config 4, Wilson-clover, fp32 inner / fp64 outer) ----
    e2e = None
    if not args.skip_e2e:
        seed4 = inputs.BASE_SEED + 4
        U4 = inputs.gauge(L, seed4, 0.5)
        b_host = torch.from_numpy(inputs.spinor(L, seed4)).pin_memory()
        x_host = torch.zeros_like(b_host).pin_memory()
        lat4 = bq.Lattice(L)
        bq.bq_gauge_load(lat4.h, U4)
        opts = bq.bq_solve_opts(inner_prec=bq.BQ_FP32, recon=bq.BQ_RECON18, csw=1.0, x0_zero=1)   # x is output only
        times, infos, hops = [], [], []
        for it in range(1 + args.e2e_steps):      # first solve = warm-up (clover build, workspace allocation)
            k0 = bq.bq_get_counters(lat4.h)
            barrier()
            t0 = time.perf_counter()
            info = bq.bq_solve(lat4.h, b_host.numpy(), x_host.numpy(), 0.1215, 1e-10, opts)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            k1 = bq.bq_get_counters(lat4.h)
            if it > 0:
                times.append(dt); infos.append(info)
                hops.append(sum(int(k1[k] - k0[k]) for k in ("hop_fp64", "hop_fp32", "hop_half")))
        dt = replicas.max_over_ranks(max(times))
        nbytes = b_host.numel() * 16
        e2e = {"value": world * FLOP_PER_SITE * Vh * hops[-1] / dt / 1e9, "unit": "GFlop/s",
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "what": "bq_solve host->host, BASELINE config 4 (32^3x64 Wilson-clover csw=1 kappa=0.1215, fp32 inner / fp64 outer "
                       "BiCGStab to 1e-10, zero initial guess declared with opts.x0_zero): hop flops executed / wall time incl. H2D of b, "
                       "layout conversion, solve, D2H of x",
               "time_to_solution_s": dt, "device_seconds": infos[-1].seconds,
               "phase_seconds": dict(zip(("h2d+import", "prepare", "iterate", "reconstruct+residual", "export+d2h"), list(infos[-1].phase_seconds))), "inner_iters": infos[-1].inner_iters,
               "outer_cycles": infos[-1].outer_cycles, "hop_launches": hops[-1], "true_rel_residual": infos[-1].true_rel_residual}
        # the plain operator through host buffers, for completeness: canonical fp64 field on the (pinned) host -> H2D -> layout
        # conversion -> ONE hop -> conversion back -> D2H.  PCIe moves 2 x 402 MB for 1.38 GFlop: transfer-bound by construction.
        psi_host = torch.from_numpy(psi).pin_memory()
        out_host = torch.zeros_like(psi_host).pin_memory()
        dev_in = torch.empty_like(psi_host, device="cuda")
        dev_out = torch.zeros_like(dev_in)
        buf_in, buf_out = lat.field(prec, bq.BQ_ODD), lat.field(prec, bq.BQ_EVEN)
        ts = []
        for it in range(3):
            barrier()
            t0 = time.perf_counter()
            dev_in.copy_(psi_host, non_blocking=True)
            bq.bq_field_import(lat.h, buf_in, dev_in, bq.BQ_ODD, prec)
            bq.bq_wilson_apply(lat.h, buf_out, buf_in, kappa, bq.BQ_EVEN, prec, recon)
            bq.bq_field_export(lat.h, dev_out, buf_out, bq.BQ_EVEN, prec)
            out_host.copy_(dev_out, non_blocking=True)
            torch.cuda.synchronize()
            ts.append(time.perf_counter() - t0)
        ta = replicas.max_over_ranks(min(ts[1:]))
        e2e["host_apply"] = {"value": world * FLOP_PER_SITE * Vh / ta / 1e9, "unit": "GFlop/s", "seconds": ta,
                             "h2d_bytes_per_step": psi_host.numel() * 16, "d2h_bytes_per_step": out_host.numel() * 16,
                             "what": "one bq_wilson_apply(EVEN) from a pinned host canonical field to a pinned host canonical field "
                                     "(H2D, bq_field_import, hop, bq_field_export, D2H)"}
        lat4.close()

    # ---- the rest of the path, per kernel (bq_bench_kernel hooks; device times, operands rotated out of L2) ----
    extras = None
    if rank == 0 and world == 1 and not args.skip_e2e and L == (32, 32, 32, 64):
        def gbs(us, nb):
            return {"us": us, "gbs": nb / us / 1e3, "frac_of_peak": nb / us / 1e3 / peak}
        extras = {"note": "device time per launch and algorithmic GB/s (every operand once) of other kernels of the path, same lattice"}
        for name, which, pr, rc, csw in (("hop_fp32_12", "hop", 1, 1, 0.0), ("hop_fp64_18", "hop", 0, 0, 0.0), ("hop_half_18", "hop", 2, 0, 0.0),
                                         ("bicg_iter_fp32_wilson", "bicg_iter", 1, 0, 0.0), ("bicg_iter_fp32_clover", "bicg_iter", 1, 0, 1.0),
                                         ("bicg_iter_half_wilson", "bicg_iter", 2, 0, 0.0)):
            extras[name] = gbs(*bq.bq_bench_kernel(lat.h, which, pr, rc, csw, 0.1215, 100, 3))
        for name, which, csw in (("hop_fp32_18_x12", "hop", 0.0), ("bicg_iter_fp32_wilson_x12", "bicg_iter", 0.0)):
            us, nb = bq.bq_bench_kernel_multi(lat.h, which, 1, 12, 0, csw, 0.1215, 16, 2)
            extras[name] = dict(gbs(us, nb), us_per_rhs=us / 12, nrhs=12,
                                gflops_hop=(FLOP_PER_SITE * Vh * 12 / us / 1e3 if which == "hop" else None))

    cpu = None
    if rank == 0 and world == 1 and not args.skip_cpu:
        cpu, _, _ = oracle_hop_sample(U, psi, kappa, L)
    lat.close()
    replicas.finish()
    if rank != 0:
        return
    line = {
        "metric": "even-odd Wilson hop GFlop/s (1320 flop/site)", "value": gflops, "unit": "GFlop/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": {"fp64": "f64", "fp32": "f32", "half": "f16-storage/f32-math"}[args.prec],
        "data": "synthetic",
        "config": {"workload": workload_name(L, args.prec, args.recon), "kappa": kappa, "links": "exp(i*0.5*H), seeded",
                   "l2": f"inputs larger than L2, no flush: {bps * Vh / 1e6:.0f} MB per apply (links streamed once) and {NSETS} (source, result) "
                         "pairs used round-robin, so no operand of a launch is left in the 126 MB L2 by the previous ones",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "hbm_gbs": achieved, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "extras": extras,
    }
    print(json.dumps(line))


if __name__ == "__main__":
    main()

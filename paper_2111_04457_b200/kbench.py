"""Per-kernel device times of the hot path against the HBM roofline.

    python -m paper_2111_04457_b200.kbench [--lattice 32,32,32,64] [--reps 200] [--nsets 3] [--json]

Each line: kernel, storage precision, link form, microseconds per launch (CUDA events inside libbq's
bq_bench_kernel, operands rotated over `nsets` scratch sets so that nothing is found in L2), algorithmic
GB/s (every operand once) and its fraction of the measured copy bandwidth (MEASURED_PEAKS.json).
Inputs: seeded synthetic gauge field of BASELINE config 3/4 (exp(i*0.5*H)); vector contents are irrelevant.
"""
from __future__ import annotations

import argparse
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", default="32,32,32,64")
    ap.add_argument("--reps", type=int, default=200)
    ap.add_argument("--nsets", type=int, default=3)
    ap.add_argument("--json", action="store_true")
    ap.add_argument("--precs", default="fp64,fp32,half")
    ap.add_argument("--nrhs", default="2,4,8,12,16", help="right-hand sides per launch for the multi-rhs lines ('' = none)")
    ap.add_argument("--solve", type=int, default=0, metavar="NRHS",
                    help="also time bq_solve_multi on NRHS point sources against NRHS separate bq_solve calls (device buffers)")
    ap.add_argument("--only", default="", help="comma-separated kernel names to run (e.g. 'hop,hop x12'); default all")
    args = ap.parse_args()
    only = [v.strip().replace("_x", " x") for v in args.only.split(",") if v.strip()]     # "hop_x12" = "hop x12"
    import torch
    from . import bq, build, inputs
    assert torch.cuda.is_available(), "kbench needs a CUDA device"
    build.build()
    L = tuple(int(v) for v in args.lattice.split(","))
    peak = 6650.0
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        with open(pk) as f:
            peak = float(json.load(f)["hbm_gbs"])
    U = inputs.gauge(L, inputs.BASE_SEED + 4, 0.5)
    rows = []
    with bq.Lattice(L) as lat:
        bq.bq_gauge_load(lat.h, U)
        for pname in args.precs.split(","):
            prec = {"fp64": 0, "fp32": 1, "half": 2}[pname]
            for which, recon, csw in ([("hop", r, 0.0) for r in (0, 1)] + [("hop_xpay", 0, 0.0), ("hop_clovinv", 0, 1.0), ("hop_clov_xpay", 0, 1.0),
                                      ("schur", 0, 0.0), ("schur", 0, 1.0), ("norm2", 0, 0.0), ("p_update", 0, 0.0), ("alpha", 0, 0.0),
                                      ("s_update", 0, 0.0), ("omega", 0, 0.0), ("final", 0, 0.0), ("hop_xpay_alpha", 0, 0.0),
                                      ("hop_xpay_omega", 0, 0.0), ("hop_xpay_alpha", 0, 1.0), ("hop_xpay_omega", 0, 1.0),
                                      ("bicg_iter_unfused", 0, 0.0), ("bicg_iter", 0, 0.0), ("bicg_iter", 1, 0.0),
                                      ("bicg_iter_unfused", 0, 1.0), ("bicg_iter", 0, 1.0)]):
                if only and which not in only:
                    continue
                us, nb = bq.bq_bench_kernel(lat.h, which, prec, recon, csw, 0.1215, args.reps, args.nsets)
                rows.append({"kernel": which, "prec": pname, "recon": 12 if recon else 18, "csw": csw, "us": us, "bytes": nb,
                             "gbs": nb / us / 1e3, "frac": nb / us / 1e3 / peak})
        # multi-rhs kernels: one launch covers nrhs right-hand sides; bytes count the links once
        for pname in args.precs.split(","):
            prec = {"fp64": 0, "fp32": 1, "half": 2}[pname]
            for nrhs in [int(v) for v in args.nrhs.split(",") if v]:
                for which, recon, csw in (("hop", 0, 0.0), ("hop", 1, 0.0), ("schur", 0, 0.0), ("schur", 0, 1.0), ("bicg_iter", 0, 0.0),
                                          ("bicg_iter", 0, 1.0)):
                    if only and f"{which} x{nrhs}" not in only:
                        continue
                    us, nb = bq.bq_bench_kernel_multi(lat.h, which, prec, nrhs, recon, csw, 0.1215, max(8, args.reps // nrhs), 2)
                    rows.append({"kernel": f"{which} x{nrhs}", "prec": pname, "recon": 12 if recon else 18, "csw": csw, "us": us,
                                 "bytes": nb, "gbs": nb / us / 1e3, "frac": nb / us / 1e3 / peak, "nrhs": nrhs, "us_per_rhs": us / nrhs})
        solve = None
        if args.solve > 0:
            # the paper's propagator workload: point sources e_s (x) e_c at the origin, one gauge field
            n = args.solve
            Lx, Ly, Lz, Lt = L
            b = torch.zeros((n, Lt, Lz, Ly, Lx, 4, 3), dtype=torch.complex128, device="cuda")
            for k in range(n):
                b[k, 0, 0, 0, 0, (k // 3) % 4, k % 3] = 1.0
            x = torch.zeros_like(b)
            solve = []
            for pname, csw in (("fp32", 0.0), ("fp32", 1.0), ("half", 0.0)):
                opts = bq.bq_solve_opts(inner_prec={"fp32": 1, "half": 2}[pname], csw=csw)
                for rep in range(2):                       # first pass = warm-up (workspace, clover build)
                    x.zero_()
                    infos = bq.bq_solve_multi(lat.h, b, x, n, 0.1215, 1e-10, opts)
                    t_multi = infos[0].seconds
                    t_single = 0.0
                    x.zero_()
                    for k in range(n):
                        t_single += bq.bq_solve(lat.h, b[k], x[k], 0.1215, 1e-10, opts).seconds
                solve.append({"prec": pname, "csw": csw, "nrhs": n, "multi_s": t_multi, "single_s": t_single,
                              "iters": [i.inner_iters for i in infos], "res": max(i.true_rel_residual for i in infos)})
    if args.json:
        print(json.dumps({"lattice": L, "peak_gbs": peak, "rows": rows, "solve": solve}))
        return
    print(f"# lattice {L}, reps {args.reps}, nsets {args.nsets}, peak {peak:.0f} GB/s (measured copy)")
    print(f"{'kernel':18s} {'prec':5s} {'links':5s} {'csw':>4s} {'us':>9s} {'MB':>9s} {'GB/s':>8s} {'frac':>6s}")
    for r in rows:
        tail = f"   {r['us_per_rhs']:7.1f} us/rhs" if "nrhs" in r else ""
        print(f"{r['kernel']:18s} {r['prec']:5s} {r['recon']:<5d} {r['csw']:4.1f} {r['us']:9.1f} {r['bytes'] / 1e6:9.1f} {r['gbs']:8.0f} {r['frac']:6.3f}{tail}")
    for r in solve or []:
        print(f"# solve x{r['nrhs']} {r['prec']} inner, csw {r['csw']}: bq_solve_multi {r['multi_s'] * 1e3:.1f} ms vs {r['nrhs']} x bq_solve "
              f"{r['single_s'] * 1e3:.1f} ms (device time incl. layout conversion), inner iterations {r['iters']}, worst |r|/|b| {r['res']:.1e}")


if __name__ == "__main__":
    main()

"""Time (or profile under ncu) the fused Mpc / Mpc^dagger kernels on one of BASELINE.json's workloads.

  python timeop.py --workload 3 --prec fp32,half --reps 5 --warmup 2

Prints one JSON line per (op, precision): ms per application and per kernel, model GB/s, TFLOP/s.
Few launches, so it is the command the ncu captures under profiles/ are taken with.
"""
import argparse
import json
import time

import torch

from paper_1701_07559_b200 import binding, build, inputs


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", type=int, default=3)
    ap.add_argument("--prec", default="fp64,fp32,half")
    ap.add_argument("--ops", default="0,1")
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--reconstruct", default=None)
    ap.add_argument("--fma-rates", action="store_true", help="also print the measured FFMA / FFMA2 rates")
    ap.add_argument("--l2-rates", action="store_true", help="also print the measured L2 -> SM and DRAM streaming rates")
    ap.add_argument("--opt", action="append", default=[], help="extra mdwf_set_option key=value")
    ap.add_argument("--batch", type=int, default=0, help="also time the batched operator (mdwf_apply_batch kernels, NEXT-2) on this "
                    "many right-hand sides; fp32 / half only; compare with --opt kernels=v3")
    ap.add_argument("--repeat", type=int, default=1, help="time every (op, precision) this many times in a row")
    ap.add_argument("--sleep", type=float, default=0.0, help="idle seconds before each timing (burst against sustained: the "
                    "kernels run into the board's power cap when launched back to back)")
    args = ap.parse_args()
    build.build()
    cfg = inputs.CONFIGS[args.workload]
    L, L5 = cfg["L"], cfg["L5"]
    recon = int(args.reconstruct or cfg["reconstruct"])
    m = binding.Mdwf(L, L5, cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"])
    m.set_option("reconstruct", recon)
    for kv in args.opt:
        m.set_option(*kv.split("=", 1))
    m.load_gauge(inputs.gauge_field(L, cfg["eps"], cfg["seed"], device="cuda"))
    torch.cuda.empty_cache()
    h = L[0] * L[1] * L[2] * L[3] // 2 * L5
    if args.fma_rates:
        r = m.fma_rates()
        print(json.dumps({"ffma_tfma_per_s": r[0], "ffma2_tfma_per_s": r[1], "ffma_tflops": 2 * r[0], "ffma2_tflops": 2 * r[1]}), flush=True)
    if args.l2_rates:
        r = m.l2_rates()
        print(json.dumps({"l2_ldg_GBs": r[0], "l2_bulk_GBs": r[1], "dram_ldg_GBs": r[2], "dram_bulk_GBs": r[3]}), flush=True)
    F = m.flops_per_site()
    for prec in args.prec.split(","):
        rb, extra = {"fp64": (8, 0), "fp32": (4, 0), "half": (2, 4)}[prec]
        b_site = 5 * (24 * rb + extra) + 2 * 8 * recon * rb / L5
        for op in (int(o) for o in args.ops.split(",") for _ in range(args.repeat)):
            time.sleep(args.sleep)
            r = m.time_op(op, prec, reps=args.reps, warmup=args.warmup)
            r.update(op=("Mpc", "Mpcdag")[op], prec=prec, workload=cfg["name"], reconstruct=recon,
                     tflops=F * h / (r["ms"] * 1e-3) / 1e12, GBs_model=b_site * h / (r["ms"] * 1e-3) / 1e9)
            print(json.dumps(r), flush=True)
            if args.batch > 0 and prec != "fp64":
                rb_ = m.time_op_batch(op, prec, args.batch, reps=max(1, args.reps // 2), warmup=min(args.warmup, 2))
                rb_.update(op=("Mpc", "Mpcdag")[op] + "_batch", prec=prec, nrhs=args.batch, ms_per_rhs=rb_["ms"] / args.batch,
                           single_ms=r["ms"], workload=cfg["name"])
                print(json.dumps(rb_), flush=True)
    m.close()


if __name__ == "__main__":
    main()

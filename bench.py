#!/usr/bin/env python
"""bench.py -- the measurement contract.

A "step" is one pass of the whole hot path: one mdwf_solve (Schur preparation, mixed-precision CG on
Mpc^+ Mpc with reliable updates to tol 1e-10, reconstruction, fp64 true residual) of the headline workload
BASELINE.json quotes its metric on: configs[3] = 32^3 x 96, L5 = 12, double/single/half ladder, 12-real links,
synthetic exp(i 0.1 H) links, Gaussian source.  `value` is the sustained operator TFLOP/s over the step
(the paper's Table VI quantity) at the fixed count 2880 + 48 L5 flop per odd 5D site per
Mpc / Mpc^+ application; the Dslash (Mpc) GB/s and TFLOP/s per precision and the solve seconds are in
"mpc" and "solve".  Multi-GPU = replicas only: every rank solves its own right-hand side, no collective on
the data path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload 0..4]
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "mdwf_eo_dslash_sustained_tflops_in_mixed_precision_cg_solve"
UNIT = "TFLOP/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for ln in self.f.read().splitlines():
            c = [v.strip() for v in ln.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(cfg, U_host, b_host, n_tslices, steps=1, warmup=0):
    """The CPU oracle, as it stands, on a bounded sample of the workload: Mpc then Mpc^+ (the operator work
    of one CG iteration) evaluated on the odd sites of the first n_tslices time slices of the lattice."""
    import numpy as np
    from oracle import mdwf_oracle as mo
    L, L5 = cfg["L"], cfg["L5"]
    orc = mo.MdwfOracle(L, L5, cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"], U_host)
    Lx, Ly, Lz, Lt = L
    sites = orc.sites_odd[orc.sites_odd < Lx * Ly * Lz * n_tslices]
    v = orc.parity_part(b_host, 1) if b_host.shape == orc.shape else b_host
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        orc.Mpc(v, sites)
        orc.Mpcdag(v, sites)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    flops = 2.0 * mo.flops_per_site(L5) * len(sites) * L5
    sec = sum(times) / len(times)
    return {"value": flops / sec / 1e12, "unit": UNIT, "cores": mo.num_threads(), "kind": "oracle",
            "sample": "Mpc + Mpc^dagger (operator work of one CG iteration) on the odd sites of %d of %d time "
                      "slices of %s (%d 5D sites), %.2f s per pass, halo sites recomputed"
                      % (n_tslices, Lt, cfg["name"], len(sites) * L5, sec),
            "seconds_per_pass": sec}


def run_reference(args, rank, world):
    """--impl reference: the oracle timed on the host cores (rank 0 only), same config / metric / unit."""
    if rank != 0:
        return
    import torch
    from paper_1701_07559_b200 import inputs
    cfg = inputs.CONFIGS[args.workload]
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    U = inputs.gauge_field(cfg["L"], cfg["eps"], cfg["seed"], device=dev).cpu().numpy()
    b = inputs.gaussian_source(cfg["L"], cfg["L5"], cfg["seed"], device=dev).cpu().numpy()
    nts = min(cfg["L"][3], args.ref_tslices)
    r = oracle_sample(cfg, U, b, nts, steps=args.steps, warmup=args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["seconds_per_pass"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args),
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(cfg, args):
    return {"workload": "BASELINE.json configs[%d]: %s, M5=%g b5=%g c5=%g m_f=%g, links exp(i %g H) seed %d, "
                        "%s, ladder %s, reconstruct %d, tol 1e-10%s"
                        % (args.workload, cfg["name"], cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"], cfg["eps"],
                           cfg["seed"], "point source at the origin x 12 spin-colour columns per step" if cfg["source"] == "point12"
                           else "Gaussian source", cfg["ladder"], cfg["reconstruct"],
                           "".join(", " + kv for kv in getattr(args, "opt", []))),
            "parallelism": "replicas only: one right-hand side per GPU, no data-path collective",
            "l2": "every vector of the step (>= 0.9 GB) is larger than the 126 MB L2; no explicit flush"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", type=int, default=3, help="index into BASELINE.json configs (default 3 = 32^3x96xL5=12)")
    ap.add_argument("--ref-tslices", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--op-reps", type=int, default=20)
    ap.add_argument("--opt", action="append", default=[], help="extra mdwf_set_option key=value (e.g. matpc=sym, kernels=v3)")
    ap.add_argument("--oracle-solve", action="store_true",
                    help="also run the FULL oracle CG solve of this workload on the host cores and report its iterations and seconds "
                         "beside the GPU's (feasible for workloads 0 and 1)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1701_07559_b200 import binding, build, inputs, replicas
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = inputs.CONFIGS[args.workload]
    L, L5 = cfg["L"], cfg["L5"]
    Vh = L[0] * L[1] * L[2] * L[3] // 2
    h = Vh * L5
    hbm_peak, peak_src = measured_peaks()

    # ---- inputs: same gauge field on every rank, one right-hand side per rank ---------------------------
    U = inputs.gauge_field(L, cfg["eps"], cfg["seed"], device="cuda")
    if cfg["source"] == "point12":      # configs[2]: the 12 spin-colour columns of a point source at the origin; a step solves all of them
        srcs = [inputs.point_source(L, L5, sp, col, device="cuda") for sp in range(4) for col in range(3)]
    else:
        srcs = [inputs.gaussian_source(L, L5, replicas.source_seed(cfg["seed"], rank), device="cuda")]
    src = srcs[0]
    m = binding.Mdwf(L, L5, cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"])
    m.set_option("reconstruct", cfg["reconstruct"])
    m.set_option("ladder", cfg["ladder"])
    for kv in args.opt:
        m.set_option(*kv.split("=", 1))
    m.load_gauge(U)
    # the library keeps its own copies of the links; the canonical field goes back to the host (configs[4] needs the memory)
    want_cpu = rank == 0 and world == 1 and not args.no_cpu_baseline
    U_host = U.cpu().numpy() if want_cpu else None
    del U
    torch.cuda.empty_cache()
    F = m.flops_per_site()
    torch.cuda.empty_cache()          # hand the generators' temporaries back: the library allocates with cudaMalloc
    sol = torch.empty_like(src)
    tol, maxiter = 1e-10, 100000

    def one_solve(host=False, ss=None, x=None):
        """one step: every right-hand side of the workload (1, or the 12 columns of configs[2])"""
        ss = srcs if ss is None else ss
        x = sol if x is None else x
        its, trs, na, sec = [], [], 0.0, 0.0
        for s in ss:
            rc, it, tr = binding.mdwf_solve(m.h, s.data_ptr(), x.data_ptr(), tol, maxiter, host=host)
            if rc != 0 or not (tr <= tol * 1.001):
                raise SystemExit("solve failed: rc=%d true residual %.3e" % (rc, tr))
            its.append(it); trs.append(tr); na += m.stat("op_applications"); sec += m.stat("solve_seconds")
        return max(its), max(trs), na, sec

    # ---- per-kernel Dslash numbers: every kernel timed ALONE, before the solves heat the device into its power cap, because the
    #      roofline they are compared with (MEASURED_PEAKS.json hbm_gbs) is the burst figure of a copy kernel timed alone ----
    gl = {18: {"fp64": 8, "fp32": 4, "half": 2}, 12: {"fp64": 8, "fp32": 4, "half": 2}}
    recon = int(cfg["reconstruct"])
    mpc = {}
    for prec, rb, extra in (("fp32", 4, 0), ("half", 2, 4), ("fp64", 8, 0)):
        # two-pass algorithmic bytes per odd 5D site: K1 reads psi, writes t; K2 reads t, psi,
        # writes out (5 spinor streams) + 2 hops x 8 links x recon reals / L5 (+ one fp32 scale per 16-bit spinor)
        b_site = 5 * (24 * rb + extra) + 2 * 8 * recon * rb / L5
        m.set_option("release_workspace", "1")
        for op, name in ((binding.OP_MPC, "Mpc"), (binding.OP_MPCDAG, "Mpcdag")):
            r = m.time_op(op, prec, reps=args.op_reps, warmup=3)
            # The same pair the way the peak was measured (MEASURED_PEAKS.json: best of 10, a burst): 3 launches after 0.3 s
            # of idle, best of 3 such bursts.  Back to back, these kernels pull the board to its 1000 W power cap within
            # ~100 ms and the SM clock drops (fp32 tile sweep: 1965 -> ~1550 MHz); "ms" above is that
            # sustained mean and the one every other number of this line is derived from.
            burst = []
            for _ in range(3):
                time.sleep(0.3)
                burst.append(m.time_op(op, prec, reps=3, warmup=1)["ms"])
            mpc["%s_%s" % (name, prec)] = {
                "ms": r["ms"], "ms_k1": r["ms_k1"], "ms_k2": r["ms_k2"],
                "tflops": F * h / (r["ms"] * 1e-3) / 1e12,
                "GBs_model": b_site * h / (r["ms"] * 1e-3) / 1e9,
                "frac_hbm": b_site * h / (r["ms"] * 1e-3) / 1e9 / hbm_peak,
                "ms_burst": min(burst), "frac_hbm_burst": b_site * h / (min(burst) * 1e-3) / 1e9 / hbm_peak,
                "bytes_per_site_model": b_site}
    m.set_option("release_workspace", "1")     # the timing vectors make room for the solver's (configs[4]: 157 GB in use)
    torch.cuda.empty_cache()

    # ---- device-resident steps -----------------------------------------------------------------------------
    for _ in range(args.warmup):
        one_solve()
    m.set_option("time_hops", "1")             # two event records around each hop launch of the timed solves (3440 per solve)
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    l0 = m.stat("launches")
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    apps = 0
    for _ in range(args.steps):
        it, tr, na, _ = one_solve()
        apps += na
    ev1.record()
    barrier()
    clocks = sampler.stop()
    launches = m.stat("launches") - l0
    ms_total = ev0.elapsed_time(ev1)
    apps_all, ms_total = replicas.aggregate(apps, ms_total, device="cuda")     # sum of work, max of device time
    value = apps_all * F * h / (ms_total * 1e-3) / 1e12
    iters, true_res, n_upd = it, tr, m.stat("reliable_updates")
    # average duration of the four hop kernels of a CG iteration INSIDE the last timed solve (CUDA events on the library's stream)
    in_solve = {k: (m.stat("hop_ms_" + k), int(m.stat("hop_n_" + k))) for k in ("k1", "k2", "k1dag", "k2dag")}
    m.set_option("time_hops", "0")

    # ---- end to end: host buffers, H2D of the source and D2H of the solution inside the timed region ----------
    srcs_h = [x.cpu().pin_memory() for x in srcs]
    src_h = srcs_h[0]
    sol_h = torch.empty_like(src_h).pin_memory()
    n_rhs = len(srcs)
    del srcs, src, sol                 # the host arm stages through the library's own device buffers (configs[4]: 2 x 24.5 GB)
    torch.cuda.empty_cache()
    one_solve(True, srcs_h, sol_h)
    barrier()
    t0 = time.perf_counter()
    apps_e = 0
    for _ in range(args.steps):
        apps_e += one_solve(True, srcs_h, sol_h)[2]
    barrier()
    e2e_s = time.perf_counter() - t0
    apps_e_all, e2e_s_max = replicas.aggregate(apps_e, e2e_s, device="cuda")
    e2e_value = apps_e_all * F * h / e2e_s_max / 1e12
    nbytes = src_h.numel() * 16 * n_rhs

    # ---- the roofline of the dominant kernel (per-kernel timings: taken before the solves, see above) ------------------
    recon = int(cfg["reconstruct"])
    sloppy = {"d": "fp64", "ds": "fp32", "dh": "half", "dsh": "half"}[cfg["ladder"]]
    rb, extra = {"fp64": (8, 0), "fp32": (4, 0), "half": (2, 4)}[sloppy]
    # the four hop kernels of one CG iteration in the sloppy precision; the roofline object describes the slowest
    b1 = (2 * (24 * rb + extra) + 8 * recon * rb / L5) * h      # K1 / K1+: read one vector, write one, 8 links / L5
    b2 = (3 * (24 * rb + extra) + 8 * recon * rb / L5) * h      # K2 / K2+: read two vectors, write one
    fam = "hop_kernel" if sloppy == "fp64" else "hop3_kernel"
    tiles = (L[1] * (L[0] // 2) // 32) * (L[2] // 2) * (L[3] // 2) if (L[0] // 2) in (2, 4, 8, 16) and (L[1] * (L[0] // 2)) % 32 == 0 else 0
    swept = L5 in (8, 12) and tiles >= 8 * 148            # the library's rule for the tile-sweep kernels (hop5 / hop6 launchers)
    pname = {"fp64": "PD", "fp32": "PS", "half": "PH"}[sloppy]
    k1b = sloppy == "half"                                      # 16-bit CG: K1 reads the B p stream, no B on load

    def kernel(dag, pre, post, own):
        # the kernel the library launches for this (precision, variant): mdwf_launch_hop in mdwf_api.cu
        if sloppy == "fp32" and swept and pre == 0:
            return "hop5_kernel<PS,%d,0,%d,%d,%d>" % (dag, post, own, L5)
        if sloppy == "half" and swept and pre == 0 and post != 2:
            return "hop6_kernel<%d,%d,%d,%d>" % (dag, post, own, L5)      # two sweep sets, 16-bit storage; K2^+ stays on hop3
        return "%s<%s,%d,%d,%d,%d,%d%s>" % (fam, pname, dag, pre, post, own, L5, ",3" if fam == "hop_kernel" or post == 1 else "")

    mp, md = mpc["Mpc_%s" % sloppy], mpc["Mpcdag_%s" % sloppy]
    cands = [
        ("%s (K1 of Mpc: t_e = B A^-1 H_eo %s)" % (kernel(0, 0 if k1b else 1, 1, 0),
                                                  "(B psi)_o, B psi streamed by the CG update" if k1b else "B psi_o"),
         mp["ms_k1"], b1, 1320 + (0 if k1b else 72) + 72 + 48 * L5 - 24, "k1"),
        ("%s (K2 of Mpc: A psi_o - 1/4 H_oe t_e)" % kernel(0, 0, 0, 2), mp["ms_k2"], b2, 1320 + 72 + 48, "k2"),
        ("%s (K1 of Mpc^dagger: u_e = A^-+ B^+ H'_eo psi_o)" % kernel(1, 0, 1, 0), md["ms_k1"], b1,
         1320 + 72 + 48 * L5 - 24, "k1"),
        ("%s (K2 of Mpc^dagger: A^+ psi_o - 1/4 B^+ H'_oe u_e)" % kernel(1, 0, 2, 3), md["ms_k2"], b2,
         1320 + 72 + 72 + 48, "k2"),
    ]
    # the dominant kernel and its duration: the average launch duration inside the timed solve; the same
    # kernels timed alone, back to back, before the solves are kept beside it
    alone = {c[0].split(" ")[0]: c[1] for c in cands}
    tags = ("k1", "k2", "k1dag", "k2dag")
    if all(in_solve[t][1] > 0 for t in tags):
        cands = [(c[0], in_solve[t][0], c[2], c[3], c[4]) for c, t in zip(cands, tags)]
    kname, k_ms, k_bytes, k_flops_site, k_key = max(cands, key=lambda c: c[1])
    roofline = {"kernel": kname,
                "bound": "hbm", "achieved": k_bytes / (k_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "peak_source": peak_src, "traffic": None,
                "algorithmic_bytes_per_launch": k_bytes, "ms_per_launch": k_ms,
                "ms_per_launch_is": "average over the %d launches of this kernel inside the last timed solve (CUDA events on the "
                                    "library's stream, option time_hops)" % in_solve[tags[[c[0] for c in cands].index(kname)]][1],
                "all_hop_kernels_ms": {c[0].split(" ")[0]: c[1] for c in cands},
                "all_hop_kernels_ms_timed_alone": alone}
    roofline["frac"] = roofline["achieved"] / roofline["peak"]
    tf = os.path.join(ROOT, "profiles", "r02_traffic.csv")   # dram bytes per launch from the committed ncu capture
    if os.path.exists(tf):
        for ln in open(tf).read().splitlines()[1:]:
            k, _, v = ln.partition(",")
            if k.strip() == "%s_%s" % (k_key, sloppy):
                roofline["traffic"] = float(v)

    ffma, ffma2 = m.fma_rates()
    # counted flops of that kernel
    alu = {"achieved": k_flops_site * h / (k_ms * 1e-3) / 1e12, "peak": 2 * ffma2, "unit": "TFLOP/s",
           "peak_source": "measured live: packed FFMA2 stream on all SMs (mdwf_fma_rates); scalar FFMA gives %.1f" % (2 * ffma)}
    alu["frac"] = alu["achieved"] / alu["peak"]
    # which ceiling binds this kernel: the larger of its two ideal times
    t_hbm = k_bytes / (hbm_peak * 1e9)
    t_alu = k_flops_site * h / (alu["peak"] * 1e12)
    if t_alu > t_hbm:
        hbm_view = {k: roofline[k] for k in ("achieved", "peak", "unit", "frac", "peak_source")}
        roofline.update({"bound": "alu", "achieved": alu["achieved"], "peak": alu["peak"], "unit": alu["unit"],
                         "frac": alu["frac"], "peak_source": alu["peak_source"], "hbm": hbm_view})
    else:
        roofline["alu"] = alu
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp64": "f64", "fp32": "f32", "half": "i16 storage / f32 arithmetic"}[sloppy],
            "data": "synthetic", "config": workload_config(cfg, args), "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                    "seconds_per_step": e2e_s_max / args.steps},
            "gpu_launches": int(launches),
            "solve": {"seconds": ms_total * 1e-3 / args.steps, "iterations": int(iters), "reliable_updates": int(n_upd),
                      "true_residual": true_res, "op_applications_per_solve": apps / args.steps,
                      "flops_per_site": F, "sites": h},
            "mpc": mpc, "roofline": roofline}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nts = min(L[3], args.ref_tslices)
        r = oracle_sample(cfg, U_host, src_h.numpy(), nts)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        # the oracle's time for the operator work of one CG iteration on the whole lattice, EXTRAPOLATED from the sample,
        # and for the whole solve at the GPU's iteration count (BLAS-1 not included): context, labelled as extrapolated
        per_it = r["seconds_per_pass"] * L[3] / nts
        line["cpu_baseline"]["extrapolated"] = {
            "oracle_seconds_per_cg_iteration": per_it,
            "oracle_solve_seconds_at_gpu_iterations": per_it * int(iters) * n_rhs,
            "note": "sample seconds x (Lt / sampled time slices) x GPU iteration count x right-hand sides; not measured"}
        if args.oracle_solve:
            from oracle import mdwf_oracle as mo
            orc = mo.MdwfOracle(L, L5, cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"], U_host)
            t0 = time.perf_counter()
            x_ref, it_ref, res_ref = orc.solve(src_h.numpy(), tol=1e-10)
            line["cpu_baseline"]["oracle_full_solve"] = {"iterations": int(it_ref), "seconds": time.perf_counter() - t0,
                                                         "true_residual": res_ref, "gpu_iterations": int(iters)}
    if rank == 0:
        print(json.dumps(line), flush=True)
    m.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- one JSON line for the MDWF hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A step = one pass of the whole solve path over one batch of synthetic input: for every right-hand side of
the configuration, even-odd source preparation, batched mixed-precision CG on the normal equations (16-bit
inner storage / fp32 arithmetic, fp64 reliable updates), reconstruction of the other parity and unpacking,
all through the C-ABI call mdwf_solve.  `value` is the metric's "mixed-prec CG seconds per RHS"; the Dslash
GB/s and GFLOP/s of the same run are in `dslash` and `roofline` (the hop kernel inside the timed solves,
timed per launch with CUDA events on the launching stream).
N > 1: the path does not shard ("replicas only"): every rank solves its own replica.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "MDWF Dslash GB/s & GFLOP/s vs HBM roofline; mixed-prec CG seconds per RHS"


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def run(self):
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 6:
                    self.rows.append(f)
            except Exception:
                pass
            self._halt.wait(0.2)

    def finish(self):
        self._halt.set()
        self.join(timeout=6)
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": int(self.rows[0][1]) if self.rows and self.rows[0][1].isdigit() else None,
                "samples": len(self.rows), "reasons": reasons}


def max_over_ranks(ms, world, device=None):
    """Multi-GPU timing rule: every rank times on its own device, the job's time is the MAX over ranks.
    (The path does not shard -- "replicas only" -- so this reduce is the only collective; gloo on CPU in tests.)"""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(sec_per_rhs_per_replica, world):
    """N independent replicas finish N*nrhs solves in the time one replica needs for nrhs: whole-job s/RHS."""
    return sec_per_rhs_per_replica / world


def oracle_baseline(cfg, budget_s=20.0):
    """The CPU oracle as it stands (oracle.solve_eo: its own even-odd CG, fp64, OpenMP over the host cores),
    timed on a bounded sample of the workload: the same operator parameters and link recipe on a small
    sub-lattice, one Gaussian rhs, same tolerance.  Returns (dict, seconds per (5D site x CG iteration))."""
    import numpy as np
    import oracle
    import synth
    dims = tuple(min(d, s) for d, s in zip(cfg.dims, (8, 8, 8, 16)))
    p = oracle.Params(dims=dims, Ls=cfg.Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=cfg.mf, bc=cfg.bc)
    U = synth.gauge_field(dims, cfg.eps, synth.seed_for(cfg.index, 1)).numpy()
    b = synth.gaussian_spinor(dims, cfg.Ls, 1, synth.seed_for(cfg.index, 2)).numpy()
    oracle.schur(p, U, b, 0, False, True)          # warm-up (page in, OpenMP team)
    t0 = time.time()
    x, its, _ = oracle.solve_eo(p, U, b, parity=0, symmetric=True, tol=cfg.tol, max_iter=100000)
    dt = time.time() - t0
    tr = float(oracle.true_residual(p, U, x, b).max())
    n5 = int(np.prod(dims)) * cfg.Ls
    per_site_iter = dt / (n5 * max(1, its[0]))
    d = {"value": dt, "unit": "s/RHS", "cores": oracle.num_threads(), "kind": "oracle",
         "sample": "oracle.solve_eo (fp64 even-odd CG, symmetric) on a %s x Ls=%d sub-lattice of the workload "
                   "(same M5,b5,c5,mf, link recipe and tol %.0e), 1 Gaussian rhs: %d iterations in %.2f s, "
                   "true residual %.2e" % ("x".join(map(str, dims)), cfg.Ls, cfg.tol, its[0], dt, tr),
         "s_per_5Dsite_iteration": per_site_iter, "iterations": its[0]}
    return d, per_site_iter


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    import synth
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = synth.CONFIGS[args.config]
    vals = []
    base = None
    for i in range(args.warmup + args.steps):
        base, _ = oracle_baseline(cfg)
        if i >= args.warmup:
            vals.append(base["value"])
    v = sum(vals) / len(vals)
    base["value"] = v
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "s/RHS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": v * 1e3, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "note": "each step is the bounded sample described in cpu_baseline.sample"},
            "cpu_baseline": base,
            "e2e": {"value": v, "unit": "s/RHS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    import synth
    import paper_1810_01609_b200 as mdwf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = synth.CONFIGS[args.config]
    nrhs = args.nrhs or cfg.nrhs
    inner, recon = args.inner, args.recon
    hbm_peak, peak_src = peaks()

    # ---- inputs (untimed): links of the config's recipe, Gaussian 5D right-hand sides --------------------
    ctx = mdwf.Context(cfg.dims, cfg.Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc, device=local)
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(cfg.index, 1), device=dev)
    ctx.mdwf_load_gauge(U, 64, 18)
    ctx.mdwf_load_gauge(U, inner, recon)
    del U
    torch.cuda.empty_cache()
    b = synth.gaussian_spinor_device(cfg.dims, cfg.Ls, nrhs, synth.seed_for(cfg.index, 2) + 7 * rank, device=dev)
    x = torch.empty_like(b)
    kw = dict(tol=cfg.tol, inner_prec=inner, recon=recon, symmetric=not args.asym, batch=args.batch, check_every=args.check_every, delta=args.delta)

    def step():
        _, res = ctx.mdwf_solve(b, out=x, **kw)
        if res.status != 0:
            raise RuntimeError("solve did not converge: %r" % (res,))
        return res

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        res = step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = ctx.mdwf_launch_count()
    ctx.mdwf_profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        res = step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.finish()
    launches = ctx.mdwf_launch_count() - l0
    prof = {c: ctx.mdwf_profile_read(c) for c in (0, 1, 2)}
    ctx.mdwf_profile(False)
    ms_total = max_over_ranks(ms_total, world, dev)
    ms_step = ms_total / args.steps
    sec_per_rhs = ms_step * 1e-3 / nrhs          # per replica; N replicas solve N*nrhs in the same time

    # ---- roofline of the dominant kernel: the hop (Dslash stencil) launches inside the timed solves ------
    cls = {16: 0, 32: 1, 64: 2}[inner]
    pms, pby, pfl, pn = prof[cls]
    roof = {"bound": "hbm", "kernel": "hop_kernel<%s,%d> (inner-precision Dslash stencil incl. fused Ls epilogue)"
            % ({16: "__half", 32: "float", 64: "double"}[inner], recon),
            "achieved": pby / pms / 1e6 if pms > 0 else None, "peak": hbm_peak, "unit": "GB/s",
            "frac": (pby / pms / 1e6) / hbm_peak if pms > 0 else None, "traffic": None, "peak_source": peak_src,
            "launches": pn, "avg_launch_ms": pms / pn if pn else None, "gflops": pfl / pms / 1e6 if pms > 0 else None,
            "share_of_step": pms / (ms_total if world == 1 else ms_step * args.steps)}
    # the 16-bit kernel is co-bound by FP32 issue: report it against the plain-FP32 FMA peak
    # 148 SMs x 128 lanes x 2 flop x max SM clock, with the 1320 flop/site convention
    fp32_peak = 148 * 128 * 2 * (clocks.get("sm_max_mhz") or 1965) * 1e-6
    if roof["gflops"]:
        roof["co_bound"] = {"bound": "alu", "achieved": roof["gflops"] * 1e-3, "peak": fp32_peak, "unit": "TFLOP/s",
                            "frac": roof["gflops"] * 1e-3 / fp32_peak,
                            "note": "convention flops (1320 per 5D site) / FP32 FMA peak; ncu: issue slots 68-70 % busy"}
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic_r1.csv")) as f:
            rows = {r["key"]: r for r in csv.DictReader(f)}
        tr = rows.get("%s|inner%d|recon%d" % (cfg.name, inner, recon))
        if tr:
            roof["traffic"] = float(tr["dram_bytes_per_launch"])
            roof["traffic_source"] = tr["source"]
            roof["algorithmic_bytes_per_launch"] = pby / pn if pn else None
    except Exception:
        pass
    h64 = prof[2]
    dsl = {"inner_hop_GBps": roof["achieved"], "inner_hop_GFLOPs": roof["gflops"],
           "fp64_hop_GBps": h64[1] / h64[0] / 1e6 if h64[0] > 0 else None,
           "fp64_hop_GFLOPs": h64[2] / h64[0] / 1e6 if h64[0] > 0 else None, "fp64_hop_launches": h64[3]}
    return dict(ctx=ctx, cfg=cfg, nrhs=nrhs, b=b, x=x, kw=kw, res=res, ms_step=ms_step, sec_per_rhs=sec_per_rhs,
                clocks=clocks, launches=launches, roof=roof, dsl=dsl, rank=rank, world=world, dev=dev)


def run_e2e(st, args):
    """Same metric through the C-ABI call with HOST buffers (mdwf_solve_host): every step copies the step's
    right-hand sides host->device and the solutions device->host inside the timed region."""
    import torch
    import torch.distributed as dist
    ctx, b, x, nrhs = st["ctx"], st["b"], st["x"], st["nrhs"]
    if st["world"] > 1 and nrhs > 1:
        # N ranks share one host: bound the pinned staging memory per rank (2 x 13.6 GB instead of 2 x 54 GB);
        # seconds per rhs is the same metric, the solver handles one rhs at a time at this size anyway
        nrhs = 1
        b = b[:1].contiguous()
    nbytes = b.numel() * b.element_size()
    try:
        bh = torch.empty(b.shape, dtype=b.dtype, pin_memory=True)
        xh = torch.empty(b.shape, dtype=b.dtype, pin_memory=True)
        pinned = True
    except Exception:
        bh = torch.empty(b.shape, dtype=b.dtype)
        xh = torch.empty(b.shape, dtype=b.dtype)
        pinned = False
    bh.copy_(b)
    torch.cuda.synchronize()
    st["b"] = st["x"] = None
    del b, x
    torch.cuda.empty_cache()
    kw = dict(st["kw"])

    def step():
        _, res = ctx.mdwf_solve_host(bh, xh, **kw)
        if res.status != 0:
            raise RuntimeError("host-buffer solve did not converge: %r" % (res,))
        return res

    for _ in range(args.e2e_warmup):
        step()
    if st["world"] > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.e2e_steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, st["world"], st["dev"])
    return {"value": ms * 1e-3 / args.e2e_steps / nrhs, "unit": "s/RHS", "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "steps": args.e2e_steps, "warmup": args.e2e_warmup, "pinned_host": pinned,
            "api": "mdwf_solve_host", "nrhs": nrhs}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json configs index (1-based); 5 = 48^3x64 Ls=10")
    ap.add_argument("--nrhs", type=int, default=0)
    ap.add_argument("--inner", type=int, default=16)
    ap.add_argument("--recon", type=int, default=12)
    ap.add_argument("--batch", type=int, default=0)
    ap.add_argument("--check-every", type=int, default=1)
    ap.add_argument("--asym", action="store_true", help="solve with Dhat instead of Mhat = M5^-1 Dhat")
    ap.add_argument("--delta", type=float, default=0.0, help="reliable-update threshold (0 = library default)")
    ap.add_argument("--e2e-steps", type=int, default=1)
    ap.add_argument("--e2e-warmup", type=int, default=1)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    st = run_ours(args)
    cfg, nrhs, res, world = st["cfg"], st["nrhs"], st["res"], st["world"]
    e2e = None if args.no_e2e else run_e2e(st, args)
    if st["rank"] != 0:
        return
    line = {"metric": METRIC, "value": aggregate(st["sec_per_rhs"], world), "unit": "s/RHS", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": st["ms_step"], "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": {16: "f32", 32: "f32", 64: "f64"}[args.inner],
            "data": "synthetic",
            "config": {"workload": cfg.name, "lattice": list(cfg.dims), "Ls": cfg.Ls, "nrhs_per_gpu": nrhs, "tol": cfg.tol,
                       "mf": cfg.mf, "inner_prec": args.inner, "recon": args.recon,
                       "arithmetic": {16: "inner CG: fp16 storage (+fp32 scale per site), fp32 arithmetic, fp64 reductions; outer: fp64 reliable updates",
                                      32: "inner CG: fp32 storage and arithmetic, fp64 reductions; outer: fp64 reliable updates",
                                      64: "fp64 throughout"}[args.inner], "links": "reunit(exp(i*%.3f*H))" % cfg.eps,
                       "rhs": "Gaussian complex 5D, device-drawn, seeded", "parallelism": "replicas only",
                       "l2": "inputs larger than L2 (half-lattice 16-bit spinor %.0f MB per rhs)" % (cfg.V4 / 2 * cfg.Ls * 52 / 1e6)},
            "cg": {"seconds_per_rhs_per_replica": st["sec_per_rhs"], "iters": res.iters, "reliable_updates": res.reliable_updates,
                   "true_resid": res.true_resid, "seconds_inner_last_step": res.seconds_inner, "seconds_last_step": res.seconds},
            "dslash": st["dsl"], "roofline": st["roof"], "gpu_launches": st["launches"], "clocks": st["clocks"]}
    if e2e is not None:
        e2e["value"] = aggregate(e2e["value"], world)
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        base, per = oracle_baseline(cfg)
        it = max(res.iters) if res.iters else 0
        base["extrapolated_s_per_rhs_on_workload"] = per * cfg.V4 * cfg.Ls * max(1, base["iterations"])
        base["note"] = "value is the measured sample; the extrapolation multiplies the measured s/(5D site x iteration) by the workload's 5D volume and the sample's iteration count (GPU needed %d inner iterations)" % it
        line["cpu_baseline"] = base
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()

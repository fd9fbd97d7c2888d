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


def sample_dims(cfg):
    """the bounded sub-lattice of the workload that the CPU oracle is timed on"""
    return tuple(min(d, s) for d, s in zip(cfg.dims, (8, 8, 8, 16)))


def oracle_baseline(cfg, workload_iters=None):
    """The CPU oracle as it stands (fp64, OpenMP over the host cores), timed on a bounded sample of the workload: the
    same operator parameters and link recipe on a small sub-lattice.  (i) hop and Mhat applications (median of 3;
    sites/s, GB/s and GFLOP/s under the same byte / flop convention as the GPU lines); (ii) its own
    even-odd CG (oracle.solve_eo) on one Gaussian rhs at the workload's tolerance.
    Returns (dict, seconds per (5D site x CG iteration))."""
    import numpy as np
    import oracle
    import synth
    dims = sample_dims(cfg)
    p = oracle.Params(dims=dims, Ls=cfg.Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=cfg.mf, bc=cfg.bc)
    U = synth.gauge_field(dims, cfg.eps, synth.seed_for(cfg.index, 1)).numpy()
    b = synth.gaussian_spinor(dims, cfg.Ls, 1, synth.seed_for(cfg.index, 2)).numpy()
    oracle.schur(p, U, b, 0, False, True)          # warm-up (page in, OpenMP team)
    n5h = int(np.prod(dims)) // 2 * cfg.Ls         # 5D sites of one parity
    other = oracle.mask(p, b, 1)
    same = oracle.mask(p, b, 0)

    def med3(fn):
        ts = []
        for _ in range(3):
            t0 = time.time()
            fn()
            ts.append(time.time() - t0)
        return sorted(ts)[1]

    t_hop = med3(lambda: oracle.hop(p, U, other, dagger=False, out_parity=0))
    t_mhat = med3(lambda: oracle.schur(p, U, same, 0, False, True))
    # same convention as mdwf_dslash_cost for fp64 / 18 reals: hop 2*192 B + links, 1320 flop; Mhat 5 passes + 2 link passes
    links = 8 * 18 * 8 * (int(np.prod(dims)) // 2)
    hop_bytes, hop_flops = 2 * 192.0 * n5h + links, 1320.0 * n5h
    mh_bytes, mh_flops = 5 * 192.0 * n5h + 2 * links, (2832.0 + 96.0 * cfg.Ls) * n5h
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
         "s_per_5Dsite_iteration": per_site_iter, "iterations": its[0],
         "dslash": {"sample_lattice": list(dims), "hop_ms": t_hop * 1e3, "hop_sites_per_s": n5h / t_hop,
                    "hop_GBps": hop_bytes / t_hop / 1e9, "hop_GFLOPs": hop_flops / t_hop / 1e9,
                    "mhat_ms": t_mhat * 1e3, "mhat_sites_per_s": n5h / t_mhat, "mhat_GBps": mh_bytes / t_mhat / 1e9,
                    "mhat_GFLOPs": mh_flops / t_mhat / 1e9, "convention": "fp64, 18-real links; median of 3"}}
    if workload_iters:
        d["extrapolated_s_per_rhs_on_workload"] = per_site_iter * cfg.V4 * cfg.Ls * workload_iters
        d["note"] = ("value is the measured sample; the extrapolation multiplies the measured s/(5D site x iteration) by the "
                     "workload's 5D volume and the workload's own iteration count (%d)" % workload_iters)
    return d, per_site_iter


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only).  Each step is the bounded sample
    described in cpu_baseline.sample; config.workload names that sub-lattice (it is NOT the GPU arm's workload)."""
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
    sd = sample_dims(cfg)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "s/RHS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": v * 1e3, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "oracle sample %s_Ls%d of %s" % ("x".join(map(str, sd)), cfg.Ls, cfg.name),
                       "of_workload": cfg.name, "sites_ratio_workload_to_sample": cfg.V4 / float(sd[0] * sd[1] * sd[2] * sd[3]),
                       "note": "each step is the bounded sample described in cpu_baseline.sample, not the GPU arm's workload"},
            "cpu_baseline": base,
            "e2e": {"value": v, "unit": "s/RHS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def fill_packed_rhs(fields, cfg, nrhs, seed, dev, scratch):
    """Gaussian complex 5D right-hand sides, drawn by the seeded device generator one (rhs, parity) half-lattice
    column at a time and packed straight into the fp64 half-lattice fields (no canonical full-lattice copy exists)."""
    import torch
    g = torch.Generator(device=dev)
    for par in (0, 1):
        for r in range(nrhs):
            g.manual_seed(int(seed) * 1000 + 2 * r + par)
            torch.view_as_real(scratch).normal_(0.0, 1.0, generator=g)
            fields[par].mdwf_field_pack_rhs(r, scratch)


def dslash_legs(ctx, cfg, nrhs, formats, dev, hbm_peak, iters=10):
    """Dslash-only leg through mdwf_dslash_packed on the bench lattice: plain hop and Mhat per (prec, recon), CUDA events
    around `iters` back-to-back calls; algorithmic bytes / flops from mdwf_dslash_cost."""
    import torch
    import synth
    import paper_1810_01609_b200 as mdwf
    out = []
    Vh = cfg.V4 // 2
    g = torch.Generator(device=dev).manual_seed(synth.seed_for(cfg.index, 3))
    for prec, recon in formats:
        fin, fout = ctx.mdwf_field_create(prec, nrhs), ctx.mdwf_field_create(prec, nrhs)
        src = torch.empty((nrhs, cfg.Ls, Vh, 4, 3), dtype=torch.complex128, device=dev)
        torch.view_as_real(src).normal_(0.0, 1.0, generator=g)
        fin.mdwf_field_pack(src)
        del src
        for name, op in (("hop", mdwf.OP_HOP), ("mhat", mdwf.OP_DHAT_SYM)):
            for _ in range(3):
                ctx.mdwf_dslash_packed(op, fout, fin, 0, False, recon)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(iters):
                ctx.mdwf_dslash_packed(op, fout, fin, 0, False, recon)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / iters
            by, fl = ctx.mdwf_dslash_cost(op, prec, recon, nrhs)
            out.append({"lattice": cfg.name, "nrhs": nrhs, "prec": prec, "recon": recon, "op": name, "ms": ms,
                        "GBps": by / ms / 1e6, "GFLOPs": fl / ms / 1e6, "frac_of_measured_hbm": by / ms / 1e6 / hbm_peak})
        fin.mdwf_field_destroy()
        fout.mdwf_field_destroy()
        torch.cuda.empty_cache()
    return out


def config2_sweep(dev, hbm_peak, rotate=4, iters=20):
    """BASELINE.json configs[1]: 16^3x32, Ls=8 Dslash-only sweep over {fp64, fp32, fp16} x {18, 12, 8 reals}; the lattice
    fits in L2, so `rotate` independent in/out buffer sets are cycled (SURVEY 8(d) config-2 caveat)."""
    import torch
    import synth
    import paper_1810_01609_b200 as mdwf
    cfg = synth.CONFIGS[2]
    ctx = mdwf.Context(cfg.dims, cfg.Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc, device=dev.index or 0)
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(2, 1), device=dev)
    Vh = cfg.V4 // 2
    g = torch.Generator(device=dev).manual_seed(synth.seed_for(2, 2))
    rows = []
    for prec in (64, 32, 16):
        for recon in (18, 12, 8):
            ctx.mdwf_load_gauge(U, prec, recon)
            fin = [ctx.mdwf_field_create(prec, 1) for _ in range(rotate)]
            fout = [ctx.mdwf_field_create(prec, 1) for _ in range(rotate)]
            for f in fin:
                src = torch.empty((1, cfg.Ls, Vh, 4, 3), dtype=torch.complex128, device=dev)
                torch.view_as_real(src).normal_(0.0, 1.0, generator=g)
                f.mdwf_field_pack(src)
            for name, op in (("hop", mdwf.OP_HOP), ("mhat", mdwf.OP_DHAT_SYM)):
                for k in range(3):
                    ctx.mdwf_dslash_packed(op, fout[k % rotate], fin[k % rotate], 0, False, recon)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for k in range(iters):
                    ctx.mdwf_dslash_packed(op, fout[k % rotate], fin[k % rotate], 0, False, recon)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / iters
                by, fl = ctx.mdwf_dslash_cost(op, prec, recon, 1)
                rows.append({"prec": prec, "recon": recon, "op": name, "ms": ms, "GBps": by / ms / 1e6,
                             "GFLOPs": fl / ms / 1e6, "frac_of_measured_hbm": by / ms / 1e6 / hbm_peak})
            for f in fin + fout:
                f.mdwf_field_destroy()
    ctx.mdwf_destroy()
    return {"lattice": cfg.name, "rotate": rotate, "rows": rows}


def run_ours(args):
    import torch
    import torch.distributed as dist
    import synth
    import paper_1810_01609_b200 as mdwf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(1, args.gpus):
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d (launch with torchrun --nproc-per-node %d, or let bench.py "
                         "spawn the ranks by not setting WORLD_SIZE)" % (args.gpus, world, args.gpus))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = synth.CONFIGS[args.config]
    nrhs = args.nrhs or cfg.nrhs
    inner, recon = args.inner, args.recon
    hbm_peak, peak_src = peaks()
    Vh = cfg.V4 // 2

    # ---- inputs (untimed): links of the config's recipe, Gaussian 5D right-hand sides as packed fp64 halves ----
    ctx = mdwf.Context(cfg.dims, cfg.Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc, device=local)
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(cfg.index, 1), device=dev)
    ctx.mdwf_load_gauge(U, 64, 18)
    ctx.mdwf_load_gauge(U, inner, recon)
    del U
    torch.cuda.empty_cache()
    # launch parameters: the library's run-time autotuner, before anything is timed
    tuned = {}
    if not args.no_autotune:
        t0 = time.time()
        ctx.mdwf_autotune(inner, recon, nrhs)
        ctx.mdwf_autotune(64, 18, 1)
        lat = "%dx%dx%dx%d/Ls%d" % (tuple(cfg.dims) + (cfg.Ls,))
        if inner == 16:
            rows = cfg.Ls * max(r for r in (1, 2, 4) if r < 2 * nrhs and r * cfg.Ls <= 48)     # rhs per interleave group
            tuned["hop16 tile (lx, ly, lz, lt, warps)"] = ctx.mdwf_tune_get("hop16/%s/rows%d" % (lat, rows))
        else:
            tuned["hop%d zc" % inner] = ctx.mdwf_tune_get("hop%d/%s/rhs%d" % (inner, lat, nrhs))
        tuned["hop64 zc"] = ctx.mdwf_tune_get("hop64/%s/rhs1" % lat)
        tuned["seconds"] = time.time() - t0
    # the solver workspace comes from PyTorch's allocator (mdwf_set_workspace)
    ws = torch.empty(ctx.mdwf_workspace_bytes(nrhs, inner, packed=True) + (1 << 20), dtype=torch.uint8, device=dev)
    ctx.mdwf_set_workspace(ws)
    psi = [ctx.mdwf_field_create(64, nrhs), ctx.mdwf_field_create(64, nrhs)]
    scratch = torch.empty((1, cfg.Ls, Vh, 4, 3), dtype=torch.complex128, device=dev)
    seed = synth.seed_for(cfg.index, 2) + 7 * rank
    kw = dict(tol=cfg.tol, inner_prec=inner, recon=recon, symmetric=not args.asym, delta=args.delta)

    def step():
        # the solve is in place (b -> psi), so every step first restores the right-hand sides (inside the timed region:
        # ~0.3 % of a config-5 step)
        fill_packed_rhs(psi, cfg, nrhs, seed, dev, scratch)
        res = ctx.mdwf_solve_packed(psi[0], psi[1], **kw)
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
    ms_total = max_over_ranks(ms_total, world, dev)
    ms_step = ms_total / args.steps
    sec_per_rhs = ms_step * 1e-3 / nrhs          # per replica; N replicas solve N*nrhs in the same time

    # ---- roofline of the dominant kernel: the inner-precision hop (Dslash stencil incl. fused epilogue) launches of one
    # more, UNTIMED solve, each timed with CUDA events on the launching stream (the per-launch events would otherwise sit
    # inside the timed region) ----------------------------------------------------------------------------------
    ctx.mdwf_profile(True)
    res_p = step()
    torch.cuda.synchronize()
    prof = {c: ctx.mdwf_profile_read(c) for c in range(8)}
    ctx.mdwf_profile(False)
    cls = {16: 0, 32: 1, 64: 2}[inner]
    pms, pby, pfl, pn = prof[cls]
    kname = ("hop16_kernel (tensor-core fp16 Dslash stencil incl. fused Ls epilogue, mma.sync f16->f32)" if inner == 16 else
             "hop_kernel<%s,%d> (Dslash stencil incl. fused Ls epilogue)" % ("float" if inner == 32 else "double", recon))
    roof = {"bound": "hbm", "kernel": kname,
            "achieved": pby / pms / 1e6 if pms > 0 else None, "peak": hbm_peak, "unit": "GB/s",
            "frac": (pby / pms / 1e6) / hbm_peak if pms > 0 else None, "traffic": None,
            "traffic_note": "not measured in this run; ncu dram bytes per launch of the same kernel are in profiles/ (per capture, with its commit)",
            "peak_source": peak_src, "launches": pn, "avg_launch_ms": pms / pn if pn else None,
            "algorithmic_bytes_per_launch": pby / pn if pn else None, "rhs_in_flight": res.batch,
            "gflops": pfl / pms / 1e6 if pms > 0 else None,
            "share_of_step": pms / (res_p.seconds * 1e3) if res_p.seconds > 0 else None,
            "timing": "per-launch CUDA events on the launching stream, over one extra solve after the timed region"}
    names = {0: "hop fp16 (tensor cores)", 1: "hop fp32", 2: "hop fp64 (reliable updates)", 3: "s-direction kernel", 4: "cg x/r update",
             5: "cg p update (+ A p)", 6: "reduction finish", 7: "axpby / convert"}
    roof["step_breakdown_ms"] = {names[c]: {"ms": prof[c][0], "launches": prof[c][3]} for c in range(8) if prof[c][3]}
    roof["step_breakdown_ms"]["whole solve (4 rhs)" if nrhs == 4 else "whole solve"] = res_p.seconds * 1e3
    h64 = prof[2]
    dsl = {"inner_hop_GBps": roof["achieved"], "inner_hop_GFLOPs": roof["gflops"],
           "fp64_hop_GBps": h64[1] / h64[0] / 1e6 if h64[0] > 0 else None,
           "fp64_hop_GFLOPs": h64[2] / h64[0] / 1e6 if h64[0] > 0 else None, "fp64_hop_launches": h64[3]}
    return dict(tuned=tuned, ctx=ctx, cfg=cfg, nrhs=nrhs, psi=psi, scratch=scratch, ws=ws, kw=kw, res=res, ms_step=ms_step,
                sec_per_rhs=sec_per_rhs, clocks=clocks, launches=launches, roof=roof, dsl=dsl, rank=rank, world=world, dev=dev,
                hbm_peak=hbm_peak)


def run_e2e(st, args):
    """Same metric through the C-ABI call with HOST buffers (mdwf_solve_host): every step copies the step's
    right-hand sides host->device and the solutions device->host inside the timed region (canonical fp64 5D fields;
    the library streams them through two staging chunks into / out of its packed fields, so the same number of
    right-hand sides is in flight as in the device-resident leg)."""
    import torch
    import torch.distributed as dist
    import synth
    ctx, cfg, nrhs, dev = st["ctx"], st["cfg"], st["nrhs"], st["dev"]
    # the packed fields and the torch-owned workspace of the device-resident leg are released first
    for f in st["psi"]:
        f.mdwf_field_destroy()
    ctx.mdwf_set_workspace(None)
    st["psi"] = st["ws"] = st["scratch"] = None
    torch.cuda.empty_cache()
    if st["world"] > 1 and nrhs > 1:
        nrhs = 1          # N ranks share one host: bound the pinned staging memory per rank
    shape = (nrhs, cfg.Ls, cfg.V4, 4, 3)
    try:
        bh = torch.empty(shape, dtype=torch.complex128, pin_memory=True)
        xh = torch.empty(shape, dtype=torch.complex128, pin_memory=True)
        pinned = True
    except Exception:
        bh = torch.empty(shape, dtype=torch.complex128)
        xh = torch.empty(shape, dtype=torch.complex128)
        pinned = False
    one = torch.empty((1,) + shape[1:], dtype=torch.complex128, device=dev)
    for r in range(nrhs):                       # device-drawn (seeded), copied to the host buffer column by column
        synth.gaussian_spinor_device(cfg.dims, cfg.Ls, 1, synth.seed_for(cfg.index, 2) + 7 * st["rank"] + 100 * r, device=dev, out=one)
        bh[r].copy_(one[0])
    del one
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    nbytes = bh.numel() * bh.element_size()
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
        res = step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, st["world"], st["dev"])
    ctx.mdwf_set_workspace(None)          # drop the library's cached workspace: the Dslash legs allocate their own fields
    return {"value": ms * 1e-3 / args.e2e_steps / nrhs, "unit": "s/RHS", "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "steps": args.e2e_steps, "warmup": args.e2e_warmup, "pinned_host": pinned,
            "api": "mdwf_solve_host", "nrhs": nrhs, "rhs_in_flight": res.batch}


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per GPU, torchrun)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


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
    ap.add_argument("--asym", action="store_true", help="solve with Dhat instead of Mhat = M5^-1 Dhat")
    ap.add_argument("--delta", type=float, default=0.0, help="reliable-update threshold (0 = library default)")
    ap.add_argument("--e2e-steps", type=int, default=1)
    ap.add_argument("--e2e-warmup", type=int, default=1)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-autotune", action="store_true", help="keep the library's default launch parameters")
    ap.add_argument("--no-dslash", action="store_true", help="skip the Dslash-only legs (bench lattice and config-2 sweep)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    st = run_ours(args)
    cfg, nrhs, res, world = st["cfg"], st["nrhs"], st["res"], st["world"]
    e2e = None if args.no_e2e else run_e2e(st, args)
    if st["rank"] != 0:
        return
    import torch
    if args.no_e2e:
        for f in st["psi"]:
            f.mdwf_field_destroy()
        st["ctx"].mdwf_set_workspace(None)
        st["psi"] = st["ws"] = st["scratch"] = None
        torch.cuda.empty_cache()
    dsl = st["dsl"]
    if not args.no_dslash and world == 1:
        import synth
        U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(cfg.index, 1), device=st["dev"])
        st["ctx"].mdwf_load_gauge(U, 32, 12)
        del U
        torch.cuda.empty_cache()
        fmts = [(16, args.recon), (32, 12)] if args.inner == 16 else [(args.inner, args.recon)]
        dsl["bench_lattice"] = dslash_legs(st["ctx"], cfg, nrhs, fmts, st["dev"], st["hbm_peak"])
        if nrhs > 1:
            dsl["bench_lattice"] += dslash_legs(st["ctx"], cfg, 1, fmts, st["dev"], st["hbm_peak"])
        dsl["config2_sweep"] = config2_sweep(st["dev"], st["hbm_peak"])
    line = {"metric": METRIC, "value": aggregate(st["sec_per_rhs"], world), "unit": "s/RHS", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": st["ms_step"], "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": {16: "f32", 32: "f32", 64: "f64"}[args.inner],
            "data": "synthetic",
            "config": {"workload": cfg.name, "lattice": list(cfg.dims), "Ls": cfg.Ls, "nrhs_per_gpu": nrhs,
                       "rhs_in_flight": res.batch, "tol": cfg.tol, "mf": cfg.mf, "inner_prec": args.inner, "recon": args.recon,
                       "arithmetic": {16: "inner CG: IEEE fp16 storage (one power-of-two scale per field and rhs), fp16 x fp16 products accumulated in fp32 on the tensor cores, fp32 epilogues, fp64 reductions; outer: fp64 reliable updates",
                                      32: "inner CG: fp32 storage and arithmetic, fp64 reductions; outer: fp64 reliable updates",
                                      64: "fp64 throughout"}[args.inner], "links": "reunit(exp(i*%.3f*H))" % cfg.eps,
                       "rhs": "Gaussian complex 5D, device-drawn, seeded, restored inside every step (in-place packed solve)",
                       "api": "mdwf_solve_packed (device-resident); mdwf_solve_host (e2e)", "parallelism": "replicas only",
                       "l2": "inputs larger than L2 (half-lattice 16-bit spinor %.0f MB per rhs)" % (cfg.V4 / 2 * cfg.Ls * 48 / 1e6)},
            "cg": {"seconds_per_rhs_per_replica": st["sec_per_rhs"], "iters": res.iters, "reliable_updates": res.reliable_updates,
                   "true_resid": res.true_resid, "seconds_inner_last_step": res.seconds_inner, "seconds_last_step": res.seconds,
                   "kernel_launches_last_step": res.kernel_launches},
            "dslash": dsl, "roofline": st["roof"], "gpu_launches": st["launches"], "clocks": st["clocks"],
            "autotune": st["tuned"] or None}
    if e2e is not None:
        e2e["value"] = aggregate(e2e["value"], world)
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        base, _ = oracle_baseline(cfg, workload_iters=max(res.iters) if res.iters else None)
        line["cpu_baseline"] = base
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()

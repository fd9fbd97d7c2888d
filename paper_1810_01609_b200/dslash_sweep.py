"""Dslash throughput sweep (BASELINE.json configs[1]: "Dslash-only throughput sweep in fp64/fp32/fp16
storage with 18-, 12- and 8-real link formats"), through the packed C-ABI calls.

    python -m paper_1810_01609_b200.dslash_sweep --config 2 [--nrhs 1] [--formats 32x12,16x12] [--ops hop,mhat]
                                                  [--iters 20] [--rotate 4] [--zc 0]

Prints one JSON line per (format, op): device time per call (CUDA events around `iters` back-to-back
calls), algorithmic GB/s and GFLOP/s under DESIGN.md's cost convention, fraction of the measured HBM peak.
--rotate R cycles over R independent in/out buffer sets so that small lattices are not L2-resident.
"""
import argparse
import json
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import synth  # noqa: E402
import paper_1810_01609_b200 as mdwf  # noqa: E402

OPS = {"hop": mdwf.OP_HOP, "mhat": mdwf.OP_DHAT_SYM, "dhat": mdwf.OP_DHAT_ASYM, "m5inv": mdwf.OP_M5INV,
       "normal": mdwf.OP_NORMAL_SYM}


def measurement_kernels(ctx, cfg, iters, peak):
    """Feynman-Hellmann sequential source and nucleon two-point contraction on random 12-column 4D propagators
    (SURVEY a10, a11): device time, algorithmic GB/s (seq source: read + write one propagator; contraction: read
    three), and GFLOP/s of the contraction at ~2.0e4 flop per site."""
    import numpy as np
    g = torch.Generator(device="cuda").manual_seed(synth.seed_for(cfg.index, 9))
    props = []
    for _ in range(3):
        S = torch.empty((12, cfg.V4, 4, 3), dtype=torch.complex128, device="cuda")
        torch.view_as_real(S).normal_(0.0, 1.0, generator=g)
        props.append(S)
    out = torch.empty_like(props[0])
    G = np.zeros((4, 4), dtype=np.complex128)
    G[0, 2], G[1, 3], G[2, 0], G[3, 1] = 1j, -1j, 1j, -1j          # a signed permutation like gamma_z gamma_5
    P = np.diag([1.0, 1.0, 0.0, 0.0]).astype(np.complex128)
    pbytes = props[0].numel() * 16

    def timed(fn):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(iters):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / iters

    ms = timed(lambda: ctx.mdwf_seq_source(props[0], G, out=out))
    print(json.dumps({"workload": cfg.name, "op": "seq_source", "ms": round(ms, 4), "GBps": round(2 * pbytes / ms / 1e6, 1),
                      "frac_of_measured_hbm": round(2 * pbytes / ms / 1e6 / peak, 4)}), flush=True)
    # gauge-covariant Gaussian smearing (NEXT-3): needs links; one step reads and writes the propagator and reads 3 x 144 B
    # of links per site
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(cfg.index, 1), device="cuda")
    ctx.mdwf_load_gauge(U, 64, 18)
    del U
    n_smear = 30
    ms = timed(lambda: ctx.mdwf_smear_gaussian(props[0], 3.0, n_smear, out=out))
    sbytes = n_smear * (2 * pbytes + 3 * 144 * cfg.V4)
    print(json.dumps({"workload": cfg.name, "op": "smear_gaussian", "steps": n_smear, "ms": round(ms, 4), "ms_per_step": round(ms / n_smear, 4),
                      "GBps": round(sbytes / ms / 1e6, 1), "frac_of_measured_hbm": round(sbytes / ms / 1e6 / peak, 4)}), flush=True)
    ms = timed(lambda: ctx.mdwf_nucleon_2pt(props[0], props[1], props[2], P))
    print(json.dumps({"workload": cfg.name, "op": "nucleon_2pt", "ms": round(ms, 4), "GBps": round(3 * pbytes / ms / 1e6, 1),
                      "GFLOPs": round(2.0e4 * cfg.V4 / ms / 1e6, 1),
                      "frac_of_measured_hbm": round(3 * pbytes / ms / 1e6 / peak, 4)}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--nrhs", type=int, default=1)
    ap.add_argument("--formats", default="64x18,64x12,64x8,32x18,32x12,32x8,16x18,16x12,16x8")
    ap.add_argument("--ops", default="hop,mhat")
    ap.add_argument("--iters", type=int, default=20)
    ap.add_argument("--rotate", type=int, default=4)
    ap.add_argument("--zc", type=int, default=0)
    ap.add_argument("--dagger", type=int, default=0)
    ap.add_argument("--tile", default="", help="fp16 stencil box and warps per block: lx,ly,lz,lt[,warps]")
    ap.add_argument("--autotune", action="store_true", help="run mdwf_autotune for every format first and print what it chose")
    ap.add_argument("--meas", action="store_true", help="time the sequential-source and nucleon 2-pt kernels instead")
    a = ap.parse_args()
    cfg = synth.CONFIGS[a.config]
    peak = 6650.0
    pk = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        peak = float(json.load(open(pk))["hbm_gbs"])
    ctx = mdwf.Context(cfg.dims, cfg.Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc)
    ctx.mdwf_set_tiling(a.zc)
    if a.tile:
        t = [int(v) for v in a.tile.split(",")]
        ctx.mdwf_set_hop16_tile(t[0], t[1], t[2], t[3], t[4] if len(t) > 4 else 0)
    if a.meas:
        measurement_kernels(ctx, cfg, a.iters, peak)
        return
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(cfg.index, 1), device="cuda")
    fmts = [tuple(int(v) for v in f.split("x")) for f in a.formats.split(",")]
    for prec, recon in fmts:
        ctx.mdwf_load_gauge(U, prec, recon)
    del U
    torch.cuda.empty_cache()
    if a.autotune:
        for prec, recon in fmts:
            ctx.mdwf_autotune(prec, recon, a.nrhs)
        tmp = "/tmp/mdwf_tune_%d.txt" % os.getpid()
        ctx.mdwf_tune_save(tmp)
        print(json.dumps({"autotune": [l.split() for l in open(tmp).read().splitlines() if l and l[0] != "#"]}), flush=True)
        os.remove(tmp)
    Vh = cfg.V4 // 2
    g = torch.Generator(device="cuda").manual_seed(synth.seed_for(cfg.index, 2))
    for prec, recon in fmts:
        fin = [ctx.mdwf_field_create(prec, a.nrhs) for _ in range(a.rotate)]
        fout = [ctx.mdwf_field_create(prec, a.nrhs) for _ in range(a.rotate)]
        for f in fin:
            src = torch.empty((a.nrhs, cfg.Ls, Vh, 4, 3), dtype=torch.complex128, device="cuda")
            torch.view_as_real(src).normal_(0.0, 1.0, generator=g)
            f.mdwf_field_pack(src)
            del src
        for name in a.ops.split(","):
            op = OPS[name]
            for k in range(3):
                ctx.mdwf_dslash_packed(op, fout[k % a.rotate], fin[k % a.rotate], 0, bool(a.dagger), recon)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for k in range(a.iters):
                ctx.mdwf_dslash_packed(op, fout[k % a.rotate], fin[k % a.rotate], 0, bool(a.dagger), recon)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / a.iters
            by, fl = ctx.mdwf_dslash_cost(op, prec, recon, a.nrhs)
            print(json.dumps({"workload": cfg.name, "nrhs": a.nrhs, "prec": prec, "recon": recon, "op": name,
                              "ms": round(ms, 5), "GBps": round(by / ms / 1e6, 1), "GFLOPs": round(fl / ms / 1e6, 1),
                              "frac_of_measured_hbm": round(by / ms / 1e6 / peak, 4), "rotate": a.rotate}), flush=True)
        for f in fin + fout:
            f.mdwf_field_destroy()


if __name__ == "__main__":
    main()

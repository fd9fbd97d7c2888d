"""GPU parity at the shape of BASELINE.json configs[1] (16^3x32, Ls=8), in the launch configuration bench.py times:
every even-odd operator for both parities and +-dagger in all nine {fp64, fp32, fp16} x {18, 12, 8 real} formats against
the fp64 CPU oracle on the whole field, and one full mixed-precision solve against the oracle's own even-odd CG
("both parities, +-dagger; parity of each vs oracle")."""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5, 16: 2e-3}      # north_star (fp64, fp32); fp16: DESIGN.md "Tolerances"


def rel(a, b):
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.fixture(scope="module")
def c2():
    import paper_1810_01609_b200 as mdwf
    cfg = synth.CONFIGS[2]
    p = oracle.Params(dims=cfg.dims, Ls=cfg.Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=cfg.mf, bc=cfg.bc)
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(2, 1))
    psi = synth.gaussian_spinor(cfg.dims, cfg.Ls, 1, synth.seed_for(2, 2)).numpy()
    ctx = mdwf.Context(cfg.dims, cfg.Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc)
    Un = U.numpy()
    ref = {}
    for parity in (0, 1):
        same, other = oracle.mask(p, psi, parity), oracle.mask(p, psi, 1 - parity)
        for dagger in (False, True):
            ref[(mdwf.OP_HOP, parity, dagger)] = (oracle.to_half(other, cfg.dims, 1 - parity),
                                                  oracle.to_half(oracle.hop(p, Un, other, dagger=dagger, out_parity=parity), cfg.dims, parity))
            for op, sym in ((mdwf.OP_DHAT_ASYM, False), (mdwf.OP_DHAT_SYM, True)):
                ref[(op, parity, dagger)] = (oracle.to_half(same, cfg.dims, parity),
                                             oracle.to_half(oracle.schur(p, Un, same, parity, dagger, sym), cfg.dims, parity))
    yield mdwf, cfg, p, U, ctx, ref
    ctx.mdwf_destroy()


@pytest.mark.parametrize("prec", [64, 32, 16])
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_config2_operators_all_formats(c2, prec, recon):
    mdwf, cfg, p, U, ctx, ref = c2
    ctx.mdwf_load_gauge(U.cuda(), prec, recon)
    for (op, parity, dagger), (inp, exp) in ref.items():
        got = ctx.mdwf_dslash(op, torch.from_numpy(inp).cuda(), parity=parity, dagger=dagger, prec=prec, recon=recon)
        e = rel(got.cpu().numpy(), exp)
        assert e <= TOL[prec] * (4 if op != mdwf.OP_HOP and prec == 16 else 1), (op, parity, dagger, prec, recon, e)


def test_config2_mixed_precision_solve_vs_oracle(c2):
    """16-bit inner CG with fp64 reliable updates to 1e-8: true residual by the ORACLE's full operator and solution
    against the oracle's even-odd CG solved 100x tighter."""
    mdwf, cfg, p, U, ctx, ref = c2
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    b = synth.gaussian_spinor(cfg.dims, cfg.Ls, 1, synth.seed_for(2, 3))
    x, res = ctx.mdwf_solve(b.cuda(), tol=cfg.tol, inner_prec=16, recon=12)
    assert res.status == mdwf.OK, res
    xn, bn, Un = x.cpu().numpy(), b.numpy(), U.numpy()
    tr = oracle.true_residual(p, Un, xn, bn)
    assert tr.max() <= cfg.tol, tr
    xo, its, _ = oracle.solve_eo(p, Un, bn, parity=0, symmetric=True, tol=cfg.tol * 1e-2, max_iter=100000)
    assert rel(xn, xo) <= 1e-6, rel(xn, xo)

"""GPU parity: every operator of mdwf_dslash (C-ABI) against the fp64 CPU oracle, element by element on
the same seeded inputs (tolerances: north_star fp64 <= 1e-12, fp32 <= 1e-5 rel-L2;
16-bit bound derived in DESIGN.md "Tolerances")."""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5, 16: 2e-3}


def rel(a, b):
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def setup(dims, Ls, mf, eps=0.3, seed=1001, bc=(1, 1, 1, -1), b5=1.5, c5=0.5, M5=1.3):
    import paper_1810_01609_b200 as mdwf
    p = oracle.Params(dims=tuple(dims), Ls=Ls, M5=M5, b5=b5, c5=c5, mf=mf, bc=tuple(bc))
    U = synth.gauge_field(dims, eps, seed)
    ctx = mdwf.Context(dims, Ls, M5, b5, c5, mf, bc=bc)
    return mdwf, p, U, ctx


def half_ops(mdwf, p, U, psi_full, parity, dagger):
    """oracle results on half-lattice inputs: dict op -> (input half field, expected half field)"""
    Un = U.numpy()
    dims = p.dims
    same = oracle.mask(p, psi_full, parity)
    other = oracle.mask(p, psi_full, 1 - parity)
    h_same, h_other = oracle.to_half(same, dims, parity), oracle.to_half(other, dims, 1 - parity)
    out = {}
    out[mdwf.OP_HOP] = (h_other, oracle.to_half(oracle.hop(p, Un, other, dagger=dagger, out_parity=parity), dims, parity))
    out[mdwf.OP_M4PRE] = (h_same, oracle.to_half(oracle.M4pre(p, same, dagger), dims, parity))
    out[mdwf.OP_M5] = (h_same, oracle.to_half(oracle.M5op(p, same, dagger), dims, parity))
    out[mdwf.OP_M5INV] = (h_same, oracle.to_half(oracle.M5inv(p, same, dagger), dims, parity))
    out[mdwf.OP_DHAT_ASYM] = (h_same, oracle.to_half(oracle.schur(p, Un, same, parity, dagger, False), dims, parity))
    out[mdwf.OP_DHAT_SYM] = (h_same, oracle.to_half(oracle.schur(p, Un, same, parity, dagger, True), dims, parity))
    for op, sym in ((mdwf.OP_NORMAL_ASYM, False), (mdwf.OP_NORMAL_SYM, True)):
        t = oracle.schur(p, Un, same, parity, False, sym)
        out[op] = (h_same, oracle.to_half(oracle.schur(p, Un, t, parity, True, sym), dims, parity))
    return out


@pytest.mark.parametrize("dims,Ls,mf", [((4, 4, 4, 4), 4, 0.1), ((6, 4, 2, 8), 5, 0.05), ((8, 8, 4, 6), 12, 0.02)])
@pytest.mark.parametrize("prec,recon", [(64, 18), (64, 12), (64, 8), (32, 18), (32, 12), (32, 8), (16, 18), (16, 12), (16, 8)])
def test_all_ops_match_oracle(dims, Ls, mf, prec, recon):
    mdwf, p, U, ctx = setup(dims, Ls, mf)
    ctx.mdwf_load_gauge(U.cuda(), prec, recon)
    nrhs = 2
    psi = synth.gaussian_spinor(dims, Ls, nrhs, 1002).numpy()
    for parity in (0, 1):
        for dagger in (False, True):
            ref = half_ops(mdwf, p, U, psi, parity, dagger)
            for op, (inp, exp) in ref.items():
                got = ctx.mdwf_dslash(op, torch.from_numpy(inp).cuda(), parity=parity, dagger=dagger, prec=prec, recon=recon)
                torch.cuda.synchronize()
                e = rel(got.cpu().numpy(), exp)
                assert e <= TOL[prec] * (4 if op >= mdwf.OP_DHAT_ASYM and prec == 16 else 1), (op, parity, dagger, prec, recon, e)


@pytest.mark.parametrize("prec,recon", [(64, 18), (32, 12), (16, 12)])
def test_full_operator_matches_oracle(prec, recon):
    dims, Ls = (4, 6, 4, 8), 6
    mdwf, p, U, ctx = setup(dims, Ls, 0.07, bc=(-1, 1, 1, -1))
    ctx.mdwf_load_gauge(U.cuda(), prec, recon)
    psi = synth.gaussian_spinor(dims, Ls, 3, 1003)
    for dagger in (False, True):
        got = ctx.mdwf_dslash(mdwf.OP_FULL, psi.cuda(), dagger=dagger, prec=prec, recon=recon).cpu().numpy()
        exp = oracle.D(p, U.numpy(), psi.numpy(), dagger=dagger)
        assert rel(got, exp) <= TOL[prec], (dagger, rel(got, exp))


def test_free_field_unit_links_and_extent2():
    """unit links (18/12 formats), extent-2 directions (both hops hit the same neighbour, A21), Ls = 1"""
    dims, Ls = (2, 2, 4, 2), 1
    mdwf, p, _, ctx = setup(dims, Ls, 0.3)
    U = synth.unit_gauge(dims)
    psi = synth.gaussian_spinor(dims, Ls, 1, 1004)
    for recon in (18, 12):
        ctx.mdwf_load_gauge(U.cuda(), 64, recon)
        got = ctx.mdwf_dslash(mdwf.OP_FULL, psi.cuda(), prec=64, recon=recon).cpu().numpy()
        assert rel(got, oracle.D(p, U.numpy(), psi.numpy())) <= 1e-12
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_load_gauge(U.cuda(), 64, 8)      # 8-real format is singular on unit links: loud failure


def test_config2_shape_sampled():
    """16^3x32, Ls=8 (BASELINE configs[1]) in the launch configuration bench.py times: hop in all three
    precisions against the oracle on the full field (the oracle does this size in seconds)."""
    cfg = synth.CONFIGS[2]
    mdwf, p, U, ctx = setup(cfg.dims, cfg.Ls, cfg.mf, eps=cfg.eps, seed=synth.seed_for(2, 1))
    psi = synth.gaussian_spinor(cfg.dims, cfg.Ls, 1, synth.seed_for(2, 2)).numpy()
    other = oracle.mask(p, psi, 1)
    exp = oracle.to_half(oracle.hop(p, U.numpy(), other, out_parity=0), cfg.dims, 0)
    inp = torch.from_numpy(oracle.to_half(other, cfg.dims, 1)).cuda()
    Ud = U.cuda()
    for prec, recon in [(64, 18), (32, 18), (32, 12), (32, 8), (16, 18), (16, 12), (16, 8)]:
        ctx.mdwf_load_gauge(Ud, prec, recon)
        got = ctx.mdwf_dslash(mdwf.OP_HOP, inp, parity=0, prec=prec, recon=recon).cpu().numpy()
        assert rel(got, exp) <= TOL[prec], (prec, recon, rel(got, exp))


def test_errors_are_loud():
    import paper_1810_01609_b200 as mdwf
    with pytest.raises(mdwf.MdwfError):
        mdwf.Context((3, 4, 4, 4), 4, 1.3, 1.5, 0.5, 0.1)
    ctx = mdwf.Context((4, 4, 4, 4), 4, 1.3, 1.5, 0.5, 0.1)
    x = torch.zeros((1, 4, 128, 4, 3), dtype=torch.complex128, device="cuda")
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_dslash(mdwf.OP_HOP, x, prec=32, recon=12)   # gauge not loaded


def test_traversal_order_does_not_change_results():
    """the z-slab depth (mdwf_set_tiling) only reorders blocks: results are bit-identical for every legal depth"""
    dims, Ls = (8, 8, 8, 4), 8          # blocks are whole (x, y) planes here, so every divisor of Z is a legal depth
    mdwf, p, U, ctx = setup(dims, Ls, 0.1)
    ctx.mdwf_load_gauge(U.cuda(), 32, 12)
    Vh = int(np.prod(dims)) // 2
    inp = synth.gaussian_spinor(dims, Ls, 3, 1010)[:, :, :Vh].contiguous().cuda()
    ref = None
    for zc in (0, 1, 2, 4, 8):
        ctx.mdwf_set_tiling(zc)
        out = ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, inp, parity=1, prec=32, recon=12)
        if ref is None:
            ref = out
        assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref)), zc
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_set_tiling(3)


def test_maximum_ls_and_empty_batch():
    """Ls = 32 (the maximum the library accepts: 8 resp. 4 sites per block) through the fused Schur operator in all
    three storage precisions; Ls = 33 and an empty batch are refused."""
    dims, Ls = (4, 4, 2, 4), 32
    mdwf, p, U, ctx = setup(dims, Ls, 0.05)
    psi = synth.gaussian_spinor(dims, Ls, 2, 1020).numpy()
    same = oracle.mask(p, psi, 0)
    inp = torch.from_numpy(oracle.to_half(same, dims, 0)).cuda()
    for prec, recon in [(64, 18), (32, 12), (16, 8)]:
        ctx.mdwf_load_gauge(U.cuda(), prec, recon)
        for dagger in (False, True):
            exp = oracle.to_half(oracle.schur(p, U.numpy(), same, 0, dagger, True), dims, 0)
            got = ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, inp, parity=0, dagger=dagger, prec=prec, recon=recon)
            assert rel(got.cpu().numpy(), exp) <= TOL[prec] * (4 if prec == 16 else 1), (prec, dagger)
    with pytest.raises(mdwf.MdwfError):
        mdwf.Context(dims, 33, 1.3, 1.5, 0.5, 0.1)
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_dslash(mdwf.OP_HOP, inp[:0].contiguous(), prec=64, recon=18)

"""GPU parity: mdwf_solve (mixed-precision CG with reliable updates) and the FH chain against the oracle.
Acceptance (north_star / SURVEY O2): full-system true residual <= tol with the ORACLE's D in fp64;
solution rel-L2 vs the oracle solution <= 1e-6; manufactured solution b = D psi*."""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def make(cfg_index, dims=None, Ls=None, mf=None):
    import paper_1810_01609_b200 as mdwf
    cfg = synth.CONFIGS[cfg_index]
    dims = dims or cfg.dims
    Ls = Ls or cfg.Ls
    mf = mf if mf is not None else cfg.mf
    p = oracle.Params(dims=tuple(dims), Ls=Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=mf, bc=cfg.bc)
    U = synth.gauge_field(dims, cfg.eps, synth.seed_for(cfg_index, 1))
    ctx = mdwf.Context(dims, Ls, cfg.M5, cfg.b5, cfg.c5, mf, bc=cfg.bc)
    Ud = U.cuda()
    ctx.mdwf_load_gauge(Ud, 64, 18)
    return mdwf, cfg, p, U, ctx, Ud


@pytest.mark.parametrize("inner,recon", [(64, 18), (32, 12), (16, 12), (16, 8)])
@pytest.mark.parametrize("symmetric", [True, False])
def test_config1_solve(inner, recon, symmetric):
    """BASELINE configs[0]: 4^4, Ls=4, CG to 1e-10; oracle variant A (unpreconditioned) is the reference."""
    mdwf, cfg, p, U, ctx, Ud = make(1)
    if inner != 64:
        ctx.mdwf_load_gauge(Ud, inner, recon)
    elif recon != 18:
        ctx.mdwf_load_gauge(Ud, 64, recon)
    b = synth.gaussian_spinor(cfg.dims, cfg.Ls, 1, synth.seed_for(1, 2))
    x, res = ctx.mdwf_solve(b.cuda(), tol=1e-10, inner_prec=inner, recon=recon, symmetric=symmetric)
    assert res.status == mdwf.OK, res
    xn = x.cpu().numpy()
    tr = oracle.true_residual(p, U.numpy(), xn, b.numpy())
    assert tr.max() <= 1e-10, (tr, res)
    assert abs(res.true_resid[0] - tr[0]) <= 0.05 * tr[0] + 1e-13      # library's own residual is the true one
    xo, _, _ = oracle.solve_full(p, U.numpy(), b.numpy(), tol=1e-13)
    assert rel(xn, xo) <= 1e-6


@pytest.mark.parametrize("parity", [0, 1])
def test_multi_rhs_batched_manufactured(parity):
    """8^3x16, Ls=8, 5 rhs in batches of 2 (ragged last batch): psi* Gaussian, b = D psi* by the oracle."""
    mdwf, cfg, p, U, ctx, Ud = make(3, dims=(8, 8, 8, 16))
    ctx.mdwf_load_gauge(Ud, 16, 12)
    star = synth.gaussian_spinor(p.dims, p.Ls, 5, synth.seed_for(3, 50)).numpy()
    b = oracle.D(p, U.numpy(), star)
    x, res = ctx.mdwf_solve(torch.from_numpy(b).cuda(), tol=1e-9, inner_prec=16, recon=12, parity=parity, batch=2)
    assert res.status == mdwf.OK, res
    xn = x.cpu().numpy()
    for r in range(5):
        assert rel(xn[r], star[r]) <= 1e-6, (r, rel(xn[r], star[r]))
    assert oracle.true_residual(p, U.numpy(), xn, b).max() <= 1e-9
    assert all(n >= 1 for n in res.reliable_updates)


def test_point_source_propagator_4d():
    """configs[2] shape scaled to 8^3x16: 12 point sources on the walls (O3), 4D in / 4D out; checked against
    the oracle's wall_inject -> solve_eo -> wall_project, and through the true residual of the 5D system."""
    mdwf, cfg, p, U, ctx, Ud = make(3, dims=(8, 8, 8, 16))
    ctx.mdwf_load_gauge(Ud, 16, 12)
    eta = synth.point_sources_4d(p.dims)
    q, res = ctx.mdwf_solve(eta.cuda(), tol=1e-9, inner_prec=16, recon=12, src_kind=1, out_kind=1)
    assert res.status == mdwf.OK, res
    Un = U.numpy()
    cols = [0, 7]
    b5 = oracle.wall_inject(p, Un, eta.numpy()[cols])
    assert rel(ctx.mdwf_wall_inject(eta.cuda()).cpu().numpy()[cols], b5) <= 1e-12
    xo, _, _ = oracle.solve_eo(p, Un, b5, tol=1e-12)
    qo = oracle.wall_project(p, xo)
    assert rel(q.cpu().numpy()[cols], qo) <= 1e-6
    # 5D output of the same solve satisfies the full system
    x5, res5 = ctx.mdwf_solve(eta.cuda()[cols], tol=1e-9, inner_prec=16, recon=12, src_kind=1, out_kind=0)
    assert oracle.true_residual(p, Un, x5.cpu().numpy(), b5).max() <= 1e-9
    assert rel(ctx.mdwf_wall_project(x5).cpu().numpy(), qo) <= 1e-6


def test_host_buffer_solve_matches_device_solve():
    mdwf, cfg, p, U, ctx, Ud = make(1)
    ctx.mdwf_load_gauge(Ud, 32, 12)
    b = synth.gaussian_spinor(cfg.dims, cfg.Ls, 3, synth.seed_for(1, 3))
    xh = torch.empty_like(b).pin_memory()
    _, res = ctx.mdwf_solve_host(b.pin_memory(), xh, tol=1e-10, inner_prec=32, recon=12, batch=2)
    assert res.status == mdwf.OK
    assert oracle.true_residual(p, U.numpy(), xh.numpy(), b.numpy()).max() <= 1e-10


@pytest.mark.parametrize("slices", [1, 3])
def test_host_buffer_solve_streams_in_chunks(slices, monkeypatch):
    """mdwf_solve_host streams every right-hand side through two staging chunks of whole s-slices.  At test
    sizes one chunk would hold all of Ls, so MDWF_STAGE_SLICES forces chunks of 1 and of 3 slices (Ls = 8: ragged last
    chunk), with 3 rhs in batches of 2 (the chunk buffers are re-used across right-hand sides, batches, upload and
    download).  Same packed fields, same solve: the result must equal the device-buffer solve bit for bit."""
    import paper_1810_01609_b200 as mdwf
    dims, Ls, mf = (4, 4, 4, 6), 8, 0.08
    p = oracle.Params(dims=dims, Ls=Ls, M5=1.3, b5=1.5, c5=0.5, mf=mf, bc=(1, 1, 1, -1))
    U = synth.gauge_field(dims, 0.3, 6101)
    ctx = mdwf.Context(dims, Ls, 1.3, 1.5, 0.5, mf)
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    b = synth.gaussian_spinor(dims, Ls, 3, 6102)
    kw = dict(tol=1e-9, inner_prec=16, recon=12, batch=2)
    xd, rd = ctx.mdwf_solve(b.cuda(), **kw)
    monkeypatch.setenv("MDWF_STAGE_SLICES", str(slices))
    xh = torch.full(b.shape, float("nan"), dtype=b.dtype).pin_memory()
    _, rh = ctx.mdwf_solve_host(b.pin_memory(), xh, **kw)
    assert rd.status == mdwf.OK and rh.status == mdwf.OK and rh.iters == rd.iters
    assert torch.equal(torch.view_as_real(xh), torch.view_as_real(xd.cpu()))
    assert oracle.true_residual(p, U.numpy(), xh.numpy(), b.numpy()).max() <= 1e-9


def test_not_converged_is_reported():
    mdwf, cfg, p, U, ctx, Ud = make(1)
    b = synth.gaussian_spinor(cfg.dims, cfg.Ls, 1, synth.seed_for(1, 2))
    x, res = ctx.mdwf_solve(b.cuda(), tol=1e-10, inner_prec=64, recon=18, max_iter=3)
    assert res.status == mdwf.NOT_CONVERGED and res.rhs_status[0] == mdwf.NOT_CONVERGED


def test_edge_cases_zero_rhs_max_batch_and_ls1():
    """degenerate inputs: an all-zero rhs inside a batch (solution 0, converged at once), the maximum batch of 64 rhs
    through mdwf_dslash, and Ls = 1 (L has only the -mf wraps, A21) solved in the asymmetric form on parity 1."""
    import paper_1810_01609_b200 as mdwf
    cfg = synth.CONFIGS[1]
    p = oracle.Params(dims=cfg.dims, Ls=cfg.Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=cfg.mf, bc=cfg.bc)
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(1, 1))
    ctx = mdwf.Context(cfg.dims, cfg.Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc)
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    b = synth.gaussian_spinor(cfg.dims, cfg.Ls, 3, synth.seed_for(1, 4))
    b[1] = 0
    x, res = ctx.mdwf_solve(b.cuda(), tol=1e-9, inner_prec=16, recon=12)
    assert res.status == mdwf.OK and res.iters[1] == 0
    xn = x.cpu().numpy()
    assert np.all(xn[1] == 0)
    tr = oracle.true_residual(p, U.numpy(), xn[[0, 2]], b.numpy()[[0, 2]])
    assert tr.max() <= 1e-9
    # 64 rhs through the Dslash entry point
    psi = synth.gaussian_spinor(cfg.dims, cfg.Ls, 64, synth.seed_for(1, 5)).numpy()
    same = oracle.mask(p, psi, 0)
    exp = oracle.to_half(oracle.schur(p, U.numpy(), same, 0, False, True), cfg.dims, 0)
    got = ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, torch.from_numpy(oracle.to_half(same, cfg.dims, 0)).cuda(), prec=64, recon=18)
    assert rel(got.cpu().numpy(), exp) <= 1e-12
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_dslash(mdwf.OP_HOP, torch.zeros((65, cfg.Ls, cfg.V4 // 2, 4, 3), dtype=torch.complex128, device="cuda"))
    # Ls = 1
    dims = (4, 2, 6, 4)
    p1 = oracle.Params(dims=dims, Ls=1, M5=1.4, b5=1.2, c5=0.3, mf=0.2, bc=(1, -1, 1, -1))
    U1 = synth.gauge_field(dims, 0.3, 77)
    c1 = mdwf.Context(dims, 1, 1.4, 1.2, 0.3, 0.2, bc=(1, -1, 1, -1))
    c1.mdwf_load_gauge(U1.cuda(), 64, 18)
    c1.mdwf_load_gauge(U1.cuda(), 32, 8)
    b1 = synth.gaussian_spinor(dims, 1, 2, 78)
    x1, r1 = c1.mdwf_solve(b1.cuda(), tol=1e-10, inner_prec=32, recon=8, parity=1, symmetric=False)
    assert r1.status == mdwf.OK
    assert oracle.true_residual(p1, U1.numpy(), x1.cpu().numpy(), b1.numpy()).max() <= 1e-10


def test_bit_reproducible_and_packed_api_and_profile():
    """fixed-order reductions: two solves of the same input are bit-identical; the packed-field calls give
    the same numbers as mdwf_dslash; the hop profiler counts launches and the documented algorithmic bytes."""
    import paper_1810_01609_b200 as mdwf
    dims, Ls = (8, 8, 4, 8), 10
    cfg = synth.CONFIGS[5]
    U = synth.gauge_field(dims, cfg.eps, 901).cuda()
    ctx = mdwf.Context(dims, Ls, cfg.M5, cfg.b5, cfg.c5, cfg.mf, bc=cfg.bc)
    ctx.mdwf_load_gauge(U, 64, 18)
    ctx.mdwf_load_gauge(U, 16, 12)
    b = synth.gaussian_spinor(dims, Ls, 3, 902).cuda()
    x1, r1 = ctx.mdwf_solve(b, tol=1e-9, inner_prec=16, recon=12, batch=2)
    x2, r2 = ctx.mdwf_solve(b, tol=1e-9, inner_prec=16, recon=12, batch=2)
    assert r1.status == mdwf.OK and r1.iters == r2.iters
    assert torch.equal(torch.view_as_real(x1), torch.view_as_real(x2))
    # packed API == canonical API
    V4 = int(np.prod(dims))
    half = synth.gaussian_spinor(dims, Ls, 2, 903)[:, :, : V4 // 2].contiguous().cuda()
    fin, fout = ctx.mdwf_field_create(16, 2), ctx.mdwf_field_create(16, 2)
    fin.mdwf_field_pack(half)
    ctx.mdwf_profile(True)
    ctx.mdwf_dslash_packed(mdwf.OP_DHAT_SYM, fout, fin, parity=1, dagger=True, recon=12)
    out = torch.empty_like(half)
    fout.mdwf_field_unpack(out)
    ms, by, fl, n = ctx.mdwf_profile_read(0)
    ctx.mdwf_profile(False)
    ref = ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, half, parity=1, dagger=True, prec=16, recon=12)
    assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref))
    n5 = (V4 // 2) * Ls * 2
    assert n == 2 and ms > 0 and fl == 2 * 1320.0 * n5
    assert by == (2 + 3) * 48.0 * n5 + 2 * 8 * 12 * 2 * (V4 // 2)      # one plain-input and one xpay-input fused hop
    cb, cf = ctx.mdwf_dslash_cost(mdwf.OP_HOP, 16, 12, 2)
    assert cb == 2 * 48.0 * n5 + 8 * 12 * 2 * (V4 // 2) and cf == 1320.0 * n5
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_dslash_packed(mdwf.OP_HOP, fin, fin, recon=12)          # out must not alias in

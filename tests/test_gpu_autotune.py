"""Run-time autotuner (PAPER.md:92-94 IV: "brute-force search over the launch parameters ... stored in a std::map ...
written to disk"): the search must leave every result unchanged (launch parameters only regroup the work),
record an admissible entry per (kernel, lattice, Ls, rhs count), and survive a save / load round trip into a fresh
context."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

DIMS, LS = (8, 8, 8, 8), 10


def make_ctx():
    import paper_1810_01609_b200 as mdwf
    U = synth.gauge_field(DIMS, 0.3, 4101).cuda()
    ctx = mdwf.Context(DIMS, LS, 1.3, 1.5, 0.5, 0.05)
    for prec, recon in ((16, 12), (32, 12), (64, 18)):
        ctx.mdwf_load_gauge(U, prec, recon)
    return mdwf, ctx


def test_autotune_keeps_results_and_round_trips(tmp_path):
    mdwf, ctx = make_ctx()
    Vh = int(np.prod(DIMS)) // 2
    nrhs = 4
    inp = synth.gaussian_spinor(DIMS, LS, nrhs, 4102)[:, :, :Vh].contiguous().cuda()
    fmts = ((16, 12), (32, 12), (64, 18))
    before = {f: ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, inp, parity=0, prec=f[0], recon=f[1]) for f in fmts}
    for prec, recon in fmts:
        ctx.mdwf_autotune(prec, recon, nrhs)
    lat = "%dx%dx%dx%d/Ls%d" % (DIMS + (LS,))
    t16 = ctx.mdwf_tune_get("hop16/%s/rows%d" % (lat, 4 * LS))
    assert len(t16) == 5 and t16[0] % 2 == 0 and all(d % t == 0 for d, t in zip(DIMS, t16[:4])) and t16[4] in (4, 8, 16)
    for name in ("hop32", "hop64"):
        zc = ctx.mdwf_tune_get("%s/%s/rhs%d" % (name, lat, nrhs))
        assert len(zc) == 1 and zc[0] >= 1 and DIMS[2] % zc[0] == 0
    assert ctx.mdwf_tune_get("hop32/%s/rhs%d" % (lat, 63)) == []
    # tuned launches give the same numbers: bit-identical stencil outputs (the tile / slab depth only regroups the work)
    for f in fmts:
        after = ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, inp, parity=0, prec=f[0], recon=f[1])
        assert torch.equal(torch.view_as_real(after), torch.view_as_real(before[f])), f
    # save -> load into a fresh context -> identical entries, identical results
    path = tmp_path / "mdwf_tune.txt"
    ctx.mdwf_tune_save(path)
    text = path.read_text()
    assert "hop16/" in text and "hop32/" in text and "hop64/" in text
    mdwf2, ctx2 = make_ctx()
    ctx2.mdwf_tune_load(path)
    assert ctx2.mdwf_tune_get("hop16/%s/rows%d" % (lat, 4 * LS)) == t16
    path2 = tmp_path / "again.txt"
    ctx2.mdwf_tune_save(path2)
    assert path2.read_text() == text
    for f in fmts:
        again = ctx2.mdwf_dslash(mdwf.OP_DHAT_SYM, inp, parity=0, prec=f[0], recon=f[1])
        assert torch.equal(torch.view_as_real(again), torch.view_as_real(before[f])), f


def test_autotune_refuses_what_is_not_loaded(tmp_path):
    mdwf, ctx = make_ctx()
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_autotune(32, 8, 1)                    # format not loaded
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_tune_load(tmp_path / "missing.txt")
    bad = tmp_path / "bad.txt"
    bad.write_text("hop32/oops\n")
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_tune_load(bad)


def test_solve_after_autotune_matches_solve_before():
    """the solver sees the tuned parameters through the same launchers: same iteration counts, same solution up to the
    order of the fp32 partial sums inside the tensor-core stencil's reductions"""
    mdwf, ctx = make_ctx()
    b = synth.gaussian_spinor(DIMS, LS, 2, 4103).cuda()
    x0, r0 = ctx.mdwf_solve(b, tol=1e-9, inner_prec=16, recon=12)
    ctx.mdwf_autotune(16, 12, 2)
    ctx.mdwf_autotune(64, 18, 1)
    x1, r1 = ctx.mdwf_solve(b, tol=1e-9, inner_prec=16, recon=12)
    assert r1.status == 0 and max(r1.true_resid) <= 1e-9
    assert abs(r1.iters[0] - r0.iters[0]) <= 2
    assert (x1 - x0).norm() / x0.norm() < 1e-8

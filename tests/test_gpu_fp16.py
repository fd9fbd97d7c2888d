"""The 16-bit storage path ("16-bit precision ... storage (utilizing single-precision computation)";
DESIGN.md R11: IEEE fp16 values with one power-of-two scale per field and rhs, products on the tensor cores accumulated in
fp32).  SURVEY O1's isolating check: the GPU operator against the oracle applied to the DEQUANTISED packed inputs, which
separates the arithmetic from the storage rounding."""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu


def setup(dims, Ls, mf, seed=2101):
    import paper_1810_01609_b200 as mdwf
    p = oracle.Params(dims=tuple(dims), Ls=Ls, M5=1.3, b5=1.5, c5=0.5, mf=mf, bc=(1, 1, 1, -1))
    U = synth.gauge_field(dims, 0.3, seed)
    ctx = mdwf.Context(dims, Ls, 1.3, 1.5, 0.5, mf)
    return mdwf, p, U, ctx


def dequantised_links(U):
    """what the stencil multiplies for the 18-real fp16 format: every real rounded double -> float -> half"""
    Un = U.numpy()
    re = Un.real.astype(np.float32).astype(np.float16).astype(np.float64)
    im = Un.imag.astype(np.float32).astype(np.float16).astype(np.float64)
    return re + 1j * im


@pytest.mark.parametrize("dims,Ls,nrhs", [((8, 4, 4, 6), 10, 4), ((4, 4, 4, 4), 8, 1), ((6, 4, 2, 8), 5, 3)])
def test_hop_on_dequantised_inputs_is_exact_to_half_an_ulp(dims, Ls, nrhs):
    """out = H in with in, U taken at their stored (dequantised) values: the only remaining error is the rounding of the
    result to half precision, so every element must sit within half an fp16 ulp of the oracle's value (slack 2 % of an
    ulp ~ 1e-5 relative: the fp32 accumulation of exact half x half products).  An arithmetic slip at the 1e-4 level --
    a wrong sign on one leg, a link entry misplaced in a fragment -- breaks this, while the 2e-3 bound of the plain
    parity tests would not see it."""
    mdwf, p, U, ctx = setup(dims, Ls, 0.05)
    ctx.mdwf_load_gauge(U.cuda(), 16, 18)
    Vh = int(np.prod(dims)) // 2
    Uq = dequantised_links(U)
    for parity in (0, 1):
        for dagger in (False, True):
            psi = synth.gaussian_spinor(dims, Ls, nrhs, 2102 + parity).numpy()
            psi *= np.array([1.0, 30.0, 1e-3, 7.0][:nrhs]).reshape(nrhs, 1, 1, 1, 1)      # different scales per rhs
            inp = oracle.to_half(oracle.mask(p, psi, 1 - parity), dims, 1 - parity)
            fin, fout = ctx.mdwf_field_create(16, nrhs), ctx.mdwf_field_create(16, nrhs)
            fin.mdwf_field_pack(torch.from_numpy(inp).cuda())
            inq = torch.empty((nrhs, Ls, Vh, 4, 3), dtype=torch.complex128, device="cuda")
            fin.mdwf_field_unpack(inq)                                                    # the stored values
            ctx.mdwf_dslash_packed(mdwf.OP_HOP, fout, fin, parity, dagger, 18)
            got = torch.empty_like(inq)
            fout.mdwf_field_unpack(got)
            exp = oracle.to_half(oracle.hop(p, Uq, oracle.from_half(inq.cpu().numpy(), dims, 1 - parity), dagger=dagger,
                                            out_parity=parity), dims, parity)
            g = torch.view_as_real(got).cpu().numpy().reshape(nrhs, -1)
            e = np.ascontiguousarray(exp).view(np.float64).reshape(nrhs, -1)
            for r in range(nrhs):
                err = np.abs(g[r] - e[r])
                # half an ulp of a normal half is <= 2^-11 |value|.  Absolute floor: the fp32 accumulation of 8 x 24 exact
                # products of typical size (a few 2^-24 of the largest element; it matters only where the legs cancel)
                floor = 3e-6 * np.abs(e[r]).max()
                assert (err <= 2.0 ** -11 * 1.02 * np.abs(e[r]) + floor).all(), (parity, dagger, r, (err / (np.abs(e[r]) + 1e-300)).max())
                # and the rounding errors are unbiased, as roundings are
                assert abs(np.mean((g[r] - e[r]) / (np.abs(e[r]) + 1e-300))) <= 2e-5
            fin.mdwf_field_destroy()
            fout.mdwf_field_destroy()


def test_pack_unpack_round_trip_is_half_precision():
    mdwf, p, U, ctx = setup((4, 4, 4, 4), 6, 0.1)
    Vh = 128
    x = synth.gaussian_spinor((4, 4, 4, 4), 6, 3, 2110)[:, :, :Vh].contiguous().cuda()
    f = ctx.mdwf_field_create(16, 3)
    f.mdwf_field_pack(x)
    y = torch.empty_like(x)
    f.mdwf_field_unpack(y)
    a, b = torch.view_as_real(x).cpu().numpy().reshape(3, -1), torch.view_as_real(y).cpu().numpy().reshape(3, -1)
    for r in range(3):
        floor = np.linalg.norm(a[r]) * 2.0 ** -39 * 8
        assert (np.abs(a[r] - b[r]) <= 2.0 ** -11 * np.abs(a[r]) + floor).all()


def test_tile_choice_does_not_change_the_result():
    """the 4D box a block owns and the warps per block only regroup the work: every output is bit-identical"""
    dims, Ls = (8, 8, 4, 4), 10
    mdwf, p, U, ctx = setup(dims, Ls, 0.05)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    Vh = int(np.prod(dims)) // 2
    inp = synth.gaussian_spinor(dims, Ls, 4, 2120)[:, :, :Vh].contiguous().cuda()
    ref = None
    for tile in [(0, 0, 0, 0, 0), (2, 2, 2, 2, 8), (4, 2, 2, 2, 16), (4, 2, 2, 2, 8), (2, 1, 1, 1, 1), (8, 4, 2, 2, 16)]:
        ctx.mdwf_set_hop16_tile(*tile)
        out = ctx.mdwf_dslash(mdwf.OP_DHAT_SYM, inp, parity=1, prec=16, recon=12)
        if ref is None:
            ref = out
        assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref)), tile
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_set_hop16_tile(3, 2, 2, 2, 8)
        ctx.mdwf_dslash(mdwf.OP_HOP, inp, parity=1, prec=16, recon=12)


def test_packed_solve_equals_canonical_solve_and_workspace():
    """mdwf_solve_packed (in place, no canonical copies) runs the same arithmetic as mdwf_solve: bit-identical solution,
    same iteration counts; with a caller-supplied workspace (mdwf_workspace_bytes / mdwf_set_workspace) too."""
    dims, Ls, nrhs = (8, 8, 4, 8), 8, 3
    mdwf, p, U, ctx = setup(dims, Ls, 0.05)
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    b = synth.gaussian_spinor(dims, Ls, nrhs, 2130)
    x, res = ctx.mdwf_solve(b.cuda(), tol=1e-9, inner_prec=16, recon=12)
    assert res.status == mdwf.OK and res.batch == nrhs
    bn = b.numpy()
    Vh = int(np.prod(dims)) // 2
    ws = torch.empty(ctx.mdwf_workspace_bytes(nrhs, 16, packed=True), dtype=torch.uint8, device="cuda")
    ctx.mdwf_set_workspace(ws)
    f = [ctx.mdwf_field_create(64, nrhs), ctx.mdwf_field_create(64, nrhs)]
    for par in (0, 1):
        h = oracle.to_half(oracle.mask(p, bn, par), dims, par)
        for r in range(nrhs):
            f[par].mdwf_field_pack_rhs(r, torch.from_numpy(np.ascontiguousarray(h[r:r + 1])).cuda())
    res2 = ctx.mdwf_solve_packed(f[0], f[1], tol=1e-9, inner_prec=16, recon=12)
    assert res2.status == mdwf.OK and res2.iters == res.iters and res2.reliable_updates == res.reliable_updates
    xs = np.zeros_like(bn)
    for par in (0, 1):
        out = torch.empty((nrhs, Ls, Vh, 4, 3), dtype=torch.complex128, device="cuda")
        f[par].mdwf_field_unpack(out)
        xs += oracle.from_half(out.cpu().numpy(), dims, par)
    assert np.array_equal(xs, x.cpu().numpy())
    assert oracle.true_residual(p, U.numpy(), xs, bn).max() <= 1e-9
    # a workspace that is too small is refused loudly
    ctx.mdwf_set_workspace(torch.empty(1 << 20, dtype=torch.uint8, device="cuda"))
    with pytest.raises(mdwf.MdwfError):
        ctx.mdwf_solve_packed(f[0], f[1], tol=1e-9, inner_prec=16, recon=12)
    ctx.mdwf_set_workspace(None)

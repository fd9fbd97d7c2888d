"""GPU parity for the fuller Feynman-Hellmann workload (R25):
gauge-covariant Gaussian smearing against the oracle element by element, and the whole chain -- smeared source, solve,
smeared sink, sequential source, solve, u- and d-quark FH correlators with the unpolarised and the polarised projector,
effective derivative -- against the oracle chain on a small lattice."""
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


def crandn(shape, seed):
    g = torch.Generator().manual_seed(seed)
    return torch.complex(torch.randn(shape, generator=g, dtype=torch.float64), torch.randn(shape, generator=g, dtype=torch.float64))


@pytest.mark.parametrize("dims,bc,ncol", [((2, 2, 2, 2), (1, 1, 1, -1), 1), ((6, 4, 2, 2), (-1, 1, 1, -1), 3),
                                          ((6, 6, 4, 2), (1, 1, 1, -1), 12), ((4, 2, 6, 4), (1, -1, 1, 1), 5)])
def test_smear_matches_oracle(dims, bc, ncol):
    """ragged shapes: fewer sites than one block, a partial last block, extent-2 directions, antiperiodic spatial bc"""
    import paper_1810_01609_b200 as mdwf
    V4 = int(np.prod(dims))
    U = synth.gauge_field(dims, 0.35, 5100)
    ctx = mdwf.Context(dims, 2, 1.3, 1.5, 0.5, 0.1, bc=bc)
    psi = crandn((ncol, V4, 4, 3), 5101)
    with pytest.raises(mdwf.MdwfError):                       # links not loaded yet
        ctx.mdwf_smear_gaussian(psi.cuda(), 3.0, 4)
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    for width, n in ((3.0, 0), (1.0, 1), (2.0, 2), (3.0, 5), (3.0, 30)):
        got = ctx.mdwf_smear_gaussian(psi.cuda(), width, n).cpu().numpy()
        exp = oracle.smear_gaussian(dims, U.numpy(), psi.numpy(), width, n, bc=bc)
        assert rel(got, exp) <= 1e-13, (width, n, rel(got, exp))
    d = psi.cuda()
    with pytest.raises(mdwf.MdwfError):                       # in place is refused
        ctx.mdwf_smear_gaussian(d, 3.0, 4, out=d)


def test_effective_derivative_matches_oracle():
    import paper_1810_01609_b200 as mdwf
    dims = (2, 2, 2, 12)
    ctx = mdwf.Context(dims, 2, 1.3, 1.5, 0.5, 0.1)
    c2, cf = crandn((12,), 5201), crandn((12,), 5202)
    got = ctx.mdwf_fh_effective_derivative(c2.cuda(), cf.cuda()).cpu().numpy()
    assert rel(got, oracle.fh_effective_derivative(c2.numpy(), cf.numpy())) <= 1e-14


def fh_workload_gpu(ctx, src, width, n_smear, projs):
    """the NEXT-3 workload on the GPU: returns S, S_FH (smeared-smeared), and per projector (C_2pt, C_FH^u, C_FH^d, g_eff^u, g_eff^d)"""
    kw = dict(tol=1e-10, inner_prec=16, recon=12, src_kind=1, out_kind=1)
    eta = ctx.mdwf_smear_gaussian(src, width, n_smear)                     # source smearing
    S_ps, r1 = ctx.mdwf_solve(eta, **kw)
    G = oracle.gamma(2) @ oracle.gamma(4)                                  # gamma_z gamma_5 (A14)
    SFH_ps, r2 = ctx.mdwf_solve(ctx.mdwf_seq_source(S_ps, G), **kw)        # current on the unsmeared propagator
    assert r1.status == 0 and r2.status == 0
    S, SFH = ctx.mdwf_smear_gaussian(S_ps, width, n_smear), ctx.mdwf_smear_gaussian(SFH_ps, width, n_smear)    # sink smearing
    out = []
    for P in projs:
        c2 = ctx.mdwf_nucleon_2pt(S, S, S, P)
        cu = ctx.mdwf_nucleon_2pt(SFH, S, S, P) + ctx.mdwf_nucleon_2pt(S, S, SFH, P)     # insertion on either u quark
        cd = ctx.mdwf_nucleon_2pt(S, SFH, S, P)                                           # insertion on the d quark
        out.append((c2, cu, cd, ctx.mdwf_fh_effective_derivative(c2, cu), ctx.mdwf_fh_effective_derivative(c2, cd)))
    return S, SFH, out


def test_fh_workload_small_vs_oracle_chain():
    import paper_1810_01609_b200 as mdwf
    dims, Ls, mf = (4, 4, 4, 8), 4, 0.1
    cfg = synth.CONFIGS[4]
    p = oracle.Params(dims=dims, Ls=Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=mf, bc=cfg.bc)
    U = synth.gauge_field(dims, cfg.eps, synth.seed_for(4, 1))
    Un = U.numpy()
    ctx = mdwf.Context(dims, Ls, cfg.M5, cfg.b5, cfg.c5, mf, bc=cfg.bc)
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    g = [oracle.gamma(m) for m in range(4)]
    projs = [0.5 * (np.eye(4) + g[3]), 0.25 * (np.eye(4) + g[3]) @ (np.eye(4) + 1j * g[0] @ g[1])]     # unpolarised, polarised
    width, n_smear = 2.0, 8
    src = synth.point_sources_4d(dims)
    S, SFH, res = fh_workload_gpu(ctx, src.cuda(), width, n_smear, projs)

    def oprop(eta):
        x, _, _ = oracle.solve_eo(p, Un, oracle.wall_inject(p, Un, eta), tol=1e-12)
        return oracle.wall_project(p, x)
    sm = lambda f: oracle.smear_gaussian(dims, Un, f, width, n_smear, bc=cfg.bc)
    So_ps = oprop(sm(src.numpy()))
    SFHo_ps = oprop(oracle.seq_source(dims, So_ps, g[2] @ oracle.gamma(4)))
    So, SFHo = sm(So_ps), sm(SFHo_ps)
    assert rel(S.cpu().numpy(), So) <= 1e-6 and rel(SFH.cpu().numpy(), SFHo) <= 1e-6
    for P, (c2, cu, cd, gu, gd) in zip(projs, res):
        c2o = oracle.nucleon_2pt(dims, So, So, So, P)
        cuo = oracle.nucleon_2pt(dims, SFHo, So, So, P) + oracle.nucleon_2pt(dims, So, So, SFHo, P)
        cdo = oracle.nucleon_2pt(dims, So, SFHo, So, P)
        assert rel(c2.cpu().numpy(), c2o) <= 1e-5 and rel(cu.cpu().numpy(), cuo) <= 1e-5 and rel(cd.cpu().numpy(), cdo) <= 1e-5
        assert rel(gu.cpu().numpy(), oracle.fh_effective_derivative(c2o, cuo)) <= 1e-4
        assert rel(gd.cpu().numpy(), oracle.fh_effective_derivative(c2o, cdo)) <= 1e-4


def test_fh_correlators_are_gauge_invariant_with_covariant_smearing():
    """with gauge-covariant smearing at source and sink the correlators do not change under U -> U^g (SURVEY A16 notes
    that the non-covariant Gaussian source of config 4 does NOT have this property): a whole-chain check that needs no
    oracle solve"""
    import paper_1810_01609_b200 as mdwf
    dims, Ls, mf = (4, 4, 4, 8), 4, 0.1
    cfg = synth.CONFIGS[4]
    V4 = int(np.prod(dims))
    U = synth.gauge_field(dims, cfg.eps, 5301).numpy()
    Gt = synth.random_su3_field(V4, 5302).numpy()
    Gt[0] = np.eye(3)                                         # keep the colour frame at the source point
    X, Y, Z, T = dims
    x4 = np.arange(V4)
    co = [x4 % X, (x4 // X) % Y, (x4 // (X * Y)) % Z, x4 // (X * Y * Z)]
    st = [1, X, X * Y, X * Y * Z]
    Ug = np.empty_like(U)
    for mu in range(4):
        nb = x4 + st[mu] * (((co[mu] + 1) % dims[mu]) - co[mu])
        Ug[mu] = np.einsum("xab,xbc,xdc->xad", Gt, U[mu], Gt[nb].conj())
    P = [0.5 * (np.eye(4) + oracle.gamma(3))]
    src = synth.point_sources_4d(dims).cuda()
    res = []
    for links in (U, Ug):
        ctx = mdwf.Context(dims, Ls, cfg.M5, cfg.b5, cfg.c5, mf, bc=cfg.bc)
        Ut = torch.from_numpy(np.ascontiguousarray(links)).cuda()
        ctx.mdwf_load_gauge(Ut, 64, 18)
        ctx.mdwf_load_gauge(Ut, 16, 12)
        res.append(fh_workload_gpu(ctx, src, 2.0, 6, P)[2][0])
    for a, b in zip(res[0][:3], res[1][:3]):
        assert rel(a.cpu().numpy(), b.cpu().numpy()) <= 1e-6

"""GPU parity: sequential source and nucleon contraction against the oracle's literal index sums (O3/O4)."""
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


def test_seq_source_matches_oracle():
    import paper_1810_01609_b200 as mdwf
    dims = (4, 6, 4, 8)
    ctx = mdwf.Context(dims, 4, 1.3, 1.5, 0.5, 0.1)
    V4 = int(np.prod(dims))
    S = crandn((12, V4, 4, 3), 4001)
    G = oracle.gamma(2) @ oracle.gamma(4)                     # gamma_z gamma_5 (A14)
    for (t0, t1) in [(0, 7), (2, 5), (3, 3)]:
        got = ctx.mdwf_seq_source(S.cuda(), G, t0, t1).cpu().numpy()
        exp = oracle.seq_source(dims, S.numpy(), G, t0, t1)
        assert np.array_equal(got, exp) or rel(got, exp) <= 1e-15
    Gr = crandn((4, 4), 4002).numpy()                          # a dense Gamma exercises every entry
    assert rel(ctx.mdwf_seq_source(S.cuda(), Gr).cpu().numpy(), oracle.seq_source(dims, S.numpy(), Gr)) <= 1e-14


@pytest.mark.parametrize("t0", [0, 3])
def test_nucleon_2pt_matches_oracle(t0):
    import paper_1810_01609_b200 as mdwf
    dims = (4, 4, 2, 6)
    ctx = mdwf.Context(dims, 4, 1.3, 1.5, 0.5, 0.1)
    V4 = int(np.prod(dims))
    S1, S2, S3 = (crandn((12, V4, 4, 3), 4100 + i) for i in range(3))
    g = [oracle.gamma(m) for m in range(4)]
    P_unpol = 0.5 * (np.eye(4) + g[3])
    P_pol = 0.25 * (np.eye(4) + g[3]) @ (np.eye(4) + 1j * g[0] @ g[1])
    for P in (P_unpol, P_pol, crandn((4, 4), 4200).numpy()):
        got = ctx.mdwf_nucleon_2pt(S1.cuda(), S2.cuda(), S3.cuda(), P, t0=t0).cpu().numpy()
        exp = oracle.nucleon_2pt(dims, S1.numpy(), S2.numpy(), S3.numpy(), P, t0=t0)
        assert rel(got, exp) <= 1e-12, rel(got, exp)


def test_nucleon_static_limit():
    """S = delta_ab (1+gamma_t)/2 on every site: C(t) = 36 * V3 with P=(1+gamma_t)/2 and 0 with (1-gamma_t)/2 (A15)."""
    import paper_1810_01609_b200 as mdwf
    dims = (2, 4, 2, 4)
    ctx = mdwf.Context(dims, 2, 1.3, 1.5, 0.5, 0.1)
    V4 = int(np.prod(dims))
    gt = oracle.gamma(3)
    Pp = 0.5 * (np.eye(4) + gt)
    S = np.zeros((12, V4, 4, 3), dtype=np.complex128)
    for be in range(4):
        for b in range(3):
            for al in range(4):
                S[3 * be + b, :, al, b] = Pp[al, be]
    Sd = torch.from_numpy(S).cuda()
    V3 = V4 // dims[3]
    c_plus = ctx.mdwf_nucleon_2pt(Sd, Sd, Sd, Pp).cpu().numpy()
    c_minus = ctx.mdwf_nucleon_2pt(Sd, Sd, Sd, 0.5 * (np.eye(4) - gt)).cpu().numpy()
    assert np.allclose(c_plus, 36.0 * V3, atol=1e-10)
    assert np.allclose(c_minus, 0.0, atol=1e-10)


def test_fh_chain_small():
    """configs[3] scaled to 4^3x8, Ls=4: smeared source -> S ; eta_seq = gamma_z gamma_5 S on all t ; S_FH ;
    C(t) with and without the insertion; every stage against the oracle chain."""
    import paper_1810_01609_b200 as mdwf
    dims, Ls, mf = (4, 4, 4, 8), 4, 0.1
    cfg = synth.CONFIGS[4]
    p = oracle.Params(dims=dims, Ls=Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=mf, bc=cfg.bc)
    U = synth.gauge_field(dims, cfg.eps, synth.seed_for(4, 1))
    ctx = mdwf.Context(dims, Ls, cfg.M5, cfg.b5, cfg.c5, mf, bc=cfg.bc)
    ctx.mdwf_load_gauge(U.cuda(), 64, 18)
    ctx.mdwf_load_gauge(U.cuda(), 16, 12)
    eta = synth.gaussian_smeared_sources_4d(dims, width=3.0)
    kw = dict(tol=1e-10, inner_prec=16, recon=12, src_kind=1, out_kind=1)
    S, r1 = ctx.mdwf_solve(eta.cuda(), **kw)
    G = oracle.gamma(2) @ oracle.gamma(4)
    seq = ctx.mdwf_seq_source(S, G)
    SFH, r2 = ctx.mdwf_solve(seq, **kw)
    assert r1.status == 0 and r2.status == 0
    Un = U.numpy()

    def oprop(src):
        x, _, _ = oracle.solve_eo(p, Un, oracle.wall_inject(p, Un, src), tol=1e-12)
        return oracle.wall_project(p, x)
    So = oprop(eta.numpy())
    SFHo = oprop(oracle.seq_source(dims, So, G))
    assert rel(S.cpu().numpy(), So) <= 1e-6
    assert rel(SFH.cpu().numpy(), SFHo) <= 1e-6
    P = 0.5 * (np.eye(4) + oracle.gamma(3))
    c0 = ctx.mdwf_nucleon_2pt(S, S, S, P).cpu().numpy()
    cfh = (ctx.mdwf_nucleon_2pt(SFH, S, S, P) + ctx.mdwf_nucleon_2pt(S, S, SFH, P) - ctx.mdwf_nucleon_2pt(S, SFH, S, P)).cpu().numpy()
    c0o = oracle.nucleon_2pt(dims, So, So, So, P)
    cfho = (oracle.nucleon_2pt(dims, SFHo, So, So, P) + oracle.nucleon_2pt(dims, So, So, SFHo, P) - oracle.nucleon_2pt(dims, So, SFHo, So, P))
    assert rel(c0, c0o) <= 1e-5 and rel(cfh, cfho) <= 1e-5


def test_static_limit_matches_golden_file():
    import os
    import paper_1810_01609_b200 as mdwf
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "static_nucleon.txt")) as f:
        for line in f:
            if not line.startswith("#") and line.strip():
                k, v = line.split()
                vals[k] = float(v)
    dims = (2, 2, 4, 2)
    ctx = mdwf.Context(dims, 2, 1.3, 1.5, 0.5, 0.1)
    V4 = int(np.prod(dims))
    gt = oracle.gamma(3)
    Pp, Pm = 0.5 * (np.eye(4) + gt), 0.5 * (np.eye(4) - gt)
    S = np.zeros((12, V4, 4, 3), dtype=np.complex128)
    for be in range(4):
        for b in range(3):
            for al in range(4):
                S[3 * be + b, :, al, b] = Pp[al, be]
    Sd = torch.from_numpy(S).cuda()
    V3 = V4 // dims[3]
    assert np.allclose(ctx.mdwf_nucleon_2pt(Sd, Sd, Sd, Pp).cpu().numpy(), vals["(1+gamma_t)/2"] * V3, atol=1e-10)
    assert np.allclose(ctx.mdwf_nucleon_2pt(Sd, Sd, Sd, Pm).cpu().numpy(), vals["(1-gamma_t)/2"] * V3, atol=1e-10)


@pytest.mark.parametrize("prec,tol", [(64, 0.0), (32, 1e-7), (16, 6e-4)])
def test_pack_unpack_round_trip(prec, tol):
    """layout round trip: canonical -> packed -> canonical; exact in fp64, storage rounding otherwise.
    Ragged shape: N5h = 3*5*... not a multiple of the 32-site storage block."""
    import paper_1810_01609_b200 as mdwf
    dims, Ls = (6, 2, 2, 4), 5
    ctx = mdwf.Context(dims, Ls, 1.3, 1.5, 0.5, 0.1)
    Vh = int(np.prod(dims)) // 2
    src = crandn((3, Ls, Vh, 4, 3), 4300).cuda()
    f = ctx.mdwf_field_create(prec, 3)
    f.mdwf_field_pack(src)
    out = torch.zeros_like(src)
    f.mdwf_field_unpack(out)
    err = float((out - src).abs().max() / src.abs().max())
    assert err <= tol, err

"""Oracle pins for the Feynman-Hellmann chain and the nucleon contraction (SURVEY.md 8(c) O3, O4,
A14, A15) and for the solver variants on config 1 (O2).  CPU only."""
import numpy as np
import pytest

import oracle
import synth

RNG = np.random.default_rng(999)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def rel(a, b):
    return np.linalg.norm((a - b).reshape(-1)) / np.linalg.norm(b.reshape(-1))


def _dense(apply, n):
    M = np.empty((n, n), dtype=complex)
    e = np.zeros(n, dtype=complex)
    for j in range(n):
        e[:] = 0
        e[j] = 1
        M[:, j] = apply(e).reshape(-1)
    return M


G = [oracle.gamma(m) for m in range(4)]
G5 = oracle.gamma(4)
CG5 = G[1] @ G[3] @ G5
P_UNPOL = 0.5 * (np.eye(4) + G[3])
P_NEG = 0.5 * (np.eye(4) - G[3])
P_POL = 0.25 * (np.eye(4) + G[3]) @ (np.eye(4) + 1j * G[0] @ G[1])


def test_Cgamma5_matrix_value():
    # SURVEY 8 Notation prints C gamma5 explicitly
    assert np.allclose(CG5, np.array([[0, -1, 0, 0], [1, 0, 0, 0], [0, 0, 0, -1], [0, 0, 1, 0]]))
    Gt = G[3] @ CG5.conj().T @ G[3]
    assert np.allclose(Gt, -CG5)


# ------------------------------------------------------------------ FH chain: S_FH = S Gamma S (A14)
def test_sequential_propagator_is_S_Gamma_S_dense():
    dims, Ls = (2, 2, 2, 2), 2
    p = oracle.Params(dims=dims, Ls=Ls, M5=1.3, b5=1.5, c5=0.5, mf=0.1)
    U = synth.gauge_field(dims, 0.3, 3).numpy()
    n4, shp5 = p.V4 * 12, (1, Ls, p.V4, 4, 3)
    n5 = int(np.prod(shp5))
    D5inv = np.linalg.inv(_dense(lambda e: oracle.D(p, U, e.reshape(shp5)), n5))

    def prop(eta):                       # eta [ncol][V4][4][3] -> S eta, dense 5D solve
        b5 = oracle.wall_inject(p, U, eta)
        psi = (D5inv @ b5.reshape(eta.shape[0], n5).T).T.reshape(eta.shape[0], Ls, p.V4, 4, 3)
        return oracle.wall_project(p, psi)

    S4 = prop(np.eye(n4, dtype=complex).reshape(n4, p.V4, 4, 3)).reshape(n4, n4).T
    Gam = G[2] @ G5                                                       # gamma_z gamma5
    Gbig = np.kron(np.eye(p.V4), np.kron(Gam, np.eye(3)))
    eta = synth.point_sources_4d(dims).numpy()                            # 12 columns at the origin
    S = prop(eta)
    seq = oracle.seq_source(dims, S, Gam)
    assert rel(seq.reshape(12, n4).T, Gbig @ S.reshape(12, n4).T) < 1e-14
    Sfh = prop(seq)
    ref = S4 @ Gbig @ S4 @ eta.reshape(12, n4).T
    assert rel(Sfh.reshape(12, n4).T, ref) < 1e-11
    # time window: only t = 1 inserted
    seq1 = oracle.seq_source(dims, S, Gam, 1, 1)
    tmask = np.kron(np.diag((np.arange(p.V4) // (p.V4 // dims[3]) == 1).astype(float)), np.eye(12))
    assert rel(seq1.reshape(12, n4).T, tmask @ Gbig @ S.reshape(12, n4).T) < 1e-14


# ------------------------------------------------------------------ nucleon contraction (A15)
def _eps():
    e = np.zeros((3, 3, 3))
    for a, b, c in [(0, 1, 2), (1, 2, 0), (2, 0, 1)]:
        e[a, b, c] = 1
        e[a, c, b] = -1
    return e


def _as5(S, V4):
    """prop[col=3*beta+b][x][alpha][a] -> S[x, alpha, a, beta, b]"""
    return S.reshape(4, 3, V4, 4, 3).transpose(2, 3, 4, 0, 1)


def _nucleon_einsum(dims, Su1, Sd, Su2, P, t0=0):
    V4 = int(np.prod(dims))
    T = dims[3]
    e = _eps()
    Gm = CG5
    Gt = G[3] @ Gm.conj().T @ G[3]
    u1, d, u2 = _as5(Su1, V4), _as5(Sd, V4), _as5(Su2, V4)
    # Q[x, alpha, b, alpha', b'] = G[alpha,beta] Sd[x,beta,b,beta',b'] Gt[beta',alpha']
    Q = np.einsum("AB,xBbCc,CD->xAbDc", Gm, d, Gt)
    direct = np.einsum("abc,def,xAbDe,xAaDd,GH,xHcGf->x", e, e, Q, u1, P, u2, optimize=True)
    exch = np.einsum("abc,def,xAbDe,xAaGf,GH,xHcDd->x", e, e, Q, u1, P, u2, optimize=True)
    site = (direct - exch).reshape(T, -1).sum(1)
    return np.roll(site, -t0)


def test_nucleon_matches_independent_einsum_form():
    dims = (2, 2, 2, 4)
    V4 = int(np.prod(dims))
    Su1, Sd, Su2 = crandn(12, V4, 4, 3), crandn(12, V4, 4, 3), crandn(12, V4, 4, 3)
    for P in (P_UNPOL, P_POL):
        for t0 in (0, 3):
            c = oracle.nucleon_2pt(dims, Su1, Sd, Su2, P, t0=t0)
            assert rel(c, _nucleon_einsum(dims, Su1, Sd, Su2, P, t0)) < 1e-13


def test_nucleon_static_quark_limit_closed_form():
    """S = delta_ab M per site: colour sums give +6 (direct) and -6 (exchange), so per site
    C = 6 tr[(G M Gt) M^T] tr[P M] + 6 tr[(G M Gt)^T M P M]  (derived by hand from C-def)."""
    dims = (2, 2, 2, 2)
    V4 = 16
    M = P_UNPOL
    S = np.zeros((12, V4, 4, 3), dtype=complex)
    for be in range(4):
        for b in range(3):
            S[3 * be + b, :, :, b] = M[:, be]
    Gt = G[3] @ CG5.conj().T @ G[3]
    K = CG5 @ M @ Gt
    for P, expect in ((P_UNPOL, 36.0), (P_NEG, 0.0)):
        site = 6 * np.trace(K @ M.T) * np.trace(P @ M) + 6 * np.trace(K.T @ M @ P @ M)
        assert abs(site - expect) < 1e-13           # +36 and 0
        c = oracle.nucleon_2pt(dims, S, S, S, P)
        assert np.allclose(c, site * (V4 // dims[3]))


def test_nucleon_gauge_invariance_scaling_and_fh_linearity():
    dims = (2, 2, 2, 4)
    V4 = int(np.prod(dims))
    S = [crandn(12, V4, 4, 3) for _ in range(3)]
    c0 = oracle.nucleon_2pt(dims, *S, P_UNPOL)
    # S(x) -> Gx S(x) G0^dag for all three slots leaves C unchanged (det = 1)
    Gx = synth.random_su3_field(V4, 5).numpy()
    G0 = Gx[0]
    St = []
    for s in S:
        s5 = _as5(s, V4)
        r = np.einsum("xac,xAcBd,bd->xAaBb", Gx, s5, G0.conj())
        St.append(np.ascontiguousarray(r.transpose(3, 4, 0, 1, 2)).reshape(12, V4, 4, 3))
    assert rel(oracle.nucleon_2pt(dims, *St, P_UNPOL), c0) < 1e-12
    # cubic: C(2S) = 8 C
    assert rel(oracle.nucleon_2pt(dims, *[2 * s for s in S], P_UNPOL), 8 * c0) < 1e-14
    # linear in each slot separately (the Feynman-Hellmann terms are first derivatives)
    F = crandn(12, V4, 4, 3)
    lam = 0.37
    for slot in range(3):
        a = list(S)
        a[slot] = S[slot] + lam * F
        b = list(S)
        b[slot] = F
        assert rel(oracle.nucleon_2pt(dims, *a, P_POL),
                   oracle.nucleon_2pt(dims, *S, P_POL) + lam * oracle.nucleon_2pt(dims, *b, P_POL)) < 1e-12


# ------------------------------------------------------------------ solver variants on config 1 (O2)
def test_config1_solver_variants_agree_and_manufactured_solution():
    cfg = synth.CONFIGS[1]
    p = oracle.Params(dims=cfg.dims, Ls=cfg.Ls, M5=cfg.M5, b5=cfg.b5, c5=cfg.c5, mf=cfg.mf, bc=cfg.bc)
    U = synth.gauge_field(cfg.dims, cfg.eps, synth.seed_for(1, 1)).numpy()
    xstar = synth.gaussian_spinor(cfg.dims, cfg.Ls, 1, synth.seed_for(1, 50)).numpy()
    b = oracle.D(p, U, xstar)                         # manufactured: the solution is known exactly
    xa, ita, _ = oracle.solve_full(p, U, b, tol=1e-13)
    assert rel(xa, xstar) < 1e-10
    for sym in (False, True):
        xb, itb, _ = oracle.solve_eo(p, U, b, parity=0, symmetric=sym, tol=1e-13)
        assert rel(xb, xstar) < 1e-10
        assert itb[0] < ita[0]                        # preconditioning helps (SURVEY: 64 vs 165 at 1e-10)
        assert oracle.true_residual(p, U, xb, b)[0] < 1e-11

"""More oracle pins (SURVEY.md 8(c) pins 6-13): an independently coded Shamir operator, dense brute
force with library LU, the closed form of M5^-1, the 4D overlap identity, input properties, the
Feynman-Hellmann chain and the nucleon contraction.  CPU only."""
import numpy as np
import pytest

import oracle
import synth

RNG = np.random.default_rng(4321)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def rel(a, b):
    return np.linalg.norm((a - b).reshape(-1)) / np.linalg.norm(b.reshape(-1))


def make(dims=(4, 4, 4, 4), Ls=4, b5=1.5, c5=0.5, mf=0.1, M5=1.3, bc=(1, 1, 1, -1), eps=0.3, seed=11):
    p = oracle.Params(dims=tuple(dims), Ls=Ls, M5=M5, b5=b5, c5=c5, mf=mf, bc=tuple(bc))
    U = synth.gauge_field(dims, eps, seed).numpy()
    return p, U


# ------------------------------------------------------------------ pin 6: Shamir limit, independent code
# Independent implementation: vectorised numpy on [T,Z,Y,X] arrays with np.roll, gamma matrices
# typed here from the Pauli-block form of the DeGrand-Rossi basis:
#   gamma_k = [[0, i s_k'],[-i s_k', 0]] with (s_x', s_y', s_z') = (s_x, -s_y, s_z);  gamma_t = [[0,1],[1,0]]
_sx = np.array([[0, 1], [1, 0]], dtype=complex)
_sy = np.array([[0, -1j], [1j, 0]], dtype=complex)
_sz = np.array([[1, 0], [0, -1]], dtype=complex)
_Z2 = np.zeros((2, 2), dtype=complex)
_G = [np.block([[_Z2, 1j * s], [-1j * s, _Z2]]) for s in (_sx, -_sy, _sz)] + [np.block([[_Z2, np.eye(2)], [np.eye(2), _Z2]])]


def test_typed_gammas_agree_with_oracle():
    for m in range(4):
        assert np.allclose(_G[m], oracle.gamma(m))


def _wilson_indep(dims, bc, U, psi, M5):
    """D_W psi = (4 - M5) psi - 1/2 sum_mu [(1-g)U(x)psi(x+mu) + (1+g)U(x-mu)^dag psi(x-mu)], roll-based."""
    X, Y, Z, T = dims
    ax = {0: 3, 1: 2, 2: 1, 3: 0}                      # array axes of [T,Z,Y,X]
    f = psi.reshape(T, Z, Y, X, 4, 3)
    out = (4.0 - M5) * f
    for mu in range(4):
        Um = U[mu].reshape(T, Z, Y, X, 3, 3)
        a = ax[mu]
        Lm = dims[mu]
        idx = np.arange(Lm).reshape([-1 if i == a else 1 for i in range(4)] + [1, 1])
        fwd = np.roll(f, -1, axis=a) * np.where(idx == Lm - 1, bc[mu], 1)          # psi(x+mu), wrapped hop gets bc
        Ufwd = np.einsum("...ab,...sb->...sa", Um, fwd)
        UdagF = np.einsum("...ba,...sb->...sa", Um.conj(), f)                       # U(x)^dag psi(x), then shift to x+mu
        bwd = np.roll(UdagF, 1, axis=a) * np.where(idx == 0, bc[mu], 1)
        out = out - 0.5 * (Ufwd - np.einsum("st,...tc->...sc", _G[mu], Ufwd))
        out = out - 0.5 * (bwd + np.einsum("st,...tc->...sc", _G[mu], bwd))
    return out.reshape(-1, 4, 3)


def _shamir_indep(p, U, psi):
    """(D psi)_s = (D_W + 1) psi_s - P- psi_{s+1} - P+ psi_{s-1}, +mf on the wraps."""
    Pp = np.diag([1, 1, 0, 0]).astype(complex)
    Pm = np.diag([0, 0, 1, 1]).astype(complex)
    out = np.empty_like(psi)
    Ls = p.Ls
    for s in range(Ls):
        up = psi[(s + 1) % Ls] * (-p.mf if s == Ls - 1 else 1.0)
        dn = psi[(s - 1) % Ls] * (-p.mf if s == 0 else 1.0)
        out[s] = _wilson_indep(p.dims, p.bc, U, psi[s], p.M5) + psi[s] \
            - np.einsum("st,xtc->xsc", Pm, up) - np.einsum("st,xtc->xsc", Pp, dn)
    return out


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 6, 2)])
def test_shamir_limit_vs_independent_operator(dims):
    p, U = make(dims=dims, Ls=5, b5=1.0, c5=0.0, mf=0.07)
    psi = crandn(p.Ls, p.V4, 4, 3)
    assert rel(oracle.D(p, U, psi[None])[0], _shamir_indep(p, U, psi)) < 1e-14
    # and the Wilson operator alone, including an extent-2 direction (A21)
    p1 = oracle.Params(dims=dims, Ls=1, M5=1.3, b5=1, c5=0, mf=0, bc=p.bc)
    assert rel(oracle.wilson(p1, U, psi[:1])[0], _wilson_indep(dims, p.bc, U, psi[0], 1.3)) < 1e-14


def test_moebius_equals_textbook_combination_of_independent_wilson():
    """D = (b5 D_W + 1) + (c5 D_W - 1) L with D_W from the independent code and L typed here."""
    p, U = make(Ls=4)
    psi = crandn(p.Ls, p.V4, 4, 3)
    Lpsi = np.empty_like(psi)
    for s in range(p.Ls):
        up = psi[(s + 1) % p.Ls] * (-p.mf if s == p.Ls - 1 else 1.0)
        dn = psi[(s - 1) % p.Ls] * (-p.mf if s == 0 else 1.0)
        Lpsi[s, :, :2] = dn[:, :2]
        Lpsi[s, :, 2:] = up[:, 2:]
    ref = np.empty_like(psi)
    for s in range(p.Ls):
        ref[s] = p.b5 * _wilson_indep(p.dims, p.bc, U, psi[s], p.M5) + psi[s] \
            + p.c5 * _wilson_indep(p.dims, p.bc, U, Lpsi[s], p.M5) - Lpsi[s]
    assert rel(oracle.D(p, U, psi[None])[0], ref) < 1e-14


# ------------------------------------------------------------------ pin 8: M5 M5^-1 = 1, closed form
@pytest.mark.parametrize("Ls", [1, 2, 4, 8, 12])
def test_m5inv_closed_form_and_identity(Ls):
    p = oracle.Params(dims=(2, 2, 2, 2), Ls=Ls, M5=1.3, b5=1.5, c5=0.5, mf=0.05)
    psi = crandn(2, Ls, p.V4, 4, 3)
    for dg in (False, True):
        assert rel(oracle.M5op(p, oracle.M5inv(p, psi, dg), dg), psi) < 1e-14
        assert rel(oracle.M5inv(p, oracle.M5op(p, psi, dg), dg), psi) < 1e-14
    # closed form (SURVEY 8 Notation): kappa = -d/a
    a, d, mf = p.a, p.d, p.mf
    k = -d / a
    Mp = np.zeros((Ls, Ls))
    Mm = np.zeros((Ls, Ls))
    for s in range(Ls):
        for t in range(Ls):
            Mp[s, t] = k ** ((s - t) % Ls) * (1.0 if s >= t else -mf) / (a * (1 + mf * k ** Ls))
            Mm[s, t] = k ** ((t - s) % Ls) * (1.0 if t >= s else -mf) / (a * (1 + mf * k ** Ls))
    ref = np.empty_like(psi)
    ref[:, :, :, :2] = np.einsum("st,rtxjc->rsxjc", Mp, psi[:, :, :, :2])
    ref[:, :, :, 2:] = np.einsum("st,rtxjc->rsxjc", Mm, psi[:, :, :, 2:])
    assert rel(oracle.M5inv(p, psi), ref) < 1e-14


# ------------------------------------------------------------------ pin 7: dense brute force on 2^4 x Ls=2
def _dense(apply, n):
    M = np.empty((n, n), dtype=complex)
    e = np.zeros(n, dtype=complex)
    for j in range(n):
        e[:] = 0
        e[j] = 1
        M[:, j] = apply(e).reshape(-1)
    return M


def test_dense_brute_force_2x2x2x2_Ls2():
    p, U = make(dims=(2, 2, 2, 2), Ls=2, mf=0.1)
    shp = (1, p.Ls, p.V4, 4, 3)
    n = int(np.prod(shp))
    assert n == 384
    Dm = _dense(lambda e: oracle.D(p, U, e.reshape(shp)), n)
    Dd = _dense(lambda e: oracle.D(p, U, e.reshape(shp), dagger=True), n)
    assert np.allclose(Dd, Dm.conj().T, atol=1e-13)
    b = crandn(*shp)
    x_lu = np.linalg.solve(Dm, b.reshape(-1)).reshape(shp)
    xa, ita, _ = oracle.solve_full(p, U, b, tol=1e-13)
    assert rel(xa, x_lu) < 1e-11
    for parity in (0, 1):
        for sym in (False, True):
            xb, itb, _ = oracle.solve_eo(p, U, b, parity=parity, symmetric=sym, tol=1e-13)
            assert rel(xb, x_lu) < 1e-11
            assert oracle.true_residual(p, U, xb, b)[0] < 1e-11
    # Schur complement identity: Dhat = D_pp - D_ppbar D_pbarpbar^-1 D_pbarp from the dense matrix
    par = np.broadcast_to(oracle.parity_of_sites(p.dims)[None, None, :, None, None], shp).reshape(-1)
    for parity in (0, 1):
        ip, iq = np.nonzero(par == parity)[0], np.nonzero(par != parity)[0]
        S = Dm[np.ix_(ip, ip)] - Dm[np.ix_(ip, iq)] @ np.linalg.solve(Dm[np.ix_(iq, iq)], Dm[np.ix_(iq, ip)])
        v = oracle.mask(p, crandn(*shp), parity)
        ref = np.zeros(n, dtype=complex)
        ref[ip] = S @ v.reshape(-1)[ip]
        assert rel(oracle.schur(p, U, v, parity, False, False).reshape(-1), ref) < 1e-13
        # prepared source and reconstruction (SURVEY 8 Even-odd form)
        bh = oracle.prepare_source(p, U, b, parity).reshape(-1)
        refb = np.zeros(n, dtype=complex)
        refb[ip] = b.reshape(-1)[ip] - Dm[np.ix_(ip, iq)] @ np.linalg.solve(Dm[np.ix_(iq, iq)], b.reshape(-1)[iq])
        assert rel(bh, refb) < 1e-13
        xp = oracle.mask(p, x_lu, parity)
        assert rel(oracle.reconstruct(p, U, xp, b, parity), x_lu) < 1e-13


# ------------------------------------------------------------------ pin 9: 4D overlap identity (O3, A3, A13)
def _matfun_eps(h, Ls):
    w, V = np.linalg.eig(h)
    e = ((1 + w) ** Ls - (1 - w) ** Ls) / ((1 + w) ** Ls + (1 - w) ** Ls)
    return V @ np.diag(e) @ np.linalg.inv(V)


@pytest.mark.parametrize("Ls", [2, 4])
def test_overlap_identity_for_4d_propagator(Ls):
    """S eta = P- psi_0 + P+ psi_{Ls-1}, D psi = -D_-(P+eta@0 (+) P-eta@Ls-1) satisfies
    [1 + (1-mf) S]^-1 = D_ov(mf) = 1/2[(1+mf) + (1-mf) g5 eps_Ls(H_M)],
    H_M = g5 (b5+c5) D_W [2 + (b5-c5) D_W]^-1."""
    p, U = make(dims=(2, 2, 2, 2), Ls=Ls, mf=0.1)
    n4 = p.V4 * 12
    p1 = oracle.Params(dims=p.dims, Ls=1, M5=p.M5, b5=1, c5=0, mf=0, bc=p.bc)
    DW = _dense(lambda e: oracle.wilson(p1, U, e.reshape(1, p.V4, 4, 3)), n4)
    g5 = np.kron(np.eye(p.V4), np.kron(np.diag([1, 1, -1, -1]), np.eye(3)))
    HM = g5 @ ((p.b5 + p.c5) * DW) @ np.linalg.inv(2 * np.eye(n4) + (p.b5 - p.c5) * DW)
    Dov = 0.5 * ((1 + p.mf) * np.eye(n4) + (1 - p.mf) * g5 @ _matfun_eps(HM, Ls))
    # dense 5D operator and the 4D propagator through the oracle's inject / project
    shp5 = (1, Ls, p.V4, 4, 3)
    n5 = int(np.prod(shp5))
    D5 = _dense(lambda e: oracle.D(p, U, e.reshape(shp5)), n5)
    eta = np.eye(n4, dtype=complex).reshape(n4, p.V4, 4, 3)
    b5 = oracle.wall_inject(p, U, eta)                                   # [n4][Ls][V4][4][3]
    psi = np.linalg.solve(D5, b5.reshape(n4, n5).T).T.reshape(n4, Ls, p.V4, 4, 3)
    S = oracle.wall_project(p, psi).reshape(n4, n4).T                    # S[:, j] = S eta_j
    lhs = np.linalg.inv(np.eye(n4) + (1 - p.mf) * S)
    assert np.abs(lhs - Dov).max() < 1e-12
    # S is gamma5-hermitian
    assert np.abs(g5 @ S @ g5 - S.conj().T).max() < 1e-12


# ------------------------------------------------------------------ pin 10: input properties
def test_links_are_su3_and_plaquette_matches_c_eps_4():
    dims = (8, 8, 8, 8)
    U = synth.gauge_field(dims, 0.306, 5).numpy()
    UUd = np.einsum("mxab,mxcb->mxac", U, U.conj())
    assert np.abs(UUd - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-13
    X, Y, Z, T = dims
    x4 = np.arange(X * Y * Z * T)
    co = [x4 % X, (x4 // X) % Y, (x4 // (X * Y)) % Z, x4 // (X * Y * Z)]
    st = [1, X, X * Y, X * Y * Z]
    nb = [x4 + st[m] * (((co[m] + 1) % dims[m]) - co[m]) for m in range(4)]
    plaq = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P = np.einsum("xab,xbc,xdc,xed->xae", U[mu], U[nu][nb[mu]], U[mu][nb[nu]].conj(), U[nu].conj())
            plaq += np.einsum("xaa->x", P).real.mean() / 3.0
    plaq /= 6.0
    c = synth.mean_trace(synth.gauge_field(dims, 0.306, 5))
    assert abs(plaq - c ** 4) < 5e-3
    assert abs(plaq - 0.600) < 0.01

"""Pins for the CPU oracle (SURVEY.md 8(c) "Pins with no implementation to compare against").

None of these compares the oracle with itself or with a stored oracle output: each one checks a
value or identity that the physics / mathematics fixes (closed forms, symmetries, an independently
coded textbook operator, dense library solves).  CPU only (-m "not gpu").
"""
import numpy as np
import pytest

import oracle
import synth

RNG = np.random.default_rng(1234)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def vdot(a, b):
    return np.vdot(a.reshape(-1), b.reshape(-1))


def rel(a, b):
    return np.linalg.norm((a - b).reshape(-1)) / np.linalg.norm(b.reshape(-1))


def make(dims=(4, 4, 4, 4), Ls=4, b5=1.5, c5=0.5, mf=0.1, M5=1.3, bc=(1, 1, 1, -1), eps=0.3, seed=11):
    p = oracle.Params(dims=tuple(dims), Ls=Ls, M5=M5, b5=b5, c5=c5, mf=mf, bc=tuple(bc))
    U = synth.gauge_field(dims, eps, seed).numpy()
    return p, U


# ----------------------------------------------------------------------------- gamma algebra (A2)
def test_gamma_clifford_hermitian_gamma5():
    g = [oracle.gamma(m) for m in range(4)]
    g5 = oracle.gamma(4)
    for m in range(4):
        assert np.allclose(g[m], g[m].conj().T)
        for n in range(4):
            anti = g[m] @ g[n] + g[n] @ g[m]
            assert np.allclose(anti, 2.0 * np.eye(4) * (m == n))
    assert np.allclose(g[0] @ g[1] @ g[2] @ g[3], g5)
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))
    C = g[1] @ g[3]
    for m in range(4):
        assert np.allclose(C @ g[m] @ np.linalg.inv(C), -g[m].T)
    # spin-up projector has rank 1; Sigma_z = i gx gy is diagonal (A15 / O4)
    Sz = 1j * g[0] @ g[1]
    assert np.allclose(Sz, np.diag([1, -1, 1, -1]))
    Ppol = 0.25 * (np.eye(4) + g[3]) @ (np.eye(4) + Sz)
    assert np.linalg.matrix_rank(Ppol) == 1


# ----------------------------------------------------------------------------- free field (pin 1)
@pytest.mark.parametrize("dims,bc", [((4, 2, 6, 4), (1, 1, 1, -1)), ((2, 4, 4, 6), (-1, 1, -1, 1))])
def test_free_field_plane_wave_spectrum(dims, bc):
    """U = 1: D_W e^{ipx}u = [(4-M5-sum cos p) + i sum g_mu sin p] e^{ipx}u, so for ANY spinor u
    (D_W - c)^2 psi = -(sum sin^2 p) psi with c = 4 - M5 - sum cos p; eigenvalues c +- i sqrt(sum sin^2)."""
    M5 = 1.3
    p = oracle.Params(dims=dims, Ls=1, M5=M5, b5=1.0, c5=0.0, mf=0.0, bc=bc)
    U = synth.unit_gauge(dims).numpy()
    X, Y, Z, T = dims
    x4 = np.arange(p.V4)
    co = [x4 % X, (x4 // X) % Y, (x4 // (X * Y)) % Z, x4 // (X * Y * Z)]
    for n in [(1, 0, 2, 1), (0, 1, 1, 3), (1, 1, 0, 0)]:
        mom = [2 * np.pi * (n[m] + (0.5 if bc[m] == -1 else 0.0)) / dims[m] for m in range(4)]
        phase = np.exp(1j * sum(mom[m] * co[m] for m in range(4)))
        u = crandn(4, 3)
        psi = (phase[:, None, None] * u[None])[None]          # [1][V4][4][3]
        c = 4 - M5 - sum(np.cos(mom))
        s2 = sum(np.sin(mom) ** 2)
        w1 = oracle.wilson(p, U, psi) - c * psi
        w2 = oracle.wilson(p, U, w1) - c * w1
        assert rel(w2, -s2 * psi) < 1e-13
        # and the eigenvectors themselves: u_pm = (sqrt(s2) +- sum g sin p) v  has eigenvalue c +- i sqrt(s2)
        gs = sum(np.sin(mom[m]) * oracle.gamma(m) for m in range(4))
        for sign in (+1, -1):
            ue = (np.sqrt(s2) * np.eye(4) + sign * gs) @ u
            pe = (phase[:, None, None] * ue[None])[None]
            assert rel(oracle.wilson(p, U, pe), (c + sign * 1j * np.sqrt(s2)) * pe) < 1e-13


# ----------------------------------------------------------------------------- gamma5-hermiticity (pin 2)
def test_gamma5_hermiticity_and_adjoint_of_wilson():
    p, U = make(dims=(4, 2, 4, 6), Ls=1)
    psi, chi = crandn(1, p.V4, 4, 3), crandn(1, p.V4, 4, 3)
    g5 = np.array([1, 1, -1, -1])[None, None, :, None]
    lhs = g5 * oracle.wilson(p, U, g5 * psi)
    assert rel(lhs, oracle.wilson(p, U, psi, dagger=True)) < 1e-14
    assert abs(vdot(chi, oracle.wilson(p, U, psi)) - vdot(oracle.wilson(p, U, chi, dagger=True), psi)) < 1e-11
    assert rel(g5 * oracle.hop(p, U, g5 * psi), oracle.hop(p, U, psi, dagger=True)) < 1e-14


# ----------------------------------------------------------------------------- adjoints (pin 4)
@pytest.mark.parametrize("name", ["H", "L", "A", "M5", "M5inv", "D", "Dhat0", "Dhat1", "Mhat0", "Mhat1", "Dminus"])
def test_adjoint_consistency(name):
    p, U = make()
    ops = {
        "H": lambda v, dg: oracle.hop(p, U, v, dagger=dg),
        "L": lambda v, dg: oracle.L(p, v, dagger=dg),
        "A": lambda v, dg: oracle.M4pre(p, v, dagger=dg),
        "M5": lambda v, dg: oracle.M5op(p, v, dagger=dg),
        "M5inv": lambda v, dg: oracle.M5inv(p, v, dagger=dg),
        "D": lambda v, dg: oracle.D(p, U, v, dagger=dg),
        "Dminus": lambda v, dg: oracle.Dminus(p, U, v, dagger=dg),
        "Dhat0": lambda v, dg: oracle.schur(p, U, v, 0, dg, False),
        "Dhat1": lambda v, dg: oracle.schur(p, U, v, 1, dg, False),
        "Mhat0": lambda v, dg: oracle.schur(p, U, v, 0, dg, True),
        "Mhat1": lambda v, dg: oracle.schur(p, U, v, 1, dg, True),
    }
    op = ops[name]
    psi, chi = crandn(1, p.Ls, p.V4, 4, 3), crandn(1, p.Ls, p.V4, 4, 3)
    if name[:4] in ("Dhat", "Mhat"):
        par = int(name[-1])
        psi, chi = oracle.mask(p, psi, par), oracle.mask(p, chi, par)
    a = vdot(chi, op(psi, False))
    b = vdot(op(chi, True), psi)
    assert abs(a - b) / abs(a) < 1e-13


# ----------------------------------------------------------------------------- A8: reflection-gamma5 hermiticity
def _Gamma5(p, v):
    g5 = np.array([1, 1, -1, -1])[None, None, None, :, None]
    return g5 * v[:, ::-1]


def test_reflection_gamma5_hermiticity():
    # c5 = 0 (any b5): Gamma5 D Gamma5 = D^dag
    p, U = make(b5=1.7, c5=0.0)
    psi = crandn(1, p.Ls, p.V4, 4, 3)
    assert rel(_Gamma5(p, oracle.D(p, U, _Gamma5(p, psi))), oracle.D(p, U, psi, dagger=True)) < 1e-14
    # c5 != 0: it FAILS for D, but holds for D D_- (A8)
    p, U = make(b5=1.5, c5=0.5)
    assert rel(_Gamma5(p, oracle.D(p, U, _Gamma5(p, psi))), oracle.D(p, U, psi, dagger=True)) > 1e-3
    lhs = _Gamma5(p, oracle.D(p, U, oracle.Dminus(p, U, _Gamma5(p, psi))))
    rhs = oracle.Dminus(p, U, oracle.D(p, U, psi, dagger=True), dagger=True)
    assert rel(lhs, rhs) < 1e-14


# ----------------------------------------------------------------------------- gauge covariance (pin 5)
def _transform(dims, U, G):
    X, Y, Z, T = dims
    V4 = X * Y * Z * T
    x4 = np.arange(V4)
    co = [x4 % X, (x4 // X) % Y, (x4 // (X * Y)) % Z, x4 // (X * Y * Z)]
    st = [1, X, X * Y, X * Y * Z]
    Up = np.empty_like(U)
    for mu in range(4):
        nb = x4 + st[mu] * (((co[mu] + 1) % dims[mu]) - co[mu])
        Up[mu] = np.einsum("xab,xbc,xdc->xad", G, U[mu], G[nb].conj())
    return Up


def test_gauge_covariance():
    p, U = make()
    G = synth.random_su3_field(p.V4, 77).numpy()
    Up = _transform(p.dims, U, G)
    psi = crandn(1, p.Ls, p.V4, 4, 3)
    gpsi = np.einsum("xab,rsxjb->rsxja", G, psi)
    for f in (lambda UU, v: oracle.D(p, UU, v), lambda UU, v: oracle.D(p, UU, v, dagger=True),
              lambda UU, v: oracle.schur(p, UU, v, 0, False, False), lambda UU, v: oracle.schur(p, UU, v, 1, True, True)):
        lhs = f(Up, gpsi)
        rhs = np.einsum("xab,rsxjb->rsxja", G, f(U, psi))
        assert rel(lhs, rhs) < 1e-13

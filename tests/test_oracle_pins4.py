"""Oracle pins for the fuller Feynman-Hellmann workload (R25): the
gauge-covariant Gaussian smearing psi' = (1 + sigma^2/(4N) Lap)^N psi and the effective derivative.  CPU only.  Each pin
is something other than the oracle's own formula: the free-field Fourier symbol, the exact second moment of the random
walk, gauge covariance, and literal per-site index loops on a tiny lattice."""
import numpy as np

import oracle
import synth

RNG = np.random.default_rng(4242)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def rel(a, b):
    return np.linalg.norm((a - b).reshape(-1)) / np.linalg.norm(b.reshape(-1))


def test_free_field_symbol():
    """unit links, periodic: (1 + a Lap)^N is diagonal in Fourier space with symbol (1 + a sum_j (2 cos p_j - 2))^N on every
    timeslice, spin and colour"""
    dims = (6, 4, 8, 2)
    X, Y, Z, T = dims
    U = synth.unit_gauge(dims).numpy()
    psi = crandn(2, X * Y * Z * T, 4, 3)
    width, N = 2.5, 7
    a = width ** 2 / (4 * N)
    got = oracle.smear_gaussian(dims, U, psi, width, N, bc=(1, 1, 1, -1)).reshape(2, T, Z, Y, X, 4, 3)
    f = np.fft.fftn(psi.reshape(2, T, Z, Y, X, 4, 3), axes=(2, 3, 4))
    pz, py, px = np.meshgrid(2 * np.pi * np.fft.fftfreq(Z), 2 * np.pi * np.fft.fftfreq(Y), 2 * np.pi * np.fft.fftfreq(X), indexing="ij")
    sym = (1 + a * (2 * np.cos(px) + 2 * np.cos(py) + 2 * np.cos(pz) - 6)) ** N
    exp = np.fft.ifftn(f * sym[None, None, :, :, :, None, None], axes=(2, 3, 4))
    assert rel(got, exp) < 1e-13


def test_point_source_moments_give_the_width():
    """unit links, point source: each step is a lazy random walk with per-axis variance 2a, so after N steps the profile
    has sum = 1 and <x_j^2> = 2 a N = sigma^2 / 2 exactly (as long as the support, radius N, does not wrap)"""
    dims = (12, 12, 12, 2)
    X, Y, Z, T = dims
    U = synth.unit_gauge(dims).numpy()
    psi = np.zeros((1, X * Y * Z * T, 4, 3), dtype=complex)
    psi[0, 0, 1, 2] = 1.0                                        # origin of timeslice 0, one spin-colour component
    width, N = 1.6, 5
    out = oracle.smear_gaussian(dims, U, psi, width, N).reshape(T, Z, Y, X, 4, 3)
    prof = out[0, :, :, :, 1, 2]
    assert np.abs(out[1]).max() == 0.0                           # timeslices do not mix
    assert abs(prof.sum() - 1.0) < 1e-13 and np.abs(prof.imag).max() == 0.0
    coord = lambda L: np.minimum(np.arange(L), L - np.arange(L))   # min-image distance from the origin
    for axis, L in ((2, X), (1, Y), (0, Z)):
        sh = [1, 1, 1]
        sh[axis] = L
        m2 = (prof.real * coord(L).reshape(sh) ** 2).sum()
        assert abs(m2 - width ** 2 / 2) < 1e-12, (axis, m2)


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
    """smear(g psi ; U^g) = g smear(psi ; U)"""
    dims = (4, 4, 6, 4)
    V4 = int(np.prod(dims))
    U = synth.gauge_field(dims, 0.3, 31).numpy()
    G = synth.random_su3_field(V4, 32).numpy()
    psi = crandn(3, V4, 4, 3)
    lhs = oracle.smear_gaussian(dims, _transform(dims, U, G), np.einsum("xab,cxsb->cxsa", G, psi), 3.0, 6)
    rhs = np.einsum("xab,cxsb->cxsa", G, oracle.smear_gaussian(dims, U, psi, 3.0, 6))
    assert rel(lhs, rhs) < 1e-13


def test_one_step_against_literal_site_loops():
    """one application on 4x2x2x2 with an antiperiodic x direction, written as explicit loops over sites and legs
    (extent-2 directions: forward and backward neighbours coincide and both terms are added)"""
    dims, bc = (4, 2, 2, 2), (-1, 1, 1, -1)
    X, Y, Z, T = dims
    V4 = X * Y * Z * T
    U = synth.gauge_field(dims, 0.4, 33).numpy()
    psi = crandn(1, V4, 4, 3)
    width = 1.2
    a = width ** 2 / 4
    exp = np.zeros_like(psi)
    for t in range(T):
        for z in range(Z):
            for y in range(Y):
                for x in range(X):
                    co = [x, y, z, t]
                    i = x + X * (y + Y * (z + Z * t))
                    acc = -6.0 * psi[0, i]
                    for j in range(3):
                        cf = list(co)
                        cf[j] = (co[j] + 1) % dims[j]
                        sf = bc[j] if co[j] == dims[j] - 1 else 1
                        i_f = cf[0] + X * (cf[1] + Y * (cf[2] + Z * cf[3]))
                        cb = list(co)
                        cb[j] = (co[j] - 1) % dims[j]
                        sb = bc[j] if co[j] == 0 else 1
                        i_b = cb[0] + X * (cb[1] + Y * (cb[2] + Z * cb[3]))
                        for s in range(4):
                            acc[s] = acc[s] + sf * U[j, i] @ psi[0, i_f, s] + sb * U[j, i_b].conj().T @ psi[0, i_b, s]
                    exp[0, i] = psi[0, i] + a * acc
    got = oracle.smear_gaussian(dims, U, psi, width, 1, bc=bc)
    assert rel(got, exp) < 1e-14
    assert rel(oracle.smear_gaussian(dims, U, psi, width, 0, bc=bc), psi) == 0.0


def test_laplacian_is_hermitian_and_negative():
    dims = (4, 4, 4, 2)
    V4 = int(np.prod(dims))
    U = synth.gauge_field(dims, 0.3, 35).numpy()
    a, b = crandn(1, V4, 4, 3), crandn(1, V4, 4, 3)
    La, Lb = oracle.covariant_laplacian_3d(dims, U, a), oracle.covariant_laplacian_3d(dims, U, b)
    assert abs(np.vdot(b, La) - np.vdot(Lb, a)) < 1e-11 * np.linalg.norm(a) * np.linalg.norm(b)
    assert np.vdot(a, La).real < 0.0


def test_effective_derivative_closed_form():
    """C_FH(t) = C(t) (c + g t)  =>  g_eff(t) = g for every t"""
    t = np.arange(10)
    C = 3.0 * np.exp(-0.7 * t) * (1 + 0.1j)
    g = 1.271
    geff = oracle.fh_effective_derivative(C, C * (0.4 + g * t))
    assert geff.shape == (9,) and np.allclose(geff, g, atol=1e-13)

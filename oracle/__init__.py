"""CPU ORACLE binding (test infrastructure only -- see oracle/mdwf_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_1810_01609_b200 and shares no code with it.

All arrays are numpy complex128 in the canonical layouts of SURVEY.md 8(b):
  5D field [nrhs][Ls][V4][4][3],  gauge [4][V4][3][3],  4D propagator [ncol][V4][4][3].
Half-lattice fields ("sites of one parity in increasing x4") are produced by to_half / from_half;
every even-odd oracle routine itself works on full-lattice arrays that are zero on the other
parity (the even-odd objects are derived by masking).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = ["mdwf_oracle.cpp", "mdwf_oracle_dwf.cpp", "mdwf_oracle_meas.cpp"]
_LIB_PATH = os.path.join(_HERE, "libmdwf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP, no fast-math).  Returns the .so path."""
    srcs = [os.path.join(_HERE, s) for s in _SRC]
    deps = srcs + [os.path.join(_HERE, "mdwf_oracle.h")]
    if (not force) and os.path.exists(_LIB_PATH) and all(
            os.path.getmtime(_LIB_PATH) >= os.path.getmtime(d) for d in deps):
        return _LIB_PATH
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB_PATH] + srcs
    subprocess.run(cmd, check=True)
    return _LIB_PATH


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


@dataclass(frozen=True)
class Params:
    dims: tuple
    Ls: int
    M5: float
    b5: float
    c5: float
    mf: float
    bc: tuple = (1, 1, 1, -1)

    @property
    def V4(self):
        return int(np.prod(self.dims))

    @property
    def a(self):
        return self.b5 * (4.0 - self.M5) + 1.0

    @property
    def d(self):
        return self.c5 * (4.0 - self.M5) - 1.0


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _ints(v):
    return (ctypes.c_int * len(v))(*[int(i) for i in v])


def _dbls(v):
    return (ctypes.c_double * len(v))(*[float(i) for i in v])


def _par(p: Params):
    return _dbls([p.M5, p.b5, p.c5, p.mf])


def gamma(mu: int) -> np.ndarray:
    """gamma_mu for mu = 0..3 (x,y,z,t); mu = 4 gives gamma5."""
    buf = (ctypes.c_double * 32)()
    lib().oracle_gamma(int(mu), buf)
    a = np.array(buf[:], dtype=np.float64).reshape(4, 4, 2)
    return a[..., 0] + 1j * a[..., 1]


# ------------------------------------------------------------------ site bookkeeping (numpy only)
def parity_of_sites(dims) -> np.ndarray:
    X, Y, Z, T = dims
    x4 = np.arange(X * Y * Z * T)
    x = x4 % X
    y = (x4 // X) % Y
    z = (x4 // (X * Y)) % Z
    t = x4 // (X * Y * Z)
    return ((x + y + z + t) & 1).astype(np.int8)


def sites_of_parity(dims, parity: int) -> np.ndarray:
    return np.nonzero(parity_of_sites(dims) == parity)[0]


def to_half(full: np.ndarray, dims, parity: int) -> np.ndarray:
    """[..., V4, 4, 3] -> [..., Vh, 4, 3] (sites of `parity` in increasing x4)."""
    return np.ascontiguousarray(full[..., sites_of_parity(dims, parity), :, :])


def from_half(half: np.ndarray, dims, parity: int) -> np.ndarray:
    V4 = int(np.prod(dims))
    out = np.zeros(half.shape[:-3] + (V4, 4, 3), dtype=np.complex128)
    out[..., sites_of_parity(dims, parity), :, :] = half
    return out


# ------------------------------------------------------------------ operators
def hop(p: Params, U, psi, dagger=False, out_parity=-1):
    psi, pp = _c(psi)
    U, pu = _c(U)
    out = np.empty_like(psi)
    n5 = int(np.prod(psi.shape[:-3]))
    lib().oracle_hop(out.ctypes.data_as(ctypes.c_void_p), pp, pu, _ints(p.dims), _ints(p.bc), n5, int(dagger),
                     int(out_parity))
    return out


def wilson(p: Params, U, psi, dagger=False):
    psi, pp = _c(psi)
    U, pu = _c(U)
    out = np.empty_like(psi)
    n5 = int(np.prod(psi.shape[:-3]))
    lib().oracle_wilson(out.ctypes.data_as(ctypes.c_void_p), pp, pu, _ints(p.dims), _ints(p.bc), n5,
                        ctypes.c_double(p.M5), int(dagger))
    return out


def _ls_shape(p: Params, psi):
    assert psi.shape[-4] == p.Ls, psi.shape
    nrhs = int(np.prod(psi.shape[:-4])) if psi.ndim > 4 else 1
    return nrhs


def ls_hop(p: Params, psi, c0, c1, dagger=False):
    """c0*psi + c1*L psi   (L^dag if dagger)."""
    psi, pp = _c(psi)
    out = np.empty_like(psi)
    lib().oracle_ls_hop(out.ctypes.data_as(ctypes.c_void_p), pp, ctypes.c_int64(psi.shape[-3]), p.Ls,
                        _ls_shape(p, psi), ctypes.c_double(p.mf), ctypes.c_double(c0), ctypes.c_double(c1),
                        int(dagger))
    return out


def ls_inv(p: Params, psi, c0, c1, dagger=False):
    """(c0 + c1 L)^-1 psi by generic dense LU."""
    psi, pp = _c(psi)
    out = np.empty_like(psi)
    lib().oracle_ls_inv(out.ctypes.data_as(ctypes.c_void_p), pp, ctypes.c_int64(psi.shape[-3]), p.Ls,
                        _ls_shape(p, psi), ctypes.c_double(p.mf), ctypes.c_double(c0), ctypes.c_double(c1),
                        int(dagger))
    return out


def L(p, psi, dagger=False):
    return ls_hop(p, psi, 0.0, 1.0, dagger)


def M5op(p, psi, dagger=False):
    return ls_hop(p, psi, p.a, p.d, dagger)


def M4pre(p, psi, dagger=False):
    return ls_hop(p, psi, p.b5, p.c5, dagger)


def M5inv(p, psi, dagger=False):
    return ls_inv(p, psi, p.a, p.d, dagger)


def D(p: Params, U, psi, dagger=False):
    psi, pp = _c(psi)
    U, pu = _c(U)
    out = np.empty_like(psi)
    lib().oracle_D(out.ctypes.data_as(ctypes.c_void_p), pp, pu, _ints(p.dims), _ints(p.bc), p.Ls,
                   _ls_shape(p, psi), _par(p), int(dagger))
    return out


def Dminus(p: Params, U, psi, dagger=False):
    psi, pp = _c(psi)
    U, pu = _c(U)
    out = np.empty_like(psi)
    lib().oracle_Dminus(out.ctypes.data_as(ctypes.c_void_p), pp, pu, _ints(p.dims), _ints(p.bc), p.Ls,
                        _ls_shape(p, psi), _par(p), int(dagger))
    return out


def mask(p: Params, psi, keep: int):
    psi = np.array(psi, dtype=np.complex128, order="C", copy=True)
    n5 = int(np.prod(psi.shape[:-3]))
    lib().oracle_mask(psi.ctypes.data_as(ctypes.c_void_p), _ints(p.dims), n5, int(keep))
    return psi


def schur(p: Params, U, psi, parity=0, dagger=False, symmetric=False):
    """Dhat (symmetric=False) or Mhat = M5^-1 Dhat (True) on a full-lattice array; input is masked to `parity`."""
    psi, pp = _c(psi)
    U, pu = _c(U)
    out = np.empty_like(psi)
    lib().oracle_schur(out.ctypes.data_as(ctypes.c_void_p), pp, pu, _ints(p.dims), _ints(p.bc), p.Ls,
                       _ls_shape(p, psi), _par(p), int(parity), int(dagger), int(symmetric))
    return out


def prepare_source(p: Params, U, b, parity=0):
    b, pb = _c(b)
    U, pu = _c(U)
    out = np.empty_like(b)
    lib().oracle_prepare_source(out.ctypes.data_as(ctypes.c_void_p), pb, pu, _ints(p.dims), _ints(p.bc), p.Ls,
                                _ls_shape(p, b), _par(p), int(parity))
    return out


def reconstruct(p: Params, U, psi_p, b, parity=0):
    b, pb = _c(b)
    psi_p, pp = _c(psi_p)
    U, pu = _c(U)
    out = np.empty_like(b)
    lib().oracle_reconstruct(out.ctypes.data_as(ctypes.c_void_p), pp, pb, pu, _ints(p.dims), _ints(p.bc), p.Ls,
                             _ls_shape(p, b), _par(p), int(parity))
    return out


# ------------------------------------------------------------------ solves
def solve_full(p: Params, U, b, tol=1e-12, max_iter=20000):
    """Variant A: CG on D^dag D, full lattice.  Returns (x, iters[nrhs], normal-eq rel. residual[nrhs])."""
    b, pb = _c(b)
    U, pu = _c(U)
    nrhs = _ls_shape(p, b)
    x = np.empty_like(b)
    it = (ctypes.c_int * nrhs)()
    rs = (ctypes.c_double * nrhs)()
    lib().oracle_solve_full(x.ctypes.data_as(ctypes.c_void_p), pb, pu, _ints(p.dims), _ints(p.bc), p.Ls, nrhs,
                            _par(p), ctypes.c_double(tol), int(max_iter), it, rs)
    return x, list(it), list(rs)


def solve_eo(p: Params, U, b, parity=0, symmetric=False, tol=1e-12, max_iter=20000):
    """Variant B: the oracle's own even-odd CG + reconstruction."""
    b, pb = _c(b)
    U, pu = _c(U)
    nrhs = _ls_shape(p, b)
    x = np.empty_like(b)
    it = (ctypes.c_int * nrhs)()
    rs = (ctypes.c_double * nrhs)()
    lib().oracle_solve_eo(x.ctypes.data_as(ctypes.c_void_p), pb, pu, _ints(p.dims), _ints(p.bc), p.Ls, nrhs,
                          _par(p), int(parity), int(symmetric), ctypes.c_double(tol), int(max_iter), it, rs)
    return x, list(it), list(rs)


def true_residual(p: Params, U, x, b):
    """||b - D x|| / ||b|| per rhs, with the oracle's FULL operator (SURVEY A9 'solver true residual')."""
    r = np.asarray(b) - D(p, U, x)
    nr = np.sqrt((np.abs(r) ** 2).reshape(r.shape[0], -1).sum(1))
    nb = np.sqrt((np.abs(np.asarray(b)) ** 2).reshape(r.shape[0], -1).sum(1))
    return nr / nb


# ------------------------------------------------------------------ 4D <-> 5D, FH chain, contraction
def wall_inject(p: Params, U, eta4):
    eta4, pe = _c(eta4)
    U, pu = _c(U)
    ncol = eta4.shape[0]
    out = np.empty((ncol, p.Ls) + eta4.shape[1:], dtype=np.complex128)
    lib().oracle_wall_inject(out.ctypes.data_as(ctypes.c_void_p), pe, pu, _ints(p.dims), _ints(p.bc), p.Ls, ncol,
                             _par(p))
    return out


def wall_project(p: Params, psi5):
    psi5, pp = _c(psi5)
    ncol = psi5.shape[0]
    out = np.empty((ncol,) + psi5.shape[2:], dtype=np.complex128)
    lib().oracle_wall_project(out.ctypes.data_as(ctypes.c_void_p), pp, ctypes.c_int64(psi5.shape[2]), p.Ls, ncol)
    return out


def _mat32(M):
    M = np.asarray(M, dtype=np.complex128).reshape(4, 4)
    return _dbls(np.stack([M.real, M.imag], -1).reshape(-1))


def seq_source(dims, prop4, Gamma, t_min=0, t_max=None):
    prop4, pp = _c(prop4)
    if t_max is None:
        t_max = dims[3] - 1
    out = np.empty_like(prop4)
    lib().oracle_seq_source(out.ctypes.data_as(ctypes.c_void_p), pp, _mat32(Gamma), _ints(dims), prop4.shape[0],
                            int(t_min), int(t_max))
    return out


def nucleon_2pt(dims, Su1, Sd, Su2, proj, t0=0, t_lo=0, t_hi=None):
    Su1, p1 = _c(Su1)
    Sd, p2 = _c(Sd)
    Su2, p3 = _c(Su2)
    T = dims[3]
    if t_hi is None:
        t_hi = T - 1
    corr = (ctypes.c_double * (2 * T))()
    lib().oracle_nucleon_2pt(corr, p1, p2, p3, _mat32(proj), _ints(dims), int(t0), int(t_lo), int(t_hi))
    c = np.array(corr[:], dtype=np.float64).reshape(T, 2)
    return c[:, 0] + 1j * c[:, 1]


# ---------------------------------------------------------------------------------------------------------------
# NEXT-3: the fuller Feynman-Hellmann workload.  The paper names "smeared" sources but
# prints no smearing formula; R25 fixes the reading: gauge-covariant Gaussian smearing
#     psi' = (1 + sigma^2/(4 N) Lap)^N psi,
#     (Lap psi)(x) = sum_{j=x,y,z} [ U_j(x) psi(x+j) + U_j(x-j)^dag psi(x-j) - 2 psi(x) ]        (3D, per timeslice)
# with the geometry's boundary sign bc_j on hops that wrap.  Plain numpy on the canonical fields
# U[4][x4][3][3], psi[col][x4][4][3], x4 = x + X(y + Y(z + Z t)).
# ---------------------------------------------------------------------------------------------------------------
def covariant_laplacian_3d(dims, U, psi4, bc=(1, 1, 1, -1)):
    X, Y, Z, T = dims
    ncol = psi4.shape[0]
    f = np.asarray(psi4, dtype=np.complex128).reshape(ncol, T, Z, Y, X, 4, 3)
    Ur = np.asarray(U, dtype=np.complex128).reshape(4, T, Z, Y, X, 3, 3)
    lap = -6.0 * f
    for j in range(3):
        axis = 4 - j                                   # x is the fastest index
        L = dims[j]
        # forward: U_j(x) psi(x + j); the hop from coordinate L-1 wraps
        fwd = np.roll(f, -1, axis=axis).copy()
        idx = [slice(None)] * 7
        idx[axis] = L - 1
        fwd[tuple(idx)] *= bc[j]
        lap = lap + np.einsum("tzyxab,ctzyxsb->ctzyxsa", Ur[j], fwd)
        # backward: U_j(x - j)^dag psi(x - j); the hop from coordinate 0 wraps
        w = np.einsum("tzyxba,ctzyxsb->ctzyxsa", Ur[j].conj(), f)
        bwd = np.roll(w, 1, axis=axis).copy()
        idx[axis] = 0
        bwd[tuple(idx)] *= bc[j]
        lap = lap + bwd
    return lap.reshape(psi4.shape)


def smear_gaussian(dims, U, psi4, width, n_iter, bc=(1, 1, 1, -1)):
    """psi' = (1 + width^2/(4 n_iter) Lap)^n_iter psi  (n_iter = 0: the identity)."""
    out = np.array(psi4, dtype=np.complex128, copy=True)
    if n_iter <= 0:
        return out
    a = float(width) ** 2 / (4.0 * n_iter)
    for _ in range(int(n_iter)):
        out = out + a * covariant_laplacian_3d(dims, U, out, bc)
    return out


def fh_effective_derivative(c2pt, cfh):
    """Feynman-Hellmann effective derivative ("Fig. 1"): with R(t) = C_FH(t) / C_2pt(t), the derivative of
    the effective mass with respect to the source strength is g_eff(t) = R(t+1) - R(t), t = 0..T-2 (R25)."""
    R = np.asarray(cfh) / np.asarray(c2pt)
    return R[1:] - R[:-1]

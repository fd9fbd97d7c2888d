"""Seeded synthetic input generators (SURVEY.md §8(c) A16-A18, §8(d) "Synthetic inputs").

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of the
method's arithmetic: no Dirac operator, no gamma matrices, no even-odd logic, no solver.
It only draws seeded random numbers and shapes them like the paper's workloads
("SU(3) ... gauge", "12x12" spin-colour propagator columns;
BASELINE.json configs[0..4]).  The production ensembles of the paper
are not available; these inputs stand in for them.

Canonical interchange layouts:
  gauge   U[mu][x4][row][col]            complex128, x4 = x + X*(y + Y*(z + Z*t))
  spinor  psi[rhs][s][x4][spin][colour]  complex128
  4D prop S[col][x4][spin][colour]       complex128, col = 3*spin_src + colour_src
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

__all__ = [
    "Config", "CONFIGS", "gauge_field", "unit_gauge", "gaussian_spinor", "point_sources_4d",
    "gaussian_smeared_sources_4d", "random_su3_field", "mean_trace", "seed_for",
]


@dataclass(frozen=True)
class Config:
    """One of BASELINE.json's five workloads (shape + physics parameters only)."""
    name: str
    dims: tuple          # (X, Y, Z, T)
    Ls: int
    nrhs: int
    mf: float
    tol: float
    eps: float           # link roughness: U = reunit(exp(i*eps*H)), SURVEY A17
    M5: float = 1.3
    b5: float = 1.5
    c5: float = 0.5
    bc: tuple = (1, 1, 1, -1)
    index: int = 0

    @property
    def V4(self):
        return int(np.prod(self.dims))


# eps = 0.306 gives mean plaquette 0.600 for independent links (plaquette = c(eps)^4);
# config 1 fixes eps = 0.3 exactly (BASELINE.json configs[0]).
CONFIGS = {
    1: Config("c1_4^4_Ls4", (4, 4, 4, 4), 4, 1, 0.1, 1e-10, 0.3, index=1),
    2: Config("c2_16^3x32_Ls8", (16, 16, 16, 32), 8, 1, 0.05, 1e-8, 0.306, index=2),
    3: Config("c3_24^3x64_Ls8", (24, 24, 24, 64), 8, 12, 0.02, 1e-8, 0.306, index=3),
    4: Config("c4_32^3x48_Ls12", (32, 32, 32, 48), 12, 12, 0.015, 1e-8, 0.306, index=4),
    5: Config("c5_48^3x64_Ls10", (48, 48, 48, 64), 10, 4, 0.01, 1e-10, 0.306, index=5),
}


def seed_for(config_index: int, stream: int) -> int:
    """seed = 1000*config + stream id (1 = gauge, 2.. = sources, 50.. = manufactured)."""
    return 1000 * int(config_index) + int(stream)


def _randn_complex(shape, seed: int) -> torch.Tensor:
    """N(0,1) + i N(0,1), fp64, drawn on the CPU so the stream is device independent."""
    g = torch.Generator(device="cpu")
    g.manual_seed(int(seed))
    re = torch.randn(shape, generator=g, dtype=torch.float64)
    im = torch.randn(shape, generator=g, dtype=torch.float64)
    return torch.complex(re, im)


def _reunitarize(U: torch.Tensor) -> torch.Tensor:
    """Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1)  ->  exactly SU(3) up to rounding."""
    r0 = U[..., 0, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
    r1 = U[..., 1, :]
    r1 = r1 - (r0.conj() * r1).sum(-1, keepdim=True) * r0
    r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
    r2 = torch.stack([
        r0[..., 1] * r1[..., 2] - r0[..., 2] * r1[..., 1],
        r0[..., 2] * r1[..., 0] - r0[..., 0] * r1[..., 2],
        r0[..., 0] * r1[..., 1] - r0[..., 1] * r1[..., 0],
    ], dim=-1).conj()
    return torch.stack([r0, r1, r2], dim=-2)


def _exp_i_eps_H(H: torch.Tensor, eps: float, order: int = 30) -> torch.Tensor:
    """exp(i*eps*H) by its Taylor series (||eps*H|| ~ 1, 30 terms reach rounding), batched."""
    A = (1j * eps) * H
    eye = torch.eye(3, dtype=H.dtype, device=H.device).expand_as(H)
    term = eye.clone()
    out = eye.clone()
    for n in range(1, order + 1):
        term = torch.matmul(term, A) / n
        out = out + term
    return out


def gauge_field(dims, eps: float, seed: int, device="cpu", chunk: int = 1 << 21) -> torch.Tensor:
    """Links U_mu(x) = reunit(exp(i*eps*H)), H = (A+A^dag)/2 - tr/3, A_ij = N(0,1)+iN(0,1);
    independent per link (BASELINE.json configs[0], configs[1]).
    Returns complex128 [4][V4][3][3] on `device` (the random numbers are always CPU-drawn)."""
    V4 = int(np.prod(dims))
    n = 4 * V4
    A = _randn_complex((n, 3, 3), seed)
    out = torch.empty((n, 3, 3), dtype=torch.complex128, device=device)
    for lo in range(0, n, chunk):
        a = A[lo:lo + chunk].to(device)
        H = 0.5 * (a + a.conj().transpose(-1, -2))
        tr = (H[..., 0, 0] + H[..., 1, 1] + H[..., 2, 2]) / 3.0
        H = H - tr[..., None, None] * torch.eye(3, dtype=H.dtype, device=H.device)
        out[lo:lo + chunk] = _reunitarize(_exp_i_eps_H(H, eps))
    return out.reshape(4, V4, 3, 3)


def unit_gauge(dims, device="cpu") -> torch.Tensor:
    """Free field: every link the identity."""
    V4 = int(np.prod(dims))
    U = torch.zeros((4, V4, 3, 3), dtype=torch.complex128, device=device)
    for a in range(3):
        U[..., a, a] = 1.0
    return U


def random_su3_field(V4: int, seed: int, eps: float = 1.0) -> torch.Tensor:
    """One random SU(3) matrix per 4D site (a gauge transformation G(x)); [V4][3][3]."""
    A = _randn_complex((V4, 3, 3), seed)
    H = 0.5 * (A + A.conj().transpose(-1, -2))
    tr = (H[..., 0, 0] + H[..., 1, 1] + H[..., 2, 2]) / 3.0
    H = H - tr[..., None, None] * torch.eye(3, dtype=H.dtype)
    return _reunitarize(_exp_i_eps_H(H, eps))


def mean_trace(U: torch.Tensor) -> float:
    """<1/3 Re tr U> over all links: c(eps) of SURVEY A17 (a property of the INPUT, no physics)."""
    return float((U[..., 0, 0].real + U[..., 1, 1].real + U[..., 2, 2].real).mean() / 3.0)


def gaussian_spinor(dims, Ls: int, nrhs: int, seed: int) -> torch.Tensor:
    """Gaussian complex random 5D spinor(s), canonical [rhs][s][x4][4][3] complex128 (CPU)."""
    V4 = int(np.prod(dims))
    return _randn_complex((nrhs, Ls, V4, 4, 3), seed)


def point_sources_4d(dims, site=(0, 0, 0, 0)) -> torch.Tensor:
    """12 unit spin-colour vectors at one site: eta[col][x4][spin][colour], col = 3*spin+colour
    (BASELINE.json configs[2])."""
    X, Y, Z, T = dims
    V4 = X * Y * Z * T
    x4 = site[0] + X * (site[1] + Y * (site[2] + Z * site[3]))
    eta = torch.zeros((12, V4, 4, 3), dtype=torch.complex128)
    for sp in range(4):
        for c in range(3):
            eta[3 * sp + c, x4, sp, c] = 1.0
    return eta


def gaussian_smeared_sources_4d(dims, width: float = 3.0, t0: int = 0) -> torch.Tensor:
    """non-covariant profile exp(-|x|^2_min-image / (2 width^2)) on timeslice t0,
    centred at the spatial origin, ||profile||_2 = 1, times the 12 unit spin-colour vectors."""
    X, Y, Z, T = dims
    V4 = X * Y * Z * T
    def mind(L):
        c = np.arange(L)
        return np.minimum(c, L - c).astype(np.float64)
    dx, dy, dz = mind(X), mind(Y), mind(Z)
    r2 = dx[None, None, :] ** 2 + dy[None, :, None] ** 2 + dz[:, None, None] ** 2   # [z][y][x]
    prof = np.exp(-r2 / (2.0 * width * width))
    prof /= math.sqrt(float((prof ** 2).sum()))
    full = np.zeros((T, Z, Y, X), dtype=np.float64)
    full[t0] = prof
    p = torch.from_numpy(full.reshape(V4))
    eta = torch.zeros((12, V4, 4, 3), dtype=torch.complex128)
    for sp in range(4):
        for c in range(3):
            eta[3 * sp + c, :, sp, c] = p
    return eta


def gaussian_spinor_device(dims, Ls: int, nrhs: int, seed: int, device="cuda", out=None) -> torch.Tensor:
    """Full-size workloads only (bench.py, full-size parity tests): the same N(0,1)+iN(0,1) field as
    gaussian_spinor but drawn by the DEVICE generator (seeded; one rhs at a time to bound memory), because
    drawing 54 GB on the host would dominate the run.  The stream differs from the CPU-drawn one, so a
    check that needs the oracle copies the slices it wants back to the host."""
    V4 = int(np.prod(dims))
    if out is None:
        out = torch.empty((nrhs, Ls, V4, 4, 3), dtype=torch.complex128, device=device)
    g = torch.Generator(device=device)
    for r in range(nrhs):
        g.manual_seed(int(seed) * 1000 + r)
        torch.view_as_real(out[r]).normal_(0.0, 1.0, generator=g)
    return out

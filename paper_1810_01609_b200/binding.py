"""Thin ctypes binding of libmdwf.so (include/mdwf.h): argument marshalling only.

Every function here has the name of the C entry point it calls; all arithmetic runs in the CUDA
kernels of csrc/.  PyTorch is used for device memory and streams only.  There is no CPU
fallback: if libmdwf.so is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MDWF_LIB", os.path.join(_HERE, "libmdwf.so"))   # MDWF_LIB: alternative build of the same library

OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4
NOT_CONVERGED, BREAKDOWN = 1, 2
OP_HOP, OP_M4PRE, OP_M5, OP_M5INV, OP_DHAT_ASYM, OP_DHAT_SYM, OP_NORMAL_ASYM, OP_NORMAL_SYM, OP_FULL = range(9)
MAX_RHS = 64

EXPORTS = [
    "mdwf_create", "mdwf_destroy", "mdwf_last_error", "mdwf_load_gauge", "mdwf_dslash", "mdwf_field_create",
    "mdwf_field_destroy", "mdwf_field_pack", "mdwf_field_unpack", "mdwf_dslash_packed", "mdwf_dslash_cost",
    "mdwf_solve", "mdwf_solve_host", "mdwf_seq_source", "mdwf_nucleon_2pt", "mdwf_wall_inject",
    "mdwf_wall_project", "mdwf_launch_count", "mdwf_set_tiling", "mdwf_profile", "mdwf_profile_read", "mdwf_selftest_host", "mdwf_solve_packed",
    "mdwf_workspace_bytes", "mdwf_set_workspace", "mdwf_set_hop16_tile", "mdwf_field_pack_rhs", "mdwf_field_unpack_rhs",
    "mdwf_autotune", "mdwf_tune_save", "mdwf_tune_load", "mdwf_tune_get",
    "mdwf_nucleon_2pt_noalloc", "mdwf_nucleon_2pt_noalloc_max_bytes",
    "mdwf_smear_gaussian", "mdwf_fh_effective_derivative",
]


class MdwfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libmdwf error %d: %s" % (code, msg))
        self.code = code


class Geometry(ctypes.Structure):
    _fields_ = [("dims", ctypes.c_int32 * 4), ("Ls", ctypes.c_int32), ("bc", ctypes.c_int32 * 4),
                ("device", ctypes.c_int32)]


class SolveOpts(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("max_iter", ctypes.c_int32), ("inner_prec", ctypes.c_int32),
                ("recon", ctypes.c_int32), ("parity", ctypes.c_int32), ("symmetric", ctypes.c_int32),
                ("delta", ctypes.c_double), ("src_kind", ctypes.c_int32), ("out_kind", ctypes.c_int32),
                ("batch", ctypes.c_int32), ("check_every", ctypes.c_int32)]


class SolveInfo(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int32 * MAX_RHS), ("reliable_updates", ctypes.c_int32 * MAX_RHS),
                ("status", ctypes.c_int32 * MAX_RHS), ("true_resid", ctypes.c_double * MAX_RHS),
                ("seconds", ctypes.c_double), ("seconds_inner", ctypes.c_double),
                ("kernel_launches", ctypes.c_int64), ("batch", ctypes.c_int32)]


_lib = None


def lib():
    """Load libmdwf.so (raises if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libmdwf.so not built: run `python -m paper_1810_01609_b200.build` "
                               "(the CUDA library is the only implementation; there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.mdwf_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(Geometry), cd, cd, cd, cd]
        L.mdwf_destroy.argtypes = [vp]
        L.mdwf_last_error.argtypes = [vp]
        L.mdwf_last_error.restype = ctypes.c_char_p
        L.mdwf_load_gauge.argtypes = [vp, vp, ci, ci, vp]
        L.mdwf_dslash.argtypes = [vp, ci, ci, ci, ci, ci, vp, vp, ci, vp]
        L.mdwf_field_create.argtypes = [vp, ci, ci, ctypes.POINTER(vp)]
        L.mdwf_field_destroy.argtypes = [vp]
        L.mdwf_field_pack.argtypes = [vp, vp, vp]
        L.mdwf_field_unpack.argtypes = [vp, vp, vp]
        L.mdwf_dslash_packed.argtypes = [vp, ci, ci, ci, ci, vp, vp, vp]
        L.mdwf_dslash_cost.argtypes = [vp, ci, ci, ci, ci, ctypes.POINTER(cd), ctypes.POINTER(cd)]
        L.mdwf_solve.argtypes = [vp, vp, vp, ci, ctypes.POINTER(SolveOpts), ctypes.POINTER(SolveInfo), vp]
        L.mdwf_solve_host.argtypes = [vp, vp, vp, ci, ctypes.POINTER(SolveOpts), ctypes.POINTER(SolveInfo), vp]
        L.mdwf_seq_source.argtypes = [vp, vp, vp, ci, ctypes.POINTER(cd), ci, ci, vp]
        L.mdwf_nucleon_2pt.argtypes = [vp, vp, vp, vp, vp, ctypes.POINTER(cd), ci, vp]
        L.mdwf_nucleon_2pt_noalloc.argtypes = [vp, vp, vp, vp, vp, ctypes.POINTER(cd), ci, vp]
        L.mdwf_nucleon_2pt_noalloc_max_bytes.argtypes = []
        L.mdwf_smear_gaussian.argtypes = [vp, vp, vp, ci, cd, ci, vp]
        L.mdwf_fh_effective_derivative.argtypes = [vp, vp, vp, vp, vp]
        L.mdwf_nucleon_2pt_noalloc_max_bytes.restype = ctypes.c_int64
        L.mdwf_wall_inject.argtypes = [vp, vp, vp, ci, ci, vp]
        L.mdwf_wall_project.argtypes = [vp, vp, vp, ci, vp]
        L.mdwf_launch_count.argtypes = [vp]
        L.mdwf_launch_count.restype = ctypes.c_int64
        L.mdwf_set_tiling.argtypes = [vp, ci]
        L.mdwf_profile.argtypes = [vp, ci]
        L.mdwf_profile_read.argtypes = [vp, ci, ctypes.POINTER(cd), ctypes.POINTER(cd), ctypes.POINTER(cd),
                                        ctypes.POINTER(ctypes.c_int64)]
        L.mdwf_selftest_host.argtypes = [cd, cd, cd, cd]
        L.mdwf_solve_packed.argtypes = [vp, vp, vp, ctypes.POINTER(SolveOpts), ctypes.POINTER(SolveInfo), vp]
        L.mdwf_workspace_bytes.argtypes = [vp, ci, ci, ci, ctypes.POINTER(ctypes.c_int64)]
        L.mdwf_set_workspace.argtypes = [vp, vp, ctypes.c_int64]
        L.mdwf_set_hop16_tile.argtypes = [vp, ci, ci, ci, ci, ci]
        L.mdwf_autotune.argtypes = [vp, ci, ci, ci, vp]
        L.mdwf_tune_save.argtypes = [vp, ctypes.c_char_p]
        L.mdwf_tune_load.argtypes = [vp, ctypes.c_char_p]
        L.mdwf_tune_get.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(ctypes.c_int), ci]
        L.mdwf_field_pack_rhs.argtypes = [vp, ci, vp, vp]
        L.mdwf_field_unpack_rhs.argtypes = [vp, ci, vp, vp]
        _lib = L
    return _lib


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t: torch.Tensor, what="tensor"):
    if not t.is_cuda:
        raise ValueError("%s must be a CUDA tensor" % what)
    if not t.is_contiguous():
        raise ValueError("%s must be contiguous" % what)
    if t.dtype not in (torch.complex128, torch.float64):
        raise ValueError("%s must be complex128/float64 (canonical fp64 layout)" % what)
    return ctypes.c_void_p(t.data_ptr())


def _mat32(M):
    M = torch.as_tensor(M, dtype=torch.complex128).reshape(4, 4).cpu()
    flat = torch.view_as_real(M).reshape(-1).tolist()
    return (ctypes.c_double * 32)(*flat)


@dataclass
class SolveResult:
    status: int
    iters: list
    reliable_updates: list
    rhs_status: list
    true_resid: list
    seconds: float
    seconds_inner: float
    kernel_launches: int
    batch: int = 0


def mdwf_selftest_host(M5=1.3, b5=1.5, c5=0.5, mf=0.05):
    """Host-only checks of the library's index arithmetic and s-direction matrices (no GPU needed)."""
    return int(lib().mdwf_selftest_host(M5, b5, c5, mf))


class Field:
    """Packed device field (mdwf_field_*)."""

    def __init__(self, ctx: "Context", prec: int, nrhs: int):
        self.ctx, self.prec, self.nrhs = ctx, prec, nrhs
        h = ctypes.c_void_p()
        ctx._chk(lib().mdwf_field_create(ctx._h, prec, nrhs, ctypes.byref(h)))
        self._h = h

    def mdwf_field_pack(self, canonical: torch.Tensor):
        self.ctx._chk(lib().mdwf_field_pack(self._h, _dev(canonical), _stream()))

    def mdwf_field_unpack(self, canonical: torch.Tensor):
        self.ctx._chk(lib().mdwf_field_unpack(self._h, _dev(canonical), _stream()))

    def mdwf_field_pack_rhs(self, rhs: int, canonical: torch.Tensor):
        self.ctx._chk(lib().mdwf_field_pack_rhs(self._h, rhs, _dev(canonical), _stream()))

    def mdwf_field_unpack_rhs(self, rhs: int, canonical: torch.Tensor):
        self.ctx._chk(lib().mdwf_field_unpack_rhs(self._h, rhs, _dev(canonical), _stream()))

    def mdwf_field_destroy(self):
        if self._h:
            lib().mdwf_field_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.mdwf_field_destroy()
        except Exception:
            pass


class Context:
    """mdwf_create(geometry, M5, b5, c5, mf) and the calls that take the context."""

    def __init__(self, dims, Ls, M5, b5, c5, mf, bc=(1, 1, 1, -1), device=0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1810_01609_b200 needs a CUDA device (no CPU fallback)")
        self.dims, self.Ls, self.bc = tuple(int(d) for d in dims), int(Ls), tuple(bc)
        self.V4 = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        g = Geometry()
        for i in range(4):
            g.dims[i] = self.dims[i]
            g.bc[i] = int(bc[i])
        g.Ls = int(Ls)
        g.device = int(device)
        self._h = ctypes.c_void_p()
        rc = lib().mdwf_create(ctypes.byref(self._h), ctypes.byref(g), M5, b5, c5, mf)
        if rc != OK:
            msg = lib().mdwf_last_error(self._h).decode() if self._h else "mdwf_create failed"
            if self._h:
                lib().mdwf_destroy(self._h)
                self._h = None
            raise MdwfError(rc, msg)

    def _chk(self, rc, soft_ok=False):
        if rc < 0 or (rc > 0 and not soft_ok):
            raise MdwfError(rc, lib().mdwf_last_error(self._h).decode())
        return rc

    def mdwf_destroy(self):
        if self._h:
            lib().mdwf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.mdwf_destroy()
        except Exception:
            pass

    def mdwf_load_gauge(self, U: torch.Tensor, store_prec=64, recon=18):
        assert U.shape == (4, self.V4, 3, 3), U.shape
        self._chk(lib().mdwf_load_gauge(self._h, _dev(U, "U"), store_prec, recon, _stream()))

    def mdwf_dslash(self, op, inp: torch.Tensor, parity=0, dagger=False, prec=64, recon=18):
        """inp: [nrhs][Ls][Vh or V4][4][3] complex128 on the device; returns a new tensor of the same shape."""
        nrhs = inp.shape[0]
        out = torch.empty_like(inp)
        self._chk(lib().mdwf_dslash(self._h, op, parity, int(bool(dagger)), prec, recon, _dev(out), _dev(inp), nrhs,
                                    _stream()))
        return out

    def mdwf_field_create(self, prec, nrhs):
        return Field(self, prec, nrhs)

    def mdwf_dslash_packed(self, op, out: Field, inp: Field, parity=0, dagger=False, recon=18):
        self._chk(lib().mdwf_dslash_packed(self._h, op, parity, int(bool(dagger)), recon, out._h, inp._h, _stream()))

    def mdwf_dslash_cost(self, op, prec, recon, nrhs):
        b, f = ctypes.c_double(), ctypes.c_double()
        self._chk(lib().mdwf_dslash_cost(self._h, op, prec, recon, nrhs, ctypes.byref(b), ctypes.byref(f)))
        return b.value, f.value

    def _opts(self, tol, max_iter, inner_prec, recon, parity, symmetric, delta, src_kind, out_kind, batch, check_every):
        o = SolveOpts()
        o.tol, o.max_iter, o.inner_prec, o.recon, o.parity = tol, max_iter, inner_prec, recon, parity
        o.symmetric, o.delta, o.src_kind, o.out_kind, o.batch, o.check_every = (int(symmetric), delta, src_kind,
                                                                                 out_kind, batch, check_every)
        return o

    @staticmethod
    def _result(rc, info, nrhs):
        return SolveResult(rc, list(info.iters[:nrhs]), list(info.reliable_updates[:nrhs]), list(info.status[:nrhs]),
                           list(info.true_resid[:nrhs]), info.seconds, info.seconds_inner, info.kernel_launches,
                           info.batch)

    def mdwf_solve(self, b: torch.Tensor, tol=1e-8, max_iter=20000, inner_prec=16, recon=12, parity=0, symmetric=True,
                   delta=0.1, src_kind=0, out_kind=0, batch=0, check_every=1, out=None):
        """b: [nrhs][Ls][V4][4][3] (src_kind 0) or [nrhs][V4][4][3] (src_kind 1), complex128 device tensor.
        Returns (x, SolveResult)."""
        nrhs = b.shape[0]
        shape = (nrhs, self.Ls, self.V4, 4, 3) if out_kind == 0 else (nrhs, self.V4, 4, 3)
        x = out if out is not None else torch.empty(shape, dtype=torch.complex128, device=b.device)
        o = self._opts(tol, max_iter, inner_prec, recon, parity, symmetric, delta, src_kind, out_kind, batch, check_every)
        info = SolveInfo()
        rc = self._chk(lib().mdwf_solve(self._h, _dev(x), _dev(b), nrhs, ctypes.byref(o), ctypes.byref(info), _stream()),
                       soft_ok=True)
        return x, self._result(rc, info, nrhs)

    def mdwf_solve_host(self, b_host: torch.Tensor, x_host: torch.Tensor, **kw):
        """Same with HOST (CPU, ideally pinned) complex128 tensors; all copies happen inside the call."""
        assert not b_host.is_cuda and not x_host.is_cuda and b_host.is_contiguous() and x_host.is_contiguous()
        nrhs = b_host.shape[0]
        o = self._opts(kw.get("tol", 1e-8), kw.get("max_iter", 20000), kw.get("inner_prec", 16), kw.get("recon", 12),
                       kw.get("parity", 0), kw.get("symmetric", True), kw.get("delta", 0.1), kw.get("src_kind", 0),
                       kw.get("out_kind", 0), kw.get("batch", 0), kw.get("check_every", 1))
        info = SolveInfo()
        rc = self._chk(lib().mdwf_solve_host(self._h, ctypes.c_void_p(x_host.data_ptr()),
                                             ctypes.c_void_p(b_host.data_ptr()), nrhs, ctypes.byref(o),
                                             ctypes.byref(info), _stream()), soft_ok=True)
        return x_host, self._result(rc, info, nrhs)

    def mdwf_solve_packed(self, psi_even: Field, psi_odd: Field, **kw):
        """In-place solve on packed fp64 half-lattice fields (b on entry, solution on exit)."""
        nrhs = psi_even.nrhs
        o = self._opts(kw.get("tol", 1e-8), kw.get("max_iter", 20000), kw.get("inner_prec", 16), kw.get("recon", 12),
                       kw.get("parity", 0), kw.get("symmetric", True), kw.get("delta", 0.1), 0, 0, 0,
                       kw.get("check_every", 1))
        info = SolveInfo()
        rc = self._chk(lib().mdwf_solve_packed(self._h, psi_even._h, psi_odd._h, ctypes.byref(o), ctypes.byref(info),
                                               _stream()), soft_ok=True)
        return self._result(rc, info, nrhs)

    def mdwf_workspace_bytes(self, nrhs, inner_prec=16, packed=False):
        n = ctypes.c_int64()
        self._chk(lib().mdwf_workspace_bytes(self._h, nrhs, inner_prec, int(bool(packed)), ctypes.byref(n)))
        return n.value

    def mdwf_set_workspace(self, buf):
        """buf: a CUDA uint8 tensor the library uses as its solver workspace (kept alive here), or None."""
        self._ws = buf
        if buf is None:
            self._chk(lib().mdwf_set_workspace(self._h, None, 0))
        else:
            self._chk(lib().mdwf_set_workspace(self._h, ctypes.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size()))

    def mdwf_set_hop16_tile(self, lx, ly, lz, lt, warps=0):
        self._chk(lib().mdwf_set_hop16_tile(self._h, lx, ly, lz, lt, warps))

    def mdwf_autotune(self, prec, recon, nrhs=1):
        self._chk(lib().mdwf_autotune(self._h, prec, recon, nrhs, _stream()))

    def mdwf_tune_save(self, path):
        self._chk(lib().mdwf_tune_save(self._h, str(path).encode()))

    def mdwf_tune_load(self, path):
        self._chk(lib().mdwf_tune_load(self._h, str(path).encode()))

    def mdwf_tune_get(self, key):
        buf = (ctypes.c_int * 8)()
        n = lib().mdwf_tune_get(self._h, key.encode(), buf, 8)
        if n < 0:
            raise MdwfError(n, "mdwf_tune_get")
        return [buf[i] for i in range(min(n, 8))]

    def mdwf_seq_source(self, prop4d: torch.Tensor, Gamma, t_min=0, t_max=None, out=None):
        ncol = prop4d.shape[0]
        if t_max is None:
            t_max = self.dims[3] - 1
        o = out if out is not None else torch.empty_like(prop4d)
        self._chk(lib().mdwf_seq_source(self._h, _dev(o), _dev(prop4d), ncol, _mat32(Gamma), t_min, t_max, _stream()))
        return o

    def mdwf_nucleon_2pt(self, S_u1, S_d, S_u2, proj, t0=0):
        T = self.dims[3]
        corr = torch.empty((T, 2), dtype=torch.float64, device=S_d.device)
        for S in (S_u1, S_d, S_u2):
            assert S.shape == (12, self.V4, 4, 3), S.shape
        self._chk(lib().mdwf_nucleon_2pt(self._h, _dev(corr), _dev(S_u1), _dev(S_d), _dev(S_u2), _mat32(proj), t0,
                                         _stream()))
        return torch.view_as_complex(corr)

    def mdwf_nucleon_2pt_noalloc(self, S_u1, S_d, S_u2, proj, corr, t0=0):
        """mdwf_nucleon_2pt without any device allocation: the caller supplies corr (float64 [T][2], device) as well."""
        T = self.dims[3]
        assert corr.shape == (T, 2) and corr.dtype == torch.float64 and corr.is_cuda and corr.is_contiguous()
        for S in (S_u1, S_d, S_u2):
            assert S.shape == (12, self.V4, 4, 3), S.shape
        self._chk(lib().mdwf_nucleon_2pt_noalloc(self._h, _dev(corr), _dev(S_u1), _dev(S_d), _dev(S_u2), _mat32(proj), t0,
                                                 _stream()))
        return torch.view_as_complex(corr)

    def mdwf_smear_gaussian(self, psi4: torch.Tensor, width, n_iter, out=None):
        ncol = psi4.shape[0]
        assert psi4.shape == (ncol, self.V4, 4, 3) and psi4.dtype == torch.complex128 and psi4.is_contiguous()
        if out is None:
            out = torch.empty_like(psi4)
        self._chk(lib().mdwf_smear_gaussian(self._h, _dev(out), _dev(psi4), ncol, float(width), int(n_iter), _stream()))
        return out

    def mdwf_fh_effective_derivative(self, c2pt: torch.Tensor, cfh: torch.Tensor):
        T = self.dims[3]
        c2, cf = torch.view_as_real(c2pt.contiguous()), torch.view_as_real(cfh.contiguous())
        assert c2.shape == (T, 2) and cf.shape == (T, 2) and c2.dtype == torch.float64 and cf.dtype == torch.float64
        geff = torch.empty((T - 1, 2), dtype=torch.float64, device=c2pt.device)
        self._chk(lib().mdwf_fh_effective_derivative(self._h, _dev(geff), _dev(c2), _dev(cf), _stream()))
        return torch.view_as_complex(geff)

    def mdwf_wall_inject(self, eta4: torch.Tensor, recon=18):
        ncol = eta4.shape[0]
        b5 = torch.empty((ncol, self.Ls, self.V4, 4, 3), dtype=torch.complex128, device=eta4.device)
        self._chk(lib().mdwf_wall_inject(self._h, _dev(b5), _dev(eta4), ncol, recon, _stream()))
        return b5

    def mdwf_wall_project(self, psi5: torch.Tensor):
        ncol = psi5.shape[0]
        q4 = torch.empty((ncol, self.V4, 4, 3), dtype=torch.complex128, device=psi5.device)
        self._chk(lib().mdwf_wall_project(self._h, _dev(q4), _dev(psi5), ncol, _stream()))
        return q4

    def mdwf_launch_count(self):
        return int(lib().mdwf_launch_count(self._h))

    def mdwf_set_tiling(self, zc):
        self._chk(lib().mdwf_set_tiling(self._h, zc))

    def mdwf_profile(self, enable):
        self._chk(lib().mdwf_profile(self._h, int(bool(enable))))

    def mdwf_profile_read(self, cls):
        """(ms, bytes, flops, launches) of the hop kernel for storage class cls (0 fp16, 1 fp32, 2 fp64)."""
        ms, by, fl, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_double(), ctypes.c_int64()
        self._chk(lib().mdwf_profile_read(self._h, cls, ctypes.byref(ms), ctypes.byref(by), ctypes.byref(fl),
                                          ctypes.byref(n)))
        return ms.value, by.value, fl.value, n.value

"""ctypes binding of libdwf.so (include/dwf.h).  Same names as the C ABI, marshalling only.

torch is used for device memory and streams: every field is a torch CUDA tensor whose data_ptr()
is handed to the library.  Canonical arrays are complex tensors
[nrhs][Ls][t][z][y][x][4][3] (spinor) / [4][t][z][y][x][3][3] (gauge); native fields are opaque
real tensors allocated by `Dwf.field()`.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# DWF_LIB: load another build of the same library (kernel tuning); the default is the in-tree libdwf.so
_LIB_PATH = os.environ.get("DWF_LIB") or os.path.join(_HERE, "libdwf.so")

DWF_F32, DWF_F64 = 0, 1
DWF_DHOP, DWF_DDW, DWF_HDW, DWF_DPV, DWF_SCHUR_EO, DWF_MEE, DWF_MOOINV, DWF_MPVDAG_M, DWF_SCHUR_EO_ALT = range(9)
DWF_DAGGER = 0x100
_HALF_OPS = (DWF_SCHUR_EO, DWF_MEE, DWF_MOOINV, DWF_SCHUR_EO_ALT)

_SIGNATURES = {
    "dwf_create": (ctypes.c_int, [ctypes.POINTER(ctypes.c_int), ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                  ctypes.c_int, ctypes.POINTER(ctypes.c_void_p)]),
    "dwf_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "dwf_set_stream": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "dwf_workspace_bytes": (ctypes.c_size_t, [ctypes.c_void_p, ctypes.c_int]),
    "dwf_set_workspace": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]),
    "dwf_set_gauge": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "dwf_field_bytes": (ctypes.c_size_t, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
    "dwf_import": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
    "dwf_export": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
    "dwf_apply": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dwf_apply_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dwf_chebyshev": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                     ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dwf_chebyshev_subspace": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dwf_chebyshev_smoother": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                              ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dwf_power_lambda_max": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double),
                                            ctypes.POINTER(ctypes.c_double)]),
    "dwf_axpy": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_void_p, ctypes.c_void_p,
                                ctypes.c_int, ctypes.c_int]),
    "dwf_inner": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double),
                                 ctypes.c_int, ctypes.c_int]),
    "dwf_norm2": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int,
                                 ctypes.c_int]),
    "dwf_norm2_static": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
    "dwf_cg_schur": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
                                    ctypes.POINTER(ctypes.c_double)]),
    "dwf_cg_schur_multi": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                          ctypes.POINTER(ctypes.c_double)]),
    "dwf_cg_normal": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                     ctypes.POINTER(ctypes.c_double)]),
    "dwf_bicgstab_pv": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]),
    "dwf_solve": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_int,
                                 ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)]),
    "dwf_convert": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dwf_solve_mixed": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_double,
                                       ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int),
                                       ctypes.POINTER(ctypes.c_double)]),
    "dwf_launch_count": (ctypes.c_longlong, [ctypes.c_void_p]),
    "dwf_last_error": (ctypes.c_char_p, [ctypes.c_void_p]),
}


def lib_path() -> str:
    return _LIB_PATH


def exported_symbols():
    """Names include/dwf.h declares (and this binding expects)."""
    return sorted(_SIGNATURES)


DWF_EINVAL, DWF_ENOGAUGE, DWF_ENOMEM, DWF_ECUDA, DWF_EUNSUPPORTED, DWF_ENOWORKSPACE, DWF_ERANGE = -1, -2, -3, -4, -5, -6, -7


class DwfError(RuntimeError):
    """A negative return code of the C ABI; `.code` is that code."""

    def __init__(self, msg, code=None):
        super().__init__(msg)
        self.code = code


_lib = None


def load():
    """Load libdwf.so; raise loudly if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise DwfError(f"{_LIB_PATH} is missing: run `python -m paper_2103_05034_b200.build` "
                           "(or __graft_entry__.build()); there is no CPU fallback")
        lib = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


class Dwf:
    """One dwf_handle.  Methods are the C calls without the `dwf_` prefix."""

    def __init__(self, L, Ls: int, M5: float, mass: float, precision: int, device="cuda:0"):
        self._h = None
        self.lib = load()
        if not torch.cuda.is_available():
            raise DwfError("no CUDA device: libdwf has no CPU path")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.L = tuple(int(v) for v in L)
        self.Ls, self.M5, self.mass, self.precision = int(Ls), float(M5), float(mass), int(precision)
        self.rdtype = torch.float32 if precision == DWF_F32 else torch.float64
        self.cdtype = torch.complex64 if precision == DWF_F32 else torch.complex128
        h = ctypes.c_void_p()
        rc = self.lib.dwf_create((ctypes.c_int * 4)(*self.L), self.Ls, self.M5, self.mass, self.precision, ctypes.byref(h))
        if rc != 0:
            raise DwfError(f"dwf_create failed with code {rc}")
        self._h = h
        self._ws = None
        self.set_stream(torch.cuda.current_stream(self.device))

    # -- plumbing -------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise DwfError(f"libdwf error {rc}: {self.lib.dwf_last_error(self._h).decode()}", rc)

    def close(self):
        if self._h is not None:
            torch.cuda.synchronize(self.device)
            self.lib.dwf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        self._check(self.lib.dwf_set_stream(self._h, ctypes.c_void_p(stream.cuda_stream)))

    def workspace_bytes(self, nrhs: int) -> int:
        return int(self.lib.dwf_workspace_bytes(self._h, nrhs))

    def set_workspace(self, nrhs: int, half_fields: int = None):
        """Allocate (torch) and register a workspace for `nrhs` right-hand sides: big enough for every call of the library
        (dwf_workspace_bytes), or for `half_fields` half fields when the caller knows which calls it makes (include/dwf.h
        states each call's need; e.g. 5 for dwf_cg_schur at 48^3 x 96 x 24, where the full 12 would not fit beside the fields)."""
        n = self.workspace_bytes(nrhs) if half_fields is None else self.field_bytes(nrhs, half=True) * half_fields + 256
        if self._ws is None or self._ws.numel() < n:
            self._ws = None
            self._ws = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._check(self.lib.dwf_set_workspace(self._h, ctypes.c_void_p(self._ws.data_ptr()), self._ws.numel()))

    def field_bytes(self, nrhs: int, half: bool = False) -> int:
        return int(self.lib.dwf_field_bytes(self._h, nrhs, int(half)))

    def field(self, nrhs: int, half: bool = False, zero: bool = False) -> torch.Tensor:
        """Allocate a native field (opaque 1-D real tensor)."""
        n = self.field_bytes(nrhs, half) // (4 if self.precision == DWF_F32 else 8)
        return (torch.zeros if zero else torch.empty)(n, dtype=self.rdtype, device=self.device)

    def canonical_shape(self, nrhs: int):
        Lx, Ly, Lz, Lt = self.L
        return (nrhs, self.Ls, Lt, Lz, Ly, Lx, 4, 3)

    # -- C ABI ----------------------------------------------------------------------------------
    def set_gauge(self, U: torch.Tensor):
        Lx, Ly, Lz, Lt = self.L
        assert U.is_cuda and U.dtype == self.cdtype and U.is_contiguous() and tuple(U.shape) == (4, Lt, Lz, Ly, Lx, 3, 3)
        self._check(self.lib.dwf_set_gauge(self._h, ctypes.c_void_p(U.data_ptr())))

    def import_(self, canonical: torch.Tensor, native: torch.Tensor = None, parity: int = -1) -> torch.Tensor:
        nrhs = canonical.shape[0]
        assert canonical.is_cuda and canonical.dtype == self.cdtype and canonical.is_contiguous()
        assert tuple(canonical.shape) == self.canonical_shape(nrhs)
        if native is None:
            native = self.field(nrhs, half=(parity >= 0))
        self._check(self.lib.dwf_import(self._h, ctypes.c_void_p(canonical.data_ptr()), ctypes.c_void_p(native.data_ptr()), nrhs, parity))
        return native

    def export(self, native: torch.Tensor, nrhs: int, parity: int = -1, canonical: torch.Tensor = None) -> torch.Tensor:
        if canonical is None:
            canonical = torch.zeros(self.canonical_shape(nrhs), dtype=self.cdtype, device=self.device)
        assert canonical.is_contiguous() and canonical.dtype == self.cdtype
        self._check(self.lib.dwf_export(self._h, ctypes.c_void_p(native.data_ptr()), ctypes.c_void_p(canonical.data_ptr()), nrhs, parity))
        return canonical

    def apply(self, op: int, inp: torch.Tensor, out: torch.Tensor, nrhs: int) -> torch.Tensor:
        self._check(self.lib.dwf_apply(self._h, op, ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr()), nrhs))
        return out

    def apply_host(self, op: int, in_host: torch.Tensor, out_host: torch.Tensor, nrhs: int) -> torch.Tensor:
        assert not in_host.is_cuda and not out_host.is_cuda and in_host.is_contiguous() and out_host.is_contiguous()
        self._check(self.lib.dwf_apply_host(self._h, op, ctypes.c_void_p(in_host.data_ptr()), ctypes.c_void_p(out_host.data_ptr()), nrhs))
        return out_host

    def chebyshev(self, order: int, lo: float, hi: float, inp: torch.Tensor, out: torch.Tensor, nrhs: int) -> torch.Tensor:
        self._check(self.lib.dwf_chebyshev(self._h, order, lo, hi, ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr()), nrhs))
        return out

    def chebyshev_subspace(self, m: int, lambda_lo: float, lambda_max: float, delta: int, nvec: int, eta: torch.Tensor,
                           phi: torch.Tensor, nrhs: int) -> torch.Tensor:
        """phi: 1-D native tensor of nvec * field elements (phi_k = phi[k * n : (k + 1) * n])."""
        assert phi.numel() == nvec * eta.numel()
        self._check(self.lib.dwf_chebyshev_subspace(self._h, m, lambda_lo, lambda_max, delta, nvec, ctypes.c_void_p(eta.data_ptr()),
                                                    ctypes.c_void_p(phi.data_ptr()), nrhs))
        return phi

    def chebyshev_smoother(self, N: int, a: float, b: float, r: torch.Tensor, out: torch.Tensor, nrhs: int) -> torch.Tensor:
        self._check(self.lib.dwf_chebyshev_smoother(self._h, N, a, b, ctypes.c_void_p(r.data_ptr()), ctypes.c_void_p(out.data_ptr()), nrhs))
        return out

    def power_lambda_max(self, iters: int, v: torch.Tensor):
        lam = ctypes.c_double()
        hist = (ctypes.c_double * iters)()
        self._check(self.lib.dwf_power_lambda_max(self._h, iters, ctypes.c_void_p(v.data_ptr()), ctypes.byref(lam), hist))
        return float(lam.value), [float(x) for x in hist]

    def axpy(self, a, x: torch.Tensor, y: torch.Tensor, nrhs: int, half: bool = False):
        a = [complex(v) for v in a]
        assert len(a) == nrhs
        buf = (ctypes.c_double * (2 * nrhs))()
        for r, v in enumerate(a):
            buf[2 * r], buf[2 * r + 1] = v.real, v.imag
        self._check(self.lib.dwf_axpy(self._h, buf, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(y.data_ptr()), nrhs, int(half)))
        return y

    def inner(self, x: torch.Tensor, y: torch.Tensor, nrhs: int, half: bool = False):
        buf = (ctypes.c_double * (2 * nrhs))()
        self._check(self.lib.dwf_inner(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(y.data_ptr()), buf, nrhs, int(half)))
        return [complex(buf[2 * r], buf[2 * r + 1]) for r in range(nrhs)]

    def norm2(self, x: torch.Tensor, nrhs: int, half: bool = False):
        buf = (ctypes.c_double * nrhs)()
        self._check(self.lib.dwf_norm2(self._h, ctypes.c_void_p(x.data_ptr()), buf, nrhs, int(half)))
        return [float(buf[r]) for r in range(nrhs)]

    def norm2_static(self, x: torch.Tensor, out_dev: torch.Tensor, nrhs: int, half: bool = False) -> torch.Tensor:
        """out_dev: float64 CUDA tensor of nrhs elements; no allocation on the C side, asynchronous."""
        assert out_dev.is_cuda and out_dev.dtype == torch.float64 and out_dev.numel() >= nrhs and out_dev.is_contiguous()
        self._check(self.lib.dwf_norm2_static(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(out_dev.data_ptr()), nrhs, int(half)))
        return out_dev

    def cg_schur(self, b_even: torch.Tensor, x_even: torch.Tensor, iters: int):
        hist = (ctypes.c_double * (iters + 1))()
        self._check(self.lib.dwf_cg_schur(self._h, ctypes.c_void_p(b_even.data_ptr()), ctypes.c_void_p(x_even.data_ptr()), iters, hist))
        return [float(v) for v in hist]

    def cg_schur_multi(self, b_even: torch.Tensor, x_even: torch.Tensor, iters: int, nrhs: int):
        """Returns the history as a list of (iters+1) lists of nrhs values."""
        hist = (ctypes.c_double * ((iters + 1) * nrhs))()
        self._check(self.lib.dwf_cg_schur_multi(self._h, ctypes.c_void_p(b_even.data_ptr()), ctypes.c_void_p(x_even.data_ptr()), iters, nrhs, hist))
        return [[float(hist[k * nrhs + r]) for r in range(nrhs)] for k in range(iters + 1)]

    def cg_normal(self, b: torch.Tensor, x: torch.Tensor, iters: int, nrhs: int):
        hist = (ctypes.c_double * ((iters + 1) * nrhs))()
        self._check(self.lib.dwf_cg_normal(self._h, ctypes.c_void_p(b.data_ptr()), ctypes.c_void_p(x.data_ptr()), iters, nrhs, hist))
        return [[float(hist[k * nrhs + r]) for r in range(nrhs)] for k in range(iters + 1)]

    def bicgstab_pv(self, b: torch.Tensor, x: torch.Tensor, iters: int):
        """BiCGSTAB on D_PV^dag D_DW x = b (full fields, nrhs = 1); returns the |r_i|^2 history (iters + 1 values)."""
        hist = (ctypes.c_double * (iters + 1))()
        self._check(self.lib.dwf_bicgstab_pv(self._h, ctypes.c_void_p(b.data_ptr()), ctypes.c_void_p(x.data_ptr()), iters, hist))
        return [float(v) for v in hist]

    def solve(self, eta: torch.Tensor, psi: torch.Tensor, tol: float, max_iters: int):
        """D_DW psi = eta by the complete red-black CGNR solve; returns (iterations, true relative residual)."""
        it, rr = ctypes.c_int(), ctypes.c_double()
        self._check(self.lib.dwf_solve(self._h, ctypes.c_void_p(eta.data_ptr()), ctypes.c_void_p(psi.data_ptr()), tol, max_iters,
                                       ctypes.byref(it), ctypes.byref(rr)))
        return int(it.value), float(rr.value)

    def convert_to(self, dst: "Dwf", inp: torch.Tensor, nrhs: int, out: torch.Tensor = None) -> torch.Tensor:
        """Native field of this handle -> native field of `dst` (other precision / site order)."""
        if out is None:
            out = dst.field(nrhs)
        self._check(self.lib.dwf_convert(self._h, dst._h, ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr()), nrhs))
        return out

    def solve_mixed(self, h32: "Dwf", eta: torch.Tensor, psi: torch.Tensor, tol: float, inner_tol: float, max_outer: int, max_inner: int):
        """self = the fp64 handle.  Returns (outer corrections, total fp32 CG iterations, final relative residual)."""
        o, i, rr = ctypes.c_int(), ctypes.c_int(), ctypes.c_double()
        self._check(self.lib.dwf_solve_mixed(self._h, h32._h, ctypes.c_void_p(eta.data_ptr()), ctypes.c_void_p(psi.data_ptr()), tol, inner_tol,
                                             max_outer, max_inner, ctypes.byref(o), ctypes.byref(i), ctypes.byref(rr)))
        return int(o.value), int(i.value), float(rr.value)

    def launch_count(self) -> int:
        return int(self.lib.dwf_launch_count(self._h))

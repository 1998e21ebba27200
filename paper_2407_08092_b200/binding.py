"""Thin ctypes binding of libddamg.so (include/ddamg.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for
device buffers and streams, nothing else.  There is no CPU fallback: if the shared
library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libddamg.so")

OK, EINVAL, ENOMEM, ESTATE, ECUDA, ESINGULAR = 0, -1, -2, -3, -4, -5
F32, F64 = 0, 1
BC_PERIODIC, BC_ANTIPERIODIC_T = 0, 1
SMOOTHER_RICHARDSON, SMOOTHER_GMRES, SMOOTHER_GCR, SMOOTHER_SAP = 0, 1, 2, 3

_STATUS = {0: "DDAMG_OK", -1: "DDAMG_EINVAL", -2: "DDAMG_ENOMEM", -3: "DDAMG_ESTATE",
           -4: "DDAMG_ECUDA", -5: "DDAMG_ESINGULAR"}

# every symbol include/ddamg.h declares: name -> (restype, argtypes)
_vp, _i, _d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
_dp, _ip, _llp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_longlong)
SYMBOLS = {
    "ddamg_version": (ctypes.c_char_p, []),
    "ddamg_create": (_i, [ctypes.POINTER(_vp), _i, _i, _d, _d, _i, _i, _vp]),
    "ddamg_destroy": (_i, [_vp]),
    "ddamg_last_error": (ctypes.c_char_p, [_vp]),
    "ddamg_half_spinor_bytes": (ctypes.c_size_t, [_vp]),
    "ddamg_load_gauge": (_i, [_vp, _vp, _i, _i]),
    "ddamg_build_clover": (_i, [_vp]),
    "ddamg_apply_schur": (_i, [_vp, _vp, _vp]),
    "ddamg_apply_schur_noalloc": (_i, [_vp, _vp, _vp]),
    "ddamg_noalloc_max_bytes": (ctypes.c_size_t, []),
    "ddamg_richardson": (_i, [_vp, _vp, _vp, _i, _d, _i, _dp]),
    "ddamg_gmres_oe": (_i, [_vp, _vp, _vp, _i, _i, _d, _i, _dp, _ip]),
    "ddamg_gcr_oe": (_i, [_vp, _vp, _vp, _i, _i, _d, _i, _dp, _ip]),
    "ddamg_apply_full": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "ddamg_fgmres": (_i, [_vp, _vp, _vp, _vp, _vp, _i, _i, _d, _i, _i, _i, _d, _i, _dp, _ip]),
    "ddamg_sap": (_i, [_vp, _vp, _vp, _vp, _vp, _i, _i, _ip, _i, _dp]),
    "ddamg_reconstruct_odd": (_i, [_vp, _vp, _vp, _vp]),
    "ddamg_prepare_rhs": (_i, [_vp, _vp, _vp, _vp]),
    "ddamg_power_iteration": (_i, [_vp, _vp, _i, _dp]),
    "ddamg_pack_spinor": (_i, [_vp, _vp, _vp, _vp]),
    "ddamg_unpack_spinor": (_i, [_vp, _vp, _vp, _vp]),
    "ddamg_get_clover": (_i, [_vp, _vp, _vp]),
    "ddamg_batch_spinor_bytes": (ctypes.c_size_t, [_vp, _i]),
    "ddamg_batch_interleave": (_i, [_vp, _i, _vp, _vp]),
    "ddamg_batch_deinterleave": (_i, [_vp, _i, _vp, _vp]),
    "ddamg_apply_schur_batch": (_i, [_vp, _i, _vp, _vp]),
    "ddamg_richardson_batch": (_i, [_vp, _i, _vp, _vp, _i, _d, _i, _dp]),
    "ddamg_reconstruct_odd_batch": (_i, [_vp, _i, _vp, _vp, _vp]),
    "ddamg_prepare_rhs_batch": (_i, [_vp, _i, _vp, _vp, _vp]),
    "ddamg_set_option": (_i, [_vp, ctypes.c_char_p, _d]),
    "ddamg_launch_count": (ctypes.c_longlong, [_vp]),
    "ddamg_kernel_timing": (_i, [_vp, _i]),
    "ddamg_kernel_time_ms": (_i, [_vp, _i, _dp, _llp, _i]),
}

_lib = None


class DdamgError(RuntimeError):
    def __init__(self, status: int, where: str, msg: str):
        super().__init__(f"{where}: {_STATUS.get(status, status)} ({msg})")
        self.status = status


def load_library() -> ctypes.CDLL:
    """dlopen libddamg.so (built in-tree by paper_2407_08092_b200.build). Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


class Ddamg:
    """One lattice / one precision / one stream (``ddamg_ctx``).

    Spinor arguments are native half-lattice device tensors created by :meth:`half_spinor`
    or :meth:`pack`; methods mirror the C entry points one to one.
    """

    def __init__(self, L: int, T: int, csw: float, m0: float, bc: int = BC_ANTIPERIODIC_T,
                 prec: int = F32, stream: Optional[torch.cuda.Stream] = None, device="cuda:0"):
        self.lib = load_library()
        self.L, self.T, self.prec = L, T, prec
        self.V = L * L * L * T
        self.device = torch.device(device)
        self.rdtype = torch.float32 if prec == F32 else torch.float64
        self.cdtype = torch.complex64 if prec == F32 else torch.complex128
        self.stream = stream
        self._h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            s = self.lib.ddamg_create(ctypes.byref(self._h), L, T, csw, m0, bc, prec,
                                      ctypes.c_void_p(stream.cuda_stream if stream is not None else 0))
        if s != OK:
            raise DdamgError(s, "ddamg_create", self.lib.ddamg_last_error(None).decode())
        self.half_bytes = self.lib.ddamg_half_spinor_bytes(self._h)

    # -- plumbing -------------------------------------------------------------
    def _ck(self, s: int, where: str):
        if s != OK:
            raise DdamgError(s, where, self.lib.ddamg_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.lib.ddamg_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def half_spinor(self, zero: bool = False) -> torch.Tensor:
        """A native half-lattice spinor buffer (flat real tensor of 24 * V/2 entries)."""
        n = 12 * self.V
        return (torch.zeros if zero else torch.empty)(n, dtype=self.rdtype, device=self.device)

    def _chk_half(self, *ts):
        for t in ts:
            if t is None:
                continue
            assert t.is_cuda and t.dtype == self.rdtype and t.is_contiguous() and t.numel() == 12 * self.V, \
                "expected a native half-lattice spinor of this context"

    # -- setup ----------------------------------------------------------------
    def load_gauge(self, U: torch.Tensor):
        """U: natural layout (T,L,L,L,4,3,3) complex64/complex128, host or device tensor."""
        assert U.is_contiguous() and U.numel() == self.V * 36
        assert U.dtype in (torch.complex64, torch.complex128)
        u_prec = F32 if U.dtype == torch.complex64 else F64
        self._ck(self.lib.ddamg_load_gauge(self._h, _ptr(U), u_prec, 1 if U.is_cuda else 0), "ddamg_load_gauge")

    def build_clover(self):
        self._ck(self.lib.ddamg_build_clover(self._h), "ddamg_build_clover")

    def pack(self, nat: torch.Tensor, want_even=True, want_odd=True):
        """natural (T,L,L,L,4,3) complex device tensor -> (x_e, x_o) native halves."""
        assert nat.is_cuda and nat.dtype == self.cdtype and nat.is_contiguous() and nat.numel() == 12 * self.V
        xe = self.half_spinor() if want_even else None
        xo = self.half_spinor() if want_odd else None
        self._ck(self.lib.ddamg_pack_spinor(self._h, _ptr(nat), _ptr(xe), _ptr(xo)), "ddamg_pack_spinor")
        return xe, xo

    def unpack(self, x_e: Optional[torch.Tensor], x_o: Optional[torch.Tensor]) -> torch.Tensor:
        self._chk_half(x_e, x_o)
        nat = torch.empty((self.T, self.L, self.L, self.L, 4, 3), dtype=self.cdtype, device=self.device)
        self._ck(self.lib.ddamg_unpack_spinor(self._h, _ptr(x_e), _ptr(x_o), _ptr(nat)), "ddamg_unpack_spinor")
        return nat

    def get_clover(self):
        """(A on even sites, A^-1 on odd sites) as dense (T,L,L,L,2,6,6) complex device tensors."""
        shape = (self.T, self.L, self.L, self.L, 2, 6, 6)
        A = torch.empty(shape, dtype=self.cdtype, device=self.device)
        Ai = torch.empty(shape, dtype=self.cdtype, device=self.device)
        self._ck(self.lib.ddamg_get_clover(self._h, _ptr(A), _ptr(Ai)), "ddamg_get_clover")
        return A, Ai

    # -- hot path ---------------------------------------------------------------
    def apply_schur(self, x_e: torch.Tensor, y_e: Optional[torch.Tensor] = None) -> torch.Tensor:
        y_e = self.half_spinor() if y_e is None else y_e
        self._chk_half(x_e, y_e)
        self._ck(self.lib.ddamg_apply_schur(self._h, _ptr(x_e), _ptr(y_e)), "ddamg_apply_schur")
        return y_e

    def apply_schur_noalloc(self, x_e: torch.Tensor, y_e: torch.Tensor) -> torch.Tensor:
        """ddamg_apply_schur_noalloc: no allocation inside the call (the caller passes y_e); the scratch half
        spinor is a static 8 MiB device array of the library, shared by all calls on the device."""
        self._chk_half(x_e, y_e)
        self._ck(self.lib.ddamg_apply_schur_noalloc(self._h, _ptr(x_e), _ptr(y_e)), "ddamg_apply_schur_noalloc")
        return y_e

    def richardson(self, b_e: torch.Tensor, x_e: torch.Tensor, nu: int, omega: float,
                   zero_init: bool = False, history: bool = False):
        self._chk_half(b_e, x_e)
        hist = (ctypes.c_double * max(nu, 1))() if history else None
        self._ck(self.lib.ddamg_richardson(self._h, _ptr(b_e), _ptr(x_e), nu, omega, int(zero_init), hist),
                 "ddamg_richardson")
        return list(hist)[:nu] if history else None

    def gmres_oe(self, b_e: torch.Tensor, x_e: torch.Tensor, k: int, cycles: int, tol: float = 0.0,
                 zero_init: bool = False):
        self._chk_half(b_e, x_e)
        n = cycles * (k + 1) + 1
        hist = (ctypes.c_double * n)()
        nh = ctypes.c_int(0)
        self._ck(self.lib.ddamg_gmres_oe(self._h, _ptr(b_e), _ptr(x_e), k, cycles, tol, int(zero_init), hist,
                                         ctypes.byref(nh)), "ddamg_gmres_oe")
        return list(hist)[:nh.value]

    def gcr_oe(self, b_e: torch.Tensor, x_e: torch.Tensor, k: int, cycles: int, tol: float = 0.0,
               zero_init: bool = False):
        self._chk_half(b_e, x_e)
        n = cycles * (k + 1) + 1
        hist = (ctypes.c_double * n)()
        nh = ctypes.c_int(0)
        self._ck(self.lib.ddamg_gcr_oe(self._h, _ptr(b_e), _ptr(x_e), k, cycles, tol, int(zero_init), hist,
                                       ctypes.byref(nh)), "ddamg_gcr_oe")
        return list(hist)[:nh.value]

    def apply_full(self, x_e: torch.Tensor, x_o: torch.Tensor):
        """(y_e, y_o) = D (x_e, x_o), the full Wilson-clover operator."""
        y_e, y_o = self.half_spinor(), self.half_spinor()
        self._chk_half(x_e, x_o)
        self._ck(self.lib.ddamg_apply_full(self._h, _ptr(x_e), _ptr(x_o), _ptr(y_e), _ptr(y_o)), "ddamg_apply_full")
        return y_e, y_o

    def fgmres(self, b_e, b_o, x_e, x_o, k: int, cycles: int, tol: float = 0.0, smoother: int = SMOOTHER_RICHARDSON,
               s_n: int = 4, s_m: int = 1, omega: float = 1.0, zero_init: bool = True):
        self._chk_half(b_e, b_o, x_e, x_o)
        n = cycles * (k + 1) + 1
        hist = (ctypes.c_double * n)()
        nh = ctypes.c_int(0)
        self._ck(self.lib.ddamg_fgmres(self._h, _ptr(b_e), _ptr(b_o), _ptr(x_e), _ptr(x_o), k, cycles, tol, smoother,
                                       s_n, s_m, omega, int(zero_init), hist, ctypes.byref(nh)), "ddamg_fgmres")
        return list(hist)[:nh.value]

    def sap(self, b_e, b_o, x_e, x_o, n: int, m: int, block=(4, 4, 4, 4), zero_init: bool = False,
            history: bool = False):
        """Alg. 1: SAP(n, m) on D x = b, in place on (x_e, x_o); history = ||b - D x^(i)||, i = 0..n."""
        self._chk_half(b_e, b_o, x_e, x_o)
        blk = (ctypes.c_int * 4)(*[int(v) for v in block])
        hist = (ctypes.c_double * (n + 1))() if history else None
        self._ck(self.lib.ddamg_sap(self._h, _ptr(b_e), _ptr(b_o), _ptr(x_e), _ptr(x_o), n, m, blk, int(zero_init),
                                    hist), "ddamg_sap")
        return list(hist) if history else None

    def reconstruct_odd(self, b_o: torch.Tensor, x_e: torch.Tensor, x_o: Optional[torch.Tensor] = None):
        x_o = self.half_spinor() if x_o is None else x_o
        self._chk_half(b_o, x_e, x_o)
        self._ck(self.lib.ddamg_reconstruct_odd(self._h, _ptr(b_o), _ptr(x_e), _ptr(x_o)), "ddamg_reconstruct_odd")
        return x_o

    def prepare_rhs(self, b_e: torch.Tensor, b_o: torch.Tensor, bhat_e: Optional[torch.Tensor] = None):
        bhat_e = self.half_spinor() if bhat_e is None else bhat_e
        self._chk_half(b_e, b_o, bhat_e)
        self._ck(self.lib.ddamg_prepare_rhs(self._h, _ptr(b_e), _ptr(b_o), _ptr(bhat_e)), "ddamg_prepare_rhs")
        return bhat_e

    def power_iteration(self, v_e: torch.Tensor, iters: int) -> float:
        self._chk_half(v_e)
        lam = ctypes.c_double(0.0)
        self._ck(self.lib.ddamg_power_iteration(self._h, _ptr(v_e), iters, ctypes.byref(lam)), "ddamg_power_iteration")
        return lam.value

    # -- multi-rhs batching (NEXT-2) ------------------------------------------------
    def batch_numel(self, nrhs: int) -> int:
        """Reals in a batch buffer of nrhs right-hand sides (ddamg_batch_spinor_bytes: an fp32 batch holds
        PAIRS of right-hand sides, so an odd nrhs is padded by one slot)."""
        nbytes = self.lib.ddamg_batch_spinor_bytes(self._h, nrhs)
        return nbytes // (4 if self.rdtype == torch.float32 else 8)

    def batch_spinor(self, nrhs: int, zero: bool = False) -> torch.Tensor:
        """A batch buffer: nrhs native half spinors interleaved per site (flat real tensor)."""
        return (torch.zeros if zero else torch.empty)(self.batch_numel(nrhs), dtype=self.rdtype, device=self.device)

    def _chk_batch(self, nrhs, *ts):
        n = self.batch_numel(nrhs)
        for t in ts:
            assert t.is_cuda and t.dtype == self.rdtype and t.is_contiguous() and t.numel() == n, \
                "expected a batch of nrhs native half spinors of this context"

    def batch_interleave(self, halves, X: Optional[torch.Tensor] = None) -> torch.Tensor:
        """halves: list of native half spinors, or an (nrhs, 12 V) tensor of them -> batch."""
        H = torch.stack(list(halves)) if not isinstance(halves, torch.Tensor) else halves
        nrhs = H.shape[0]
        H = H.contiguous().view(-1)
        X = self.batch_spinor(nrhs) if X is None else X
        assert H.is_cuda and H.dtype == self.rdtype and H.numel() == nrhs * 12 * self.V
        self._chk_batch(nrhs, X)
        self._ck(self.lib.ddamg_batch_interleave(self._h, nrhs, _ptr(H), _ptr(X)), "ddamg_batch_interleave")
        return X

    def batch_deinterleave(self, nrhs: int, X: torch.Tensor) -> torch.Tensor:
        """batch -> (nrhs, 12 V) tensor whose rows are native half spinors."""
        self._chk_batch(nrhs, X)
        H = torch.empty(nrhs * 12 * self.V, dtype=self.rdtype, device=self.device)
        self._ck(self.lib.ddamg_batch_deinterleave(self._h, nrhs, _ptr(X), _ptr(H)), "ddamg_batch_deinterleave")
        return H.view(nrhs, 12 * self.V)

    def apply_schur_batch(self, nrhs: int, X_e: torch.Tensor, Y_e: Optional[torch.Tensor] = None) -> torch.Tensor:
        Y_e = self.batch_spinor(nrhs) if Y_e is None else Y_e
        self._chk_batch(nrhs, X_e, Y_e)
        self._ck(self.lib.ddamg_apply_schur_batch(self._h, nrhs, _ptr(X_e), _ptr(Y_e)), "ddamg_apply_schur_batch")
        return Y_e

    def richardson_batch(self, nrhs: int, B_e: torch.Tensor, X_e: torch.Tensor, nu: int, omega: float,
                         zero_init: bool = False, history: bool = False):
        """history -> list of nu lists of nrhs residual norms."""
        self._chk_batch(nrhs, B_e, X_e)
        hist = (ctypes.c_double * max(nu * nrhs, 1))() if history else None
        self._ck(self.lib.ddamg_richardson_batch(self._h, nrhs, _ptr(B_e), _ptr(X_e), nu, omega, int(zero_init),
                                                 hist), "ddamg_richardson_batch")
        if not history:
            return None
        flat = list(hist)
        return [flat[i * nrhs:(i + 1) * nrhs] for i in range(nu)]

    def reconstruct_odd_batch(self, nrhs: int, B_o: torch.Tensor, X_e: torch.Tensor,
                              X_o: Optional[torch.Tensor] = None) -> torch.Tensor:
        X_o = self.batch_spinor(nrhs) if X_o is None else X_o
        self._chk_batch(nrhs, B_o, X_e, X_o)
        self._ck(self.lib.ddamg_reconstruct_odd_batch(self._h, nrhs, _ptr(B_o), _ptr(X_e), _ptr(X_o)),
                 "ddamg_reconstruct_odd_batch")
        return X_o

    def prepare_rhs_batch(self, nrhs: int, B_e: torch.Tensor, B_o: torch.Tensor,
                          Bhat_e: Optional[torch.Tensor] = None) -> torch.Tensor:
        Bhat_e = self.batch_spinor(nrhs) if Bhat_e is None else Bhat_e
        self._chk_batch(nrhs, B_e, B_o, Bhat_e)
        self._ck(self.lib.ddamg_prepare_rhs_batch(self._h, nrhs, _ptr(B_e), _ptr(B_o), _ptr(Bhat_e)),
                 "ddamg_prepare_rhs_batch")
        return Bhat_e

    def set_option(self, name: str, value: float):
        self._ck(self.lib.ddamg_set_option(self._h, name.encode(), float(value)), "ddamg_set_option")

    # -- accounting ---------------------------------------------------------------
    def launch_count(self) -> int:
        return int(self.lib.ddamg_launch_count(self._h))

    def kernel_timing(self, on: bool):
        self._ck(self.lib.ddamg_kernel_timing(self._h, int(on)), "ddamg_kernel_timing")

    def kernel_time_ms(self, which: int, reset: bool = True):
        ms = ctypes.c_double(0.0)
        n = ctypes.c_longlong(0)
        self._ck(self.lib.ddamg_kernel_time_ms(self._h, which, ctypes.byref(ms), ctypes.byref(n), int(reset)),
                 "ddamg_kernel_time_ms")
        return ms.value, n.value

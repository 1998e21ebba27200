"""CPU fp64 oracle for the odd-even Wilson-clover hot path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It shares no code with
``paper_2407_08092_b200`` (the CUDA library) and neither imports the other.

The operator arithmetic lives in ``oracle/wilson_clover.c`` (plain C, natural
layout, full 4x4 spin matrices); this file is the ctypes marshalling around
it.  The iterations (Richardson, Alg. 4; GMRES, Alg. 2; GCR, Alg. 3; FGMRES) are
written out step by step in ``oracle/iterations.py``, SAP (Alg. 1) in ``oracle/sap.py``.

Parity status: every function is pinned by ``tests/test_oracle_*.py`` against
closed forms / invariants / dense linear algebra; the only *unpinned* items
are the paper's Fig. 1 spectra (gauge field not given -- qualitative check
only) and the paper's Tables 1-2 timings (need the CLQCD ensemble and ORISE).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from .build import build as _build, LIB as _LIB

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        path = os.environ.get("ORACLE_LIB")          # a sanitizer build (tests/test_oracle_sanitizers.py)
        if not path:
            _build()
            path = _LIB
        _lib = ctypes.CDLL(path)
        _lib.oracle_invert_sites.restype = ctypes.c_long
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.complex128 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=np.complex128)


def gamma_matrices() -> np.ndarray:
    """The four 4x4 gamma matrices the oracle uses (reading R1), shape (4,4,4)."""
    g = np.zeros((4, 4, 4), dtype=np.complex128)
    lib().oracle_gamma(_p(g))
    return g


def parity_mask(L: int, T: int) -> np.ndarray:
    """(T,L,L,L) array of (x+y+z+t) mod 2  (even = 0)."""
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    return (x + y + z + t) & 1


class WilsonClover:
    """D = A + H on an L^3 x T lattice and its Schur complement (eq. 1-3).

    ``U``: natural-layout gauge field, shape (T,L,L,L,4,3,3), WITHOUT boundary sign.
    ``bc``: 0 periodic, 1 antiperiodic in time (reading R2).
    All spinors are full-lattice arrays of shape (T,L,L,L,4,3), complex128;
    "x_e" means such an array that is zero on odd sites.
    """

    def __init__(self, L: int, T: int, csw: float, m0: float, bc: int, U):
        self.L, self.T, self.csw, self.m0, self.bc = int(L), int(T), float(csw), float(m0), int(bc)
        self.V = L * L * L * T
        self.shape = (T, L, L, L, 4, 3)
        self.U = _c(U).reshape(T, L, L, L, 4, 3, 3)
        self.Ubc = np.empty_like(self.U)
        lib().oracle_apply_bc(L, T, self.bc, _p(self.U), _p(self.Ubc))
        self.A = np.empty((T, L, L, L, 12, 12), dtype=np.complex128)
        lib().oracle_clover(L, T, ctypes.c_double(self.csw), ctypes.c_double(self.m0), _p(self.U), _p(self.A))
        self.Ainv = np.empty_like(self.A)
        self.n_singular = int(lib().oracle_invert_sites(ctypes.c_long(self.V), _p(self.A), _p(self.Ainv),
                                                        ctypes.c_double(1e-12)))
        self.par = parity_mask(L, T)
        self.even = (self.par == 0)[..., None, None]
        self.odd = (self.par == 1)[..., None, None]

    # -- pieces ------------------------------------------------------------
    def hop(self, psi, sel: int = 2, Ubc=None) -> np.ndarray:
        """(H psi) on even (sel=0), odd (sel=1) or all (sel=2) sites; 0 elsewhere.
        ``Ubc``: link field to use instead of this operator's own (SAP's block-diagonal
        operator is the hopping term of a link field with the inter-block links zeroed)."""
        psi = _c(psi)
        links = self.Ubc if Ubc is None else _c(Ubc)
        out = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_hop(self.L, self.T, _p(links), _p(psi), _p(out), int(sel))
        return out

    def site_matvec(self, M, psi, sel: int = 2) -> np.ndarray:
        psi = _c(psi)
        out = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_site_matvec(self.L, self.T, _p(M), _p(psi), _p(out), int(sel))
        return out

    # -- operators -----------------------------------------------------------
    def apply_D(self, x) -> np.ndarray:
        x = _c(x)
        y = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_apply_D(self.L, self.T, _p(self.Ubc), _p(self.A), _p(x), _p(y))
        return y

    def apply_schur(self, x_e) -> np.ndarray:
        x_e = _c(x_e)
        y = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_apply_schur(self.L, self.T, _p(self.Ubc), _p(self.A), _p(self.Ainv), _p(x_e), _p(y))
        return y

    def prepare_rhs(self, b) -> np.ndarray:
        b = _c(b)
        y = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_prepare_rhs(self.L, self.T, _p(self.Ubc), _p(self.Ainv), _p(b), _p(y))
        return y

    def reconstruct_odd(self, b, x_e) -> np.ndarray:
        b, x_e = _c(b), _c(x_e)
        y = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_reconstruct_odd(self.L, self.T, _p(self.Ubc), _p(self.Ainv), _p(b), _p(x_e), _p(y))
        return y

    # -- dense assembly (tiny lattices only; used by the pins) ---------------
    def dense(self, op) -> np.ndarray:
        """Matrix of a linear map on full-lattice vectors, column by column."""
        n = 12 * self.V
        M = np.empty((n, n), dtype=np.complex128)
        e = np.zeros(n, dtype=np.complex128)
        for j in range(n):
            e[j] = 1.0
            M[:, j] = op(e.reshape(self.shape)).reshape(n)
            e[j] = 0.0
        return M


from .iterations import richardson, richardson_multi, gmres, gcr, fgmres, power_iteration  # noqa: E402,F401
from .sap import sap, BlockOperators, block_index, cut_links, minimal_residual  # noqa: E402,F401

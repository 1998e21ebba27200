"""SAP(n, m), Alg. 1, step by step -- TEST INFRASTRUCTURE.

Plain numpy, fp64, full-lattice vectors in the natural layout, built only from the pieces of
``oracle.WilsonClover`` (hopping term with a chosen link field, site-matrix products).

What the paper fixes: the lattice is divided into contiguous, disjoint
four-dimensional blocks; the blocks are coloured red/black so that no two contiguous blocks
share a colour; per outer iteration the red blocks are processed first ("approximately
solving the linear systems defined on each block"), then the black ones; the block solves
are done via Minimal Residual, m iterations; Alg. 1 recomputes ``r = b - D x`` before each
colour (lines 2 and 7).  With odd-even preconditioning "it is not the whole lattice what is
reordered but rather each of the domain decomposition blocks ... minimal residual is used for
solving the linear systems with the Schur complement of each block".

Readings (R20-R24; the paper gives no formula for any of them):

* R20  block geometry: block extents ``B = (Bx, By, Bz, Bt)``, each dividing the lattice
  extent with an EVEN quotient (so that the two-colouring closes under the periodic wrap);
  block coordinate ``c_mu = x_mu // B_mu``; colour = parity of ``c_x + c_y + c_z + c_t``,
  red = 0.
* R21  "the linear system defined on block k": ``D_k = P_k D P_k^T``, the rows and columns of
  D belonging to the sites of block k.  Equivalently D with every link that joins two
  different blocks set to zero -- which is how it is evaluated here: ``cut_links`` zeroes
  ``U_mu(x)`` whenever ``x`` and ``x + mu`` lie in different blocks, and the ordinary hopping
  routine is then called with that link field.  The site-diagonal part A is unchanged.
* R22  Minimal Residual (the paper cites Saad's book): ``e = 0, rho = rhs``; m times
  ``q = M rho; alpha = <q, rho>/<q, q>; e += alpha rho; rho -= alpha q`` with
  ``<q, rho> = q^H rho`` restricted to the block (local dot products).  No
  relaxation factor.  A block whose ``<q, q>`` is exactly 0 takes alpha = 0.
* R23  block odd-even: eq. 2 written for D_k -- ``rhat_e = r_e - H^k_eo
  A_oo^-1 r_o``; MR(m) on ``D^k_S = A_ee - H^k_eo A_oo^-1 H^k_oe`` from ``e_e = 0``;
  ``e_o = A_oo^-1 (r_o - H^k_oe e_e)``; parity is the GLOBAL site parity.
* R24  history: ``hist[i] = ||b - D x^(i)||_2`` for i = 0..n-1 (the residual of Alg. 1
  line 2, computed anyway), plus the true final residual as the last entry.

Parity status: pinned by ``tests/test_oracle_sap.py`` -- block operator against the dense
sub-blocks of D, Minimal Residual against per-block 1-D least squares and the residual
identity, the odd-even block solve against the plain one, and the converged-block-solve
limit against multiplicative Schwarz with dense block inverses.
"""
from __future__ import annotations

import numpy as np


def _norm(v) -> float:
    return float(np.sqrt(np.vdot(v, v).real))


def block_index(L: int, T: int, block):
    """(T,L,L,L) integer arrays: block number of every site and its colour (R20)."""
    Bx, By, Bz, Bt = (int(v) for v in block)
    ext = (L, L, L, T)
    for e, B in zip(ext, (Bx, By, Bz, Bt)):
        if B < 1 or e % B != 0 or (e // B) % 2 != 0:
            raise ValueError("block extents must divide the lattice with an even quotient")
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    cx, cy, cz, ct = x // Bx, y // By, z // Bz, t // Bt
    nx, ny, nz = L // Bx, L // By, L // Bz
    bid = cx + nx * (cy + ny * (cz + nz * ct))
    colour = (cx + cy + cz + ct) & 1
    return bid, colour


def cut_links(Ubc: np.ndarray, L: int, T: int, block) -> np.ndarray:
    """R21: the link field of the block-diagonal operator.  ``U_mu(x)`` joins x and x + mu; it is
    set to zero when those two sites lie in different blocks, i.e. when x is on the upper
    mu-face of its block (x_mu mod B_mu == B_mu - 1; this includes the periodic wrap)."""
    Ucut = np.array(Ubc, dtype=np.complex128, copy=True).reshape(T, L, L, L, 4, 3, 3)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    for mu, coord in enumerate((x, y, z, t)):
        leaves = (coord % int(block[mu])) == int(block[mu]) - 1
        Ucut[..., mu, :, :][leaves] = 0.0
    return Ucut


def _per_block_sum(vals: np.ndarray, bid: np.ndarray, nblk: int) -> np.ndarray:
    """sum of a per-site quantity over each block (local dot products)."""
    out = np.zeros(nblk, dtype=vals.dtype)
    np.add.at(out, bid.reshape(-1), vals.reshape(-1))
    return out


def minimal_residual(apply, rhs, m: int, bid, nblk: int, return_residual: bool = False):
    """R22 on every block at once: ``apply`` must be block-diagonal, so each block runs its own
    independent iteration with its own alpha.  Vectors have shape (T,L,L,L,4,3)."""
    e = np.zeros_like(rhs)
    rho = np.array(rhs, copy=True)
    for _ in range(m):
        q = apply(rho)
        num = _per_block_sum(np.sum(np.conj(q) * rho, axis=(-1, -2)), bid, nblk)     # <q, rho> = q^H rho
        den = _per_block_sum(np.sum(np.abs(q) ** 2, axis=(-1, -2)), bid, nblk)       # <q, q>
        alpha = np.where(den > 0.0, num / np.where(den > 0.0, den, 1.0), 0.0)
        a = alpha[bid][..., None, None]
        e = e + a * rho
        rho = rho - a * q
    if return_residual:
        return e, rho
    return e


class BlockOperators:
    """The block-diagonal operator sum_k P_k^T D_k P_k (R21) and its block odd-even Schur
    complement (R23) for a ``WilsonClover`` oracle ``op`` and block extents ``block``."""

    def __init__(self, op, block):
        self.op = op
        self.block = tuple(int(v) for v in block)
        self.bid, self.colour = block_index(op.L, op.T, self.block)
        self.nblk = int(self.bid.max()) + 1
        self.Ucut = cut_links(op.Ubc, op.L, op.T, self.block)

    def hop(self, psi, sel: int = 2):
        return self.op.hop(psi, sel, Ubc=self.Ucut)

    def apply_D(self, psi):
        """sum_k P_k^T D_k P_k psi = A psi + H[Ucut] psi."""
        return self.op.site_matvec(self.op.A, psi, 2) + self.hop(psi, 2)

    def apply_schur(self, x_e):
        """D^k_S x_e = A_ee x_e - H^k_eo A_oo^-1 H^k_oe x_e on every block (R23)."""
        op = self.op
        t_o = op.site_matvec(op.Ainv, self.hop(x_e, 1), 1)
        return op.site_matvec(op.A, x_e, 0) - self.hop(t_o, 0)

    def solve(self, r, m: int, odd_even: bool = True):
        """m Minimal Residual iterations on D_k e_k = r_k for every block in the support of r."""
        op = self.op
        if not odd_even:
            return minimal_residual(self.apply_D, r, m, self.bid, self.nblk)
        r_e = np.where(op.even, r, 0.0)
        r_o = np.where(op.odd, r, 0.0)
        rhat_e = r_e - self.hop(op.site_matvec(op.Ainv, r_o, 1), 0)                 # eq. 2, right factor
        e_e = minimal_residual(self.apply_schur, rhat_e, m, self.bid, self.nblk)
        e_o = op.site_matvec(op.Ainv, r_o - self.hop(e_e, 1), 1)                    # eq. 2, left factor
        return e_e + e_o


def sap(op, b, x0, n: int, m: int, block, odd_even: bool = True):
    """Alg. 1: SAP(n, m) on D x = b.  Returns (x^(n), hist) (R24)."""
    blk = BlockOperators(op, block)
    red = (blk.colour == 0)[..., None, None]
    black = (blk.colour == 1)[..., None, None]
    x = np.array(x0, dtype=np.complex128, copy=True)
    b = np.asarray(b, dtype=np.complex128)
    hist = []
    for _ in range(n):                                     # line 1
        r = b - op.apply_D(x)                              # line 2
        hist.append(_norm(r))
        x = x + blk.solve(np.where(red, r, 0.0), m, odd_even)        # lines 4-6: red blocks
        r = b - op.apply_D(x)                              # line 7
        x = x + blk.solve(np.where(black, r, 0.0), m, odd_even)      # lines 8-10: black blocks
    hist.append(_norm(b - op.apply_D(x)))
    return x, hist

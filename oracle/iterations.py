"""The two smoother iterations of the hot path, step by step -- TEST INFRASTRUCTURE.

Plain numpy, fp64, in the paper's order and notation.  ``apply`` is any
callable computing ``D_S x`` (in the tests: ``WilsonClover.apply_schur`` or a
dense matrix).  Vectors are numpy arrays of any shape; inner products run
over all entries.

* ``richardson``  -- Alg. 4 with omega supplied
  (readings R11, R12, R14 of SURVEY.md section 8(c) / DESIGN.md).
* ``gmres``       -- Alg. 2, restarted GMRES(n, m) with the
  modified Gram-Schmidt loop exactly as printed (line 6-7) and the least
  squares problem of line 10 solved by Givens rotations updated every step
  (readings R7, R8, R9, R10, R13).
* ``power_iteration`` -- Alg. 4 line 1 ("approximately compute
  omega = delta/|lambda_max(D)|"; "a few iterations of power
  iteration").
"""
from __future__ import annotations

import numpy as np


def _norm(v) -> float:
    return float(np.sqrt(np.vdot(v, v).real))


def richardson(apply, b, x0, nu: int, omega: float):
    """Alg. 4, lines 2-4:  for i=1..nu:  r = b - D x;  x = x + omega r.

    Returns (x^(nu), hist) with hist[i] = ||b - D x^(i)||_2 for i = 0..nu-1
    (R14: the norm of the residual each sweep computes anyway).
    """
    x = np.array(x0, dtype=np.complex128, copy=True)
    hist = []
    for _ in range(nu):
        r = b - apply(x)                 # Alg. 4 line 3
        hist.append(_norm(r))
        x = x + omega * r                # Alg. 4 line 4
    return x, hist


def gmres(apply, b, x0, k: int, cycles: int, tol: float = 0.0, return_basis: bool = False):
    """Alg. 2: GMRES(n = cycles, m = k) on  D x = b.

    History (R13) = [ ||r|| at the start of every cycle, then the k Givens
    estimates |gamma_{j+1}| of that cycle, ..., and the true ||r|| at the end ].
    With tol > 0 (R10) the cycle is cut as soon as an estimate is
    <= tol * ||b||, and no further cycle starts once the true residual is.
    """
    x = np.array(x0, dtype=np.complex128, copy=True)
    bnorm = _norm(b)
    hist = []
    basis = None
    done = False
    for _ in range(cycles):
        r = b - apply(x)                                   # line 2
        beta = _norm(r)
        hist.append(beta)
        if tol > 0.0 and beta <= tol * bnorm:              # line 3
            done = True
            break
        V = [r / beta]                                     # v_1 = r / beta        (R7)
        H = np.zeros((k + 1, k), dtype=np.complex128)
        cs = np.zeros(k, dtype=np.complex128)
        sn = np.zeros(k, dtype=np.complex128)
        g = np.zeros(k + 1, dtype=np.complex128)           # rotated beta e_1
        g[0] = beta
        m = 0
        for j in range(k):                                 # line 4
            w = apply(V[j])                                # line 5: w = D v_j
            for i in range(j + 1):                         # line 6
                H[i, j] = np.vdot(V[i], w)                 # line 7: h_ij = v_i^H w   (R8)
                w = w - H[i, j] * V[i]
            H[j + 1, j] = _norm(w)                         # line 8
            if H[j + 1, j].real > 0.0:
                V.append(w / H[j + 1, j])                  # v_{j+1}
            else:                                          # exact breakdown
                V.append(np.zeros_like(w))
            # line 10, done incrementally (R9): apply old rotations, make a new one
            for i in range(j):
                t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
                H[i + 1, j] = -np.conj(sn[i]) * H[i, j] + np.conj(cs[i]) * H[i + 1, j]
                H[i, j] = t
            a, c = H[j, j], H[j + 1, j]
            d = np.sqrt(abs(a) ** 2 + abs(c) ** 2)
            cs[j], sn[j] = np.conj(a) / d, np.conj(c) / d
            H[j, j] = cs[j] * a + sn[j] * c                # = d
            H[j + 1, j] = 0.0
            g[j + 1] = -np.conj(sn[j]) * g[j]
            g[j] = cs[j] * g[j]
            hist.append(abs(g[j + 1]))                     # |gamma_{j+1}| = ||beta e_1 - H y||
            m = j + 1
            if tol > 0.0 and abs(g[j + 1]) <= tol * bnorm:
                break
        # back-substitution  R y = g,  then  x = x + V_m y       (line 10)
        y = np.zeros(m, dtype=np.complex128)
        for i in range(m - 1, -1, -1):
            y[i] = (g[i] - np.dot(H[i, i + 1:m], y[i + 1:m])) / H[i, i]
        for i in range(m):
            x = x + y[i] * V[i]
        basis = V
    if not done:
        hist.append(_norm(b - apply(x)))
    if return_basis:
        return x, hist, basis
    return x, hist


def power_iteration(apply, v0, iters: int) -> float:
    """A few power iterations for |lambda_max(D)| (Alg. 4 line 1).

    v <- D v / ||D v||, estimate = ||D v|| / ||v|| of the last step.
    """
    v = np.array(v0, dtype=np.complex128, copy=True)
    v = v / _norm(v)
    lam = 0.0
    for _ in range(iters):
        w = apply(v)
        lam = _norm(w)
        v = w / lam
    return lam


def richardson_multi(apply, B, X0, nu: int, omega: float):
    """Multiple right-hand sides ("apply each block to many vectors",
    multiple rhs): the same Alg. 4 run on every column independently.  ``B``, ``X0`` are
    sequences of vectors; returns (list of x^(nu), hist) with hist[i][r] the residual norm
    of rhs r before sweep i+1.  No new arithmetic: it calls :func:`richardson` per rhs, so
    it inherits that function's pins.
    """
    xs, hists = [], []
    for b, x0 in zip(B, X0):
        x, h = richardson(apply, b, x0, nu, omega)
        xs.append(x)
        hists.append(h)
    return xs, [[hists[r][i] for r in range(len(xs))] for i in range(nu)]


def gcr(apply, b, x0, k: int, cycles: int, tol: float = 0.0):
    """Alg. 3 (PAPER.md:113-131 and the algorithm box after it): GCR(n = cycles, m = k) on D x = b.

    Followed line by line: p_1 = r, z_1 = D p_1; for each step delta_k = (z_k, z_k),
    alpha = (r, z_k)/delta_k, x += alpha p_k, r -= alpha z_k, w = D r,
    beta_j = -(w, z_j)/delta_j, p_{k+1} = r + sum beta_j p_j, z_{k+1} = w + sum beta_j z_j.
    Inner products are conjugate-linear in the direction vector z (reading R8): (a, z) = z^H a.
    The D r / p_{k+1} / z_{k+1} of the last step of a cycle are never used and are skipped.
    History (same layout as ``gmres``, R13): the true ||b - D x|| at the start of every cycle,
    then ||r|| after each of the k updates of line 8 (the recursively updated residual), and
    the true residual norm at the end.  With tol > 0 (R10) stop as soon as ||r|| <= tol ||b||.
    """
    x = np.array(x0, dtype=np.complex128, copy=True)
    bnorm = _norm(b)
    hist = []
    done = False
    for _ in range(cycles):
        r = b - apply(x)                                   # line 2
        hist.append(_norm(r))
        if tol > 0.0 and hist[-1] <= tol * bnorm:          # line 3
            done = True
            break
        P = [r.copy()]                                     # line 4: p_1 = r
        Z = [apply(P[0])]                                  #         z_1 = D p_1
        delta = []
        for j in range(k):                                 # line 5
            delta.append(np.vdot(Z[j], Z[j]).real)         # line 6
            alpha = np.vdot(Z[j], r) / delta[j]            # line 7: (r, z_k) / delta_k
            x = x + alpha * P[j]                           # line 8
            r = r - alpha * Z[j]                           # line 9
            hist.append(_norm(r))
            if tol > 0.0 and hist[-1] <= tol * bnorm:
                break
            if j == k - 1:
                break
            w = apply(r)                                   # line 10
            p_new = r.copy()
            z_new = w.copy()
            for i in range(j + 1):                         # line 11
                beta = -np.vdot(Z[i], w) / delta[i]        # line 12
                p_new = p_new + beta * P[i]                # line 13
                z_new = z_new + beta * Z[i]                # line 14
            P.append(p_new)
            Z.append(z_new)
    if not done:
        hist.append(_norm(b - apply(x)))
    return x, hist


def fgmres(apply, precond, b, x0, k: int, cycles: int, tol: float = 0.0, return_basis: bool = False):
    """Flexible GMRES(n = cycles, m = k): the outer solver of DD-alphaAMG (PAPER.md:77,
    "FGMRES ... preconditioned by" the multigrid cycle; here by the smoother alone).

    The paper prints no algorithm for it; this is Alg. 2 with the one change that makes GMRES
    flexible (reading R19): the Krylov vector is preconditioned before the operator is
    applied, z_j = M(v_j), w = D z_j, the z_j are kept, and the update is x += Z_m y.
    ``precond`` may be any (even non-linear) map.  History layout as in ``gmres``.
    """
    x = np.array(x0, dtype=np.complex128, copy=True)
    bnorm = _norm(b)
    hist = []
    Zs = None
    done = False
    for _ in range(cycles):
        r = b - apply(x)
        beta = _norm(r)
        hist.append(beta)
        if tol > 0.0 and beta <= tol * bnorm:
            done = True
            break
        V = [r / beta]
        Zs = []
        H = np.zeros((k + 1, k), dtype=np.complex128)
        cs = np.zeros(k, dtype=np.complex128)
        sn = np.zeros(k, dtype=np.complex128)
        g = np.zeros(k + 1, dtype=np.complex128)
        g[0] = beta
        m = 0
        for j in range(k):
            Zs.append(precond(V[j]))                       # z_j = M v_j
            w = apply(Zs[j])                               # w = D z_j
            for i in range(j + 1):
                H[i, j] = np.vdot(V[i], w)
                w = w - H[i, j] * V[i]
            H[j + 1, j] = _norm(w)
            V.append(w / H[j + 1, j] if H[j + 1, j].real > 0.0 else np.zeros_like(w))
            for i in range(j):
                t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
                H[i + 1, j] = -np.conj(sn[i]) * H[i, j] + np.conj(cs[i]) * H[i + 1, j]
                H[i, j] = t
            a, c = H[j, j], H[j + 1, j]
            d = np.sqrt(abs(a) ** 2 + abs(c) ** 2)
            cs[j], sn[j] = np.conj(a) / d, np.conj(c) / d
            H[j, j] = cs[j] * a + sn[j] * c
            H[j + 1, j] = 0.0
            g[j + 1] = -np.conj(sn[j]) * g[j]
            g[j] = cs[j] * g[j]
            hist.append(abs(g[j + 1]))
            m = j + 1
            if tol > 0.0 and abs(g[j + 1]) <= tol * bnorm:
                break
        y = np.zeros(m, dtype=np.complex128)
        for i in range(m - 1, -1, -1):
            y[i] = (g[i] - np.dot(H[i, i + 1:m], y[i + 1:m])) / H[i, i]
        for i in range(m):
            x = x + y[i] * Zs[i]                           # x += Z_m y
    if not done:
        hist.append(_norm(b - apply(x)))
    if return_basis:
        return x, hist, Zs
    return x, hist

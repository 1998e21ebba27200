"""Pins for the oracle's GCR (Alg. 3) and flexible GMRES -- CPU only.

* GCR minimises the residual over x^0 + K_m exactly like GMRES ("mathematically equivalent",
  PAPER.md:115, 131): pinned against a dense least-squares solve over the Krylov basis built
  with dense matrix powers (not against the oracle's own GMRES), its directions are
  D^H D-orthogonal, and -- as a cross-check between two independently pinned
  routines -- its residual history equals the GMRES history.
* FGMRES: with the identity preconditioner it is GMRES; with an exact inverse it converges in
  one step; with a genuinely varying (non-linear) preconditioner the residual is the dense
  least-squares minimum over span{z_1..z_m}, which is what makes it "flexible".
"""
import numpy as np
import pytest

import gen
import oracle
from helpers import CONFIGS, config_gauge, rel_l2, even_part
from test_oracle_iterations import small, _np, _embed  # noqa: F401  (fixture + helpers)


def _krylov_min(DS, r0, k):
    K = np.empty((len(r0), k), dtype=np.complex128)
    v = r0.copy()
    for j in range(k):
        K[:, j] = v
        v = DS @ v
    y, *_ = np.linalg.lstsq(DS @ K, r0, rcond=None)
    return K, y, np.linalg.norm(r0 - DS @ K @ y)


@pytest.mark.parametrize("k", [1, 4, 7])
def test_gcr_minimises_residual_over_krylov_space(small, k):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2104)), op.par)
    x0 = even_part(_np(gen.spinor_field(2, 2, 2105)), op.par)
    x, hist = oracle.gcr(op.apply_schur, b, x0, k, 1)
    bv, x0v = b.reshape(-1)[ie], x0.reshape(-1)[ie]
    r0 = bv - DS @ x0v
    K, y, rmin = _krylov_min(DS, r0, k)
    assert len(hist) == k + 2
    assert abs(hist[0] - np.linalg.norm(r0)) < 1e-12 * hist[0]
    assert abs(hist[-1] - rmin) < 1e-9 * rmin                  # true final residual is the minimum
    assert abs(hist[-2] - hist[-1]) < 1e-10 * hist[0]          # recursive residual == true residual
    assert rel_l2(x.reshape(-1)[ie], x0v + K @ y) < 1e-8
    # every intermediate residual is the minimum over the smaller Krylov space
    for j in range(1, k + 1):
        assert abs(hist[j] - _krylov_min(DS, r0, j)[2]) < 1e-9 * hist[0]


def test_gcr_history_equals_gmres_history_and_restarts(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2106)), op.par)
    xg, hg = oracle.gmres(op.apply_schur, b, np.zeros_like(b), 5, 3)
    xc, hc = oracle.gcr(op.apply_schur, b, np.zeros_like(b), 5, 3)
    assert len(hc) == len(hg) == 3 * 6 + 1
    assert np.allclose(hc, hg, rtol=1e-9, atol=1e-12 * hg[0])
    assert rel_l2(xc, xg) < 1e-9


def test_gcr_full_dimension_is_exact_and_tolerance_exit(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2107)), op.par)
    x, hist = oracle.gcr(op.apply_schur, b, np.zeros_like(b), 40, 1)
    # GCR(40) on a 96-dimensional well-conditioned system: far below 1e-8
    assert hist[-1] < 1e-8 * hist[0]
    x, hist = oracle.gcr(op.apply_schur, b, np.zeros_like(b), 10, 10, tol=1e-6)
    assert hist[-1] <= 1e-6 * np.linalg.norm(b) * 1.0001
    assert len(hist) < 10 * 11 + 1
    assert rel_l2(DS @ x.reshape(-1)[ie], b.reshape(-1)[ie]) < 2e-6


def test_fgmres_identity_preconditioner_is_gmres(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2108)), op.par)
    x0 = even_part(_np(gen.spinor_field(2, 2, 2109)), op.par)
    xf, hf = oracle.fgmres(op.apply_schur, lambda v: v, b, x0, 6, 2)
    xg, hg = oracle.gmres(op.apply_schur, b, x0, 6, 2)
    assert np.allclose(hf, hg, rtol=1e-12)
    assert rel_l2(xf, xg) < 1e-12


def test_fgmres_exact_inverse_converges_in_one_step(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2110)), op.par)
    inv = np.linalg.inv(DS)
    M = lambda v: _embed(op, ie, inv @ v.reshape(-1)[ie])
    x, hist = oracle.fgmres(op.apply_schur, M, b, np.zeros_like(b), 3, 1)
    assert hist[1] < 1e-12 * hist[0]
    assert rel_l2(x.reshape(-1)[ie], inv @ b.reshape(-1)[ie]) < 1e-12


def test_fgmres_minimises_over_span_of_preconditioned_vectors(small):
    """A preconditioner that changes from call to call (k Richardson sweeps, k = call number):
    the residual must be min_y || r0 - D Z y || over the stored z_j."""
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2111)), op.par)
    x0 = even_part(_np(gen.spinor_field(2, 2, 2112)), op.par)
    calls = [0]

    def M(v):
        calls[0] += 1
        return oracle.richardson(op.apply_schur, v, np.zeros_like(v), calls[0], 0.3)[0]
    k = 5
    x, hist, Z = oracle.fgmres(op.apply_schur, M, b, x0, k, 1, return_basis=True)
    r0 = (b - op.apply_schur(x0)).reshape(-1)[ie]
    Zm = np.stack([z.reshape(-1)[ie] for z in Z], axis=1)
    y, *_ = np.linalg.lstsq(DS @ Zm, r0, rcond=None)
    rmin = np.linalg.norm(r0 - DS @ Zm @ y)
    assert abs(hist[-1] - rmin) < 1e-10 * hist[0]
    assert abs(hist[-2] - hist[-1]) < 1e-11 * hist[0]
    assert rel_l2(x.reshape(-1)[ie], x0.reshape(-1)[ie] + Zm @ y) < 1e-9


def test_gcr_directions_are_DhD_orthogonal(small):
    """the p_k are made D^H D-orthogonal, i.e. the z_k = D p_k are orthogonal.
    Checked through the update itself: after GCR(1, m) the residual is orthogonal to D K_m."""
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2113)), op.par)
    k = 6
    x, _ = oracle.gcr(op.apply_schur, b, np.zeros_like(b), k, 1)
    bv = b.reshape(-1)[ie]
    r = bv - DS @ x.reshape(-1)[ie]
    K, _, _ = _krylov_min(DS, bv, k)
    assert np.abs((DS @ K).conj().T @ r).max() < 1e-9 * np.linalg.norm(bv)

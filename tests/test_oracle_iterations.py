"""Pins for the oracle's iterations (oracle/iterations.py) -- CPU only.

* Richardson: closed form  x^(k) = x^0 + (I - (I - w D_S)^k) D_S^-1 r^0
  with dense matrices; the M_3 preconditioner statement of PAPER.md:185-187.
* GMRES (Alg. 2): residual minimisation over x^0 + K_m
   against a dense least-squares solve; orthonormal basis;
  Givens estimate == true residual; GMRES(dim) is exact; monotone estimates.
* Power iteration (Alg. 4 line 1) against dense eigenvalues.
"""
import numpy as np
import pytest

import gen
import oracle
from helpers import CONFIGS, config_gauge, config_spinor, rel_l2, even_part


def _np(t):
    return t.cpu().numpy()


@pytest.fixture(scope="module")
def small():
    """Config-1 recipe on 2^4: operator, dense D_S on the even sites, index set."""
    c = CONFIGS[1]
    op = oracle.WilsonClover(2, 2, c["csw"], c["m0"], c["bc"], _np(config_gauge(1, 2, 2)))
    par = np.repeat(op.par.reshape(-1), 12)
    ie = np.where(par == 0)[0]
    DS = op.dense(op.apply_schur)[np.ix_(ie, ie)]
    return op, DS, ie


def _embed(op, ie, v):
    out = np.zeros(12 * op.V, dtype=np.complex128)
    out[ie] = v
    return out.reshape(op.shape)


@pytest.mark.parametrize("omega,k", [(1.0, 4), (0.3, 3), (0.9, 8)])
def test_richardson_closed_form(small, omega, k):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2001)), op.par)
    x0 = even_part(_np(gen.spinor_field(2, 2, 2002)), op.par)
    x, hist = oracle.richardson(op.apply_schur, b, x0, k, omega)
    n = len(ie)
    r0 = b.reshape(-1)[ie] - DS @ x0.reshape(-1)[ie]
    E = np.linalg.matrix_power(np.eye(n) - omega * DS, k)
    expect = x0.reshape(-1)[ie] + (np.eye(n) - E) @ np.linalg.solve(DS, r0)
    assert rel_l2(x.reshape(-1)[ie], expect) < 1e-12
    assert np.all(x.reshape(-1)[np.setdiff1d(np.arange(12 * op.V), ie)] == 0)
    # history: hist[i] = ||(I - w D_S)^i r0||
    r = r0.copy()
    for i in range(k):
        assert abs(hist[i] - np.linalg.norm(r)) < 1e-12 * np.linalg.norm(r)
        r = r - omega * (DS @ r)


def test_richardson_m3_preconditioner_identity():
    """M_3 = eq. 2 with D_S^-1 -> p_{R,3}(D_S); the smoother call
    prepare_rhs -> 3 Richardson sweeps from 0 -> reconstruct_odd applies exactly M_3."""
    c = CONFIGS[1]
    op = oracle.WilsonClover(2, 2, c["csw"], c["m0"], c["bc"], _np(config_gauge(1, 2, 2)))
    D = op.dense(op.apply_D)
    par = np.repeat(op.par.reshape(-1), 12)
    ie, io = np.where(par == 0)[0], np.where(par == 1)[0]
    Dee, Deo, Doe, Doo = D[np.ix_(ie, ie)], D[np.ix_(ie, io)], D[np.ix_(io, ie)], D[np.ix_(io, io)]
    DS = Dee - Deo @ np.linalg.solve(Doo, Doe)
    ne, no = len(ie), len(io)
    omega = 0.3
    pR3 = (np.eye(ne) - np.linalg.matrix_power(np.eye(ne) - omega * DS, 3)) @ np.linalg.inv(DS)
    Dooi = np.linalg.inv(Doo)
    Lf = np.block([[np.eye(ne), np.zeros((ne, no))], [-Dooi @ Doe, np.eye(no)]])
    Mid = np.block([[pR3, np.zeros((ne, no))], [np.zeros((no, ne)), Dooi]])
    Rf = np.block([[np.eye(ne), -Deo @ Dooi], [np.zeros((no, ne)), np.eye(no)]])
    M3 = Lf @ Mid @ Rf
    b = _np(gen.spinor_field(2, 2, 2003))
    bperm = np.concatenate([b.reshape(-1)[ie], b.reshape(-1)[io]])
    expect = M3 @ bperm
    bhat = op.prepare_rhs(b)
    xe, _ = oracle.richardson(op.apply_schur, bhat, np.zeros_like(bhat), 3, omega)
    xo = op.reconstruct_odd(b, xe)
    got = np.concatenate([xe.reshape(-1)[ie], xo.reshape(-1)[io]])
    assert rel_l2(got, expect) < 1e-12


def test_gmres_minimises_residual_over_krylov_space(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2004)), op.par)
    x0 = even_part(_np(gen.spinor_field(2, 2, 2005)), op.par)
    k = 7
    x, hist, V = oracle.gmres(op.apply_schur, b, x0, k, 1, return_basis=True)
    bv, x0v = b.reshape(-1)[ie], x0.reshape(-1)[ie]
    r0 = bv - DS @ x0v
    K = np.empty((len(ie), k), dtype=np.complex128)
    v = r0.copy()
    for j in range(k):
        K[:, j] = v
        v = DS @ v
    # dense least squares: min_y || r0 - D_S K y ||
    y, *_ = np.linalg.lstsq(DS @ K, r0, rcond=None)
    rmin = np.linalg.norm(r0 - DS @ K @ y)
    assert len(hist) == k + 2
    assert abs(hist[0] - np.linalg.norm(r0)) < 1e-12 * hist[0]
    assert abs(hist[-1] - rmin) < 1e-10 * rmin                     # true final residual is the minimum
    assert abs(hist[-2] - hist[-1]) < 1e-12 * hist[0]              # Givens estimate == true residual
    assert rel_l2(x.reshape(-1)[ie], x0v + K @ y) < 1e-9
    # orthonormal Arnoldi basis
    Vm = np.stack([w.reshape(-1) for w in V[:k + 1]], axis=1)
    assert np.abs(Vm.conj().T @ Vm - np.eye(k + 1)).max() < 1e-13
    # monotone non-increasing estimates
    est = np.array(hist[:-1])
    assert np.all(np.diff(est) <= 1e-14 * est[0])


def test_gmres_restart_history_layout_and_cycle_consistency(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2006)), op.par)
    x, hist = oracle.gmres(op.apply_schur, b, np.zeros_like(b), 5, 3)
    assert len(hist) == 3 * (5 + 1) + 1
    for c in range(3):
        end_est = hist[c * 6 + 5]
        nxt_true = hist[(c + 1) * 6] if c < 2 else hist[-1]
        assert abs(end_est - nxt_true) < 1e-12 * hist[0]
    bv = b.reshape(-1)[ie]
    assert abs(np.linalg.norm(bv - DS @ x.reshape(-1)[ie]) - hist[-1]) < 1e-12 * hist[0]


def test_gmres_full_dimension_is_exact_solve(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2007)), op.par)
    x, hist = oracle.gmres(op.apply_schur, b, np.zeros_like(b), len(ie), 1)
    expect = np.linalg.solve(DS, b.reshape(-1)[ie])
    assert rel_l2(x.reshape(-1)[ie], expect) < 1e-10
    assert hist[-1] < 1e-10 * hist[0]


def test_gmres_tolerance_exit(small):
    op, DS, ie = small
    b = even_part(_np(gen.spinor_field(2, 2, 2008)), op.par)
    x, hist = oracle.gmres(op.apply_schur, b, np.zeros_like(b), 10, 10, tol=1e-6)
    assert hist[-1] <= 1e-6 * np.linalg.norm(b) * 1.0001
    assert len(hist) < 10 * 11 + 1


def test_power_iteration_against_dense_spectrum(small):
    op, DS, ie = small
    lam_max = np.abs(np.linalg.eigvals(DS)).max()
    v0 = even_part(_np(gen.spinor_field(2, 2, 2009)), op.par)
    est = oracle.power_iteration(op.apply_schur, v0, 200)
    assert abs(est - lam_max) < 0.05 * lam_max
    few = oracle.power_iteration(op.apply_schur, v0, 10)          # "approximately"
    assert 0.7 * lam_max < few < 1.1 * lam_max


def test_config1_richardson_diverges_at_prescribed_omega_and_converges_at_papers():
    """with omega = 1.0 (config 1) rho(I - w D_S) > 1, the history grows;
    with the paper's omega = 1.5/|lambda_max| it decreases."""
    c = CONFIGS[1]
    op = oracle.WilsonClover(4, 4, c["csw"], c["m0"], c["bc"], _np(config_gauge(1)))
    b = even_part(_np(config_spinor(1, 0)), op.par)
    _, h1 = oracle.richardson(op.apply_schur, b, np.zeros_like(b), 6, 1.0)
    assert np.all(np.diff(h1) > 0)
    lam = oracle.power_iteration(op.apply_schur, b, 20)
    _, h2 = oracle.richardson(op.apply_schur, b, np.zeros_like(b), 6, 1.5 / lam)
    assert np.all(np.diff(h2) < 0)

"""Pins for the oracle's SAP(n, m) (Alg. 1; oracle/sap.py) -- CPU only.

None of these re-types the oracle's recurrences; each compares with dense linear algebra on
the matrix of the oracle's own (separately pinned) D, or with a property the paper states.

* block operator (R21): its dense matrix equals the diagonal blocks P_k D P_k^T of dense D and
  is exactly zero between different blocks ("linear systems defined on each block", Alg. 1
  lines 5, 9); two-colouring: no two contiguous blocks share a colour.
* Minimal Residual (R22): each step's alpha is the 1-D least-squares minimiser of
  ||rho - alpha M rho|| on every block separately (numpy lstsq); the recursive residual equals
  rhs - M e; residual norms never increase.
* block odd-even (R23): with converged block solves the odd-even and the plain
  variant give the same e_k = D_k^-1 r_k (dense solve).
* whole iteration: with converged block solves SAP(n, .) equals multiplicative Schwarz,
  x <- x + sum_{k red} P_k^T D_k^-1 P_k (b - D x), then black (dense block inverses);
  SAP reduces the residual monotonically on the config-1 recipe.
"""
import numpy as np
import pytest

import gen
import oracle
from helpers import CONFIGS, config_gauge, rel_l2


def _np(t):
    return t.cpu().numpy()


@pytest.fixture(scope="module")
def lat4():
    """Config-1 recipe on 4^4 with 2^4 blocks (16 blocks, 8 per colour); dense D (3072^2)."""
    c = CONFIGS[1]
    op = oracle.WilsonClover(4, 4, c["csw"], c["m0"], c["bc"], _np(config_gauge(1, 4, 4)))
    blk = oracle.BlockOperators(op, (2, 2, 2, 2))
    D = op.dense(op.apply_D)
    dof_bid = np.repeat(blk.bid.reshape(-1), 12)
    dof_col = np.repeat(blk.colour.reshape(-1), 12)
    return op, blk, D, dof_bid, dof_col


def test_two_colouring_no_contiguous_blocks_share_a_colour():
    for (L, T, block) in [(4, 4, (2, 2, 2, 2)), (8, 8, (4, 4, 4, 4)), (8, 16, (4, 2, 4, 4)), (4, 8, (2, 2, 2, 2))]:
        bid, col = oracle.block_index(L, T, block)
        for axis in range(4):                       # arrays are (t,z,y,x)
            nb_bid = np.roll(bid, -1, axis=axis)
            nb_col = np.roll(col, -1, axis=axis)
            crossing = nb_bid != bid
            assert crossing.any()
            assert np.all(nb_col[crossing] != col[crossing])
        # blocks are contiguous boxes of the stated size, each with one colour
        sizes = np.bincount(bid.reshape(-1))
        assert np.all(sizes == np.prod(block))
        for k in range(sizes.size):
            assert np.unique(col[bid == k]).size == 1
        assert np.sum(col == 0) == np.sum(col == 1)
    with pytest.raises(ValueError):
        oracle.block_index(4, 4, (4, 2, 2, 2))      # one block along x: the wrap would join it to itself
    with pytest.raises(ValueError):
        oracle.block_index(12, 12, (4, 4, 4, 4))    # three blocks per axis cannot be two-coloured


def test_block_operator_is_block_diagonal_part_of_dense_D(lat4):
    op, blk, D, dof_bid, _ = lat4
    Dblk = op.dense(blk.apply_D)
    same = dof_bid[:, None] == dof_bid[None, :]
    assert np.abs(Dblk[~same]).max() == 0.0
    assert np.abs(Dblk[same] - D[same]).max() < 1e-14
    # and D really couples different blocks (the cut is not vacuous)
    assert np.abs(D[~same]).max() > 0.1


def test_block_schur_is_schur_complement_of_each_dense_block(lat4):
    op, blk, D, dof_bid, _ = lat4
    par = np.repeat(op.par.reshape(-1), 12)
    rng = np.random.default_rng(5)
    x_e = np.where(op.even, rng.standard_normal(op.shape) + 1j * rng.standard_normal(op.shape), 0.0)
    y = blk.apply_schur(x_e).reshape(-1)
    assert np.all(y[par == 1] == 0)
    for k in (0, 5, 15):
        e = np.where((dof_bid == k) & (par == 0))[0]
        o = np.where((dof_bid == k) & (par == 1))[0]
        S = D[np.ix_(e, e)] - D[np.ix_(e, o)] @ np.linalg.solve(D[np.ix_(o, o)], D[np.ix_(o, e)])
        assert rel_l2(y[e], S @ x_e.reshape(-1)[e]) < 1e-13


def test_minimal_residual_steps_are_blockwise_least_squares(lat4):
    op, blk, D, dof_bid, _ = lat4
    rng = np.random.default_rng(6)
    rhs = rng.standard_normal(op.shape) + 1j * rng.standard_normal(op.shape)
    prev_rho = rhs
    prev_e = np.zeros_like(rhs)
    for m in (1, 2, 3):
        e, rho = oracle.minimal_residual(blk.apply_D, rhs, m, blk.bid, blk.nblk, return_residual=True)
        # recursive residual is the true residual of the block system
        assert rel_l2(rho, rhs - blk.apply_D(e)) < 1e-13
        q = blk.apply_D(prev_rho).reshape(-1)
        for k in (0, 3, 9, 15):
            idx = np.where(dof_bid == k)[0]
            alpha, *_ = np.linalg.lstsq(q[idx, None], prev_rho.reshape(-1)[idx], rcond=None)
            assert rel_l2(e.reshape(-1)[idx], prev_e.reshape(-1)[idx] + alpha[0] * prev_rho.reshape(-1)[idx]) < 1e-12
            assert np.linalg.norm(rho.reshape(-1)[idx]) <= np.linalg.norm(prev_rho.reshape(-1)[idx]) * (1 + 1e-14)
        prev_rho, prev_e = rho, e


def test_converged_block_solves_equal_dense_block_inverse_with_and_without_odd_even(lat4):
    op, blk, D, dof_bid, dof_col = lat4
    rng = np.random.default_rng(7)
    r = rng.standard_normal(op.shape) + 1j * rng.standard_normal(op.shape)
    r_red = np.where((blk.colour == 0)[..., None, None], r, 0.0)
    e_oe = blk.solve(r_red, 150, odd_even=True).reshape(-1)
    e_pl = blk.solve(r_red, 400, odd_even=False).reshape(-1)
    assert np.all(e_oe[dof_col == 1] == 0)                       # untouched blocks get no correction
    for k in np.unique(dof_bid[dof_col == 0])[:4]:
        idx = np.where(dof_bid == k)[0]
        exact = np.linalg.solve(D[np.ix_(idx, idx)], r.reshape(-1)[idx])
        assert rel_l2(e_oe[idx], exact) < 1e-10
        assert rel_l2(e_pl[idx], exact) < 1e-8


def _schwarz_dense(D, dof_bid, dof_col, b, x, n):
    for _ in range(n):
        for colour in (0, 1):
            r = b - D @ x
            for k in np.unique(dof_bid[dof_col == colour]):
                idx = np.where(dof_bid == k)[0]
                x[idx] += np.linalg.solve(D[np.ix_(idx, idx)], r[idx])
    return x


def test_sap_with_converged_block_solves_is_multiplicative_schwarz(lat4):
    op, blk, D, dof_bid, dof_col = lat4
    b = _np(gen.spinor_field(4, 4, 2301))
    x0 = _np(gen.spinor_field(4, 4, 2302))
    x, hist = oracle.sap(op, b, x0, 2, 150, (2, 2, 2, 2))
    expect = _schwarz_dense(D, dof_bid, dof_col, b.reshape(-1).copy(), x0.reshape(-1).copy(), 2)
    assert rel_l2(x.reshape(-1), expect) < 1e-9
    assert len(hist) == 3
    assert abs(hist[0] - np.linalg.norm(b.reshape(-1) - D @ x0.reshape(-1))) < 1e-11 * hist[0]
    assert abs(hist[-1] - np.linalg.norm(b.reshape(-1) - D @ expect)) < 1e-7 * hist[0]


def test_sap_one_mr_step_by_hand_on_one_block(lat4):
    """SAP(1,1) from x = 0, plain (non odd-even) block solve: on a red block k the update is
    alpha_k r_k with alpha_k = <D_k r_k, r_k>/<D_k r_k, D_k r_k>, r = b -- dense arithmetic."""
    op, blk, D, dof_bid, dof_col = lat4
    b = _np(gen.spinor_field(4, 4, 2303))
    # stop after the red half: compare only on red blocks, which the black half does not touch
    x, _ = oracle.sap(op, b, np.zeros_like(b), 1, 1, (2, 2, 2, 2), odd_even=False)
    bv = b.reshape(-1)
    for k in np.unique(dof_bid[dof_col == 0])[:3]:
        idx = np.where(dof_bid == k)[0]
        q = D[np.ix_(idx, idx)] @ bv[idx]
        alpha = np.vdot(q, bv[idx]) / np.vdot(q, q)
        assert rel_l2(x.reshape(-1)[idx], alpha * bv[idx]) < 1e-13


def test_sap_reduces_the_residual_and_odd_even_helps_the_block_solves():
    c = CONFIGS[1]
    op = oracle.WilsonClover(4, 4, c["csw"], c["m0"], c["bc"], _np(config_gauge(1, 4, 4)))
    b = _np(gen.spinor_field(4, 4, 2304))
    _, h_oe = oracle.sap(op, b, np.zeros_like(b), 3, 4, (2, 2, 2, 2), odd_even=True)
    _, h_pl = oracle.sap(op, b, np.zeros_like(b), 3, 4, (2, 2, 2, 2), odd_even=False)
    assert all(h_oe[i + 1] < h_oe[i] for i in range(3))
    assert all(h_pl[i + 1] < h_pl[i] for i in range(3))
    assert h_oe[0] == h_pl[0] == pytest.approx(np.linalg.norm(b))
    assert h_oe[-1] < h_pl[-1]          # "it only helps the block solves in SAP to converge faster"

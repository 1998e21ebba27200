"""GPU parity of the multi-rhs (batched) path -- SURVEY.md NEXT-2.

Each *_batch entry point must compute, per right-hand side, what its single-rhs namesake
computes: checked element by element against the fp64 oracle (same tolerances as the
single-rhs path) and, GPU against GPU, bit for bit against the single-rhs kernels.
"""
import numpy as np
import pytest
import torch

from helpers import CONFIGS, rel_l2
from test_gpu_parity import make_pair, _mods

pytestmark = pytest.mark.gpu


def _spinors(p, nrhs, seed0):
    """nrhs full-lattice spinors: (list of numpy complex128, list of (x_e, x_o) native halves)."""
    nps, halves = [], []
    for r in range(nrhs):
        a, d = p.spinor(seed0 + r)
        nps.append(a)
        halves.append(p.ctx.pack(d))
    return nps, halves


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("nrhs", [1, 2, 3, 4, 8])
def test_batch_interleave_layout_and_roundtrip(prec, nrhs):
    p = make_pair(1, prec, 4, 6)
    _, halves = _spinors(p, nrhs, 7000)
    H = torch.stack([h[0] for h in halves])                  # (nrhs, 24 * Vh)
    X = p.ctx.batch_interleave(H)
    Vh = p.ctx.V // 2
    if prec == "f64":
        # documented layout (include/ddamg.h): plane j of double2, vector index cb * nrhs + r
        expect = H.view(nrhs, 12, Vh, 2).permute(1, 2, 0, 3).contiguous().view(-1)
    else:
        # documented fp32 layout: 12 half-planes of float4; half-plane h, vector cb * npairs + p =
        # (re, re', im, im') of complex number h of the site for the rhs 2p, 2p+1 (odd nrhs: zero padding)
        npairs = (nrhs + 1) // 2
        Hp = torch.zeros(2 * npairs, 24 * Vh, dtype=H.dtype, device=H.device)
        Hp[:nrhs] = H
        c = Hp.view(npairs, 2, 6, Vh, 2, 2)                  # pair, lane, plane, cb, complex-in-vector, re/im
        expect = c.permute(2, 4, 3, 0, 5, 1).contiguous().view(-1)     # plane, complex, cb, pair, re/im, lane
    assert X.numel() == expect.numel()
    assert torch.equal(X, expect)
    assert torch.equal(p.ctx.batch_deinterleave(nrhs, X), H)


CASES = [
    (1, "f64", 4, 4, 3), (1, "f32", 4, 4, 4), (1, "f64", 2, 2, 2),
    (3, "f32", 6, 8, 5),        # V/2 * 5 = 4320 threads: ragged last CTA, rhs groups straddle warps
    (3, "f32", 6, 8, 8), (2, "f32", 8, 8, 32), (3, "f64", 4, 6, 7),
]


@pytest.mark.parametrize("cfg,prec,L,T,nrhs", CASES)
def test_batch_apply_prepare_reconstruct(cfg, prec, L, T, nrhs):
    p = make_pair(cfg, prec, L, T)
    x_np, xh = _spinors(p, nrhs, 7100)
    b_np, bh = _spinors(p, nrhs, 7200)
    X_e = p.ctx.batch_interleave([h[0] for h in xh])
    B_e = p.ctx.batch_interleave([h[0] for h in bh])
    B_o = p.ctx.batch_interleave([h[1] for h in bh])
    Y = p.ctx.batch_deinterleave(nrhs, p.ctx.apply_schur_batch(nrhs, X_e))
    Bh = p.ctx.batch_deinterleave(nrhs, p.ctx.prepare_rhs_batch(nrhs, B_e, B_o))
    Xo = p.ctx.batch_deinterleave(nrhs, p.ctx.reconstruct_odd_batch(nrhs, B_o, X_e))
    for r in range(nrhs):
        # vs the oracle (eq. 3, eq. 2 right and left factors)
        assert rel_l2(p.to_np(Y[r].contiguous(), None), p.ora.apply_schur(p.even(x_np[r]))) <= p.apply_tol
        assert rel_l2(p.to_np(Bh[r].contiguous(), None), p.ora.prepare_rhs(b_np[r])) <= p.apply_tol
        assert rel_l2(p.to_np(None, Xo[r].contiguous()),
                      p.ora.reconstruct_odd(b_np[r], p.even(x_np[r]))) <= p.apply_tol
        # vs the single-rhs kernels: same arithmetic in the same order
        assert torch.equal(Y[r], p.ctx.apply_schur(xh[r][0]))
        assert torch.equal(Bh[r], p.ctx.prepare_rhs(bh[r][0], bh[r][1]))
        assert torch.equal(Xo[r], p.ctx.reconstruct_odd(bh[r][1], xh[r][0]))


@pytest.mark.parametrize("cfg,prec,L,T,nrhs,nu", [
    (1, "f64", 4, 4, 3, 4), (1, "f32", 4, 4, 4, 4), (3, "f32", 8, 8, 4, 4), (3, "f32", 6, 8, 5, 3),
    (2, "f32", 8, 8, 8, 8),
])
def test_batch_richardson_matches_oracle(cfg, prec, L, T, nrhs, nu):
    oracle, _ = _mods()
    p = make_pair(cfg, prec, L, T)
    omega = CONFIGS[cfg]["omega"]
    b_np, bh = _spinors(p, nrhs, 7300)
    x_np, xh = _spinors(p, nrhs, 7400)
    B_e = p.ctx.batch_interleave([h[0] for h in bh])
    X_e = p.ctx.batch_interleave([h[0] for h in xh])
    X_nohist = X_e.clone()
    hist = p.ctx.richardson_batch(nrhs, B_e, X_e, nu, omega, history=True)
    xs_ref, h_ref = oracle.richardson_multi(p.ora.apply_schur, [p.even(b) for b in b_np],
                                            [p.even(x) for x in x_np], nu, omega)
    got = p.ctx.batch_deinterleave(nrhs, X_e)
    for r in range(nrhs):
        assert rel_l2(p.to_np(got[r].contiguous(), None), xs_ref[r]) <= (1e-11 if p.f64 else 2e-5)
        for i in range(nu):
            assert abs(hist[i][r] - h_ref[i][r]) <= 1e-4 * h_ref[i][r]
        # bit-identical to the single-rhs call
        x1 = xh[r][0].clone()
        h1 = p.ctx.richardson(bh[r][0], x1, nu, omega, history=True)
        assert torch.equal(got[r], x1)
        assert np.allclose([hist[i][r] for i in range(nu)], h1, rtol=1e-13, atol=0)
    # the history-free call (the one bench.py times) gives the same iterate
    p.ctx.richardson_batch(nrhs, B_e, X_nohist, nu, omega)
    assert torch.equal(X_nohist, X_e)
    # x0 = 0
    Z = torch.full_like(X_e, 3.0)
    p.ctx.richardson_batch(nrhs, B_e, Z, 1, omega, zero_init=True)
    assert torch.equal(Z, B_e * omega)                      # (padding lanes of an odd fp32 batch are 0 in both)


def test_batch_error_codes():
    _, dd = _mods()
    p = make_pair(1, "f32", 4, 4)
    X = p.ctx.batch_spinor(2, zero=True)
    Y = p.ctx.batch_spinor(2)
    lib, h = p.ctx.lib, p.ctx._h
    import ctypes
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    assert lib.ddamg_apply_schur_batch(h, 0, vp(X), vp(Y)) == dd.binding.EINVAL
    assert lib.ddamg_apply_schur_batch(h, 33, vp(X), vp(Y)) == dd.binding.EINVAL
    assert lib.ddamg_apply_schur_batch(h, 2, vp(X), vp(X)) == dd.binding.EINVAL
    assert lib.ddamg_richardson_batch(h, 2, vp(X), vp(Y), -1, 1.0, 0, None) == dd.binding.EINVAL
    assert lib.ddamg_batch_interleave(h, 2, None, vp(Y)) == dd.binding.EINVAL
    fresh = dd.Ddamg(4, 4, 1.0, 0.0, 1, dd.F32)
    assert fresh.lib.ddamg_apply_schur_batch(fresh._h, 2, vp(X), vp(Y)) == dd.binding.ESTATE
    assert lib.ddamg_apply_schur_batch(h, 2, vp(X), vp(Y)) == dd.binding.OK


@pytest.mark.parametrize("budget", [0.0, 3 * 2 * 4 * 8 * 4 * 96.0, 1e12])
def test_batch_z_chunked_traversal_is_bit_identical(budget):
    """The z-chunked CTA order (option batch_l2_bytes) only permutes which CTA does which sites:
    results, including the per-rhs residual history, are bit-identical to the single-rhs path.
    8^3 x 6, nrhs = 4: one (z,t) plane = 4 * 8 * 4 threads = 1 CTA, so chunking is active for
    budget 0 (zc = 1) and for a budget of two planes (zc = 2), and off for the huge one."""
    p = make_pair(3, "f32", 8, 6)
    nrhs, nu, omega = 4, 3, 0.9
    _, bh = _spinors(p, nrhs, 7500)
    _, xh = _spinors(p, nrhs, 7600)
    p.ctx.set_option("batch_l2_bytes", budget)
    B_e = p.ctx.batch_interleave([h[0] for h in bh])
    X_e = p.ctx.batch_interleave([h[0] for h in xh])
    Y = p.ctx.batch_deinterleave(nrhs, p.ctx.apply_schur_batch(nrhs, X_e))
    hist = p.ctx.richardson_batch(nrhs, B_e, X_e, nu, omega, history=True)
    got = p.ctx.batch_deinterleave(nrhs, X_e)
    for r in range(nrhs):
        assert torch.equal(Y[r], p.ctx.apply_schur(xh[r][0]))
        x1 = xh[r][0].clone()
        h1 = p.ctx.richardson(bh[r][0], x1, nu, omega, history=True)
        assert torch.equal(got[r], x1)
        assert np.allclose([hist[i][r] for i in range(nu)], h1, rtol=1e-13, atol=0)
    with pytest.raises(Exception):
        p.ctx.set_option("no_such_option", 1.0)

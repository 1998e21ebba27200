"""GPU parity of SAP(n, m) (Alg. 1) vs the oracle.

The oracle (oracle/sap.py) recomputes r = b - D x before each colour and runs the per-block
odd-even Minimal Residual with numpy on full-lattice vectors; the CUDA path does the block
solves with one CTA per block out of shared memory.  Same seeded inputs, element by element.
"""
import ctypes

import numpy as np
import pytest
import torch

from helpers import rel_l2
from test_gpu_parity import make_pair, _mods

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,prec,L,T,block,n,m", [
    (1, "f64", 4, 4, (2, 2, 2, 2), 2, 3),        # config 1, smallest blocks (8 of 32 lanes active)
    (1, "f32", 4, 4, (2, 2, 2, 2), 2, 3),
    (4, "f32", 8, 8, (4, 4, 4, 4), 3, 4),        # the paper's SAP(3,4) on 4^4 blocks (Tables 1, 2, 6)
    (4, "f64", 8, 8, (4, 4, 4, 4), 3, 4),
    (3, "f32", 8, 16, (4, 2, 4, 4), 2, 4),       # anisotropic block, ragged last warp (64 of 64), 4 blocks along t
    (2, "f64", 8, 8, (2, 4, 2, 4), 1, 5),
    (3, "f32", 8, 16, (4, 4, 4, 8), 1, 2),       # 512-site blocks: 256 threads, the fp32 maximum
    (2, "f32", 16, 16, (4, 4, 4, 4), 2, 4),      # 256 blocks: several CTAs per SM wave
    (1, "f32", 4, 8, (2, 2, 2, 4), 2, 1),        # m = 1
])
def test_sap_matches_oracle(cfg, prec, L, T, block, n, m):
    oracle, _ = _mods()
    p = make_pair(cfg, prec, L, T)
    b_np, b_d = p.spinor(9000 + cfg)
    x_np, x_d = p.spinor(9050 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    x_e, x_o = p.ctx.pack(x_d)
    hist = p.ctx.sap(b_e, b_o, x_e, x_o, n, m, block, zero_init=False, history=True)
    x_ref, h_ref = oracle.sap(p.ora, b_np, x_np, n, m, block)
    assert len(hist) == n + 1
    tol_h = 1e-10 if p.f64 else 1e-4
    for a, r in zip(hist, h_ref):
        assert abs(a - r) <= tol_h * r, (hist, h_ref)
    assert rel_l2(p.to_np(x_e, x_o), x_ref) <= (1e-11 if p.f64 else 2e-5)
    # zero initial guess, no history (asynchronous path): bit-identical to the history path
    y_e, y_o = p.ctx.half_spinor(), p.ctx.half_spinor()
    y_e.fill_(7.0); y_o.fill_(-3.0)                                   # must be ignored
    p.ctx.sap(b_e, b_o, y_e, y_o, n, m, block, zero_init=True)
    z_e, z_o = p.ctx.half_spinor(zero=True), p.ctx.half_spinor(zero=True)
    h0 = p.ctx.sap(b_e, b_o, z_e, z_o, n, m, block, zero_init=False, history=True)
    assert torch.equal(y_e, z_e) and torch.equal(y_o, z_o)
    x0_ref, h0_ref = oracle.sap(p.ora, b_np, np.zeros_like(b_np), n, m, block)
    assert rel_l2(p.to_np(y_e, y_o), x0_ref) <= (1e-11 if p.f64 else 2e-5)
    assert abs(h0[0] - np.linalg.norm(b_np)) <= (1e-12 if p.f64 else 1e-6) * h0[0]
    assert all(abs(a - r) <= tol_h * r for a, r in zip(h0, h0_ref))


@pytest.mark.parametrize("cfg,prec,L,T,block", [
    (4, "f32", 8, 8, (4, 4, 4, 4)),
    (3, "f32", 8, 16, (4, 2, 4, 4)),
    (1, "f64", 4, 8, (2, 2, 2, 4)),
])
def test_sap_block_ordered_and_native_residual_storage_agree(cfg, prec, L, T, block):
    """Option "sap_blocked": r and e kept block-ordered (default) or as native half spinors.  Same arithmetic per
    site, so the iterate is bit-identical; only the summation order of the history norms differs."""
    p = make_pair(cfg, prec, L, T)
    _, b_d = p.spinor(9100 + cfg)
    _, x_d = p.spinor(9150 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    out = {}
    for mode in (1, 0):
        p.ctx.set_option("sap_blocked", mode)
        for zero_init in (False, True):
            x_e, x_o = p.ctx.pack(x_d)
            hist = p.ctx.sap(b_e, b_o, x_e, x_o, 2, 3, block, zero_init=zero_init, history=True)
            out[(mode, zero_init)] = (x_e, x_o, hist)
    p.ctx.set_option("sap_blocked", 1)
    for zero_init in (False, True):
        a, b = out[(1, zero_init)], out[(0, zero_init)]
        assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
        assert all(abs(u - v) <= (1e-13 if p.f64 else 1e-6) * v for u, v in zip(a[2], b[2]))


def test_sap_smooths_and_m0_is_identity():
    """SAP(n, 4) reduces the residual every iteration; SAP(n, 0) leaves x untouched."""
    p = make_pair(4, "f32", 8, 8)
    b_np, b_d = p.spinor(9101)
    b_e, b_o = p.ctx.pack(b_d)
    x_e, x_o = p.ctx.half_spinor(zero=True), p.ctx.half_spinor(zero=True)
    hist = p.ctx.sap(b_e, b_o, x_e, x_o, 4, 4, (4, 4, 4, 4), history=True)
    assert all(hist[i + 1] < 0.7 * hist[i] for i in range(4)), hist
    keep_e, keep_o = x_e.clone(), x_o.clone()
    h = p.ctx.sap(b_e, b_o, x_e, x_o, 2, 0, (4, 4, 4, 4), history=True)
    assert torch.equal(keep_e, x_e) and torch.equal(keep_o, x_o)
    assert h[0] == h[1] == h[2] and abs(h[0] - hist[-1]) <= 1e-5 * hist[-1]


def test_sap_error_codes():
    _, dd = _mods()
    E = dd.binding
    p = make_pair(1, "f64", 8, 8)
    b = [p.ctx.half_spinor(zero=True) for _ in range(4)]
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    lib, h = p.ctx.lib, p.ctx._h
    blk = lambda *v: (ctypes.c_int * 4)(*v)
    call = lambda block, n=1, m=1, xe=b[2]: lib.ddamg_sap(h, vp(b[0]), vp(b[1]), vp(xe), vp(b[3]), n, m, block, 0, None)
    assert call(blk(4, 4, 4, 4)) == E.OK
    assert call(blk(8, 4, 4, 4)) == E.EINVAL          # one block along x
    assert call(blk(3, 4, 4, 4)) == E.EINVAL          # odd extent
    assert call(blk(4, 4, 4, 4), n=-1) == E.EINVAL
    assert call(blk(4, 4, 4, 4), m=-1) == E.EINVAL
    assert call(blk(4, 4, 4, 4), xe=b[0]) == E.EINVAL  # x_e aliases b_e
    assert call(None) == E.EINVAL
    p2 = make_pair(1, "f64", 8, 16)
    c = [p2.ctx.half_spinor(zero=True) for _ in range(4)]
    # 512-site blocks in fp64: 295 KB of links, more than a CTA's shared memory
    assert p2.ctx.lib.ddamg_sap(p2.ctx._h, vp(c[0]), vp(c[1]), vp(c[2]), vp(c[3]), 1, 1, blk(4, 4, 4, 8), 0, None) == E.EINVAL
    assert b"shared memory" in p2.ctx.lib.ddamg_last_error(p2.ctx._h)


@pytest.mark.parametrize("cfg,prec,L,T,block,k,s_n,s_m", [
    (1, "f64", 4, 4, (2, 2, 2, 2), 5, 2, 3),
    (4, "f32", 8, 8, (4, 4, 4, 4), 6, 1, 4),
])
def test_fgmres_with_sap_smoother_matches_oracle(cfg, prec, L, T, block, k, s_n, s_m):
    """Outer FGMRES preconditioned by z = SAP(s_n, s_m) v from z = 0: the paper's default solver
    configuration (Table 6) minus the coarse grid.  SAP is a fixed linear map, so the oracle's
    FGMRES with the oracle's SAP as preconditioner is the reference."""
    from test_gpu_parity import _check_history
    oracle, dd = _mods()
    p = make_pair(cfg, prec, L, T)
    for name, B in zip(("sap_block_x", "sap_block_y", "sap_block_z", "sap_block_t"), block):
        p.ctx.set_option(name, B)
    b_np, b_d = p.spinor(9200 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    x_e, x_o = p.ctx.half_spinor(), p.ctx.half_spinor()
    hist = p.ctx.fgmres(b_e, b_o, x_e, x_o, k, 1, 0.0, dd.SMOOTHER_SAP, s_n, s_m, 0.0, zero_init=True)
    M = lambda v: oracle.sap(p.ora, v, np.zeros_like(v), s_n, s_m, block)[0]
    x_ref, h_ref = oracle.fgmres(p.ora.apply_D, M, b_np, np.zeros_like(b_np), k, 1)
    _check_history(hist, h_ref, np.linalg.norm(b_np), p.f64)
    assert rel_l2(p.to_np(x_e, x_o), x_ref) <= (1e-8 if p.f64 else 1e-4)
    assert hist[-1] < 1e-2 * hist[0]                       # SAP-preconditioned FGMRES converges fast


def test_sap_options_error_codes():
    _, dd = _mods()
    p = make_pair(1, "f32")
    with pytest.raises(dd.DdamgError):
        p.ctx.set_option("sap_block_x", 3)
    with pytest.raises(dd.DdamgError):
        p.ctx.set_option("sap_block_q", 4)
    b_e, b_o, x_e, x_o = (p.ctx.half_spinor(zero=True) for _ in range(4))
    # default 4^4 blocks do not two-colour a 4^4 lattice: the smoother reports it
    with pytest.raises(dd.DdamgError):
        p.ctx.fgmres(b_e, b_o, x_e, x_o, 2, 1, 0.0, dd.SMOOTHER_SAP, 1, 1, 0.0)
    with pytest.raises(dd.DdamgError):
        p.ctx.fgmres(b_e, b_o, x_e, x_o, 2, 1, 0.0, dd.SMOOTHER_SAP, 1, 0, 0.0)

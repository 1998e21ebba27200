"""GPU parity of odd-even GCR(n, m) (Alg. 3) vs the oracle."""
import numpy as np
import pytest
import torch

from helpers import rel_l2
from test_gpu_parity import make_pair, _mods, _check_history

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,prec,k,cycles,L,T", [
    (1, "f64", 5, 2, None, None),
    (1, "f32", 5, 2, None, None),
    (4, "f32", 10, 2, 8, 8),          # config 4 recipe, GCR(2,10) on a small lattice
    (4, "f64", 10, 2, 8, 8),
    (2, "f32", 14, 1, 8, 8),          # k > 12: lines 11-14 run in more than one fused chunk
    (3, "f64", 1, 3, 6, 8),           # m = 1: every cycle is one minimal-residual step
])
def test_gcr_matches_oracle(cfg, prec, k, cycles, L, T):
    oracle, _ = _mods()
    p = make_pair(cfg, prec, L, T)
    b_np, b_d = p.spinor(2000 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    bhat = p.ctx.prepare_rhs(b_e, b_o)
    bhat_np = p.to_np(bhat, None)
    x_e = p.ctx.half_spinor()
    hist = p.ctx.gcr_oe(bhat, x_e, k, cycles, zero_init=True)
    x_ref, h_ref = oracle.gcr(p.ora.apply_schur, bhat_np, np.zeros_like(bhat_np), k, cycles)
    assert len(hist) == cycles * (k + 1) + 1
    _check_history(hist, h_ref, np.linalg.norm(bhat_np), p.f64)
    assert rel_l2(p.to_np(x_e, None), x_ref) <= (1e-9 if p.f64 else 5e-5)
    # non-zero initial guess
    x_np, x_d = p.spinor(2070 + cfg)
    x_e2, _ = p.ctx.pack(x_d)
    hist2 = p.ctx.gcr_oe(bhat, x_e2, k, 1, zero_init=False)
    x_ref2, h_ref2 = oracle.gcr(p.ora.apply_schur, bhat_np, p.even(x_np), k, 1)
    _check_history(hist2, h_ref2, np.linalg.norm(bhat_np), p.f64)
    assert rel_l2(p.to_np(x_e2, None), x_ref2) <= (1e-9 if p.f64 else 5e-5)


def test_gcr_equals_gmres_on_the_gpu_and_tolerance_exit():
    """the two methods minimise the same residual over the same space."""
    p = make_pair(1, "f64")
    b_np, b_d = p.spinor(2001)
    b_e, b_o = p.ctx.pack(b_d)
    bhat = p.ctx.prepare_rhs(b_e, b_o)
    xg, xc = p.ctx.half_spinor(), p.ctx.half_spinor()
    hg = p.ctx.gmres_oe(bhat, xg, 6, 2, zero_init=True)
    hc = p.ctx.gcr_oe(bhat, xc, 6, 2, zero_init=True)
    assert np.allclose(hc, hg, rtol=1e-8)
    assert rel_l2(xc.cpu().numpy(), xg.cpu().numpy()) < 1e-9
    # eq. 2 end to end with a tolerance
    x_e = p.ctx.half_spinor()
    hist = p.ctx.gcr_oe(bhat, x_e, 10, 20, tol=1e-10, zero_init=True)
    assert len(hist) < 20 * 11 + 1
    x = p.to_np(x_e, p.ctx.reconstruct_odd(b_o, x_e))
    assert rel_l2(p.ora.apply_D(x), b_np) < 1e-9


def test_gcr_error_codes():
    _, dd = _mods()
    p = make_pair(1, "f32")
    b = p.ctx.half_spinor(zero=True)
    x = p.ctx.half_spinor(zero=True)
    import ctypes
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    lib, h = p.ctx.lib, p.ctx._h
    assert lib.ddamg_gcr_oe(h, vp(b), vp(x), 0, 1, 0.0, 1, None, None) == dd.binding.EINVAL
    assert lib.ddamg_gcr_oe(h, vp(b), vp(b), 2, 1, 0.0, 1, None, None) == dd.binding.EINVAL
    assert lib.ddamg_gcr_oe(h, vp(b), vp(x), 65, 1, 0.0, 1, None, None) == dd.binding.EINVAL
    assert lib.ddamg_gcr_oe(h, vp(b), vp(x), 2, 1, 0.0, 1, None, None) == dd.binding.OK

"""GPU parity with two-row (12-real) link storage (option "gauge_recon" = 12).

The fused hopping kernels read rows 0, 1 of each SU(3) link and rebuild row 2 in registers.
Same bars as the 18-real path (north_star): fp64 apply <= 1e-12, fp32 apply <= 5e-6 relative
L2 against the oracle, which always consumes the full (rounded) links.
"""
import numpy as np
import pytest
import torch

import gen
from helpers import CONFIGS, rel_l2
from test_gpu_parity import make_pair, _mods

pytestmark = pytest.mark.gpu


def make_pair12(cfg, prec, L=None, T=None, bc=None):
    p = make_pair(cfg, prec, L, T, bc)
    p.ctx.set_option("gauge_recon", 12)
    return p


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("cfg,L,T,bc", [(1, 2, 2, 1), (1, 4, 4, 1), (1, 4, 6, 0), (3, 6, 8, 1), (2, 16, 16, 1)])
def test_recon12_schur_apply_and_eq2_factors(prec, cfg, L, T, bc):
    p = make_pair12(cfg, prec, L, T, bc)
    xn, xd = p.spinor(2000 + cfg)
    bn, bd = p.spinor(2100 + cfg)
    x_e, _ = p.ctx.pack(xd)
    b_e, b_o = p.ctx.pack(bd)
    y = p.to_np(p.ctx.apply_schur(x_e), None)
    assert rel_l2(y, p.ora.apply_schur(p.even(xn))) <= p.apply_tol
    assert np.all(y[p.ora.par == 1] == 0)
    bh = p.to_np(p.ctx.prepare_rhs(b_e, b_o), None)
    assert rel_l2(bh, p.ora.prepare_rhs(bn)) <= p.apply_tol
    xo = p.to_np(None, p.ctx.reconstruct_odd(b_o, x_e))
    assert rel_l2(xo, p.ora.reconstruct_odd(bn, p.even(xn))) <= p.apply_tol


@pytest.mark.parametrize("cfg,prec,nu,L,T", [(1, "f64", 4, None, None), (2, "f32", 8, None, None), (3, "f32", 4, 8, 8)])
def test_recon12_richardson_matches_oracle(cfg, prec, nu, L, T):
    oracle, _ = _mods()
    p = make_pair12(cfg, prec, L, T)
    omega = CONFIGS[cfg]["omega"]
    bn, bd = p.spinor(2000 + cfg)
    xn, xd = p.spinor(2050 + cfg)
    b_e, _ = p.ctx.pack(bd)
    x_e, _ = p.ctx.pack(xd)
    hist = p.ctx.richardson(b_e, x_e, nu, omega, zero_init=False, history=True)
    x_ref, h_ref = oracle.richardson(p.ora.apply_schur, p.even(bn), p.even(xn), nu, omega)
    assert max(abs(a - r) / r for a, r in zip(hist, h_ref)) <= 1e-4
    assert rel_l2(p.to_np(x_e, None), x_ref) <= (1e-11 if p.f64 else 2e-5)


def test_recon12_gmres_full_operator_and_batch():
    """Every other consumer of the fused hopping kernel reads the two-row links too."""
    oracle, _ = _mods()
    p = make_pair12(3, "f32", 8, 8)
    bn, bd = p.spinor(2003)
    b_e, b_o = p.ctx.pack(bd)
    x_e = p.ctx.half_spinor(zero=True)
    gh = p.ctx.gmres_oe(b_e, x_e, 6, 1, zero_init=True)
    be = p.even(bn)
    _, g_ref = oracle.gmres(p.ora.apply_schur, be, np.zeros_like(be), 6, 1)
    nb = np.linalg.norm(be)
    assert all(abs(a - r) <= 1e-4 * r + 32 * np.finfo(np.float32).eps * nb for a, r in zip(gh, g_ref))
    y_e, y_o = p.ctx.apply_full(b_e, b_o)
    assert rel_l2(p.to_np(y_e, y_o), p.ora.apply_D(bn)) <= p.apply_tol
    nrhs = 3
    halves = [p.ctx.pack(p.spinor(2200 + r)[1])[0] for r in range(nrhs)]
    Y = p.ctx.batch_deinterleave(nrhs, p.ctx.apply_schur_batch(nrhs, p.ctx.batch_interleave(halves)))
    for r in range(nrhs):
        assert torch.equal(Y[r], p.ctx.apply_schur(halves[r]))      # batch = single-rhs kernel, bit for bit


def test_recon12_close_to_full_links_and_option_order():
    """Set before or after load_gauge: same result; 12 vs 18 differ by rounding only."""
    _, dd = _mods()
    c = CONFIGS[3]
    U = gen.gauge_field(8, 8, 1003, c["eps"], c["reunit"]).to(torch.complex64).cuda()
    x = gen.spinor_field(8, 8, 7).to(torch.complex64).cuda()
    outs = []
    for mode in ("18", "before", "after"):
        ctx = dd.Ddamg(8, 8, c["csw"], c["m0"], 1, dd.F32)
        if mode == "before":
            ctx.set_option("gauge_recon", 12)
        ctx.load_gauge(U)
        if mode == "after":
            ctx.set_option("gauge_recon", 12)
        ctx.build_clover()
        x_e, _ = ctx.pack(x)
        outs.append(ctx.apply_schur(x_e))
    assert torch.equal(outs[1], outs[2])
    d = (outs[1] - outs[0]).norm() / outs[0].norm()
    assert 0 < d < 1e-6
    ctx.set_option("gauge_recon", 18)                               # and back
    assert torch.equal(ctx.apply_schur(x_e), outs[0])


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_recon12_refuses_non_su3_links(prec):
    _, dd = _mods()
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    U = gen.gauge_field(4, 4, 11, 0.3, False).to(cdt)
    U[1, 2, 3, 0, 2] *= 1.001                                        # one link no longer unitary
    ctx = dd.Ddamg(4, 4, 1.0, -0.1, 1, dd.F64 if prec == "f64" else dd.F32)
    ctx.load_gauge(U.cuda())
    with pytest.raises(dd.DdamgError) as e:
        ctx.set_option("gauge_recon", 12)
    assert e.value.status == dd.EINVAL and "SU(3)" in str(e.value)
    ctx.build_clover()                                               # context still usable, on 18-real links
    x_e, _ = ctx.pack(gen.spinor_field(4, 4, 3).to(cdt).cuda())
    assert torch.isfinite(torch.view_as_real(ctx.unpack(ctx.apply_schur(x_e), None))).all()
    with pytest.raises(dd.DdamgError):
        ctx.set_option("gauge_recon", 16)

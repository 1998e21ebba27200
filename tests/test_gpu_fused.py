"""Fused sweep (option "fused_sweep"): kernels A and B / B' of one Schur apply / Richardson sweep
as ONE launch, pipelined time slice by time slice through L2 (csrc/ddamg_sweep_kernel.cuh).

The per-site arithmetic is the two-launch path's, so every result must be BIT-identical to it
(which the other GPU tests compare with the oracle); here additionally one direct oracle check.
Covers the task order for T = 2, T = lag + 2, T > lag + 2, several lags, both link formats,
the in-place Richardson update, the fused residual-norm history, and lattices whose time slice
is not a whole number of CTA tiles (silently served by the two-launch path).
"""
import numpy as np
import pytest
import torch

import gen
from helpers import CONFIGS, rel_l2
from test_gpu_parity import make_pair, _mods

pytestmark = pytest.mark.gpu


def _ctx(L, T, prec, recon, bc=1):
    _, dd = _mods()
    c = CONFIGS[3]
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    ctx = dd.Ddamg(L, T, c["csw"], c["m0"], bc, dd.F64 if prec == "f64" else dd.F32)
    ctx.load_gauge(gen.gauge_field(L, T, 77, c["eps"], True).to(cdt).cuda())
    ctx.build_clover()
    if recon == 12:
        ctx.set_option("gauge_recon", 12)
    x_e, _ = ctx.pack(gen.spinor_field(L, T, 5).to(cdt).cuda())
    b_e, _ = ctx.pack(gen.spinor_field(L, T, 6).to(cdt).cuda())
    return ctx, x_e, b_e


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("L,T,prec,lag", [
    (8, 2, "f32", 2),        # T = 2: both time neighbours coincide, all A tasks first
    (8, 4, "f32", 2),        # T = lag + 2: all A tasks first
    (8, 8, "f32", 1),        # minimal lag: B(t) directly behind the A task it needs
    (8, 8, "f64", 2),
    (8, 12, "f32", 3),
    (16, 16, "f32", 2),      # 16 tiles per slice
    (16, 6, "f32", 64),      # lag larger than T
])
def test_fused_sweep_is_bit_identical_to_two_launches(L, T, prec, lag, recon):
    ctx, x_e, b_e = _ctx(L, T, prec, recon)
    y_ref = ctx.apply_schur(x_e)
    xr = x_e.clone()
    h_ref = ctx.richardson(b_e, xr, 3, 0.9, history=True)
    xr2 = x_e.clone()
    ctx.richardson(b_e, xr2, 3, 0.9)
    n0 = ctx.launch_count()
    ctx.set_option("fused_sweep", 1)
    ctx.set_option("sweep_lag", lag)
    for _ in range(3):                                   # repeated: the ticket / counters are re-armed every launch
        assert torch.equal(ctx.apply_schur(x_e), y_ref)
    xf = x_e.clone()
    h = ctx.richardson(b_e, xf, 3, 0.9, history=True)    # in place, fused ||r||^2 partials
    assert h == h_ref and torch.equal(xf, xr)
    xf2 = x_e.clone()
    n1 = ctx.launch_count()
    ctx.richardson(b_e, xf2, 3, 0.9)
    assert ctx.launch_count() - n1 == 3                  # one launch per sweep instead of two
    assert torch.equal(xf2, xr2)
    assert n0 > 0


def test_fused_sweep_matches_oracle():
    oracle, _ = _mods()
    p = make_pair(3, "f32", 8, 8)
    p.ctx.set_option("fused_sweep", 1)
    xn, xd = p.spinor(2003)
    bn, bd = p.spinor(2053)
    x_e, _ = p.ctx.pack(xd)
    b_e, _ = p.ctx.pack(bd)
    assert rel_l2(p.to_np(p.ctx.apply_schur(x_e), None), p.ora.apply_schur(p.even(xn))) <= 5e-6
    hist = p.ctx.richardson(b_e, x_e, 4, 0.9, history=True)
    x_ref, h_ref = oracle.richardson(p.ora.apply_schur, p.even(bn), p.even(xn), 4, 0.9)
    assert max(abs(a - r) / r for a, r in zip(hist, h_ref)) <= 1e-4
    assert rel_l2(p.to_np(x_e, None), x_ref) <= 2e-5


@pytest.mark.parametrize("L,T", [(4, 4), (6, 8)])
def test_fused_sweep_falls_back_when_a_slice_is_not_whole_tiles(L, T):
    ctx, x_e, b_e = _ctx(L, T, "f32", 18)
    y_ref = ctx.apply_schur(x_e)
    ctx.set_option("fused_sweep", 1)
    n = ctx.launch_count()
    assert torch.equal(ctx.apply_schur(x_e), y_ref)
    assert ctx.launch_count() - n == 2                   # kernel A + kernel B


def test_fused_sweep_option_validation():
    _, dd = _mods()
    ctx = dd.Ddamg(8, 8, 1.0, 0.0, 1, dd.F32)
    for name, bad in (("fused_sweep", 2), ("sweep_lag", 0), ("sweep_lag", 2.5)):
        with pytest.raises(dd.DdamgError) as e:
            ctx.set_option(name, bad)
        assert e.value.status == dd.EINVAL

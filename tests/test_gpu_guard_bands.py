"""Out-of-bounds writes: every output-producing entry point writes into a buffer that sits between
two guard bands filled with a sentinel bit pattern; afterwards the bands must be bit-unchanged and
the payload fully overwritten (no sentinel left).  compute-sanitizer is closed on this GPU pool, so
this is the memory check of the CUDA path: ragged lattices (V/2 not a multiple
of the CTA size), the smallest lattice, both precisions, both link formats, multi-rhs, SAP.
"""
import pytest
import torch

import gen
from helpers import CONFIGS
from test_gpu_parity import _mods

pytestmark = pytest.mark.gpu

GUARD = 4096                      # reals on each side (16-byte aligned for fp32 and fp64)
SENT32, SENT64 = -1.2345678e30, -1.2345678901234567e300


class Guarded:
    def __init__(self, ctx, n, dtype):
        self.sent = SENT32 if dtype == torch.float32 else SENT64
        self.big = torch.full((n + 2 * GUARD,), self.sent, dtype=dtype, device="cuda")
        self.view = self.big[GUARD:GUARD + n]
        assert self.view.data_ptr() % 16 == 0

    def check(self, what):
        torch.cuda.synchronize()
        s = torch.tensor(self.sent, dtype=self.big.dtype, device="cuda")
        assert torch.equal(self.big[:GUARD], s.expand(GUARD)), f"{what}: wrote below the buffer"
        assert torch.equal(self.big[-GUARD:], s.expand(GUARD)), f"{what}: wrote above the buffer"
        assert not (self.view == s).any(), f"{what}: part of the output was never written"
        self.big.fill_(self.sent)


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("L,T", [(2, 2), (6, 8), (4, 6), (8, 8)])
def test_outputs_stay_inside_their_buffers(L, T, prec, recon):
    _, dd = _mods()
    c = CONFIGS[3]
    f64 = prec == "f64"
    cdt, rdt = (torch.complex128, torch.float64) if f64 else (torch.complex64, torch.float32)
    ctx = dd.Ddamg(L, T, c["csw"], c["m0"], 1, dd.F64 if f64 else dd.F32)
    ctx.load_gauge(gen.gauge_field(L, T, 9, c["eps"], True).to(cdt).cuda())
    ctx.build_clover()
    if recon == 12:
        ctx.set_option("gauge_recon", 12)
    nat = gen.spinor_field(L, T, 4).to(cdt).cuda()
    n = 12 * L ** 3 * T
    ge, go = Guarded(ctx, n, rdt), Guarded(ctx, n, rdt)
    ctx.lib.ddamg_pack_spinor(ctx._h, nat.data_ptr(), ge.view.data_ptr(), go.view.data_ptr())
    x_e, x_o = ge.view.clone(), go.view.clone()
    ge.check("pack_spinor even"); go.check("pack_spinor odd")
    b_e, b_o = ctx.pack(gen.spinor_field(L, T, 5).to(cdt).cuda())

    ctx.apply_schur(x_e, ge.view); ge.check("apply_schur")
    ctx.prepare_rhs(b_e, b_o, ge.view); ge.check("prepare_rhs")
    ctx.reconstruct_odd(b_o, x_e, go.view); go.check("reconstruct_odd")
    ge.view.copy_(x_e)
    ctx.richardson(b_e, ge.view, 3, 0.3, history=True); ge.check("richardson")
    ctx.richardson(b_e, ge.view, 2, 0.3, zero_init=True); ge.check("richardson zero_init")
    ctx.gmres_oe(b_e, ge.view, 4, 2, zero_init=True); ge.check("gmres_oe")
    ctx.gcr_oe(b_e, ge.view, 4, 2, zero_init=True); ge.check("gcr_oe")
    ge.view.copy_(x_e); go.view.copy_(x_o)
    if L % 4 == 0 and T % 4 == 0:                         # 2^4 blocks need an even number of blocks per axis
        ctx.sap(b_e, b_o, ge.view, go.view, 2, 2, block=(2, 2, 2, 2)); ge.check("sap even"); go.check("sap odd")
    ctx.fgmres(b_e, b_o, ge.view, go.view, 3, 1, zero_init=True); ge.check("fgmres even"); go.check("fgmres odd")
    # natural-layout output
    gn = Guarded(ctx, 24 * L ** 3 * T, rdt)
    ctx.lib.ddamg_unpack_spinor(ctx._h, x_e.data_ptr(), x_o.data_ptr(), gn.view.data_ptr()); gn.check("unpack_spinor")
    # multi-rhs
    nrhs = 3
    gb = Guarded(ctx, ctx.batch_numel(nrhs), rdt)               # fp32: rhs pairs, the odd rhs is padded
    X = ctx.batch_interleave([x_e, b_e, x_e])
    ctx.apply_schur_batch(nrhs, X, gb.view); gb.check("apply_schur_batch")
    gb.view.copy_(X)
    ctx.richardson_batch(nrhs, ctx.batch_interleave([b_e, b_e, x_e]), gb.view, 2, 0.3); gb.check("richardson_batch")

"""SAP(n, m) (Alg. 1) at FULL size -- config 5, 64^3 x 128, fp32, two-row links, 4^4 blocks: the
launch configuration of bench.py's SAP row (65536 CTAs per colour, TMA-staged links and 6x6 blocks, block-ordered
residual) -- on sampled blocks the oracle can compute.

One SAP iteration is local: the update of a red block depends on r = b - D x on that block (x within one site, links
within two sites of it); the update of a black block additionally on the updates of its red face neighbours.  So the
oracle is run on a box of 6^4 blocks (24^4 sites) cut out of the GPU's own inputs as if it were periodic (the
antiperiodic sign applied to the cut links by hand, as in test_gpu_fullsize.py); its SAP(1, m) result is exact on the
2^4 blocks at the centre of the box (local block coordinates 2..3: 8 red and 8 black blocks, 8^4 sites), whose red
neighbours (block coordinates 1..4) and their halos (reaching into blocks 0 and 5) lie inside the box.  The box origin
is a block corner with an even sum of block coordinates, so that the box-local two-colouring is the global one.
Box 0 is interior; box 1 has the periodic seams of all four axes and the antiperiodic time boundary running through
the compared core.  Both entry modes are compared: a non-zero initial guess with history, and the zero initial guess
without history (the smoother use, which reads b in place and assigns x).
"""
import numpy as np
import pytest
import torch

from helpers import rel_l2
from test_gpu_fullsize import FullSize, _cut

pytestmark = pytest.mark.gpu

BLOCK = (4, 4, 4, 4)
M = 4
B = 24                     # box extent: 6 blocks
LO, HI = 8, 16             # compared core: blocks 2..3 of the box


@pytest.fixture(scope="module")
def fs5():
    f = FullSize(5, 12)
    f.b_e2, f.b_o2 = f.ctx.pack(f.b_nat)
    yield f
    f.ctx.close()


def _origin(fs, name):
    L, T = fs.L, fs.T
    o = (20, 28, 40, 48) if name == "interior" else (L - 12, L - 12, L - 12, T - 12)
    assert all(v % 4 == 0 for v in o) and sum(v // 4 for v in o) % 2 == 0
    return o


def _box(fs, origin):
    """Oracle operator on the box and the cut full-lattice b, x (complex128 numpy)."""
    L, T, c = fs.L, fs.T, fs.c
    Ub = _cut(fs.U, origin, B, L, T).cpu().to(torch.complex128).numpy()
    if c["bc"] == 1:
        tg = (np.arange(B) + origin[3]) % T
        Ub[tg == T - 1, :, :, :, 3] *= -1.0
    ora = fs.oracle.WilsonClover(B, B, c["csw"], c["m0"], 0, Ub)
    xb = _cut(fs.x_nat, origin, B, L, T).cpu().to(torch.complex128).numpy()
    bb = _cut(fs.b_nat, origin, B, L, T).cpu().to(torch.complex128).numpy()
    return ora, bb, xb


def _core(a):
    return a[LO:HI, LO:HI, LO:HI, LO:HI]


@pytest.mark.parametrize("name", ["interior", "wrap corner + antiperiodic seam"])
def test_sap_full_size_sampled(fs5, name):
    fs = fs5
    origin = _origin(fs, name)
    ora, bb, xb = _box(fs, origin)
    # ---- non-zero initial guess, with history (one full residual, then the incremental one)
    x_e, x_o = fs.ctx.pack(fs.x_nat)
    hist = fs.ctx.sap(fs.b_e2, fs.b_o2, x_e, x_o, 1, M, BLOCK, zero_init=False, history=True)
    got = _cut(fs.ctx.unpack(x_e, x_o), origin, B, fs.L, fs.T).cpu().to(torch.complex128).numpy()
    ref, _ = fs.oracle.sap(ora, bb, xb, 1, M, BLOCK)
    assert np.linalg.norm(_core(ref) - _core(xb)) > 1e-2 * np.linalg.norm(_core(xb))      # the update is not small
    assert rel_l2(_core(got), _core(ref)) <= 2e-5, name
    assert rel_l2(got, ref) > 1e-3                         # the box surface differs: the cut is live
    # history at full size: ||b - D x0|| and ||b - D x1|| against separate fp64 reductions of the full operator
    for h, (xe, xo) in zip(hist, (fs.ctx.pack(fs.x_nat), (x_e, x_o))):
        y_e, y_o = fs.ctx.apply_full(xe, xo)
        r = torch.sqrt(torch.linalg.vector_norm((fs.b_e2 - y_e).double()) ** 2 +
                       torch.linalg.vector_norm((fs.b_o2 - y_o).double()) ** 2).item()
        assert abs(h - r) <= 1e-4 * r, (hist, r)
    assert hist[1] < 0.7 * hist[0]
    # ---- zero initial guess, no history: the smoother use (b read in place, x assigned; garbage in x is ignored)
    z_e, z_o = fs.ctx.half_spinor(), fs.ctx.half_spinor()
    z_e.fill_(3.0); z_o.fill_(-5.0)
    fs.ctx.sap(fs.b_e2, fs.b_o2, z_e, z_o, 1, M, BLOCK, zero_init=True)
    got0 = _cut(fs.ctx.unpack(z_e, z_o), origin, B, fs.L, fs.T).cpu().to(torch.complex128).numpy()
    ref0, _ = fs.oracle.sap(ora, bb, np.zeros_like(bb), 1, M, BLOCK)
    assert rel_l2(_core(got0), _core(ref0)) <= 2e-5, name

"""Multi-rhs batching (NEXT-2) at FULL size -- config 5, 64^3 x 128, fp32, two-row links: the
launch configuration of bench.py's multi-rhs rows, in which (unlike on the small lattices of test_gpu_batch.py) the
z-chunked CTA traversal is really in effect (one time slice of nrhs spinors no longer fits the L2 budget).

The single-rhs kernels are compared with the oracle at this size in test_gpu_fullsize.py; the batched kernels
perform per right-hand side the same operations in the same order, so each rhs of a batched Richardson call must
be BIT-IDENTICAL to the single-rhs call on that rhs -- for an odd nrhs (a padded last pair) as well, histories
included to the last bit but the order of the block sums."""
import pytest
import torch

import gen
from test_gpu_fullsize import FullSize

pytestmark = pytest.mark.gpu

NU = 2


@pytest.fixture(scope="module")
def fs5():
    f = FullSize(5, 12)
    yield f
    f.ctx.close()


@pytest.mark.parametrize("nrhs", [3, 8])
def test_batched_richardson_full_size_bit_identical_per_rhs(fs5, nrhs):
    fs, ctx = fs5, fs5.ctx
    omega = fs.c["omega"]
    bs, xs = [], []
    for r in range(nrhs):
        b, _ = ctx.pack(gen.spinor_field(fs.L, fs.T, 5100 + r, device="cuda", dtype=torch.complex64), want_odd=False)
        x, _ = ctx.pack(gen.spinor_field(fs.L, fs.T, 5200 + r, device="cuda", dtype=torch.complex64), want_odd=False)
        bs.append(b); xs.append(x)
    Bb, Xb = ctx.batch_interleave(bs), ctx.batch_interleave(xs)
    hist_b = ctx.richardson_batch(nrhs, Bb, Xb, NU, omega, history=True)
    out = ctx.batch_deinterleave(nrhs, Xb)
    del Bb, Xb
    for r in range(nrhs):
        x = xs[r].clone()
        hist = ctx.richardson(bs[r], x, NU, omega, history=True)
        torch.cuda.synchronize()
        assert torch.equal(out[r], x.view(-1)), r
        for i in range(NU):
            assert abs(hist_b[i][r] - hist[i]) <= 1e-12 * hist[i], (r, i)

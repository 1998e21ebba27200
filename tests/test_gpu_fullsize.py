"""Full-size parity (BASELINE.json configs[4]: 64^3 x 128, fp32) in the launch configuration
bench.py times, on sampled outputs the oracle can compute one by one; the same at the other
full-size shapes of BASELINE.json (configs[2]: 32^3 x 64, configs[3]: 48^3 x 96).

The oracle cannot run on 33.5 M sites in seconds, but one Schur apply depends only on spinors
within 2 sites and links within 3 sites of the output site, and nu Richardson sweeps on 2 nu
(+1 for the clover leaves).  So the oracle is run on a small box cut out of the GPU's own
input buffers (global wrap-around, the antiperiodic sign applied to the cut links by hand)
as if the box were periodic; its result is exact on the core of the box that lies at least
that far from the box surface, and that core is compared element by element.
Box 0 is interior; box 1 contains the (x,y,z,t) wrap corner, i.e. the periodic seams of all
four axes and the antiperiodic time boundary.

Properties that hold at any size are checked on the whole lattice: gamma5-hermiticity of D_S
and the fused residual-norm reduction against a separate fp64 reduction of b - D_S x.
"""
import numpy as np
import pytest
import torch

import gen
from helpers import CONFIGS, rel_l2

pytestmark = pytest.mark.gpu

NU = 4


def _cut(field: torch.Tensor, origin, B, L, T) -> torch.Tensor:
    """field[(ot+i)%T, (oz+j)%L, (oy+k)%L, (ox+l)%L, ...] for i,j,k,l in range(B) (device gather)."""
    ox, oy, oz, ot = origin
    dev = field.device
    it = (torch.arange(B, device=dev) + ot) % T
    iz = (torch.arange(B, device=dev) + oz) % L
    iy = (torch.arange(B, device=dev) + oy) % L
    ix = (torch.arange(B, device=dev) + ox) % L
    return field.index_select(0, it).index_select(1, iz).index_select(2, iy).index_select(3, ix).contiguous()


class FullSize:
    def __init__(self, cfg=5, recon=18):
        import oracle
        import paper_2407_08092_b200 as dd
        self.oracle, self.dd = oracle, dd
        c = CONFIGS[cfg]
        self.c = c
        self.L, self.T = c["L"], c["T"]
        dev = "cuda"
        self.U = gen.gauge_field(self.L, self.T, 1000 + cfg, c["eps"], c["reunit"], device=dev,
                                 dtype=torch.complex64)
        self.ctx = dd.Ddamg(self.L, self.T, c["csw"], c["m0"], c["bc"], dd.F32)
        self.ctx.load_gauge(self.U)
        self.ctx.build_clover()
        if recon == 12:                        # bench.py --gauge-recon 12: two-row links in the hopping kernels
            self.ctx.set_option("gauge_recon", 12)
        self.x_nat = gen.spinor_field(self.L, self.T, 3000 + cfg, device=dev, dtype=torch.complex64)
        self.b_nat = gen.spinor_field(self.L, self.T, 2000 + cfg, device=dev, dtype=torch.complex64)
        self.x_e, _ = self.ctx.pack(self.x_nat, want_odd=False)
        self.b_e, _ = self.ctx.pack(self.b_nat, want_odd=False)

    def box_oracle(self, origin, B):
        """Oracle operator on the box + the cut (even-masked) x and b, all complex128 numpy."""
        assert sum(origin) % 2 == 0, "box origin must be an even site so that parities agree"
        L, T, c = self.L, self.T, self.c
        Ub = _cut(self.U, origin, B, L, T).cpu().to(torch.complex128).numpy()
        if c["bc"] == 1:                       # reading R2: -1 on U_t of the global slice t = T-1
            tg = (np.arange(B) + origin[3]) % T
            Ub[tg == T - 1, :, :, :, 3] *= -1.0
        ora = self.oracle.WilsonClover(B, B, c["csw"], c["m0"], 0, Ub)
        xb = _cut(self.x_nat, origin, B, L, T).cpu().to(torch.complex128).numpy()
        bb = _cut(self.b_nat, origin, B, L, T).cpu().to(torch.complex128).numpy()
        return ora, np.where(ora.even, xb, 0.0), np.where(ora.even, bb, 0.0)


# config 5 = the bench workload (both link formats); configs 3 and 4 = the other full-size shapes
# of BASELINE.json (32^3 x 64, 48^3 x 96) in the bench's default link format
@pytest.fixture(scope="module", params=[(5, 18), (5, 12), (3, 12), (4, 12)],
                ids=["cfg5-links18", "cfg5-links12", "cfg3-links12", "cfg4-links12"])
def fs(request):
    f = FullSize(*request.param)
    yield f
    f.ctx.close()


def _core(a, m):
    return a[m:-m, m:-m, m:-m, m:-m]


def _origin(fs, name):
    """Even-parity box origins: one interior, one whose box crosses the periodic seam of all four
    axes and the antiperiodic time boundary (for config 5: (20,30,40,50) and (58,60,56,122))."""
    L, T = fs.L, fs.T
    if name == "interior":
        return (5 * L // 16, 15 * L // 32, 5 * L // 8, 25 * T // 64)
    return (L - 6, L - 4, L - 8, T - 6)


BOXES = ["interior", "wrap corner + antiperiodic seam"]


@pytest.mark.parametrize("name", BOXES)
def test_schur_apply_full_size_sampled(fs, name):
    origin = _origin(fs, name)
    B, m = 12, 4                                        # dependence radius 3 < margin 4; core 4^4
    y = fs.ctx.apply_schur(fs.x_e)
    y_nat = fs.ctx.unpack(y, None)
    got = _cut(y_nat, origin, B, fs.L, fs.T).cpu().to(torch.complex128).numpy()
    ora, xb, _ = fs.box_oracle(origin, B)
    ref = ora.apply_schur(xb)
    assert np.linalg.norm(_core(ref, m)) > 0
    assert rel_l2(_core(got, m), _core(ref, m)) <= 5e-6, name
    # the box surface, where the oracle's wrap-around is wrong, must indeed differ (the cut is live)
    assert rel_l2(got, ref) > 1e-3


@pytest.mark.parametrize("name", BOXES)
def test_richardson_full_size_sampled(fs, name):
    origin = _origin(fs, name)
    omega = fs.c["omega"]
    m = 2 * NU + 2                                      # dependence radius 2 nu + 1
    B = 4 + 2 * m
    x = fs.x_e.clone()
    hist = fs.ctx.richardson(fs.b_e, x, NU, omega, history=True)
    x2 = fs.x_e.clone()
    fs.ctx.richardson(fs.b_e, x2, NU, omega)            # bench.py's launch configuration (no history)
    torch.cuda.synchronize()
    assert torch.equal(x, x2)
    x_nat = fs.ctx.unpack(x, None)
    got = _cut(x_nat, origin, B, fs.L, fs.T).cpu().to(torch.complex128).numpy()
    ora, xb, bb = fs.box_oracle(origin, B)
    ref, _ = fs.oracle.richardson(ora.apply_schur, bb, xb, NU, omega)
    assert rel_l2(_core(got, m), _core(ref, m)) <= 2e-5, name
    # fused norm reduction at full size: hist[0] = || b - D_S x0 ||, reduced separately in fp64
    y = fs.ctx.apply_schur(fs.x_e)
    r0 = torch.linalg.vector_norm((fs.b_e - y).double()).item()
    assert abs(hist[0] - r0) <= 1e-6 * r0
    assert all(np.isfinite(hist)) and len(hist) == NU


def test_gamma5_hermiticity_full_size(fs):
    """<y, g5 D_S x> = <g5 D_S y, x> on the whole 64^3 x 128 lattice (holds at any size)."""
    ctx = fs.ctx
    g5 = torch.ones(4, 3, dtype=torch.complex64, device="cuda")
    g5[2:] = -1.0

    def g5mul(v_e):
        nat = ctx.unpack(v_e, None)
        out, _ = ctx.pack(nat * g5, want_odd=False)
        return out

    def dot(a, b):                                      # complex inner product of native halves
        a = torch.view_as_complex(a.view(-1, 2).contiguous()).to(torch.complex128)
        b = torch.view_as_complex(b.view(-1, 2).contiguous()).to(torch.complex128)
        return torch.vdot(a, b).item()

    x, yv = fs.x_e, fs.b_e
    lhs = dot(yv, g5mul(ctx.apply_schur(x)))
    rhs = dot(g5mul(ctx.apply_schur(yv)), x)
    scale = torch.linalg.vector_norm(x.double()).item() * torch.linalg.vector_norm(yv.double()).item()
    assert abs(lhs - rhs) <= 1e-7 * scale

"""GPU parity: libddamg.so (through the C ABI) vs the CPU fp64 oracle, element by element.

Tolerances are BASELINE.json's (north_star): fp64 apply <= 1e-12, fp32 apply <= 5e-6 relative
L2; fp32 Richardson / GMRES residual history <= 1e-4 per entry (plus the fp32 floor term
32 * eps32 * ||b|| of DESIGN.md for converged GMRES residuals).  The oracle always consumes
the same rounded inputs as the GPU (fp32 fields promoted to fp64).
"""
import numpy as np
import pytest
import torch

import gen
from helpers import CONFIGS, rel_l2

pytestmark = pytest.mark.gpu

EPS32 = float(np.finfo(np.float32).eps)


def _mods():
    import oracle
    import paper_2407_08092_b200 as dd
    return oracle, dd


class Pair:
    """An oracle operator and a GPU context built from the same rounded inputs."""

    def __init__(self, L, T, csw, m0, bc, prec_name, gauge_seed, eps, reunit, unit=False):
        oracle, dd = _mods()
        self.dd = dd
        self.L, self.T = L, T
        self.f64 = prec_name == "f64"
        self.cdt = torch.complex128 if self.f64 else torch.complex64
        if unit:
            U = gen.unit_gauge_field(L, T)
        else:
            U = gen.gauge_field(L, T, gauge_seed, eps, reunit)
        U = U.to(self.cdt)
        self.ora = oracle.WilsonClover(L, T, csw, m0, bc, U.to(torch.complex128).numpy())
        self.ctx = dd.Ddamg(L, T, csw, m0, bc, dd.F64 if self.f64 else dd.F32)
        self.ctx.load_gauge(U.cuda())
        self.ctx.build_clover()
        self.apply_tol = 1e-12 if self.f64 else 5e-6

    def spinor(self, seed):
        """(numpy complex128 full-lattice array, device tensor) of the same rounded values."""
        s = gen.spinor_field(self.L, self.T, seed).to(self.cdt)
        return s.to(torch.complex128).numpy(), s.cuda()

    def to_np(self, x_e=None, x_o=None):
        return self.ctx.unpack(x_e, x_o).cpu().to(torch.complex128).numpy()

    def even(self, a):
        return np.where(self.ora.even, a, 0.0)

    def odd(self, a):
        return np.where(self.ora.odd, a, 0.0)


def make_pair(cfg, prec, L=None, T=None, bc=None):
    c = CONFIGS[cfg]
    return Pair(L or c["L"], T or c["T"], c["csw"], c["m0"], c["bc"] if bc is None else bc, prec,
                1000 + cfg, c["eps"], c["reunit"])


# ------------------------------------------------------------------------- layout

@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("L,T", [(2, 2), (4, 4), (6, 4), (8, 10)])
def test_pack_unpack_roundtrip_bit_exact(prec, L, T):
    _, dd = _mods()
    ctx = dd.Ddamg(L, T, 1.0, 0.0, 1, dd.F64 if prec == "f64" else dd.F32)
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    nat = gen.spinor_field(L, T, 5).to(cdt).cuda()
    xe, xo = ctx.pack(nat)
    assert torch.equal(ctx.unpack(xe, xo), nat)
    par = gen.site_parity(L, T, "cuda")[..., None, None]
    assert torch.equal(ctx.unpack(xe, None), torch.where(par == 0, nat, torch.zeros_like(nat)))
    assert torch.equal(ctx.unpack(None, xo), torch.where(par == 1, nat, torch.zeros_like(nat)))


# ------------------------------------------------------------------------- clover (a1)

@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("cfg,L,T", [(1, 4, 4), (3, 6, 4), (1, 2, 2)])
def test_clover_blocks_match_oracle(prec, cfg, L, T):
    p = make_pair(cfg, prec, L, T)
    A, Ai = p.ctx.get_clover()
    A = A.cpu().to(torch.complex128).numpy()
    Ai = Ai.cpu().to(torch.complex128).numpy()
    ev, od = p.ora.par == 0, p.ora.par == 1
    tol = 1e-13 if p.f64 else 2e-7
    for blk, sl in ((0, slice(0, 6)), (1, slice(6, 12))):
        ref_A = p.ora.A[..., sl, sl]
        ref_Ai = p.ora.Ainv[..., sl, sl]
        assert np.abs(A[ev][:, blk] - ref_A[ev]).max() <= tol * np.abs(ref_A).max()
        assert np.abs(Ai[od][:, blk] - ref_Ai[od]).max() <= 4 * tol * np.abs(ref_Ai).max()
        assert np.all(A[od][:, blk] == 0) and np.all(Ai[ev][:, blk] == 0)


def test_clover_constant_flux_closed_form_on_gpu():
    """Same closed form that pins the oracle (tests/test_oracle_operator.py), straight on the GPU."""
    _, dd = _mods()
    L, T, csw, m0, nflux = 4, 4, 1.3, -0.15, 3
    phi = 2 * np.pi * nflux / L ** 2
    T3 = np.array([1.0, -1.0, 0.0])
    U = gen.unit_gauge_field(L, T).numpy()
    for y in range(L):
        U[:, :, y, :, 0] = np.diag(np.exp(-1j * phi * y * T3))
    for x in range(L):
        U[:, :, L - 1, x, 1] = np.diag(np.exp(1j * phi * L * x * T3))
    ctx = dd.Ddamg(L, T, csw, m0, 1, dd.F64)
    ctx.load_gauge(torch.from_numpy(U).cuda())
    ctx.build_clover()
    A, Ai = ctx.get_clover()
    blk = (m0 + 4.0) * np.eye(6) + 0.5 * csw * np.sin(phi) * np.kron(np.diag([1.0, -1.0]), np.diag(T3))
    par = gen.site_parity(L, T).numpy()
    A = A.cpu().numpy()
    Ai = Ai.cpu().numpy()
    assert np.abs(A[par == 0] - blk).max() < 1e-13
    assert np.abs(Ai[par == 1] - np.linalg.inv(blk)).max() < 1e-13


def test_singular_clover_block_is_reported():
    _, dd = _mods()
    ctx = dd.Ddamg(4, 4, 0.0, -4.0, 0, dd.F64)          # A = (m0 + 4) 1 = 0
    ctx.load_gauge(gen.unit_gauge_field(4, 4).cuda())
    with pytest.raises(dd.DdamgError) as e:
        ctx.build_clover()
    assert e.value.status == dd.ESINGULAR


# ------------------------------------------------------------------------- apply (a2-a6, a10)

CASES = [
    # cfg, prec, L, T, bc
    (1, "f64", None, None, None),     # config 1: 4^4 fp64
    (1, "f32", None, None, None),
    (1, "f64", 2, 2, None),           # smallest lattice: both hops of an extent-2 axis add
    (1, "f64", 4, 6, 0),              # periodic time, T != L
    (3, "f32", 6, 8, None),           # L not a power of two, V/2 = 864: ragged last CTA
    (3, "f64", 6, 8, None),
    (2, "f32", None, None, None),     # config 2: 16^4
    (2, "f64", None, None, None),
]


@pytest.mark.parametrize("cfg,prec,L,T,bc", CASES)
def test_schur_apply_prepare_reconstruct(cfg, prec, L, T, bc):
    p = make_pair(cfg, prec, L, T, bc)
    x_np, x_d = p.spinor(2000 + cfg)
    b_np, b_d = p.spinor(2100 + cfg)
    x_e, x_o = p.ctx.pack(x_d)
    b_e, b_o = p.ctx.pack(b_d)
    # eq. 3
    y = p.to_np(p.ctx.apply_schur(x_e), None)
    y_ref = p.ora.apply_schur(p.even(x_np))
    assert np.all(y[p.ora.par == 1] == 0)
    assert rel_l2(y, y_ref) <= p.apply_tol
    # eq. 2 right factor
    bh = p.to_np(p.ctx.prepare_rhs(b_e, b_o), None)
    assert rel_l2(bh, p.ora.prepare_rhs(b_np)) <= p.apply_tol
    # eq. 2 left factor
    xo = p.to_np(None, p.ctx.reconstruct_odd(b_o, x_e))
    assert np.all(xo[p.ora.par == 0] == 0)
    assert rel_l2(xo, p.ora.reconstruct_odd(b_np, p.even(x_np))) <= p.apply_tol


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("bc", [0, 1])
def test_free_field_plane_wave_closed_form_on_gpu(prec, bc):
    """D_S psi_e = (a - s^2/a) psi_e for a free plane wave (closed form, no oracle involved)."""
    oracle, dd = _mods()
    L, T, m0 = 8, 12, -0.1
    p = Pair(L, T, 1.7, m0, bc, prec, 0, 0.0, False, unit=True)
    g = oracle.gamma_matrices()
    n = (1, 3, 2, 5)
    mom = np.array([2 * np.pi * n[0] / L, 2 * np.pi * n[1] / L, 2 * np.pi * n[2] / L,
                    (2 * n[3] + 1) * np.pi / T if bc == 1 else 2 * np.pi * n[3] / T])
    K = sum(np.sin(mom[mu]) * g[mu] for mu in range(4))
    evals, evecs = np.linalg.eigh(K)
    u = evecs[:, 3]
    w = np.kron(u, np.array([0.3 - 0.2j, 1.0, -0.7j]))
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    psi = np.exp(1j * (mom[0] * x + mom[1] * y + mom[2] * z + mom[3] * t))[..., None, None] * w.reshape(4, 3)
    psi_d = torch.from_numpy(psi).to(p.cdt).cuda()
    x_e, _ = p.ctx.pack(psi_d)
    got = p.to_np(p.ctx.apply_schur(x_e), None)
    a = m0 + 4.0
    s = -np.sum(np.cos(mom)) + 1j * np.sqrt(np.sum(np.sin(mom) ** 2))
    expect = (a - s * s / a) * p.even(psi_d.cpu().to(torch.complex128).numpy())
    assert rel_l2(got, expect) <= (1e-12 if p.f64 else 5e-6)


# ------------------------------------------------------------------------- Richardson (a7)

@pytest.mark.parametrize("cfg,prec,nu,L,T", [
    (1, "f64", 4, None, None),        # config 1: 4 sweeps, omega = 1.0
    (1, "f32", 4, None, None),
    (2, "f32", 8, None, None),        # config 2: 8 sweeps, omega = 1.0
    (2, "f64", 8, None, None),
    (3, "f32", 4, 8, 8),              # config 3 recipe (omega = 0.9, nu = 4) on a small lattice
])
def test_richardson_matches_oracle(cfg, prec, nu, L, T):
    oracle, _ = _mods()
    p = make_pair(cfg, prec, L, T)
    omega = CONFIGS[cfg]["omega"]
    b_np, b_d = p.spinor(2000 + cfg)
    x_np, x_d = p.spinor(2050 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    bhat = p.ctx.prepare_rhs(b_e, b_o)
    bhat_np = p.to_np(bhat, None)                       # same rounded rhs for both sides
    x_e, _ = p.ctx.pack(x_d)
    hist = p.ctx.richardson(bhat, x_e, nu, omega, zero_init=False, history=True)
    x_ref, h_ref = oracle.richardson(p.ora.apply_schur, bhat_np, p.even(x_np), nu, omega)
    assert len(hist) == nu
    tol_h = 1e-11 if p.f64 else 1e-4
    for a, r in zip(hist, h_ref):
        assert abs(a - r) <= tol_h * r
    assert rel_l2(p.to_np(x_e, None), x_ref) <= (1e-11 if p.f64 else 2e-5)
    # same call without history (no reductions, asynchronous) gives the same iterate bit for bit
    x_e2, _ = p.ctx.pack(x_d)
    assert p.ctx.richardson(bhat, x_e2, nu, omega) is None
    torch.cuda.synchronize()
    assert torch.equal(x_e2, x_e)
    # zero initial guess (reading R12): first sweep is x = omega * b
    x_e3 = p.ctx.half_spinor()
    x_e3.fill_(float("nan"))
    h0 = p.ctx.richardson(bhat, x_e3, nu, omega, zero_init=True, history=True)
    x0_ref, h0_ref = oracle.richardson(p.ora.apply_schur, bhat_np, np.zeros_like(bhat_np), nu, omega)
    for a, r in zip(h0, h0_ref):
        assert abs(a - r) <= tol_h * r
    assert rel_l2(p.to_np(x_e3, None), x0_ref) <= (1e-11 if p.f64 else 2e-5)


def test_richardson_cuda_graph_replay_is_bit_identical():
    """Option cuda_graph: the history-free call replays its 2 nu launches through a captured CUDA graph
    (SURVEY.md 3.4); same kernels, same order -> same bits, also after the arguments change (re-capture)."""
    p = make_pair(2, "f32", 8, 8)
    _, b_d = p.spinor(11)
    _, c_d = p.spinor(12)
    _, x_d = p.spinor(13)
    b_e, _ = p.ctx.pack(b_d)
    c_e, _ = p.ctx.pack(c_d)
    outs = {}
    for mode in (0, 1):
        p.ctx.set_option("cuda_graph", mode)
        res = []
        for rhs, nu, omega, zi in ((b_e, 4, 0.3, False), (b_e, 4, 0.3, False), (c_e, 4, 0.3, False), (c_e, 3, 0.25, True),
                                   (b_e, 4, 0.3, False)):
            x_e, _ = p.ctx.pack(x_d)
            l0 = p.ctx.launch_count()
            p.ctx.richardson(rhs, x_e, nu, omega, zero_init=zi)
            torch.cuda.synchronize()
            res.append((x_e.clone(), p.ctx.launch_count() - l0))
        outs[mode] = res
    for (xa, la), (xb, lb) in zip(outs[0], outs[1]):
        assert torch.equal(xa, xb)
        assert la == lb                                   # the launch accounting counts the kernels inside the graph
    p.ctx.set_option("cuda_graph", 1)
    p.ctx.set_option("gauge_recon", 12)                   # link format is part of the capture key
    x12, _ = p.ctx.pack(x_d)
    p.ctx.richardson(b_e, x12, 4, 0.3)
    p.ctx.set_option("cuda_graph", 0)
    y12, _ = p.ctx.pack(x_d)
    p.ctx.richardson(b_e, y12, 4, 0.3)
    torch.cuda.synchronize()
    assert torch.equal(x12, y12)
    with pytest.raises(p.dd.DdamgError):
        p.ctx.set_option("cuda_graph", 2)


def test_richardson_nu_zero_is_identity():
    p = make_pair(1, "f64")
    _, b_d = p.spinor(1)
    _, x_d = p.spinor(2)
    b_e, _ = p.ctx.pack(b_d)
    x_e, _ = p.ctx.pack(x_d)
    keep = x_e.clone()
    assert p.ctx.richardson(b_e, x_e, 0, 1.0, history=True) == []
    assert torch.equal(x_e, keep)


# ------------------------------------------------------------------------- GMRES (a8, a9)

def _check_history(got, ref, bnorm, f64):
    assert len(got) == len(ref)
    for a, r in zip(got, ref):
        if f64:
            assert abs(a - r) <= 1e-9 * r + 1e-13 * bnorm
        else:
            assert abs(a - r) <= 1e-4 * r + 32 * EPS32 * bnorm


@pytest.mark.parametrize("cfg,prec,k,cycles,L,T", [
    (1, "f64", 5, 2, None, None),
    (1, "f32", 5, 2, None, None),
    (4, "f32", 10, 2, 8, 8),          # config 4 recipe GMRES(2,10) on a small lattice
    (4, "f64", 10, 2, 8, 8),
    (4, "f32", 10, 2, 16, 32),        # config 4 recipe GMRES(2,10), T = 2L shape, 65,536 even sites (512 CTAs)
    (2, "f32", 14, 1, None, None),    # k > 12: more than one fused multi-dot chunk, second Gram-Schmidt pass (CGS2)
    (3, "f32", 40, 1, 8, 8),          # a long fp32 cycle: four chunks, CGS2 keeps the Givens estimates on the oracle's
])
def test_gmres_matches_oracle(cfg, prec, k, cycles, L, T):
    oracle, _ = _mods()
    p = make_pair(cfg, prec, L, T)
    b_np, b_d = p.spinor(2000 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    bhat = p.ctx.prepare_rhs(b_e, b_o)
    bhat_np = p.to_np(bhat, None)
    x_e = p.ctx.half_spinor()
    hist = p.ctx.gmres_oe(bhat, x_e, k, cycles, zero_init=True)
    x_ref, h_ref = oracle.gmres(p.ora.apply_schur, bhat_np, np.zeros_like(bhat_np), k, cycles)
    assert len(hist) == cycles * (k + 1) + 1
    _check_history(hist, h_ref, np.linalg.norm(bhat_np), p.f64)
    assert rel_l2(p.to_np(x_e, None), x_ref) <= (1e-9 if p.f64 else 5e-5)
    # non-zero initial guess
    x_np, x_d = p.spinor(2070 + cfg)
    x_e2, _ = p.ctx.pack(x_d)
    hist2 = p.ctx.gmres_oe(bhat, x_e2, k, 1, zero_init=False)
    x_ref2, h_ref2 = oracle.gmres(p.ora.apply_schur, bhat_np, p.even(x_np), k, 1)
    _check_history(hist2, h_ref2, np.linalg.norm(bhat_np), p.f64)
    assert rel_l2(p.to_np(x_e2, None), x_ref2) <= (1e-9 if p.f64 else 5e-5)


def test_gmres_tolerance_exit_and_full_smoother_call():
    """eq. 2 end to end: prepare_rhs -> GMRES to 1e-10 -> reconstruct_odd solves D x = b."""
    oracle, _ = _mods()
    p = make_pair(1, "f64")
    b_np, b_d = p.spinor(2001)
    b_e, b_o = p.ctx.pack(b_d)
    bhat = p.ctx.prepare_rhs(b_e, b_o)
    x_e = p.ctx.half_spinor()
    hist = p.ctx.gmres_oe(bhat, x_e, 10, 20, tol=1e-10, zero_init=True)
    assert len(hist) < 20 * 11 + 1
    x_o = p.ctx.reconstruct_odd(b_o, x_e)
    x = p.to_np(x_e, x_o)
    assert rel_l2(p.ora.apply_D(x), b_np) < 1e-9


def test_power_iteration_matches_oracle():
    oracle, _ = _mods()
    p = make_pair(1, "f64")
    v_np, v_d = p.spinor(2009)
    v_e, _ = p.ctx.pack(v_d)
    lam = p.ctx.power_iteration(v_e, 10)
    ref = oracle.power_iteration(p.ora.apply_schur, p.even(v_np), 10)
    assert abs(lam - ref) < 1e-10 * ref


# ------------------------------------------------------------------------- error behaviour

def test_error_codes():
    _, dd = _mods()
    for bad in [(3, 4), (4, 5), (0, 4)]:
        with pytest.raises(dd.DdamgError) as e:
            dd.Ddamg(bad[0], bad[1], 1.0, 0.0)
        assert e.value.status == dd.EINVAL
    ctx = dd.Ddamg(4, 4, 1.0, -0.1, 1, dd.F32)
    x = ctx.half_spinor(zero=True)
    y = ctx.half_spinor()
    with pytest.raises(dd.DdamgError) as e:
        ctx.apply_schur(x, y)                               # no gauge yet
    assert e.value.status == dd.ESTATE
    with pytest.raises(dd.DdamgError) as e:
        ctx.build_clover()
    assert e.value.status == dd.ESTATE
    ctx.load_gauge(gen.gauge_field(4, 4, 1, 0.3).to(torch.complex64))      # host tensor path
    with pytest.raises(dd.DdamgError) as e:
        ctx.apply_schur(x, y)                               # clover not built
    assert e.value.status == dd.ESTATE
    ctx.build_clover()
    ctx.apply_schur(x, y)
    torch.cuda.synchronize()
    assert torch.all(y == 0)                                # D_S 0 = 0
    with pytest.raises(dd.DdamgError) as e:
        ctx.apply_schur(x, x)                               # aliasing
    assert e.value.status == dd.EINVAL
    with pytest.raises(dd.DdamgError) as e:
        ctx.richardson(x, y, -1, 1.0)
    assert e.value.status == dd.EINVAL
    with pytest.raises(dd.DdamgError) as e:
        ctx.gmres_oe(x, y, 0, 1)
    assert e.value.status == dd.EINVAL
    # the layout converters move 16-byte vectors: a natural buffer that is only 8-byte aligned is refused
    buf = torch.zeros(12 * 256 + 1, dtype=torch.complex64, device="cuda")
    with pytest.raises(dd.DdamgError) as e:
        ctx.pack(buf[1:])
    assert e.value.status == dd.EINVAL


def test_host_and_device_gauge_paths_agree():
    _, dd = _mods()
    U = gen.gauge_field(4, 4, 9, 0.3)
    outs = []
    for src in (U, U.cuda()):
        ctx = dd.Ddamg(4, 4, 1.0, -0.1, 1, dd.F64)
        ctx.load_gauge(src)
        ctx.build_clover()
        x_e, _ = ctx.pack(gen.spinor_field(4, 4, 3).cuda())
        outs.append(ctx.apply_schur(x_e).clone())
    assert torch.equal(outs[0], outs[1])

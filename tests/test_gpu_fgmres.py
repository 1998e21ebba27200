"""GPU parity of the full operator D and the outer FGMRES preconditioned by one odd-even
smoother call (eq. 1-2) vs the oracle."""
import numpy as np
import pytest
import torch

from helpers import CONFIGS, rel_l2
from test_gpu_parity import make_pair, _mods, _check_history

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,prec,L,T,bc", [
    (1, "f64", 4, 4, None), (1, "f32", 4, 4, None), (1, "f64", 2, 2, None), (3, "f32", 6, 8, None),
    (1, "f64", 4, 6, 0), (2, "f32", 16, 16, None),
])
def test_apply_full_matches_oracle(cfg, prec, L, T, bc):
    p = make_pair(cfg, prec, L, T, bc)
    x_np, x_d = p.spinor(8000 + cfg)
    x_e, x_o = p.ctx.pack(x_d)
    y_e, y_o = p.ctx.apply_full(x_e, x_o)
    assert rel_l2(p.to_np(y_e, y_o), p.ora.apply_D(x_np)) <= p.apply_tol
    # A_oo (built lazily) times the stored A_oo^-1 is the identity:  A_oo^-1 (D x)_o with x_e = 0 gives x_o
    z = torch.zeros_like(x_e)
    _, w_o = p.ctx.apply_full(z, x_o)
    back = p.ctx.reconstruct_odd(w_o, z)             # A_oo^-1 (w_o - H_oe 0)
    assert rel_l2(back.cpu().numpy(), x_o.cpu().numpy()) <= (1e-12 if p.f64 else 2e-6)


def _oracle_smoother(oracle, ora, kind, s_n, s_m, omega):
    """z = M v: eq. 2 around the chosen oracle iteration, zero initial guess."""
    def M(v):
        bhat = ora.prepare_rhs(v)
        z0 = np.zeros_like(bhat)
        if kind == 0:
            ze, _ = oracle.richardson(ora.apply_schur, bhat, z0, s_n, omega)
        elif kind == 1:
            ze, _ = oracle.gmres(ora.apply_schur, bhat, z0, s_m, s_n)
        else:
            ze, _ = oracle.gcr(ora.apply_schur, bhat, z0, s_m, s_n)
        return ze + ora.reconstruct_odd(v, ze)
    return M


@pytest.mark.parametrize("cfg,prec,L,T,k,cycles,kind,s_n,s_m,omega", [
    (1, "f64", 4, 4, 5, 2, 0, 3, 1, 0.3),       # Richardson(3, paper-like omega)
    (1, "f32", 4, 4, 5, 2, 0, 3, 1, 0.3),
    (4, "f32", 8, 8, 6, 1, 1, 1, 4, 0.0),       # GMRES(1,4) smoother
    (4, "f64", 6, 8, 4, 2, 2, 1, 3, 0.0),       # GCR(1,3) smoother
    (3, "f32", 6, 8, 14, 1, 0, 2, 1, 0.25),     # k > 12: two orthogonalisation chunks
])
def test_fgmres_matches_oracle(cfg, prec, L, T, k, cycles, kind, s_n, s_m, omega):
    oracle, dd = _mods()
    p = make_pair(cfg, prec, L, T)
    b_np, b_d = p.spinor(8100 + cfg)
    b_e, b_o = p.ctx.pack(b_d)
    x_e, x_o = p.ctx.half_spinor(), p.ctx.half_spinor()
    hist = p.ctx.fgmres(b_e, b_o, x_e, x_o, k, cycles, 0.0, kind, s_n, s_m, omega, zero_init=True)
    M = _oracle_smoother(oracle, p.ora, kind, s_n, s_m, omega)
    x_ref, h_ref = oracle.fgmres(p.ora.apply_D, M, b_np, np.zeros_like(b_np), k, cycles)
    assert len(hist) == cycles * (k + 1) + 1
    _check_history(hist, h_ref, np.linalg.norm(b_np), p.f64)
    assert rel_l2(p.to_np(x_e, x_o), x_ref) <= (1e-8 if p.f64 else 1e-4)
    # the recorded final residual is the true one
    y_e, y_o = p.ctx.apply_full(x_e, x_o)
    res = np.linalg.norm(b_np - p.to_np(y_e, y_o))
    assert abs(res - hist[-1]) <= (1e-9 if p.f64 else 1e-3) * hist[0]


def test_fgmres_solves_D_x_equals_b_end_to_end():
    """Outer FGMRES + odd-even Richardson smoother (omega from the power iteration, Alg. 4
    line 1) drives D x = b to 1e-10 on config 1 -- the paper's solver minus the coarse grid."""
    oracle, dd = _mods()
    p = make_pair(1, "f64")
    b_np, b_d = p.spinor(8201)
    b_e, b_o = p.ctx.pack(b_d)
    v = p.ctx.pack(p.spinor(8202)[1])[0]
    omega = 1.5 / p.ctx.power_iteration(v, 12)
    x0_np, x0_d = p.spinor(8203)
    x_e, x_o = p.ctx.pack(x0_d)                       # non-zero initial guess
    hist = p.ctx.fgmres(b_e, b_o, x_e, x_o, 10, 20, 1e-10, dd.SMOOTHER_RICHARDSON, 3, 1, omega, zero_init=False)
    assert len(hist) < 20 * 11 + 1
    x = p.to_np(x_e, x_o)
    assert rel_l2(p.ora.apply_D(x), b_np) < 2e-10
    # fewer outer iterations than unpreconditioned-size Krylov: the smoother is doing work
    assert len(hist) < 60


def test_fgmres_error_codes():
    _, dd = _mods()
    p = make_pair(1, "f32")
    b_e, b_o, x_e, x_o = (p.ctx.half_spinor(zero=True) for _ in range(4))
    import ctypes
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    lib, h = p.ctx.lib, p.ctx._h
    call = lambda *a: lib.ddamg_fgmres(h, vp(b_e), vp(b_o), vp(x_e), vp(x_o), *a, None, None)
    assert call(0, 1, 0.0, 0, 1, 1, 1.0, 1) == dd.EINVAL
    assert call(2, 1, 0.0, 7, 1, 1, 1.0, 1) == dd.EINVAL
    assert call(2, 1, 0.0, 1, 1, 0, 1.0, 1) == dd.EINVAL
    assert call(2, 1, 0.0, 0, 2, 0, 0.3, 1) == dd.OK
    assert lib.ddamg_apply_full(h, vp(x_e), vp(x_o), vp(x_e), vp(b_o)) == dd.EINVAL

"""Pins for the CPU oracle's operator (oracle/wilson_clover.c) -- CPU only.

Each test checks the oracle against something the paper or the mathematics
fixes, never against a re-typed copy of the oracle's own formula:

* Clifford algebra / gamma5 of the basis (reading R1; needed for the 6x6 block
  claim of PAPER.md:173);
* free-field plane waves: closed-form eigenpairs of D and of D_S (BASELINE.json
  north_star);
* gamma5-hermiticity, gauge covariance;
* clover term: constant abelian flux closed form (fixes sign and the 1/32),
  an independent numpy (np.roll) field strength in the chiral block form,
  6x6 block structure, A * A^-1 = 1 to 1e-13;
* D_S == D_ee - D_eo D_oo^-1 D_oe assembled from dense blocks of D (eq. 3);
* Schur solve + odd reconstruction == dense LU of the full D on 2^4 (eq. 2);
* Fig. 1 qualitative statements on a 4^4 lattice.
"""
import numpy as np
import pytest

import gen
import oracle
from helpers import CONFIGS, config_gauge, config_spinor, rel_l2, even_part, odd_part

G5 = np.array([1, 1, -1, -1], dtype=np.float64)[:, None]       # gamma5 on (spin, colour)


def _np(t):
    return t.cpu().numpy()


def make(cfg=1, L=None, T=None, bc=None, csw=None, m0=None, U=None):
    c = CONFIGS[cfg]
    L = L or c["L"]
    T = T or c["T"]
    if U is None:
        U = _np(config_gauge(cfg, L, T))
    return oracle.WilsonClover(L, T, c["csw"] if csw is None else csw, c["m0"] if m0 is None else m0,
                               c["bc"] if bc is None else bc, U)


# ------------------------------------------------------------------ gamma basis

def test_gamma_clifford_algebra_and_gamma5():
    g = oracle.gamma_matrices()
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T, atol=0)                       # Hermitian
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu), atol=1e-15)
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    assert np.allclose(g5, np.diag([1, 1, -1, -1]), atol=1e-15)                # chiral: gamma5 diagonal
    # chiral basis: gamma_mu is block off-diagonal, so gamma_mu gamma_nu is block diagonal
    for mu in range(4):
        assert np.all(g[mu][:2, :2] == 0) and np.all(g[mu][2:, 2:] == 0)


# ------------------------------------------------------------------ free field

def _momenta(L, T, bc, n):
    p = np.array([2 * np.pi * n[0] / L, 2 * np.pi * n[1] / L, 2 * np.pi * n[2] / L,
                  (2 * n[3] + 1) * np.pi / T if bc == 1 else 2 * np.pi * n[3] / T])
    return p


def _plane_wave(L, T, p, w):
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return phase[..., None, None] * w.reshape(4, 3)


@pytest.mark.parametrize("bc", [0, 1])
def test_free_field_plane_wave_eigenpairs(bc):
    """D e^{ipx} u(x)c = (m0 + 4 - sum cos p_mu +- i sqrt(sum sin^2 p_mu)) e^{ipx} u(x)c."""
    L, T, m0 = 4, 6, -0.1
    op = oracle.WilsonClover(L, T, 1.7, m0, bc, _np(gen.unit_gauge_field(L, T)))
    g = oracle.gamma_matrices()
    rng = np.random.default_rng(7)
    for n in [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 2, 3, 4), (3, 1, 2, 5)]:
        p = _momenta(L, T, bc, n)
        K = sum(np.sin(p[mu]) * g[mu] for mu in range(4))           # Hermitian, K^2 = sum sin^2
        s2 = np.sum(np.sin(p) ** 2)
        evals, evecs = np.linalg.eigh(K)
        for sign, col in ((-1, 0), (+1, 3)):
            u = evecs[:, col]
            assert abs(evals[col] - sign * np.sqrt(s2)) < 1e-13
            c = rng.normal(size=3) + 1j * rng.normal(size=3)
            w = np.kron(u, c)
            psi = _plane_wave(L, T, p, w)
            lam = m0 + 4.0 - np.sum(np.cos(p)) + 1j * sign * np.sqrt(s2)
            assert rel_l2(op.apply_D(psi), lam * psi) < 1e-13
            # Schur complement on the even sublattice: (a - s^2/a) psi_e, s = lam - a
            a = m0 + 4.0
            s = lam - a
            psi_e = even_part(psi, op.par)
            assert rel_l2(op.apply_schur(psi_e), (a - s * s / a) * psi_e) < 1e-13


def test_free_field_full_spectrum():
    """Whole spectrum of the dense free D on 2^3 x 4 (extent-2 axes: both hops add)."""
    L, T, m0, bc = 2, 4, -0.1, 1
    op = oracle.WilsonClover(L, T, 1.0, m0, bc, _np(gen.unit_gauge_field(L, T)))
    ev = np.linalg.eigvals(op.dense(op.apply_D))
    expect = []
    for n0 in range(L):
        for n1 in range(L):
            for n2 in range(L):
                for n3 in range(T):
                    p = _momenta(L, T, bc, (n0, n1, n2, n3))
                    re = m0 + 4.0 - np.sum(np.cos(p))
                    im = np.sqrt(np.sum(np.sin(p) ** 2))
                    expect += [re + 1j * im] * 6 + [re - 1j * im] * 6
    expect = np.array(expect)
    # match as multisets
    used = np.zeros(len(ev), dtype=bool)
    for lam in expect:
        d = np.abs(ev - lam) + used * 1e9
        j = int(np.argmin(d))
        assert d[j] < 1e-9
        used[j] = True


def test_pure_gauge_field_reproduces_free_operator():
    """U_mu(x) = W(x) W(x+mu)^H is gauge-equivalent to the free field: D[U] = W D[1] W^H."""
    L, T = 4, 4
    W = _np(gen.random_su3_per_site(L, T, 11))
    U = np.empty((T, L, L, L, 4, 3, 3), dtype=np.complex128)
    for mu, ax in enumerate((3, 2, 1, 0)):
        Wf = np.roll(W, -1, axis=ax)
        U[..., mu, :, :] = W @ np.conj(np.swapaxes(Wf, -1, -2))
    op = oracle.WilsonClover(L, T, 1.3, -0.2, 0, U)
    free = oracle.WilsonClover(L, T, 1.3, -0.2, 0, _np(gen.unit_gauge_field(L, T)))
    psi = _np(config_spinor(1))
    lhs = op.apply_D(np.einsum("...ab,...sb->...sa", W, psi))
    rhs = np.einsum("...ab,...sb->...sa", W, free.apply_D(psi))
    assert rel_l2(lhs, rhs) < 1e-13


# ------------------------------------------------------- symmetries, random field

@pytest.mark.parametrize("bc", [0, 1])
def test_gamma5_hermiticity(bc):
    op = make(1, bc=bc)
    x = _np(config_spinor(1, 0))
    y = _np(config_spinor(1, 1))
    lhs = np.vdot(y, G5 * op.apply_D(x))
    rhs = np.vdot(G5 * op.apply_D(y), x)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    xe, ye = even_part(x, op.par), even_part(y, op.par)
    lhs = np.vdot(ye, G5 * op.apply_schur(xe))
    rhs = np.vdot(G5 * op.apply_schur(ye), xe)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)


def _gauge_transform(U, Om):
    """U^Om_mu(x) = Om(x) U_mu(x) Om(x+mu)^H."""
    out = np.empty_like(U)
    for mu, ax in enumerate((3, 2, 1, 0)):
        Of = np.roll(Om, -1, axis=ax)
        out[..., mu, :, :] = Om @ U[..., mu, :, :] @ np.conj(np.swapaxes(Of, -1, -2))
    return out


def test_gauge_covariance():
    L, T = 4, 6
    U = _np(config_gauge(1, L, T))
    Om = _np(gen.random_su3_per_site(L, T, 5))
    op = make(1, L, T, U=U)
    opg = make(1, L, T, U=_gauge_transform(U, Om))
    psi = _np(gen.spinor_field(L, T, 77))
    rot = lambda v: np.einsum("...ab,...sb->...sa", Om, v)
    assert rel_l2(opg.apply_D(rot(psi)), rot(op.apply_D(psi))) < 1e-13
    pe = even_part(psi, op.par)
    assert rel_l2(opg.apply_schur(rot(pe)), rot(op.apply_schur(pe))) < 1e-13
    # clover blocks rotate as A(x) -> Om(x) A(x) Om(x)^H  (colour index inside each spin)
    A = op.A.reshape(T, L, L, L, 4, 3, 4, 3)
    Ag = opg.A.reshape(T, L, L, L, 4, 3, 4, 3)
    Arot = np.einsum("...ab,...sbrc,...dc->...sard", Om, A, np.conj(Om))
    assert rel_l2(Ag, Arot) < 1e-13


# ---------------------------------------------------------------- clover term

def test_clover_constant_abelian_flux_closed_form():
    """U_x = exp(-i phi y T3), U_y = exp(+i phi L x T3) on y = L-1, phi = 2 pi n / L^2:
    every xy plaquette is exp(i phi T3) and
    A_upper = A_lower = (m0+4) 1_6 + (csw/2) sin(phi) sigma_3 (x) T3   exactly."""
    L, T, csw, m0, nflux = 4, 4, 1.3, -0.15, 3
    phi = 2 * np.pi * nflux / L ** 2
    T3 = np.array([1.0, -1.0, 0.0])
    U = _np(gen.unit_gauge_field(L, T))
    for y in range(L):
        U[:, :, y, :, 0] = np.diag(np.exp(-1j * phi * y * T3))
    for x in range(L):
        U[:, :, L - 1, x, 1] = np.diag(np.exp(1j * phi * L * x * T3))
    op = oracle.WilsonClover(L, T, csw, m0, 1, U)
    s3 = np.diag([1.0, -1.0])
    blk = (m0 + 4.0) * np.eye(6) + 0.5 * csw * np.sin(phi) * np.kron(s3, np.diag(T3))
    expect = np.zeros((12, 12), dtype=np.complex128)
    expect[:6, :6] = blk
    expect[6:, 6:] = blk
    assert np.abs(op.A - expect).max() < 1e-14


def _field_strength_numpy(U):
    """Independent (np.roll based) F'_{mu nu} = Q - Q^H, all sites at once."""
    AX = (3, 2, 1, 0)                                   # array axis of direction mu
    dag = lambda M: np.conj(np.swapaxes(M, -1, -2))
    sh = lambda M, mu, s: np.roll(M, -s, axis=AX[mu])   # sh(M,mu,+1)(x) = M(x+mu)

    def F(mu, nu):
        Um, Un = U[..., mu, :, :], U[..., nu, :, :]
        l1 = Um @ sh(Un, mu, 1) @ dag(sh(Um, nu, 1)) @ dag(Un)
        l2 = Un @ dag(sh(sh(Um, mu, -1), nu, 1)) @ dag(sh(Un, mu, -1)) @ sh(Um, mu, -1)
        l3 = dag(sh(Um, mu, -1)) @ dag(sh(sh(Un, mu, -1), nu, -1)) @ sh(sh(Um, mu, -1), nu, -1) @ sh(Un, nu, -1)
        l4 = dag(sh(Un, nu, -1)) @ sh(Um, nu, -1) @ sh(sh(Un, mu, 1), nu, -1) @ dag(Um)
        Q = l1 + l2 + l3 + l4
        return Q - dag(Q)
    return F


def test_clover_chiral_block_form_and_6x6_structure():
    """D_ee, D_oo are block diagonal with 6x6 blocks.  In the chiral basis
    A = A_upper (+) A_lower with
      A_upper = (m0+4) - (csw/16) sum_k sigma_k (x) i (F'_ij - F'_kt),
      A_lower = (m0+4) - (csw/16) sum_k sigma_k (x) i (F'_ij + F'_kt),  (i,j,k) cyclic."""
    L, T = 4, 6
    c = CONFIGS[3]
    U = _np(gen.gauge_field(L, T, 1003, c["eps"], True))
    op = oracle.WilsonClover(L, T, c["csw"], c["m0"], 1, U)
    A = op.A
    assert np.all(A[..., :6, 6:] == 0) and np.all(A[..., 6:, :6] == 0)        # exactly decoupled
    assert np.abs(A - np.conj(np.swapaxes(A, -1, -2))).max() < 1e-14           # Hermitian
    F = _field_strength_numpy(U)
    sig = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
    up = (c["m0"] + 4.0) * np.eye(6)[None, None, None, None] + 0j
    lo = up.copy()
    for k, (i, j) in enumerate(((1, 2), (2, 0), (0, 1))):
        Fij, Fkt = F(i, j), F(k, 3)
        up = up - (c["csw"] / 16.0) * np.einsum("st,...ab->...satb", sig[k], 1j * (Fij - Fkt)).reshape(T, L, L, L, 6, 6)
        lo = lo - (c["csw"] / 16.0) * np.einsum("st,...ab->...satb", sig[k], 1j * (Fij + Fkt)).reshape(T, L, L, L, 6, 6)
    assert np.abs(A[..., :6, :6] - up).max() < 1e-13
    assert np.abs(A[..., 6:, 6:] - lo).max() < 1e-13


@pytest.mark.parametrize("cfg", [1, 3])
def test_clover_blocks_are_constant_plus_spin_traceless(cfg):
    """The property the CUDA path's compact storage of A_ee / A_oo relies on: each
    6x6 block is (m0+4) 1 + sum_k sigma_k (x) G_k, so with rows ordered (spin, colour) its lower-right 3x3
    sub-block equals 2(m0+4) - (upper-left sub-block) and its off-diagonal sub-blocks are each other's
    adjoint.  Checked on the oracle's own A (which is built entry by entry from gamma_mu gamma_nu (x) F'),
    so the statement does not depend on the chiral-block restatement above.  The INVERSE has no such
    structure (it is stored in full)."""
    op = make(cfg, 4, 4)
    c0 = CONFIGS[cfg]["m0"] + 4.0
    for b in (0, 1):
        B = op.A[..., 6 * b:6 * b + 6, 6 * b:6 * b + 6]
        ul, lr, ll, ur = B[..., :3, :3], B[..., 3:, 3:], B[..., 3:, :3], B[..., :3, 3:]
        assert np.abs(lr - (2.0 * c0 * np.eye(3) - ul)).max() < 1e-14
        assert np.abs(ll - np.conj(np.swapaxes(ur, -1, -2))).max() < 1e-14
        Bi = op.Ainv[..., 6 * b:6 * b + 6, 6 * b:6 * b + 6]
        assert np.abs(Bi[..., 3:, 3:] + Bi[..., :3, :3] - 2.0 / c0 * np.eye(3)).max() > 1e-3


def test_clover_independent_of_time_boundary_sign():
    """Every leaf crosses the t boundary an even number of times (reading R2)."""
    U = _np(config_gauge(1))
    Uflip = U.copy()
    Uflip[-1, ..., 3, :, :] *= -1.0
    a = make(1, U=U).A
    b = make(1, U=Uflip).A
    assert np.abs(a - b).max() < 1e-14


@pytest.mark.parametrize("cfg", [1, 3])
def test_clover_inverse(cfg):
    """BASELINE.json: a clover block times its inverse equals the identity to 1e-13."""
    op = make(cfg, 4, 4)
    assert op.n_singular == 0
    prod = op.A @ op.Ainv
    assert np.abs(prod - np.eye(12)).max() <= 1e-13
    assert np.all(op.Ainv[..., :6, 6:] == 0) and np.all(op.Ainv[..., 6:, :6] == 0)


def test_singular_site_is_reported():
    A = np.zeros((2, 12, 12), dtype=np.complex128)
    A[0] = np.eye(12)
    A[1] = np.eye(12)
    A[1, 5, 5] = 0.0
    Ainv = np.zeros_like(A)
    import ctypes
    bad = oracle.lib().oracle_invert_sites(ctypes.c_long(2), A.ctypes.data_as(ctypes.c_void_p),
                                           Ainv.ctypes.data_as(ctypes.c_void_p), ctypes.c_double(1e-12))
    assert bad == 1


# ------------------------------------------------------ eq. 1-3 on dense matrices

@pytest.fixture(scope="module")
def dense_2x4():
    """Config-1 recipe on 2^4 (192 x 192): dense D and the parity index sets."""
    op = make(1, 2, 2)
    D = op.dense(op.apply_D)
    par = np.repeat(op.par.reshape(-1), 12)
    return op, D, np.where(par == 0)[0], np.where(par == 1)[0]


def test_sparsity_nine_blocks_per_block_row():
    """nine 12x12 blocks per block-row (self + 8 neighbours) on 4^4."""
    op = make(1)
    V = op.V
    rng = np.random.default_rng(3)
    for n in rng.choice(V, size=6, replace=False):
        e = np.zeros((V, 12), dtype=np.complex128)
        e[n] = rng.normal(size=12) + 1j * rng.normal(size=12)
        y = op.apply_D(e.reshape(op.shape)).reshape(V, 12)
        touched = np.where(np.abs(y).sum(axis=1) > 0)[0]
        assert len(touched) == 9


def test_schur_equals_dense_block_definition(dense_2x4):
    """eq. 3: D_S = D_ee - D_eo D_oo^-1 D_oe from the blocks of the oracle's own dense D."""
    op, D, ie, io = dense_2x4
    Dee, Deo, Doe, Doo = D[np.ix_(ie, ie)], D[np.ix_(ie, io)], D[np.ix_(io, ie)], D[np.ix_(io, io)]
    DS = Dee - Deo @ np.linalg.solve(Doo, Doe)
    DS_oracle = op.dense(op.apply_schur)
    assert np.abs(DS_oracle[np.ix_(ie, ie)] - DS).max() < 1e-13
    # nothing is read from or written to odd sites
    assert np.all(DS_oracle[io, :] == 0) and np.all(DS_oracle[:, io] == 0)


def test_schur_solve_plus_reconstruction_equals_dense_lu(dense_2x4):
    """eq. 2: prepare_rhs + D_S^-1 + reconstruct_odd == dense LU solve of the full D on 2^4."""
    op, D, ie, io = dense_2x4
    b = _np(gen.spinor_field(2, 2, 2001))
    x_ref = np.linalg.solve(D, b.reshape(-1))
    bhat = op.prepare_rhs(b)
    DS = op.dense(op.apply_schur)[np.ix_(ie, ie)]
    xe = np.zeros(12 * op.V, dtype=np.complex128)
    xe[ie] = np.linalg.solve(DS, bhat.reshape(-1)[ie])
    xe = xe.reshape(op.shape)
    xo = op.reconstruct_odd(b, xe)
    assert np.all(even_part(xo, op.par) == 0)
    assert rel_l2((xe + xo).reshape(-1), x_ref) < 1e-13


def test_schur_block_definition_on_4x4_sampled_columns():
    """Same as above on config 1 (4^4) through D applied to vectors: D_S x_e computed from
    D_ee, D_eo, D_oe, D_oo actions (dense D_oo solve per site is block diagonal)."""
    op = make(1)
    x = _np(config_spinor(1))
    xe = even_part(x, op.par)
    # D (x_e, 0) = (D_ee x_e, D_oe x_e)
    Dx = op.apply_D(xe)
    Dee_x, Doe_x = even_part(Dx, op.par), odd_part(Dx, op.par)
    # D_oo^-1 via numpy solve of the oracle's site matrices
    t = np.linalg.solve(op.A, Doe_x.reshape(*op.shape[:4], 12, 1)).reshape(op.shape)
    t = odd_part(t, op.par)
    Dt = op.apply_D(t)                       # (D_eo t, D_oo t)
    expect = Dee_x - even_part(Dt, op.par)
    assert rel_l2(op.apply_schur(xe), expect) < 1e-13


# --------------------------------------------------------------------- Fig. 1

def test_fig1_qualitative_spectra():
    """spec(D) extends beyond 6.0; D_S is better conditioned, its largest
    eigenvalues moved towards zero and its smallest away from zero (4^4 lattice).
    The figure's gauge field is not given: qualitative only (parity unpinned for exact values)."""
    op = make(1)
    D = op.dense(op.apply_D)
    par = np.repeat(op.par.reshape(-1), 12)
    ie, io = np.where(par == 0)[0], np.where(par == 1)[0]
    DS = D[np.ix_(ie, ie)] - D[np.ix_(ie, io)] @ np.linalg.solve(D[np.ix_(io, io)], D[np.ix_(io, ie)])
    lD = np.abs(np.linalg.eigvals(D))
    lS = np.abs(np.linalg.eigvals(DS))
    assert lD.max() > 6.0
    assert lS.max() < lD.max()
    assert lS.min() > lD.min()
    assert np.linalg.cond(DS) < np.linalg.cond(D)

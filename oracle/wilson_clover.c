/*
 * oracle/wilson_clover.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the hot path computes:
 * the Wilson-clover Dirac operator D = A + H on a periodic L^3 x T lattice and
 * its odd-even Schur complement (eq. 1-3)
 *
 *        D_S = D_ee - D_eo D_oo^{-1} D_oe ,
 *
 * with A the site-diagonal (mass + clover) part (the paper's D_ee (+) D_oo) and
 * H the nearest-neighbour hopping part (the paper's D_eo (+) D_oe).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant with paper_2407_08092_b200/ (the CUDA library) and neither imports
 * the other.
 *
 * Everything is written in the natural layout with full-lattice vectors:
 *   site index   n = x0 + L*(x1 + L*(x2 + L*x3)),  x3 = t in [0,T)
 *   parity       (x0+x1+x2+x3) mod 2, even = 0
 *   spinor       psi[n][spin(4)][colour(3)]                   (12 d.o.f./site)
 *   gauge        U[n][mu(4)][row(3)][col(3)],  mu = x,y,z,t
 *   site matrix  A[n][12][12], row/col index = 3*spin + colour
 * "Half-lattice" vectors x_e / x_o are full-lattice arrays that are zero on
 * the other parity; no checkerboard indexing tricks are used anywhere.
 *
 * The paper never writes the operator down; the definitions below are the
 * readings R1-R5 of SURVEY.md section 8(c) (restated in DESIGN.md):
 *   R1  gamma_mu = [[0, B_mu],[B_mu^H, 0]],  B_k = -i sigma_k (k=x,y,z), B_t = 1
 *   R2  antiperiodic time = sign -1 on U_t of the slice t = T-1 (hopping only)
 *   R3  (H psi)(x) = -1/2 sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu)
 *                                + (1+gamma_mu) U_mu(x-mu)^H psi(x-mu) ]
 *   R4  A(x) = (m0+4) - (csw/32) sum_{mu != nu} gamma_mu gamma_nu (x) F'_{mu nu}(x),
 *       F' = Q - Q^H,  Q = sum of the four plaquette leaves at x
 *   R5  no trace subtraction in F'
 *
 * Pins (tests/test_oracle_*.py, none of them re-types these formulas):
 * free-field plane-wave eigenvalues, gamma5-hermiticity, gauge covariance,
 * constant-abelian-flux closed form of the clover term, A*A^{-1} = 1,
 * Schur + reconstruction == dense LU of the full D on 2^4.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

/* ------------------------------------------------------------------ geometry */

static inline long site_of(int L, int T, const int x[4])
{
    (void)T;
    return (long)x[0] + (long)L * ((long)x[1] + (long)L * ((long)x[2] + (long)L * (long)x[3]));
}

static inline void coords_of(int L, long n, int x[4])
{
    x[0] = (int)(n % L); n /= L;
    x[1] = (int)(n % L); n /= L;
    x[2] = (int)(n % L); n /= L;
    x[3] = (int)n;
}

static inline int extent(int L, int T, int mu) { return mu == 3 ? T : L; }

/* site x + s*mu_hat (s = +1 or -1), periodic wrap */
static inline long shifted(int L, int T, const int x[4], int mu, int s)
{
    int y[4] = { x[0], x[1], x[2], x[3] };
    int e = extent(L, T, mu);
    y[mu] = (y[mu] + s + e) % e;
    return site_of(L, T, y);
}

static inline int parity_of(const int x[4]) { return (x[0] + x[1] + x[2] + x[3]) & 1; }

/* selects which sites a routine writes: 0 = even only, 1 = odd only, 2 = all */
static inline int selected(int sel, int par) { return sel == 2 || sel == par; }

/* ------------------------------------------------------------ gamma matrices */

/* R1: chiral basis.  g[mu][r][c], 4x4 each. */
static void build_gamma(cplx g[4][4][4])
{
    const cplx sig[3][2][2] = {
        { { 0, 1 }, { 1, 0 } },
        { { 0, -I }, { I, 0 } },
        { { 1, 0 }, { 0, -1 } },
    };
    memset(g, 0, sizeof(cplx) * 64);
    for (int mu = 0; mu < 4; ++mu) {
        cplx B[2][2];
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                B[a][b] = (mu < 3) ? (-I * sig[mu][a][b]) : (a == b ? 1.0 : 0.0);
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b) {
                g[mu][a][2 + b] = B[a][b];            /* upper-right block  B      */
                g[mu][2 + a][b] = conj(B[b][a]);      /* lower-left  block  B^H    */
            }
    }
}

/* exported so the tests can pin the Clifford algebra, hermiticity and gamma5 */
void oracle_gamma(cplx* out /* [4][4][4] */)
{
    cplx g[4][4][4];
    build_gamma(g);
    memcpy(out, g, sizeof(g));
}

/* ----------------------------------------------------------- 3x3 helpers */

static inline void m3_mul(const cplx* a, const cplx* b, cplx* c)   /* c = a b */
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            cplx s = 0;
            for (int k = 0; k < 3; ++k) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}

static inline void m3_dag(const cplx* a, cplx* c)                  /* c = a^H */
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c[3 * i + j] = conj(a[3 * j + i]);
}

/* c = a1 a2 a3 a4 */
static void m3_mul4(const cplx* a1, const cplx* a2, const cplx* a3, const cplx* a4, cplx* c)
{
    cplx t1[9], t2[9];
    m3_mul(a1, a2, t1);
    m3_mul(t1, a3, t2);
    m3_mul(t2, a4, c);
}

/* --------------------------------------------------------- boundary condition */

/* R2: Ubc = U, except U_t(x) -> -U_t(x) on the slice t = T-1 when bc == 1. */
void oracle_apply_bc(int L, int T, int bc, const cplx* U, cplx* Ubc)
{
    long V = (long)L * L * L * T;
    memcpy(Ubc, U, sizeof(cplx) * 36 * (size_t)V);
    if (bc != 1) return;
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        if (x[3] == T - 1)
            for (int k = 0; k < 9; ++k) Ubc[36 * n + 9 * 3 + k] = -Ubc[36 * n + 9 * 3 + k];
    }
}

/* ------------------------------------------------------------- hopping term */

/* R3.  out(x) = (H psi)(x) on the selected sites, 0 elsewhere.
 * Ubc must already carry the boundary sign. */
void oracle_hop(int L, int T, const cplx* Ubc, const cplx* psi, cplx* out, int sel)
{
    long V = (long)L * L * L * T;
    cplx g[4][4][4];
    build_gamma(g);
#pragma omp parallel for schedule(static)
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        cplx acc[4][3];
        memset(acc, 0, sizeof(acc));
        if (selected(sel, parity_of(x))) {
            for (int mu = 0; mu < 4; ++mu) {
                /* forward: (1 - gamma_mu) (x) U_mu(x) psi(x+mu) */
                {
                    long nf = shifted(L, T, x, mu, +1);
                    const cplx* u = Ubc + 36 * n + 9 * mu;
                    const cplx* p = psi + 12 * nf;
                    cplx chi[4][3];
                    for (int s = 0; s < 4; ++s)
                        for (int a = 0; a < 3; ++a) {
                            cplx t = 0;
                            for (int b = 0; b < 3; ++b) t += u[3 * a + b] * p[3 * s + b];
                            chi[s][a] = t;
                        }
                    for (int r = 0; r < 4; ++r)
                        for (int s = 0; s < 4; ++s) {
                            cplx w = (r == s ? 1.0 : 0.0) - g[mu][r][s];
                            for (int a = 0; a < 3; ++a) acc[r][a] += w * chi[s][a];
                        }
                }
                /* backward: (1 + gamma_mu) (x) U_mu(x-mu)^H psi(x-mu) */
                {
                    long nb = shifted(L, T, x, mu, -1);
                    const cplx* u = Ubc + 36 * nb + 9 * mu;
                    const cplx* p = psi + 12 * nb;
                    cplx chi[4][3];
                    for (int s = 0; s < 4; ++s)
                        for (int a = 0; a < 3; ++a) {
                            cplx t = 0;
                            for (int b = 0; b < 3; ++b) t += conj(u[3 * b + a]) * p[3 * s + b];
                            chi[s][a] = t;
                        }
                    for (int r = 0; r < 4; ++r)
                        for (int s = 0; s < 4; ++s) {
                            cplx w = (r == s ? 1.0 : 0.0) + g[mu][r][s];
                            for (int a = 0; a < 3; ++a) acc[r][a] += w * chi[s][a];
                        }
                }
            }
            for (int r = 0; r < 4; ++r)
                for (int a = 0; a < 3; ++a) acc[r][a] *= -0.5;
        }
        memcpy(out + 12 * n, acc, sizeof(acc));
    }
}

/* -------------------------------------------------------------- clover term */

/* R4/R5.  A[n][12][12] for every site.  U is the field WITHOUT the boundary
 * sign (the sign cancels in every leaf; tests check that). */
void oracle_clover(int L, int T, double csw, double m0, const cplx* U, cplx* A)
{
    long V = (long)L * L * L * T;
    cplx g[4][4][4];
    build_gamma(g);
#pragma omp parallel for schedule(static)
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        cplx* An = A + 144 * n;
        for (int i = 0; i < 144; ++i) An[i] = 0;
        for (int i = 0; i < 12; ++i) An[13 * i] = m0 + 4.0;

        for (int mu = 0; mu < 4; ++mu)
            for (int nu = 0; nu < 4; ++nu) {
                if (mu == nu) continue;
                /* neighbouring sites of the four leaves */
                int xm[4], xn[4];
                long n_pm = shifted(L, T, x, mu, +1);           /* x+mu      */
                long n_pn = shifted(L, T, x, nu, +1);           /* x+nu      */
                long n_mm = shifted(L, T, x, mu, -1);           /* x-mu      */
                long n_mn = shifted(L, T, x, nu, -1);           /* x-nu      */
                coords_of(L, n_mm, xm);
                coords_of(L, n_mn, xn);
                long n_mm_pn = shifted(L, T, xm, nu, +1);       /* x-mu+nu   */
                long n_mm_mn = shifted(L, T, xm, nu, -1);       /* x-mu-nu   */
                long n_pm_mn = shifted(L, T, xn, mu, +1);       /* x+mu-nu   */
#define LINK(site, dir) (U + 36 * (site) + 9 * (dir))
                cplx d1[9], d2[9], leaf[9], Q[9];
                for (int k = 0; k < 9; ++k) Q[k] = 0;
                /* leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^H U_nu(x)^H */
                m3_dag(LINK(n_pn, mu), d1);
                m3_dag(LINK(n, nu), d2);
                m3_mul4(LINK(n, mu), LINK(n_pm, nu), d1, d2, leaf);
                for (int k = 0; k < 9; ++k) Q[k] += leaf[k];
                /* leaf 2: U_nu(x) U_mu(x-mu+nu)^H U_nu(x-mu)^H U_mu(x-mu) */
                m3_dag(LINK(n_mm_pn, mu), d1);
                m3_dag(LINK(n_mm, nu), d2);
                m3_mul4(LINK(n, nu), d1, d2, LINK(n_mm, mu), leaf);
                for (int k = 0; k < 9; ++k) Q[k] += leaf[k];
                /* leaf 3: U_mu(x-mu)^H U_nu(x-mu-nu)^H U_mu(x-mu-nu) U_nu(x-nu) */
                m3_dag(LINK(n_mm, mu), d1);
                m3_dag(LINK(n_mm_mn, nu), d2);
                m3_mul4(d1, d2, LINK(n_mm_mn, mu), LINK(n_mn, nu), leaf);
                for (int k = 0; k < 9; ++k) Q[k] += leaf[k];
                /* leaf 4: U_nu(x-nu)^H U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^H */
                m3_dag(LINK(n_mn, nu), d1);
                m3_dag(LINK(n, mu), d2);
                m3_mul4(d1, LINK(n_mn, mu), LINK(n_pm_mn, nu), d2, leaf);
                for (int k = 0; k < 9; ++k) Q[k] += leaf[k];
#undef LINK
                /* F' = Q - Q^H */
                cplx F[9];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) F[3 * a + b] = Q[3 * a + b] - conj(Q[3 * b + a]);
                /* gamma_mu gamma_nu */
                cplx gg[4][4];
                for (int r = 0; r < 4; ++r)
                    for (int s = 0; s < 4; ++s) {
                        cplx t = 0;
                        for (int k = 0; k < 4; ++k) t += g[mu][r][k] * g[nu][k][s];
                        gg[r][s] = t;
                    }
                /* A -= (csw/32) gg (x) F' */
                for (int r = 0; r < 4; ++r)
                    for (int s = 0; s < 4; ++s)
                        for (int a = 0; a < 3; ++a)
                            for (int b = 0; b < 3; ++b)
                                An[12 * (3 * r + a) + (3 * s + b)] -= (csw / 32.0) * gg[r][s] * F[3 * a + b];
            }
    }
}

/* ------------------------------------------------------- site-matrix inverse */

/* Ainv[n] = A[n]^{-1}, 12x12 Gauss-Jordan with partial pivoting.  Returns the
 * number of sites whose pivot fell below tol * (largest |entry| of the site
 * matrix) -- 0 means every site was inverted. */
long oracle_invert_sites(long nsites, const cplx* A, cplx* Ainv, double tol)
{
    long bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (long n = 0; n < nsites; ++n) {
        cplx M[12][24];
        double scale = 0;
        for (int i = 0; i < 12; ++i)
            for (int j = 0; j < 12; ++j) {
                M[i][j] = A[144 * n + 12 * i + j];
                M[i][12 + j] = (i == j) ? 1.0 : 0.0;
                double a = cabs(M[i][j]);
                if (a > scale) scale = a;
            }
        int singular = 0;
        for (int c = 0; c < 12; ++c) {
            int p = c;
            for (int i = c + 1; i < 12; ++i)
                if (cabs(M[i][c]) > cabs(M[p][c])) p = i;
            if (!(cabs(M[p][c]) > tol * scale)) { singular = 1; break; }
            if (p != c)
                for (int j = 0; j < 24; ++j) { cplx t = M[c][j]; M[c][j] = M[p][j]; M[p][j] = t; }
            cplx inv = 1.0 / M[c][c];
            for (int j = 0; j < 24; ++j) M[c][j] *= inv;
            for (int i = 0; i < 12; ++i) {
                if (i == c) continue;
                cplx f = M[i][c];
                if (f == 0) continue;
                for (int j = 0; j < 24; ++j) M[i][j] -= f * M[c][j];
            }
        }
        if (singular) { bad += 1; continue; }
        for (int i = 0; i < 12; ++i)
            for (int j = 0; j < 12; ++j) Ainv[144 * n + 12 * i + j] = M[i][12 + j];
    }
    return bad;
}

/* out(x) = M(x) psi(x) on the selected sites, 0 elsewhere */
void oracle_site_matvec(int L, int T, const cplx* M, const cplx* psi, cplx* out, int sel)
{
    long V = (long)L * L * L * T;
#pragma omp parallel for schedule(static)
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        int on = selected(sel, parity_of(x));
        for (int i = 0; i < 12; ++i) {
            cplx s = 0;
            if (on)
                for (int j = 0; j < 12; ++j) s += M[144 * n + 12 * i + j] * psi[12 * n + j];
            out[12 * n + i] = s;
        }
    }
}

/* ------------------------------------------------------------ the operators */

/* y = D x = A x + H x on the whole lattice (the paper's D of "D x = b"). */
void oracle_apply_D(int L, int T, const cplx* Ubc, const cplx* A, const cplx* x, cplx* y)
{
    long V = (long)L * L * L * T;
    cplx* h = (cplx*)malloc(sizeof(cplx) * 12 * (size_t)V);
    oracle_hop(L, T, Ubc, x, h, 2);
    oracle_site_matvec(L, T, A, x, y, 2);
    for (long i = 0; i < 12 * V; ++i) y[i] += h[i];
    free(h);
}

/* eq. 3:  y_e = A_ee x_e - H_eo A_oo^{-1} H_oe x_e.
 * x_e is read on even sites only; y_e is written on even sites, 0 on odd. */
void oracle_apply_schur(int L, int T, const cplx* Ubc, const cplx* A, const cplx* Ainv,
                        const cplx* x_e, cplx* y_e)
{
    long V = (long)L * L * L * T;
    size_t bytes = sizeof(cplx) * 12 * (size_t)V;
    cplx* xe = (cplx*)calloc(1, bytes);
    cplx* t1 = (cplx*)malloc(bytes);
    cplx* t2 = (cplx*)malloc(bytes);
    /* mask x_e to even sites so that the caller's odd entries cannot leak in */
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        int ev = parity_of(x) == 0;
        for (int i = 0; i < 12; ++i) xe[12 * n + i] = ev ? x_e[12 * n + i] : 0.0;
    }
    oracle_hop(L, T, Ubc, xe, t1, 1);                 /* t1 = H_oe x_e        (odd)  */
    oracle_site_matvec(L, T, Ainv, t1, t2, 1);        /* t2 = A_oo^{-1} t1    (odd)  */
    oracle_hop(L, T, Ubc, t2, t1, 0);                 /* t1 = H_eo t2         (even) */
    oracle_site_matvec(L, T, A, xe, y_e, 0);          /* y  = A_ee x_e        (even) */
    for (long i = 0; i < 12 * V; ++i) y_e[i] -= t1[i];
    free(xe); free(t1); free(t2);
}

/* eq. 2, right factor:  bhat_e = b_e - H_eo A_oo^{-1} b_o.
 * b is a full-lattice vector; bhat_e is written on even sites, 0 on odd. */
void oracle_prepare_rhs(int L, int T, const cplx* Ubc, const cplx* Ainv, const cplx* b, cplx* bhat_e)
{
    long V = (long)L * L * L * T;
    size_t bytes = sizeof(cplx) * 12 * (size_t)V;
    cplx* t1 = (cplx*)malloc(bytes);
    cplx* t2 = (cplx*)malloc(bytes);
    oracle_site_matvec(L, T, Ainv, b, t1, 1);         /* t1 = A_oo^{-1} b_o   (odd)  */
    oracle_hop(L, T, Ubc, t1, t2, 0);                 /* t2 = H_eo t1         (even) */
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        int ev = parity_of(x) == 0;
        for (int i = 0; i < 12; ++i) bhat_e[12 * n + i] = ev ? b[12 * n + i] - t2[12 * n + i] : 0.0;
    }
    free(t1); free(t2);
}

/* eq. 2, left factor:  x_o = A_oo^{-1} (b_o - H_oe x_e).
 * b: full-lattice rhs (odd part used); x_e: even part used; x_o written on odd
 * sites, 0 on even. */
void oracle_reconstruct_odd(int L, int T, const cplx* Ubc, const cplx* Ainv, const cplx* b,
                            const cplx* x_e, cplx* x_o)
{
    long V = (long)L * L * L * T;
    size_t bytes = sizeof(cplx) * 12 * (size_t)V;
    cplx* xe = (cplx*)calloc(1, bytes);
    cplx* t1 = (cplx*)malloc(bytes);
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        int ev = parity_of(x) == 0;
        for (int i = 0; i < 12; ++i) xe[12 * n + i] = ev ? x_e[12 * n + i] : 0.0;
    }
    oracle_hop(L, T, Ubc, xe, t1, 1);                 /* t1 = H_oe x_e        (odd)  */
    for (long n = 0; n < V; ++n) {
        int x[4];
        coords_of(L, n, x);
        int od = parity_of(x) == 1;
        for (int i = 0; i < 12; ++i) t1[12 * n + i] = od ? b[12 * n + i] - t1[12 * n + i] : 0.0;
    }
    oracle_site_matvec(L, T, Ainv, t1, x_o, 1);
    free(xe); free(t1);
}

/*
 * ddamg.h -- C ABI of libddamg.so: the finest-level hot path of DD-alphaAMG as
 * extended by arXiv:2407.08092, hand-written for NVIDIA B200 (sm_100a).
 *
 * The path (PAPER.md = /root/reference/PAPER.md, the paper's text):
 *   * odd-even reordering of D x = b                        eq. 1
 *   * Schur factorisation of D^-1                           eq. 2
 *   * Schur complement  D_S = D_ee - D_eo D_oo^-1 D_oe      eq. 3
 *   * modified Richardson on D_S x_e = bhat_e               Alg. 4
 *   * restarted GMRES(n, m) on D_S x_e = bhat_e             Alg. 2
 *   * "odd-even + {GMRES, Richardson}": whole lattice reordered, iteration runs on the
 *     Schur system
 * D is the Wilson-clover operator with 12 d.o.f. per site;
 * D_ee, D_oo are block diagonal with 6x6 blocks and D_oo^-1 is stored.
 * The paper never writes D down; DESIGN.md lists the readings (gamma basis, hopping
 * normalisation, clover leaves, boundary condition) this library and the oracle use:
 *   D = A + H,  A(x) = (m0+4) - (csw/32) sum_{mu!=nu} gamma_mu gamma_nu (x) F'_munu(x),
 *   (H psi)(x) = -1/2 sum_mu [(1-gamma_mu) U_mu(x) psi(x+mu) + (1+gamma_mu) U_mu(x-mu)^H psi(x-mu)].
 *
 * Conventions
 *   * One context = one lattice, one precision, one CUDA stream, one GPU (the current
 *     device at ddamg_create).  No multi-GPU sharding, no collectives.
 *   * "natural" layout (external): site n = x + L*(y + L*(z + L*t)); complex numbers are
 *     (re, im) pairs of the context precision unless an argument says otherwise.
 *       gauge   U[n][mu][row][col]      mu = 0..3 = x,y,z,t       (72 reals / site)
 *       spinor  psi[n][spin][colour]                              (24 reals / site)
 *   * "native" layout (internal, checkerboarded SoA): a half-lattice spinor of parity p
 *     holds the V/2 sites with (x+y+z+t) mod 2 == p (even = 0) at
 *     checkerboard index cb = n >> 1, as 24/NV planes of V/2 16-byte vectors
 *     (NV = 4 floats or 2 doubles); plane j holds reals NV*j .. NV*j+NV-1 of the site's
 *     24 reals (spin-major, then colour, then re/im).  Size: 12*V complex = 24*(V/2) reals.
 *     Callers obtain native buffers only through ddamg_pack_spinor / ddamg_unpack_spinor;
 *     every x_e / x_o / b_e / b_o argument below is a DEVICE pointer to such a buffer,
 *     16-byte aligned, of ddamg_half_spinor_bytes() bytes, owned by the caller.
 *   * All work is enqueued on the context's stream.  Functions that return a residual
 *     history synchronise that stream once before returning; the others are asynchronous.
 *   * Every function returns DDAMG_OK (0) or a negative status and never aborts, exits
 *     or throws.  A CUDA error is sticky: all later calls return DDAMG_ECUDA until
 *     ddamg_destroy.  ddamg_last_error() gives a human-readable message.
 *   * There is no CPU fallback: without a CUDA device ddamg_create returns DDAMG_ECUDA.
 */
#ifndef DDAMG_H
#define DDAMG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ddamg_ctx ddamg_ctx;   /* opaque; owns all internal device memory */

enum {
    DDAMG_OK = 0,
    DDAMG_EINVAL = -1,     /* bad argument (null pointer, odd L/T, nu < 0, k < 1, ...) */
    DDAMG_ENOMEM = -2,     /* device or host allocation failed                        */
    DDAMG_ESTATE = -3,     /* call out of order (no gauge loaded / clover not built)  */
    DDAMG_ECUDA = -4,      /* CUDA runtime error (sticky)                             */
    DDAMG_ESINGULAR = -5   /* a 6x6 clover block is numerically singular              */
};
enum { DDAMG_F32 = 0, DDAMG_F64 = 1 };
enum { DDAMG_BC_PERIODIC = 0, DDAMG_BC_ANTIPERIODIC_T = 1 };
enum { DDAMG_SMOOTHER_RICHARDSON = 0, DDAMG_SMOOTHER_GMRES = 1, DDAMG_SMOOTHER_GCR = 2, DDAMG_SMOOTHER_SAP = 3 };

/* Library version string, e.g. "ddamg-b200 0.1 (sm_100a)". Never NULL. */
const char* ddamg_version(void);

/*
 * Create a context for an L^3 x T lattice (L, T even, >= 2; L^3*T/2 < 2^31).
 *   csw, m0   clover coefficient and bare mass of D (Table 5 names them)
 *   bc        DDAMG_BC_PERIODIC or DDAMG_BC_ANTIPERIODIC_T (time links of slice T-1 negated)
 *   prec      DDAMG_F32 or DDAMG_F64: precision of every stored field and of every
 *             spinor argument (reductions always accumulate in fp64)
 *   cuda_stream  a cudaStream_t (host value) or NULL for the legacy default stream
 * On success *out is a new context (caller destroys it).  EINVAL / ENOMEM / ECUDA.
 */
int ddamg_create(ddamg_ctx** out, int L, int T, double csw, double m0, int bc, int prec,
                 void* cuda_stream);

/* Free everything the context owns (synchronises its stream first). NULL is a no-op. */
int ddamg_destroy(ddamg_ctx* ctx);

/* Message of the last failure on this context ("" if none).  ctx may be NULL. */
const char* ddamg_last_error(ddamg_ctx* ctx);

/* Bytes of one native half-lattice spinor = 24 * (V/2) * sizeof(real).  0 if ctx is NULL. */
size_t ddamg_half_spinor_bytes(ddamg_ctx* ctx);

/*
 * Load the gauge field (step a0).  U: natural layout, u_prec = DDAMG_F32/F64 complex,
 * HOST pointer if on_device == 0 (copied with cudaMemcpyAsync, then the stream is
 * synchronised), DEVICE pointer otherwise.  The field is rounded to the context
 * precision, repacked per parity and direction, and the antiperiodic sign is folded into
 * the time links of slice T-1.  The caller keeps U.  Invalidates a previously built clover.
 */
int ddamg_load_gauge(ddamg_ctx* ctx, const void* U, int u_prec, int on_device);

/*
 * Build the clover term (step a1) from the loaded links: per site the two Hermitian 6x6
 * blocks of A(x), computed in fp64, stored in the context precision;
 * A itself is kept on even sites, its INVERSE on odd sites ("explicitly storing the data
 * for D_oo^-1 is cheap").  Storage (internal): the inverses as packed Hermitian blocks (36
 * reals each); the blocks themselves in a compact 28-real form that uses their structure
 * A_+- = (m0+4) + sum_k sigma_k (x) G_k (the lower-right 3x3 sub-block is 2(m0+4) minus the
 * upper-left one), 224 instead of 288 bytes per even site in fp32.  Synchronises.  ESTATE without a gauge field; ESINGULAR if an
 * odd-site block has a pivot below 1e-12 * (largest entry of the block).
 */
int ddamg_build_clover(ddamg_ctx* ctx);

/* eq. 3:  y_e = D_S x_e = A_ee x_e - H_eo A_oo^-1 H_oe x_e.   y_e must not alias x_e. */
int ddamg_apply_schur(ddamg_ctx* ctx, const void* x_e, void* y_e);

/*
 * The same operator (eq. 3), for callers that must not allocate: code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc.  The call performs NO cudaMalloc / cudaFree
 * and calls no allocating library routine: the intermediate t_o = A_oo^-1 H_oe x_e lives in a static device
 * array inside libddamg.so of ddamg_noalloc_max_bytes() = 8 MiB (held by every GPU that loads the library until
 * the process exits) instead of in context-owned memory.  Same two kernels, same arithmetic: results are
 * bit-identical to ddamg_apply_schur.
 *   x_e, y_e   DEVICE native half spinors as for ddamg_apply_schur (caller-owned, must not alias).
 * Limit: one half spinor (ddamg_half_spinor_bytes) must fit the array -- fp32 lattices up to V/2 = 87381
 * sites (e.g. 16^3 x 32), fp64 up to 43690 (e.g. 16^4); EINVAL with a message naming both sizes beyond that.
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress; no allocation): make
 * it once per device, with that device current, before entering a capture.  ALL contexts and calls on a device
 * share the one array, which keeps the last call's contents; nothing in it has to start at zero (kernel A
 * overwrites every element kernel B reads), but two calls that overlap on the GPU (different streams or
 * contexts without ordering between them) RACE on it: serialise them.
 * ESTATE before the gauge field and the clover term are set up, or while ddamg_kernel_timing is on (its event
 * pool may grow); ECUDA if the address cannot be resolved.
 */
int ddamg_apply_schur_noalloc(ddamg_ctx* ctx, const void* x_e, void* y_e);
size_t ddamg_noalloc_max_bytes(void);

/*
 * Alg. 4 with omega supplied (lines 2-4):  nu times  r = b_e - D_S x_e;  x_e += omega r.
 *   x_e        in: x^(0) (ignored if zero_init != 0, then x^(0) = 0 and the first sweep is
 *              x = omega b_e without an operator application); out: x^(nu).  In place.
 *   res_hist   HOST array of nu doubles or NULL; res_hist[i] = || b_e - D_S x^(i) ||_2,
 *              i = 0..nu-1 (by-product of sweep i+1).  NULL skips the reductions and the
 *              stream synchronisation.
 * EINVAL if nu < 0 or b_e aliases x_e.
 */
int ddamg_richardson(ddamg_ctx* ctx, const void* b_e, void* x_e, int nu, double omega,
                     int zero_init, double* res_hist);

/*
 * Alg. 2: restarted GMRES(n = cycles, m = k) on D_S x_e = b_e.
 *   x_e        in: x^(0) (ignored if zero_init); out: the final iterate.
 *   tol        0: run all cycles*k steps (smoother use); > 0: stop as soon as the Givens
 *              residual estimate <= tol * ||b_e|| (checked on the host every step)
 *   res_hist   HOST array of cycles*(k+1)+1 doubles or NULL: for each cycle the true
 *              ||b_e - D_S x|| at its start followed by the k residual estimates, then the
 *              true residual norm at the end.  *n_hist (may be NULL) = entries written.
 * Orthogonalisation: classical Gram-Schmidt in two fused passes (one multi-dot, one
 * multi-axpy + norm), partial sums in fp64 (reading R15); for k > 12 or tol > 0 the two
 * passes are repeated once (CGS2) so that the Givens residual estimates stay reliable in fp32.
 * The basis is kept lazily normalised (vector + device scalar, reading R15b): no separate
 * normalisation pass.
 * EINVAL if k < 1, cycles < 1 or b_e aliases x_e.  ENOMEM if the Krylov basis
 * ((k+1) half spinors) cannot be allocated.
 */
int ddamg_gmres_oe(ddamg_ctx* ctx, const void* b_e, void* x_e, int k, int cycles, double tol,
                   int zero_init, double* res_hist, int* n_hist);

/*
 * Alg. 3: GCR(n = cycles, m = k) on D_S x_e = b_e -- SURVEY.md NEXT-4.
 * Arguments, history layout (cycles*(k+1)+1 entries: true residual at each cycle start, the
 * recursively updated ||r|| after each of the k steps, true residual at the end), tol and
 * error behaviour as ddamg_gmres_oe.  Mathematically equivalent to GMRES but
 * keeps 2k+1 half spinors (p_j, z_j = D_S p_j, r) and does one D_S application per step;
 * lines 11-14 run as one fused pass that also yields delta_{k+1} and (r, z_{k+1}).
 */
int ddamg_gcr_oe(ddamg_ctx* ctx, const void* b_e, void* x_e, int k, int cycles, double tol,
                 int zero_init, double* res_hist, int* n_hist);

/*
 * The full operator of eq. 1 on both parities:
 *   y_e = A_ee x_e + H_eo x_o,   y_o = A_oo x_o + H_oe x_e.
 * Builds and keeps A_oo itself on first use (the Schur path stores only A_oo^-1).
 * No output may alias an input.
 */
int ddamg_apply_full(ddamg_ctx* ctx, const void* x_e, const void* x_o, void* y_e, void* y_o);

/*
 * Outer solver: flexible GMRES(n = cycles, m = k) on the full system
 * D x = b (PAPER.md:77 names FGMRES as DD-alphaAMG's outer solver), preconditioned by ONE
 * odd-even smoother call per Krylov vector and nothing else (no coarse grid):
 *   z = M v:  bhat_e = v_e - H_eo A_oo^-1 v_o;  z_e = smoother on D_S z_e = bhat_e from z_e = 0;
 *             z_o = A_oo^-1 (v_o - H_oe z_e)                                   (eq. 2)
 *   smoother = DDAMG_SMOOTHER_RICHARDSON: s_n sweeps with weight omega (s_m ignored)
 *              DDAMG_SMOOTHER_GMRES / _GCR: (n = s_n cycles, m = s_m) without tolerance
 *              DDAMG_SMOOTHER_SAP: z = SAP(s_n, s_m) on D z = v from z = 0 (Alg. 1; acts on the
 *              full system, no eq.-2 wrapper; block extents from the "sap_block_*" options,
 *              default 4^4 as in Table 6; s_m = 0 is rejected)
 * The paper prints no FGMRES algorithm; reading R19: Alg. 2 with z_j = M v_j,
 * w = D z_j, x += Z_m y.  History layout, tol, zero_init as ddamg_gmres_oe (norms over both
 * parities).  x_e / x_o: initial guess in, solution out.  Keeps 2k+1 full-lattice vectors.
 */
int ddamg_fgmres(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* x_e, void* x_o, int k, int cycles,
                 double tol, int smoother, int s_n, int s_m, double omega, int zero_init, double* res_hist,
                 int* n_hist);

/*
 * Alg. 1: SAP(n, m) on the full system D x = b -- SURVEY.md NEXT-3.
 * The lattice is cut into 4-D blocks of block[0..3] = (Bx, By, Bz, Bt) sites, coloured
 * red/black by the parity of the sum of their block coordinates.  Each of the
 * n outer iterations computes r = b - D x (line 2), approximately solves D_k e_k = r_k on every
 * red block and adds e_k to x_k (lines 4-6), recomputes r (line 7) and does the same on the
 * black blocks (lines 8-10).  D_k = P_k D P_k^T (hops leaving the block dropped).  The block
 * solve is m Minimal Residual iterations with block-local odd-even preconditioning
 * (PAPER.md:179): rhat_e = r_e - H^k_eo A_oo^-1 r_o; e = 0, rho = rhat_e, m times
 * { q = D^k_S rho; alpha = <q,rho>/<q,q>; e += alpha rho; rho -= alpha q };
 * e_o = A_oo^-1 (r_o - H^k_oe e)  (readings R20-R24).  All dot products are
 * block-local; one CTA per block, the block's links staged in shared memory.
 *   block      HOST array of 4 ints; each even, dividing L (L, L, T) with an EVEN quotient, at
 *              most 512 sites per block, links of one block must fit in shared memory
 *              (fp32: up to 512 sites, fp64: up to 256 sites) -- else EINVAL
 *   x_e, x_o   in: x^(0) (ignored if zero_init != 0); out: x^(n).  In place.  With zero_init and
 *              res_hist == NULL the first residual is b itself (b - D 0) and is not computed.
 *   res_hist   HOST array of n+1 doubles or NULL: ||b - D x^(i)||_2 for i = 0..n (the first n
 *              are the residuals of line 2; the last costs one extra residual).  NULL skips
 *              the reductions and the stream synchronisation.
 * m = 0 leaves x unchanged.  Builds and keeps A_oo on first use (as ddamg_apply_full), and
 * block-ordered copies of the links and of A_ee / A_oo^-1 for the block geometry last used
 * (2 x the size of the gauge field; rebuilt when the geometry, the links or the clover change).
 */
int ddamg_sap(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* x_e, void* x_o, int n, int m,
              const int* block, int zero_init, double* res_hist);

/* eq. 2, left factor:  x_o = A_oo^-1 (b_o - H_oe x_e). */
int ddamg_reconstruct_odd(ddamg_ctx* ctx, const void* b_o, const void* x_e, void* x_o);

/* eq. 2, right factor: bhat_e = b_e - H_eo A_oo^-1 b_o.   bhat_e may alias b_e. */
int ddamg_prepare_rhs(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* bhat_e);

/*
 * Alg. 4 line 1: a few power iterations for |lambda_max(D_S)| starting from v_e
 * (overwritten).  *lambda_max (HOST) = ||D_S v|| / ||v|| of the last iteration.  Synchronises.
 */
int ddamg_power_iteration(ddamg_ctx* ctx, void* v_e, int iters, double* lambda_max);

/* natural (DEVICE, context precision, full lattice, 16-byte aligned: EINVAL otherwise) -> native halves.
 * x_e or x_o may be NULL. */
int ddamg_pack_spinor(ddamg_ctx* ctx, const void* nat, void* x_e, void* x_o);
/* native halves -> natural (DEVICE).  A NULL half writes zeros on that parity. */
int ddamg_unpack_spinor(ddamg_ctx* ctx, const void* x_e, const void* x_o, void* nat);

/*
 * ---- Multi-rhs batching (PAPER.md:310-312 names "applying each block to
 * many vectors" / multiple right-hand sides as the way to raise cache reuse).  The same D_S is
 * applied to nrhs (1..32, V/2 * nrhs < 2^31) right-hand sides in one pass: links and clover
 * blocks, 78 % of the bytes of a single-rhs pass, are fetched once per site for all of them.
 * A BATCH is a DEVICE buffer of ddamg_batch_spinor_bytes(ctx, nrhs) bytes holding nrhs native
 * half spinors interleaved per site.
 *   fp64 context: nrhs * half-spinor bytes; plane j (double2), vector index cb * nrhs + r
 *     (r = rhs index, fastest).
 *   fp32 context: right-hand sides travel in PAIRS (2p, 2p+1), one thread per (site, pair), every
 *     operation a packed f32x2 instruction whose two lanes are the two right-hand sides (links,
 *     rebuilt third rows, clover entries and index arithmetic are shared by the pair):
 *     2 * ceil(nrhs / 2) * half-spinor bytes; 12 half-planes of float4; half-plane h (= complex
 *     number h = 3 * spin + colour of the site), vector index cb * npairs + p =
 *     (re of rhs 2p, re of rhs 2p+1, im of rhs 2p, im of rhs 2p+1).  With an odd nrhs the second
 *     lane of the last pair is padding (written as 0 by ddamg_batch_interleave, ignored by
 *     ddamg_batch_deinterleave and by the residual history).
 * Callers build batches with ddamg_batch_interleave from nrhs native half spinors stored back
 * to back (halves = [r][native half spinor]) and read them back with ddamg_batch_deinterleave;
 * both are asynchronous, neither may alias.
 * Every *_batch function computes, for each r independently, exactly what its single-rhs
 * namesake computes (same arithmetic, same order: results are bit-identical per rhs).
 */
size_t ddamg_batch_spinor_bytes(ddamg_ctx* ctx, int nrhs);
int ddamg_batch_interleave(ddamg_ctx* ctx, int nrhs, const void* halves, void* X);
int ddamg_batch_deinterleave(ddamg_ctx* ctx, int nrhs, const void* X, void* halves);
/* eq. 3 for every rhs:  Y_e[r] = D_S X_e[r].  Y_e must not alias X_e. */
int ddamg_apply_schur_batch(ddamg_ctx* ctx, int nrhs, const void* X_e, void* Y_e);
/*
 * Alg. 4 (omega supplied) on every rhs, in place.  res_hist: HOST array of nu * nrhs doubles
 * or NULL, res_hist[i * nrhs + r] = || B_e[r] - D_S X^(i)[r] ||_2.  zero_init != 0 starts from
 * X = 0 (run as a full sweep on a zeroed batch; the result equals X = omega B bit for bit).
 * EINVAL if nu < 0, nrhs out of range, nu * nrhs > 8192 with a history, or B_e aliases X_e.
 */
int ddamg_richardson_batch(ddamg_ctx* ctx, int nrhs, const void* B_e, void* X_e, int nu, double omega,
                           int zero_init, double* res_hist);
/* eq. 2 factors for every rhs (see ddamg_reconstruct_odd / ddamg_prepare_rhs). */
int ddamg_reconstruct_odd_batch(ddamg_ctx* ctx, int nrhs, const void* B_o, const void* X_e, void* X_o);
int ddamg_prepare_rhs_batch(ddamg_ctx* ctx, int nrhs, const void* B_e, const void* B_o, void* Bhat_e);

/*
 * Debug / parity: the stored clover blocks as dense matrices, natural site order, DEVICE
 * buffers of V*2*6*6 complex numbers of the context precision ([n][block][row][col],
 * block 0 = spins 0,1, block 1 = spins 2,3, row = 3*(spin mod 2) + colour).
 *   A_nat     A(x) blocks on even sites, zeros on odd sites  (may be NULL)
 *   Ainv_nat  A(x)^-1 blocks on odd sites, zeros on even     (may be NULL)
 */
int ddamg_get_clover(ddamg_ctx* ctx, void* A_nat, void* Ainv_nat);

/*
 * Options:
 *   "batch_l2_bytes"  L2 budget (bytes, default 40e6) of the multi-rhs kernels' z-chunked
 *                     traversal: CTAs visit the lattice in chunks of zc z-planes (zc = largest
 *                     divisor of L with 3 * zc * one (z,t)-plane of batch spinors <= budget)
 *                     so that t-neighbours are re-read from L2, not HBM.  0 = smallest chunks;
 *                     a huge value = plain lexicographic order.  Never changes results.
 *   "sap_block_x", "sap_block_y", "sap_block_z", "sap_block_t"
 *                     block extents SAP uses as the FGMRES smoother (even integers >= 2,
 *                     default 4; checked against the lattice when the smoother runs).
 *   "gauge_recon"     18 (default) or 12.  12 = two-row link storage: the
 *                     fused hopping kernels (Schur apply, Richardson, GMRES, GCR, eq.-2
 *                     factors, full operator, multi-rhs) read rows 0 and 1 of each SU(3) link
 *                     (48 B instead of 72 B in fp32) from a second, context-owned copy and
 *                     rebuild row 2 = conj(row0 x row1) in registers (sign of the antiperiodic
 *                     boundary restored).  May be set before or after ddamg_load_gauge; every
 *                     later ddamg_load_gauge re-compresses.  The links must be SU(3): if any
 *                     stored third row differs from the rebuilt one by more than 2e-6 (fp32
 *                     context) / 1e-12 (fp64) the call returns EINVAL and the context stays
 *                     on 18-real links.  Results change by rounding only (third rows are
 *                     rebuilt from rounded rows).  Clover build and SAP block solves always
 *                     use the full links.
 *   "cuda_graph"      -1 (default, auto), 0 or 1.  A history-free ddamg_richardson call (res_hist NULL,
 *                     nu > 1: the smoother use) is 2 nu kernel launches with no host work between
 *                     them; with 1 they are captured once into a CUDA graph and replayed by one
 *                     graph launch per call (re-captured when b_e, x_e, nu, omega, zero_init or the
 *                     link format change).  Auto = on for lattices up to 2^19 sites per parity,
 *                     where the kernels are short enough for launch gaps to show.  Same kernels,
 *                     same order: bit-identical results.  Off while ddamg_kernel_timing is on.
 *   "sap_blocked"     1 (default) or 0.  ddamg_sap keeps its residual and update vectors block-ordered
 *                     (contiguous per domain-decomposition block) instead of in the native half-spinor
 *                     layout; same arithmetic per site, results identical up to the summation order of
 *                     the residual-history norms.
 * EINVAL for an unknown name or a bad value.
 */
int ddamg_set_option(ddamg_ctx* ctx, const char* name, double value);

/* Number of kernel launches this context has enqueued since creation (bench accounting). */
long long ddamg_launch_count(ddamg_ctx* ctx);

/*
 * Time the kernels of the last ddamg_apply_schur / ddamg_richardson call pattern:
 * when enabled (on != 0) every hot-path kernel launch is bracketed by CUDA events on the
 * context's stream; ddamg_kernel_time_ms returns the accumulated device time (ms) and the
 * number of launches of kernel class `which` (0 = kernel A: A_oo^-1 H_oe, 1 = kernel B /
 * B': A_ee x - H_eo t with optional Richardson update, 2 = eq.-2 factors, 3 / 4 = the
 * multi-rhs forms of kernel A / kernel B, B', 5 = one parity of the full operator /
 * residual, 6 = SAP block-solve kernel, 8 = fused multi-dot, 9 = fused
 * multi-axpy (+ norm), 10 = the other streaming BLAS-1 passes of GMRES / GCR) since the last
 * reset, after synchronising the stream.  The event pairs come from a pool created by
 * ddamg_kernel_timing(ctx, 1) (4096 pairs, grown in chunks if a measurement records more):
 * no event is created inside a timed call.  Used by bench.py for the per-kernel roofline.
 */
int ddamg_kernel_timing(ddamg_ctx* ctx, int on);
int ddamg_kernel_time_ms(ddamg_ctx* ctx, int which, double* ms, long long* launches, int reset);

#ifdef __cplusplus
}
#endif
#endif /* DDAMG_H */

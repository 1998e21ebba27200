// ddamg_internal.h -- declarations shared by the translation units of libddamg.so.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include "ddamg_common.cuh"

namespace ddamg {

#ifndef DDAMG_DSLASH_THREADS
#define DDAMG_DSLASH_THREADS 128
#endif
constexpr int DSLASH_THREADS = DDAMG_DSLASH_THREADS;
constexpr int BLAS_THREADS = 256;
constexpr int GMRES_KMAX = 64;          // largest cycle length m of GMRES(n, m)
constexpr int HIST_MAX = 8192;         // residual-history entries kept on the device
constexpr int NRHS_MAX = 32;            // right-hand sides per multi-rhs batch
constexpr int MDOT_NB = 12;             // basis vectors handled per fused multi-dot / multi-axpy pass
constexpr int SAP_MAX_THREADS = 256;    // SAP: sites per parity of one domain-decomposition block (<= 512-site blocks)

// epilogues of the fused hopping kernel (ddamg_dslash.cu)
enum {
    EPI_CLOV_HOP = 0,            // out = Cl (H in)                         kernel A
    EPI_CLOV_RHS_MINUS_HOP = 1,  // out = Cl (rhs - H in)                   reconstruct_odd
    EPI_RHS_MINUS_HOP = 2,       // out = rhs - H in                        prepare_rhs
    EPI_SCHUR = 3,               // out = Cl own - H in                     kernel B
    EPI_RICHARDSON = 4,          // r = rhs - (Cl own - H in); out = own + w r   kernel B'
    EPI_RESIDUAL = 5,            // out = rhs - (Cl own - H in)
    EPI_FULL = 6,                // out = Cl own + H in                     one parity of D = A + H
    EPI_FULL_RESIDUAL = 7        // out = rhs - (Cl own + H in)             one parity of b - D x
};

template <typename T>
void launch_dslash(const Geom& g, int epi, bool norm, int parity, const void* in, const void* gauge_own,
                   const void* gauge_opp, const void* clov, const void* own, const void* rhs, void* out,
                   double omega, double c0, double* partials, int units, double batch_l2_bytes, int recon, int apbc,
                   cudaStream_t st);
// clov: for EPI_CLOV_* the INVERSE blocks (packed 36 reals per block), for EPI >= EPI_SCHUR the blocks themselves in
// the compact form of load_clover_A (CLOVA_REALS per block; c0 = m0 + 4)
// `units`: 0 = one right-hand side in the native half-spinor layout; >= 1 = multi-rhs batch processed by that
// many threads per site: fp32 -> pairs of right-hand sides (pair layout, batch_units()), fp64 -> right-hand sides
inline int batch_units(int nrhs, size_t real_bytes) { return real_bytes == 4 ? (nrhs + 1) / 2 : nrhs; }
inline int batch_slots(int nrhs, size_t real_bytes) { return real_bytes == 4 ? 2 * ((nrhs + 1) / 2) : nrhs; }   // rhs slots incl. padding
// two-row copy of the packed gauge field (option "gauge_recon" = 12) + max deviation of the
// stored third rows from conj(row0 x row1): *dev_max_bits = bit pattern of the largest
// absolute deviation as a non-negative float (atomicMax on the bits; zero it first)
template <typename T>
void launch_compress_gauge(const Geom& g, int bc, const void* gauge, void* gauge12, unsigned int* dev_max_bits,
                           cudaStream_t st);
template <typename T>
void launch_clover_apply(const Geom& g, const void* clov, const void* in, void* out, int units, cudaStream_t st);
int dslash_grid(const Geom& g, int units = 1);

// ---- SAP block solves (ddamg_sap.cu)
struct SapGeom {
    int B[4];            // block extents (each even, dividing the lattice extent with an even quotient)
    int Bxh;             // B[0] / 2
    int Vbh;             // sites per parity of one block
    int nb[4];           // blocks per direction
    int nbxh;            // nb[0] / 2
};
size_t sap_smem_bytes(const SapGeom& sg, size_t real_bytes, int recon);
// block-ordered copies of the links (2 * 4 * recon reals per site pair; recon = 18, or 12: rows 0 and 1) and of
// A_ee / A_oo^-1 (slots of 72 reals per site; A_ee keeps its compact form and uses 2 * CLOVA_REALS of its slot),
// V/2 site pairs each, for one block geometry; clov_e is the context's compact A_ee
template <typename T>
void launch_sap_reorder(const Geom& g, const SapGeom& sg, int recon, const void* gauge, const void* clov_e,
                        const void* clov_oinv, void* blk_links, void* blk_clov, cudaStream_t st);
// block solves of one colour: x += e, e -> (e_e, e_o), residual (rho, 0) -> (rn_e, rn_o) on those blocks
template <typename T>
cudaError_t launch_sap_blocks(const Geom& g, const SapGeom& sg, int recon, double c0, int colour, int m, const void* blk_links,
                              const void* blk_clov, const void* r_e, const void* r_o, void* rn_e, void* rn_o,
                              void* e_e, void* e_o, void* x_e, void* x_o, int blocked, int rin_native, int x_assign,
                              cudaStream_t st);
// rin_native: (blocked only) the input residual is still a native half-spinor pair; x_assign: x = e instead of x += e
// blocked != 0: r, rn, e are block-ordered arrays (per parity [block][24/N planes][n] 16-byte vectors) instead of
// native half spinors; launch_sap_spinor_to_blocked converts a native pair, launch_sap_boundary_blocked is the
// in-place incremental residual on them (links from the block-ordered link copy)
template <typename T>
void launch_sap_spinor_to_blocked(const Geom& g, const SapGeom& sg, const void* s_e, const void* s_o, void* b_e, void* b_o,
                                  cudaStream_t st);
template <typename T>
void launch_sap_boundary_blocked(const Geom& g, const SapGeom& sg, int recon, int target, int apbc, const void* blk_links,
                                 const void* e_e, const void* e_o, void* r_e, void* r_o, const void* native_in_e,
                                 const void* native_in_o, cudaStream_t st);
// native_in_* != NULL: the input residual of the target blocks is read from that native pair (and every site of the
// block written block-ordered) instead of in place
// rn = r - (hops across block faces) e on the sites of colour `target`; gauge: the hopping kernels' link blocks
// (recon reals per link), apbc as in launch_dslash
template <typename T>
void launch_sap_boundary(const Geom& g, const SapGeom& sg, int recon, int target, int apbc, const void* gauge,
                         const void* e_e, const void* e_o, const void* r_e, const void* r_o, void* rn_e, void* rn_o,
                         cudaStream_t st);

// ---- setup (ddamg_setup.cu)
template <typename Tin, typename T>
void launch_pack_gauge(const Geom& g, int bc, const void* U_nat, void* gauge, cudaStream_t st);
template <typename T>
void launch_pack_spinor(const Geom& g, const void* nat, void* x_e, void* x_o, cudaStream_t st);
template <typename T>
void launch_unpack_spinor(const Geom& g, const void* x_e, const void* x_o, void* nat, cudaStream_t st);
template <typename T>
void launch_batch_interleave(const Geom& g, int nrhs, bool to_batch, void* halves, void* X, cudaStream_t st);
// fast path (unpivoted LDL^H; *need_pivot_flag is raised when a block needs the pivoted rebuild) and the
// pivoted Gauss-Jordan build (*singular_flag raised for a numerically singular block)
template <typename T>
void launch_build_clover(const Geom& g, double csw, double m0, const void* gauge, void* clov_e, void* clov_o,
                         void* clov_o_plain, int* need_pivot_flag, cudaStream_t st);
template <typename T>
void launch_build_clover_pivoted(const Geom& g, double csw, double m0, const void* gauge, void* clov_e, void* clov_o,
                                 void* clov_o_plain, int* singular_flag, cudaStream_t st);
template <typename T>
void launch_get_clover(const Geom& g, double c0, const void* clov_e, const void* clov_o, void* A_nat, void* Ainv_nat,
                       cudaStream_t st);

// ---- BLAS-1 and the small dense part of GMRES (ddamg_blas.cu)
// device scalar block used by Richardson / GMRES / power iteration (all fp64)
struct Scalars {
    double hist[HIST_MAX];                              // residual history
    double H[(GMRES_KMAX + 1) * GMRES_KMAX * 2];        // Hessenberg / R factor, column major, complex
    double cs[GMRES_KMAX * 2], sn[GMRES_KMAX * 2];      // Givens rotations
    double gvec[(GMRES_KMAX + 1) * 2];                  // rotated beta e_1
    double y[GMRES_KMAX * 2];                           // least-squares solution
    double ys[GMRES_KMAX * 2];                          // y_i * vs[i]: coefficients of the stored basis vectors
    double vs[GMRES_KMAX + 1];                          // GMRES: v_i = vs[i] * stored_i (lazy normalisation)
    double hcol[(GMRES_KMAX + 1) * 2];                  // current column h_{1..j,j}
    double negh[(GMRES_KMAX + 1) * 2];                  // -hcol (axpy coefficients)
    double delta[GMRES_KMAX];                           // GCR: delta_j = (z_j, z_j)
    double alpha[2];                                    // GCR: alpha of the current step
    double scale;                                       // 1/beta or 1/h_{j+1,j}
    double value;                                       // last reduced norm
    int nhist;
};

// Every BLAS-1 launch below is one wave of resident CTAs; the functions that write per-block
// partial sums RETURN their grid (= number of partial blocks, <= blas_grid_cap()) for the
// finalize_* kernel that follows.
int blas_grid_cap();
// dst = sqrt(sum partials); stores into sc->value, optionally appends to sc->hist, sets sc->scale = 1/value
void launch_finalize_norm(const double* partials, int n, Scalars* sc, int append_hist, cudaStream_t st);
// multi-rhs: partials[block][stride], the first nrhs of each row are right-hand sides (the rest padding)
void launch_finalize_norm_batch(const double* partials, int nblocks, int nrhs, int stride, Scalars* sc, int offset, cudaStream_t st);
template <typename T>
int launch_copy_norm(size_t nreal, const void* src, void* dst, double* partials, cudaStream_t st);
template <typename T>
void launch_scale_by_dev(size_t nreal, void* v, const double* scale, cudaStream_t st);
template <typename T>
int launch_axpy_norm(size_t nreal, double alpha, const void* x, void* y, double* partials, cudaStream_t st); // y = alpha*x (+norm of x)
// partial complex dots <v_i, w>, i = 0..nb-1 (nb <= MDOT_NB): partials[block][2*nb]
template <typename T>
int launch_multi_dot(size_t nreal, int nb, const void* V, size_t vstride_real, const void* w, double* partials,
                      cudaStream_t st);
void launch_finalize_dots(const double* partials, int nblocks, int nb, Scalars* sc, int first, cudaStream_t st);
void launch_finalize_dots_lazy(const double* partials, int nblocks, int nb, Scalars* sc, int first, int j, cudaStream_t st);
void launch_finalize_dots_lazy2(const double* partials, int nblocks, int nb, Scalars* sc, int first, cudaStream_t st);   // CGS2 correction
// w <- (*wscale) w + sum_i coef[i] v_i (complex coef and real wscale on device, nb <= MDOT_NB;
// wscale NULL = 1); optional |w|^2 partials
template <typename T>
int launch_multi_axpy(size_t nreal, int nb, const void* V, size_t vstride_real, const double* coef, void* w,
                       double* partials, cudaStream_t st, const double* wscale = nullptr);
// GCR (Alg. 3)
template <typename T>
int launch_gcr_form(size_t nreal, int nb, const void* Z0, const void* P0, size_t vstride_real, const double* coef,
                     void* z_io, const void* r, void* p_out, int init_p, double* partials, cudaStream_t st);
void launch_gcr_alpha(const double* partials, int nblocks, Scalars* sc, int j, cudaStream_t st);
void launch_gcr_beta(Scalars* sc, int first, int nb, cudaStream_t st);
template <typename T>
int launch_gcr_update(size_t nreal, const double* alpha, const void* p, const void* z, void* x, void* r,
                       double* partials, cudaStream_t st);
void launch_gmres_begin_cycle(Scalars* sc, cudaStream_t st);                 // g = beta e_1 (beta = sc->value)
void launch_gmres_givens(Scalars* sc, int j, cudaStream_t st);               // after the norm of w is in sc->value
void launch_gmres_solve(Scalars* sc, int m, cudaStream_t st);                // y = R^-1 g

}  // namespace ddamg

// ddamg_dslash.cu -- the fused hopping + clover kernels of the Schur complement (eq. 3).
//
//   kernel A   t_o = A_oo^-1 (H_oe x_e)                         EPI_CLOV_HOP      (steps a2-a5)
//   kernel B   y_e = A_ee x_e - H_eo t_o                         EPI_SCHUR         (step a6)
//   kernel B'  r = b_e - (A_ee x_e - H_eo t_o); x_e += w r       EPI_RICHARDSON    (step a7)
//              out = b_e - (A_ee x_e - H_eo t_o)  (+ ||out||^2)  EPI_RESIDUAL      (GMRES line 2)
//              x_o = A_oo^-1 (b_o - H_oe x_e)                    EPI_CLOV_RHS_MINUS_HOP (eq. 2 left)
//              bhat_e = b_e - H_eo t_o                           EPI_RHS_MINUS_HOP (eq. 2 right)
//              y_p = A_pp x_p + H_pq x_q  (one parity of D x)    EPI_FULL          (outer FGMRES)
//              out = b_p - (A_pp x_p + H_pq x_q)  (+ ||out||^2)  EPI_FULL_RESIDUAL
//
// One thread per output site; consecutive threads = consecutive checkerboard indices, so
// every plane access of a warp is one contiguous 512-byte (16-byte vectors) run.
#include "ddamg_dslash_kernel.cuh"

namespace ddamg {

template void launch_dslash_recon<float, 18>(const Geom&, int, bool, int, const void*, const void*, const void*, const void*,
                                             const void*, const void*, void*, double, double, double*, int, double, int, cudaStream_t);
template void launch_dslash_recon<double, 18>(const Geom&, int, bool, int, const void*, const void*, const void*, const void*,
                                              const void*, const void*, void*, double, double, double*, int, double, int, cudaStream_t);

// instantiated in ddamg_dslash12.cu
extern template void launch_dslash_recon<float, 12>(const Geom&, int, bool, int, const void*, const void*, const void*,
                                                    const void*, const void*, const void*, void*, double, double, double*,
                                                    int, double, int, cudaStream_t);
extern template void launch_dslash_recon<double, 12>(const Geom&, int, bool, int, const void*, const void*, const void*,
                                                     const void*, const void*, const void*, void*, double, double, double*,
                                                     int, double, int, cudaStream_t);

// recon = 18: gauge_* point into the full link blocks; recon = 12: into the two-row blocks
template <typename T>
void launch_dslash(const Geom& g, int epi, bool norm, int parity, const void* in, const void* gauge_own,
                   const void* gauge_opp, const void* clov, const void* own, const void* rhs, void* out,
                   double omega, double c0, double* partials, int units, double batch_l2_bytes, int recon, int apbc,
                   cudaStream_t st)
{
    if (recon == 12)
        launch_dslash_recon<T, 12>(g, epi, norm, parity, in, gauge_own, gauge_opp, clov, own, rhs, out, omega, c0, partials,
                                   units, batch_l2_bytes, apbc, st);
    else
        launch_dslash_recon<T, 18>(g, epi, norm, parity, in, gauge_own, gauge_opp, clov, own, rhs, out, omega, c0, partials,
                                   units, batch_l2_bytes, apbc, st);
}
template void launch_dslash<float>(const Geom&, int, bool, int, const void*, const void*, const void*, const void*,
                                   const void*, const void*, void*, double, double, double*, int, double, int, int, cudaStream_t);
template void launch_dslash<double>(const Geom&, int, bool, int, const void*, const void*, const void*, const void*,
                                    const void*, const void*, void*, double, double, double*, int, double, int, int, cudaStream_t);

// out = Cl in on one parity (right factor of eq. 2: t_o = A_oo^-1 b_o); units as in launch_dslash
template <typename T, bool BATCH>
__global__ void __launch_bounds__(DSLASH_THREADS)
clover_apply_kernel(Geom g, int units, const T* __restrict__ clov, const T* __restrict__ in, T* __restrict__ out)
{
    using S = typename ValueOf<T, BATCH>::type;
    const int tid = blockIdx.x * DSLASH_THREADS + threadIdx.x;
    const int cb = tid / units;
    if (cb >= g.Vh) return;
    S v[24], res[24];
    load_spinor<T, true>(in, g.Vh * units, tid, v);
    clover_site_mul<T>(clov, g.Vh, cb, v, res);
    store_spinor<T>(out, g.Vh * units, tid, res);
}

template <typename T>
void launch_clover_apply(const Geom& g, const void* clov, const void* in, void* out, int units, cudaStream_t st)
{
    if (units > 0)
        clover_apply_kernel<T, true><<<dslash_grid(g, units), DSLASH_THREADS, 0, st>>>(g, units, (const T*)clov, (const T*)in, (T*)out);
    else
        clover_apply_kernel<T, false><<<dslash_grid(g, 1), DSLASH_THREADS, 0, st>>>(g, 1, (const T*)clov, (const T*)in, (T*)out);
}
template void launch_clover_apply<float>(const Geom&, const void*, const void*, void*, int, cudaStream_t);
template void launch_clover_apply<double>(const Geom&, const void*, const void*, void*, int, cudaStream_t);

int dslash_grid(const Geom& g, int units)
{
    return (int)(((long long)g.Vh * units + DSLASH_THREADS - 1) / DSLASH_THREADS);
}

}  // namespace ddamg

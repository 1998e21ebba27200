// ddamg_dslash12.cu -- the fused hopping + clover kernels for two-row (12-real) link storage
// (option "gauge_recon" = 12): same kernels as ddamg_dslash.cu, the third row of every link is
// rebuilt in registers as conj(row0 x row1).  A separate translation unit so that the two
// instantiation sets compile in parallel.
#include "ddamg_dslash_kernel.cuh"

namespace ddamg {

template void launch_dslash_recon<float, 12>(const Geom&, int, bool, int, const void*, const void*, const void*, const void*,
                                             const void*, const void*, void*, double, double, double*, int, double, int, cudaStream_t);
template void launch_dslash_recon<double, 12>(const Geom&, int, bool, int, const void*, const void*, const void*, const void*,
                                              const void*, const void*, void*, double, double, double*, int, double, int, cudaStream_t);

}  // namespace ddamg

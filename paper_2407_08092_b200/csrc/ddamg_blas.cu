// ddamg_blas.cu -- device-wide reductions and the BLAS-1 / small dense part of GMRES
// (steps a8, a9; Alg. 2 lines 2, 7, 8, 10).
//
// BLAS-1 kernels see a half-lattice spinor as a flat array of 16-byte vectors; in the native
// layout the two (fp64: one) complex numbers of a vector are (re, im) pairs, so complex inner
// products can be formed without knowing the site structure.
//
// All of them are HBM streams: every kernel is ONE wave of resident CTAs
// (grid = SMs x occupancy, grid-stride loop), every thread first issues ALL the 16-byte loads of
// an iteration (NB + 1 vectors; small NB: several elements per iteration) and only then computes,
// so that ~100 KB per SM are in flight.  fp32 data: the products of one 16-byte vector (4 reals)
// are formed with fp32 FMAs and folded into fp64 accumulators once per vector -- the fp64 pipe
// and the F2F conversion pipe see 2 operations per (vector, basis vector) instead of 12; axpy
// forms are evaluated in fp32 (the result is stored in fp32 anyway).  fp64 data: fp64 throughout.
// Each block writes its fp64 partials, a single-block kernel finishes them in a fixed order
// (deterministic), and every scalar (norms, Hessenberg column, Givens rotations, the
// least-squares solution) stays on the device: no host synchronisation inside a cycle.
#include "ddamg_internal.h"

namespace ddamg {

static int sm_count()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            cudaGetLastError();
            n = 148;
        }
    }
    return n;
}

// upper bound of every BLAS-1 grid (sizes the partial-sum scratch): 2048 resident threads per SM
int blas_grid_cap() { return sm_count() * (2048 / BLAS_THREADS); }

// one wave: as many CTAs as are resident at once, at most one per BLAS_THREADS * unroll vectors
template <typename K>
static int wave_grid(K kernel, size_t nvec, int unroll)
{
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, BLAS_THREADS, 0) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    const size_t per_cta = (size_t)BLAS_THREADS * unroll;
    const size_t need = (nvec + per_cta - 1) / per_cta;
    const size_t cap = (size_t)sm_count() * per_sm;
    return (int)(need < cap ? (need ? need : 1) : cap);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sums NV values per thread across the block; result valid in thread 0 (written to out[0..NV-1])
template <int NV>
__device__ __forceinline__ void block_sum_n(double (&v)[NV], double* out)
{
    __shared__ double sh[BLAS_THREADS / 32][NV];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const double s = warp_sum(v[i]);
        if (lane == 0) sh[w][i] = s;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double s = 0;
        for (int k = 0; k < BLAS_THREADS / 32; ++k) s += sh[k][threadIdx.x];
        out[threadIdx.x] = s;
    }
}

// ---- per-vector arithmetic in the data precision (fp32 vectors: 4 reals = 2 complex numbers)
__device__ __forceinline__ float4 ld_once(const float4* p) { return __ldcs(p); }
__device__ __forceinline__ double2 ld_once(const double2* p) { return __ldcs(p); }

// conj(v) . w over the complex numbers of one vector, added to (ar, ai)
__device__ __forceinline__ void cdot_add(const float4& v, const float4& w, double& ar, double& ai)
{
    float pr = v.x * w.x;
    pr = fmaf(v.y, w.y, pr); pr = fmaf(v.z, w.z, pr); pr = fmaf(v.w, w.w, pr);
    float pi = v.x * w.y;
    pi = fmaf(-v.y, w.x, pi); pi = fmaf(v.z, w.w, pi); pi = fmaf(-v.w, w.z, pi);
    ar += (double)pr;
    ai += (double)pi;
}
__device__ __forceinline__ void cdot_add(const double2& v, const double2& w, double& ar, double& ai)
{
    ar = fma(v.x, w.x, ar); ar = fma(v.y, w.y, ar);
    ai = fma(v.x, w.y, ai); ai = fma(-v.y, w.x, ai);
}
// |v|^2 added to a
__device__ __forceinline__ void norm_add(const float4& v, double& a)
{
    float p = v.x * v.x;
    p = fmaf(v.y, v.y, p); p = fmaf(v.z, v.z, p); p = fmaf(v.w, v.w, p);
    a += (double)p;
}
__device__ __forceinline__ void norm_add(const double2& v, double& a) { a = fma(v.x, v.x, a); a = fma(v.y, v.y, a); }
// w += (cr + i ci) v, complex number by complex number
__device__ __forceinline__ void caxpy(float cr, float ci, const float4& v, float4& w)
{
    w.x = fmaf(cr, v.x, w.x); w.x = fmaf(-ci, v.y, w.x);
    w.y = fmaf(cr, v.y, w.y); w.y = fmaf(ci, v.x, w.y);
    w.z = fmaf(cr, v.z, w.z); w.z = fmaf(-ci, v.w, w.z);
    w.w = fmaf(cr, v.w, w.w); w.w = fmaf(ci, v.z, w.w);
}
__device__ __forceinline__ void caxpy(double cr, double ci, const double2& v, double2& w)
{
    w.x = fma(cr, v.x, w.x); w.x = fma(-ci, v.y, w.x);
    w.y = fma(cr, v.y, w.y); w.y = fma(ci, v.x, w.y);
}
__device__ __forceinline__ void vscale(float s, float4& w) { w.x *= s; w.y *= s; w.z *= s; w.w *= s; }
__device__ __forceinline__ void vscale(double s, double2& w) { w.x *= s; w.y *= s; }

// elements per thread and iteration: enough independent 16-byte loads in flight for every NB
__host__ __device__ constexpr int unroll_for(int nloads) { return nloads >= 7 ? 1 : nloads >= 4 ? 2 : nloads >= 2 ? 4 : 8; }

// ------------------------------------------------------------------ norm finish
__global__ void finalize_norm_kernel(const double* __restrict__ partials, int n, Scalars* sc, int append)
{
    double v[1] = { 0.0 };
    for (int i = threadIdx.x; i < n; i += BLAS_THREADS) v[0] += partials[i];
    __shared__ double tot[1];
    block_sum_n<1>(v, tot);
    __syncthreads();
    if (threadIdx.x == 0) {
        const double nrm = sqrt(tot[0]);
        sc->value = nrm;
        sc->scale = nrm > 0.0 ? 1.0 / nrm : 0.0;
        if (append && sc->nhist < HIST_MAX) sc->hist[sc->nhist++] = nrm;
    }
}
void launch_finalize_norm(const double* partials, int n, Scalars* sc, int append_hist, cudaStream_t st)
{
    finalize_norm_kernel<<<1, BLAS_THREADS, 0, st>>>(partials, n, sc, append_hist);
}

// multi-rhs: partials[block][stride]; block r < nrhs of this kernel finishes rhs r into hist[offset + r]
__global__ void finalize_norm_batch_kernel(const double* __restrict__ partials, int nblocks, int nrhs, int stride, Scalars* sc,
                                           int offset)
{
    const int r = blockIdx.x;
    double v[1] = { 0.0 };
    for (int i = threadIdx.x; i < nblocks; i += BLAS_THREADS) v[0] += partials[(size_t)i * stride + r];
    __shared__ double tot[1];
    block_sum_n<1>(v, tot);
    __syncthreads();
    if (threadIdx.x == 0 && offset + r < HIST_MAX) sc->hist[offset + r] = sqrt(tot[0]);
    if (threadIdx.x == 0 && r == nrhs - 1) sc->nhist = (offset + nrhs < HIST_MAX) ? offset + nrhs : HIST_MAX;
}
void launch_finalize_norm_batch(const double* partials, int nblocks, int nrhs, int stride, Scalars* sc, int offset, cudaStream_t st)
{
    finalize_norm_batch_kernel<<<nrhs, BLAS_THREADS, 0, st>>>(partials, nblocks, nrhs, stride, sc, offset);
}

// ------------------------------------------------------------------ y = alpha * x, partial |x|^2
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
axpy_norm_kernel(size_t nvec, T alpha, const typename VecOf<T>::type* x,
                 typename VecOf<T>::type* y, double* __restrict__ partials)   // x may alias y
{
    using V = typename VecOf<T>::type;
    constexpr int U = 8;
    double acc[1] = { 0.0 };
    const size_t step = (size_t)gridDim.x * BLAS_THREADS * U;
    for (size_t base = (size_t)blockIdx.x * BLAS_THREADS * U + threadIdx.x; base < nvec; base += step) {
        V v[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (base + (size_t)u * BLAS_THREADS < nvec) v[u] = x[base + (size_t)u * BLAS_THREADS];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (base + (size_t)u * BLAS_THREADS < nvec) {
                norm_add(v[u], acc[0]);
                vscale(alpha, v[u]);
                y[base + (size_t)u * BLAS_THREADS] = v[u];
            }
    }
    if (partials) block_sum_n<1>(acc, partials + blockIdx.x);
}
template <typename T>
int launch_axpy_norm(size_t nreal, double alpha, const void* x, void* y, double* partials, cudaStream_t st)
{
    using V = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N;
    const int grid = wave_grid(axpy_norm_kernel<T>, nvec, 8);
    axpy_norm_kernel<T><<<grid, BLAS_THREADS, 0, st>>>(nvec, (T)alpha, (const V*)x, (V*)y, partials);
    return grid;
}
template <typename T>
int launch_copy_norm(size_t nreal, const void* src, void* dst, double* partials, cudaStream_t st)
{
    return launch_axpy_norm<T>(nreal, 1.0, src, dst, partials, st);
}
template int launch_axpy_norm<float>(size_t, double, const void*, void*, double*, cudaStream_t);
template int launch_axpy_norm<double>(size_t, double, const void*, void*, double*, cudaStream_t);
template int launch_copy_norm<float>(size_t, const void*, void*, double*, cudaStream_t);
template int launch_copy_norm<double>(size_t, const void*, void*, double*, cudaStream_t);

// ------------------------------------------------------------------ v *= *scale (device scalar)
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
scale_kernel(size_t nvec, typename VecOf<T>::type* __restrict__ v, const double* __restrict__ scale)
{
    using V = typename VecOf<T>::type;
    constexpr int U = 8;
    const T s = (T)(*scale);
    const size_t step = (size_t)gridDim.x * BLAS_THREADS * U;
    for (size_t base = (size_t)blockIdx.x * BLAS_THREADS * U + threadIdx.x; base < nvec; base += step) {
        V r[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (base + (size_t)u * BLAS_THREADS < nvec) r[u] = v[base + (size_t)u * BLAS_THREADS];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (base + (size_t)u * BLAS_THREADS < nvec) {
                vscale(s, r[u]);
                v[base + (size_t)u * BLAS_THREADS] = r[u];
            }
    }
}
template <typename T>
void launch_scale_by_dev(size_t nreal, void* v, const double* scale, cudaStream_t st)
{
    using V = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N;
    scale_kernel<T><<<wave_grid(scale_kernel<T>, nvec, 8), BLAS_THREADS, 0, st>>>(nvec, (V*)v, scale);
}
template void launch_scale_by_dev<float>(size_t, void*, const double*, cudaStream_t);
template void launch_scale_by_dev<double>(size_t, void*, const double*, cudaStream_t);

// ------------------------------------------------------------------ fused multi-dot  <v_i, w>
template <typename T, int NB>
__global__ void __launch_bounds__(BLAS_THREADS)
multi_dot_kernel(size_t nvec, const typename VecOf<T>::type* __restrict__ V0, size_t vstride,
                 const typename VecOf<T>::type* __restrict__ w, double* __restrict__ partials)
{
    using V = typename VecOf<T>::type;
    constexpr int U = unroll_for(NB + 1);
    double acc[2 * NB];
#pragma unroll
    for (int i = 0; i < 2 * NB; ++i) acc[i] = 0.0;
    const size_t step = (size_t)gridDim.x * BLAS_THREADS * U;
    for (size_t base = (size_t)blockIdx.x * BLAS_THREADS * U + threadIdx.x; base < nvec; base += step) {
        V wv[U], vv[U][NB];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) {
                wv[u] = ld_once(w + i);
#pragma unroll
                for (int b = 0; b < NB; ++b) vv[u][b] = ld_once(V0 + (size_t)b * vstride + i);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (base + (size_t)u * BLAS_THREADS < nvec) {
#pragma unroll
                for (int b = 0; b < NB; ++b) cdot_add(vv[u][b], wv[u], acc[2 * b], acc[2 * b + 1]);    // conj(v) * w
            }
        }
    }
    block_sum_n<2 * NB>(acc, partials + (size_t)blockIdx.x * 2 * NB);
}
template <typename T>
int launch_multi_dot(size_t nreal, int nb, const void* V, size_t vstride_real, const void* w, double* partials,
                     cudaStream_t st)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N, vs = vstride_real / VecOf<T>::N;
    int grid = 0;
#define MD(NB) case NB: grid = wave_grid(multi_dot_kernel<T, NB>, nvec, unroll_for(NB + 1)); \
        multi_dot_kernel<T, NB><<<grid, BLAS_THREADS, 0, st>>>(nvec, (const VT*)V, vs, (const VT*)w, partials); break;
    switch (nb) { MD(1) MD(2) MD(3) MD(4) MD(5) MD(6) MD(7) MD(8) MD(9) MD(10) MD(11) MD(12) }
    static_assert(MDOT_NB == 12, "one case per NB");
#undef MD
    return grid;
}
template int launch_multi_dot<float>(size_t, int, const void*, size_t, const void*, double*, cudaStream_t);
template int launch_multi_dot<double>(size_t, int, const void*, size_t, const void*, double*, cudaStream_t);

// hcol[first .. first+nb-1] = sum over blocks; negh = -hcol.  One warp per real component,
// lanes stride over the blocks, fixed shuffle tree: deterministic.
__global__ void finalize_dots_kernel(const double* __restrict__ partials, int nblocks, int nb, Scalars* sc, int first)
{
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (c < 2 * nb) {
        double s = 0;
        for (int b = lane; b < nblocks; b += 32) s += partials[(size_t)b * 2 * nb + c];
        s = warp_sum(s);
        if (lane == 0) {
            sc->hcol[2 * first + c] = s;
            sc->negh[2 * first + c] = -s;
        }
    }
}
void launch_finalize_dots(const double* partials, int nblocks, int nb, Scalars* sc, int first, cudaStream_t st)
{
    finalize_dots_kernel<<<1, 32 * 2 * MDOT_NB, 0, st>>>(partials, nblocks, nb, sc, first);
}

// GMRES with a lazily normalised basis (v_i = vs[i] * stored_i, DESIGN.md section 7 "GMRES"):
// the raw sums are <stored_i, D_S stored_j>, so  h_ij = vs[i] vs[j] sum  and the coefficient of
// stored_i in  w~ = vs[j] D_S stored_j - sum_i h_ij vs[i] stored_i  is  negh_i = -h_ij vs[i].
__global__ void finalize_dots_lazy_kernel(const double* __restrict__ partials, int nblocks, int nb, Scalars* sc,
                                          int first, int j)
{
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (c < 2 * nb) {
        double s = 0;
        for (int b = lane; b < nblocks; b += 32) s += partials[(size_t)b * 2 * nb + c];
        s = warp_sum(s);
        if (lane == 0) {
            const double si = sc->vs[first + (c >> 1)];
            const double h = s * si * sc->vs[j];
            sc->hcol[2 * first + c] = h;
            sc->negh[2 * first + c] = -h * si;
        }
    }
}
void launch_finalize_dots_lazy(const double* partials, int nblocks, int nb, Scalars* sc, int first, int j, cudaStream_t st)
{
    finalize_dots_lazy_kernel<<<1, 32 * 2 * MDOT_NB, 0, st>>>(partials, nblocks, nb, sc, first, j);
}

// Second Gram-Schmidt pass (CGS2): the raw sums are <stored_i, w> with w already orthogonalised once and in true
// units, so the correction is  h'_i = vs[i] sum;  h_ij += h'_i;  coefficient of stored_i:  -h'_i vs[i].
__global__ void finalize_dots_lazy2_kernel(const double* __restrict__ partials, int nblocks, int nb, Scalars* sc, int first)
{
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (c < 2 * nb) {
        double s = 0;
        for (int b = lane; b < nblocks; b += 32) s += partials[(size_t)b * 2 * nb + c];
        s = warp_sum(s);
        if (lane == 0) {
            const double si = sc->vs[first + (c >> 1)];
            const double h = s * si;
            sc->hcol[2 * first + c] += h;
            sc->negh[2 * first + c] = -h * si;
        }
    }
}
void launch_finalize_dots_lazy2(const double* partials, int nblocks, int nb, Scalars* sc, int first, cudaStream_t st)
{
    finalize_dots_lazy2_kernel<<<1, 32 * 2 * MDOT_NB, 0, st>>>(partials, nblocks, nb, sc, first);
}

// ------------------------------------------------------------------ w <- ws w + sum_i coef_i v_i  (+ |w|^2)
template <typename T, int NB>
__global__ void __launch_bounds__(BLAS_THREADS)
multi_axpy_kernel(size_t nvec, const typename VecOf<T>::type* __restrict__ V0, size_t vstride,
                  const double* __restrict__ coef, typename VecOf<T>::type* __restrict__ w,
                  double* __restrict__ partials, const double* __restrict__ wscale)
{
    using V = typename VecOf<T>::type;
    constexpr int U = unroll_for(NB + 1);
    T cr[NB], ci[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) { cr[b] = (T)coef[2 * b]; ci[b] = (T)coef[2 * b + 1]; }
    const T ws = wscale ? (T)(*wscale) : (T)1;
    double acc[1] = { 0.0 };
    const size_t step = (size_t)gridDim.x * BLAS_THREADS * U;
    for (size_t base = (size_t)blockIdx.x * BLAS_THREADS * U + threadIdx.x; base < nvec; base += step) {
        V wv[U], vv[U][NB];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) {
                wv[u] = w[i];
#pragma unroll
                for (int b = 0; b < NB; ++b) vv[u][b] = ld_once(V0 + (size_t)b * vstride + i);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) {
                if (wscale) vscale(ws, wv[u]);
#pragma unroll
                for (int b = 0; b < NB; ++b) caxpy(cr[b], ci[b], vv[u][b], wv[u]);
                norm_add(wv[u], acc[0]);
                w[i] = wv[u];
            }
        }
    }
    if (partials) block_sum_n<1>(acc, partials + blockIdx.x);
}
template <typename T>
int launch_multi_axpy(size_t nreal, int nb, const void* V, size_t vstride_real, const double* coef, void* w,
                      double* partials, cudaStream_t st, const double* wscale)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N, vs = vstride_real / VecOf<T>::N;
    int grid = 0;
#define MA(NB) case NB: grid = wave_grid(multi_axpy_kernel<T, NB>, nvec, unroll_for(NB + 1)); \
        multi_axpy_kernel<T, NB><<<grid, BLAS_THREADS, 0, st>>>(nvec, (const VT*)V, vs, coef, (VT*)w, partials, wscale); break;
    switch (nb) { MA(1) MA(2) MA(3) MA(4) MA(5) MA(6) MA(7) MA(8) MA(9) MA(10) MA(11) MA(12) }
#undef MA
    return grid;
}
template int launch_multi_axpy<float>(size_t, int, const void*, size_t, const double*, void*, double*, cudaStream_t, const double*);
template int launch_multi_axpy<double>(size_t, int, const void*, size_t, const double*, void*, double*, cudaStream_t, const double*);

// ------------------------------------------------------------------ GCR (Alg. 3)
// lines 11-14 in one pass:  z = w + sum_j beta_j z_j  (in place on w),  p = r + sum_j beta_j p_j,
// plus the partial sums the next step needs: |z|^2 (line 6) and <z, r> (line 7).
// NB = 0 is the start of a cycle: p_1 = r, z_1 = D p_1 untouched, same partial sums.
template <typename T, int NB>
__global__ void __launch_bounds__(BLAS_THREADS)
gcr_form_kernel(size_t nvec, const typename VecOf<T>::type* __restrict__ Z0,
                const typename VecOf<T>::type* __restrict__ P0, size_t vstride,
                const double* __restrict__ coef, typename VecOf<T>::type* __restrict__ z_io,
                const typename VecOf<T>::type* __restrict__ r, typename VecOf<T>::type* __restrict__ p_out,
                int init_p, double* __restrict__ partials)
{
    using V = typename VecOf<T>::type;
    constexpr int NBA = NB > 0 ? NB : 1;
    constexpr int U = unroll_for(2 * NB + 3);
    T cr[NBA], ci[NBA];
#pragma unroll
    for (int b = 0; b < NB; ++b) { cr[b] = (T)coef[2 * b]; ci[b] = (T)coef[2 * b + 1]; }
    double acc[3] = { 0.0, 0.0, 0.0 };
    const size_t step = (size_t)gridDim.x * BLAS_THREADS * U;
    for (size_t base = (size_t)blockIdx.x * BLAS_THREADS * U + threadIdx.x; base < nvec; base += step) {
        V zv[U], rv[U], pv[U], zb[U][NBA], pb[U][NBA];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) {
                zv[u] = z_io[i];
                rv[u] = r[i];
                if (!init_p) pv[u] = p_out[i];
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    zb[u][b] = ld_once(Z0 + (size_t)b * vstride + i);
                    pb[u][b] = ld_once(P0 + (size_t)b * vstride + i);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) {
                if (init_p) pv[u] = rv[u];
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    caxpy(cr[b], ci[b], zb[u][b], zv[u]);
                    caxpy(cr[b], ci[b], pb[u][b], pv[u]);
                }
                if (NB > 0) z_io[i] = zv[u];
                p_out[i] = pv[u];
                if (partials) {
                    norm_add(zv[u], acc[0]);
                    cdot_add(zv[u], rv[u], acc[1], acc[2]);          // conj(z) * r
                }
            }
        }
    }
    if (partials) block_sum_n<3>(acc, partials + (size_t)blockIdx.x * 3);
}
template <typename T>
int launch_gcr_form(size_t nreal, int nb, const void* Z0, const void* P0, size_t vstride_real, const double* coef,
                    void* z_io, const void* r, void* p_out, int init_p, double* partials, cudaStream_t st)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N, vs = vstride_real / VecOf<T>::N;
    int grid = 0;
#define GF(NB) case NB: grid = wave_grid(gcr_form_kernel<T, NB>, nvec, unroll_for(2 * NB + 3)); \
        gcr_form_kernel<T, NB><<<grid, BLAS_THREADS, 0, st>>>(nvec, (const VT*)Z0, (const VT*)P0, vs, coef, (VT*)z_io, (const VT*)r, (VT*)p_out, init_p, partials); break;
    switch (nb) { GF(0) GF(1) GF(2) GF(3) GF(4) GF(5) GF(6) GF(7) GF(8) GF(9) GF(10) GF(11) GF(12) }
#undef GF
    return grid;
}
template int launch_gcr_form<float>(size_t, int, const void*, const void*, size_t, const double*, void*, const void*, void*, int, double*, cudaStream_t);
template int launch_gcr_form<double>(size_t, int, const void*, const void*, size_t, const double*, void*, const void*, void*, int, double*, cudaStream_t);

// lines 6-7: delta_j = sum |z|^2, alpha = <z, r> / delta_j  (partials[block][3] from gcr_form)
__global__ void gcr_alpha_kernel(const double* __restrict__ partials, int nblocks, Scalars* sc, int j)
{
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;       // 3 warps, one per component
    __shared__ double tot[3];
    double s = 0;
    for (int b = lane; b < nblocks; b += 32) s += partials[(size_t)b * 3 + c];
    s = warp_sum(s);
    if (lane == 0) tot[c] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        const double d = tot[0];
        sc->delta[j] = d;
        sc->alpha[0] = d > 0.0 ? tot[1] / d : 0.0;
        sc->alpha[1] = d > 0.0 ? tot[2] / d : 0.0;
    }
}
void launch_gcr_alpha(const double* partials, int nblocks, Scalars* sc, int j, cudaStream_t st)
{
    gcr_alpha_kernel<<<1, 96, 0, st>>>(partials, nblocks, sc, j);
}

// line 12: beta_i = -<z_i, w> / delta_i for i = first..first+nb-1 (hcol holds the dots) -> sc->negh
__global__ void gcr_beta_kernel(Scalars* sc, int first, int nb)
{
    const int i = first + threadIdx.x;
    if ((int)threadIdx.x < nb) {
        const double d = sc->delta[i];
        sc->negh[2 * i] = d > 0.0 ? -sc->hcol[2 * i] / d : 0.0;
        sc->negh[2 * i + 1] = d > 0.0 ? -sc->hcol[2 * i + 1] / d : 0.0;
    }
}
void launch_gcr_beta(Scalars* sc, int first, int nb, cudaStream_t st) { gcr_beta_kernel<<<1, 32, 0, st>>>(sc, first, nb); }

// lines 8-9:  x += alpha p,  r -= alpha z,  partial |r|^2
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
gcr_update_kernel(size_t nvec, const double* __restrict__ alpha, const typename VecOf<T>::type* __restrict__ p,
                  const typename VecOf<T>::type* __restrict__ z, typename VecOf<T>::type* __restrict__ x,
                  typename VecOf<T>::type* __restrict__ r, double* __restrict__ partials)
{
    using V = typename VecOf<T>::type;
    constexpr int U = 2;
    const T ar = (T)alpha[0], ai = (T)alpha[1];
    double acc[1] = { 0.0 };
    const size_t step = (size_t)gridDim.x * BLAS_THREADS * U;
    for (size_t base = (size_t)blockIdx.x * BLAS_THREADS * U + threadIdx.x; base < nvec; base += step) {
        V xv[U], rv[U], pv[U], zv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) { xv[u] = x[i]; rv[u] = r[i]; pv[u] = ld_once(p + i); zv[u] = ld_once(z + i); }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const size_t i = base + (size_t)u * BLAS_THREADS;
            if (i < nvec) {
                caxpy(ar, ai, pv[u], xv[u]);
                caxpy(-ar, -ai, zv[u], rv[u]);
                norm_add(rv[u], acc[0]);
                x[i] = xv[u];
                r[i] = rv[u];
            }
        }
    }
    block_sum_n<1>(acc, partials + blockIdx.x);
}
template <typename T>
int launch_gcr_update(size_t nreal, const double* alpha, const void* p, const void* z, void* x, void* r,
                      double* partials, cudaStream_t st)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N;
    const int grid = wave_grid(gcr_update_kernel<T>, nvec, 2);
    gcr_update_kernel<T><<<grid, BLAS_THREADS, 0, st>>>(nvec, alpha, (const VT*)p, (const VT*)z, (VT*)x, (VT*)r, partials);
    return grid;
}
template int launch_gcr_update<float>(size_t, const double*, const void*, const void*, void*, void*, double*, cudaStream_t);
template int launch_gcr_update<double>(size_t, const double*, const void*, const void*, void*, void*, double*, cudaStream_t);

// ------------------------------------------------------------------ small dense part (1 thread)
__global__ void gmres_begin_cycle_kernel(Scalars* sc)
{
    for (int i = 0; i < 2 * (GMRES_KMAX + 1); ++i) sc->gvec[i] = 0.0;
    sc->gvec[0] = sc->value;          // beta e_1
    sc->vs[0] = sc->scale;            // v_1 = r / beta, kept as (1 / beta, r)
}
void launch_gmres_begin_cycle(Scalars* sc, cudaStream_t st) { gmres_begin_cycle_kernel<<<1, 1, 0, st>>>(sc); }

// column j: hcol[0..j] hold h_{i,j}; sc->value holds h_{j+1,j} = ||w||.  Applies the previous
// rotations, forms rotation j, updates g and appends |g_{j+1}| to the history (Alg. 2 line 10
// done incrementally; reading R9).
__global__ void gmres_givens_kernel(Scalars* sc, int j)
{
    double* H = sc->H + (size_t)j * (GMRES_KMAX + 1) * 2;      // column j
    for (int i = 0; i <= j; ++i) { H[2 * i] = sc->hcol[2 * i]; H[2 * i + 1] = sc->hcol[2 * i + 1]; }
    H[2 * (j + 1)] = sc->value;
    H[2 * (j + 1) + 1] = 0.0;
    sc->vs[j + 1] = sc->scale;        // v_{j+1} = w / h_{j+1,j}, kept as (1 / h_{j+1,j}, w)
    for (int i = 0; i < j; ++i) {
        const double cr = sc->cs[2 * i], ci = sc->cs[2 * i + 1], sr = sc->sn[2 * i], si = sc->sn[2 * i + 1];
        const double ar = H[2 * i], ai = H[2 * i + 1], br = H[2 * i + 2], bi = H[2 * i + 3];
        // t = c a + s b ;  b' = -conj(s) a + conj(c) b
        const double tr = cr * ar - ci * ai + sr * br - si * bi;
        const double ti = cr * ai + ci * ar + sr * bi + si * br;
        const double ur = -(sr * ar + si * ai) + (cr * br + ci * bi);
        const double ui = -(sr * ai - si * ar) + (cr * bi - ci * br);
        H[2 * i] = tr; H[2 * i + 1] = ti; H[2 * i + 2] = ur; H[2 * i + 3] = ui;
    }
    const double ar = H[2 * j], ai = H[2 * j + 1], c = H[2 * j + 2];
    const double d = sqrt(ar * ar + ai * ai + c * c);
    double cr = 1, ci = 0, sr = 0, si = 0;
    if (d > 0) { cr = ar / d; ci = -ai / d; sr = c / d; si = 0; }       // cs = conj(a)/d, sn = conj(c)/d
    sc->cs[2 * j] = cr; sc->cs[2 * j + 1] = ci; sc->sn[2 * j] = sr; sc->sn[2 * j + 1] = si;
    H[2 * j] = d; H[2 * j + 1] = 0.0; H[2 * j + 2] = 0.0; H[2 * j + 3] = 0.0;
    const double gr = sc->gvec[2 * j], gi = sc->gvec[2 * j + 1];
    // g_{j+1} = -conj(s) g_j ; g_j = c g_j
    sc->gvec[2 * j + 2] = -(sr * gr + si * gi);
    sc->gvec[2 * j + 3] = -(sr * gi - si * gr);
    sc->gvec[2 * j] = cr * gr - ci * gi;
    sc->gvec[2 * j + 1] = cr * gi + ci * gr;
    const double est = hypot(sc->gvec[2 * j + 2], sc->gvec[2 * j + 3]);
    if (sc->nhist < HIST_MAX) sc->hist[sc->nhist++] = est;
    sc->scale = sc->value > 0.0 ? 1.0 / sc->value : 0.0;                 // for v_{j+1} = w / h_{j+1,j}
}
void launch_gmres_givens(Scalars* sc, int j, cudaStream_t st) { gmres_givens_kernel<<<1, 1, 0, st>>>(sc, j); }

// back-substitution R y = g (R = rotated H, upper triangular m x m)
__global__ void gmres_solve_kernel(Scalars* sc, int m)
{
    for (int i = m - 1; i >= 0; --i) {
        double sr = sc->gvec[2 * i], si = sc->gvec[2 * i + 1];
        for (int c = i + 1; c < m; ++c) {
            const double* h = sc->H + ((size_t)c * (GMRES_KMAX + 1) + i) * 2;
            sr -= h[0] * sc->y[2 * c] - h[1] * sc->y[2 * c + 1];
            si -= h[0] * sc->y[2 * c + 1] + h[1] * sc->y[2 * c];
        }
        const double* d = sc->H + ((size_t)i * (GMRES_KMAX + 1) + i) * 2;
        const double den = d[0] * d[0] + d[1] * d[1];
        sc->y[2 * i] = den > 0 ? (sr * d[0] + si * d[1]) / den : 0.0;
        sc->y[2 * i + 1] = den > 0 ? (si * d[0] - sr * d[1]) / den : 0.0;
        sc->ys[2 * i] = sc->y[2 * i] * sc->vs[i];            // x += sum_i y_i vs[i] stored_i
        sc->ys[2 * i + 1] = sc->y[2 * i + 1] * sc->vs[i];
    }
}
void launch_gmres_solve(Scalars* sc, int m, cudaStream_t st) { gmres_solve_kernel<<<1, 1, 0, st>>>(sc, m); }

}  // namespace ddamg

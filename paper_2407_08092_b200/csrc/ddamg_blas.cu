// ddamg_blas.cu -- device-wide reductions and the BLAS-1 / small dense part of GMRES
// (steps a8, a9; Alg. 2 lines 2, 7, 8, 10).
//
// BLAS-1 kernels see a half-lattice spinor as a flat array of 16-byte vectors; in the native
// layout the two (fp64: one) complex numbers of a vector are (re, im) pairs, so complex inner
// products can be formed without knowing the site structure.  All partial sums are fp64;
// each block writes its partials, a single-block kernel finishes them in a fixed order
// (deterministic), and every scalar (norms, Hessenberg column, Givens rotations, the
// least-squares solution) stays on the device: no host synchronisation inside a cycle.
#include "ddamg_internal.h"

namespace ddamg {

int blas_grid(size_t nvec)
{
    size_t b = (nvec + BLAS_THREADS - 1) / BLAS_THREADS;
    const size_t cap = 148 * 8;
    return (int)(b < cap ? (b ? b : 1) : cap);
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

__device__ __forceinline__ void cvt(const float4& v, double (&r)[4]) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void cvt(const double2& v, double (&r)[2]) { r[0] = v.x; r[1] = v.y; }

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

// multi-rhs: partials[block][nrhs]; block r of this kernel finishes rhs r into hist[offset + r]
__global__ void finalize_norm_batch_kernel(const double* __restrict__ partials, int nblocks, int nrhs, Scalars* sc,
                                           int offset)
{
    const int r = blockIdx.x;
    double v[1] = { 0.0 };
    for (int i = threadIdx.x; i < nblocks; i += BLAS_THREADS) v[0] += partials[(size_t)i * nrhs + r];
    __shared__ double tot[1];
    block_sum_n<1>(v, tot);
    __syncthreads();
    if (threadIdx.x == 0 && offset + r < HIST_MAX) sc->hist[offset + r] = sqrt(tot[0]);
    if (threadIdx.x == 0 && r == nrhs - 1) sc->nhist = (offset + nrhs < HIST_MAX) ? offset + nrhs : HIST_MAX;
}
void launch_finalize_norm_batch(const double* partials, int nblocks, int nrhs, Scalars* sc, int offset, cudaStream_t st)
{
    finalize_norm_batch_kernel<<<nrhs, BLAS_THREADS, 0, st>>>(partials, nblocks, nrhs, sc, offset);
}

// ------------------------------------------------------------------ y = alpha * x, partial |x|^2
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
axpy_norm_kernel(size_t nvec, T alpha, const typename VecOf<T>::type* x,
                 typename VecOf<T>::type* y, double* __restrict__ partials)   // x may alias y
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    double acc[1] = { 0.0 };
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        const V v = x[i];
        T r[N];
        unpack(v, r);
#pragma unroll
        for (int k = 0; k < N; ++k) { acc[0] += (double)r[k] * (double)r[k]; r[k] *= alpha; }
        y[i] = pack(r);
    }
    if (partials) block_sum_n<1>(acc, partials + blockIdx.x);
}
template <typename T>
void launch_axpy_norm(size_t nreal, double alpha, const void* x, void* y, double* partials, cudaStream_t st)
{
    using V = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N;
    axpy_norm_kernel<T><<<blas_grid(nvec), BLAS_THREADS, 0, st>>>(nvec, (T)alpha, (const V*)x, (V*)y, partials);
}
template <typename T>
void launch_copy_norm(size_t nreal, const void* src, void* dst, double* partials, cudaStream_t st)
{
    launch_axpy_norm<T>(nreal, 1.0, src, dst, partials, st);
}
template void launch_axpy_norm<float>(size_t, double, const void*, void*, double*, cudaStream_t);
template void launch_axpy_norm<double>(size_t, double, const void*, void*, double*, cudaStream_t);
template void launch_copy_norm<float>(size_t, const void*, void*, double*, cudaStream_t);
template void launch_copy_norm<double>(size_t, const void*, void*, double*, cudaStream_t);

// ------------------------------------------------------------------ v *= *scale (device scalar)
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
scale_kernel(size_t nvec, typename VecOf<T>::type* __restrict__ v, const double* __restrict__ scale)
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    const T s = (T)(*scale);
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T r[N];
        unpack(v[i], r);
#pragma unroll
        for (int k = 0; k < N; ++k) r[k] *= s;
        v[i] = pack(r);
    }
}
template <typename T>
void launch_scale_by_dev(size_t nreal, void* v, const double* scale, cudaStream_t st)
{
    using V = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N;
    scale_kernel<T><<<blas_grid(nvec), BLAS_THREADS, 0, st>>>(nvec, (V*)v, scale);
}
template void launch_scale_by_dev<float>(size_t, void*, const double*, cudaStream_t);
template void launch_scale_by_dev<double>(size_t, void*, const double*, cudaStream_t);

// ------------------------------------------------------------------ fused multi-dot  <v_i, w>
template <typename T, int NB>
__global__ void __launch_bounds__(BLAS_THREADS)
multi_dot_kernel(size_t nvec, const typename VecOf<T>::type* __restrict__ V0, size_t vstride,
                 const typename VecOf<T>::type* __restrict__ w, double* __restrict__ partials)
{
    constexpr int N = VecOf<T>::N;
    double acc[2 * NB];
#pragma unroll
    for (int i = 0; i < 2 * NB; ++i) acc[i] = 0.0;
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        double wr[N];
        cvt(w[i], wr);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            double vr[N];
            cvt(V0[(size_t)b * vstride + i], vr);
#pragma unroll
            for (int c = 0; c < N; c += 2) {          // conj(v) * w
                acc[2 * b] += vr[c] * wr[c] + vr[c + 1] * wr[c + 1];
                acc[2 * b + 1] += vr[c] * wr[c + 1] - vr[c + 1] * wr[c];
            }
        }
    }
    block_sum_n<2 * NB>(acc, partials + (size_t)blockIdx.x * 2 * NB);
}
template <typename T>
void launch_multi_dot(size_t nreal, int nb, const void* V, size_t vstride_real, const void* w, double* partials,
                      cudaStream_t st)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N, vs = vstride_real / VecOf<T>::N;
    const int grid = blas_grid(nvec);
#define MD(NB) case NB: multi_dot_kernel<T, NB><<<grid, BLAS_THREADS, 0, st>>>(nvec, (const VT*)V, vs, (const VT*)w, partials); break;
    switch (nb) { MD(1) MD(2) MD(3) MD(4) MD(5) MD(6) MD(7) MD(8) MD(9) MD(10) MD(11) MD(12) }
    static_assert(MDOT_NB == 12, "one case per NB");
#undef MD
}
template void launch_multi_dot<float>(size_t, int, const void*, size_t, const void*, double*, cudaStream_t);
template void launch_multi_dot<double>(size_t, int, const void*, size_t, const void*, double*, cudaStream_t);

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

// ------------------------------------------------------------------ w += sum_i coef_i v_i  (+ |w|^2)
template <typename T, int NB>
__global__ void __launch_bounds__(BLAS_THREADS)
multi_axpy_kernel(size_t nvec, const typename VecOf<T>::type* __restrict__ V0, size_t vstride,
                  const double* __restrict__ coef, typename VecOf<T>::type* __restrict__ w,
                  double* __restrict__ partials, const double* __restrict__ wscale)
{
    constexpr int N = VecOf<T>::N;
    double cr[NB], ci[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) { cr[b] = coef[2 * b]; ci[b] = coef[2 * b + 1]; }
    const double ws = wscale ? *wscale : 1.0;        // w <- ws * w + sum_i coef_i v_i
    double acc[1] = { 0.0 };
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        double wr[N];
        cvt(w[i], wr);
        if (wscale) {
#pragma unroll
            for (int c = 0; c < N; ++c) wr[c] *= ws;
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            double vr[N];
            cvt(V0[(size_t)b * vstride + i], vr);
#pragma unroll
            for (int c = 0; c < N; c += 2) {
                wr[c] += cr[b] * vr[c] - ci[b] * vr[c + 1];
                wr[c + 1] += cr[b] * vr[c + 1] + ci[b] * vr[c];
            }
        }
        T o[N];
#pragma unroll
        for (int c = 0; c < N; ++c) { o[c] = (T)wr[c]; acc[0] += (double)o[c] * (double)o[c]; }
        w[i] = pack(o);
    }
    if (partials) block_sum_n<1>(acc, partials + blockIdx.x);
}
template <typename T>
void launch_multi_axpy(size_t nreal, int nb, const void* V, size_t vstride_real, const double* coef, void* w,
                       double* partials, cudaStream_t st, const double* wscale)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N, vs = vstride_real / VecOf<T>::N;
    const int grid = blas_grid(nvec);
#define MA(NB) case NB: multi_axpy_kernel<T, NB><<<grid, BLAS_THREADS, 0, st>>>(nvec, (const VT*)V, vs, coef, (VT*)w, partials, wscale); break;
    switch (nb) { MA(1) MA(2) MA(3) MA(4) MA(5) MA(6) MA(7) MA(8) MA(9) MA(10) MA(11) MA(12) }
#undef MA
}
template void launch_multi_axpy<float>(size_t, int, const void*, size_t, const double*, void*, double*, cudaStream_t, const double*);
template void launch_multi_axpy<double>(size_t, int, const void*, size_t, const double*, void*, double*, cudaStream_t, const double*);

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
    constexpr int N = VecOf<T>::N;
    double cr[NB > 0 ? NB : 1], ci[NB > 0 ? NB : 1];
#pragma unroll
    for (int b = 0; b < NB; ++b) { cr[b] = coef[2 * b]; ci[b] = coef[2 * b + 1]; }
    double acc[3] = { 0.0, 0.0, 0.0 };
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        double zr[N], pr[N], rr[N];
        cvt(z_io[i], zr);
        cvt(r[i], rr);
        if (init_p) {
#pragma unroll
            for (int c = 0; c < N; ++c) pr[c] = rr[c];
        } else {
            cvt(p_out[i], pr);
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            double zv[N], pv[N];
            cvt(Z0[(size_t)b * vstride + i], zv);
            cvt(P0[(size_t)b * vstride + i], pv);
#pragma unroll
            for (int c = 0; c < N; c += 2) {
                zr[c] += cr[b] * zv[c] - ci[b] * zv[c + 1];
                zr[c + 1] += cr[b] * zv[c + 1] + ci[b] * zv[c];
                pr[c] += cr[b] * pv[c] - ci[b] * pv[c + 1];
                pr[c + 1] += cr[b] * pv[c + 1] + ci[b] * pv[c];
            }
        }
        T zo[N], po[N];
#pragma unroll
        for (int c = 0; c < N; ++c) { zo[c] = (T)zr[c]; po[c] = (T)pr[c]; }
        if (NB > 0) z_io[i] = pack(zo);
        p_out[i] = pack(po);
        if (partials) {
#pragma unroll
            for (int c = 0; c < N; c += 2) {              // conj(z) * r
                const double a = zo[c], bq = zo[c + 1];
                acc[0] += a * a + bq * bq;
                acc[1] += a * rr[c] + bq * rr[c + 1];
                acc[2] += a * rr[c + 1] - bq * rr[c];
            }
        }
    }
    if (partials) block_sum_n<3>(acc, partials + (size_t)blockIdx.x * 3);
}
template <typename T>
void launch_gcr_form(size_t nreal, int nb, const void* Z0, const void* P0, size_t vstride_real, const double* coef,
                     void* z_io, const void* r, void* p_out, int init_p, double* partials, cudaStream_t st)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N, vs = vstride_real / VecOf<T>::N;
    const int grid = blas_grid(nvec);
#define GF(NB) case NB: gcr_form_kernel<T, NB><<<grid, BLAS_THREADS, 0, st>>>(nvec, (const VT*)Z0, (const VT*)P0, vs, coef, (VT*)z_io, (const VT*)r, (VT*)p_out, init_p, partials); break;
    switch (nb) { GF(0) GF(1) GF(2) GF(3) GF(4) GF(5) GF(6) GF(7) GF(8) GF(9) GF(10) GF(11) GF(12) }
#undef GF
}
template void launch_gcr_form<float>(size_t, int, const void*, const void*, size_t, const double*, void*, const void*, void*, int, double*, cudaStream_t);
template void launch_gcr_form<double>(size_t, int, const void*, const void*, size_t, const double*, void*, const void*, void*, int, double*, cudaStream_t);

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
    constexpr int N = VecOf<T>::N;
    const double ar = alpha[0], ai = alpha[1];
    double acc[1] = { 0.0 };
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        double xv[N], rv[N], pv[N], zv[N];
        cvt(x[i], xv); cvt(r[i], rv); cvt(p[i], pv); cvt(z[i], zv);
        T xo[N], ro[N];
#pragma unroll
        for (int c = 0; c < N; c += 2) {
            xo[c] = (T)(xv[c] + ar * pv[c] - ai * pv[c + 1]);
            xo[c + 1] = (T)(xv[c + 1] + ar * pv[c + 1] + ai * pv[c]);
            ro[c] = (T)(rv[c] - (ar * zv[c] - ai * zv[c + 1]));
            ro[c + 1] = (T)(rv[c + 1] - (ar * zv[c + 1] + ai * zv[c]));
        }
#pragma unroll
        for (int c = 0; c < N; ++c) acc[0] += (double)ro[c] * (double)ro[c];
        x[i] = pack(xo);
        r[i] = pack(ro);
    }
    block_sum_n<1>(acc, partials + blockIdx.x);
}
template <typename T>
void launch_gcr_update(size_t nreal, const double* alpha, const void* p, const void* z, void* x, void* r,
                       double* partials, cudaStream_t st)
{
    using VT = typename VecOf<T>::type;
    const size_t nvec = nreal / VecOf<T>::N;
    gcr_update_kernel<T><<<blas_grid(nvec), BLAS_THREADS, 0, st>>>(nvec, alpha, (const VT*)p, (const VT*)z, (VT*)x, (VT*)r, partials);
}
template void launch_gcr_update<float>(size_t, const double*, const void*, const void*, void*, void*, double*, cudaStream_t);
template void launch_gcr_update<double>(size_t, const double*, const void*, const void*, void*, void*, double*, cudaStream_t);

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

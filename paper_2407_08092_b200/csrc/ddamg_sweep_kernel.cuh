// ddamg_sweep_kernel.cuh -- one Schur apply / one Richardson sweep as ONE launch:
// kernel A (t_o = A_oo^-1 H_oe x_e) and kernel B / B' (y_e = A_ee x_e - H_eo t_o, Richardson
// update) pipelined time slice by time slice, so that t_o and the second read of x_e are served
// by L2 instead of HBM ("A->B slab pipelining in L2"; eq. 3, Alg. 4).
//
// Work is cut into tiles of DSLASH_THREADS sites; S tiles make one time slice.  Tiles are
// handed out in a fixed global order through an atomic ticket (so a tile only ever waits for
// tiles with smaller tickets: no deadlock whatever the CTA scheduling order):
//
//     A(T-1) A(0) .. A(lag) | B(0) A(lag+1) | B(1) A(lag+2) | ... | B(..) .. B(T-1)
//
// A(t) = kernel A on the odd sites of slice t, B(t) = kernel B / B' on the even sites of slice t.
// B(t) reads t_o on slices t-1, t, t+1 (periodic), so it waits until the three counters
// done[t-1], done[t], done[t+1] (incremented by every finished A tile, release / acquire at
// gpu scope) have reached S.  With lag >= 2 the A tiles B(t) needs were handed out a whole
// slice earlier and the wait is a single load.  In-place Richardson (out == x_e) is race-free
// under the same rule: x_e on slice t is read by A(t-1), A(t), A(t+1) only, exactly the tasks
// B(t) waits for.  Per-site arithmetic is the code of dslash_kernel: results are bit-identical
// to the two-launch path.
#pragma once
#include "ddamg_internal.h"
#include "ddamg_hop.cuh"

namespace ddamg {

template <typename T>
struct SweepArgs {
    Geom g;
    const T* x;              // x_e: neighbours of kernel A, own-site operand of kernel B
    T* t;                    // t_o scratch (written by A tiles, read by B tiles)
    const T* gauge_e;        // link blocks of the even / odd sites (18- or 12-real)
    const T* gauge_o;
    const T* clov_e;         // A_ee
    const T* clov_oinv;      // A_oo^-1
    const T* rhs;            // b_e (EPI_RICHARDSON / EPI_RESIDUAL)
    T* out;                  // y_e, or x_e itself for the in-place Richardson update
    T omega;
    double* partials;        // NORM: per-tile sums of |r|^2, indexed like the two-launch path
    unsigned int* sync;      // [0] ticket, [1 + t] finished A tiles of slice t; zeroed before the launch
    int S;                   // tiles per time slice = Lh * L * L / DSLASH_THREADS
    int nA0;                 // A tasks handed out before the first B task = min(lag + 2, T)
    int apbc;
};

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <typename T, int EPI_B, bool NORM, int RECON>
__global__ void __launch_bounds__(DSLASH_THREADS) __maxnreg__(sizeof(T) == 4 ? 128 : 255)
sweep_kernel(const SweepArgs<T> a)
{
    __shared__ unsigned int s_ticket;
    __shared__ double warp_part[DSLASH_THREADS / 32];
    if (threadIdx.x == 0) s_ticket = atomicAdd(&a.sync[0], 1u);
    __syncthreads();
    const int task = (int)(s_ticket / (unsigned)a.S), tile = (int)(s_ticket - (unsigned)task * a.S);
    const int Tt = a.g.T, R = Tt - a.nA0;
    int phase, t;                                   // phase 0 = A, 1 = B
    if (task < a.nA0) { phase = 0; t = task == 0 ? Tt - 1 : task - 1; }
    else {
        const int k = task - a.nA0;
        if (k < 2 * R) { phase = (k & 1) ^ 1; t = (k & 1) ? a.nA0 - 1 + (k >> 1) : (k >> 1); }
        else { phase = 1; t = R + (k - 2 * R); }
    }
    const int cb = (t * a.S + tile) * DSLASH_THREADS + threadIdx.x;
    if (phase == 0) {
        const Site s = site_of_cb(a.g, cb, 1);
        T acc[24], res[24];
        hop_site<T, RECON>(a.g, cb, s, a.x, 1, 0, a.gauge_o, a.gauge_e, acc, a.apbc);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] *= (T)(-0.5);
        clover_site_mul<T>(a.clov_oinv, a.g.Vh, cb, acc, res);
        store_spinor<T>(a.t, a.g.Vh, cb, res);
        __syncthreads();                            // all stores of the tile, then release by thread 0
        if (threadIdx.x == 0) {
            __threadfence();
            atomicAdd(&a.sync[1 + t], 1u);
        }
        return;
    }
    if (threadIdx.x == 0) {
        const int tm = t == 0 ? Tt - 1 : t - 1, tp = t == Tt - 1 ? 0 : t + 1;
        while (ld_acquire_gpu(&a.sync[1 + t]) < (unsigned)a.S) __nanosleep(200);
        while (ld_acquire_gpu(&a.sync[1 + tm]) < (unsigned)a.S) __nanosleep(200);
        while (ld_acquire_gpu(&a.sync[1 + tp]) < (unsigned)a.S) __nanosleep(200);
    }
    __syncthreads();
    const Site s = site_of_cb(a.g, cb, 0);
    T acc[24], res[24], x[24], ax[24];
    hop_site<T, RECON>(a.g, cb, s, a.t, 1, 0, a.gauge_e, a.gauge_o, acc, a.apbc);
    load_spinor<T, true>(a.x, a.g.Vh, cb, x);
    clover_site_mul<T>(a.clov_e, a.g.Vh, cb, x, ax);
    double nrm = 0.0;
    if (EPI_B == EPI_SCHUR) {
#pragma unroll
        for (int i = 0; i < 24; ++i) res[i] = ax[i] + (T)0.5 * acc[i];
    } else {
        T b[24];
        load_spinor<T, true>(a.rhs, a.g.Vh, cb, b);
#pragma unroll
        for (int i = 0; i < 24; ++i) {
            const T r = b[i] - (ax[i] + (T)0.5 * acc[i]);
            if (NORM) nrm += (double)r * (double)r;
            res[i] = (EPI_B == EPI_RICHARDSON) ? x[i] + a.omega * r : r;
        }
    }
    store_spinor<T>(a.out, a.g.Vh, cb, res);
    if (NORM) {                                     // same reduction tree as dslash_kernel's block_sum
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        if (lane == 0) warp_part[w] = nrm;
        __syncthreads();
        double v = (threadIdx.x < DSLASH_THREADS / 32) ? warp_part[threadIdx.x] : 0.0;
        if (w == 0) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) a.partials[t * a.S + tile] = v;
        }
    }
}

// epi_b: EPI_SCHUR (y_e = D_S x_e), EPI_RICHARDSON (in place when out == x) or EPI_RESIDUAL.
// Requires sweep_eligible(g).  sync: T + 1 device words owned by the context.
template <typename T, int RECON>
cudaError_t launch_sweep_recon(const Geom& g, int epi_b, bool norm, const void* x, void* t, const void* gauge_e,
                               const void* gauge_o, const void* clov_e, const void* clov_oinv, const void* rhs,
                               void* out, double omega, double* partials, unsigned int* sync, int lag, int apbc,
                               cudaStream_t st)
{
    SweepArgs<T> a;
    a.g = g;
    a.x = (const T*)x; a.t = (T*)t;
    a.gauge_e = (const T*)gauge_e; a.gauge_o = (const T*)gauge_o;
    a.clov_e = (const T*)clov_e; a.clov_oinv = (const T*)clov_oinv;
    a.rhs = (const T*)rhs; a.out = (T*)out; a.omega = (T)omega; a.partials = partials; a.sync = sync;
    a.S = g.Lh * g.L * g.L / DSLASH_THREADS;
    a.nA0 = lag + 2 < g.T ? lag + 2 : g.T;
    a.apbc = apbc;
    cudaError_t e = cudaMemsetAsync(sync, 0, sizeof(unsigned int) * (size_t)(g.T + 1), st);
    if (e != cudaSuccess) return e;
    const int grid = 2 * g.T * a.S;
    if (epi_b == EPI_SCHUR) sweep_kernel<T, EPI_SCHUR, false, RECON><<<grid, DSLASH_THREADS, 0, st>>>(a);
    else if (epi_b == EPI_RICHARDSON) {
        if (norm) sweep_kernel<T, EPI_RICHARDSON, true, RECON><<<grid, DSLASH_THREADS, 0, st>>>(a);
        else sweep_kernel<T, EPI_RICHARDSON, false, RECON><<<grid, DSLASH_THREADS, 0, st>>>(a);
    } else {
        if (norm) sweep_kernel<T, EPI_RESIDUAL, true, RECON><<<grid, DSLASH_THREADS, 0, st>>>(a);
        else sweep_kernel<T, EPI_RESIDUAL, false, RECON><<<grid, DSLASH_THREADS, 0, st>>>(a);
    }
    return cudaSuccess;
}

}  // namespace ddamg

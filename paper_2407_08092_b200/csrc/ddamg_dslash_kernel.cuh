// ddamg_dslash_kernel.cuh -- the fused hopping + clover kernel template, instantiated once per
// link storage format: RECON = 18 in ddamg_dslash.cu, RECON = 12 (two-row links) in
// ddamg_dslash12.cu.
#pragma once
#include "ddamg_internal.h"
#include "ddamg_hop.cuh"

namespace ddamg {

template <typename T>
struct DslashArgs {
    Geom g;
    int parity;              // parity of the output sites
    const T* in;             // opposite-parity spinor (the 8 neighbours)
    const T* gauge_own;      // 4 link blocks of the output parity
    const T* gauge_opp;      // 4 link blocks of the opposite parity
    const T* clov;           // clover blocks of the output parity: the inverses (packed 36 reals per block) for
                             // EPI_CLOV_*, the blocks themselves (compact 28 reals per block) for EPI >= EPI_SCHUR
    T c0;                    // m0 + 4, the constant part of the compact blocks
    const T* own;            // own-site spinor (EPI_SCHUR / RICHARDSON / RESIDUAL)
    const T* rhs;            // b (EPI_RICHARDSON / RESIDUAL / *_RHS_*)
    T* out;
    T omega;
    double* partials;        // per-block sum of |r|^2 (NORM) or nullptr; batch: [block][units * lanes]
    int nrhs;                // BATCH kernels: threads (units) per site = rhs pairs (fp32) or rhs (fp64); else 1
    int zc;                  // BATCH: z-chunk of the CTA traversal (0 = plain lexicographic order)
    int cpp;                 // BATCH: CTAs per (z,t) plane = Lh * L * nrhs / DSLASH_THREADS (when zc > 0)
    int apbc;                // RECON = 12: antiperiodic time boundary (sign of the rebuilt third row of U_t(T-1))
};

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double warp_part[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) warp_part[w] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? warp_part[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    }
    return v;     // valid in thread 0
}

// Register budget per thread (ptxas trades registers for loads in flight; measured on B200,
// 128 registers = 4 CTAs of 128 threads per SM is the optimum for both
// the kernel-A class (EPI <= EPI_RHS_MINUS_HOP) and the kernel-B class).
#ifndef DDAMG_MAXREG_A
#define DDAMG_MAXREG_A 128
#endif
#ifndef DDAMG_MAXREG_B
#define DDAMG_MAXREG_B 128
#endif
#ifndef DDAMG_MAXREG_BATCH
#define DDAMG_MAXREG_BATCH 128     // multi-rhs kernels
#endif

// spinor value type of a kernel: one value per thread, or (fp32 multi-rhs) a packed pair of
// right-hand sides per thread
template <typename T, bool BATCH> struct ValueOf { using type = T; static constexpr int LANES = 1; };
template <> struct ValueOf<float, true> { using type = P2; static constexpr int LANES = 2; };

// BATCH (multi-rhs): one thread per (site, unit), unit fastest, so that the
// threads of a site share every link / clover vector they load while all spinor planes stay
// contiguous per warp (vector index cb * units + r).  fp32: a unit is a PAIR of right-hand
// sides carried through the whole site update as the two lanes of packed f32x2 instructions
// (links, the rebuilt third rows, clover entries and every index computation are shared by
// the pair); fp64: a unit is one right-hand side.  a.nrhs = units per site.
template <typename T, int EPI, bool NORM, bool BATCH, int RECON>
__global__ void __launch_bounds__(DSLASH_THREADS)
__maxnreg__(sizeof(T) == 4 ? (BATCH ? DDAMG_MAXREG_BATCH : EPI <= EPI_RHS_MINUS_HOP ? DDAMG_MAXREG_A : DDAMG_MAXREG_B) : 255)
dslash_kernel(const DslashArgs<T> a)
{
    using S = typename ValueOf<T, BATCH>::type;
    constexpr int LANES = ValueOf<T, BATCH>::LANES;
    // BATCH: with several spinors per site one time slice of neighbour spinors no longer fits L2
    // (64^3: nrhs * 12.6 MB), so the t-1 neighbours would be re-fetched from HBM.  CTAs therefore
    // walk the lattice in z-chunks: for each chunk of zc z-planes, t runs over the whole time
    // extent before the next chunk starts, which keeps three t-slabs of the chunk L2-resident.
    int blk = blockIdx.x;
    if (BATCH && a.zc > 0) {
        const int plane = blk / a.cpp, within = blk - plane * a.cpp;     // plane in chunked order
        const int per_chunk = a.zc * a.g.T;
        const int chunk = plane / per_chunk, rem = plane - chunk * per_chunk;
        const int t = rem / a.zc, z = chunk * a.zc + (rem - t * a.zc);
        blk = (t * a.g.L + z) * a.cpp + within;
    }
    const int tid = blk * DSLASH_THREADS + threadIdx.x;
    const int units = BATCH ? a.nrhs : 1;
    const int cb = BATCH ? tid / units : tid;
    const int rr = BATCH ? tid - cb * units : 0;
    const int Vs = a.g.Vh * units;         // vectors per spinor plane
    const int sv = cb * units + rr;        // this thread's vector index in a spinor plane (== tid)
    double nrm[2] = { 0.0, 0.0 };
    if (cb < a.g.Vh) {
        const Site s = site_of_cb(a.g, cb, a.parity);
        S acc[24];
        hop_site<T, RECON, S>(a.g, cb, s, a.in, units, rr, a.gauge_own, a.gauge_opp, acc, a.apbc);
        S res[24];
        if (EPI == EPI_CLOV_HOP) {
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = vmul((T)(-0.5), acc[i]);
            clover_site_mul<T>(a.clov, a.g.Vh, cb, acc, res);
        } else if (EPI == EPI_CLOV_RHS_MINUS_HOP) {
            S b[24];
            load_spinor<T, true>(a.rhs, Vs, sv, b);
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = vfma((T)0.5, acc[i], b[i]);
            clover_site_mul<T>(a.clov, a.g.Vh, cb, acc, res);
        } else if (EPI == EPI_RHS_MINUS_HOP) {
            S b[24];
            load_spinor<T, true>(a.rhs, Vs, sv, b);
#pragma unroll
            for (int i = 0; i < 24; ++i) res[i] = vfma((T)0.5, acc[i], b[i]);
        } else {
            S x[24], ax[24];
            load_spinor<T, true>(a.own, Vs, sv, x);
            clover_site_mul<T, LD_STREAM, true>(a.clov, a.g.Vh, cb, x, ax, a.c0);
            // H = -1/2 acc:  Schur forms subtract H t (+1/2 acc), the full operator adds H x (-1/2 acc)
            constexpr bool FULL = (EPI == EPI_FULL || EPI == EPI_FULL_RESIDUAL);
            const T hs = FULL ? (T)(-0.5) : (T)0.5;
            if (EPI == EPI_SCHUR || EPI == EPI_FULL) {
#pragma unroll
                for (int i = 0; i < 24; ++i) res[i] = vfma(hs, acc[i], ax[i]);     // A x - H t   or   A x + H x'
            } else {
                S b[24];
                load_spinor<T, true>(a.rhs, Vs, sv, b);
#pragma unroll
                for (int i = 0; i < 24; ++i) {
                    const S r = b[i] - vfma(hs, acc[i], ax[i]);
                    if (NORM) vnorm_add(r, nrm);
                    res[i] = (EPI == EPI_RICHARDSON) ? vfma(a.omega, r, x[i]) : r;
                }
            }
        }
        store_spinor<T>(a.out, Vs, sv, res);
    }
    if (NORM) {
        if (BATCH) {
            // per-rhs partial sums of this block: thread q < units * LANES adds the entries of rhs q
            // (rhs = unit * LANES + lane); partials[block][units * LANES]
            __shared__ double per_thread[LANES][DSLASH_THREADS];
            per_thread[0][threadIdx.x] = nrm[0];
            if (LANES == 2) per_thread[LANES - 1][threadIdx.x] = nrm[1];
            __syncthreads();
            if ((int)threadIdx.x < units * LANES) {
                const int unit = (int)threadIdx.x / LANES, lane = (int)threadIdx.x - unit * LANES;
                const int first = (int)(((long long)blk * DSLASH_THREADS) % units);          // unit of thread 0
                int i = unit - first;
                if (i < 0) i += units;
                double tot = 0.0;
                for (; i < DSLASH_THREADS; i += units) tot += per_thread[lane][i];
                a.partials[(size_t)blk * units * LANES + threadIdx.x] = tot;
            }
        } else {
            const double tot = block_sum(nrm[0]);
            if (threadIdx.x == 0) a.partials[blockIdx.x] = tot;
        }
    }
}

template <typename T, int EPI, bool NORM, int RECON>
static void launch(const DslashArgs<T>& a, cudaStream_t st)
{
    if (a.nrhs > 0) dslash_kernel<T, EPI, NORM, true, RECON><<<dslash_grid(a.g, a.nrhs), DSLASH_THREADS, 0, st>>>(a);
    else dslash_kernel<T, EPI, NORM, false, RECON><<<dslash_grid(a.g, 1), DSLASH_THREADS, 0, st>>>(a);
}

template <typename T, int RECON>
void launch_dslash_recon(const Geom& g, int epi, bool norm, int parity, const void* in, const void* gauge_own,
                         const void* gauge_opp, const void* clov, const void* own, const void* rhs, void* out,
                         double omega, double c0, double* partials, int units, double batch_l2_bytes, int apbc, cudaStream_t st)
{
    // units = 0: one right-hand side in the native half-spinor layout; units >= 1: multi-rhs batch with
    // that many threads per site (fp32: rhs pairs, fp64: rhs)
    DslashArgs<T> a;
    a.apbc = apbc;
    a.nrhs = units;
    a.zc = 0;
    a.cpp = 0;
    const long long plane_threads = (long long)g.Lh * g.L * units;
    const int lanes = sizeof(T) == 4 ? 2 : 1;
    if (units * lanes > 1 && plane_threads % DSLASH_THREADS == 0) {
        // largest divisor zc of L whose three t-slabs of spinors (zc planes each) fit the L2 budget
        const double plane_bytes = (double)g.Lh * g.L * units * lanes * 24 * sizeof(T);
        int zc = 0;
        for (int d = 1; d <= g.L; ++d)
            if (g.L % d == 0 && 3.0 * d * plane_bytes <= batch_l2_bytes) zc = d;
        if (zc == 0) zc = 1;
        if (zc < g.L) {
            a.zc = zc;
            a.cpp = (int)(plane_threads / DSLASH_THREADS);
        }
    }
    a.g = g;
    a.parity = parity;
    a.in = (const T*)in;
    a.gauge_own = (const T*)gauge_own;
    a.gauge_opp = (const T*)gauge_opp;
    a.clov = (const T*)clov;
    a.own = (const T*)own;
    a.rhs = (const T*)rhs;
    a.out = (T*)out;
    a.omega = (T)omega;
    a.c0 = (T)c0;
    a.partials = partials;
    switch (epi) {
    case EPI_CLOV_HOP: launch<T, EPI_CLOV_HOP, false, RECON>(a, st); break;
    case EPI_CLOV_RHS_MINUS_HOP: launch<T, EPI_CLOV_RHS_MINUS_HOP, false, RECON>(a, st); break;
    case EPI_RHS_MINUS_HOP: launch<T, EPI_RHS_MINUS_HOP, false, RECON>(a, st); break;
    case EPI_SCHUR: launch<T, EPI_SCHUR, false, RECON>(a, st); break;
    case EPI_RICHARDSON:
        if (norm) launch<T, EPI_RICHARDSON, true, RECON>(a, st);
        else launch<T, EPI_RICHARDSON, false, RECON>(a, st);
        break;
    case EPI_RESIDUAL:
        if (norm) launch<T, EPI_RESIDUAL, true, RECON>(a, st);
        else launch<T, EPI_RESIDUAL, false, RECON>(a, st);
        break;
    case EPI_FULL: launch<T, EPI_FULL, false, RECON>(a, st); break;
    case EPI_FULL_RESIDUAL:
        if (norm) launch<T, EPI_FULL_RESIDUAL, true, RECON>(a, st);
        else launch<T, EPI_FULL_RESIDUAL, false, RECON>(a, st);
        break;
    }
}

}  // namespace ddamg

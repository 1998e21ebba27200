// ddamg_setup.cu -- setup steps a0 (gauge repack) and a1 (clover build + 6x6 inversion),
// plus the layout converters that hide the native layout from callers.
//
// The clover term ("Wilson-Dirac discretization with a clover improvement";
// DESIGN.md readings R4, R5) is assembled directly in its chiral 6x6 block form
// (D_ee, D_oo block diagonal with 6x6 blocks):
//   A_upper = (m0+4) - (csw/16) sum_k sigma_k (x) i (F'_ij - F'_kt)
//   A_lower = (m0+4) - (csw/16) sum_k sigma_k (x) i (F'_ij + F'_kt),  (i,j,k) cyclic,
// with F' = Q - Q^H and Q the sum of the four plaquette leaves.  All arithmetic in fp64;
// the result is rounded once to the context precision.
#include <cstdint>
#include "ddamg_internal.h"

namespace ddamg {

// ------------------------------------------------------------------ coordinates (setup only)
struct Coord { int x[4]; };

__device__ __forceinline__ Coord coord_of(const Geom& g, int cb, int parity)
{
    const Site s = site_of_cb(g, cb, parity);
    Coord c;
    c.x[0] = 2 * s.xh + s.q; c.x[1] = s.y; c.x[2] = s.z; c.x[3] = s.t;
    return c;
}
__device__ __forceinline__ int parity_of(const Coord& c) { return (c.x[0] + c.x[1] + c.x[2] + c.x[3]) & 1; }
__device__ __forceinline__ int cb_of(const Geom& g, const Coord& c)
{
    return (c.x[0] >> 1) + g.Lh * (c.x[1] + g.L * (c.x[2] + g.L * c.x[3]));
}
__device__ __forceinline__ size_t nat_of(const Geom& g, const Coord& c)
{
    return (size_t)c.x[0] + (size_t)g.L * (c.x[1] + (size_t)g.L * (c.x[2] + (size_t)g.L * c.x[3]));
}
__device__ __forceinline__ Coord shift(const Geom& g, Coord c, int mu, int d)
{
    const int e = (mu == 3) ? g.T : g.L;
    c.x[mu] = (c.x[mu] + d + e) % e;
    return c;
}

// ------------------------------------------------------------------ a0: gauge repack
// VEC: the natural field is 16-byte aligned, so a site's 72 input reals are read as whole 16-byte vectors
// (18 float4 / 36 double2 / ...) instead of 72 scalars.
template <typename Tin, typename T, bool VEC>
__global__ void pack_gauge_kernel(Geom g, int bc, const Tin* __restrict__ U, T* __restrict__ gauge)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    const Coord c = coord_of(g, cb, parity);
    const size_t n = nat_of(g, c);
    const size_t lblk = (size_t)18 * g.Vh;
    Tin r[72];
    if (VEC) {
        using Vin = typename VecOf<Tin>::type;
        constexpr int NI = VecOf<Tin>::N;
        const Vin* src = reinterpret_cast<const Vin*>(U) + n * (72 / NI);
#pragma unroll
        for (int k = 0; k < 72 / NI; ++k) unpack(ld_stream(src + k), &r[k * NI]);
    } else {
#pragma unroll
        for (int k = 0; k < 72; ++k) r[k] = U[n * 72 + k];
    }
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        T u[18];
        const T sgn = (bc == 1 && mu == 3 && c.x[3] == g.T - 1) ? (T)-1 : (T)1;
#pragma unroll
        for (int k = 0; k < 18; ++k) u[k] = sgn * (T)r[18 * mu + k];
        store_link(gauge + ((size_t)parity * 4 + mu) * lblk, g.Vh, cb, u);
    }
}

template <typename Tin, typename T>
void launch_pack_gauge(const Geom& g, int bc, const void* U_nat, void* gauge, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    if (((uintptr_t)U_nat & 15) == 0)
        pack_gauge_kernel<Tin, T, true><<<(n + 127) / 128, 128, 0, st>>>(g, bc, (const Tin*)U_nat, (T*)gauge);
    else
        pack_gauge_kernel<Tin, T, false><<<(n + 127) / 128, 128, 0, st>>>(g, bc, (const Tin*)U_nat, (T*)gauge);
}
template void launch_pack_gauge<float, float>(const Geom&, int, const void*, void*, cudaStream_t);
template void launch_pack_gauge<double, float>(const Geom&, int, const void*, void*, cudaStream_t);
template void launch_pack_gauge<float, double>(const Geom&, int, const void*, void*, cudaStream_t);
template void launch_pack_gauge<double, double>(const Geom&, int, const void*, void*, cudaStream_t);

// ------------------------------------------------------------------ two-row link copy
// gauge12 = rows 0, 1 of every packed link (sign of the antiperiodic boundary included, as in
// `gauge`).  Also measures how far the stored third rows are from sgn * conj(row0 x row1): the
// caller refuses two-row storage for links that are not SU(3) to working precision.
template <typename T>
__global__ void compress_gauge_kernel(Geom g, int bc, const T* __restrict__ gauge, T* __restrict__ gauge12,
                                      unsigned int* __restrict__ dev_max_bits)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    float dev = 0.f;
    if (idx < 2 * g.Vh) {
        const int parity = idx / g.Vh, cb = idx % g.Vh;
        const Site s = site_of_cb(g, cb, parity);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            T u[18], v[18];
            load_link(gauge + ((size_t)parity * 4 + mu) * (size_t)18 * g.Vh, g.Vh, cb, u);
#pragma unroll
            for (int k = 0; k < 12; ++k) v[k] = u[k];
            const T sgn = (bc == 1 && mu == 3 && s.t == g.T - 1) ? (T)-1 : (T)1;
            reconstruct_row2<T>(sgn, v);
#pragma unroll
            for (int k = 12; k < 18; ++k) {
                const float d = fabsf((float)(v[k] - u[k]));
                dev = (d > dev || !(d == d)) ? d : dev;          // NaN-propagating max (fmaxf would drop a NaN)
            }
            store_link12(gauge12 + ((size_t)parity * 4 + mu) * (size_t)12 * g.Vh, g.Vh, cb, u);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o));
    // fmaxf drops NaNs: a non-finite link must not pass as "deviation 0", so it is reported as +Inf
    bool bad = !isfinite(dev);
    bad = __any_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && (bad || dev > 0.f)) atomicMax(dev_max_bits, bad ? 0x7f800000u : __float_as_uint(dev));
}

template <typename T>
void launch_compress_gauge(const Geom& g, int bc, const void* gauge, void* gauge12, unsigned int* dev_max_bits,
                           cudaStream_t st)
{
    const int n = 2 * g.Vh;
    compress_gauge_kernel<T><<<(n + 255) / 256, 256, 0, st>>>(g, bc, (const T*)gauge, (T*)gauge12, dev_max_bits);
}
template void launch_compress_gauge<float>(const Geom&, int, const void*, void*, unsigned int*, cudaStream_t);
template void launch_compress_gauge<double>(const Geom&, int, const void*, void*, unsigned int*, cudaStream_t);

// ------------------------------------------------------------------ spinor layout converters
// A site's 24 reals are 24/N 16-byte vectors in the natural layout as well, and vector k of the site IS plane k of
// the native layout: both converters move whole vectors (natural side: 6 / 12 accesses of 16 bytes per thread at
// a 96 / 192-byte stride, all sectors fully used between them; native side: one contiguous run per plane and warp).
template <typename T>
__global__ void pack_spinor_kernel(Geom g, const T* __restrict__ nat, T* __restrict__ xe, T* __restrict__ xo)
{
    using V = typename VecOf<T>::type;
    constexpr int NV = 24 / VecOf<T>::N;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    T* dst = parity ? xo : xe;
    if (!dst) return;
    const size_t n = nat_of(g, coord_of(g, cb, parity));
    const V* src = reinterpret_cast<const V*>(nat) + n * NV;
    V v[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = ld_stream(src + k);
    V* d = reinterpret_cast<V*>(dst) + cb;
#pragma unroll
    for (int k = 0; k < NV; ++k) d[(size_t)k * g.Vh] = v[k];
}

template <typename T>
__global__ void unpack_spinor_kernel(Geom g, const T* __restrict__ xe, const T* __restrict__ xo, T* __restrict__ nat)
{
    using V = typename VecOf<T>::type;
    constexpr int NV = 24 / VecOf<T>::N;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    const T* src = parity ? xo : xe;
    const size_t n = nat_of(g, coord_of(g, cb, parity));
    V v[NV];
    if (src) {
        const V* sp = reinterpret_cast<const V*>(src) + cb;
#pragma unroll
        for (int k = 0; k < NV; ++k) v[k] = ld_stream(sp + (size_t)k * g.Vh);
    } else {
        T z[VecOf<T>::N] = {};
#pragma unroll
        for (int k = 0; k < NV; ++k) v[k] = pack(z);
    }
    V* d = reinterpret_cast<V*>(nat) + n * NV;
#pragma unroll
    for (int k = 0; k < NV; ++k) d[k] = v[k];
}

template <typename T>
void launch_pack_spinor(const Geom& g, const void* nat, void* x_e, void* x_o, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    pack_spinor_kernel<T><<<(n + 255) / 256, 256, 0, st>>>(g, (const T*)nat, (T*)x_e, (T*)x_o);
}
template <typename T>
void launch_unpack_spinor(const Geom& g, const void* x_e, const void* x_o, void* nat, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    unpack_spinor_kernel<T><<<(n + 255) / 256, 256, 0, st>>>(g, (const T*)x_e, (const T*)x_o, (T*)nat);
}
template void launch_pack_spinor<float>(const Geom&, const void*, void*, void*, cudaStream_t);
template void launch_pack_spinor<double>(const Geom&, const void*, void*, void*, cudaStream_t);
template void launch_unpack_spinor<float>(const Geom&, const void*, const void*, void*, cudaStream_t);
template void launch_unpack_spinor<double>(const Geom&, const void*, const void*, void*, cudaStream_t);

// ------------------------------------------------------------------ multi-rhs interleave
// fp64:  X[plane][cb * nrhs + r] = halves[r][plane][cb]  (TO_BATCH) or the inverse.  One thread per
// vector of the batch; writes (TO_BATCH) / reads (inverse) of the batch are contiguous.
template <bool TO_BATCH>
__global__ void batch_interleave_kernel(int Vh, int nrhs, double2* __restrict__ halves, double2* __restrict__ X)
{
    constexpr int NP = 12;
    const size_t per_plane = (size_t)Vh * nrhs;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per_plane * NP) return;
    const int plane = (int)(i / per_plane);
    const size_t rem = i - (size_t)plane * per_plane;
    const int cb = (int)(rem / nrhs), r = (int)(rem - (size_t)cb * nrhs);
    const size_t h = ((size_t)r * NP + plane) * Vh + cb;
    if (TO_BATCH) X[i] = halves[h];
    else halves[h] = X[i];
}
// fp32 pair layout (ddamg_common.cuh, load_spinor of P2): 12 half-planes of float4; half-plane h, vector
// cb * npairs + p = (re, re', im, im') of complex number h of the site for the rhs 2p and 2p+1.  An odd nrhs
// leaves the second lane of the last pair as padding: written as 0 (TO_BATCH), ignored (inverse).
template <bool TO_BATCH>
__global__ void batch_interleave_pairs_kernel(int Vh, int nrhs, float2* __restrict__ halves, float4* __restrict__ X)
{
    const int npairs = (nrhs + 1) / 2;
    const size_t per_plane = (size_t)Vh * npairs;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per_plane * 12) return;
    const int h = (int)(i / per_plane);
    const size_t rem = i - (size_t)h * per_plane;
    const int cb = (int)(rem / npairs), p = (int)(rem - (size_t)cb * npairs);
    // complex number h of a native half spinor = float2 number (h & 1) of the float4 at plane h / 2
    const size_t per_rhs = (size_t)12 * Vh;                       // float2 per half spinor
    const size_t src = ((size_t)(h >> 1) * Vh + cb) * 2 + (h & 1);
    const int r0 = 2 * p, r1 = 2 * p + 1;
    if (TO_BATCH) {
        const float2 a = halves[(size_t)r0 * per_rhs + src];
        const float2 b = r1 < nrhs ? halves[(size_t)r1 * per_rhs + src] : make_float2(0.f, 0.f);
        X[i] = make_float4(a.x, b.x, a.y, b.y);
    } else {
        const float4 v = X[i];
        halves[(size_t)r0 * per_rhs + src] = make_float2(v.x, v.z);
        if (r1 < nrhs) halves[(size_t)r1 * per_rhs + src] = make_float2(v.y, v.w);
    }
}
template <typename T>
void launch_batch_interleave(const Geom& g, int nrhs, bool to_batch, void* halves, void* X, cudaStream_t st);
template <>
void launch_batch_interleave<double>(const Geom& g, int nrhs, bool to_batch, void* halves, void* X, cudaStream_t st)
{
    const size_t n = (size_t)g.Vh * nrhs * 12;
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (to_batch) batch_interleave_kernel<true><<<grid, 256, 0, st>>>(g.Vh, nrhs, (double2*)halves, (double2*)X);
    else batch_interleave_kernel<false><<<grid, 256, 0, st>>>(g.Vh, nrhs, (double2*)halves, (double2*)X);
}
template <>
void launch_batch_interleave<float>(const Geom& g, int nrhs, bool to_batch, void* halves, void* X, cudaStream_t st)
{
    const size_t n = (size_t)g.Vh * ((nrhs + 1) / 2) * 12;
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (to_batch) batch_interleave_pairs_kernel<true><<<grid, 256, 0, st>>>(g.Vh, nrhs, (float2*)halves, (float4*)X);
    else batch_interleave_pairs_kernel<false><<<grid, 256, 0, st>>>(g.Vh, nrhs, (float2*)halves, (float4*)X);
}

// ------------------------------------------------------------------ a1: clover build
struct M3 { double re[9], im[9]; };

template <typename T>
__device__ void link_at(const Geom& g, const T* __restrict__ gauge, const Coord& c, int mu, M3& m)
{
    const int par = parity_of(c), cb = cb_of(g, c);
    T u[18];
    load_link(gauge + ((size_t)par * 4 + mu) * (size_t)18 * g.Vh, g.Vh, cb, u);
#pragma unroll
    for (int k = 0; k < 9; ++k) { m.re[k] = (double)u[2 * k]; m.im[k] = (double)u[2 * k + 1]; }
}

// c = op(a) * op(b),  op = identity or Hermitian conjugate
template <bool DA, bool DB>
__device__ void mm(const M3& a, const M3& b, M3& c)
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double sr = 0, si = 0;
            for (int k = 0; k < 3; ++k) {
                const int ia = DA ? 3 * k + i : 3 * i + k;
                const int ib = DB ? 3 * j + k : 3 * k + j;
                const double ar = a.re[ia], ai = DA ? -a.im[ia] : a.im[ia];
                const double br = b.re[ib], bi = DB ? -b.im[ib] : b.im[ib];
                sr += ar * br - ai * bi;
                si += ar * bi + ai * br;
            }
            c.re[3 * i + j] = sr;
            c.im[3 * i + j] = si;
        }
}

// F'_{mu nu}(x) = Q - Q^H, Q = sum of the four leaves at x (reading R4)
template <typename T>
__device__ void field_strength(const Geom& g, const T* __restrict__ gauge, const Coord& x, int mu, int nu, M3& F)
{
    M3 Q, a, b, t1, t2;
    for (int k = 0; k < 9; ++k) Q.re[k] = Q.im[k] = 0;
    const Coord xpm = shift(g, x, mu, +1), xpn = shift(g, x, nu, +1);
    const Coord xmm = shift(g, x, mu, -1), xmn = shift(g, x, nu, -1);
    const Coord xmm_pn = shift(g, xmm, nu, +1), xmm_mn = shift(g, xmm, nu, -1), xpm_mn = shift(g, xpm, nu, -1);
    // leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^H U_nu(x)^H
    link_at(g, gauge, x, mu, a); link_at(g, gauge, xpm, nu, b); mm<false, false>(a, b, t1);
    link_at(g, gauge, xpn, mu, a); mm<false, true>(t1, a, t2);
    link_at(g, gauge, x, nu, a); mm<false, true>(t2, a, t1);
    for (int k = 0; k < 9; ++k) { Q.re[k] += t1.re[k]; Q.im[k] += t1.im[k]; }
    // leaf 2: U_nu(x) U_mu(x-mu+nu)^H U_nu(x-mu)^H U_mu(x-mu)
    link_at(g, gauge, x, nu, a); link_at(g, gauge, xmm_pn, mu, b); mm<false, true>(a, b, t1);
    link_at(g, gauge, xmm, nu, a); mm<false, true>(t1, a, t2);
    link_at(g, gauge, xmm, mu, a); mm<false, false>(t2, a, t1);
    for (int k = 0; k < 9; ++k) { Q.re[k] += t1.re[k]; Q.im[k] += t1.im[k]; }
    // leaf 3: U_mu(x-mu)^H U_nu(x-mu-nu)^H U_mu(x-mu-nu) U_nu(x-nu)
    link_at(g, gauge, xmm, mu, a); link_at(g, gauge, xmm_mn, nu, b); mm<true, true>(a, b, t1);
    link_at(g, gauge, xmm_mn, mu, a); mm<false, false>(t1, a, t2);
    link_at(g, gauge, xmn, nu, a); mm<false, false>(t2, a, t1);
    for (int k = 0; k < 9; ++k) { Q.re[k] += t1.re[k]; Q.im[k] += t1.im[k]; }
    // leaf 4: U_nu(x-nu)^H U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^H
    link_at(g, gauge, xmn, nu, a); link_at(g, gauge, xmn, mu, b); mm<true, false>(a, b, t1);
    link_at(g, gauge, xpm_mn, nu, a); mm<false, false>(t1, a, t2);
    link_at(g, gauge, x, mu, a); mm<false, true>(t2, a, t1);
    for (int k = 0; k < 9; ++k) { Q.re[k] += t1.re[k]; Q.im[k] += t1.im[k]; }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            F.re[3 * i + j] = Q.re[3 * i + j] - Q.re[3 * j + i];
            F.im[3 * i + j] = Q.im[3 * i + j] + Q.im[3 * j + i];
        }
}

// in-place inverse of a dense 6x6 complex matrix, Gauss-Jordan with partial pivoting.
// Returns false if a pivot is below 1e-12 * max|entry|.
__device__ bool invert6(double (&mr)[6][6], double (&mi)[6][6])
{
    double ar[6][12], ai[6][12];
    double scale = 0;
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            ar[i][j] = mr[i][j]; ai[i][j] = mi[i][j];
            ar[i][6 + j] = (i == j) ? 1.0 : 0.0; ai[i][6 + j] = 0.0;
            scale = fmax(scale, hypot(mr[i][j], mi[i][j]));
        }
    for (int c = 0; c < 6; ++c) {
        int p = c;
        double best = ar[c][c] * ar[c][c] + ai[c][c] * ai[c][c];
        for (int i = c + 1; i < 6; ++i) {
            const double v = ar[i][c] * ar[i][c] + ai[i][c] * ai[i][c];
            if (v > best) { best = v; p = i; }
        }
        if (!(sqrt(best) > 1e-12 * scale)) return false;
        if (p != c)
            for (int j = 0; j < 12; ++j) {
                double t = ar[c][j]; ar[c][j] = ar[p][j]; ar[p][j] = t;
                t = ai[c][j]; ai[c][j] = ai[p][j]; ai[p][j] = t;
            }
        const double ir = ar[c][c] / best, ii = -ai[c][c] / best;      // 1 / pivot
        for (int j = 0; j < 12; ++j) {
            const double xr = ar[c][j], xi = ai[c][j];
            ar[c][j] = xr * ir - xi * ii;
            ai[c][j] = xr * ii + xi * ir;
        }
        for (int i = 0; i < 6; ++i) {
            if (i == c) continue;
            const double fr = ar[i][c], fi = ai[i][c];
            for (int j = 0; j < 12; ++j) {
                ar[i][j] -= fr * ar[c][j] - fi * ai[c][j];
                ai[i][j] -= fr * ai[c][j] + fi * ar[c][j];
            }
        }
    }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) { mr[i][j] = ar[i][6 + j]; mi[i][j] = ai[i][6 + j]; }
    return true;
}

template <typename T>
__global__ void build_clover_pivoted_kernel(Geom g, double csw, double m0, const T* __restrict__ gauge,
                                    T* __restrict__ clov_e, T* __restrict__ clov_o, T* __restrict__ clov_o_plain,
                                    int* singular)
{
    // clov_e: A on even sites; clov_o: A^-1 on odd sites; clov_o_plain: A itself on odd sites
    // (needed only by the full operator D = A + H).  A NULL output skips that part.
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    if (parity == 0 && !clov_e) return;
    const Coord x = coord_of(g, cb, parity);
    // dense blocks, index 3*s + c
    double ur[6][6], ui[6][6], lr[6][6], li[6][6];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            ur[i][j] = lr[i][j] = (i == j) ? m0 + 4.0 : 0.0;
            ui[i][j] = li[i][j] = 0.0;
        }
    const double kap = csw / 16.0;
    for (int k = 0; k < 3; ++k) {
        const int i = (k + 1) % 3, j = (k + 2) % 3;
        M3 Fij, Fkt;
        field_strength<T>(g, gauge, x, i, j, Fij);
        field_strength<T>(g, gauge, x, k, 3, Fkt);
        // G^-+ = i (F_ij -+ F_kt)  (Hermitian 3x3):  i*(a + ib) = -b + ia
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                const int e = 3 * a + b;
                const double gmr = -(Fij.im[e] - Fkt.im[e]), gmi = (Fij.re[e] - Fkt.re[e]);
                const double gpr = -(Fij.im[e] + Fkt.im[e]), gpi = (Fij.re[e] + Fkt.re[e]);
                if (k == 2) {            // sigma_z: diag(+G, -G)
                    ur[a][b] -= kap * gmr; ui[a][b] -= kap * gmi;
                    ur[3 + a][3 + b] += kap * gmr; ui[3 + a][3 + b] += kap * gmi;
                    lr[a][b] -= kap * gpr; li[a][b] -= kap * gpi;
                    lr[3 + a][3 + b] += kap * gpr; li[3 + a][3 + b] += kap * gpi;
                } else if (k == 0) {     // sigma_x: off-diagonal G, G
                    ur[a][3 + b] -= kap * gmr; ui[a][3 + b] -= kap * gmi;
                    ur[3 + a][b] -= kap * gmr; ui[3 + a][b] -= kap * gmi;
                    lr[a][3 + b] -= kap * gpr; li[a][3 + b] -= kap * gpi;
                    lr[3 + a][b] -= kap * gpr; li[3 + a][b] -= kap * gpi;
                } else {                 // sigma_y: [0,1] = -i G, [1,0] = +i G ;  -i*(r+ii') = i' - i r
                    ur[a][3 + b] -= kap * gmi;  ui[a][3 + b] -= kap * (-gmr);
                    ur[3 + a][b] -= kap * (-gmi); ui[3 + a][b] -= kap * gmr;
                    lr[a][3 + b] -= kap * gpi;  li[a][3 + b] -= kap * (-gpr);
                    lr[3 + a][b] -= kap * (-gpi); li[3 + a][b] -= kap * gpr;
                }
            }
    }
    T c[36];
    for (int pass = 0; pass < 2; ++pass) {
      // pass 0: the block itself (even sites -> clov_e, odd sites -> clov_o_plain);
      // pass 1: odd sites only, the inverse -> clov_o
      T* dst;
      if (pass == 0) {
          dst = parity ? clov_o_plain : clov_e;
      } else {
          if (parity == 0 || !clov_o) break;
          const bool ok1 = invert6(ur, ui);
          const bool ok2 = invert6(lr, li);
          if (!(ok1 && ok2)) atomicOr(singular, 1);
          dst = clov_o;
      }
      if (!dst) continue;
      for (int blk = 0; blk < 2; ++blk) {
        double (&mr)[6][6] = blk ? lr : ur;
        double (&mi)[6][6] = blk ? li : ui;
        double pd[36];
        for (int i = 0; i < 6; ++i) pd[i] = mr[i][i];
        for (int i = 1; i < 6; ++i)
            for (int j = 0; j < i; ++j) {
                // Hermitian part of the lower triangle (rounding-level symmetrisation)
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                pd[k] = 0.5 * (mr[i][j] + mr[j][i]);
                pd[k + 1] = 0.5 * (mi[i][j] - mi[j][i]);
            }
        if (pass == 0) {
            // the block itself: compact form (ddamg_common.cuh)
            const double delta[3] = { mr[0][0] - (m0 + 4.0), mr[1][1] - (m0 + 4.0), mr[2][2] - (m0 + 4.0) };
            T a[CLOVA_REALS];
            compact_clover_A<T>(pd, delta, a);
            store_clover_A<T>(dst, g.Vh, cb, blk, a);
        } else {
            for (int q = 0; q < 36; ++q) c[q] = (T)pd[q];
            store_clover_block<T>(dst, g.Vh, cb, blk, c);
        }
      }
    }
}


// ---- a1, fast path.  One CTA = CLOV_SITES sites x 3 thread groups; group k (warp-uniform) forms the two
// field strengths of the plane pair k  (F'_ij, F'_kt; (i, j, k) cyclic)  for its site with all 3x3
// products fully unrolled in fp64 registers (no local arrays), and leaves the two Hermitian 3x3 matrices
// G^-+_k = i (F'_ij -+ F'_kt)  in shared memory.  Groups 0 / 1 then assemble the upper / lower chirality block
//   A = [[c - kap G_z, -kap (G_x - i G_y)], [-kap (G_x + i G_y), c + kap G_z]],  c = m0 + 4, kap = csw / 16,
// directly in the packed Hermitian format and, on odd sites, invert it by an unpivoted LDL^H in registers.
// A pivot below 1e-2 * max|A_ij| (never the case for a clover block with its dominant diagonal; possible for
// an indefinite or singular block) raises *need_pivot: the host then rebuilds everything with the pivoted
// Gauss-Jordan kernel above, which also decides DDAMG_ESINGULAR (reading C6: pivot < 1e-12 ||block||).
#ifndef DDAMG_CLOV_SITES
#define DDAMG_CLOV_SITES 64
#endif
#ifndef DDAMG_CLOV_MINB
#define DDAMG_CLOV_MINB 2
#endif
constexpr int CLOV_SITES = DDAMG_CLOV_SITES;

struct M3d { double re[9], im[9]; };
struct X4 { int x, y, z, t; };

__device__ __forceinline__ X4 shift4(const Geom& g, X4 c, int mu, int d)
{
    if (mu == 0) { c.x += d; c.x = c.x < 0 ? c.x + g.L : (c.x >= g.L ? c.x - g.L : c.x); }
    else if (mu == 1) { c.y += d; c.y = c.y < 0 ? c.y + g.L : (c.y >= g.L ? c.y - g.L : c.y); }
    else if (mu == 2) { c.z += d; c.z = c.z < 0 ? c.z + g.L : (c.z >= g.L ? c.z - g.L : c.z); }
    else { c.t += d; c.t = c.t < 0 ? c.t + g.T : (c.t >= g.T ? c.t - g.T : c.t); }
    return c;
}

// links are re-read by the neighbouring sites' leaves: cacheable loads (not the streaming ones of the hot path)
__device__ __forceinline__ void link_cached(const Geom& g, const float* __restrict__ gauge, const X4& c, int mu, M3d& m)
{
    const int par = (c.x + c.y + c.z + c.t) & 1;
    const int cb = (c.x >> 1) + g.Lh * (c.y + g.L * (c.z + g.L * c.t));
    const float* blk = gauge + ((size_t)par * 4 + mu) * (size_t)18 * g.Vh;
    const float4* p4 = reinterpret_cast<const float4*>(blk) + cb;
    float u[18];
#pragma unroll
    for (int k = 0; k < 4; ++k) unpack(__ldg(p4 + (size_t)k * g.Vh), &u[4 * k]);
    const float2 v = __ldg(reinterpret_cast<const float2*>(blk + (size_t)16 * g.Vh) + cb);
    u[16] = v.x; u[17] = v.y;
#pragma unroll
    for (int k = 0; k < 9; ++k) { m.re[k] = (double)u[2 * k]; m.im[k] = (double)u[2 * k + 1]; }
}
__device__ __forceinline__ void link_cached(const Geom& g, const double* __restrict__ gauge, const X4& c, int mu, M3d& m)
{
    const int par = (c.x + c.y + c.z + c.t) & 1;
    const int cb = (c.x >> 1) + g.Lh * (c.y + g.L * (c.z + g.L * c.t));
    const double2* p = reinterpret_cast<const double2*>(gauge + ((size_t)par * 4 + mu) * (size_t)18 * g.Vh) + cb;
#pragma unroll
    for (int k = 0; k < 9; ++k) { const double2 v = __ldg(p + (size_t)k * g.Vh); m.re[k] = v.x; m.im[k] = v.y; }
}

// c = op(a) * op(b), fully unrolled (every index is a compile-time constant: registers only)
template <bool DA, bool DB>
__device__ __forceinline__ void mm_u(const M3d& a, const M3d& b, M3d& c)
{
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            double sr = 0.0, si = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int ia = DA ? 3 * k + i : 3 * i + k;
                const int ib = DB ? 3 * j + k : 3 * k + j;
                const double ar = a.re[ia], ai = DA ? -a.im[ia] : a.im[ia];
                const double br = b.re[ib], bi = DB ? -b.im[ib] : b.im[ib];
                sr = fma(ar, br, sr); sr = fma(-ai, bi, sr);
                si = fma(ar, bi, si); si = fma(ai, br, si);
            }
            c.re[3 * i + j] = sr;
            c.im[3 * i + j] = si;
        }
}

// Q += op(U1) op(U2) op(U3) op(U4) with U_n = U_{d_n}(s_n)
template <bool D1, bool D2, bool D3, bool D4, typename T>
__device__ __forceinline__ void leaf(const Geom& g, const T* __restrict__ gauge, const X4& s1, int d1, const X4& s2, int d2,
                                     const X4& s3, int d3, const X4& s4, int d4, M3d& Q)
{
    M3d a, b, t;
    link_cached(g, gauge, s1, d1, a);
    link_cached(g, gauge, s2, d2, b);
    mm_u<D1, D2>(a, b, t);
    link_cached(g, gauge, s3, d3, a);
    mm_u<false, D3>(t, a, b);
    link_cached(g, gauge, s4, d4, a);
    mm_u<false, D4>(b, a, t);
#pragma unroll
    for (int k = 0; k < 9; ++k) { Q.re[k] += t.re[k]; Q.im[k] += t.im[k]; }
}

// F'_{mu nu}(x) = Q - Q^H (anti-Hermitian), Q = sum of the four leaves at x (reading R4).  Returned as the 9 reals
// f[0..2] = Im F_aa,  f[3 + 2 e], f[4 + 2 e] = Re, Im of the strictly-lower entries e = (1,0), (2,0), (2,1).
template <typename T>
__device__ __forceinline__ void field_strength_u(const Geom& g, const T* __restrict__ gauge, const X4& x, int mu, int nu,
                                                 double (&f)[9])
{
    M3d Q;
#pragma unroll
    for (int k = 0; k < 9; ++k) Q.re[k] = Q.im[k] = 0.0;
    const X4 xpm = shift4(g, x, mu, +1), xpn = shift4(g, x, nu, +1);
    const X4 xmm = shift4(g, x, mu, -1), xmn = shift4(g, x, nu, -1);
    const X4 xmm_pn = shift4(g, xmm, nu, +1), xmm_mn = shift4(g, xmm, nu, -1), xpm_mn = shift4(g, xpm, nu, -1);
    leaf<false, false, true, true>(g, gauge, x, mu, xpm, nu, xpn, mu, x, nu, Q);           // U_mu(x) U_nu(x+mu) U_mu(x+nu)^H U_nu(x)^H
    leaf<false, true, true, false>(g, gauge, x, nu, xmm_pn, mu, xmm, nu, xmm, mu, Q);      // U_nu(x) U_mu(x-mu+nu)^H U_nu(x-mu)^H U_mu(x-mu)
    leaf<true, true, false, false>(g, gauge, xmm, mu, xmm_mn, nu, xmm_mn, mu, xmn, nu, Q); // U_mu(x-mu)^H U_nu(x-mu-nu)^H U_mu(x-mu-nu) U_nu(x-nu)
    leaf<true, false, false, true>(g, gauge, xmn, nu, xmn, mu, xpm_mn, nu, x, mu, Q);      // U_nu(x-nu)^H U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^H
#pragma unroll
    for (int a = 0; a < 3; ++a) f[a] = 2.0 * Q.im[4 * a];
    f[3] = Q.re[3] - Q.re[1]; f[4] = Q.im[3] + Q.im[1];      // (1,0)
    f[5] = Q.re[6] - Q.re[2]; f[6] = Q.im[6] + Q.im[2];      // (2,0)
    f[7] = Q.re[7] - Q.re[5]; f[8] = Q.im[7] + Q.im[5];      // (2,1)
}

// packed Hermitian 6x6 (6 real diagonal entries, 15 complex strictly-lower entries row by row)
__host__ __device__ constexpr int pk(int i, int j) { return 6 + 2 * (i * (i - 1) / 2 + j); }

// In-place inverse of a packed Hermitian 6x6 by unpivoted LDL^H; false if a pivot is below 1e-2 * max|entry|.
__device__ __forceinline__ bool invert6_ldl(double (&p)[36])
{
    double scale = 0.0;
#pragma unroll
    for (int i = 0; i < 6; ++i) scale = fmax(scale, fabs(p[i]));
#pragma unroll
    for (int k = 6; k < 36; ++k) scale = fmax(scale, fabs(p[k]));
    // every loop below has compile-time bounds 0..5 and the triangular structure is expressed by guards that
    // fold away after unrolling, so that all arrays stay in registers
    double Lr[6][6], Li[6][6], D[6], Di[6];
    bool ok = true;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        double d = p[j];
#pragma unroll
        for (int k = 0; k < 6; ++k)
            if (k < j) d -= (Lr[j][k] * Lr[j][k] + Li[j][k] * Li[j][k]) * D[k];
        D[j] = d;
        ok = ok && (fabs(d) > 1e-2 * scale);
        Di[j] = 1.0 / d;
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            if (i > j) {
                double sr = p[pk(i, j)], si = p[pk(i, j) + 1];
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    if (k < j) {
                        // L_ik D_k conj(L_jk)
                        const double tr = Lr[i][k] * D[k], ti = Li[i][k] * D[k];
                        sr -= tr * Lr[j][k] + ti * Li[j][k];
                        si -= ti * Lr[j][k] - tr * Li[j][k];
                    }
                }
                Lr[i][j] = sr * Di[j];
                Li[i][j] = si * Di[j];
            }
        }
    }
    // M = L^-1 (unit lower triangular), column by column
    double Mr[6][6], Mi[6][6];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            if (i > j) {
                double sr = Lr[i][j], si = Li[i][j];
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    if (k > j && k < i) {
                        sr += Lr[i][k] * Mr[k][j] - Li[i][k] * Mi[k][j];
                        si += Lr[i][k] * Mi[k][j] + Li[i][k] * Mr[k][j];
                    }
                }
                Mr[i][j] = -sr;
                Mi[i][j] = -si;
            }
        }
    }
    // A^-1 = M^H D^-1 M:  (i, j), i >= j:  sum_{k >= i} conj(M_ki) M_kj / D_k,  M_kk = 1
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        double d = Di[i];
#pragma unroll
        for (int k = 0; k < 6; ++k)
            if (k > i) d += (Mr[k][i] * Mr[k][i] + Mi[k][i] * Mi[k][i]) * Di[k];
        p[i] = d;
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            if (j < i) {
                double sr = Mr[i][j] * Di[i], si = Mi[i][j] * Di[i];          // k = i term: conj(1) M_ij / D_i
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    if (k > i) {
                        const double tr = Mr[k][j] * Di[k], ti = Mi[k][j] * Di[k];
                        sr += Mr[k][i] * tr + Mi[k][i] * ti;                  // conj(M_ki) * M_kj
                        si += Mr[k][i] * ti - Mi[k][i] * tr;
                    }
                }
                p[pk(i, j)] = sr;
                p[pk(i, j) + 1] = si;
            }
        }
    }
    return ok;
}

template <typename T>
__global__ void __launch_bounds__(3 * CLOV_SITES, DDAMG_CLOV_MINB)
build_clover_kernel(Geom g, double csw, double m0, const T* __restrict__ gauge,
                    T* __restrict__ clov_e, T* __restrict__ clov_o, T* __restrict__ clov_o_plain, int* need_pivot)
{
    // clov_e: A on even sites; clov_o: A^-1 on odd sites; clov_o_plain: A itself on odd sites
    // (needed only by the full operator D = A + H).  A NULL output skips that part.
    __shared__ double G[2][3][9][CLOV_SITES];        // [-+][k][entry][site]: diag 0..2, lower (re, im) 3..8
    const int sl = threadIdx.x % CLOV_SITES, k = threadIdx.x / CLOV_SITES;
    const int idx = blockIdx.x * CLOV_SITES + sl;
    const bool live = idx < 2 * g.Vh;
    const int parity = live ? idx / g.Vh : 0, cb = live ? idx % g.Vh : 0;
    const bool wanted = live && (parity == 1 ? (clov_o || clov_o_plain) : clov_e != nullptr);
    if (wanted) {
        const Site s = site_of_cb(g, cb, parity);
        X4 x;
        x.x = 2 * s.xh + s.q; x.y = s.y; x.z = s.z; x.t = s.t;
        const int i = k == 2 ? 0 : k + 1, j = k == 0 ? 2 : k - 1;      // (i, j, k) cyclic
        double fij[9], fkt[9];
        field_strength_u<T>(g, gauge, x, i, j, fij);
        field_strength_u<T>(g, gauge, x, k, 3, fkt);
        // G = i F:  diag = -Im F_aa;  lower: Re G = -Im F, Im G = Re F
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            G[0][k][a][sl] = -(fij[a] - fkt[a]);
            G[1][k][a][sl] = -(fij[a] + fkt[a]);
        }
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            G[0][k][3 + 2 * e][sl] = -(fij[4 + 2 * e] - fkt[4 + 2 * e]);
            G[0][k][4 + 2 * e][sl] = fij[3 + 2 * e] - fkt[3 + 2 * e];
            G[1][k][3 + 2 * e][sl] = -(fij[4 + 2 * e] + fkt[4 + 2 * e]);
            G[1][k][4 + 2 * e][sl] = fij[3 + 2 * e] + fkt[3 + 2 * e];
        }
    }
    __syncthreads();
    if (!wanted || k >= 2) return;
    const int h = k;                                  // chirality block: 0 = upper (G^-), 1 = lower (G^+)
    double gx[9], gy[9], gz[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) { gx[e] = G[h][0][e][sl]; gy[e] = G[h][1][e][sl]; gz[e] = G[h][2][e][sl]; }
    const double kap = csw / 16.0, c0 = m0 + 4.0;
    double p[36];
#pragma unroll
    for (int a = 0; a < 3; ++a) { p[a] = c0 - kap * gz[a]; p[3 + a] = c0 + kap * gz[a]; }
    // diagonal 3x3 blocks: -+ kap G_z (strictly-lower entries (1,0), (2,0), (2,1))
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int a = e == 0 ? 1 : 2, b = e == 2 ? 1 : 0;
        p[pk(a, b)] = -kap * gz[3 + 2 * e];         p[pk(a, b) + 1] = -kap * gz[4 + 2 * e];
        p[pk(3 + a, 3 + b)] = kap * gz[3 + 2 * e];  p[pk(3 + a, 3 + b) + 1] = kap * gz[4 + 2 * e];
    }
    // lower-left 3x3 block (3 + a, b) = -kap (G_x + i G_y)[a][b]
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            double xr, xi, yr, yi;
            if (a == b) { xr = gx[a]; xi = 0.0; yr = gy[a]; yi = 0.0; }
            else {
                const int hi = a > b ? a : b, lo = a > b ? b : a;
                const int e = hi == 1 ? 0 : (lo == 0 ? 1 : 2);
                const double sgn = a > b ? 1.0 : -1.0;               // upper entries are the conjugates
                xr = gx[3 + 2 * e]; xi = sgn * gx[4 + 2 * e];
                yr = gy[3 + 2 * e]; yi = sgn * gy[4 + 2 * e];
            }
            p[pk(3 + a, b)] = -kap * (xr - yi);
            p[pk(3 + a, b) + 1] = -kap * (xi + yr);
        }
    T c[36];
    T* plain = parity ? clov_o_plain : clov_e;
    if (plain) {
        // the block itself: compact form (ddamg_common.cuh), delta_a = A_aa - c0 formed before rounding
        const double delta[3] = { -kap * gz[0], -kap * gz[1], -kap * gz[2] };
        T a[CLOVA_REALS];
        compact_clover_A<T>(p, delta, a);
        store_clover_A<T>(plain, g.Vh, cb, h, a);
    }
    if (parity == 1 && clov_o) {
        if (!invert6_ldl(p)) atomicOr(need_pivot, 1);
#pragma unroll
        for (int q = 0; q < 36; ++q) c[q] = (T)p[q];
        store_clover_block<T>(clov_o, g.Vh, cb, h, c);
    }
}

template <typename T>
void launch_build_clover(const Geom& g, double csw, double m0, const void* gauge, void* clov_e, void* clov_o,
                         void* clov_o_plain, int* need_pivot_flag, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    build_clover_kernel<T><<<(n + CLOV_SITES - 1) / CLOV_SITES, 3 * CLOV_SITES, 0, st>>>(
        g, csw, m0, (const T*)gauge, (T*)clov_e, (T*)clov_o, (T*)clov_o_plain, need_pivot_flag);
}
template void launch_build_clover<float>(const Geom&, double, double, const void*, void*, void*, void*, int*, cudaStream_t);
template void launch_build_clover<double>(const Geom&, double, double, const void*, void*, void*, void*, int*, cudaStream_t);

template <typename T>
void launch_build_clover_pivoted(const Geom& g, double csw, double m0, const void* gauge, void* clov_e, void* clov_o,
                                 void* clov_o_plain, int* singular_flag, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    build_clover_pivoted_kernel<T><<<(n + 63) / 64, 64, 0, st>>>(g, csw, m0, (const T*)gauge, (T*)clov_e, (T*)clov_o,
                                                                  (T*)clov_o_plain, singular_flag);
}
template void launch_build_clover_pivoted<float>(const Geom&, double, double, const void*, void*, void*, void*, int*, cudaStream_t);
template void launch_build_clover_pivoted<double>(const Geom&, double, double, const void*, void*, void*, void*, int*, cudaStream_t);

// ------------------------------------------------------------------ debug: dense clover out
template <typename T>
__global__ void get_clover_kernel(Geom g, T c0, const T* __restrict__ clov_e, const T* __restrict__ clov_o,
                                  T* __restrict__ A_nat, T* __restrict__ Ainv_nat)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    const size_t n = nat_of(g, coord_of(g, cb, parity));
    T* mine = parity ? Ainv_nat : A_nat;
    T* other = parity ? A_nat : Ainv_nat;
    if (other)
        for (int k = 0; k < 144; ++k) other[n * 144 + k] = 0;
    if (!mine) return;
    const T* src = parity ? clov_o : clov_e;
    for (int blk = 0; blk < 2; ++blk) {
        T c[36];
        if (parity) load_clover_block<T>(src, g.Vh, cb, blk, c);      // A_oo^-1: packed
        else load_clover_A<T>(src, g.Vh, cb, blk, c0, c);             // A_ee: compact
        T* out = mine + n * 144 + blk * 72;
        for (int i = 0; i < 6; ++i)
            for (int j = 0; j < 6; ++j) {
                T re, im;
                if (i == j) { re = c[i]; im = 0; }
                else if (j < i) { const int k = 6 + 2 * (i * (i - 1) / 2 + j); re = c[k]; im = c[k + 1]; }
                else { const int k = 6 + 2 * (j * (j - 1) / 2 + i); re = c[k]; im = -c[k + 1]; }
                out[2 * (6 * i + j)] = re;
                out[2 * (6 * i + j) + 1] = im;
            }
    }
}

template <typename T>
void launch_get_clover(const Geom& g, double c0, const void* clov_e, const void* clov_o, void* A_nat, void* Ainv_nat,
                       cudaStream_t st)
{
    const int n = 2 * g.Vh;
    get_clover_kernel<T><<<(n + 127) / 128, 128, 0, st>>>(g, (T)c0, (const T*)clov_e, (const T*)clov_o, (T*)A_nat,
                                                           (T*)Ainv_nat);
}
template void launch_get_clover<float>(const Geom&, double, const void*, const void*, void*, void*, cudaStream_t);
template void launch_get_clover<double>(const Geom&, double, const void*, const void*, void*, void*, cudaStream_t);

}  // namespace ddamg

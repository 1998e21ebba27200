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
template <typename Tin, typename T>
__global__ void pack_gauge_kernel(Geom g, int bc, const Tin* __restrict__ U, T* __restrict__ gauge)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    const Coord c = coord_of(g, cb, parity);
    const size_t n = nat_of(g, c);
    const size_t lblk = (size_t)18 * g.Vh;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        T u[18];
        const T sgn = (bc == 1 && mu == 3 && c.x[3] == g.T - 1) ? (T)-1 : (T)1;
#pragma unroll
        for (int k = 0; k < 18; ++k) u[k] = sgn * (T)U[(n * 4 + mu) * 18 + k];
        store_link(gauge + ((size_t)parity * 4 + mu) * lblk, g.Vh, cb, u);
    }
}

template <typename Tin, typename T>
void launch_pack_gauge(const Geom& g, int bc, const void* U_nat, void* gauge, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    pack_gauge_kernel<Tin, T><<<(n + 255) / 256, 256, 0, st>>>(g, bc, (const Tin*)U_nat, (T*)gauge);
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
            for (int k = 12; k < 18; ++k) dev = fmaxf(dev, fabsf((float)(v[k] - u[k])));
            store_link12(gauge12 + ((size_t)parity * 4 + mu) * (size_t)12 * g.Vh, g.Vh, cb, u);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o));
    if ((threadIdx.x & 31) == 0 && dev > 0.f) atomicMax(dev_max_bits, __float_as_uint(dev));
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
template <typename T>
__global__ void pack_spinor_kernel(Geom g, const T* __restrict__ nat, T* __restrict__ xe, T* __restrict__ xo)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    T* dst = parity ? xo : xe;
    if (!dst) return;
    const size_t n = nat_of(g, coord_of(g, cb, parity));
    T s[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) s[k] = nat[n * 24 + k];
    store_spinor<T>(dst, g.Vh, cb, s);
}

template <typename T>
__global__ void unpack_spinor_kernel(Geom g, const T* __restrict__ xe, const T* __restrict__ xo, T* __restrict__ nat)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx / g.Vh, cb = idx % g.Vh;
    const T* src = parity ? xo : xe;
    const size_t n = nat_of(g, coord_of(g, cb, parity));
    T s[24];
    if (src) {
        load_spinor<T>(src, g.Vh, cb, s);
    } else {
#pragma unroll
        for (int k = 0; k < 24; ++k) s[k] = 0;
    }
#pragma unroll
    for (int k = 0; k < 24; ++k) nat[n * 24 + k] = s[k];
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
// X[plane][cb * nrhs + r] = halves[r][plane][cb]  (TO_BATCH) or the inverse.  One thread per
// vector of the batch; writes (TO_BATCH) / reads (inverse) of the batch are contiguous.
template <typename T, bool TO_BATCH>
__global__ void batch_interleave_kernel(int Vh, int nrhs, typename VecOf<T>::type* __restrict__ halves,
                                        typename VecOf<T>::type* __restrict__ X)
{
    constexpr int NP = 24 / VecOf<T>::N;
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
template <typename T>
void launch_batch_interleave(const Geom& g, int nrhs, bool to_batch, void* halves, void* X, cudaStream_t st)
{
    using V = typename VecOf<T>::type;
    const size_t n = (size_t)g.Vh * nrhs * (24 / VecOf<T>::N);
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (to_batch) batch_interleave_kernel<T, true><<<grid, 256, 0, st>>>(g.Vh, nrhs, (V*)halves, (V*)X);
    else batch_interleave_kernel<T, false><<<grid, 256, 0, st>>>(g.Vh, nrhs, (V*)halves, (V*)X);
}
template void launch_batch_interleave<float>(const Geom&, int, bool, void*, void*, cudaStream_t);
template void launch_batch_interleave<double>(const Geom&, int, bool, void*, void*, cudaStream_t);

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
__global__ void build_clover_kernel(Geom g, double csw, double m0, const T* __restrict__ gauge,
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
        for (int i = 0; i < 6; ++i) c[i] = (T)mr[i][i];
        for (int i = 1; i < 6; ++i)
            for (int j = 0; j < i; ++j) {
                // Hermitian part of the lower triangle (rounding-level symmetrisation)
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                c[k] = (T)(0.5 * (mr[i][j] + mr[j][i]));
                c[k + 1] = (T)(0.5 * (mi[i][j] - mi[j][i]));
            }
        store_clover_block<T>(dst, g.Vh, cb, blk, c);
      }
    }
}

template <typename T>
void launch_build_clover(const Geom& g, double csw, double m0, const void* gauge, void* clov_e, void* clov_o,
                         void* clov_o_plain, int* singular_flag, cudaStream_t st)
{
    const int n = 2 * g.Vh;
    build_clover_kernel<T><<<(n + 63) / 64, 64, 0, st>>>(g, csw, m0, (const T*)gauge, (T*)clov_e, (T*)clov_o,
                                                          (T*)clov_o_plain, singular_flag);
}
template void launch_build_clover<float>(const Geom&, double, double, const void*, void*, void*, void*, int*, cudaStream_t);
template void launch_build_clover<double>(const Geom&, double, double, const void*, void*, void*, void*, int*, cudaStream_t);

// ------------------------------------------------------------------ debug: dense clover out
template <typename T>
__global__ void get_clover_kernel(Geom g, const T* __restrict__ clov_e, const T* __restrict__ clov_o,
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
        load_clover_block<T>(src, g.Vh, cb, blk, c);
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
void launch_get_clover(const Geom& g, const void* clov_e, const void* clov_o, void* A_nat, void* Ainv_nat,
                       cudaStream_t st)
{
    const int n = 2 * g.Vh;
    get_clover_kernel<T><<<(n + 127) / 128, 128, 0, st>>>(g, (const T*)clov_e, (const T*)clov_o, (T*)A_nat,
                                                           (T*)Ainv_nat);
}
template void launch_get_clover<float>(const Geom&, const void*, const void*, void*, void*, cudaStream_t);
template void launch_get_clover<double>(const Geom&, const void*, const void*, void*, void*, cudaStream_t);

}  // namespace ddamg

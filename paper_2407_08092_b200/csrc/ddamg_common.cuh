// ddamg_common.cuh -- geometry, native (checkerboard SoA) layout and vector access.
//
// Native layout:
//   * site of parity p with coordinates (x,y,z,t):  cb = (x>>1) + Lh*(y + L*(z + L*t)),
//     Lh = L/2  (== natural index >> 1 because L is even and x is fastest)
//   * half-lattice spinor: 24/NV planes of Vh 16-byte vectors, plane j = reals NV*j..
//   * gauge: per (parity, mu) one block of 18*Vh reals holding U_mu(x) for the Vh sites of
//     that parity: fp32 = 4 planes of float4 (reals 0..15) + 1 plane of float2 (reals 16,17);
//     fp64 = 9 planes of double2; reals are row-major (row, col, re/im)
//   * clover: per parity 2 blocks/site, each block 36 reals = 6 real diagonal entries then
//     the 15 complex strictly-lower entries (1,0),(2,0),(2,1),(3,0),...,(5,4); stored as
//     72/NV planes of Vh vectors (block 0 first).  This is the format of the INVERSES (A_oo^-1);
//     the blocks themselves (A_ee, A_oo) use the compact 28-real form of load_clover_A below
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ddamg {

struct Geom {
    int L, T, Lh;        // Lh = L/2
    int Vh;              // sites per parity
    int sy, sz, st;      // cb strides of +1 in y, z, t:  Lh, Lh*L, Lh*L*L
};

template <typename T> struct VecOf;
template <> struct VecOf<float>  { using type = float4;  static constexpr int N = 4; };
template <> struct VecOf<double> { using type = double2; static constexpr int N = 2; };

// ----------------------------------------------------------------- cache-hinted access
// Spinor neighbours are re-read up to 8 times by different CTAs: keep them cacheable
// (read-only path).  Gauge links and clover blocks are read exactly once per kernel:
// stream them with an evict-first policy so that they do not push spinors out of L2.

__device__ __forceinline__ float4 ld_reuse(const float4* p) { return __ldg(p); }
__device__ __forceinline__ double2 ld_reuse(const double2* p) { return __ldg(p); }
__device__ __forceinline__ float4 ld_stream(const float4* p) { return __ldcs(p); }
__device__ __forceinline__ float2 ld_stream(const float2* p) { return __ldcs(p); }
__device__ __forceinline__ double2 ld_stream(const double2* p) { return __ldcs(p); }

__device__ __forceinline__ void unpack(const float4& v, float* r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void unpack(const double2& v, double* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ float4 pack(const float* r) { return make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ double2 pack(const double* r) { return make_double2(r[0], r[1]); }

// ----------------------------------------------------------------- packed fp32 pairs
// Blackwell executes two fp32 operations per instruction on an aligned register pair (FADD2 /
// FMUL2 / FFMA2, PTX add/mul/fma.rn.f32x2); one operand may be a plain 32-bit register that the
// instruction broadcasts to both lanes, with a sign modifier, at no extra cost.  Each lane is an
// ordinary IEEE fp32 operation, so a packed evaluation is bit-identical to the scalar one as
// long as the order of operations per element is the same.  P2 carries two independent values
// through the hopping / clover code: the two spin components of a half spinor (single rhs), or
// the same spinor component of two right-hand sides (multi-rhs).
struct P2 { float2 v; };
__device__ __forceinline__ P2 mkp(float a, float b) { P2 r; r.v = make_float2(a, b); return r; }
__device__ __forceinline__ P2 operator+(P2 a, P2 b) { P2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ P2 operator-(P2 a, P2 b) { P2 r; r.v = __fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y)); return r; }
__device__ __forceinline__ P2 operator-(P2 a) { return mkp(-a.v.x, -a.v.y); }

// value-type generic arithmetic: S = float, double (one value) or P2 (two fp32 values); the
// coefficient c is always a scalar of the storage precision (a link / clover entry, omega, 1/2)
__device__ __forceinline__ float vmul(float c, float a) { return c * a; }
__device__ __forceinline__ double vmul(double c, double a) { return c * a; }
__device__ __forceinline__ P2 vmul(float c, P2 a) { P2 r; r.v = __fmul2_rn(make_float2(c, c), a.v); return r; }
__device__ __forceinline__ float vfma(float c, float a, float b) { return fmaf(c, a, b); }
__device__ __forceinline__ double vfma(double c, double a, double b) { return fma(c, a, b); }
__device__ __forceinline__ P2 vfma(float c, P2 a, P2 b) { P2 r; r.v = __ffma2_rn(make_float2(c, c), a.v, b.v); return r; }
__device__ __forceinline__ float vzero(float) { return 0.f; }
__device__ __forceinline__ double vzero(double) { return 0.0; }
__device__ __forceinline__ P2 vzero(P2) { return mkp(0.f, 0.f); }
// |r|^2 accumulated per lane in fp64 (nrm[0]: the value / lane 0, nrm[1]: lane 1 of a P2)
__device__ __forceinline__ void vnorm_add(float r, double (&nrm)[2]) { nrm[0] += (double)r * (double)r; }
__device__ __forceinline__ void vnorm_add(double r, double (&nrm)[2]) { nrm[0] += r * r; }
__device__ __forceinline__ void vnorm_add(P2 r, double (&nrm)[2])
{
    nrm[0] += (double)r.v.x * (double)r.v.x;
    nrm[1] += (double)r.v.y * (double)r.v.y;
}

// 24 reals of one site of a native half-lattice spinor
template <typename T, bool STREAM = false>
__device__ __forceinline__ void load_spinor(const T* __restrict__ base, int Vh, int cb, T (&s)[24])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    const V* p = reinterpret_cast<const V*>(base) + cb;
#pragma unroll
    for (int k = 0; k < 24 / N; ++k) {
        V v = STREAM ? ld_stream(p + (size_t)k * Vh) : ld_reuse(p + (size_t)k * Vh);
        unpack(v, &s[k * N]);
    }
}

template <typename T>
__device__ __forceinline__ void store_spinor(T* __restrict__ base, int Vh, int cb, const T (&s)[24])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    V* p = reinterpret_cast<V*>(base) + cb;
#pragma unroll
    for (int k = 0; k < 24 / N; ++k) p[(size_t)k * Vh] = pack(&s[k * N]);
}

// Multi-rhs batch of fp32 spinors, two right-hand sides per thread: the
// batch is stored as 12 half-planes of float4; half-plane h, vector index cb * npairs + p holds
// complex number h of the site for the rhs pair p as (re of rhs 2p, re of rhs 2p+1, im of rhs 2p,
// im of rhs 2p+1), so that one 16-byte load leaves two ready-made register pairs.  Vs = Vh * npairs.
template <typename T, bool STREAM = false>
__device__ __forceinline__ void load_spinor(const float* __restrict__ base, int Vs, int idx, P2 (&s)[24])
{
    const float4* p = reinterpret_cast<const float4*>(base) + idx;
#pragma unroll
    for (int h = 0; h < 12; ++h) {
        const float4 v = STREAM ? ld_stream(p + (size_t)h * Vs) : ld_reuse(p + (size_t)h * Vs);
        s[2 * h] = mkp(v.x, v.y);
        s[2 * h + 1] = mkp(v.z, v.w);
    }
}
template <typename T>
__device__ __forceinline__ void store_spinor(float* __restrict__ base, int Vs, int idx, const P2 (&s)[24])
{
    float4* p = reinterpret_cast<float4*>(base) + idx;
#pragma unroll
    for (int h = 0; h < 12; ++h) p[(size_t)h * Vs] = make_float4(s[2 * h].v.x, s[2 * h].v.y, s[2 * h + 1].v.x, s[2 * h + 1].v.y);
}

// 18 reals of one link; blk = start of the (parity, mu) block
__device__ __forceinline__ void load_link(const float* __restrict__ blk, int Vh, int cb, float (&u)[18])
{
    const float4* p4 = reinterpret_cast<const float4*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 4; ++k) unpack(ld_stream(p4 + (size_t)k * Vh), &u[4 * k]);
    const float2 v = ld_stream(reinterpret_cast<const float2*>(blk + (size_t)16 * Vh) + cb);
    u[16] = v.x; u[17] = v.y;
}
__device__ __forceinline__ void load_link(const double* __restrict__ blk, int Vh, int cb, double (&u)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 9; ++k) unpack(ld_stream(p + (size_t)k * Vh), &u[2 * k]);
}
__device__ __forceinline__ void store_link(float* __restrict__ blk, int Vh, int cb, const float (&u)[18])
{
    float4* p4 = reinterpret_cast<float4*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 4; ++k) p4[(size_t)k * Vh] = pack(&u[4 * k]);
    reinterpret_cast<float2*>(blk + (size_t)16 * Vh)[cb] = make_float2(u[16], u[17]);
}
__device__ __forceinline__ void store_link(double* __restrict__ blk, int Vh, int cb, const double (&u)[18])
{
    double2* p = reinterpret_cast<double2*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 9; ++k) p[(size_t)k * Vh] = pack(&u[2 * k]);
}

// Two-row (12-real) link storage (option "gauge_recon" = 12; SURVEY.md 8(d) "two-row link
// storage"): per (parity, mu) a block of 12*Vh reals holding rows 0 and 1 of U_mu(x)
// (fp32: 3 planes of float4, fp64: 6 planes of double2).  For U in SU(3) the third row is
// conj(row0 x row1); the antiperiodic sign folded into the stored rows of U_t(T-1) does not
// survive the cross product, so the caller passes sgn = -1 for those links.
template <typename T>
__device__ __forceinline__ void reconstruct_row2(T sgn, T (&u)[18])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        // row0[a] * row1[b] - row0[b] * row1[a], conjugated
        T re = u[2 * a] * u[6 + 2 * b];
        re = fma(-u[2 * a + 1], u[6 + 2 * b + 1], re);
        re = fma(-u[2 * b], u[6 + 2 * a], re);
        re = fma(u[2 * b + 1], u[6 + 2 * a + 1], re);
        T im = u[2 * a] * u[6 + 2 * b + 1];
        im = fma(u[2 * a + 1], u[6 + 2 * b], im);
        im = fma(-u[2 * b], u[6 + 2 * a + 1], im);
        im = fma(-u[2 * b + 1], u[6 + 2 * a], im);
        u[12 + 2 * c] = sgn * re;
        u[12 + 2 * c + 1] = -sgn * im;
    }
}
__device__ __forceinline__ void load_link12(const float* __restrict__ blk, int Vh, int cb, float sgn, float (&u)[18])
{
    const float4* p4 = reinterpret_cast<const float4*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 3; ++k) unpack(ld_stream(p4 + (size_t)k * Vh), &u[4 * k]);
    reconstruct_row2<float>(sgn, u);
}
__device__ __forceinline__ void load_link12(const double* __restrict__ blk, int Vh, int cb, double sgn, double (&u)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 6; ++k) unpack(ld_stream(p + (size_t)k * Vh), &u[2 * k]);
    reconstruct_row2<double>(sgn, u);
}
__device__ __forceinline__ void store_link12(float* __restrict__ blk, int Vh, int cb, const float (&u)[18])
{
    float4* p4 = reinterpret_cast<float4*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 3; ++k) p4[(size_t)k * Vh] = pack(&u[4 * k]);
}
__device__ __forceinline__ void store_link12(double* __restrict__ blk, int Vh, int cb, const double (&u)[18])
{
    double2* p = reinterpret_cast<double2*>(blk) + cb;
#pragma unroll
    for (int k = 0; k < 6; ++k) p[(size_t)k * Vh] = pack(&u[2 * k]);
}

// load modes of the clover accessors: LD_REUSE = global, read-only path, cacheable (re-read by the same CTA);
// LD_STREAM = global, read once per kernel (evict-first); LD_PLAIN = ordinary load (shared memory: the SAP
// block kernel's staged blocks).  (false / true convert to LD_REUSE / LD_STREAM.)
enum { LD_REUSE = 0, LD_STREAM = 1, LD_PLAIN = 2 };
template <int MODE, typename V>
__device__ __forceinline__ V ld_mode(const V* p)
{
    if (MODE == LD_STREAM) return ld_stream(p);
    if (MODE == LD_REUSE) return ld_reuse(p);
    return *p;
}
// 36 reals of clover block b (0/1) of one site
template <typename T, int MODE = LD_STREAM>
__device__ __forceinline__ void load_clover_block(const T* __restrict__ base, int Vh, int cb, int b, T (&c)[36])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    const V* p = reinterpret_cast<const V*>(base) + (size_t)b * (36 / N) * Vh + cb;
#pragma unroll
    for (int k = 0; k < 36 / N; ++k) unpack(ld_mode<MODE>(p + (size_t)k * Vh), &c[k * N]);
}
template <typename T>
__device__ __forceinline__ void store_clover_block(T* __restrict__ base, int Vh, int cb, int b, const T (&c)[36])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    V* p = reinterpret_cast<V*>(base) + (size_t)b * (36 / N) * Vh + cb;
#pragma unroll
    for (int k = 0; k < 36 / N; ++k) p[(size_t)k * Vh] = pack(&c[k * N]);
}

// Compact storage of the clover blocks THEMSELVES (A_ee, and A_oo for the full operator; never the
// inverses).  In the chiral basis a block is  A_+- = c0 1_6 + sum_k sigma_k (x) G_k  with c0 = m0 + 4
// and G_k Hermitian 3x3 (R4: the clover term is traceless in spin), i.e. with rows /
// columns ordered (spin, colour)
//        [ c0 + G_3      M    ]
//        [   M^H      c0 - G_3 ]          M = G_1 - i G_2
// so the lower-right 3x3 block is 2 c0 - (upper-left block) and need not be stored: 27 reals
// instead of 36.  Stored per block (CLOVA_REALS = 28 with one pad real: 7 float4 / 14 double2
// planes): delta_i = A_ii - c0 (i = 0..2), the lower entries (1,0) (2,0) (2,1) of the upper-left
// block, the 9 complex entries (3+i, j) of M^H, pad.  224 instead of 288 bytes per site in fp32.
// load_clover_A expands into the ordinary packed 36 (6 real diagonal + 15 complex lower entries):
// 3 additions, 3 subtractions, sign flips folded into the consumers' operands.
constexpr int CLOVA_REALS = 28;
template <typename T, int MODE = LD_STREAM>
__device__ __forceinline__ void load_clover_A(const T* __restrict__ base, int Vh, int cb, int b, T c0, T (&c)[36])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    const V* p = reinterpret_cast<const V*>(base) + (size_t)b * (CLOVA_REALS / N) * Vh + cb;
    T a[CLOVA_REALS];
#pragma unroll
    for (int k = 0; k < CLOVA_REALS / N; ++k) unpack(ld_mode<MODE>(p + (size_t)k * Vh), &a[k * N]);
#pragma unroll
    for (int i = 0; i < 3; ++i) { c[i] = c0 + a[i]; c[3 + i] = c0 - a[i]; }
#pragma unroll
    for (int i = 0; i < 6; ++i) c[6 + i] = a[3 + i];                  // (1,0) (2,0) (2,1)
#pragma unroll
    for (int i = 0; i < 6; ++i) c[12 + i] = a[9 + i];                 // (3,0) (3,1) (3,2)
#pragma unroll
    for (int i = 0; i < 6; ++i) c[18 + i] = a[15 + i];                // (4,0) (4,1) (4,2)
    c[24] = -a[3]; c[25] = -a[4];                                     // (4,3) = -(1,0)
#pragma unroll
    for (int i = 0; i < 6; ++i) c[26 + i] = a[21 + i];                // (5,0) (5,1) (5,2)
    c[32] = -a[5]; c[33] = -a[6];                                     // (5,3) = -(2,0)
    c[34] = -a[7]; c[35] = -a[8];                                     // (5,4) = -(2,1)
}
// a = the CLOVA_REALS compact reals of one block (delta_0..2, (1,0) (2,0) (2,1), rows 3..5 x columns 0..2, pad);
// the builders form delta in fp64 before rounding
template <typename T>
__device__ __forceinline__ void store_clover_A(T* __restrict__ base, int Vh, int cb, int b, const T (&a)[CLOVA_REALS])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    V* p = reinterpret_cast<V*>(base) + (size_t)b * (CLOVA_REALS / N) * Vh + cb;
#pragma unroll
    for (int k = 0; k < CLOVA_REALS / N; ++k) p[(size_t)k * Vh] = pack(&a[k * N]);
}
// packed 36 (fp64, as the builders hold it) -> compact, delta passed separately
template <typename T>
__device__ __forceinline__ void compact_clover_A(const double (&p)[36], const double (&delta)[3], T (&a)[CLOVA_REALS])
{
#pragma unroll
    for (int i = 0; i < 3; ++i) a[i] = (T)delta[i];
#pragma unroll
    for (int i = 0; i < 6; ++i) { a[3 + i] = (T)p[6 + i]; a[9 + i] = (T)p[12 + i]; a[15 + i] = (T)p[18 + i]; a[21 + i] = (T)p[26 + i]; }
    a[27] = 0;
}

// ------------------------------------------------------------------------- geometry
struct Site {
    int xh, y, z, t;
    int q;               // x & 1  == (y + z + t + parity) & 1
};

__device__ __forceinline__ Site site_of_cb(const Geom& g, int cb, int parity)
{
    Site s;
    s.xh = cb % g.Lh;
    int r = cb / g.Lh;
    s.y = r % g.L;
    r /= g.L;
    s.z = r % g.L;
    s.t = r / g.L;
    s.q = (s.y + s.z + s.t + parity) & 1;
    return s;
}

// checkerboard index (in the opposite-parity arrays) of the neighbour x + dir*mu_hat
template <int MU, int DIR>
__device__ __forceinline__ int neighbour_cb(const Geom& g, int cb, const Site& s)
{
    if (MU == 0) {
        if (DIR > 0) {
            if (s.q == 0) return cb;                               // x even: x+1 shares xh
            return (s.xh == g.Lh - 1) ? cb - (g.Lh - 1) : cb + 1;
        } else {
            if (s.q == 1) return cb;                               // x odd: x-1 shares xh
            return (s.xh == 0) ? cb + (g.Lh - 1) : cb - 1;
        }
    } else if (MU == 1) {
        if (DIR > 0) return (s.y == g.L - 1) ? cb - (g.L - 1) * g.sy : cb + g.sy;
        return (s.y == 0) ? cb + (g.L - 1) * g.sy : cb - g.sy;
    } else if (MU == 2) {
        if (DIR > 0) return (s.z == g.L - 1) ? cb - (g.L - 1) * g.sz : cb + g.sz;
        return (s.z == 0) ? cb + (g.L - 1) * g.sz : cb - g.sz;
    } else {
        if (DIR > 0) return (s.t == g.T - 1) ? cb - (g.T - 1) * g.st : cb + g.st;
        return (s.t == 0) ? cb + (g.T - 1) * g.st : cb - g.st;
    }
}

}  // namespace ddamg

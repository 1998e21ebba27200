// ddamg_hop.cuh -- the hopping term and the 6x6 clover mat-vec, per output site, in registers.
//
// Steps a2-a4 of the path: for each of the 8 neighbours
//   a2  gamma-projection to a half spinor  h = psi_u -+ B_mu psi_l        (12 of 24 reals)
//   a3  SU(3) x half spinor                chi = U h   or   U^H h
//   a4  reconstruction and accumulation    (chi, -+ B_mu^H chi)
// using the chiral-basis identity (1 -+ gamma_mu) psi = (h, -+ B_mu^H h), B_k = -i sigma_k,
// B_t = 1 (reading R1; the oracle multiplies by the full 4x4 matrices instead).
// The overall -1/2 of the hopping term is applied once at the end.
//
// Everything is generic in the spinor VALUE type S (ddamg_common.cuh): S = T (float / double,
// one right-hand side) or S = P2 (fp32, two right-hand sides per thread, every operation one
// packed f32x2 instruction with the link / clover entry as its broadcast scalar operand).
// With S = float the two dense parts are packed as well: the colour multiply runs once on the
// PAIR of spin components of the half spinor (same link, same operations), the 6x6 mat-vec on
// (re, im) pairs.  The order of operations per element is the same in all three forms, so the
// fp32 single-rhs and multi-rhs kernels agree bit for bit.
#pragma once
#include "ddamg_common.cuh"

namespace ddamg {

// spinor register layout: s[6*spin + 2*colour + {0: re, 1: im}]
#define RE(s, c) (6 * (s) + 2 * (c))
#define IM(s, c) (6 * (s) + 2 * (c) + 1)

// h = a + SGN * (I ? i : 1) * b   for one colour component (pair of reals)
template <bool TIMES_I, int SGN, typename S>
__device__ __forceinline__ void proj_pair(S& hr, S& hi, S ar, S ai, S br, S bi)
{
    if (TIMES_I) {          // a + SGN * i * b = (ar - SGN*bi) + i (ai + SGN*br)
        hr = SGN > 0 ? ar - bi : ar + bi;
        hi = SGN > 0 ? ai + br : ai - br;
    } else {
        hr = SGN > 0 ? ar + br : ar - br;
        hi = SGN > 0 ? ai + bi : ai - bi;
    }
}

// acc += SGN * (I ? i : 1) * c
template <bool TIMES_I, int SGN, typename S>
__device__ __forceinline__ void acc_pair(S& ar, S& ai, S cr, S ci)
{
    if (TIMES_I) {
        ar = SGN > 0 ? ar - ci : ar + ci;
        ai = SGN > 0 ? ai + cr : ai - cr;
    } else {
        ar = SGN > 0 ? ar + cr : ar - cr;
        ai = SGN > 0 ? ai + ci : ai - ci;
    }
}

// chi = U h (DAG = false) or U^H h (DAG = true); u row-major 3x3 complex, h/chi 3 complex values
// of type S.  Explicit fma chains (4 per complex multiply-add).
template <bool DAG, typename T, typename S>
__device__ __forceinline__ void su3_mul(const T (&u)[18], const S* __restrict__ h, S* __restrict__ chi)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        S cr, ci;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const T ur = DAG ? u[2 * (3 * b + a)] : u[2 * (3 * a + b)];
            const T ui = DAG ? -u[2 * (3 * b + a) + 1] : u[2 * (3 * a + b) + 1];
            if (b == 0) {
                cr = vmul(ur, h[0]);
                ci = vmul(ur, h[1]);
            } else {
                cr = vfma(ur, h[2 * b], cr);
                ci = vfma(ur, h[2 * b + 1], ci);
            }
            cr = vfma(-ui, h[2 * b + 1], cr);
            ci = vfma(ui, h[2 * b], ci);
        }
        chi[2 * a] = cr;
        chi[2 * a + 1] = ci;
    }
}

// colour multiply of both spin components of a half spinor: h, chi = 12 values (spin, colour, re/im)
template <bool DAG, typename T, typename S>
__device__ __forceinline__ void su3_mul_half(const T (&u)[18], const S (&h)[12], S (&chi)[12])
{
    su3_mul<DAG, T, S>(u, &h[0], &chi[0]);
    su3_mul<DAG, T, S>(u, &h[6], &chi[6]);
}
// fp32, one rhs: the two spin components as the two lanes of packed operations
template <bool DAG>
__device__ __forceinline__ void su3_mul_half(const float (&u)[18], const float (&h)[12], float (&chi)[12])
{
    P2 hp[6], cp[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) hp[k] = mkp(h[k], h[6 + k]);
    su3_mul<DAG, float, P2>(u, hp, cp);
#pragma unroll
    for (int k = 0; k < 6; ++k) { chi[k] = cp[k].v.x; chi[6 + k] = cp[k].v.y; }
}
// One direction.  MU = 0..3, FWD: neighbour x+mu with U_mu(x), projector (1 - gamma_mu);
// !FWD: neighbour x-mu with U_mu(x-mu)^H, projector (1 + gamma_mu).
template <int MU, bool FWD, typename T, typename S>
__device__ __forceinline__ void hop_dir(const S (&psi)[24], const T (&u)[18], S (&acc)[24])
{
    constexpr int P = FWD ? +1 : -1;     // sign in (1 - P*gamma_mu)
    S h[12], chi[12];
    // ---- a2: h = psi_u - P * B_mu psi_l
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (MU == 0) {          // -P*B psi_l = +P*i*sigma_x psi_l = P*i*(psi_3, psi_2)
            proj_pair<true, P>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(3, c)], psi[IM(3, c)]);
            proj_pair<true, P>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(2, c)], psi[IM(2, c)]);
        } else if (MU == 1) {   // -P*B psi_l = P*(psi_3, -psi_2)
            proj_pair<false, P>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(3, c)], psi[IM(3, c)]);
            proj_pair<false, -P>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(2, c)], psi[IM(2, c)]);
        } else if (MU == 2) {   // -P*B psi_l = P*i*(psi_2, -psi_3)
            proj_pair<true, P>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(2, c)], psi[IM(2, c)]);
            proj_pair<true, -P>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(3, c)], psi[IM(3, c)]);
        } else {                // -P*B psi_l = -P*(psi_2, psi_3)
            proj_pair<false, -P>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(2, c)], psi[IM(2, c)]);
            proj_pair<false, -P>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(3, c)], psi[IM(3, c)]);
        }
    }
    // ---- a3: colour multiply of both spin components
    su3_mul_half<!FWD>(u, h, chi);
    // ---- a4: upper += chi ; lower += -P * B_mu^H chi
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[RE(0, c)] = acc[RE(0, c)] + chi[RE(0, c)];
        acc[IM(0, c)] = acc[IM(0, c)] + chi[IM(0, c)];
        acc[RE(1, c)] = acc[RE(1, c)] + chi[RE(1, c)];
        acc[IM(1, c)] = acc[IM(1, c)] + chi[IM(1, c)];
        if (MU == 0) {          // -P * i sigma_x chi = -P*i*(chi_1, chi_0)
            acc_pair<true, -P>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(1, c)], chi[IM(1, c)]);
            acc_pair<true, -P>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(0, c)], chi[IM(0, c)]);
        } else if (MU == 1) {   // -P * i sigma_y chi = -P*(chi_1, -chi_0)
            acc_pair<false, -P>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(1, c)], chi[IM(1, c)]);
            acc_pair<false, P>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(0, c)], chi[IM(0, c)]);
        } else if (MU == 2) {   // -P * i sigma_z chi = -P*i*(chi_0, -chi_1)
            acc_pair<true, -P>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(0, c)], chi[IM(0, c)]);
            acc_pair<true, P>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(1, c)], chi[IM(1, c)]);
        } else {                // -P * chi
            acc_pair<false, -P>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(0, c)], chi[IM(0, c)]);
            acc_pair<false, -P>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(1, c)], chi[IM(1, c)]);
        }
    }
}

// acc = sum over the 8 neighbours (WITHOUT the -1/2).  `in` is the opposite-parity spinor,
// gauge_own / gauge_opp the 4-direction link blocks of this site's / the other parity.
// Multi-rhs: `in` holds the spinors of `units` threads per site interleaved
// (vector index cb * units + r, plane stride Vh * units; fp32: a unit is a PAIR of right-hand
// sides, S = P2; fp64: one right-hand side); links are indexed by site only, so the threads of
// one site read the same link vectors (one DRAM fetch, L1 broadcast).
// RECON = 18: full links.  RECON = 12: two-row storage, third row rebuilt in registers
// (load_link12); apbc != 0 then restores the antiperiodic sign of the links U_t(t = T-1).
template <typename T, int RECON, typename S>
__device__ __forceinline__ void hop_site(const Geom& g, int cb, const Site& s,
                                         const T* __restrict__ in, const int units, const int r,
                                         const T* __restrict__ gauge_own,
                                         const T* __restrict__ gauge_opp, S (&acc)[24], const int apbc = 0)
{
    const int Vs = g.Vh * units;                // vectors per spinor plane
    const size_t lblk = (size_t)RECON * g.Vh;   // reals per (parity, mu) link block
    // sign of the third row of the forward / backward link in direction MU (RECON = 12 only)
    const T sgn_f3 = (apbc && s.t == g.T - 1) ? (T)-1 : (T)1;
    const T sgn_b3 = (apbc && s.t == 0) ? (T)-1 : (T)1;
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = vzero(S());
    S psi[24];
    T u[18];
    int nbs[8];
    nbs[0] = neighbour_cb<0, +1>(g, cb, s); nbs[1] = neighbour_cb<0, -1>(g, cb, s);
    nbs[2] = neighbour_cb<1, +1>(g, cb, s); nbs[3] = neighbour_cb<1, -1>(g, cb, s);
    nbs[4] = neighbour_cb<2, +1>(g, cb, s); nbs[5] = neighbour_cb<2, -1>(g, cb, s);
    nbs[6] = neighbour_cb<3, +1>(g, cb, s); nbs[7] = neighbour_cb<3, -1>(g, cb, s);
#define DDAMG_HOP(MU)                                                        \
    load_spinor<T>(in, Vs, nbs[2 * MU] * units + r, psi);                    \
    if (RECON == 12) load_link12(gauge_own + MU * lblk, g.Vh, cb, MU == 3 ? sgn_f3 : (T)1, u); \
    else load_link(gauge_own + MU * lblk, g.Vh, cb, u);                      \
    hop_dir<MU, true, T, S>(psi, u, acc);                                    \
    load_spinor<T>(in, Vs, nbs[2 * MU + 1] * units + r, psi);                \
    if (RECON == 12) load_link12(gauge_opp + MU * lblk, g.Vh, nbs[2 * MU + 1], MU == 3 ? sgn_b3 : (T)1, u); \
    else load_link(gauge_opp + MU * lblk, g.Vh, nbs[2 * MU + 1], u);         \
    hop_dir<MU, false, T, S>(psi, u, acc);
    DDAMG_HOP(0)
    DDAMG_HOP(1)
    DDAMG_HOP(2)
    DDAMG_HOP(3)
#undef DDAMG_HOP
}

// y (6 complex) = M v for a packed Hermitian 6x6 block c (6 real diag, 15 complex lower)
template <typename T, typename S>
__device__ __forceinline__ void clover_block_mul(const T (&c)[36], const S* __restrict__ v, S* __restrict__ y)
{
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        S yr = vmul(c[i], v[2 * i]);
        S yi = vmul(c[i], v[2 * i + 1]);
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            if (j < i) {                              // l_ij v_j
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                yr = vfma(c[k], v[2 * j], yr);
                yr = vfma(-c[k + 1], v[2 * j + 1], yr);
                yi = vfma(c[k], v[2 * j + 1], yi);
                yi = vfma(c[k + 1], v[2 * j], yi);
            } else if (j > i) {                       // conj(l_ji) v_j
                const int k = 6 + 2 * (j * (j - 1) / 2 + i);
                yr = vfma(c[k], v[2 * j], yr);
                yr = vfma(c[k + 1], v[2 * j + 1], yr);
                yi = vfma(c[k], v[2 * j + 1], yi);
                yi = vfma(-c[k + 1], v[2 * j], yi);
            }
        }
        y[2 * i] = yr;
        y[2 * i + 1] = yi;
    }
}
// fp32, one rhs: (re, im) of each output as the two lanes.  With V_j = (v_re, v_im) and
// W_j = (-v_im, v_re):  l v = l_re V + l_im W,  conj(l) v = l_re V - l_im W; per lane the same
// products in the same order as the scalar form above (the sign of a product does not change
// its rounding).
__device__ __forceinline__ void clover_block_mul(const float (&c)[36], const float* __restrict__ v, float* __restrict__ y)
{
    P2 V[6], W[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) { V[j] = mkp(v[2 * j], v[2 * j + 1]); W[j] = mkp(-v[2 * j + 1], v[2 * j]); }
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        P2 Y = vmul(c[i], V[i]);
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            if (j < i) {
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                Y = vfma(c[k], V[j], Y);
                Y = vfma(c[k + 1], W[j], Y);
            } else if (j > i) {
                const int k = 6 + 2 * (j * (j - 1) / 2 + i);
                Y = vfma(c[k], V[j], Y);
                Y = vfma(-c[k + 1], W[j], Y);
            }
        }
        y[2 * i] = Y.v.x;
        y[2 * i + 1] = Y.v.y;
    }
}

// out = Cl(x) v for the two blocks of one site (upper: reals 0..11, lower: 12..23).
// AFMT = false: `clov` holds general Hermitian blocks (the inverses) in the packed 36-real form;
// AFMT = true: it holds the clover blocks themselves in the compact 28-real form (c0 = m0 + 4).
// MODE: LD_STREAM / LD_REUSE (global) or LD_PLAIN (`clov` in shared memory), ddamg_common.cuh.
template <typename T, int MODE = LD_STREAM, bool AFMT = false, typename S>
__device__ __forceinline__ void clover_site_mul(const T* __restrict__ clov, int Vh, int cb,
                                                const S (&v)[24], S (&out)[24], T c0 = 0)
{
    T c[36];
    if (AFMT) load_clover_A<T, MODE>(clov, Vh, cb, 0, c0, c);
    else load_clover_block<T, MODE>(clov, Vh, cb, 0, c);
    clover_block_mul(c, &v[0], &out[0]);
    if (AFMT) load_clover_A<T, MODE>(clov, Vh, cb, 1, c0, c);
    else load_clover_block<T, MODE>(clov, Vh, cb, 1, c);
    clover_block_mul(c, &v[12], &out[12]);
}

}  // namespace ddamg

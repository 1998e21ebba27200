// ddamg_hop.cuh -- the hopping term and the 6x6 clover mat-vec, per output site, in registers.
//
// Steps a2-a4 of the path: for each of the 8 neighbours
//   a2  gamma-projection to a half spinor  h = psi_u -+ B_mu psi_l        (12 of 24 reals)
//   a3  SU(3) x half spinor                chi = U h   or   U^H h
//   a4  reconstruction and accumulation    (chi, -+ B_mu^H chi)
// using the chiral-basis identity (1 -+ gamma_mu) psi = (h, -+ B_mu^H h), B_k = -i sigma_k,
// B_t = 1 (reading R1; the oracle multiplies by the full 4x4 matrices instead).
// The overall -1/2 of the hopping term is applied once at the end.
#pragma once
#include "ddamg_common.cuh"

namespace ddamg {

// spinor register layout: s[6*spin + 2*colour + {0: re, 1: im}]
#define RE(s, c) (6 * (s) + 2 * (c))
#define IM(s, c) (6 * (s) + 2 * (c) + 1)

// h = a + SGN * (I ? i : 1) * b   for one colour component (pair of reals)
template <bool TIMES_I, int SGN, typename T>
__device__ __forceinline__ void proj_pair(T& hr, T& hi, T ar, T ai, T br, T bi)
{
    if (TIMES_I) {          // a + SGN * i * b = (ar - SGN*bi) + i (ai + SGN*br)
        hr = ar - SGN * bi;
        hi = ai + SGN * br;
    } else {
        hr = ar + SGN * br;
        hi = ai + SGN * bi;
    }
}

// acc += SGN * (I ? i : 1) * c
template <bool TIMES_I, int SGN, typename T>
__device__ __forceinline__ void acc_pair(T& ar, T& ai, T cr, T ci)
{
    if (TIMES_I) {
        ar -= SGN * ci;
        ai += SGN * cr;
    } else {
        ar += SGN * cr;
        ai += SGN * ci;
    }
}

// chi = U h (DAG = false) or U^H h (DAG = true); u row-major 3x3 complex, h/chi 3 complex.
// Written as explicit fma chains (4 FFMA per complex multiply-add): `c += a*b - d*e` would be
// evaluated as c + (a*b - d*e) = FMUL + FFMA + FADD, 50 % more instructions.
template <bool DAG, typename T>
__device__ __forceinline__ void su3_mul(const T (&u)[18], const T* __restrict__ h, T* __restrict__ chi)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T cr, ci;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const T ur = DAG ? u[2 * (3 * b + a)] : u[2 * (3 * a + b)];
            const T ui = DAG ? -u[2 * (3 * b + a) + 1] : u[2 * (3 * a + b) + 1];
            if (b == 0) {
                cr = ur * h[0];
                ci = ur * h[1];
            } else {
                cr = fma(ur, h[2 * b], cr);
                ci = fma(ur, h[2 * b + 1], ci);
            }
            cr = fma(-ui, h[2 * b + 1], cr);
            ci = fma(ui, h[2 * b], ci);
        }
        chi[2 * a] = cr;
        chi[2 * a + 1] = ci;
    }
}

// One direction.  MU = 0..3, FWD: neighbour x+mu with U_mu(x), projector (1 - gamma_mu);
// !FWD: neighbour x-mu with U_mu(x-mu)^H, projector (1 + gamma_mu).
template <int MU, bool FWD, typename T>
__device__ __forceinline__ void hop_dir(const T (&psi)[24], const T (&u)[18], T (&acc)[24])
{
    constexpr int S = FWD ? +1 : -1;     // sign in (1 - S*gamma_mu)
    T h[12], chi[12];
    // ---- a2: h = psi_u - S * B_mu psi_l
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (MU == 0) {          // -S*B psi_l = +S*i*sigma_x psi_l = S*i*(psi_3, psi_2)
            proj_pair<true, S>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(3, c)], psi[IM(3, c)]);
            proj_pair<true, S>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(2, c)], psi[IM(2, c)]);
        } else if (MU == 1) {   // -S*B psi_l = S*(psi_3, -psi_2)
            proj_pair<false, S>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(3, c)], psi[IM(3, c)]);
            proj_pair<false, -S>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(2, c)], psi[IM(2, c)]);
        } else if (MU == 2) {   // -S*B psi_l = S*i*(psi_2, -psi_3)
            proj_pair<true, S>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(2, c)], psi[IM(2, c)]);
            proj_pair<true, -S>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(3, c)], psi[IM(3, c)]);
        } else {                // -S*B psi_l = -S*(psi_2, psi_3)
            proj_pair<false, -S>(h[RE(0, c)], h[IM(0, c)], psi[RE(0, c)], psi[IM(0, c)], psi[RE(2, c)], psi[IM(2, c)]);
            proj_pair<false, -S>(h[RE(1, c)], h[IM(1, c)], psi[RE(1, c)], psi[IM(1, c)], psi[RE(3, c)], psi[IM(3, c)]);
        }
    }
    // ---- a3: colour multiply of both spin components
    su3_mul<!FWD>(u, &h[0], &chi[0]);
    su3_mul<!FWD>(u, &h[6], &chi[6]);
    // ---- a4: upper += chi ; lower += -S * B_mu^H chi
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[RE(0, c)] += chi[RE(0, c)];
        acc[IM(0, c)] += chi[IM(0, c)];
        acc[RE(1, c)] += chi[RE(1, c)];
        acc[IM(1, c)] += chi[IM(1, c)];
        if (MU == 0) {          // -S * i sigma_x chi = -S*i*(chi_1, chi_0)
            acc_pair<true, -S>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(1, c)], chi[IM(1, c)]);
            acc_pair<true, -S>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(0, c)], chi[IM(0, c)]);
        } else if (MU == 1) {   // -S * i sigma_y chi = -S*(chi_1, -chi_0)
            acc_pair<false, -S>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(1, c)], chi[IM(1, c)]);
            acc_pair<false, S>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(0, c)], chi[IM(0, c)]);
        } else if (MU == 2) {   // -S * i sigma_z chi = -S*i*(chi_0, -chi_1)
            acc_pair<true, -S>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(0, c)], chi[IM(0, c)]);
            acc_pair<true, S>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(1, c)], chi[IM(1, c)]);
        } else {                // -S * chi
            acc_pair<false, -S>(acc[RE(2, c)], acc[IM(2, c)], chi[RE(0, c)], chi[IM(0, c)]);
            acc_pair<false, -S>(acc[RE(3, c)], acc[IM(3, c)], chi[RE(1, c)], chi[IM(1, c)]);
        }
    }
}

// acc = sum over the 8 neighbours (WITHOUT the -1/2).  `in` is the opposite-parity spinor,
// gauge_own / gauge_opp the 4-direction link blocks of this site's / the other parity.
// Multi-rhs: `in` holds nrhs spinors interleaved per site (vector index
// cb * nrhs + r, plane stride Vh * nrhs); links are indexed by site only, so the nrhs
// adjacent threads of one site read the same link vectors (one DRAM fetch, L1 broadcast).
// RECON = 18: full links.  RECON = 12: two-row storage, third row rebuilt in registers
// (load_link12); apbc != 0 then restores the antiperiodic sign of the links U_t(t = T-1).
template <typename T, int RECON = 18>
__device__ __forceinline__ void hop_site(const Geom& g, int cb, const Site& s,
                                         const T* __restrict__ in, const int nrhs, const int r,
                                         const T* __restrict__ gauge_own,
                                         const T* __restrict__ gauge_opp, T (&acc)[24], const int apbc = 0)
{
    const int Vs = g.Vh * nrhs;                 // vectors per spinor plane
    const size_t lblk = (size_t)RECON * g.Vh;   // reals per (parity, mu) link block
    // sign of the third row of the forward / backward link in direction MU (RECON = 12 only)
    const T sgn_f3 = (apbc && s.t == g.T - 1) ? (T)-1 : (T)1;
    const T sgn_b3 = (apbc && s.t == 0) ? (T)-1 : (T)1;
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    T psi[24], u[18];
    int nbs[8];
    nbs[0] = neighbour_cb<0, +1>(g, cb, s); nbs[1] = neighbour_cb<0, -1>(g, cb, s);
    nbs[2] = neighbour_cb<1, +1>(g, cb, s); nbs[3] = neighbour_cb<1, -1>(g, cb, s);
    nbs[4] = neighbour_cb<2, +1>(g, cb, s); nbs[5] = neighbour_cb<2, -1>(g, cb, s);
    nbs[6] = neighbour_cb<3, +1>(g, cb, s); nbs[7] = neighbour_cb<3, -1>(g, cb, s);
#define DDAMG_HOP(MU)                                                        \
    load_spinor<T>(in, Vs, nbs[2 * MU] * nrhs + r, psi);                     \
    if (RECON == 12) load_link12(gauge_own + MU * lblk, g.Vh, cb, MU == 3 ? sgn_f3 : (T)1, u); \
    else load_link(gauge_own + MU * lblk, g.Vh, cb, u);                      \
    hop_dir<MU, true>(psi, u, acc);                                          \
    load_spinor<T>(in, Vs, nbs[2 * MU + 1] * nrhs + r, psi);                 \
    if (RECON == 12) load_link12(gauge_opp + MU * lblk, g.Vh, nbs[2 * MU + 1], MU == 3 ? sgn_b3 : (T)1, u); \
    else load_link(gauge_opp + MU * lblk, g.Vh, nbs[2 * MU + 1], u);         \
    hop_dir<MU, false>(psi, u, acc);
    DDAMG_HOP(0)
    DDAMG_HOP(1)
    DDAMG_HOP(2)
    DDAMG_HOP(3)
#undef DDAMG_HOP
}

// y (6 complex) = M v for a packed Hermitian 6x6 block c (6 real diag, 15 complex lower)
template <typename T>
__device__ __forceinline__ void clover_block_mul(const T (&c)[36], const T* __restrict__ v, T* __restrict__ y)
{
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        T yr = c[i] * v[2 * i];
        T yi = c[i] * v[2 * i + 1];
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            if (j < i) {                              // l_ij v_j
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                yr = fma(c[k], v[2 * j], yr);
                yr = fma(-c[k + 1], v[2 * j + 1], yr);
                yi = fma(c[k], v[2 * j + 1], yi);
                yi = fma(c[k + 1], v[2 * j], yi);
            } else if (j > i) {                       // conj(l_ji) v_j
                const int k = 6 + 2 * (j * (j - 1) / 2 + i);
                yr = fma(c[k], v[2 * j], yr);
                yr = fma(c[k + 1], v[2 * j + 1], yr);
                yi = fma(c[k], v[2 * j + 1], yi);
                yi = fma(-c[k + 1], v[2 * j], yi);
            }
        }
        y[2 * i] = yr;
        y[2 * i + 1] = yi;
    }
}

// out = Cl(x) v for the two blocks of one site (upper: reals 0..11, lower: 12..23)
template <typename T, bool STREAM = true>
__device__ __forceinline__ void clover_site_mul(const T* __restrict__ clov, int Vh, int cb,
                                                const T (&v)[24], T (&out)[24])
{
    T c[36];
    load_clover_block<T, STREAM>(clov, Vh, cb, 0, c);
    clover_block_mul<T>(c, &v[0], &out[0]);
    load_clover_block<T, STREAM>(clov, Vh, cb, 1, c);
    clover_block_mul<T>(c, &v[12], &out[12]);
}

}  // namespace ddamg

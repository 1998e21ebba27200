// ddamg_sap.cu -- the block solves of SAP(n, m) (Alg. 1).
//
// One CTA per domain-decomposition block of one colour (Alg. 1 lines 4-6 / 8-10): given the
// global residual r = b - D x (lines 2 / 7, computed by the streaming full-operator kernel of
// ddamg_dslash.cu, which runs at the HBM roofline; evaluating it inside this low-occupancy
// kernel was measured 1.6x slower) it runs m Minimal Residual iterations on D_k e_k = r_k with
// block-local odd-even preconditioning ("each of the domain decomposition blocks"
// is reordered and "minimal residual is used for solving the linear systems with the Schur
// complement of each block") and adds e_k to x_k:
//
//     rhat_e = r_e - H^k_eo A_oo^-1 r_o                               eq. 2 on the block
//     e = 0, rho = rhat_e;  m x { q = D^k_S rho;  alpha = <q,rho>/<q,q>;  e += alpha rho;  rho -= alpha q }
//     e_o = A_oo^-1 (r_o - H^k_oe e);   x_e += e;  x_o += e_o
//
// with D^k_S = A_ee - H^k_eo A_oo^-1 H^k_oe and H^k the hopping term with every hop that leaves
// the block dropped (D_k = P_k D P_k^T, R21).  B200 mapping: thread i owns even site i
// and odd site i of the block (all lanes busy in both half steps); the block's links (the only
// operand re-used by all 2m+3 hopping applications) are staged ONCE in shared memory, the two
// exchanged half-block spinors live in shared memory, e and rho stay in registers, the 6x6
// clover blocks are re-read through L1/L2 (73 KB per 4^4 block: L2-resident).  All dot
// products are block-local: one CTA-wide fp64 reduction per MR iteration, no
// global reduction, no host involvement.
#include "ddamg_internal.h"
#include "ddamg_hop.cuh"

namespace ddamg {

template <typename T>
struct SapArgs {
    Geom g;
    SapGeom sg;
    int colour;              // colour of the blocks this launch solves (0 = red)
    int m;                   // Minimal Residual iterations (>= 1)
    const T* blk_links;      // block-ordered links:  [block][parity][mu][18 * n]   (sap_reorder_kernel)
    const T* blk_clov;       // block-ordered A_ee / A_oo^-1 blocks:  [block][parity][72 * n]
    const T* r_e;            // global residual r = b - D x
    const T* r_o;
    T* x_e;                  // iterate, updated in place on the blocks of this colour
    T* x_o;
};

// ---- shared-memory access (plain loads/stores: the read-only global path does not apply)
template <typename T>
__device__ __forceinline__ void lds_spinor(const T* base, int n, int i, T (&s)[24])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    const V* p = reinterpret_cast<const V*>(base) + i;
#pragma unroll
    for (int k = 0; k < 24 / N; ++k) unpack(p[k * n], &s[k * N]);
}
template <typename T>
__device__ __forceinline__ void sts_spinor(T* base, int n, int i, const T (&s)[24])
{
    using V = typename VecOf<T>::type;
    constexpr int N = VecOf<T>::N;
    V* p = reinterpret_cast<V*>(base) + i;
#pragma unroll
    for (int k = 0; k < 24 / N; ++k) p[k * n] = pack(&s[k * N]);
}
__device__ __forceinline__ void lds_link(const float* blk, int n, int i, float (&u)[18])
{
    const float4* p4 = reinterpret_cast<const float4*>(blk) + i;
#pragma unroll
    for (int k = 0; k < 4; ++k) unpack(p4[k * n], &u[4 * k]);
    const float2 v = reinterpret_cast<const float2*>(blk + 16 * n)[i];
    u[16] = v.x; u[17] = v.y;
}
__device__ __forceinline__ void lds_link(const double* blk, int n, int i, double (&u)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + i;
#pragma unroll
    for (int k = 0; k < 9; ++k) unpack(p[k * n], &u[2 * k]);
}
__device__ __forceinline__ void sts_link(float* blk, int n, int i, const float (&u)[18])
{
    float4* p4 = reinterpret_cast<float4*>(blk) + i;
#pragma unroll
    for (int k = 0; k < 4; ++k) p4[k * n] = pack(&u[4 * k]);
    reinterpret_cast<float2*>(blk + 16 * n)[i] = make_float2(u[16], u[17]);
}
__device__ __forceinline__ void sts_link(double* blk, int n, int i, const double (&u)[18])
{
    double2* p = reinterpret_cast<double2*>(blk) + i;
#pragma unroll
    for (int k = 0; k < 9; ++k) p[k * n] = pack(&u[2 * k]);
}

// local site of parity p with block-checkerboard index lcb = (lx>>1) + Bxh*(ly + By*(lz + Bz*lt))
struct LSite {
    int lx, ly, lz, lt;
    int q;               // lx & 1
};
__device__ __forceinline__ LSite lsite_of(const SapGeom& sg, int lcb, int parity)
{
    LSite s;
    const int xh = lcb % sg.Bxh;
    int r = lcb / sg.Bxh;
    s.ly = r % sg.B[1];
    r /= sg.B[1];
    s.lz = r % sg.B[2];
    s.lt = r / sg.B[2];
    s.q = (s.ly + s.lz + s.lt + parity) & 1;        // block origins are even: local parity == global parity
    s.lx = 2 * xh + s.q;
    return s;
}

// acc = sum over the neighbours INSIDE the block (without the -1/2): the hopping term of
// D_k = P_k D P_k^T.  in: opposite-parity half-block spinor, links_own / links_opp: the block's
// forward links of this site's / the other parity, all in shared memory.
template <typename T>
__device__ __forceinline__ void hop_block(const SapGeom& sg, int lcb, const LSite& s, const T* in,
                                          const T* links_own, const T* links_opp, T (&acc)[24])
{
    const int n = sg.Vbh;
    const int lblk = 18 * n;
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    T psi[24], u[18];
    const int sy = sg.Bxh, sz = sg.Bxh * sg.B[1], st = sg.Bxh * sg.B[1] * sg.B[2];
#define DDAMG_BHOP(MU, IN_F, NB_F, IN_B, NB_B)                               \
    if (IN_F) {                                                              \
        lds_spinor<T>(in, n, (NB_F), psi);                                   \
        lds_link(links_own + MU * lblk, n, lcb, u);                          \
        hop_dir<MU, true>(psi, u, acc);                                      \
    }                                                                        \
    if (IN_B) {                                                              \
        lds_spinor<T>(in, n, (NB_B), psi);                                   \
        lds_link(links_opp + MU * lblk, n, (NB_B), u);                       \
        hop_dir<MU, false>(psi, u, acc);                                     \
    }
    DDAMG_BHOP(0, s.lx + 1 < sg.B[0], lcb + s.q, s.lx > 0, lcb + s.q - 1)
    DDAMG_BHOP(1, s.ly + 1 < sg.B[1], lcb + sy, s.ly > 0, lcb - sy)
    DDAMG_BHOP(2, s.lz + 1 < sg.B[2], lcb + sz, s.lz > 0, lcb - sz)
    DDAMG_BHOP(3, s.lt + 1 < sg.B[3], lcb + st, s.lt > 0, lcb - st)
#undef DDAMG_BHOP
}

template <typename T>
__global__ void __launch_bounds__(SAP_MAX_THREADS, 1) sap_block_kernel(const SapArgs<T> a)
{
    extern __shared__ __align__(16) unsigned char sap_smem[];
    const SapGeom& sg = a.sg;
    const int n = sg.Vbh;
    T* links = reinterpret_cast<T*>(sap_smem);                 // [parity][mu][18 * n]
    T* S_e = links + 2 * 4 * 18 * n;                           // even-site half-block spinor
    T* S_o = S_e + 24 * n;                                     // odd-site half-block spinor
    double* red = reinterpret_cast<double*>(S_o + 24 * n);     // [warp][3]
    const int tid = threadIdx.x;
    const bool active = tid < n;
    const int lane = tid & 31, warp = tid >> 5, nwarps = (blockDim.x + 31) >> 5;

    // which block: blocks of one colour enumerated with the x block-coordinate compressed by 2
    int r = blockIdx.x;
    const int cxh = r % sg.nbxh; r /= sg.nbxh;
    const int cy = r % sg.nb[1]; r /= sg.nb[1];
    const int cz = r % sg.nb[2];
    const int ct = r / sg.nb[2];
    const int cx = 2 * cxh + ((cy + cz + ct + a.colour) & 1);
    const int ox = cx * sg.B[0], oy = cy * sg.B[1], oz = cz * sg.B[2], ot = ct * sg.B[3];
    const size_t bid = (size_t)cx + (size_t)sg.nb[0] * (cy + (size_t)sg.nb[1] * (cz + (size_t)sg.nb[2] * ct));
    const T* clov_e = a.blk_clov + bid * 2 * 72 * n;          // this block's A_ee, in-block SoA (n sites)
    const T* clov_oinv = clov_e + 72 * n;                      // and A_oo^-1

    LSite ls[2];                                               // this thread's even / odd site in the block
    int cbg[2] = { 0, 0 };                                     // and their global checkerboard indices
    T rho[24], e[24];
    if (active) {
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            ls[p] = lsite_of(sg, tid, p);
            cbg[p] = ((ox + ls[p].lx) >> 1) + a.g.Lh * ((oy + ls[p].ly) + a.g.L * ((oz + ls[p].lz) + a.g.L * (ot + ls[p].lt)));
        }
    }
    const int sblk = 4 * 18 * n;                               // one parity's four link blocks in shared memory
    {
        // ---- stage the block's links (read once from HBM per launch): the block-ordered copy has
        // the shared-memory layout, so this is one contiguous, fully coalesced 16-byte-vector copy
        using V = typename VecOf<T>::type;
        const V* src = reinterpret_cast<const V*>(a.blk_links + bid * 2 * sblk);
        V* dst = reinterpret_cast<V*>(links);
        const int nv = 2 * sblk / VecOf<T>::N;
        for (int i = tid; i < nv; i += blockDim.x) dst[i] = ld_stream(src + i);
    }
    if (active) {
        // ---- eq. 2 right factor, odd half: t_o = A_oo^-1 r_o;  rho starts as r_e
        T v[24], t[24];
        load_spinor<T, false>(a.r_o, a.g.Vh, cbg[1], v);
        clover_site_mul<T, false>(clov_oinv, n, tid, v, t);
        sts_spinor<T>(S_o, n, tid, t);
        load_spinor<T, true>(a.r_e, a.g.Vh, cbg[0], rho);
    }
    __syncthreads();

    // ---- the block solve as 2m+2 half steps, one copy of the block hopping code:
    //   hs = 0        even:  rho = rhat_e = r_e - H^k_eo t_o;  e = 0
    //   hs odd < last odd :  t_o = A_oo^-1 H^k_oe rho
    //   hs even > 0   even:  q = A_ee rho - H^k_eo t_o;  alpha = <q,rho>/<q,q>;  e += alpha rho;  rho -= alpha q
    //   hs = 2m+1     odd :  e_o = A_oo^-1 (r_o - H^k_oe e);  x += e
    const int last = 2 * a.m + 1;
#pragma unroll 1
    for (int hs = 0; hs <= last; ++hs) {
        const int par = hs & 1;
        T acc[24];
        if (active)
            hop_block<T>(sg, tid, ls[par], par ? S_e : S_o, links + par * sblk, links + (1 - par) * sblk, acc);
        if (par) {
            if (active) {
                T v[24], t[24];
                if (hs == last) {
                    load_spinor<T, false>(a.r_o, a.g.Vh, cbg[1], v);
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] = v[i] + (T)0.5 * acc[i];          // r_o - H e
                } else {
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] = (T)(-0.5) * acc[i];              // H rho
                }
                clover_site_mul<T, false>(clov_oinv, n, tid, v, t);
                if (hs == last) {
                    load_spinor<T, true>(a.x_o, a.g.Vh, cbg[1], v);
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] += t[i];
                    store_spinor<T>(a.x_o, a.g.Vh, cbg[1], v);
                    load_spinor<T, true>(a.x_e, a.g.Vh, cbg[0], v);
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] += e[i];
                    store_spinor<T>(a.x_e, a.g.Vh, cbg[0], v);
                } else {
                    sts_spinor<T>(S_o, n, tid, t);
                }
            }
        } else if (hs == 0) {
            if (active) {
#pragma unroll
                for (int i = 0; i < 24; ++i) {
                    rho[i] = rho[i] + (T)0.5 * acc[i];
                    e[i] = 0;
                }
                sts_spinor<T>(S_e, n, tid, rho);
            }
        } else {
            T q[24];
            double nr = 0.0, ni = 0.0, dd = 0.0;
            if (active) {
                clover_site_mul<T, false>(clov_e, n, tid, rho, q);
#pragma unroll
                for (int i = 0; i < 24; ++i) q[i] = q[i] + (T)0.5 * acc[i];
                // <q, rho> = q^H rho and <q, q>, this site's share
#pragma unroll
                for (int c = 0; c < 12; ++c) {
                    const double qr = q[2 * c], qi = q[2 * c + 1], pr = rho[2 * c], pi = rho[2 * c + 1];
                    nr += qr * pr + qi * pi;
                    ni += qr * pi - qi * pr;
                    dd += qr * qr + qi * qi;
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                nr += __shfl_xor_sync(0xffffffffu, nr, o);
                ni += __shfl_xor_sync(0xffffffffu, ni, o);
                dd += __shfl_xor_sync(0xffffffffu, dd, o);
            }
            if (lane == 0) { red[3 * warp] = nr; red[3 * warp + 1] = ni; red[3 * warp + 2] = dd; }
            __syncthreads();
            nr = ni = dd = 0.0;
            for (int w = 0; w < nwarps; ++w) { nr += red[3 * w]; ni += red[3 * w + 1]; dd += red[3 * w + 2]; }
            const T ar = dd > 0.0 ? (T)(nr / dd) : (T)0, ai = dd > 0.0 ? (T)(ni / dd) : (T)0;
            if (active) {
#pragma unroll
                for (int c = 0; c < 12; ++c) {
                    const T pr = rho[2 * c], pi = rho[2 * c + 1];
                    e[2 * c] += ar * pr - ai * pi;                     // e += alpha rho
                    e[2 * c + 1] += ar * pi + ai * pr;
                    rho[2 * c] -= ar * q[2 * c] - ai * q[2 * c + 1];   // rho -= alpha q
                    rho[2 * c + 1] -= ar * q[2 * c + 1] + ai * q[2 * c];
                }
                if (hs + 1 < last) sts_spinor<T>(S_e, n, tid, rho);
                else sts_spinor<T>(S_e, n, tid, e);
            }
        }
        __syncthreads();
    }
}

// ---- block-ordered operand copies (built once per block geometry, ddamg_api.cu caches them)
// In the checkerboard layout a 4^4 block owns x-runs of two sites per parity: 32-byte runs, so
// half of every 64-byte DRAM access and three quarters of every 128-byte L2 line were wasted
// on the links and on the 6x6 blocks that all 2m+2 half steps re-read (profiles/
// r1c_ncu_full_sap.md).  Here every block's links and clover blocks are stored contiguously in
// the block's own SoA order (plane-major, n = V_b/2 sites per plane), block id = cx + nbx (cy +
// nby (cz + nbz ct)) over the blocks of BOTH colours.
template <typename T>
__global__ void sap_reorder_kernel(Geom g, SapGeom sg, const T* __restrict__ gauge, const T* __restrict__ clov_e,
                                   const T* __restrict__ clov_oinv, T* __restrict__ blk_links, T* __restrict__ blk_clov)
{
    const int n = sg.Vbh, i = threadIdx.x;
    if (i >= n) return;
    int r = blockIdx.x;
    const int cx = r % sg.nb[0]; r /= sg.nb[0];
    const int cy = r % sg.nb[1]; r /= sg.nb[1];
    const int cz = r % sg.nb[2];
    const int ct = r / sg.nb[2];
    const size_t bid = blockIdx.x;
    const size_t gblk = (size_t)18 * g.Vh;
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        const LSite ls = lsite_of(sg, i, p);
        const int cbg = ((cx * sg.B[0] + ls.lx) >> 1) +
                        g.Lh * ((cy * sg.B[1] + ls.ly) + g.L * ((cz * sg.B[2] + ls.lz) + g.L * (ct * sg.B[3] + ls.lt)));
#pragma unroll 1
        for (int mu = 0; mu < 4; ++mu) {
            T u[18];
            load_link(gauge + (size_t)(p * 4 + mu) * gblk, g.Vh, cbg, u);
            store_link(blk_links + (bid * 8 + p * 4 + mu) * 18 * n, n, i, u);
        }
        const T* src = p ? clov_oinv : clov_e;
#pragma unroll 1
        for (int b = 0; b < 2; ++b) {
            T c[36];
            load_clover_block<T, true>(src, g.Vh, cbg, b, c);
            store_clover_block<T>(blk_clov + (bid * 2 + p) * 72 * n, n, i, b, c);
        }
    }
}

template <typename T>
void launch_sap_reorder(const Geom& g, const SapGeom& sg, const void* gauge, const void* clov_e, const void* clov_oinv,
                        void* blk_links, void* blk_clov, cudaStream_t st)
{
    const int threads = (sg.Vbh + 31) / 32 * 32;
    const int grid = sg.nb[0] * sg.nb[1] * sg.nb[2] * sg.nb[3];
    sap_reorder_kernel<T><<<grid, threads, 0, st>>>(g, sg, (const T*)gauge, (const T*)clov_e, (const T*)clov_oinv,
                                                    (T*)blk_links, (T*)blk_clov);
}
template void launch_sap_reorder<float>(const Geom&, const SapGeom&, const void*, const void*, const void*, void*, void*, cudaStream_t);
template void launch_sap_reorder<double>(const Geom&, const SapGeom&, const void*, const void*, const void*, void*, void*, cudaStream_t);

size_t sap_smem_bytes(const SapGeom& sg, size_t real_bytes)
{
    return (size_t)(2 * 4 * 18 + 48) * sg.Vbh * real_bytes + (size_t)32 * 3 * sizeof(double);
}

template <typename T>
cudaError_t launch_sap_blocks(const Geom& g, const SapGeom& sg, int colour, int m, const void* blk_links,
                              const void* blk_clov, const void* r_e, const void* r_o,
                              void* x_e, void* x_o, cudaStream_t st)
{
    SapArgs<T> a;
    a.g = g; a.sg = sg; a.colour = colour; a.m = m;
    a.blk_links = (const T*)blk_links; a.blk_clov = (const T*)blk_clov;
    a.r_e = (const T*)r_e; a.r_o = (const T*)r_o; a.x_e = (T*)x_e; a.x_o = (T*)x_o;
    const size_t smem = sap_smem_bytes(sg, sizeof(T));
    cudaError_t e = cudaFuncSetAttribute(sap_block_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int threads = (sg.Vbh + 31) / 32 * 32;
    const int grid = sg.nbxh * sg.nb[1] * sg.nb[2] * sg.nb[3];
    sap_block_kernel<T><<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}
template cudaError_t launch_sap_blocks<float>(const Geom&, const SapGeom&, int, int, const void*, const void*,
                                              const void*, const void*, void*, void*, cudaStream_t);
template cudaError_t launch_sap_blocks<double>(const Geom&, const SapGeom&, int, int, const void*, const void*,
                                               const void*, const void*, void*, void*, cudaStream_t);

}  // namespace ddamg

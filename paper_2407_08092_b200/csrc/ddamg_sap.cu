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
// operand re-used by all 2m+3 hopping applications) are staged ONCE in shared memory (one TMA bulk copy), the two
// exchanged half-block spinors live in shared memory, e and rho stay in registers, the 6x6
// clover blocks are re-read through L1/L2 (65 KB per 4^4 block with A_ee in its compact form: L2-resident) or,
// in the default case (fp32, two-row links, 4^4 blocks: template flag CS), staged in shared memory by one TMA
// bulk copy per half step that lands behind the hopping sum.  All dot
// products are block-local: one CTA-wide fp64 reduction per MR iteration, no
// global reduction, no host involvement.
//
// The residual is kept up to date INCREMENTALLY (what DD-alphaAMG itself does; R24): after its
// solve the block kernel also writes e_k and the new residual of its own sites -- (rho, 0): the odd rows of
// D_k e_k = r_k hold exactly, the even rows are left with the last Minimal Residual residual -- and
// sap_boundary_kernel subtracts H e from the sites of the OTHER colour that touch a solved block (the hops
// that cross a block face, on average 2 of 8 per site for 4^4 blocks).  Alg. 1's lines 2 and 7 thus cost one
// partial hopping pass instead of two full operator applications per colour.
// RECON = 12: the block's links are staged as two rows (48 instead of 72 bytes per link in fp32; third row
// rebuilt on use), which brings a 4^4 fp32 block to 74 KB of shared memory: 3 CTAs per SM instead of 2.
#include "ddamg_internal.h"
#include "ddamg_hop.cuh"

namespace ddamg {

template <typename T>
struct SapArgs {
    Geom g;
    SapGeom sg;
    int colour;              // colour of the blocks this launch solves (0 = red)
    int m;                   // Minimal Residual iterations (>= 1)
    const T* blk_links;      // block-ordered links:  [block][parity][mu][RECON * n]   (sap_reorder_kernel)
    const T* blk_clov;       // block-ordered A_ee (compact form, 2 * CLOVA_REALS * n of the slot used) / A_oo^-1 blocks (packed):  [block][parity][72 * n]
    T c0;                    // m0 + 4, the constant part of the compact A_ee blocks
    const T* r_e;            // global residual r = b - D x (read on the blocks of this colour)
    const T* r_o;
    T* rn_e;                 // residual after the update, written on the blocks of this colour: (rho, 0)
    T* rn_o;
    T* e_e;                  // the update e_k, written on the blocks of this colour (read by sap_boundary_kernel)
    T* e_o;
    T* x_e;                  // iterate, updated in place on the blocks of this colour
    T* x_o;
    int blocked;             // r, rn, e are BLOCK-ORDERED arrays ([block][plane][n], one array per parity) instead of
                             // native half spinors: every access of a block is then a contiguous run per plane
    int rin_native;          // blocked: the INPUT residual r_e / r_o is still a native half spinor (first launch of a
                             // call from x = 0, where r = b is read in place)
    int x_assign;            // x = e instead of x += e (first solve of a colour from x = 0: x is not read)
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
// two-row links in shared memory (RECON = 12): rows 0, 1 as 3 float4 / 6 double2 planes, third row rebuilt.
// No boundary sign: a hop inside a block never uses the wrap-around link of the time boundary.
__device__ __forceinline__ void lds_link12(const float* blk, int n, int i, float (&u)[18])
{
    const float4* p4 = reinterpret_cast<const float4*>(blk) + i;
#pragma unroll
    for (int k = 0; k < 3; ++k) unpack(p4[k * n], &u[4 * k]);
    reconstruct_row2<float>(1.f, u);
}
__device__ __forceinline__ void lds_link12(const double* blk, int n, int i, double (&u)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + i;
#pragma unroll
    for (int k = 0; k < 6; ++k) unpack(p[k * n], &u[2 * k]);
    reconstruct_row2<double>(1.0, u);
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
template <typename T, int RECON>
__device__ __forceinline__ void hop_block(const SapGeom& sg, int lcb, const LSite& s, const T* in,
                                          const T* links_own, const T* links_opp, T (&acc)[24])
{
    const int n = sg.Vbh;
    const int lblk = RECON * n;
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    T psi[24], u[18];
    const int sy = sg.Bxh, sz = sg.Bxh * sg.B[1], st = sg.Bxh * sg.B[1] * sg.B[2];
#define DDAMG_BHOP(MU, IN_F, NB_F, IN_B, NB_B)                               \
    if (IN_F) {                                                              \
        lds_spinor<T>(in, n, (NB_F), psi);                                   \
        if (RECON == 12) lds_link12(links_own + MU * lblk, n, lcb, u);       \
        else lds_link(links_own + MU * lblk, n, lcb, u);                     \
        hop_dir<MU, true>(psi, u, acc);                                      \
    }                                                                        \
    if (IN_B) {                                                              \
        lds_spinor<T>(in, n, (NB_B), psi);                                   \
        if (RECON == 12) lds_link12(links_opp + MU * lblk, n, (NB_B), u);    \
        else lds_link(links_opp + MU * lblk, n, (NB_B), u);                  \
        hop_dir<MU, false>(psi, u, acc);                                     \
    }
    DDAMG_BHOP(0, s.lx + 1 < sg.B[0], lcb + s.q, s.lx > 0, lcb + s.q - 1)
    DDAMG_BHOP(1, s.ly + 1 < sg.B[1], lcb + sy, s.ly > 0, lcb - sy)
    DDAMG_BHOP(2, s.lz + 1 < sg.B[2], lcb + sz, s.lz > 0, lcb - sz)
    DDAMG_BHOP(3, s.lt + 1 < sg.B[3], lcb + st, s.lt > 0, lcb - st)
#undef DDAMG_BHOP
}

// MAXT = 128: blocks of up to 256 sites (the 4^4 default), two (18-real links) or three (two-row links, fp32)
// CTAs per SM; MAXT = 256: blocks of up to 512 sites.  B4: the block is 4^4 (Table 6's aggregate size, the
// default): every extent, stride and shared-memory plane offset is a compile-time constant, which removes the
// address arithmetic of the ~90 shared-memory and ~20 global accesses of a half step.
#ifndef DDAMG_SAP_B4_SPECIALISE
#define DDAMG_SAP_B4_SPECIALISE 1
#endif
#ifndef DDAMG_SAP_STAGE_CLOVER
#define DDAMG_SAP_STAGE_CLOVER 1
#endif
// CS (fp32, two-row links, 4^4 blocks: the default case): the 6x6 blocks of the coming half step are staged in
// shared memory as well -- one TMA bulk copy (A_oo^-1: 36.9 KB, compact A_ee: 28.7 KB) issued at the start of the
// half step by one thread, which completes behind the hopping sum; the half step's 6x6 multiplies then read
// shared memory instead of waiting for L2 / HBM (the dominant stall of the kernel without it).  111.5 KB per CTA:
// 2 CTAs per SM instead of 3.
template <typename T, int RECON, int MAXT, bool B4, bool CS>
__global__ void __launch_bounds__(MAXT, MAXT == 128 ? (RECON == 12 && sizeof(T) == 4 && !CS ? 3 : 2) : 1)
sap_block_kernel(const SapArgs<T> a)
{
    extern __shared__ __align__(16) unsigned char sap_smem[];
    SapGeom sg = a.sg;
    if (B4) {                                                  // constants the compiler propagates
        sg.B[0] = sg.B[1] = sg.B[2] = sg.B[3] = 4;
        sg.Bxh = 2;
        sg.Vbh = 128;
    }
    const int n = sg.Vbh;
    T* links = reinterpret_cast<T*>(sap_smem);                 // [parity][mu][RECON * n]
    T* S_e = links + 2 * 4 * RECON * n;                        // even-site half-block spinor
    T* S_o = S_e + 24 * n;                                     // odd-site half-block spinor
    T* C = S_o + 24 * n;                                       // CS: the staged 6x6 blocks of one parity (72 n reals)
    double* red = reinterpret_cast<double*>(C + (CS ? 72 * n : 0));    // [warp][3]
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
    // where this thread's even / odd site lives in r, rn, e: native (checkerboard index, plane stride V/2) or
    // block-ordered (local index, plane stride n, block offset 24 n reals)
    const int rstr = a.blocked ? n : a.g.Vh;
    const int ri[2] = { a.blocked ? tid : cbg[0], a.blocked ? tid : cbg[1] };
    const size_t roff = a.blocked ? bid * 24 * n : 0;
    const bool in_blk = a.blocked && !a.rin_native;            // the same for the input residual
    const int istr = in_blk ? n : a.g.Vh;
    const int ii[2] = { in_blk ? tid : cbg[0], in_blk ? tid : cbg[1] };
    const size_t ioff = in_blk ? bid * 24 * n : 0;
    const int sblk = 4 * RECON * n;                            // one parity's four link blocks in shared memory
    // ---- stage the block's links (read once from HBM per launch): the block-ordered copy has the
    // shared-memory layout, so this is ONE contiguous bulk copy (TMA engine, `cp.async.bulk`, SASS UBLKCP)
    // issued by one thread and tracked by an mbarrier; it runs behind the prologue's own global loads
    // instead of in front of them, and no thread spends instructions or registers on it.
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(red + 3 * 32);     // [0]: links (+ first blocks), [1]: 6x6 blocks
    const unsigned bar_s = (unsigned)__cvta_generic_to_shared(bar);
    const unsigned C_s = (unsigned)__cvta_generic_to_shared(C);
    if (tid == 0) {
        const unsigned bytes = (unsigned)(2 * sblk * sizeof(T));
        const unsigned cbytes = CS ? (unsigned)(72 * n * sizeof(T)) : 0u;
        const unsigned dst_s = (unsigned)__cvta_generic_to_shared(links);
        const T* src = a.blk_links + bid * 2 * sblk;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_s));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_s + 8));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_s), "r"(bytes + cbytes) : "memory");
        if (CS)                                                // A_oo^-1 first: the prologue needs it before the links
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(C_s), "l"(clov_oinv), "r"(cbytes), "r"(bar_s) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst_s), "l"(src), "r"(bytes), "r"(bar_s) : "memory");
    }
    auto wait_bar = [&](unsigned addr, unsigned parity) {
        unsigned done = 0;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    };
    if (CS) {
        __syncthreads();                                       // the barriers' init is visible
        T v[24], t[24];
        if (active) load_spinor<T, false>(a.r_o + ioff, istr, ii[1], v);
        wait_bar(bar_s, 0);                                    // links and A_oo^-1 have landed
        if (active) {
            clover_site_mul<T, LD_PLAIN>(C, n, tid, v, t);
            sts_spinor<T>(S_o, n, tid, t);
            load_spinor<T, true>(a.r_e + ioff, istr, ii[0], rho);
        }
        __syncthreads();
    } else {
        if (active) {
            // ---- eq. 2 right factor, odd half: t_o = A_oo^-1 r_o;  rho starts as r_e
            T v[24], t[24];
            load_spinor<T, false>(a.r_o + ioff, istr, ii[1], v);
            clover_site_mul<T, LD_REUSE>(clov_oinv, n, tid, v, t);
            sts_spinor<T>(S_o, n, tid, t);
            load_spinor<T, true>(a.r_e + ioff, istr, ii[0], rho);
        }
        __syncthreads();                                       // S_o complete; the barrier's init is visible
        wait_bar(bar_s, 0);                                    // wait for the links (phase 0 of the mbarrier)
    }

    // ---- the block solve as 2m+2 half steps, one copy of the block hopping code:
    //   hs = 0        even:  rho = rhat_e = r_e - H^k_eo t_o;  e = 0
    //   hs odd < last odd :  t_o = A_oo^-1 H^k_oe rho
    //   hs even > 0   even:  q = A_ee rho - H^k_eo t_o;  alpha = <q,rho>/<q,q>;  e += alpha rho;  rho -= alpha q
    //   hs = 2m+1     odd :  e_o = A_oo^-1 (r_o - H^k_oe e);  x += e
    const int last = 2 * a.m + 1;
#pragma unroll 1
    for (int hs = 0; hs <= last; ++hs) {
        const int par = hs & 1;
        if (CS && hs >= 2 && tid == 0) {
            // the 6x6 blocks of this half step (hs = 1 still finds the prologue's A_oo^-1): every thread has passed
            // the barrier that ended the previous half step, so the buffer is free; completion k = hs - 2 of bar[1]
            const unsigned cbytes = (unsigned)((par ? 72 : 2 * CLOVA_REALS) * n * sizeof(T));
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_s + 8), "r"(cbytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(C_s), "l"(par ? clov_oinv : clov_e), "r"(cbytes), "r"(bar_s + 8) : "memory");
        }
        T acc[24];
        if (active)
            hop_block<T, RECON>(sg, tid, ls[par], par ? S_e : S_o, links + par * sblk, links + (1 - par) * sblk, acc);
        if (CS && hs >= 2) wait_bar(bar_s + 8, (unsigned)par);
        if (par) {
            if (active) {
                T v[24], t[24];
                if (hs == last) {
                    load_spinor<T, false>(a.r_o + ioff, istr, ii[1], v);
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] = v[i] + (T)0.5 * acc[i];          // r_o - H e
                } else {
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] = (T)(-0.5) * acc[i];              // H rho
                }
                if (CS) clover_site_mul<T, LD_PLAIN>(C, n, tid, v, t);
                else clover_site_mul<T, LD_REUSE>(clov_oinv, n, tid, v, t);
                if (hs == last) {
                    if (a.x_assign) {
                        store_spinor<T>(a.x_o, a.g.Vh, cbg[1], t);
                        store_spinor<T>(a.x_e, a.g.Vh, cbg[0], e);
                    } else {
                        load_spinor<T, true>(a.x_o, a.g.Vh, cbg[1], v);
#pragma unroll
                        for (int i = 0; i < 24; ++i) v[i] += t[i];
                        store_spinor<T>(a.x_o, a.g.Vh, cbg[1], v);
                        load_spinor<T, true>(a.x_e, a.g.Vh, cbg[0], v);
#pragma unroll
                        for (int i = 0; i < 24; ++i) v[i] += e[i];
                        store_spinor<T>(a.x_e, a.g.Vh, cbg[0], v);
                    }
                    // the update and the residual it leaves on this block: r_k - D_k e_k = (rho, 0)
                    store_spinor<T>(a.e_o + roff, rstr, ri[1], t);
                    store_spinor<T>(a.e_e + roff, rstr, ri[0], e);
                    store_spinor<T>(a.rn_e + roff, rstr, ri[0], rho);
#pragma unroll
                    for (int i = 0; i < 24; ++i) v[i] = 0;
                    store_spinor<T>(a.rn_o + roff, rstr, ri[1], v);
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
                if (CS) clover_site_mul<T, LD_PLAIN, true>(C, n, tid, rho, q, a.c0);
                else clover_site_mul<T, LD_REUSE, true>(clov_e, n, tid, rho, q, a.c0);
#pragma unroll
                for (int i = 0; i < 24; ++i) q[i] = q[i] + (T)0.5 * acc[i];
                // <q, rho> = q^H rho and <q, q>, this site's share: the 12 complex products of the site in the
                // data precision, the sums over the block's sites in fp64
                T snr = 0, sni = 0, sdd = 0;
#pragma unroll
                for (int c = 0; c < 12; ++c) {
                    const T qr = q[2 * c], qi = q[2 * c + 1], pr = rho[2 * c], pi = rho[2 * c + 1];
                    snr = vfma(qr, pr, snr); snr = vfma(qi, pi, snr);
                    sni = vfma(qr, pi, sni); sni = vfma(-qi, pr, sni);
                    sdd = vfma(qr, qr, sdd); sdd = vfma(qi, qi, sdd);
                }
                nr = snr; ni = sni; dd = sdd;
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
template <typename T, int RECON>
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
            if (RECON == 12) store_link12(blk_links + (bid * 8 + p * 4 + mu) * 12 * n, n, i, u);
            else store_link(blk_links + (bid * 8 + p * 4 + mu) * 18 * n, n, i, u);
        }
        const T* src = p ? clov_oinv : clov_e;
#pragma unroll 1
        for (int b = 0; b < 2; ++b) {
            T c[36];
            if (p) {
                load_clover_block<T, LD_STREAM>(src, g.Vh, cbg, b, c);
                store_clover_block<T>(blk_clov + (bid * 2 + p) * 72 * n, n, i, b, c);
            } else {
                // A_ee stays in the compact form (CLOVA_REALS per block): a plain copy of its vectors
                using V = typename VecOf<T>::type;
                constexpr int NV = CLOVA_REALS / VecOf<T>::N;
                const V* sv = reinterpret_cast<const V*>(src) + (size_t)b * NV * g.Vh + cbg;
                V* dv = reinterpret_cast<V*>(blk_clov + (bid * 2 + p) * 72 * n) + (size_t)b * NV * n + i;
#pragma unroll
                for (int k = 0; k < NV; ++k) dv[(size_t)k * n] = ld_stream(sv + (size_t)k * g.Vh);
            }
        }
    }
}

template <typename T>
void launch_sap_reorder(const Geom& g, const SapGeom& sg, int recon, const void* gauge, const void* clov_e,
                        const void* clov_oinv, void* blk_links, void* blk_clov, cudaStream_t st)
{
    const int threads = (sg.Vbh + 31) / 32 * 32;
    const int grid = sg.nb[0] * sg.nb[1] * sg.nb[2] * sg.nb[3];
    if (recon == 12)
        sap_reorder_kernel<T, 12><<<grid, threads, 0, st>>>(g, sg, (const T*)gauge, (const T*)clov_e, (const T*)clov_oinv,
                                                            (T*)blk_links, (T*)blk_clov);
    else
        sap_reorder_kernel<T, 18><<<grid, threads, 0, st>>>(g, sg, (const T*)gauge, (const T*)clov_e, (const T*)clov_oinv,
                                                            (T*)blk_links, (T*)blk_clov);
}
template void launch_sap_reorder<float>(const Geom&, const SapGeom&, int, const void*, const void*, const void*, void*, void*, cudaStream_t);
template void launch_sap_reorder<double>(const Geom&, const SapGeom&, int, const void*, const void*, const void*, void*, void*, cudaStream_t);

// fp32 blocks of 4^4 sites with two-row links also stage the 6x6 blocks of one parity (sap_block_kernel<.., CS>)
static bool sap_stages_clover(const SapGeom& sg, size_t real_bytes, int recon)
{
    return DDAMG_SAP_STAGE_CLOVER && real_bytes == 4 && recon == 12 && sg.B[0] == 4 && sg.B[1] == 4 && sg.B[2] == 4 && sg.B[3] == 4;
}
size_t sap_smem_bytes(const SapGeom& sg, size_t real_bytes, int recon)
{
    return (size_t)(2 * 4 * recon + 48 + (sap_stages_clover(sg, real_bytes, recon) ? 72 : 0)) * sg.Vbh * real_bytes +
           (size_t)32 * 3 * sizeof(double) + 16;               // + the two mbarriers of the bulk copies
}

template <typename T, int RECON, int MAXT, bool B4, bool CS = false>
static cudaError_t launch_blocks_as(const SapArgs<T>& a, int threads, int grid, size_t smem, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(sap_block_kernel<T, RECON, MAXT, B4, CS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    sap_block_kernel<T, RECON, MAXT, B4, CS><<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}

template <typename T>
cudaError_t launch_sap_blocks(const Geom& g, const SapGeom& sg, int recon, double c0, int colour, int m, const void* blk_links,
                              const void* blk_clov, const void* r_e, const void* r_o, void* rn_e, void* rn_o,
                              void* e_e, void* e_o, void* x_e, void* x_o, int blocked, int rin_native, int x_assign, cudaStream_t st)
{
    SapArgs<T> a;
    a.blocked = blocked;
    a.rin_native = rin_native;
    a.x_assign = x_assign;
    a.g = g; a.sg = sg; a.colour = colour; a.m = m; a.c0 = (T)c0;
    a.blk_links = (const T*)blk_links; a.blk_clov = (const T*)blk_clov;
    a.r_e = (const T*)r_e; a.r_o = (const T*)r_o; a.rn_e = (T*)rn_e; a.rn_o = (T*)rn_o;
    a.e_e = (T*)e_e; a.e_o = (T*)e_o; a.x_e = (T*)x_e; a.x_o = (T*)x_o;
    const size_t smem = sap_smem_bytes(sg, sizeof(T), recon);
    const int threads = (sg.Vbh + 31) / 32 * 32;
    const int grid = sg.nbxh * sg.nb[1] * sg.nb[2] * sg.nb[3];
    const bool b4 = DDAMG_SAP_B4_SPECIALISE && sg.B[0] == 4 && sg.B[1] == 4 && sg.B[2] == 4 && sg.B[3] == 4;
    if constexpr (sizeof(T) == 4) {
        if (b4 && sap_stages_clover(sg, sizeof(T), recon)) return launch_blocks_as<T, 12, 128, true, true>(a, threads, grid, smem, st);
    }
    if (b4)
        return recon == 12 ? launch_blocks_as<T, 12, 128, true>(a, threads, grid, smem, st)
                           : launch_blocks_as<T, 18, 128, true>(a, threads, grid, smem, st);
    if (threads <= 128)
        return recon == 12 ? launch_blocks_as<T, 12, 128, false>(a, threads, grid, smem, st)
                           : launch_blocks_as<T, 18, 128, false>(a, threads, grid, smem, st);
    return recon == 12 ? launch_blocks_as<T, 12, SAP_MAX_THREADS, false>(a, threads, grid, smem, st)
                       : launch_blocks_as<T, 18, SAP_MAX_THREADS, false>(a, threads, grid, smem, st);
}
template cudaError_t launch_sap_blocks<float>(const Geom&, const SapGeom&, int, double, int, int, const void*, const void*,
                                              const void*, const void*, void*, void*, void*, void*, void*, void*, int, int, int, cudaStream_t);
template cudaError_t launch_sap_blocks<double>(const Geom&, const SapGeom&, int, double, int, int, const void*, const void*,
                                               const void*, const void*, void*, void*, void*, void*, void*, void*, int, int, int, cudaStream_t);

// ---- block-ordered residual and update arrays.  In the checkerboard layout a block owns 2-site (32-byte) x-runs,
// alternating with the other colour's: a launch that touches the sites of ONE colour uses every other 32-byte
// sector, i.e. half of each 64-byte DRAM access, and a warp's access to a block is 16 different lines.  r, rn and e
// are internal to SAP, so they are kept block-ordered instead -- per parity an array [block][24/N planes][n sites]
// of 16-byte vectors, block = cx + nbx (cy + nby (cz + nbz ct)) -- and every access of a block is one contiguous
// run per plane.  native -> block-ordered, both parities (Alg. 1 line 2: the first residual):
template <typename T>
__global__ void sap_spinor_to_blocked_kernel(Geom g, SapGeom sg, const T* __restrict__ s_e, const T* __restrict__ s_o,
                                             T* __restrict__ b_e, T* __restrict__ b_o)
{
    const int n = sg.Vbh, i = threadIdx.x;
    if (i >= n) return;
    int r = blockIdx.x;
    const int cx = r % sg.nb[0]; r /= sg.nb[0];
    const int cy = r % sg.nb[1]; r /= sg.nb[1];
    const int cz = r % sg.nb[2];
    const int ct = r / sg.nb[2];
    const size_t off = (size_t)blockIdx.x * 24 * n;
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        const LSite ls = lsite_of(sg, i, p);
        const int cbg = ((cx * sg.B[0] + ls.lx) >> 1) +
                        g.Lh * ((cy * sg.B[1] + ls.ly) + g.L * ((cz * sg.B[2] + ls.lz) + g.L * (ct * sg.B[3] + ls.lt)));
        T v[24];
        load_spinor<T, true>(p ? s_o : s_e, g.Vh, cbg, v);
        store_spinor<T>((p ? b_o : b_e) + off, n, i, v);
    }
}
template <typename T>
void launch_sap_spinor_to_blocked(const Geom& g, const SapGeom& sg, const void* s_e, const void* s_o, void* b_e, void* b_o,
                                  cudaStream_t st)
{
    const int threads = (sg.Vbh + 31) / 32 * 32;
    const int grid = sg.nb[0] * sg.nb[1] * sg.nb[2] * sg.nb[3];
    sap_spinor_to_blocked_kernel<T><<<grid, threads, 0, st>>>(g, sg, (const T*)s_e, (const T*)s_o, (T*)b_e, (T*)b_o);
}
template void launch_sap_spinor_to_blocked<float>(const Geom&, const SapGeom&, const void*, const void*, void*, void*, cudaStream_t);
template void launch_sap_spinor_to_blocked<double>(const Geom&, const SapGeom&, const void*, const void*, void*, void*, cudaStream_t);

// Incremental residual on block-ordered arrays, in place: for every site x of the blocks of colour `target`
//   r(x) -= sum over the neighbours y of x in OTHER blocks of H_xy e(y)
// One CTA per target block, one thread per site (even sites first); sites none of whose hops leaves the block have
// nothing to do.  Links come from the block-ordered link copy: U_mu(x) is the block's own forward link, U_mu(x - mu)
// the forward link of the neighbour block's far face.
#ifndef DDAMG_SAP_BND_MAXREG
#define DDAMG_SAP_BND_MAXREG 80      // 3 CTAs of 256 threads per SM (94 registers uncapped: 2); measured 2.05 -> 1.63 ms
#endif
template <typename T, int RECON>
__global__ void __launch_bounds__(2 * SAP_MAX_THREADS) __maxnreg__(sizeof(T) == 4 ? DDAMG_SAP_BND_MAXREG : 128)
sap_boundary_blocked_kernel(Geom g, SapGeom sg, int target, int apbc, const T* __restrict__ blk_links,
                            const T* __restrict__ e_e, const T* __restrict__ e_o, T* r_e, T* r_o,
                            const T* __restrict__ nin_e, const T* __restrict__ nin_o)
{
    // nin_e / nin_o != NULL: the input residual is still a NATIVE half-spinor pair (first pass of a call from
    // x = 0, r = b): every site of the block is read from it and written block-ordered, also those without a hop
    const int n = sg.Vbh;
    if ((int)threadIdx.x >= 2 * n) return;
    int b = blockIdx.x;
    const int cxh = b % sg.nbxh; b /= sg.nbxh;
    const int cy = b % sg.nb[1]; b /= sg.nb[1];
    const int cz = b % sg.nb[2];
    const int ct = b / sg.nb[2];
    const int cx = 2 * cxh + ((cy + cz + ct + target) & 1);
    const int c[4] = { cx, cy, cz, ct };
    const int parity = (int)threadIdx.x >= n ? 1 : 0;
    const int lcb = (int)threadIdx.x - parity * n;
    const LSite ls = lsite_of(sg, lcb, parity);
    const int l[4] = { ls.lx, ls.ly, ls.lz, ls.lt };
    bool any = false;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) any = any || l[mu] == 0 || l[mu] == sg.B[mu] - 1;
    if (!any && !nin_e) return;
    const size_t bid = (size_t)cx + (size_t)sg.nb[0] * (cy + (size_t)sg.nb[1] * (cz + (size_t)sg.nb[2] * ct));
    const T* e_in = parity ? e_e : e_o;                        // neighbours have the opposite parity
    T acc[24], psi[24], u[18];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    // neighbour across the face in direction mu (dir = +1 / -1): its block id and local index
#define DDAMG_BXHOP(MU)                                                                              \
    {                                                                                                \
        const bool t_edge_f = MU == 3 && apbc && ct == sg.nb[3] - 1;                                 \
        const bool t_edge_b = MU == 3 && apbc && ct == 0;                                            \
        if (l[MU] == sg.B[MU] - 1) {                                                                 \
            int cn[4] = { c[0], c[1], c[2], c[3] }, ln[4] = { l[0], l[1], l[2], l[3] };              \
            cn[MU] = c[MU] + 1 == sg.nb[MU] ? 0 : c[MU] + 1;                                         \
            ln[MU] = 0;                                                                              \
            const size_t nbid = (size_t)cn[0] + (size_t)sg.nb[0] * (cn[1] + (size_t)sg.nb[1] * (cn[2] + (size_t)sg.nb[2] * cn[3])); \
            const int nlcb = (ln[0] >> 1) + sg.Bxh * (ln[1] + sg.B[1] * (ln[2] + sg.B[2] * ln[3]));  \
            load_spinor<T>(e_in + nbid * 24 * n, n, nlcb, psi);                                      \
            const T* lk = blk_links + (bid * 8 + parity * 4 + MU) * RECON * n;                       \
            if (RECON == 12) load_link12(lk, n, lcb, t_edge_f ? (T)-1 : (T)1, u);                    \
            else load_link(lk, n, lcb, u);                                                           \
            hop_dir<MU, true>(psi, u, acc);                                                          \
        }                                                                                            \
        if (l[MU] == 0) {                                                                            \
            int cn[4] = { c[0], c[1], c[2], c[3] }, ln[4] = { l[0], l[1], l[2], l[3] };              \
            cn[MU] = c[MU] == 0 ? sg.nb[MU] - 1 : c[MU] - 1;                                         \
            ln[MU] = sg.B[MU] - 1;                                                                   \
            const size_t nbid = (size_t)cn[0] + (size_t)sg.nb[0] * (cn[1] + (size_t)sg.nb[1] * (cn[2] + (size_t)sg.nb[2] * cn[3])); \
            const int nlcb = (ln[0] >> 1) + sg.Bxh * (ln[1] + sg.B[1] * (ln[2] + sg.B[2] * ln[3]));  \
            load_spinor<T>(e_in + nbid * 24 * n, n, nlcb, psi);                                      \
            const T* lk = blk_links + (nbid * 8 + (1 - parity) * 4 + MU) * RECON * n;                \
            if (RECON == 12) load_link12(lk, n, nlcb, t_edge_b ? (T)-1 : (T)1, u);                   \
            else load_link(lk, n, nlcb, u);                                                          \
            hop_dir<MU, false>(psi, u, acc);                                                         \
        }                                                                                            \
    }
    DDAMG_BXHOP(0)
    DDAMG_BXHOP(1)
    DDAMG_BXHOP(2)
    DDAMG_BXHOP(3)
#undef DDAMG_BXHOP
    T* r = (parity ? r_o : r_e) + bid * 24 * n;
    T v[24];
    if (nin_e) {
        const int cbg = ((cx * sg.B[0] + l[0]) >> 1) + g.Lh * ((cy * sg.B[1] + l[1]) + g.L * ((cz * sg.B[2] + l[2]) + g.L * (ct * sg.B[3] + l[3])));
        load_spinor<T, true>(parity ? nin_o : nin_e, g.Vh, cbg, v);
    } else {
        load_spinor<T, true>(r, n, lcb, v);
    }
#pragma unroll
    for (int i = 0; i < 24; ++i) v[i] = vfma((T)0.5, acc[i], v[i]);          // r - H e,  H = -1/2 acc
    store_spinor<T>(r, n, lcb, v);
}

template <typename T>
void launch_sap_boundary_blocked(const Geom& g, const SapGeom& sg, int recon, int target, int apbc, const void* blk_links,
                                 const void* e_e, const void* e_o, void* r_e, void* r_o, const void* native_in_e,
                                 const void* native_in_o, cudaStream_t st)
{
    const int grid = sg.nbxh * sg.nb[1] * sg.nb[2] * sg.nb[3];          // blocks of one colour
    const int threads = (2 * sg.Vbh + 31) / 32 * 32;
    if (recon == 12)
        sap_boundary_blocked_kernel<T, 12><<<grid, threads, 0, st>>>(g, sg, target, apbc, (const T*)blk_links, (const T*)e_e,
                                                                     (const T*)e_o, (T*)r_e, (T*)r_o, (const T*)native_in_e,
                                                                     (const T*)native_in_o);
    else
        sap_boundary_blocked_kernel<T, 18><<<grid, threads, 0, st>>>(g, sg, target, apbc, (const T*)blk_links, (const T*)e_e,
                                                                     (const T*)e_o, (T*)r_e, (T*)r_o, (const T*)native_in_e,
                                                                     (const T*)native_in_o);
}
template void launch_sap_boundary_blocked<float>(const Geom&, const SapGeom&, int, int, int, const void*, const void*, const void*,
                                                 void*, void*, const void*, const void*, cudaStream_t);
template void launch_sap_boundary_blocked<double>(const Geom&, const SapGeom&, int, int, int, const void*, const void*, const void*,
                                                  void*, void*, const void*, const void*, cudaStream_t);

// ---- incremental residual (Alg. 1 lines 2 / 7 after the first evaluation): for every site of colour `target`
//   rn(x) = r(x) - sum over the neighbours y of x in OTHER blocks of H_xy e(y)
// Every block across a face has the other colour, i.e. was just solved and carries its update in e; hops inside
// the site's own block see no update (e is stale there and must not be read).  One thread per lattice site; the
// lanes of the other colour idle, which costs issue slots but no memory traffic (32-byte sectors: the 2-site
// x-runs of a 4-wide block are exactly one sector per plane).
template <typename T, int RECON>
__global__ void __launch_bounds__(DSLASH_THREADS)
sap_boundary_kernel(Geom g, SapGeom sg, int target, int apbc, const T* __restrict__ gauge, const T* __restrict__ e_e,
                    const T* __restrict__ e_o, const T* r_e, const T* r_o, T* rn_e, T* rn_o)
{
    const int idx = blockIdx.x * DSLASH_THREADS + threadIdx.x;
    if (idx >= 2 * g.Vh) return;
    const int parity = idx >= g.Vh ? 1 : 0, cb = idx - parity * g.Vh;
    const Site s = site_of_cb(g, cb, parity);
    const int x = 2 * s.xh + s.q;
    const int bx = x / sg.B[0], by = s.y / sg.B[1], bz = s.z / sg.B[2], bt = s.t / sg.B[3];
    if (((bx + by + bz + bt) & 1) != target) return;
    const int lx = x - bx * sg.B[0], ly = s.y - by * sg.B[1], lz = s.z - bz * sg.B[2], lt = s.t - bt * sg.B[3];
    const T* in = parity ? e_e : e_o;                          // neighbours have the opposite parity
    const size_t lblk = (size_t)RECON * g.Vh;
    const T* gauge_own = gauge + (size_t)parity * 4 * lblk;
    const T* gauge_opp = gauge + (size_t)(1 - parity) * 4 * lblk;
    const T sgn_f3 = (apbc && s.t == g.T - 1) ? (T)-1 : (T)1;
    const T sgn_b3 = (apbc && s.t == 0) ? (T)-1 : (T)1;
    T acc[24], psi[24], u[18];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
#define DDAMG_XHOP(MU, OUT_F, OUT_B)                                                           \
    if (OUT_F) {                                                                               \
        load_spinor<T>(in, g.Vh, neighbour_cb<MU, +1>(g, cb, s), psi);                         \
        if (RECON == 12) load_link12(gauge_own + MU * lblk, g.Vh, cb, MU == 3 ? sgn_f3 : (T)1, u); \
        else load_link(gauge_own + MU * lblk, g.Vh, cb, u);                                    \
        hop_dir<MU, true>(psi, u, acc);                                                        \
    }                                                                                          \
    if (OUT_B) {                                                                               \
        const int nb = neighbour_cb<MU, -1>(g, cb, s);                                         \
        load_spinor<T>(in, g.Vh, nb, psi);                                                     \
        if (RECON == 12) load_link12(gauge_opp + MU * lblk, g.Vh, nb, MU == 3 ? sgn_b3 : (T)1, u); \
        else load_link(gauge_opp + MU * lblk, g.Vh, nb, u);                                    \
        hop_dir<MU, false>(psi, u, acc);                                                       \
    }
    DDAMG_XHOP(0, lx == sg.B[0] - 1, lx == 0)
    DDAMG_XHOP(1, ly == sg.B[1] - 1, ly == 0)
    DDAMG_XHOP(2, lz == sg.B[2] - 1, lz == 0)
    DDAMG_XHOP(3, lt == sg.B[3] - 1, lt == 0)
#undef DDAMG_XHOP
    const T* r = parity ? r_o : r_e;
    T* rn = parity ? rn_o : rn_e;
    T v[24];
    load_spinor<T, true>(r, g.Vh, cb, v);
#pragma unroll
    for (int i = 0; i < 24; ++i) v[i] = vfma((T)0.5, acc[i], v[i]);          // r - H e,  H = -1/2 acc
    store_spinor<T>(rn, g.Vh, cb, v);
}

template <typename T>
void launch_sap_boundary(const Geom& g, const SapGeom& sg, int recon, int target, int apbc, const void* gauge,
                         const void* e_e, const void* e_o, const void* r_e, const void* r_o, void* rn_e, void* rn_o,
                         cudaStream_t st)
{
    const int grid = (2 * g.Vh + DSLASH_THREADS - 1) / DSLASH_THREADS;
    if (recon == 12)
        sap_boundary_kernel<T, 12><<<grid, DSLASH_THREADS, 0, st>>>(g, sg, target, apbc, (const T*)gauge, (const T*)e_e,
                                                                    (const T*)e_o, (const T*)r_e, (const T*)r_o, (T*)rn_e, (T*)rn_o);
    else
        sap_boundary_kernel<T, 18><<<grid, DSLASH_THREADS, 0, st>>>(g, sg, target, apbc, (const T*)gauge, (const T*)e_e,
                                                                    (const T*)e_o, (const T*)r_e, (const T*)r_o, (T*)rn_e, (T*)rn_o);
}
template void launch_sap_boundary<float>(const Geom&, const SapGeom&, int, int, int, const void*, const void*, const void*,
                                         const void*, const void*, void*, void*, cudaStream_t);
template void launch_sap_boundary<double>(const Geom&, const SapGeom&, int, int, int, const void*, const void*, const void*,
                                          const void*, const void*, void*, void*, cudaStream_t);

}  // namespace ddamg

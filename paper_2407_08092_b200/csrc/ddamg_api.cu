// ddamg_api.cu -- the C ABI of include/ddamg.h: context, state machine, launch order.
//
// Host orchestration only: every arithmetic step of the path runs in the kernels of
// ddamg_dslash.cu / ddamg_setup.cu / ddamg_blas.cu.  Nothing here touches spinor data on the
// host, and there is no CPU fallback.
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "../../include/ddamg.h"
#include "ddamg_internal.h"

using namespace ddamg;

struct ddamg_ctx {
    Geom g;
    double csw, m0;
    int bc, prec;
    cudaStream_t stream;
    size_t real_bytes;
    size_t half_bytes;          // one native half spinor
    size_t nreal;               // reals per half spinor = 24 * Vh
    void* gauge;                // [parity][mu] link blocks
    void* gauge12;              // two-row copy of the links (option "gauge_recon" = 12), else NULL
    int recon;                  // 18 or 12: link format read by the fused hopping kernels
    unsigned int* recon_dev;    // device: largest |stored row 2 - rebuilt row 2| of the last compression
    double recon_deviation;     // host copy of it
    void* clov[2];              // [0] = A_ee blocks (compact 28-real form), [1] = A_oo^-1 blocks (packed 36-real form)
    void* tmp_o;                // t_o of eq. 3
    void* tmp_e;                // scratch half spinor (power iteration, final residual)
    void* krylov;               // (kcap + 1) half spinors
    int kcap;
    void* clov_oo;              // A itself on odd sites, compact form (built lazily: only the full operator D needs it)
    Scalars* sc2;               // device scalars of the outer FGMRES (the inner smoother uses sc)
    void* fgm_basis;            // outer FGMRES: (fgm_cap + 1) V + fgm_cap Z full-lattice vectors
    int fgm_cap;
    void* tmp_batch;            // multi-rhs t_o (batch_cap half spinors)
    double* partials_batch;     // multi-rhs reduction scratch
    int batch_cap;
    double batch_l2_bytes;      // L2 budget of the z-chunked multi-rhs traversal (option "batch_l2_bytes")
    void* sap_links;            // SAP: block-ordered copy of the links (launch_sap_reorder), or NULL
    void* sap_clov;             // SAP: block-ordered copy of A_ee / A_oo^-1
    int sap_built[4];           // block extents the two copies were built for ({0,..} = stale)
    int sap_built_recon;        // link format (18 / 12 reals) of the block-ordered link copy
    void* sap_e;                // SAP: the update e of the last solved colour, even half then odd half
    int sap_blocked;            // SAP keeps r and e block-ordered (option "sap_blocked", default 1)
    int sap_block[4];           // SAP block extents used when SAP is the FGMRES smoother (options "sap_block_x".."_t")
    // CUDA-graph replay of a history-free Richardson call (option "cuda_graph"): the 2 nu launches are captured
    // once on cap_stream (nothing ever executes there) and replayed on the context's stream
    int graph_mode;             // 0 = off, 1 = on, -1 = auto (on for lattices whose kernels are launch-bound)
    cudaStream_t cap_stream;
    cudaGraphExec_t rich_exec;
    struct RichKey { const void* b; void* x; int nu; double omega; int zero_init; int recon; } rich_key;
    long long rich_launches;    // kernel launches inside the captured graph
    double* partials;           // reduction scratch
    size_t partials_len;
    Scalars* sc;                // device scalars
    double* host_hist;          // pinned
    int* singular;              // device flag
    bool have_gauge, have_clover, have_clov_oo;
    int sticky;                 // DDAMG_OK or DDAMG_ECUDA
    long long launches;
    std::string err;
    // optional per-kernel timing
    bool timing;
    struct Ev { cudaEvent_t a, b; int which; };
    std::vector<Ev> events;     // pool of event pairs, created by ddamg_kernel_timing(1): none is created inside a timed call
    size_t ev_used;             // pairs recorded since the last reset
};

static thread_local std::string g_err_noctx;

static int fail(ddamg_ctx* c, int code, const std::string& msg)
{
    if (c) {
        c->err = msg;
        if (code == DDAMG_ECUDA) c->sticky = DDAMG_ECUDA;
    } else {
        g_err_noctx = msg;
    }
    return code;
}

static int check_cuda(ddamg_ctx* c, cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return DDAMG_OK;
    return fail(c, DDAMG_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CK(expr)                                                     \
    do {                                                             \
        int _s = check_cuda(ctx, (expr), #expr);                     \
        if (_s != DDAMG_OK) return _s;                               \
    } while (0)

// NVTX range per API call (tracing): visible to ncu --nvtx / any NVTX-aware
// profiler, a no-op costing a few ns without one.
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

#define ENTER(ctx)                                                           \
    NvtxRange nvtx_range_(__func__);                                         \
    do {                                                                     \
        if (!(ctx)) return DDAMG_EINVAL;                                     \
        if ((ctx)->sticky != DDAMG_OK) return (ctx)->sticky;                 \
    } while (0)

// Optional per-kernel timing: brackets the launches issued during its lifetime with a pair of
// pooled CUDA events on the context's stream, tagged with the kernel class `which`.
static const size_t EV_POOL_CHUNK = 4096;
static bool grow_event_pool(ddamg_ctx* ctx, size_t n)
{
    for (size_t i = 0; i < n; ++i) {
        ddamg_ctx::Ev ev;
        if (cudaEventCreate(&ev.a) != cudaSuccess) { cudaGetLastError(); return false; }
        if (cudaEventCreate(&ev.b) != cudaSuccess) { cudaGetLastError(); cudaEventDestroy(ev.a); return false; }
        ev.which = -1;
        ctx->events.push_back(ev);
    }
    return true;
}
struct KernelTimer {
    ddamg_ctx* c;
    long idx;
    KernelTimer(ddamg_ctx* ctx, int which) : c(ctx), idx(-1)
    {
        if (!c->timing) return;
        if (c->ev_used == c->events.size() && !grow_event_pool(c, EV_POOL_CHUNK)) return;   // pool exhausted: rare, outside steady state
        idx = (long)c->ev_used++;
        c->events[idx].which = which;
        cudaEventRecord(c->events[idx].a, c->stream);
    }
    ~KernelTimer() { if (idx >= 0) cudaEventRecord(c->events[idx].b, c->stream); }
};
enum { KT_A = 0, KT_B = 1, KT_EQ2 = 2, KT_BATCH_A = 3, KT_BATCH_B = 4, KT_FULL = 5, KT_SAP = 6,
       KT_MDOT = 8, KT_MAXPY = 9, KT_BLAS1 = 10 };

static int after_launch(ddamg_ctx* ctx, int n = 1)
{
    ctx->launches += n;
    return check_cuda(ctx, cudaGetLastError(), "kernel launch");
}

static void* gauge_block(ddamg_ctx* c, int parity)
{
    return (char*)c->gauge + (size_t)parity * 4 * 18 * c->g.Vh * c->real_bytes;
}

// link blocks read by the fused hopping kernels: the two-row copy when gauge_recon = 12
static void* hop_gauge_block(ddamg_ctx* c, int parity)
{
    if (c->recon == 12) return (char*)c->gauge12 + (size_t)parity * 4 * 12 * c->g.Vh * c->real_bytes;
    return gauge_block(c, parity);
}

// (Re)build the two-row copy from the packed links; refuses links that are not SU(3).
static int compress_gauge(ddamg_ctx* ctx)
{
    if (!ctx->gauge12) {
        cudaError_t e = cudaMalloc(&ctx->gauge12, (size_t)2 * 4 * 12 * ctx->g.Vh * ctx->real_bytes);
        if (e == cudaSuccess && !ctx->recon_dev) e = cudaMalloc((void**)&ctx->recon_dev, sizeof(unsigned int));
        if (e != cudaSuccess) {
            cudaGetLastError();
            cudaFree(ctx->gauge12); ctx->gauge12 = nullptr;
            ctx->recon = 18;
            return fail(ctx, DDAMG_ENOMEM, "gauge_recon: cannot allocate the two-row link copy");
        }
    }
    int s = check_cuda(ctx, cudaMemsetAsync(ctx->recon_dev, 0, sizeof(unsigned int), ctx->stream), "gauge_recon memset");
    if (s != DDAMG_OK) return s;
    if (ctx->prec == DDAMG_F32) launch_compress_gauge<float>(ctx->g, ctx->bc, ctx->gauge, ctx->gauge12, ctx->recon_dev, ctx->stream);
    else launch_compress_gauge<double>(ctx->g, ctx->bc, ctx->gauge, ctx->gauge12, ctx->recon_dev, ctx->stream);
    ctx->launches += 1;
    s = check_cuda(ctx, cudaGetLastError(), "kernel launch");
    if (s != DDAMG_OK) return s;
    float dev = 0.f;
    s = check_cuda(ctx, cudaMemcpyAsync(&dev, ctx->recon_dev, sizeof(float), cudaMemcpyDeviceToHost, ctx->stream), "gauge_recon D2H");
    if (s == DDAMG_OK) s = check_cuda(ctx, cudaStreamSynchronize(ctx->stream), "gauge_recon sync");
    if (s != DDAMG_OK) return s;
    ctx->recon_deviation = dev;
    const double tol = ctx->prec == DDAMG_F32 ? 2e-6 : 1e-12;
    if (!(dev <= tol)) {
        ctx->recon = 18;
        char msg[200];
        snprintf(msg, sizeof msg, "gauge_recon = 12 refused: links are not SU(3) (third row differs from conj(row0 x row1) by %.3g > %.1g); using 18-real links", (double)dev, tol);
        return fail(ctx, DDAMG_EINVAL, msg);
    }
    return DDAMG_OK;
}

extern "C" const char* ddamg_version(void) { return "ddamg-b200 0.1 (sm_100a)"; }

extern "C" const char* ddamg_last_error(ddamg_ctx* ctx) { return ctx ? ctx->err.c_str() : g_err_noctx.c_str(); }

extern "C" size_t ddamg_half_spinor_bytes(ddamg_ctx* ctx) { return ctx ? ctx->half_bytes : 0; }

extern "C" long long ddamg_launch_count(ddamg_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int ddamg_create(ddamg_ctx** out, int L, int T, double csw, double m0, int bc, int prec, void* cuda_stream)
{
    if (!out) return fail(nullptr, DDAMG_EINVAL, "ddamg_create: out is NULL");
    *out = nullptr;
    if (L < 2 || T < 2 || (L & 1) || (T & 1)) return fail(nullptr, DDAMG_EINVAL, "ddamg_create: L and T must be even and >= 2");
    if (bc != DDAMG_BC_PERIODIC && bc != DDAMG_BC_ANTIPERIODIC_T) return fail(nullptr, DDAMG_EINVAL, "ddamg_create: bad bc");
    if (prec != DDAMG_F32 && prec != DDAMG_F64) return fail(nullptr, DDAMG_EINVAL, "ddamg_create: bad prec");
    const double vh = 0.5 * (double)L * L * L * T;
    if (vh >= 1073741824.0) return fail(nullptr, DDAMG_EINVAL, "ddamg_create: lattice too large");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, DDAMG_ECUDA, "ddamg_create: no CUDA device (there is no CPU fallback)");
    }
    ddamg_ctx* ctx = new (std::nothrow) ddamg_ctx();
    if (!ctx) return fail(nullptr, DDAMG_ENOMEM, "ddamg_create: host allocation failed");
    ctx->g.L = L; ctx->g.T = T; ctx->g.Lh = L / 2;
    ctx->g.Vh = (int)vh;
    ctx->g.sy = ctx->g.Lh; ctx->g.sz = ctx->g.Lh * L; ctx->g.st = ctx->g.Lh * L * L;
    ctx->csw = csw; ctx->m0 = m0; ctx->bc = bc; ctx->prec = prec;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->real_bytes = prec == DDAMG_F32 ? 4 : 8;
    ctx->nreal = (size_t)24 * ctx->g.Vh;
    ctx->half_bytes = ctx->nreal * ctx->real_bytes;
    ctx->gauge12 = nullptr; ctx->recon = 18; ctx->recon_dev = nullptr; ctx->recon_deviation = 0.0;
    ctx->gauge = ctx->clov[0] = ctx->clov[1] = ctx->tmp_o = ctx->tmp_e = ctx->krylov = nullptr;
    ctx->kcap = 0;
    ctx->clov_oo = nullptr; ctx->sc2 = nullptr; ctx->fgm_basis = nullptr; ctx->fgm_cap = 0;
    ctx->tmp_batch = nullptr; ctx->partials_batch = nullptr; ctx->batch_cap = 0; ctx->batch_l2_bytes = 40e6;
    for (int mu = 0; mu < 4; ++mu) ctx->sap_block[mu] = 4;
    ctx->sap_blocked = 1;
    ctx->sap_links = ctx->sap_clov = ctx->sap_e = nullptr; ctx->sap_built_recon = 0;
    for (int mu = 0; mu < 4; ++mu) ctx->sap_built[mu] = 0;
    ctx->partials = nullptr; ctx->sc = nullptr; ctx->host_hist = nullptr; ctx->singular = nullptr;
    ctx->have_gauge = ctx->have_clover = ctx->have_clov_oo = false;
    ctx->sticky = DDAMG_OK; ctx->launches = 0; ctx->timing = false; ctx->ev_used = 0;
    ctx->graph_mode = -1; ctx->cap_stream = nullptr; ctx->rich_exec = nullptr; ctx->rich_launches = 0;
    memset(&ctx->rich_key, 0, sizeof ctx->rich_key);

    const size_t gauge_bytes = (size_t)2 * 4 * 18 * ctx->g.Vh * ctx->real_bytes;
    const size_t clov_bytes = (size_t)72 * ctx->g.Vh * ctx->real_bytes;                   // A_oo^-1: packed 36 reals per block
    const size_t clovA_bytes = (size_t)2 * CLOVA_REALS * ctx->g.Vh * ctx->real_bytes;     // A_ee: compact 28 reals per block
    const int dgrid = dslash_grid(ctx->g);
    // reduction scratch: 2 * dgrid norm partials (both parities of the full operator), or the partials of the
    // widest BLAS-1 grid (every BLAS-1 grid is <= blas_grid_cap(), whatever the vector length)
    const int bcap = blas_grid_cap();
    ctx->partials_len = (size_t)(2 * dgrid > bcap * 2 * MDOT_NB ? 2 * dgrid : bcap * 2 * MDOT_NB);
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaMalloc(&ctx->gauge, gauge_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->clov[0], clovA_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->clov[1], clov_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->tmp_o, ctx->half_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->tmp_e, ctx->half_bytes);
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->partials, ctx->partials_len * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->sc, sizeof(Scalars));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->singular, sizeof(int));
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->host_hist, sizeof(double) * (HIST_MAX + 8));
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->sc, 0, sizeof(Scalars), ctx->stream);
    if (e != cudaSuccess) {
        const int code = (e == cudaErrorMemoryAllocation) ? DDAMG_ENOMEM : DDAMG_ECUDA;
        fail(nullptr, code, std::string("ddamg_create: ") + cudaGetErrorString(e));
        cudaGetLastError();
        ddamg_destroy(ctx);
        return code;
    }
    *out = ctx;
    return DDAMG_OK;
}

extern "C" int ddamg_destroy(ddamg_ctx* ctx)
{
    if (!ctx) return DDAMG_OK;
    cudaStreamSynchronize(ctx->stream);
    for (auto& ev : ctx->events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    if (ctx->rich_exec) cudaGraphExecDestroy(ctx->rich_exec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    cudaFree(ctx->gauge12); cudaFree(ctx->recon_dev);
    cudaFree(ctx->sap_links); cudaFree(ctx->sap_clov); cudaFree(ctx->sap_e);
    cudaFree(ctx->gauge); cudaFree(ctx->clov[0]); cudaFree(ctx->clov[1]);
    cudaFree(ctx->tmp_o); cudaFree(ctx->tmp_e); cudaFree(ctx->krylov);
    cudaFree(ctx->tmp_batch); cudaFree(ctx->partials_batch);
    cudaFree(ctx->clov_oo); cudaFree(ctx->sc2); cudaFree(ctx->fgm_basis);
    cudaFree(ctx->partials); cudaFree(ctx->sc); cudaFree(ctx->singular);
    if (ctx->host_hist) cudaFreeHost(ctx->host_hist);
    cudaGetLastError();
    delete ctx;
    return DDAMG_OK;
}

// --------------------------------------------------------------------------- setup
extern "C" int ddamg_load_gauge(ddamg_ctx* ctx, const void* U, int u_prec, int on_device)
{
    ENTER(ctx);
    if (!U) return fail(ctx, DDAMG_EINVAL, "ddamg_load_gauge: U is NULL");
    if (u_prec != DDAMG_F32 && u_prec != DDAMG_F64) return fail(ctx, DDAMG_EINVAL, "ddamg_load_gauge: bad u_prec");
    const size_t in_bytes = (size_t)2 * ctx->g.Vh * 72 * (u_prec == DDAMG_F32 ? 4 : 8);
    const void* src = U;
    void* staging = nullptr;
    if (!on_device) {
        cudaError_t e = cudaMalloc(&staging, in_bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, DDAMG_ENOMEM, "ddamg_load_gauge: staging allocation failed"); }
        int s = check_cuda(ctx, cudaMemcpyAsync(staging, U, in_bytes, cudaMemcpyHostToDevice, ctx->stream), "gauge H2D");
        if (s != DDAMG_OK) { cudaFree(staging); return s; }
        src = staging;
    }
    if (ctx->prec == DDAMG_F32) {
        if (u_prec == DDAMG_F32) launch_pack_gauge<float, float>(ctx->g, ctx->bc, src, ctx->gauge, ctx->stream);
        else launch_pack_gauge<double, float>(ctx->g, ctx->bc, src, ctx->gauge, ctx->stream);
    } else {
        if (u_prec == DDAMG_F32) launch_pack_gauge<float, double>(ctx->g, ctx->bc, src, ctx->gauge, ctx->stream);
        else launch_pack_gauge<double, double>(ctx->g, ctx->bc, src, ctx->gauge, ctx->stream);
    }
    int s = after_launch(ctx);
    if (staging) {
        int s2 = check_cuda(ctx, cudaStreamSynchronize(ctx->stream), "gauge sync");
        cudaFree(staging);
        if (s == DDAMG_OK) s = s2;
    }
    if (s != DDAMG_OK) return s;
    ctx->have_gauge = true;
    ctx->have_clover = false;
    ctx->have_clov_oo = false;
    ctx->sap_built[0] = 0;
    if (ctx->recon == 12) return compress_gauge(ctx);      // option set before the links arrived
    return DDAMG_OK;
}

extern "C" int ddamg_build_clover(ddamg_ctx* ctx)
{
    ENTER(ctx);
    if (!ctx->have_gauge) return fail(ctx, DDAMG_ESTATE, "ddamg_build_clover: no gauge field loaded");
    // fast path: register-resident leaves + unpivoted LDL^H; the flag asks for the pivoted rebuild
    CK(cudaMemsetAsync(ctx->singular, 0, sizeof(int), ctx->stream));
    if (ctx->prec == DDAMG_F32)
        launch_build_clover<float>(ctx->g, ctx->csw, ctx->m0, ctx->gauge, ctx->clov[0], ctx->clov[1], nullptr, ctx->singular, ctx->stream);
    else
        launch_build_clover<double>(ctx->g, ctx->csw, ctx->m0, ctx->gauge, ctx->clov[0], ctx->clov[1], nullptr, ctx->singular, ctx->stream);
    int s = after_launch(ctx);
    if (s != DDAMG_OK) return s;
    int flag = 0;
    CK(cudaMemcpyAsync(&flag, ctx->singular, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (flag) {
        // some odd-site block has a small unpivoted pivot (indefinite or singular block): Gauss-Jordan with
        // partial pivoting for every block, which also applies the singularity criterion of reading C6
        CK(cudaMemsetAsync(ctx->singular, 0, sizeof(int), ctx->stream));
        if (ctx->prec == DDAMG_F32)
            launch_build_clover_pivoted<float>(ctx->g, ctx->csw, ctx->m0, ctx->gauge, ctx->clov[0], ctx->clov[1], nullptr, ctx->singular, ctx->stream);
        else
            launch_build_clover_pivoted<double>(ctx->g, ctx->csw, ctx->m0, ctx->gauge, ctx->clov[0], ctx->clov[1], nullptr, ctx->singular, ctx->stream);
        s = after_launch(ctx);
        if (s != DDAMG_OK) return s;
        CK(cudaMemcpyAsync(&flag, ctx->singular, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
    }
    if (flag) return fail(ctx, DDAMG_ESINGULAR, "ddamg_build_clover: a 6x6 odd-site block is numerically singular");
    ctx->have_clover = true;
    ctx->sap_built[0] = 0;                                  // SAP operand copies are stale
    return DDAMG_OK;
}

extern "C" int ddamg_pack_spinor(ddamg_ctx* ctx, const void* nat, void* x_e, void* x_o)
{
    ENTER(ctx);
    if (!nat || (!x_e && !x_o)) return fail(ctx, DDAMG_EINVAL, "ddamg_pack_spinor: NULL argument");
    if (((uintptr_t)nat & 15) != 0) return fail(ctx, DDAMG_EINVAL, "ddamg_pack_spinor: nat must be 16-byte aligned");
    if (ctx->prec == DDAMG_F32) launch_pack_spinor<float>(ctx->g, nat, x_e, x_o, ctx->stream);
    else launch_pack_spinor<double>(ctx->g, nat, x_e, x_o, ctx->stream);
    return after_launch(ctx);
}

extern "C" int ddamg_unpack_spinor(ddamg_ctx* ctx, const void* x_e, const void* x_o, void* nat)
{
    ENTER(ctx);
    if (!nat) return fail(ctx, DDAMG_EINVAL, "ddamg_unpack_spinor: nat is NULL");
    if (((uintptr_t)nat & 15) != 0) return fail(ctx, DDAMG_EINVAL, "ddamg_unpack_spinor: nat must be 16-byte aligned");
    if (ctx->prec == DDAMG_F32) launch_unpack_spinor<float>(ctx->g, x_e, x_o, nat, ctx->stream);
    else launch_unpack_spinor<double>(ctx->g, x_e, x_o, nat, ctx->stream);
    return after_launch(ctx);
}

extern "C" int ddamg_get_clover(ddamg_ctx* ctx, void* A_nat, void* Ainv_nat)
{
    ENTER(ctx);
    if (!ctx->have_clover) return fail(ctx, DDAMG_ESTATE, "ddamg_get_clover: clover not built");
    if (!A_nat && !Ainv_nat) return fail(ctx, DDAMG_EINVAL, "ddamg_get_clover: both outputs NULL");
    if (ctx->prec == DDAMG_F32) launch_get_clover<float>(ctx->g, ctx->m0 + 4.0, ctx->clov[0], ctx->clov[1], A_nat, Ainv_nat, ctx->stream);
    else launch_get_clover<double>(ctx->g, ctx->m0 + 4.0, ctx->clov[0], ctx->clov[1], A_nat, Ainv_nat, ctx->stream);
    return after_launch(ctx);
}

// --------------------------------------------------------------------------- hot path
// One fused hopping launch.  parity = parity of the output sites.
// units: 0 = single right-hand side, >= 1 = multi-rhs batch of that many threads per site (batch_units())
static int dslash(ddamg_ctx* ctx, int epi, bool norm, int parity, const void* in, const void* own, const void* rhs,
                  void* out, double omega, int which, int units = 0, size_t partials_offset = 0,
                  const void* clov_override = nullptr)
{
    double* partials = (units > 0 ? ctx->partials_batch : ctx->partials) + partials_offset;
    const void* clov = clov_override ? clov_override : ctx->clov[parity];
    KernelTimer kt(ctx, which);
    if (ctx->prec == DDAMG_F32)
        launch_dslash<float>(ctx->g, epi, norm, parity, in, hop_gauge_block(ctx, parity), hop_gauge_block(ctx, 1 - parity),
                             clov, own, rhs, out, omega, ctx->m0 + 4.0, partials, units, ctx->batch_l2_bytes, ctx->recon, ctx->bc == 1, ctx->stream);
    else
        launch_dslash<double>(ctx->g, epi, norm, parity, in, hop_gauge_block(ctx, parity), hop_gauge_block(ctx, 1 - parity),
                              clov, own, rhs, out, omega, ctx->m0 + 4.0, partials, units, ctx->batch_l2_bytes, ctx->recon, ctx->bc == 1, ctx->stream);
    return after_launch(ctx);
}

static int need_ready(ddamg_ctx* ctx, const char* who)
{
    if (!ctx->have_gauge || !ctx->have_clover)
        return fail(ctx, DDAMG_ESTATE, std::string(who) + ": load the gauge field and build the clover term first");
    return DDAMG_OK;
}

// y_e = D_S x_e  (kernel A then kernel B)
static int schur(ddamg_ctx* ctx, const void* x_e, void* y_e)
{
    int s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, ctx->tmp_o, 0.0, 0);
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_SCHUR, false, 0, ctx->tmp_o, x_e, nullptr, y_e, 0.0, 1);
}

// --------------------------------------------------------------------------- allocation-free Schur apply
// For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
// it): ddamg_apply_schur_noalloc keeps the intermediate t_o = A_oo^-1 H_oe x_e of eq. 3 -- the scratch between kernels
// A and B -- in a file-scope device array of a fixed, modest size instead of context-owned memory.  Every GPU that
// loads the library holds the array until the process exits.  In host code the array's NAME is a host-side stand-in,
// not a device address: the address a kernel may use comes from cudaGetSymbolAddress, resolved once per device with
// that device current (noalloc_scratch below) and cached.
#define DDAMG_NOALLOC_SCRATCH_BYTES (8u << 20)
static __device__ __align__(256) unsigned char g_noalloc_scratch[DDAMG_NOALLOC_SCRATCH_BYTES];
static const int NOALLOC_MAX_DEVICES = 64;
static void* g_noalloc_ptr[NOALLOC_MAX_DEVICES];            // device address of g_noalloc_scratch on device d, or NULL
static std::mutex g_noalloc_mutex;

// set-up step: device address of the scratch array on the CURRENT device (first call on a device resolves it)
static int noalloc_scratch(ddamg_ctx* ctx, void** out)
{
    int dev = -1;
    int s = check_cuda(ctx, cudaGetDevice(&dev), "cudaGetDevice");
    if (s != DDAMG_OK) return s;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(ctx, DDAMG_EINVAL, "ddamg_apply_schur_noalloc: device index out of range");
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        s = check_cuda(ctx, cudaGetSymbolAddress(&p, g_noalloc_scratch), "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (s != DDAMG_OK) return s;
        if (!p) return fail(ctx, DDAMG_ECUDA, "ddamg_apply_schur_noalloc: cudaGetSymbolAddress returned NULL");
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return DDAMG_OK;
}

extern "C" size_t ddamg_noalloc_max_bytes(void) { return (size_t)DDAMG_NOALLOC_SCRATCH_BYTES; }

extern "C" int ddamg_apply_schur_noalloc(ddamg_ctx* ctx, const void* x_e, void* y_e)
{
    ENTER(ctx);
    if (!x_e || !y_e || x_e == y_e) return fail(ctx, DDAMG_EINVAL, "ddamg_apply_schur_noalloc: NULL or aliased arguments");
    if (ctx->half_bytes > (size_t)DDAMG_NOALLOC_SCRATCH_BYTES) {
        char msg[240];
        snprintf(msg, sizeof msg, "ddamg_apply_schur_noalloc: one half spinor of this lattice is %zu bytes, more than the %u-byte "
                 "static scratch array (ddamg_noalloc_max_bytes); use ddamg_apply_schur", ctx->half_bytes, DDAMG_NOALLOC_SCRATCH_BYTES);
        return fail(ctx, DDAMG_EINVAL, msg);
    }
    int s = need_ready(ctx, "ddamg_apply_schur_noalloc");
    if (s != DDAMG_OK) return s;
    if (ctx->timing) return fail(ctx, DDAMG_ESTATE, "ddamg_apply_schur_noalloc: switch ddamg_kernel_timing off (its event pool may grow)");
    void* t_o = nullptr;
    s = noalloc_scratch(ctx, &t_o);
    if (s != DDAMG_OK) return s;
    // kernel A writes all V/2 sites of t_o before kernel B reads them: nothing in the shared array has to start at zero
    s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, t_o, 0.0, 0);
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_SCHUR, false, 0, t_o, x_e, nullptr, y_e, 0.0, 1);
}

extern "C" int ddamg_apply_schur(ddamg_ctx* ctx, const void* x_e, void* y_e)
{
    ENTER(ctx);
    if (!x_e || !y_e || x_e == y_e) return fail(ctx, DDAMG_EINVAL, "ddamg_apply_schur: NULL or aliased arguments");
    int s = need_ready(ctx, "ddamg_apply_schur");
    if (s != DDAMG_OK) return s;
    return schur(ctx, x_e, y_e);
}

static int copy_hist(ddamg_ctx* ctx, double* dst, int n, int* n_out)
{
    // nhist, then the entries
    CK(cudaMemcpyAsync(ctx->host_hist, (char*)ctx->sc + offsetof(Scalars, hist), sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    int nh = 0;
    CK(cudaMemcpyAsync(&nh, (char*)ctx->sc + offsetof(Scalars, nhist), sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (nh > n) nh = n;
    if (dst) memcpy(dst, ctx->host_hist, sizeof(double) * nh);
    if (n_out) *n_out = nh;
    return DDAMG_OK;
}

static int reset_hist(ddamg_ctx* ctx)
{
    return check_cuda(ctx, cudaMemsetAsync((char*)ctx->sc + offsetof(Scalars, nhist), 0, sizeof(int), ctx->stream), "reset hist");
}

template <typename T>
static int t_axpy_norm(ddamg_ctx* ctx, double alpha, const void* x, void* y, double* partials)
{
    return launch_axpy_norm<T>(ctx->nreal, alpha, x, y, partials, ctx->stream);
}

// The launches of one Richardson call (Alg. 4 lines 2-4), enqueued on ctx->stream.
static int richardson_enqueue(ddamg_ctx* ctx, const void* b_e, void* x_e, int nu, double omega, int zero_init, bool hist)
{
    int s = DDAMG_OK;
    int done = 0;
    if (zero_init && nu > 0) {
        // x^(0) = 0:  r = b,  x^(1) = omega b  (no operator application; Alg. 4 line 3-4)
        const int nblk = ctx->prec == DDAMG_F32 ? t_axpy_norm<float>(ctx, omega, b_e, x_e, hist ? ctx->partials : nullptr)
                                                : t_axpy_norm<double>(ctx, omega, b_e, x_e, hist ? ctx->partials : nullptr);
        s = after_launch(ctx);
        if (s != DDAMG_OK) return s;
        if (hist) { launch_finalize_norm(ctx->partials, nblk, ctx->sc, 1, ctx->stream); s = after_launch(ctx); if (s != DDAMG_OK) return s; }
        done = 1;
    } else if (zero_init) {
        CK(cudaMemsetAsync(x_e, 0, ctx->half_bytes, ctx->stream));
    }
    for (int i = done; i < nu; ++i) {
        s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, ctx->tmp_o, 0.0, 0);            // kernel A
        if (s != DDAMG_OK) return s;
        s = dslash(ctx, EPI_RICHARDSON, hist, 0, ctx->tmp_o, x_e, b_e, x_e, omega, 1);                  // kernel B'
        if (s != DDAMG_OK) return s;
        if (hist) {
            launch_finalize_norm(ctx->partials, dslash_grid(ctx->g), ctx->sc, 1, ctx->stream);
            s = after_launch(ctx);
            if (s != DDAMG_OK) return s;
        }
    }
    return DDAMG_OK;
}

// "auto": replay through a CUDA graph where the kernels are short enough for launch gaps to show
// (measured in bench.py rows.config2_richardson_8_sweeps): up to 2^19 sites per parity
static bool use_graph(ddamg_ctx* ctx) { return ctx->graph_mode == 1 || (ctx->graph_mode < 0 && ctx->g.Vh <= (1 << 19)); }

extern "C" int ddamg_richardson(ddamg_ctx* ctx, const void* b_e, void* x_e, int nu, double omega, int zero_init,
                                double* res_hist)
{
    ENTER(ctx);
    if (!b_e || !x_e || b_e == x_e || nu < 0) return fail(ctx, DDAMG_EINVAL, "ddamg_richardson: bad arguments");
    if (res_hist && nu > HIST_MAX) return fail(ctx, DDAMG_EINVAL, "ddamg_richardson: nu exceeds the history capacity");
    int s = need_ready(ctx, "ddamg_richardson");
    if (s != DDAMG_OK) return s;
    const bool hist = res_hist != nullptr;
    if (!hist && !ctx->timing && nu > 1 && use_graph(ctx)) {
        // history-free call (the smoother use): 2 nu launches with no host work in between -> one graph launch
        const ddamg_ctx::RichKey key = { b_e, x_e, nu, omega, zero_init != 0, ctx->recon };
        const ddamg_ctx::RichKey& k0 = ctx->rich_key;
        const bool same = ctx->rich_exec && k0.b == key.b && k0.x == key.x && k0.nu == key.nu && k0.omega == key.omega &&
                          k0.zero_init == key.zero_init && k0.recon == key.recon;
        if (!same) {
            if (ctx->rich_exec) { cudaGraphExecDestroy(ctx->rich_exec); ctx->rich_exec = nullptr; }
            if (!ctx->cap_stream) CK(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
            CK(cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
            cudaStream_t user = ctx->stream;
            const long long l0 = ctx->launches;
            ctx->stream = ctx->cap_stream;
            s = richardson_enqueue(ctx, b_e, x_e, nu, omega, zero_init, false);
            ctx->stream = user;
            ctx->rich_launches = ctx->launches - l0;
            ctx->launches = l0;
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamEndCapture(ctx->cap_stream, &graph);
            if (s != DDAMG_OK) { if (graph) cudaGraphDestroy(graph); return s; }
            if (e == cudaSuccess) e = cudaGraphInstantiate(&ctx->rich_exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            if (e != cudaSuccess) { ctx->rich_exec = nullptr; return check_cuda(ctx, e, "ddamg_richardson: graph capture"); }
            ctx->rich_key = key;
        }
        CK(cudaGraphLaunch(ctx->rich_exec, ctx->stream));
        ctx->launches += ctx->rich_launches;
        return DDAMG_OK;
    }
    if (hist) { s = reset_hist(ctx); if (s != DDAMG_OK) return s; }
    s = richardson_enqueue(ctx, b_e, x_e, nu, omega, zero_init, hist);
    if (s != DDAMG_OK) return s;
    if (hist && nu > 0) return copy_hist(ctx, res_hist, nu, nullptr);
    return DDAMG_OK;
}

extern "C" int ddamg_reconstruct_odd(ddamg_ctx* ctx, const void* b_o, const void* x_e, void* x_o)
{
    ENTER(ctx);
    if (!b_o || !x_e || !x_o) return fail(ctx, DDAMG_EINVAL, "ddamg_reconstruct_odd: NULL argument");
    int s = need_ready(ctx, "ddamg_reconstruct_odd");
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_CLOV_RHS_MINUS_HOP, false, 1, x_e, nullptr, b_o, x_o, 0.0, 2);
}

extern "C" int ddamg_prepare_rhs(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* bhat_e)
{
    ENTER(ctx);
    if (!b_e || !b_o || !bhat_e) return fail(ctx, DDAMG_EINVAL, "ddamg_prepare_rhs: NULL argument");
    int s = need_ready(ctx, "ddamg_prepare_rhs");
    if (s != DDAMG_OK) return s;
    if (ctx->prec == DDAMG_F32) launch_clover_apply<float>(ctx->g, ctx->clov[1], b_o, ctx->tmp_o, 0, ctx->stream);     // t_o = A_oo^-1 b_o
    else launch_clover_apply<double>(ctx->g, ctx->clov[1], b_o, ctx->tmp_o, 0, ctx->stream);
    s = after_launch(ctx);
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_RHS_MINUS_HOP, false, 0, ctx->tmp_o, nullptr, b_e, bhat_e, 0.0, 2);         // b_e - H_eo t_o
}

// --------------------------------------------------------------------------- multi-rhs (NEXT-2)
// The same operator applied to nrhs right-hand sides per pass ("apply each
// block to many vectors"): links and clover blocks are fetched once per site for all nrhs.
static int batch_ready(ddamg_ctx* ctx, int nrhs, const char* who)
{
    if (nrhs < 1 || nrhs > NRHS_MAX) return fail(ctx, DDAMG_EINVAL, std::string(who) + ": nrhs must be 1..32");
    if ((double)ctx->g.Vh * nrhs >= 2147483648.0) return fail(ctx, DDAMG_EINVAL, std::string(who) + ": V/2 * nrhs must be < 2^31");
    int s = need_ready(ctx, who);
    if (s != DDAMG_OK) return s;
    if (nrhs > ctx->batch_cap) {
        CK(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->tmp_batch); cudaFree(ctx->partials_batch);
        ctx->tmp_batch = nullptr; ctx->partials_batch = nullptr; ctx->batch_cap = 0;
        const int slots = batch_slots(nrhs, ctx->real_bytes), units = batch_units(nrhs, ctx->real_bytes);
        cudaError_t e = cudaMalloc(&ctx->tmp_batch, (size_t)slots * ctx->half_bytes);
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->partials_batch, sizeof(double) * (size_t)dslash_grid(ctx->g, units) * slots);
        if (e != cudaSuccess) {
            cudaGetLastError();
            cudaFree(ctx->tmp_batch); ctx->tmp_batch = nullptr;
            return fail(ctx, DDAMG_ENOMEM, std::string(who) + ": cannot allocate the multi-rhs workspace");
        }
        ctx->batch_cap = nrhs;
    }
    return DDAMG_OK;
}

extern "C" size_t ddamg_batch_spinor_bytes(ddamg_ctx* ctx, int nrhs)
{
    return (ctx && nrhs > 0) ? (size_t)batch_slots(nrhs, ctx->real_bytes) * ctx->half_bytes : 0;
}

static int batch_interleave(ddamg_ctx* ctx, int nrhs, bool to_batch, void* halves, void* X, const char* who)
{
    ENTER(ctx);
    if (!halves || !X || halves == X) return fail(ctx, DDAMG_EINVAL, std::string(who) + ": NULL or aliased arguments");
    if (nrhs < 1 || nrhs > NRHS_MAX || (double)ctx->g.Vh * nrhs >= 2147483648.0)
        return fail(ctx, DDAMG_EINVAL, std::string(who) + ": bad nrhs");
    if (ctx->prec == DDAMG_F32) launch_batch_interleave<float>(ctx->g, nrhs, to_batch, halves, X, ctx->stream);
    else launch_batch_interleave<double>(ctx->g, nrhs, to_batch, halves, X, ctx->stream);
    return after_launch(ctx);
}

extern "C" int ddamg_batch_interleave(ddamg_ctx* ctx, int nrhs, const void* halves, void* X)
{
    return batch_interleave(ctx, nrhs, true, const_cast<void*>(halves), X, "ddamg_batch_interleave");
}

extern "C" int ddamg_batch_deinterleave(ddamg_ctx* ctx, int nrhs, const void* X, void* halves)
{
    return batch_interleave(ctx, nrhs, false, halves, const_cast<void*>(X), "ddamg_batch_deinterleave");
}

extern "C" int ddamg_apply_schur_batch(ddamg_ctx* ctx, int nrhs, const void* X_e, void* Y_e)
{
    ENTER(ctx);
    if (!X_e || !Y_e || X_e == Y_e) return fail(ctx, DDAMG_EINVAL, "ddamg_apply_schur_batch: NULL or aliased arguments");
    int s = batch_ready(ctx, nrhs, "ddamg_apply_schur_batch");
    if (s != DDAMG_OK) return s;
    const int units = batch_units(nrhs, ctx->real_bytes);
    s = dslash(ctx, EPI_CLOV_HOP, false, 1, X_e, nullptr, nullptr, ctx->tmp_batch, 0.0, 3, units);
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_SCHUR, false, 0, ctx->tmp_batch, X_e, nullptr, Y_e, 0.0, 4, units);
}

extern "C" int ddamg_richardson_batch(ddamg_ctx* ctx, int nrhs, const void* B_e, void* X_e, int nu, double omega,
                                      int zero_init, double* res_hist)
{
    ENTER(ctx);
    if (!B_e || !X_e || B_e == X_e || nu < 0) return fail(ctx, DDAMG_EINVAL, "ddamg_richardson_batch: bad arguments");
    int s = batch_ready(ctx, nrhs, "ddamg_richardson_batch");
    if (s != DDAMG_OK) return s;
    const bool hist = res_hist != nullptr;
    if (hist && (long long)nu * nrhs > HIST_MAX) return fail(ctx, DDAMG_EINVAL, "ddamg_richardson_batch: nu * nrhs exceeds the history capacity");
    if (hist) { s = reset_hist(ctx); if (s != DDAMG_OK) return s; }
    // x^(0) = 0 is run as a full sweep on a zeroed batch (bit-identical to x = omega b)
    const int units = batch_units(nrhs, ctx->real_bytes), slots = batch_slots(nrhs, ctx->real_bytes);
    if (zero_init) CK(cudaMemsetAsync(X_e, 0, (size_t)slots * ctx->half_bytes, ctx->stream));
    for (int i = 0; i < nu; ++i) {
        s = dslash(ctx, EPI_CLOV_HOP, false, 1, X_e, nullptr, nullptr, ctx->tmp_batch, 0.0, 3, units);
        if (s != DDAMG_OK) return s;
        s = dslash(ctx, EPI_RICHARDSON, hist, 0, ctx->tmp_batch, X_e, B_e, X_e, omega, 4, units);
        if (s != DDAMG_OK) return s;
        if (hist) {
            launch_finalize_norm_batch(ctx->partials_batch, dslash_grid(ctx->g, units), nrhs, slots, ctx->sc, i * nrhs, ctx->stream);
            s = after_launch(ctx);
            if (s != DDAMG_OK) return s;
        }
    }
    if (hist && nu > 0) return copy_hist(ctx, res_hist, nu * nrhs, nullptr);
    return DDAMG_OK;
}

extern "C" int ddamg_reconstruct_odd_batch(ddamg_ctx* ctx, int nrhs, const void* B_o, const void* X_e, void* X_o)
{
    ENTER(ctx);
    if (!B_o || !X_e || !X_o) return fail(ctx, DDAMG_EINVAL, "ddamg_reconstruct_odd_batch: NULL argument");
    int s = batch_ready(ctx, nrhs, "ddamg_reconstruct_odd_batch");
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_CLOV_RHS_MINUS_HOP, false, 1, X_e, nullptr, B_o, X_o, 0.0, 2, batch_units(nrhs, ctx->real_bytes));
}

extern "C" int ddamg_prepare_rhs_batch(ddamg_ctx* ctx, int nrhs, const void* B_e, const void* B_o, void* Bhat_e)
{
    ENTER(ctx);
    if (!B_e || !B_o || !Bhat_e) return fail(ctx, DDAMG_EINVAL, "ddamg_prepare_rhs_batch: NULL argument");
    int s = batch_ready(ctx, nrhs, "ddamg_prepare_rhs_batch");
    if (s != DDAMG_OK) return s;
    const int units = batch_units(nrhs, ctx->real_bytes);
    if (ctx->prec == DDAMG_F32) launch_clover_apply<float>(ctx->g, ctx->clov[1], B_o, ctx->tmp_batch, units, ctx->stream);
    else launch_clover_apply<double>(ctx->g, ctx->clov[1], B_o, ctx->tmp_batch, units, ctx->stream);
    s = after_launch(ctx);
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_RHS_MINUS_HOP, false, 0, ctx->tmp_batch, nullptr, B_e, Bhat_e, 0.0, 2, units);
}

// --------------------------------------------------------------------------- GMRES
template <typename T>
static int gmres_impl(ddamg_ctx* ctx, const void* b_e, void* x_e, int k, int cycles, double tol, int zero_init,
                      double* res_hist, int* n_hist)
{
    cudaStream_t st = ctx->stream;
    const size_t nreal = ctx->nreal;
    const int dgrid = dslash_grid(ctx->g);
    int nblk = 0;                                                        // partial blocks of the last BLAS-1 reduction
    char* V = (char*)ctx->krylov;
    auto Vj = [&](int j) { return (void*)(V + (size_t)j * ctx->half_bytes); };
    // The basis is kept lazily normalised: slot i holds an un-normalised vector and the device
    // scalar vs[i] its factor, v_i = vs[i] * stored_i.  The normalisation pass v_{j+1} = w / h_{j+1,j}
    // (one read and one write of a half spinor per Arnoldi step) disappears: its factor goes into the
    // dot products, the axpy coefficients and the final x += V y instead (scalar work only).
    double* coef_ys = (double*)((char*)ctx->sc + offsetof(Scalars, ys));
    double* coef_negh = (double*)((char*)ctx->sc + offsetof(Scalars, negh));
    double* vs = (double*)((char*)ctx->sc + offsetof(Scalars, vs));
    // a second Gram-Schmidt pass (CGS2) where a long cycle or a tolerance exit relies on the Givens estimates
    const bool cgs2 = k > MDOT_NB || tol > 0.0;
    int s = reset_hist(ctx);
    if (s != DDAMG_OK) return s;
    double bnorm = 0.0;
    if (tol > 0.0) {
        nblk = launch_copy_norm<T>(nreal, b_e, Vj(0), ctx->partials, st);
        launch_finalize_norm(ctx->partials, nblk, ctx->sc, 0, st);
        s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
        CK(cudaMemcpyAsync(&bnorm, (char*)ctx->sc + offsetof(Scalars, value), sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    if (zero_init) CK(cudaMemsetAsync(x_e, 0, ctx->half_bytes, st));
    bool converged = false;
    for (int c = 0; c < cycles && !converged; ++c) {
        // line 2: r = b - D_S x, beta = ||r||
        if (zero_init && c == 0) {
            { KernelTimer kt(ctx, KT_BLAS1); nblk = launch_copy_norm<T>(nreal, b_e, Vj(0), ctx->partials, st); }
            s = after_launch(ctx); if (s != DDAMG_OK) return s;
            launch_finalize_norm(ctx->partials, nblk, ctx->sc, 1, st);
        } else {
            s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, ctx->tmp_o, 0.0, 0);
            if (s != DDAMG_OK) return s;
            s = dslash(ctx, EPI_RESIDUAL, true, 0, ctx->tmp_o, x_e, b_e, Vj(0), 0.0, 1);
            if (s != DDAMG_OK) return s;
            launch_finalize_norm(ctx->partials, dgrid, ctx->sc, 1, st);
        }
        launch_gmres_begin_cycle(ctx->sc, st);                           // v_1 = r / beta as (vs[0] = 1 / beta, r)
        s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
        if (tol > 0.0) {
            double beta = 0.0;
            CK(cudaMemcpyAsync(&beta, (char*)ctx->sc + offsetof(Scalars, value), sizeof(double), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            if (beta <= tol * bnorm) { converged = true; break; }
        }
        int m = 0;
        for (int j = 0; j < k; ++j) {
            // line 5: w = D_S v_j = vs[j] * D_S stored_j;  D_S stored_j -> V[j+1]
            s = schur(ctx, Vj(j), Vj(j + 1));
            if (s != DDAMG_OK) return s;
            // lines 6-7 (fused classical Gram-Schmidt): h_ij = <v_i, w>, i = 0..j
            for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {
                const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                { KernelTimer kt(ctx, KT_MDOT); nblk = launch_multi_dot<T>(nreal, nb, Vj(i0), nreal, Vj(j + 1), ctx->partials, st); }
                launch_finalize_dots_lazy(ctx->partials, nblk, nb, ctx->sc, i0, j, st);
                s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
            }
            // w = vs[j] V[j+1] - sum_i h_ij vs[i] stored_i ; line 8: h_{j+1,j} = ||w||
            for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {
                const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                const bool last = i0 + MDOT_NB > j;
                {
                    KernelTimer kt(ctx, KT_MAXPY);
                    nblk = launch_multi_axpy<T>(nreal, nb, Vj(i0), nreal, coef_negh + 2 * i0, Vj(j + 1), last ? ctx->partials : nullptr, st,
                                                i0 == 0 ? vs + j : nullptr);
                }
                s = after_launch(ctx); if (s != DDAMG_OK) return s;
            }
            if (cgs2) {
                // second pass: one classical Gram-Schmidt pass loses orthogonality like eps * cond(basis)^2, which in
                // fp32 shows in the Givens estimates of long cycles; the correction h' = <v_i, w> is added to h_ij
                for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {
                    const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                    { KernelTimer kt(ctx, KT_MDOT); nblk = launch_multi_dot<T>(nreal, nb, Vj(i0), nreal, Vj(j + 1), ctx->partials, st); }
                    launch_finalize_dots_lazy2(ctx->partials, nblk, nb, ctx->sc, i0, st);
                    s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
                }
                for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {
                    const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                    const bool last = i0 + MDOT_NB > j;
                    { KernelTimer kt(ctx, KT_MAXPY); nblk = launch_multi_axpy<T>(nreal, nb, Vj(i0), nreal, coef_negh + 2 * i0, Vj(j + 1), last ? ctx->partials : nullptr, st); }
                    s = after_launch(ctx); if (s != DDAMG_OK) return s;
                }
            }
            launch_finalize_norm(ctx->partials, nblk, ctx->sc, 0, st);
            launch_gmres_givens(ctx->sc, j, st);                         // also vs[j+1] = 1 / h_{j+1,j}
            s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
            m = j + 1;
            if (tol > 0.0) {
                int nh = 0;
                CK(cudaMemcpyAsync(&nh, (char*)ctx->sc + offsetof(Scalars, nhist), sizeof(int), cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                double est = 0.0;
                CK(cudaMemcpyAsync(&est, (char*)ctx->sc + offsetof(Scalars, hist) + sizeof(double) * (nh - 1), sizeof(double), cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                if (est <= tol * bnorm) break;
            }
        }
        // line 10: y = argmin, x += V_m y
        launch_gmres_solve(ctx->sc, m, st);
        s = after_launch(ctx); if (s != DDAMG_OK) return s;
        for (int i0 = 0; i0 < m; i0 += MDOT_NB) {
            const int nb = (m - i0) < MDOT_NB ? (m - i0) : MDOT_NB;
            { KernelTimer kt(ctx, KT_MAXPY); launch_multi_axpy<T>(nreal, nb, Vj(i0), nreal, coef_ys + 2 * i0, x_e, nullptr, st); }
            s = after_launch(ctx); if (s != DDAMG_OK) return s;
        }
    }
    if (!converged) {
        // true residual at the end
        s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, ctx->tmp_o, 0.0, 0);
        if (s != DDAMG_OK) return s;
        s = dslash(ctx, EPI_RESIDUAL, true, 0, ctx->tmp_o, x_e, b_e, Vj(0), 0.0, 1);
        if (s != DDAMG_OK) return s;
        launch_finalize_norm(ctx->partials, dgrid, ctx->sc, 1, st);
        s = after_launch(ctx); if (s != DDAMG_OK) return s;
    }
    return copy_hist(ctx, res_hist, cycles * (k + 1) + 1, n_hist);
}

extern "C" int ddamg_gmres_oe(ddamg_ctx* ctx, const void* b_e, void* x_e, int k, int cycles, double tol, int zero_init,
                              double* res_hist, int* n_hist)
{
    ENTER(ctx);
    if (!b_e || !x_e || b_e == x_e || k < 1 || cycles < 1 || tol < 0.0)
        return fail(ctx, DDAMG_EINVAL, "ddamg_gmres_oe: bad arguments");
    if (k > GMRES_KMAX) return fail(ctx, DDAMG_EINVAL, "ddamg_gmres_oe: k exceeds GMRES_KMAX (64)");
    if ((long long)cycles * (k + 1) + 1 > HIST_MAX) return fail(ctx, DDAMG_EINVAL, "ddamg_gmres_oe: history too long");
    int s = need_ready(ctx, "ddamg_gmres_oe");
    if (s != DDAMG_OK) return s;
    if (k > ctx->kcap) {
        CK(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->krylov);
        ctx->krylov = nullptr; ctx->kcap = 0;
        cudaError_t e = cudaMalloc(&ctx->krylov, (size_t)(k + 1) * ctx->half_bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, DDAMG_ENOMEM, "ddamg_gmres_oe: cannot allocate the Krylov basis"); }
        ctx->kcap = k;
    }
    if (ctx->prec == DDAMG_F32) return gmres_impl<float>(ctx, b_e, x_e, k, cycles, tol, zero_init, res_hist, n_hist);
    return gmres_impl<double>(ctx, b_e, x_e, k, cycles, tol, zero_init, res_hist, n_hist);
}

// --------------------------------------------------------------------------- GCR (NEXT-4)
static int ensure_krylov(ddamg_ctx* ctx, int nvec, const char* who)
{
    if (nvec <= ctx->kcap + 1) return DDAMG_OK;
    CK(cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->krylov);
    ctx->krylov = nullptr; ctx->kcap = 0;
    cudaError_t e = cudaMalloc(&ctx->krylov, (size_t)nvec * ctx->half_bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, DDAMG_ENOMEM, std::string(who) + ": cannot allocate the Krylov vectors"); }
    ctx->kcap = nvec - 1;
    return DDAMG_OK;
}

template <typename T>
static int gcr_impl(ddamg_ctx* ctx, const void* b_e, void* x_e, int k, int cycles, double tol, int zero_init,
                    double* res_hist, int* n_hist)
{
    cudaStream_t st = ctx->stream;
    const size_t nreal = ctx->nreal;
    const int dgrid = dslash_grid(ctx->g);
    int nblk = 0;                                                        // partial blocks of the last BLAS-1 reduction
    char* base = (char*)ctx->krylov;
    auto P = [&](int j) { return (void*)(base + (size_t)j * ctx->half_bytes); };
    auto Z = [&](int j) { return (void*)(base + (size_t)(k + j) * ctx->half_bytes); };
    void* r = (void*)(base + (size_t)(2 * k) * ctx->half_bytes);
    double* alpha = (double*)((char*)ctx->sc + offsetof(Scalars, alpha));
    double* beta = (double*)((char*)ctx->sc + offsetof(Scalars, negh));
    int s = reset_hist(ctx);
    if (s != DDAMG_OK) return s;
    double bnorm = 0.0;
    auto last_hist = [&](double* v) -> int {
        int nh = 0;
        CK(cudaMemcpyAsync(&nh, (char*)ctx->sc + offsetof(Scalars, nhist), sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        CK(cudaMemcpyAsync(v, (char*)ctx->sc + offsetof(Scalars, hist) + sizeof(double) * (nh - 1), sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return DDAMG_OK;
    };
    if (tol > 0.0) {
        nblk = launch_copy_norm<T>(nreal, b_e, r, ctx->partials, st);
        launch_finalize_norm(ctx->partials, nblk, ctx->sc, 0, st);
        s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
        CK(cudaMemcpyAsync(&bnorm, (char*)ctx->sc + offsetof(Scalars, value), sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    if (zero_init) CK(cudaMemsetAsync(x_e, 0, ctx->half_bytes, st));
    bool converged = false;
    for (int c = 0; c < cycles && !converged; ++c) {
        // line 2: r = b - D_S x
        if (zero_init && c == 0) {
            { KernelTimer kt(ctx, KT_BLAS1); nblk = launch_copy_norm<T>(nreal, b_e, r, ctx->partials, st); }
            s = after_launch(ctx); if (s != DDAMG_OK) return s;
            launch_finalize_norm(ctx->partials, nblk, ctx->sc, 1, st);
        } else {
            s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, ctx->tmp_o, 0.0, 0);
            if (s != DDAMG_OK) return s;
            s = dslash(ctx, EPI_RESIDUAL, true, 0, ctx->tmp_o, x_e, b_e, r, 0.0, 1);
            if (s != DDAMG_OK) return s;
            launch_finalize_norm(ctx->partials, dgrid, ctx->sc, 1, st);
        }
        s = after_launch(ctx); if (s != DDAMG_OK) return s;
        if (tol > 0.0) {
            double v = 0.0;
            s = last_hist(&v); if (s != DDAMG_OK) return s;
            if (v <= tol * bnorm) { converged = true; break; }
        }
        // line 4: z_1 = D_S r (p_1 = r is written by the form pass, which also gives delta_1, <z_1, r>)
        s = schur(ctx, r, Z(0));
        if (s != DDAMG_OK) return s;
        { KernelTimer kt(ctx, KT_BLAS1); nblk = launch_gcr_form<T>(nreal, 0, nullptr, nullptr, nreal, nullptr, Z(0), r, P(0), 1, ctx->partials, st); }
        s = after_launch(ctx); if (s != DDAMG_OK) return s;
        for (int j = 0; j < k; ++j) {
            launch_gcr_alpha(ctx->partials, nblk, ctx->sc, j, st);                        // lines 6-7
            { KernelTimer kt(ctx, KT_BLAS1); nblk = launch_gcr_update<T>(nreal, alpha, P(j), Z(j), x_e, r, ctx->partials, st); }   // lines 8-9
            launch_finalize_norm(ctx->partials, nblk, ctx->sc, 1, st);
            s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
            if (tol > 0.0) {
                double v = 0.0;
                s = last_hist(&v); if (s != DDAMG_OK) return s;
                if (v <= tol * bnorm) { converged = true; break; }
            }
            if (j == k - 1) break;
            s = schur(ctx, r, Z(j + 1));                                                   // line 10: w = D_S r
            if (s != DDAMG_OK) return s;
            for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {                                     // line 12
                const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                { KernelTimer kt(ctx, KT_MDOT); nblk = launch_multi_dot<T>(nreal, nb, Z(i0), nreal, Z(j + 1), ctx->partials, st); }
                launch_finalize_dots(ctx->partials, nblk, nb, ctx->sc, i0, st);
                launch_gcr_beta(ctx->sc, i0, nb, st);
                s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
            }
            for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {                                     // lines 13-14
                const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                const bool last = i0 + MDOT_NB > j;
                {
                    KernelTimer kt(ctx, KT_BLAS1);
                    nblk = launch_gcr_form<T>(nreal, nb, Z(i0), P(i0), nreal, beta + 2 * i0, Z(j + 1), r, P(j + 1), i0 == 0,
                                              last ? ctx->partials : nullptr, st);
                }
                s = after_launch(ctx); if (s != DDAMG_OK) return s;
            }
        }
    }
    if (!converged) {
        s = dslash(ctx, EPI_CLOV_HOP, false, 1, x_e, nullptr, nullptr, ctx->tmp_o, 0.0, 0);
        if (s != DDAMG_OK) return s;
        s = dslash(ctx, EPI_RESIDUAL, true, 0, ctx->tmp_o, x_e, b_e, r, 0.0, 1);
        if (s != DDAMG_OK) return s;
        launch_finalize_norm(ctx->partials, dgrid, ctx->sc, 1, st);
        s = after_launch(ctx); if (s != DDAMG_OK) return s;
    }
    return copy_hist(ctx, res_hist, cycles * (k + 1) + 1, n_hist);
}

extern "C" int ddamg_gcr_oe(ddamg_ctx* ctx, const void* b_e, void* x_e, int k, int cycles, double tol, int zero_init,
                            double* res_hist, int* n_hist)
{
    ENTER(ctx);
    if (!b_e || !x_e || b_e == x_e || k < 1 || cycles < 1 || tol < 0.0)
        return fail(ctx, DDAMG_EINVAL, "ddamg_gcr_oe: bad arguments");
    if (k > GMRES_KMAX) return fail(ctx, DDAMG_EINVAL, "ddamg_gcr_oe: k exceeds 64");
    if ((long long)cycles * (k + 1) + 1 > HIST_MAX) return fail(ctx, DDAMG_EINVAL, "ddamg_gcr_oe: history too long");
    int s = need_ready(ctx, "ddamg_gcr_oe");
    if (s != DDAMG_OK) return s;
    s = ensure_krylov(ctx, 2 * k + 1, "ddamg_gcr_oe");
    if (s != DDAMG_OK) return s;
    if (ctx->prec == DDAMG_F32) return gcr_impl<float>(ctx, b_e, x_e, k, cycles, tol, zero_init, res_hist, n_hist);
    return gcr_impl<double>(ctx, b_e, x_e, k, cycles, tol, zero_init, res_hist, n_hist);
}

// --------------------------------------------------------------------------- full operator, outer FGMRES (NEXT-4)
// D = A + H on both parities needs A_oo itself (the Schur path stores only its inverse).
static int ensure_full(ddamg_ctx* ctx, const char* who)
{
    int s = need_ready(ctx, who);
    if (s != DDAMG_OK) return s;
    if (ctx->have_clov_oo) return DDAMG_OK;
    if (!ctx->clov_oo) {
        cudaError_t e = cudaMalloc(&ctx->clov_oo, (size_t)2 * CLOVA_REALS * ctx->g.Vh * ctx->real_bytes);
        if (e != cudaSuccess) { cudaGetLastError(); ctx->clov_oo = nullptr; return fail(ctx, DDAMG_ENOMEM, std::string(who) + ": cannot allocate A_oo"); }
    }
    if (ctx->prec == DDAMG_F32)
        launch_build_clover<float>(ctx->g, ctx->csw, ctx->m0, ctx->gauge, nullptr, nullptr, ctx->clov_oo, ctx->singular, ctx->stream);
    else
        launch_build_clover<double>(ctx->g, ctx->csw, ctx->m0, ctx->gauge, nullptr, nullptr, ctx->clov_oo, ctx->singular, ctx->stream);
    s = after_launch(ctx);
    if (s != DDAMG_OK) return s;
    ctx->have_clov_oo = true;
    return DDAMG_OK;
}

// (y_e, y_o) = D (x_e, x_o)
static int apply_full(ddamg_ctx* ctx, const void* x_e, const void* x_o, void* y_e, void* y_o)
{
    int s = dslash(ctx, EPI_FULL, false, 0, x_o, x_e, nullptr, y_e, 0.0, 5);
    if (s != DDAMG_OK) return s;
    return dslash(ctx, EPI_FULL, false, 1, x_e, x_o, nullptr, y_o, 0.0, 5, 0, 0, ctx->clov_oo);
}

extern "C" int ddamg_apply_full(ddamg_ctx* ctx, const void* x_e, const void* x_o, void* y_e, void* y_o)
{
    ENTER(ctx);
    if (!x_e || !x_o || !y_e || !y_o || x_e == y_e || x_o == y_o || x_e == y_o || x_o == y_e)
        return fail(ctx, DDAMG_EINVAL, "ddamg_apply_full: NULL or aliased arguments");
    int s = ensure_full(ctx, "ddamg_apply_full");
    if (s != DDAMG_OK) return s;
    return apply_full(ctx, x_e, x_o, y_e, y_o);
}

// z = M v: one odd-even smoother call (eq. 2) from a zero initial guess
static int smoother_call(ddamg_ctx* ctx, int smoother, int s_n, int s_m, double omega, const void* v_e, const void* v_o,
                         void* z_e, void* z_o)
{
    if (smoother == DDAMG_SMOOTHER_SAP)      // z = SAP(s_n, s_m) on D z = v from z = 0 (acts on the full system, no eq. 2 wrapper)
        return ddamg_sap(ctx, v_e, v_o, z_e, z_o, s_n, s_m, ctx->sap_block, 1, nullptr);
    int s = ddamg_prepare_rhs(ctx, v_e, v_o, ctx->tmp_e);
    if (s != DDAMG_OK) return s;
    switch (smoother) {
    case DDAMG_SMOOTHER_RICHARDSON: s = ddamg_richardson(ctx, ctx->tmp_e, z_e, s_n, omega, 1, nullptr); break;
    case DDAMG_SMOOTHER_GMRES: s = ddamg_gmres_oe(ctx, ctx->tmp_e, z_e, s_m, s_n, 0.0, 1, nullptr, nullptr); break;
    case DDAMG_SMOOTHER_GCR: s = ddamg_gcr_oe(ctx, ctx->tmp_e, z_e, s_m, s_n, 0.0, 1, nullptr, nullptr); break;
    default: return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: unknown smoother");
    }
    if (s != DDAMG_OK) return s;
    return ddamg_reconstruct_odd(ctx, v_o, z_e, z_o);
}

static int copy_hist_from(ddamg_ctx* ctx, Scalars* sc, double* dst, int n, int* n_out)
{
    CK(cudaMemcpyAsync(ctx->host_hist, (char*)sc + offsetof(Scalars, hist), sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    int nh = 0;
    CK(cudaMemcpyAsync(&nh, (char*)sc + offsetof(Scalars, nhist), sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (nh > n) nh = n;
    if (dst) memcpy(dst, ctx->host_hist, sizeof(double) * nh);
    if (n_out) *n_out = nh;
    return DDAMG_OK;
}

template <typename T>
static int fgmres_impl(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* x_e, void* x_o, int k, int cycles, double tol,
                       int smoother, int s_n, int s_m, double omega, int zero_init, double* res_hist, int* n_hist)
{
    cudaStream_t st = ctx->stream;
    Scalars* sc = ctx->sc2;
    const size_t nhalf = ctx->nreal, nfull = 2 * ctx->nreal;
    const size_t full_bytes = 2 * ctx->half_bytes;
    const int dgrid = dslash_grid(ctx->g);
    int nblk = 0, nblk_b = 0;
    char* base = (char*)ctx->fgm_basis;
    auto Ve = [&](int j) { return (void*)(base + (size_t)j * full_bytes); };                       // v_j, even half
    auto Vo = [&](int j) { return (void*)(base + (size_t)j * full_bytes + ctx->half_bytes); };
    auto Ze = [&](int j) { return (void*)(base + (size_t)(k + 1 + j) * full_bytes); };             // z_j = M v_j
    auto Zo = [&](int j) { return (void*)(base + (size_t)(k + 1 + j) * full_bytes + ctx->half_bytes); };
    double* coef_y = (double*)((char*)sc + offsetof(Scalars, y));
    double* coef_negh = (double*)((char*)sc + offsetof(Scalars, negh));
    double* scale = (double*)((char*)sc + offsetof(Scalars, scale));
    double* value = (double*)((char*)sc + offsetof(Scalars, value));
    CK(cudaMemsetAsync((char*)sc + offsetof(Scalars, nhist), 0, sizeof(int), st));
    int s;
    // r = b - D x into v_0, ||r|| appended to the history
    auto residual = [&]() -> int {
        int q = dslash(ctx, EPI_FULL_RESIDUAL, true, 0, x_o, x_e, b_e, Ve(0), 0.0, 5);
        if (q != DDAMG_OK) return q;
        q = dslash(ctx, EPI_FULL_RESIDUAL, true, 1, x_e, x_o, b_o, Vo(0), 0.0, 5, 0, (size_t)dgrid, ctx->clov_oo);
        if (q != DDAMG_OK) return q;
        launch_finalize_norm(ctx->partials, 2 * dgrid, sc, 1, st);
        return after_launch(ctx);
    };
    double bnorm = 0.0;
    {   // ||b|| (the tolerance is relative to it)
        nblk_b = launch_copy_norm<T>(nhalf, b_e, Ve(0), ctx->partials, st);
        nblk_b += launch_copy_norm<T>(nhalf, b_o, Vo(0), ctx->partials + nblk_b, st);
        launch_finalize_norm(ctx->partials, nblk_b, sc, 0, st);
        s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
        if (tol > 0.0) {
            CK(cudaMemcpyAsync(&bnorm, value, sizeof(double), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    if (zero_init) {
        CK(cudaMemsetAsync(x_e, 0, ctx->half_bytes, st));
        CK(cudaMemsetAsync(x_o, 0, ctx->half_bytes, st));
    }
    bool converged = false;
    for (int c = 0; c < cycles && !converged; ++c) {
        if (zero_init && c == 0) {
            // r = b: v_0 already holds b and sc->value its norm
            launch_finalize_norm(ctx->partials, nblk_b, sc, 1, st);
            s = after_launch(ctx); if (s != DDAMG_OK) return s;
        } else {
            s = residual(); if (s != DDAMG_OK) return s;
        }
        launch_gmres_begin_cycle(sc, st);
        launch_scale_by_dev<T>(nfull, Ve(0), scale, st);
        s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
        if (tol > 0.0) {
            double beta = 0.0;
            CK(cudaMemcpyAsync(&beta, value, sizeof(double), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            if (beta <= tol * bnorm) { converged = true; break; }
        }
        int m = 0;
        for (int j = 0; j < k; ++j) {
            s = smoother_call(ctx, smoother, s_n, s_m, omega, Ve(j), Vo(j), Ze(j), Zo(j));      // z_j = M v_j
            if (s != DDAMG_OK) return s;
            s = apply_full(ctx, Ze(j), Zo(j), Ve(j + 1), Vo(j + 1));                             // w = D z_j
            if (s != DDAMG_OK) return s;
            for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {
                const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                nblk = launch_multi_dot<T>(nfull, nb, Ve(i0), nfull, Ve(j + 1), ctx->partials, st);
                launch_finalize_dots(ctx->partials, nblk, nb, sc, i0, st);
                s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
            }
            for (int i0 = 0; i0 <= j; i0 += MDOT_NB) {
                const int nb = (j + 1 - i0) < MDOT_NB ? (j + 1 - i0) : MDOT_NB;
                const bool last = i0 + MDOT_NB > j;
                nblk = launch_multi_axpy<T>(nfull, nb, Ve(i0), nfull, coef_negh + 2 * i0, Ve(j + 1), last ? ctx->partials : nullptr, st);
                s = after_launch(ctx); if (s != DDAMG_OK) return s;
            }
            launch_finalize_norm(ctx->partials, nblk, sc, 0, st);
            launch_gmres_givens(sc, j, st);
            launch_scale_by_dev<T>(nfull, Ve(j + 1), scale, st);
            s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
            m = j + 1;
            if (tol > 0.0) {
                int nh = 0;
                CK(cudaMemcpyAsync(&nh, (char*)sc + offsetof(Scalars, nhist), sizeof(int), cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                double est = 0.0;
                CK(cudaMemcpyAsync(&est, (char*)sc + offsetof(Scalars, hist) + sizeof(double) * (nh - 1), sizeof(double), cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                if (est <= tol * bnorm) break;
            }
        }
        launch_gmres_solve(sc, m, st);
        s = after_launch(ctx); if (s != DDAMG_OK) return s;
        for (int i0 = 0; i0 < m; i0 += MDOT_NB) {                                                  // x += Z_m y
            const int nb = (m - i0) < MDOT_NB ? (m - i0) : MDOT_NB;
            launch_multi_axpy<T>(nhalf, nb, Ze(i0), nfull, coef_y + 2 * i0, x_e, nullptr, st);
            launch_multi_axpy<T>(nhalf, nb, Zo(i0), nfull, coef_y + 2 * i0, x_o, nullptr, st);
            s = after_launch(ctx, 2); if (s != DDAMG_OK) return s;
        }
    }
    if (!converged) { s = residual(); if (s != DDAMG_OK) return s; }
    return copy_hist_from(ctx, sc, res_hist, cycles * (k + 1) + 1, n_hist);
}

extern "C" int ddamg_fgmres(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* x_e, void* x_o, int k, int cycles,
                            double tol, int smoother, int s_n, int s_m, double omega, int zero_init, double* res_hist,
                            int* n_hist)
{
    ENTER(ctx);
    if (!b_e || !b_o || !x_e || !x_o || b_e == x_e || b_o == x_o || k < 1 || cycles < 1 || tol < 0.0 || s_n < 1)
        return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: bad arguments");
    if ((smoother == DDAMG_SMOOTHER_GMRES || smoother == DDAMG_SMOOTHER_GCR) && (s_m < 1 || s_m > GMRES_KMAX))
        return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: bad inner cycle length");
    if (smoother == DDAMG_SMOOTHER_SAP && s_m < 1) return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: SAP needs at least one Minimal Residual iteration");
    if (smoother < DDAMG_SMOOTHER_RICHARDSON || smoother > DDAMG_SMOOTHER_SAP)
        return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: unknown smoother");
    if (k > GMRES_KMAX) return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: k exceeds 64");
    if ((long long)cycles * (k + 1) + 1 > HIST_MAX) return fail(ctx, DDAMG_EINVAL, "ddamg_fgmres: history too long");
    int s = ensure_full(ctx, "ddamg_fgmres");
    if (s != DDAMG_OK) return s;
    if (!ctx->sc2) {
        cudaError_t e = cudaMalloc((void**)&ctx->sc2, sizeof(Scalars));
        if (e != cudaSuccess) { cudaGetLastError(); ctx->sc2 = nullptr; return fail(ctx, DDAMG_ENOMEM, "ddamg_fgmres: scalars"); }
        CK(cudaMemsetAsync(ctx->sc2, 0, sizeof(Scalars), ctx->stream));
    }
    if (k > ctx->fgm_cap) {
        CK(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->fgm_basis);
        ctx->fgm_basis = nullptr; ctx->fgm_cap = 0;
        cudaError_t e = cudaMalloc(&ctx->fgm_basis, (size_t)(2 * k + 1) * 2 * ctx->half_bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, DDAMG_ENOMEM, "ddamg_fgmres: cannot allocate the V and Z bases"); }
        ctx->fgm_cap = k;
    }
    if (ctx->prec == DDAMG_F32)
        return fgmres_impl<float>(ctx, b_e, b_o, x_e, x_o, k, cycles, tol, smoother, s_n, s_m, omega, zero_init, res_hist, n_hist);
    return fgmres_impl<double>(ctx, b_e, b_o, x_e, x_o, k, cycles, tol, smoother, s_n, s_m, omega, zero_init, res_hist, n_hist);
}

// --------------------------------------------------------------------------- SAP (NEXT-3)
// Alg. 1.  Per outer iteration and colour: the global residual r = b - D x
// (lines 2 / 7) with the fused full-operator kernels, then one launch of the block-solve
// kernel over all blocks of that colour (lines 4-6 / 8-10).
static int sap_geometry(ddamg_ctx* ctx, const int* block, SapGeom* sg, const char* who)
{
    const int ext[4] = { ctx->g.L, ctx->g.L, ctx->g.L, ctx->g.T };
    long long vb = 1;
    for (int mu = 0; mu < 4; ++mu) {
        const int B = block[mu];
        if (B < 2 || (B & 1) || ext[mu] % B != 0 || ((ext[mu] / B) & 1))
            return fail(ctx, DDAMG_EINVAL, std::string(who) + ": block extents must be even and divide the lattice extents with an even quotient");
        sg->B[mu] = B;
        sg->nb[mu] = ext[mu] / B;
        vb *= B;
    }
    if (vb / 2 > SAP_MAX_THREADS) return fail(ctx, DDAMG_EINVAL, std::string(who) + ": blocks of more than 512 sites are not supported");
    sg->Bxh = sg->B[0] / 2;
    sg->Vbh = (int)(vb / 2);
    sg->nbxh = sg->nb[0] / 2;
    int dev = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        return check_cuda(ctx, cudaGetLastError(), "cudaDeviceGetAttribute");
    if (sap_smem_bytes(*sg, ctx->real_bytes, ctx->recon) > (size_t)optin)
        return fail(ctx, DDAMG_EINVAL, std::string(who) + ": the block's links do not fit in shared memory at this precision");
    return DDAMG_OK;
}

extern "C" int ddamg_sap(ddamg_ctx* ctx, const void* b_e, const void* b_o, void* x_e, void* x_o, int n, int m,
                         const int* block, int zero_init, double* res_hist)
{
    ENTER(ctx);
    if (!b_e || !b_o || !x_e || !x_o || !block || b_e == x_e || b_o == x_o || n < 0 || m < 0)
        return fail(ctx, DDAMG_EINVAL, "ddamg_sap: bad arguments");
    if (res_hist && n + 1 > HIST_MAX) return fail(ctx, DDAMG_EINVAL, "ddamg_sap: n exceeds the history capacity");
    int s = ensure_full(ctx, "ddamg_sap");
    if (s != DDAMG_OK) return s;
    SapGeom sg;
    s = sap_geometry(ctx, block, &sg, "ddamg_sap");
    if (s != DDAMG_OK) return s;
    cudaStream_t st = ctx->stream;
    const bool hist = res_hist != nullptr;
    const bool f32 = ctx->prec == DDAMG_F32;
    const int dgrid = dslash_grid(ctx->g);
    const int recon = ctx->recon;             // two-row links (validated SU(3)) are also staged as two rows in shared memory
    // block-ordered links and clover blocks for this geometry (built once, kept until the
    // gauge field, the clover term, the link format or the block extents change)
    if (m > 0 && (memcmp(ctx->sap_built, sg.B, sizeof(int) * 4) != 0 || ctx->sap_built_recon != recon)) {
        if (!ctx->sap_links) {
            cudaError_t e = cudaMalloc(&ctx->sap_links, (size_t)2 * 4 * 18 * ctx->g.Vh * ctx->real_bytes);
            if (e == cudaSuccess) e = cudaMalloc(&ctx->sap_clov, (size_t)2 * 72 * ctx->g.Vh * ctx->real_bytes);
            if (e == cudaSuccess) e = cudaMalloc(&ctx->sap_e, 2 * ctx->half_bytes);
            if (e != cudaSuccess) {
                cudaGetLastError();
                cudaFree(ctx->sap_links); ctx->sap_links = nullptr;
                cudaFree(ctx->sap_clov); ctx->sap_clov = nullptr;
                return fail(ctx, DDAMG_ENOMEM, "ddamg_sap: cannot allocate the block-ordered operand copies");
            }
        }
        if (f32) launch_sap_reorder<float>(ctx->g, sg, recon, ctx->gauge, ctx->clov[0], ctx->clov[1], ctx->sap_links, ctx->sap_clov, st);
        else launch_sap_reorder<double>(ctx->g, sg, recon, ctx->gauge, ctx->clov[0], ctx->clov[1], ctx->sap_links, ctx->sap_clov, st);
        s = after_launch(ctx);
        if (s != DDAMG_OK) return s;
        memcpy(ctx->sap_built, sg.B, sizeof(int) * 4);
        ctx->sap_built_recon = recon;
    }
    if (hist) { s = reset_hist(ctx); if (s != DDAMG_OK) return s; }
    if (zero_init && (m == 0 || n == 0)) {                   // otherwise the first solve of each colour assigns x
        CK(cudaMemsetAsync(x_e, 0, ctx->half_bytes, st));
        CK(cudaMemsetAsync(x_o, 0, ctx->half_bytes, st));
    }
    void* r_e = ctx->tmp_e;                                  // the residual r = b - D x, kept up to date incrementally
    void* r_o = ctx->tmp_o;
    void* e_e = ctx->sap_e;
    void* e_o = ctx->sap_e ? (char*)ctx->sap_e + ctx->half_bytes : nullptr;
    // r and e are BLOCK-ORDERED (ddamg_sap.cu): every launch touches the blocks of one colour, which in the native
    // layout are every other 32-byte sector.  (Option "sap_blocked" = 0 keeps them native.)
    const int blocked = ctx->sap_blocked;
    // ||r|| of the maintained residual -> history
    auto append_norm = [&]() -> int {
        const int n1 = f32 ? launch_copy_norm<float>(ctx->nreal, r_e, r_e, ctx->partials, st)
                           : launch_copy_norm<double>(ctx->nreal, r_e, r_e, ctx->partials, st);
        const int n2 = f32 ? launch_copy_norm<float>(ctx->nreal, r_o, r_o, ctx->partials + n1, st)
                           : launch_copy_norm<double>(ctx->nreal, r_o, r_o, ctx->partials + n1, st);
        launch_finalize_norm(ctx->partials, n1 + n2, ctx->sc, 1, st);
        return after_launch(ctx, 3);
    };
    // block solves of one colour (Alg. 1 lines 4-6 / 8-10), then the residual of the other colour's sites (line 7 / 2)
    // rin_native: (blocked) rin is still the native pair b; x_assign: first solve of this colour from x = 0
    auto half_iteration = [&](int colour, const void* rin_e, const void* rin_o, bool update_other, int rin_native, int x_assign) -> int {
        {
            KernelTimer kt(ctx, KT_SAP);
            cudaError_t e = f32
                ? launch_sap_blocks<float>(ctx->g, sg, recon, ctx->m0 + 4.0, colour, m, ctx->sap_links, ctx->sap_clov, rin_e, rin_o, r_e, r_o, e_e, e_o, x_e, x_o, blocked, rin_native, x_assign, st)
                : launch_sap_blocks<double>(ctx->g, sg, recon, ctx->m0 + 4.0, colour, m, ctx->sap_links, ctx->sap_clov, rin_e, rin_o, r_e, r_o, e_e, e_o, x_e, x_o, blocked, rin_native, x_assign, st);
            if (e != cudaSuccess) return check_cuda(ctx, e, "sap_block_kernel attributes");
        }
        int q = after_launch(ctx);
        if (q != DDAMG_OK || !update_other) return q;
        {
            KernelTimer kt(ctx, KT_FULL);
            if (blocked) {
                const void* nin_e = rin_native ? rin_e : nullptr;
                const void* nin_o = rin_native ? rin_o : nullptr;
                if (f32) launch_sap_boundary_blocked<float>(ctx->g, sg, recon, 1 - colour, ctx->bc == 1, ctx->sap_links, e_e, e_o, r_e, r_o, nin_e, nin_o, st);
                else launch_sap_boundary_blocked<double>(ctx->g, sg, recon, 1 - colour, ctx->bc == 1, ctx->sap_links, e_e, e_o, r_e, r_o, nin_e, nin_o, st);
            } else {
                if (f32) launch_sap_boundary<float>(ctx->g, sg, recon, 1 - colour, ctx->bc == 1, hop_gauge_block(ctx, 0), e_e, e_o, rin_e, rin_o, r_e, r_o, st);
                else launch_sap_boundary<double>(ctx->g, sg, recon, 1 - colour, ctx->bc == 1, hop_gauge_block(ctx, 0), e_e, e_o, rin_e, rin_o, r_e, r_o, st);
            }
        }
        return after_launch(ctx);
    };
    auto to_blocked = [&](const void* s_e, const void* s_o) -> int {
        if (f32) launch_sap_spinor_to_blocked<float>(ctx->g, sg, s_e, s_o, r_e, r_o, st);
        else launch_sap_spinor_to_blocked<double>(ctx->g, sg, s_e, s_o, r_e, r_o, st);
        return after_launch(ctx);
    };
    if (m == 0 || n == 0) {
        // zero Minimal Residual iterations: every e_k = 0, SAP is the identity; the history repeats ||b - D x||
        if (hist) {
            s = dslash(ctx, EPI_FULL_RESIDUAL, true, 0, x_o, x_e, b_e, r_e, 0.0, 5);
            if (s != DDAMG_OK) return s;
            s = dslash(ctx, EPI_FULL_RESIDUAL, true, 1, x_e, x_o, b_o, r_o, 0.0, 5, 0, (size_t)dgrid, ctx->clov_oo);
            if (s != DDAMG_OK) return s;
            for (int i = 0; i <= n; ++i) { launch_finalize_norm(ctx->partials, 2 * dgrid, ctx->sc, 1, st); s = after_launch(ctx); if (s != DDAMG_OK) return s; }
            return copy_hist(ctx, res_hist, n + 1, nullptr);
        }
        return DDAMG_OK;
    }
    // Alg. 1 line 2, first iteration: r = b - D x, evaluated in full once (x = 0: r = b itself -- the smoother use,
    // PAPER.md:55); afterwards every block solve and boundary pass keeps r current
    const void* rin_e = b_e;
    const void* rin_o = b_o;
    int native0 = 0;
    if (!zero_init) {
        // blocked: the residual is formed in the (still unused) e arrays and re-ordered into r
        void* t_e = blocked ? e_e : r_e;
        void* t_o = blocked ? e_o : r_o;
        s = dslash(ctx, EPI_FULL_RESIDUAL, hist, 0, x_o, x_e, b_e, t_e, 0.0, 5);
        if (s != DDAMG_OK) return s;
        s = dslash(ctx, EPI_FULL_RESIDUAL, hist, 1, x_e, x_o, b_o, t_o, 0.0, 5, 0, (size_t)dgrid, ctx->clov_oo);
        if (s != DDAMG_OK) return s;
        if (hist) { launch_finalize_norm(ctx->partials, 2 * dgrid, ctx->sc, 1, st); s = after_launch(ctx); if (s != DDAMG_OK) return s; }
        if (blocked) { s = to_blocked(t_e, t_o); if (s != DDAMG_OK) return s; }
        rin_e = r_e; rin_o = r_o;
    } else if (blocked && hist) {
        s = to_blocked(b_e, b_o);                                                      // r = b, block-ordered
        if (s != DDAMG_OK) return s;
        s = append_norm(); if (s != DDAMG_OK) return s;                                // ||b||
        rin_e = r_e; rin_o = r_o;
    } else if (blocked) {
        native0 = 1;           // the smoother use: the first red solves and the first boundary pass read b in place
    } else if (hist) {
        // ||b||: reduce b without touching it
        const int n1 = f32 ? launch_copy_norm<float>(ctx->nreal, b_e, r_e, ctx->partials, st) : launch_copy_norm<double>(ctx->nreal, b_e, r_e, ctx->partials, st);
        const int n2 = f32 ? launch_copy_norm<float>(ctx->nreal, b_o, r_o, ctx->partials + n1, st) : launch_copy_norm<double>(ctx->nreal, b_o, r_o, ctx->partials + n1, st);
        launch_finalize_norm(ctx->partials, n1 + n2, ctx->sc, 1, st);
        s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
        rin_e = r_e; rin_o = r_o;
    }
    for (int i = 0; i < n; ++i) {
        if (i > 0 && hist) { s = append_norm(); if (s != DDAMG_OK) return s; }       // line 2: ||r|| before iteration i
        const int first = zero_init && i == 0;                                         // x = 0: the solves assign x
        s = half_iteration(0, rin_e, rin_o, true, native0 && i == 0, first);           // red blocks, then r on the black sites
        if (s != DDAMG_OK) return s;
        rin_e = r_e; rin_o = r_o;
        s = half_iteration(1, r_e, r_o, i + 1 < n || hist, 0, first);                  // black blocks, then r on the red sites
        if (s != DDAMG_OK) return s;
    }
    if (hist) {
        s = append_norm(); if (s != DDAMG_OK) return s;                                // final residual
        return copy_hist(ctx, res_hist, n + 1, nullptr);
    }
    return DDAMG_OK;
}

// --------------------------------------------------------------------------- power iteration
extern "C" int ddamg_power_iteration(ddamg_ctx* ctx, void* v_e, int iters, double* lambda_max)
{
    ENTER(ctx);
    if (!v_e || !lambda_max || iters < 1) return fail(ctx, DDAMG_EINVAL, "ddamg_power_iteration: bad arguments");
    int s = need_ready(ctx, "ddamg_power_iteration");
    if (s != DDAMG_OK) return s;
    cudaStream_t st = ctx->stream;
    int nblk = 0;
    double* scale = (double*)((char*)ctx->sc + offsetof(Scalars, scale));
    const bool f32 = ctx->prec == DDAMG_F32;
    // v <- v / ||v||
    nblk = f32 ? launch_copy_norm<float>(ctx->nreal, v_e, v_e, ctx->partials, st)
               : launch_copy_norm<double>(ctx->nreal, v_e, v_e, ctx->partials, st);
    launch_finalize_norm(ctx->partials, nblk, ctx->sc, 0, st);
    if (f32) launch_scale_by_dev<float>(ctx->nreal, v_e, scale, st);
    else launch_scale_by_dev<double>(ctx->nreal, v_e, scale, st);
    s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
    for (int i = 0; i < iters; ++i) {
        s = schur(ctx, v_e, ctx->tmp_e);                                     // w = D_S v
        if (s != DDAMG_OK) return s;
        nblk = f32 ? launch_copy_norm<float>(ctx->nreal, ctx->tmp_e, v_e, ctx->partials, st)    // v = w, |w|^2
                   : launch_copy_norm<double>(ctx->nreal, ctx->tmp_e, v_e, ctx->partials, st);
        launch_finalize_norm(ctx->partials, nblk, ctx->sc, 0, st);           // lambda = ||w||
        if (f32) launch_scale_by_dev<float>(ctx->nreal, v_e, scale, st);
        else launch_scale_by_dev<double>(ctx->nreal, v_e, scale, st);
        s = after_launch(ctx, 3); if (s != DDAMG_OK) return s;
    }
    CK(cudaMemcpyAsync(lambda_max, (char*)ctx->sc + offsetof(Scalars, value), sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return DDAMG_OK;
}

// --------------------------------------------------------------------------- options
extern "C" int ddamg_set_option(ddamg_ctx* ctx, const char* name, double value)
{
    ENTER(ctx);
    if (!name) return fail(ctx, DDAMG_EINVAL, "ddamg_set_option: name is NULL");
    if (strcmp(name, "batch_l2_bytes") == 0) {
        if (!(value >= 0.0)) return fail(ctx, DDAMG_EINVAL, "ddamg_set_option: batch_l2_bytes must be >= 0");
        ctx->batch_l2_bytes = value;
        return DDAMG_OK;
    }
    if (strcmp(name, "cuda_graph") == 0) {
        if (value != 0.0 && value != 1.0 && value != -1.0) return fail(ctx, DDAMG_EINVAL, "ddamg_set_option: cuda_graph must be 0, 1 or -1 (auto)");
        ctx->graph_mode = (int)value;
        return DDAMG_OK;
    }
    if (strcmp(name, "sap_blocked") == 0) {
        if (value != 0.0 && value != 1.0) return fail(ctx, DDAMG_EINVAL, "ddamg_set_option: sap_blocked must be 0 or 1");
        ctx->sap_blocked = (int)value;
        return DDAMG_OK;
    }
    if (strcmp(name, "gauge_recon") == 0) {
        if (value != 12.0 && value != 18.0) return fail(ctx, DDAMG_EINVAL, "ddamg_set_option: gauge_recon must be 18 or 12");
        ctx->recon = (int)value;
        if (ctx->recon == 12 && ctx->have_gauge) return compress_gauge(ctx);
        return DDAMG_OK;
    }
    static const char* const sap_names[4] = { "sap_block_x", "sap_block_y", "sap_block_z", "sap_block_t" };
    for (int mu = 0; mu < 4; ++mu)
        if (strcmp(name, sap_names[mu]) == 0) {
            const int B = (int)value;
            if ((double)B != value || B < 2 || (B & 1)) return fail(ctx, DDAMG_EINVAL, "ddamg_set_option: SAP block extents must be even integers >= 2");
            ctx->sap_block[mu] = B;
            return DDAMG_OK;
        }
    return fail(ctx, DDAMG_EINVAL, std::string("ddamg_set_option: unknown option ") + name);
}

// --------------------------------------------------------------------------- kernel timing
extern "C" int ddamg_kernel_timing(ddamg_ctx* ctx, int on)
{
    ENTER(ctx);
    if (on && ctx->events.empty() && !grow_event_pool(ctx, EV_POOL_CHUNK))      // all events are created here, not in timed calls
        return fail(ctx, DDAMG_ECUDA, "ddamg_kernel_timing: cannot create the event pool");
    ctx->timing = on != 0;
    return DDAMG_OK;
}

extern "C" int ddamg_kernel_time_ms(ddamg_ctx* ctx, int which, double* ms, long long* launches, int reset)
{
    ENTER(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    double tot = 0.0;
    long long n = 0;
    for (size_t i = 0; i < ctx->ev_used; ++i) {
        const ddamg_ctx::Ev& ev = ctx->events[i];
        if (ev.which != which) continue;
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, ev.a, ev.b));
        tot += t;
        ++n;
    }
    if (ms) *ms = tot;
    if (launches) *launches = n;
    if (reset) ctx->ev_used = 0;          // the pooled events are kept and re-recorded
    return DDAMG_OK;
}

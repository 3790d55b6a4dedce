// clt_api.cu -- the C ABI of libclt (include/clt.h): context, workspace carving, stage scheduling.
// Product code: no CPU fallback, shares nothing with oracle/.
#include "clt.h"
#include "clt_internal.h"

#include <cuda.h>

#include <math.h>
#include <new>
#include <stdio.h>
#include <string.h>
#include <vector>

using namespace clt;

// prefetch.global.L2 hints for the next plane's epilogue operands (measured choice)
#ifndef CLT_PREFETCH
#define CLT_PREFETCH 1
#endif
// L2 promotion of the TMA loads (measured choice)
#ifndef CLT_L2_PROMO
#define CLT_L2_PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_256B
#endif

struct clt_ctx {
    clt_grid grid;
    clt_params par;
    Layout L;
    Phys ph;
    cudaStream_t stream;
    // workspace carving (device)
    double *Un, *acc, *Ua, *Ub, *J1, *G, *tab, *Rtab, *invRtab, *cs, *partial, *result;
    int nblocks_diag;
    double *static_partial;        // clt_diagnostics_static: this device's address of the library's static scratch array
    int static_max_blocks;         // ... and how many reduction CTAs it holds
    bool has_state, has_v0, hall;
    int k_first, k_last, kd_first, kd_last;   // owned rows / rows of max |div_c B| (clt_set_owned_rows)
    // clt_link_rows: neighbouring slabs whose ghost rows the stage kernels of this context fill (0 = lower, 1 = upper)
    struct { clt_ctx *peer; int k0, k1, dk; } link[2];
    bool adaptive;                 // inside clt_step_cfl: stage coefficients from the device clock
    double adaptive_cfl;
    int sm_count;                  // multiprocessors of that device (automatic phi chunking of small grids)
    int device;                    // the device the workspace lives on (every call runs with it current)
    int next_stage;                // clt_step_stage: the stage expected next (1..4)
    bool spectral;                 // pseudo-spectral phi scheme (clt_set_phi_scheme)
    double *spec, *spec_ctab;      // caller-provided scratch: SPEC_COUNT derivative fields + circulant weights

    int64_t step;
    double time;
    double dt;
    int64_t launches;
    int phi_chunks, use_graph;
    int variant;      // 0 = TMA-fed fused RHS kernel (default), 1 = plain-load variant
    cudaGraphExec_t graph_exec;
    int graph_chunks;
    bool graph_v0;
    // "does the reference state move?" is decided on the device (any_nonzero_kernel) and read back lazily, so that
    // clt_set_equilibrium stays asynchronous: pinned flag + the event that marks its copy
    int *v0_flag_host;
    cudaEvent_t v0_event;
    bool v0_pending;
    char cuda_err[256];
    // per-kernel event timing (clt_set_profiling)
    bool profiling;
    std::vector<cudaEvent_t> *ev;      // pairs: start, stop
    std::vector<int> *ev_kind;         // 0..4 rhs mode, 5 curl
    std::vector<long> *ev_start;       // index of the event that marks the start of launch n (its own, or the previous end)
    bool prof_chain;                   // the last operation on the stream was the end event of the previous profiled launch
    size_t ev_used;
    int64_t ev_dropped;
};

namespace {

// makes the context's device current for the duration of an API call (callers with several GPUs in one process)
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(clt_ctx *ctx)
    {
        if (!ctx) return;
        ctx->prof_chain = false;       // whatever this call enqueues first does not follow a profiled launch back to back
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; return; }
        if (prev != ctx->device) cudaSetDevice(ctx->device); else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

constexpr size_t ALIGN = 128;   // every field and table base is 128-byte aligned
inline size_t align_up(size_t n) { return (n + ALIGN - 1) / ALIGN * ALIGN; }

bool grid_ok(const clt_grid *g)
{
    if (!g) return false;
    if (g->nR < 9 || g->nZ < 9 || g->nphi < 5) return false;
    if (g->nR > (1 << 20) || g->nZ > (1 << 20) || g->nphi > (1 << 20)) return false;
    if (!(g->Rmin > 0.0) || !(g->Rmax > g->Rmin) || !(g->Zmax > g->Zmin)) return false;
    if (!isfinite(g->Rmin) || !isfinite(g->Rmax) || !isfinite(g->Zmin) || !isfinite(g->Zmax)) return false;
    if (!isfinite(g->phi_extent) || g->phi_extent < 0.0) return false;
    return true;
}

Layout make_layout(const clt_grid *g)
{
    Layout L;
    L.nR = g->nR; L.nphi = g->nphi; L.nZ = g->nZ;
    L.pR = (LP + g->nR + 2 + 15) / 16 * 16;     // room for clamped halo reads two nodes past the edge
    L.plane = (long long)L.nZ * L.pR;
    L.field = (long long)L.nphi * L.plane;
    return L;
}

struct Carve {
    size_t field_b, table_b, rtab_b, cs_b, partial_b, result_b, total;
    int nblocks;
};
Carve carve(const clt_grid *g)
{
    Layout L = make_layout(g);
    Carve c;
    c.field_b = align_up((size_t)L.field * sizeof(double));
    c.table_b = align_up((size_t)L.plane * sizeof(double));
    c.rtab_b = align_up((size_t)L.pR * sizeof(double));
    c.cs_b = align_up((size_t)2 * g->nphi * sizeof(double));
    c.nblocks = diag_blocks(L);
    c.partial_b = align_up((size_t)c.nblocks * 6 * sizeof(double));
    // 6 diagnostics + the device clock of clt_step_cfl (6 doubles at +8) + dt minimum (at +16) + the fixed-dt stage
    // coefficients (4 doubles at +24) + the "v0 != 0" flag (at +28)
    c.result_b = align_up(32 * sizeof(double));
    c.total = 38 * c.field_b + T_COUNT * c.table_b + 2 * c.rtab_b + c.cs_b + c.partial_b + c.result_b;
    return c;
}

int cuda_fail(clt_ctx *c, cudaError_t e, const char *where)
{
    if (c) snprintf(c->cuda_err, sizeof(c->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return CLT_ECUDA;
}
#define CK(call)                                                      \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);      \
    } while (0)

// dense user array [rows][nR]  <->  padded internal rows
int copy_in(clt_ctx *ctx, double *dst_padded, const double *src, size_t rows)
{
    CK(cudaMemcpy2DAsync(dst_padded + LP, (size_t)ctx->L.pR * sizeof(double), src, (size_t)ctx->L.nR * sizeof(double),
                         (size_t)ctx->L.nR * sizeof(double), rows, cudaMemcpyDefault, ctx->stream));
    return CLT_OK;
}
int copy_out(clt_ctx *ctx, double *dst, const double *src_padded, size_t rows)
{
    CK(cudaMemcpy2DAsync(dst, (size_t)ctx->L.nR * sizeof(double), src_padded + LP, (size_t)ctx->L.pR * sizeof(double),
                         (size_t)ctx->L.nR * sizeof(double), rows, cudaMemcpyDefault, ctx->stream));
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, dst);
    if (e != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
    if (at.type != cudaMemoryTypeDevice) CK(cudaStreamSynchronize(ctx->stream));   // host destination: synchronous
    return CLT_OK;
}

void free_profile(clt_ctx *ctx)
{
    if (ctx->v0_flag_host) { cudaFreeHost(ctx->v0_flag_host); ctx->v0_flag_host = nullptr; }
    if (ctx->v0_event) { cudaEventDestroy(ctx->v0_event); ctx->v0_event = nullptr; }
    if (ctx->ev) {
        for (cudaEvent_t e : *ctx->ev) cudaEventDestroy(e);
        delete ctx->ev;
        ctx->ev = nullptr;
    }
    delete ctx->ev_kind;
    ctx->ev_kind = nullptr;
    delete ctx->ev_start;
    ctx->ev_start = nullptr;
}

void destroy_graph(clt_ctx *ctx)
{
    if (ctx->graph_exec) {
        cudaGraphExecDestroy(ctx->graph_exec);
        ctx->graph_exec = nullptr;
    }
}

// the kernels' v0 = 0 specialisation is chosen on the host: wait (once) for the flag clt_set_equilibrium requested
int resolve_v0(clt_ctx *ctx)
{
    if (!ctx->v0_pending) return CLT_OK;
    cudaError_t e = cudaEventSynchronize(ctx->v0_event);
    if (e != cudaSuccess) { snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "v0 flag: %s", cudaGetErrorString(e)); return CLT_ECUDA; }
    ctx->has_v0 = *ctx->v0_flag_host != 0;
    ctx->v0_pending = false;
    return CLT_OK;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess
            && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    }
    return fn;
}

// 4-D map (R column, Z row, phi plane, field) over nfields consecutive padded fields; box = tile with halo
// box_fields = 1: one field per copy; = nfields: one copy brings the tiles of all fields (stored field after field)
bool make_map(const clt_ctx *ctx, const double *base, int nfields, int tile_z, CUtensorMap *out, int box_fields = 1)
{
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return false;
    const Layout &L = ctx->L;
    const cuuint64_t dims[4] = { (cuuint64_t)L.pR, (cuuint64_t)L.nZ, (cuuint64_t)L.nphi, (cuuint64_t)nfields };
    const cuuint64_t strides[3] = { (cuuint64_t)L.pR * 8, (cuuint64_t)L.plane * 8, (cuuint64_t)L.field * 8 };
    const cuuint32_t box[4] = { 32 + 4, (cuuint32_t)tile_z + 4, 1, (cuuint32_t)box_fields };      // tile with the radius-2 halo
    const cuuint32_t estr[4] = { 1, 1, 1, 1 };
    return enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CLT_L2_PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)
           == CUDA_SUCCESS;
}
// phi chunks per tile (gridDim.z).  0 = automatic: one chunk, unless the grid has fewer tiles than the device has SMs
// (small grids: 128 x 16 x 128 has 64 tiles) -- then as many chunks as keep the CTA count within one wave, each at least
// 8 planes long (a chunk re-reads 4 planes of prologue).  Measured: +44 % at 128 x 16 x 128, nothing to gain from
// 256 x 32 x 256 upwards.  The result does not depend on it (bit-identical).
int effective_chunks(const clt_ctx *ctx)
{
    int c = ctx->phi_chunks;
    if (c == 0) {
        const int tiles = ((ctx->L.nR - 4 + 31) / 32) * ((ctx->L.nZ - 4 + rhs_tile_z() - 1) / rhs_tile_z());
        c = ctx->sm_count / (tiles > 0 ? tiles : 1);
        if (c > ctx->L.nphi / 8) c = ctx->L.nphi / 8;
        if (c < 1) c = 1;
    }
    if (c > ctx->L.nphi / 4) c = ctx->L.nphi / 4 > 0 ? ctx->L.nphi / 4 : 1;
    return c;
}

constexpr size_t MAX_PROFILED = 8192;

// returns the index of the event pair to use for this launch, or -1
long prof_begin(clt_ctx *ctx, int kind)
{
    if (!ctx->profiling || ctx->use_graph == 1) { ctx->prof_chain = false; return -1; }
    if (ctx->ev_used >= MAX_PROFILED) { ctx->ev_dropped++; ctx->prof_chain = false; return -1; }
    if (ctx->ev->size() < 2 * (ctx->ev_used + 1)) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
            cudaGetLastError();
            ctx->prof_chain = false;
            return -1;
        }
        ctx->ev->push_back(a); ctx->ev->push_back(b);
        ctx->ev_kind->push_back(kind);
        ctx->ev_start->push_back(0);
    }
    const long n = (long)ctx->ev_used++;
    (*ctx->ev_kind)[n] = kind;
    if (ctx->prof_chain && n > 0) {
        (*ctx->ev_start)[n] = 2 * (n - 1) + 1;      // back-to-back launches: the previous end event is this start
    } else {
        (*ctx->ev_start)[n] = 2 * n;
        cudaEventRecord((*ctx->ev)[2 * n], ctx->stream);
    }
    return n;
}
void prof_end(clt_ctx *ctx, long n)
{
    if (n >= 0) {
        cudaEventRecord((*ctx->ev)[2 * n + 1], ctx->stream);
        ctx->prof_chain = true;
    }
}

// kernels one phi pre-pass launches
int phi_launches(const clt_ctx *, int mode) { return mode == 0 ? 1 : 2; }

// NEXT-2: pseudo-spectral phi derivatives of the stage state U (mode 0: what the curl needs, 1: what the RHS needs)
int run_phi_pass(clt_ctx *ctx, int mode, const double *U)
{
    SpecArgs a;
    a.L = ctx->L; a.ph = ctx->ph;
    a.U = U; a.J1 = ctx->J1; a.tab = ctx->tab;
    a.out = ctx->spec; a.ctab = ctx->spec_ctab;
    a.mode = mode; a.hall = ctx->hall ? 1 : 0; a.has_v0 = ctx->has_v0 ? 1 : 0;
    const long pe = prof_begin(ctx, 6);
    CK(launch_phi_spectral(a, ctx->stream));
    prof_end(ctx, pe);
    ctx->launches += phi_launches(ctx, mode);
    return CLT_OK;
}

int run_curl(clt_ctx *ctx, const double *U)
{
    CurlArgs a;
    a.L = ctx->L; a.ph = ctx->ph;
    a.B = U + 5 * ctx->L.field;
    a.J1 = ctx->J1;
    a.G = ctx->G;
    a.tab = ctx->tab;
    a.R = ctx->Rtab + LP;
    a.invR = ctx->invRtab + LP;
    a.phi_chunks = effective_chunks(ctx);
    a.spec = ctx->spec;
    alignas(64) CUtensorMap tmU;
    const bool tma = ctx->variant == 0;
    if (ctx->spectral) {
        if (!tma) {
            snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "the pseudo-spectral phi scheme needs the default kernel variant");
            return CLT_EINVAL;
        }
        int r = run_phi_pass(ctx, 0, U);
        if (r) return r;
    }
    if (tma && !make_map(ctx, U, 8, curl_tma_tile_z(), &tmU)) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "cuTensorMapEncodeTiled failed");
        return CLT_ECUDA;
    }
    const long pe = prof_begin(ctx, 5);
    if (tma)
        CK(launch_curl_tma(a, &tmU, ctx->hall, ctx->spectral, ctx->stream));
    else
        CK(launch_curl(a, ctx->stream));
    prof_end(ctx, pe);
    ctx->launches++;
    return CLT_OK;
}

int run_rhs(clt_ctx *ctx, int mode, const double *in, double *out)
{
    RhsArgs a;
    a.L = ctx->L; a.ph = ctx->ph;
    a.in = in; a.J1 = ctx->J1; a.Un = ctx->Un; a.acc = ctx->acc; a.out = out;
    a.tab = ctx->tab;
    a.R = ctx->Rtab + LP;
    a.invR = ctx->invRtab + LP;
    a.phi_chunks = effective_chunks(ctx);
    a.prefetch = CLT_PREFETCH;
    a.spec = ctx->spec;
    // stage coefficients: the device clock inside clt_step_cfl, else the fixed-dt table clt_set_dt keeps up to date
    a.coef = ctx->adaptive ? ctx->result + 8 : ctx->result + 24;
    a.dtmin_bits = ctx->adaptive ? (unsigned long long *)(ctx->result + 16) : nullptr;
    a.cfl = ctx->adaptive_cfl;
    a.own_k0 = ctx->k_first; a.own_k1 = ctx->k_last;
    for (int side = 0; side < 2; ++side) {
        clt_ctx *pc = ctx->link[side].peer;
        double *pout = nullptr;
        if (pc && mode != RHS_MODE_K) pout = out == ctx->Ua ? pc->Ua : (out == ctx->Ub ? pc->Ub : (out == ctx->Un ? pc->Un : nullptr));
        a.peer[side].out = pout;
        a.peer[side].plane = pc ? pc->L.plane : 0;
        a.peer[side].field = pc ? pc->L.field : 0;
        a.peer[side].k0 = ctx->link[side].k0; a.peer[side].k1 = ctx->link[side].k1; a.peer[side].dk = ctx->link[side].dk;
    }
    const bool tma = ctx->variant == 0;
    const bool linked = ctx->link[0].peer || ctx->link[1].peer;
    const bool slab = linked || ctx->k_first != 2 || ctx->k_last != ctx->L.nZ - 3;
    if (linked && !tma) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "linked slabs (clt_link_rows) need the default kernel variant");
        return CLT_EINVAL;
    }
    if ((ctx->hall || ctx->spectral) && !tma) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err),
                 "the Hall term and the pseudo-spectral phi scheme need the default kernel variant");
        return CLT_EINVAL;
    }
    if (ctx->spectral) {
        int r = run_phi_pass(ctx, 1, in);
        if (r) return r;
    }
    alignas(64) CUtensorMap tmU, tmJ, tmV;
    const int nJ = ctx->hall ? 6 : 3;
    // static reference state: rho, p and B land in the raw buffer, v in a ring of its own (three boxes over the stage state)
    const int nU = (ctx->has_v0 || ctx->spectral) ? 8 : 2;      // must match rhs_velocity_ring() of the kernels
    if (tma && (!make_map(ctx, in, 8, rhs_tile_z(), &tmU, nU) || !make_map(ctx, in, 8, rhs_tile_z(), &tmV, 3)
                || !make_map(ctx, ctx->J1, nJ, rhs_tile_z(), &tmJ, nJ))) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "cuTensorMapEncodeTiled failed");
        return CLT_ECUDA;
    }
    const long pe = prof_begin(ctx, mode);
    if (tma)
        CK(launch_rhs_tma(a, &tmU, &tmJ, &tmV, mode, ctx->has_v0, ctx->hall, ctx->spectral, slab, ctx->stream));
    else
        CK(launch_rhs(a, mode, ctx->has_v0, ctx->stream));
    prof_end(ctx, pe);
    ctx->launches++;
    return CLT_OK;
}

// a6: one classical RK4 step in the reduced-traffic accumulator form (clt_kernels.cu):
//   s1: Ua = Un + dt/2 K1                          s2: Ub = Un + dt/2 K2, acc = Un + (Ua - Un)/3 + dt/3 K2
//   s3: Ua = Un + dt K3                            s4: Un = acc + (Ua - Un)/3 + dt/6 K4
int enqueue_stage(clt_ctx *ctx, int stage)
{
    int r;
    if ((r = resolve_v0(ctx))) return r;
    switch (stage) {
    case 1:
        if ((r = run_curl(ctx, ctx->Un))) return r;
        return run_rhs(ctx, RHS_MODE_S1, ctx->Un, ctx->Ua);
    case 2:
        if ((r = run_curl(ctx, ctx->Ua))) return r;
        return run_rhs(ctx, RHS_MODE_S2, ctx->Ua, ctx->Ub);
    case 3:
        if ((r = run_curl(ctx, ctx->Ub))) return r;
        return run_rhs(ctx, RHS_MODE_S3, ctx->Ub, ctx->Ua);
    case 4:
        if ((r = run_curl(ctx, ctx->Ua))) return r;
        return run_rhs(ctx, RHS_MODE_S4, ctx->Ua, ctx->Un);
    default:
        return CLT_EINVAL;
    }
}

int enqueue_step(clt_ctx *ctx)
{
    for (int stage = 1; stage <= 4; ++stage) {
        int r = enqueue_stage(ctx, stage);
        if (r) return r;
    }
    return CLT_OK;
}

// rows k0 .. k0+nrows-1 of one 8-field buffer  <->  dense [8][nphi][nrows][nR]
int copy_rows(clt_ctx *ctx, double *buf, int k0, int nrows, double *dense, bool to_dense)
{
    cudaMemcpy3DParms p;
    memset(&p, 0, sizeof(p));
    cudaPitchedPtr internal = make_cudaPitchedPtr(buf + (size_t)k0 * ctx->L.pR + LP, (size_t)ctx->L.pR * sizeof(double),
                                                  (size_t)ctx->L.nR, (size_t)ctx->L.nZ);
    cudaPitchedPtr user = make_cudaPitchedPtr(dense, (size_t)ctx->L.nR * sizeof(double), (size_t)ctx->L.nR, (size_t)nrows);
    p.srcPtr = to_dense ? internal : user;
    p.dstPtr = to_dense ? user : internal;
    p.extent = make_cudaExtent((size_t)ctx->L.nR * sizeof(double), (size_t)nrows, (size_t)8 * ctx->L.nphi);
    p.kind = cudaMemcpyDefault;
    CK(cudaMemcpy3DAsync(&p, ctx->stream));
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, dense);
    if (e != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
    if (at.type != cudaMemoryTypeDevice) CK(cudaStreamSynchronize(ctx->stream));
    return CLT_OK;
}

}  // namespace

extern "C" {

size_t clt_workspace_bytes(const clt_grid *grid)
{
    if (!grid_ok(grid)) return 0;
    return carve(grid).total;
}

int clt_create(const clt_grid *grid, const clt_params *params, void *d_workspace, size_t bytes, void *cuda_stream,
               clt_ctx **out)
{
    if (!out) return CLT_EINVAL;
    *out = nullptr;
    if (!grid_ok(grid) || !params || !d_workspace) return CLT_EINVAL;
    if (!isfinite(params->gamma) || !isfinite(params->eta) || !isfinite(params->nu) || !isfinite(params->D)
        || !isfinite(params->kappa) || !isfinite(params->dt) || !isfinite(params->cfl))
        return CLT_EINVAL;
    if (params->eta < 0 || params->nu < 0 || params->D < 0 || params->kappa < 0 || params->dt < 0 || params->flags != 0)
        return CLT_EINVAL;
    if (!isfinite(params->d_i) || params->d_i < 0) return CLT_EINVAL;
    const Carve c = carve(grid);
    if (bytes < c.total || ((uintptr_t)d_workspace % 256) != 0) return CLT_ENOMEM;
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, d_workspace);
    if (e != cudaSuccess) { cudaGetLastError(); return CLT_ECUDA; }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return CLT_ENOMEM;

    clt_ctx *ctx = new (std::nothrow) clt_ctx();
    if (!ctx) return CLT_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->ev = new std::vector<cudaEvent_t>();
    ctx->ev_kind = new std::vector<int>();
    ctx->ev_start = new std::vector<long>();
    ctx->grid = *grid;
    ctx->par = *params;
    ctx->L = make_layout(grid);
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->device = at.device;
    DeviceGuard device_guard(ctx);
    if (cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess) {
        cudaGetLastError();
        ctx->sm_count = 148;
    }
    ctx->dt = params->dt;
    ctx->k_first = 2; ctx->k_last = grid->nZ - 3; ctx->kd_first = 4; ctx->kd_last = grid->nZ - 5;
    ctx->next_stage = 1;
    const double Lphi = grid->phi_extent == 0.0 ? 2.0 * M_PI : grid->phi_extent;
    const double dR = (grid->Rmax - grid->Rmin) / (double)(grid->nR - 1);
    const double dZ = (grid->Zmax - grid->Zmin) / (double)(grid->nZ - 1);
    const double dphi = Lphi / (double)grid->nphi;
    Phys &ph = ctx->ph;
    ph.d_i = params->d_i;
    ctx->hall = params->d_i != 0.0;
    ph.gamma = params->gamma; ph.eta = params->eta; ph.nu = params->nu; ph.D = params->D; ph.kappa = params->kappa;
    ph.cR1 = 1.0 / (12.0 * dR); ph.cZ1 = 1.0 / (12.0 * dZ); ph.cP1 = 1.0 / (12.0 * dphi);
    ph.cR2 = 1.0 / (12.0 * dR * dR); ph.cZ2 = 1.0 / (12.0 * dZ * dZ); ph.cP2 = 1.0 / (12.0 * dphi * dphi);
    ph.dR = dR; ph.dZ = dZ; ph.dphi = dphi; ph.Lphi = Lphi;

    char *p = (char *)d_workspace;
    auto take = [&](size_t b) { double *r = (double *)p; p += b; return r; };
    ctx->Un = take(8 * c.field_b); ctx->acc = take(8 * c.field_b);
    ctx->Ua = take(8 * c.field_b); ctx->Ub = take(8 * c.field_b);
    ctx->J1 = take(3 * c.field_b);
    ctx->G = take(3 * c.field_b);      // right behind J1: one tensor map covers both (Hall variant)
    ctx->tab = take(T_COUNT * c.table_b);
    ctx->Rtab = take(c.rtab_b); ctx->invRtab = take(c.rtab_b);
    ctx->cs = take(c.cs_b);
    ctx->partial = take(c.partial_b);
    ctx->result = take(c.result_b);
    ctx->nblocks_diag = c.nblocks;
    // carve() aligns every field to 256 B but Layout::field is the unaligned stride: they must agree
    if ((size_t)ctx->L.field * sizeof(double) != c.field_b || (size_t)ctx->L.plane * sizeof(double) != c.table_b) {
        free_profile(ctx);
        delete ctx;
        return CLT_EINVAL;
    }

    int rc = CLT_OK;
    do {
        if ((e = cudaMemsetAsync(d_workspace, 0, c.total, ctx->stream)) != cudaSuccess) break;
        // R_i = Rmin + i*dR in plain double arithmetic on the host (hazard H1); pad columns repeat the edge
        std::vector<double> R(ctx->L.pR), iR(ctx->L.pR), cs(2 * (size_t)grid->nphi);
        for (int col = 0; col < ctx->L.pR; ++col) {
            int i = col - LP;
            i = i < 0 ? 0 : (i > grid->nR - 1 ? grid->nR - 1 : i);
            volatile double prod = (double)i * dR;      // no FMA contraction
            R[col] = grid->Rmin + prod;
            iR[col] = 1.0 / R[col];
        }
        for (int j = 0; j < grid->nphi; ++j) {
            const double ang = 2.0 * M_PI * (double)j / (double)grid->nphi;
            cs[j] = cos(ang);
            cs[grid->nphi + j] = sin(ang);
        }
        if ((e = cudaMemcpyAsync(ctx->Rtab, R.data(), R.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream))) break;
        if ((e = cudaMemcpyAsync(ctx->invRtab, iR.data(), iR.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream))) break;
        if ((e = cudaMemcpyAsync(ctx->cs, cs.data(), cs.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream))) break;
        if ((e = cudaStreamSynchronize(ctx->stream))) break;     // the host vectors go out of scope
        if ((e = configure_kernels())) break;                    // shared-memory opt-in of this context's device
        if ((e = diag_static_scratch(&ctx->static_partial, &ctx->static_max_blocks))) break;   // symbol address on this device
        if ((e = cudaHostAlloc((void **)&ctx->v0_flag_host, sizeof(int), cudaHostAllocDefault))) break;
        if ((e = cudaEventCreateWithFlags(&ctx->v0_event, cudaEventDisableTiming))) break;
        if ((e = launch_tables(ctx->L, ctx->ph, ctx->tab, ctx->Rtab + LP, ctx->invRtab + LP, ctx->stream))) break;
        ctx->launches++;
        if (ctx->dt > 0.0) {
            const double dt = ctx->dt, c4[4] = { dt, 0.5 * dt, dt / 3.0, dt / 6.0 };
            if ((e = cudaMemcpyAsync(ctx->result + 24, c4, sizeof(c4), cudaMemcpyHostToDevice, ctx->stream))) break;
        }
    } while (0);
    if (e != cudaSuccess) {
        free_profile(ctx);
        delete ctx;
        cudaGetLastError();
        return CLT_ECUDA;
    }
    *out = ctx;
    return rc;
}

int clt_destroy(clt_ctx *ctx)
{
    DeviceGuard device_guard(ctx);
    if (!ctx) return CLT_OK;
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    destroy_graph(ctx);
    free_profile(ctx);
    delete ctx;
    if (e != cudaSuccess) { cudaGetLastError(); return CLT_ECUDA; }
    return CLT_OK;
}

int clt_set_equilibrium(clt_ctx *ctx, const double *U0)
{
    DeviceGuard device_guard(ctx);
    if (!ctx) return CLT_EINVAL;
    ctx->has_state = false;
    const size_t rows = (size_t)8 * ctx->L.nZ;
    ctx->has_v0 = false;
    ctx->v0_pending = false;
    if (U0) {
        int r = copy_in(ctx, ctx->tab, U0, rows);          // tables 0..7 are U0 itself
        if (r) return r;
        // does the reference state move?  (selects the v0 = 0 specialisation of the kernels)  Decided on the device; the
        // flag is read back when the first kernel that needs it is launched (resolve_v0), so this call stays asynchronous
        int *flag = (int *)(ctx->result + 28);
        CK(launch_any_nonzero(ctx->tab + T_V0R * ctx->L.plane, 3 * ctx->L.plane, flag, ctx->stream));
        ctx->launches++;
        CK(cudaMemcpyAsync(ctx->v0_flag_host, flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaEventRecord(ctx->v0_event, ctx->stream));
        ctx->v0_pending = true;
        cudaPointerAttributes at;
        cudaError_t e = cudaPointerGetAttributes(&at, U0);
        if (e != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
        if (at.type != cudaMemoryTypeDevice) CK(cudaStreamSynchronize(ctx->stream));   // the caller may reuse host memory
    } else {
        CK(cudaMemsetAsync(ctx->tab, 0, (size_t)8 * ctx->L.plane * sizeof(double), ctx->stream));
    }
    CK(launch_tables(ctx->L, ctx->ph, ctx->tab, ctx->Rtab + LP, ctx->invRtab + LP, ctx->stream));
    ctx->launches++;
    return CLT_OK;
}

int clt_set_state(clt_ctx *ctx, const double *U)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !U) return CLT_EINVAL;
    ctx->adaptive = false;           // a new state ends an open clt_cfl_* sequence
    int r = copy_in(ctx, ctx->Un, U, (size_t)8 * ctx->L.nphi * ctx->L.nZ);
    if (r) return r;
    // a1: freeze the two boundary layers per R/Z side in every RK buffer
    CK(launch_copy_boundary(ctx->L, 8, ctx->Un, ctx->acc, ctx->Ua, ctx->Ub, ctx->sm_count, ctx->stream));
    ctx->launches++;
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, U);
    if (e != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
    if (at.type != cudaMemoryTypeDevice) CK(cudaStreamSynchronize(ctx->stream));   // the caller may reuse host memory
    ctx->has_state = true;
    ctx->next_stage = 1;
    ctx->step = 0;
    ctx->time = 0.0;
    return CLT_OK;
}

int clt_get_state(clt_ctx *ctx, double *U)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !U) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    return copy_out(ctx, U, ctx->Un, (size_t)8 * ctx->L.nphi * ctx->L.nZ);
}

int clt_rhs(clt_ctx *ctx, double *dUdt)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !dUdt) return CLT_EINVAL;
    if (!ctx->has_state || ctx->next_stage != 1) return CLT_ESTATE;      // U_b is the scratch buffer: not inside a step
    int r;
    if ((r = resolve_v0(ctx))) return r;
    if ((r = run_curl(ctx, ctx->Un))) return r;
    CK(launch_zero_boundary(ctx->L, 8, ctx->Ub, ctx->sm_count, ctx->stream));     // K = 0 on the boundary layers
    ctx->launches++;
    if ((r = run_rhs(ctx, RHS_MODE_K, ctx->Un, ctx->Ub))) return r;
    if ((r = copy_out(ctx, dUdt, ctx->Ub, (size_t)8 * ctx->L.nphi * ctx->L.nZ))) return r;
    CK(launch_copy_boundary(ctx->L, 8, ctx->Un, ctx->Ub, nullptr, nullptr, ctx->sm_count, ctx->stream));   // restore the scratch buffer
    ctx->launches++;
    return CLT_OK;
}

int clt_curl_J1(clt_ctx *ctx, double *J1)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !J1) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    int r;
    if ((r = resolve_v0(ctx))) return r;
    if ((r = run_curl(ctx, ctx->Un))) return r;
    return copy_out(ctx, J1, ctx->J1, (size_t)3 * ctx->L.nphi * ctx->L.nZ);
}

int clt_hall_G(clt_ctx *ctx, double *G)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !G) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    if (!ctx->hall) return CLT_EINVAL;
    int r;
    if ((r = resolve_v0(ctx))) return r;
    if ((r = run_curl(ctx, ctx->Un))) return r;
    return copy_out(ctx, G, ctx->G, (size_t)3 * ctx->L.nphi * ctx->L.nZ);
}

// { dt, dt/2, dt/3, dt/6 } -> the fixed-dt coefficient table in device memory (stream-ordered: steps already enqueued
// keep the dt they were enqueued with; a captured graph of the step stays valid)
static int upload_dt(clt_ctx *ctx)
{
    const double dt = ctx->dt;
    const double c[4] = { dt, 0.5 * dt, dt / 3.0, dt / 6.0 };
    CK(cudaMemcpyAsync(ctx->result + 24, c, sizeof(c), cudaMemcpyHostToDevice, ctx->stream));   // pageable source: staged before the call returns
    return CLT_OK;
}

int clt_set_dt(clt_ctx *ctx, double dt)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !(dt > 0.0) || !isfinite(dt)) return CLT_EINVAL;
    ctx->dt = dt;
    return upload_dt(ctx);
}

int clt_step(clt_ctx *ctx, int n)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || n < 0) return CLT_EINVAL;
    if (!ctx->has_state || ctx->next_stage != 1 || ctx->adaptive) return CLT_ESTATE;     // not between clt_cfl_open and clt_cfl_close
    if (!(ctx->dt > 0.0)) return CLT_EINVAL;
    // CUDA graph of the 8-launch step: 1 = always, 2 = never, 0 (default) = unless per-kernel profiling is on
    if (ctx->use_graph == 1 || (ctx->use_graph == 0 && !ctx->profiling)) {
        int rv = resolve_v0(ctx);
        if (rv) return rv;
        // dt is not part of the graph: the kernels read the stage coefficients from device memory (clt_set_dt)
        const bool stale = !ctx->graph_exec || ctx->graph_chunks != effective_chunks(ctx) || ctx->graph_v0 != ctx->has_v0;
        if (stale) {
            destroy_graph(ctx);
            cudaGraph_t g = nullptr;
            // capture on a private stream (the legacy default stream cannot be captured); the instantiated
            // graph is launched on the context's stream
            cudaStream_t cap = nullptr, user = ctx->stream;
            CK(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
            cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
            if (e != cudaSuccess) { cudaStreamDestroy(cap); return cuda_fail(ctx, e, "cudaStreamBeginCapture"); }
            const int64_t before = ctx->launches;
            ctx->stream = cap;
            int r = enqueue_step(ctx);
            ctx->stream = user;
            ctx->launches = before;
            e = cudaStreamEndCapture(cap, &g);
            cudaStreamDestroy(cap);
            if (r) { if (g) cudaGraphDestroy(g); return r; }
            if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamEndCapture");
            e = cudaGraphInstantiate(&ctx->graph_exec, g, 0);
            cudaGraphDestroy(g);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaGraphInstantiate");
            ctx->graph_chunks = effective_chunks(ctx); ctx->graph_v0 = ctx->has_v0;
        }
        for (int s = 0; s < n; ++s) {
            CK(cudaGraphLaunch(ctx->graph_exec, ctx->stream));
            ctx->launches += ctx->spectral ? 8 + 4 * (phi_launches(ctx, 0) + phi_launches(ctx, 1)) : 8;
        }
    } else {
        for (int s = 0; s < n; ++s) {
            int r = enqueue_step(ctx);
            if (r) return r;
        }
    }
    ctx->step += n;
    ctx->time += (double)n * ctx->dt;
    return CLT_OK;
}

// a7 + SETDT: the reduction kernels over the current state -> ctx->result[0..5] (device)
static int enqueue_diag(clt_ctx *ctx, double cfl)
{
    DiagArgs a;
    a.L = ctx->L; a.ph = ctx->ph;
    a.U = ctx->Un; a.tab = ctx->tab;
    a.R = ctx->Rtab + LP; a.invR = ctx->invRtab + LP;
    a.cs = ctx->cs; a.partial = ctx->partial; a.cfl = cfl; a.ihZ = 1.0 / ctx->ph.dZ;
    a.spec_c1 = ctx->spectral ? ctx->spec_ctab : nullptr;
    a.k_first = ctx->k_first; a.k_last = ctx->k_last; a.kd_first = ctx->kd_first; a.kd_last = ctx->kd_last;
    alignas(64) CUtensorMap tmU;
    const bool tma = ctx->variant == 0 && !ctx->spectral && make_map(ctx, ctx->Un, 8, diag_tma_tile_z(), &tmU, 8);
    CK(launch_diag(a, ctx->nblocks_diag, ctx->result, ctx->stream, tma ? &tmU : nullptr));
    ctx->launches += 2;
    return CLT_OK;
}

static int run_diag(clt_ctx *ctx, double cfl, double out6[6])
{
    int r = enqueue_diag(ctx, cfl);
    if (r) return r;
    CK(cudaMemcpyAsync(out6, ctx->result, 6 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return CLT_OK;
}

int clt_diagnostics(clt_ctx *ctx, clt_diag *out)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !out) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    double r6[6];
    int r = run_diag(ctx, ctx->par.cfl > 0 ? ctx->par.cfl : 0.5, r6);
    if (r) return r;
    out->kinetic = r6[0]; out->magnetic = r6[1]; out->magnetic_pert = r6[2]; out->magnetic_n1 = r6[3];
    out->max_divB = r6[4];
    out->step = ctx->step;
    out->time = ctx->time;
    for (int q = 0; q < 5; ++q)
        if (!isfinite(r6[q])) return CLT_ENONFINITE;
    return CLT_OK;
}

// The diagnostics reduction with NO memory but the library's own: block partials in the static device array
// (clt_kernels.cu), results to the caller's device pointer, nothing allocated, nothing copied to the host, no synchronisation.
int clt_diagnostics_static(clt_ctx *ctx, double cfl, double *d_out6)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !d_out6) return CLT_EINVAL;
    if (!(cfl > 0.0)) cfl = ctx->par.cfl > 0 ? ctx->par.cfl : 0.5;
    if (!isfinite(cfl)) return CLT_EINVAL;
    // the column kernel (pseudo-spectral scheme) has the most CTAs: one per 32 R nodes and Z row
    const int need = diag_blocks(ctx->L);
    if (need > ctx->static_max_blocks || !ctx->static_partial) {
        snprintf(ctx->cuda_err, sizeof(ctx->cuda_err),
                 "clt_diagnostics_static: this grid needs %d block partials, the static scratch holds %d (use clt_diagnostics)",
                 need, ctx->static_max_blocks);
        return CLT_ENOMEM;
    }
    if (!ctx->has_state) return CLT_ESTATE;
    cudaPointerAttributes at;
    cudaError_t pe = cudaPointerGetAttributes(&at, d_out6);
    if (pe != cudaSuccess) { cudaGetLastError(); return CLT_EINVAL; }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return CLT_EINVAL;
    DiagArgs a;
    a.L = ctx->L; a.ph = ctx->ph;
    a.U = ctx->Un; a.tab = ctx->tab;
    a.R = ctx->Rtab + LP; a.invR = ctx->invRtab + LP;
    a.cs = ctx->cs; a.partial = ctx->static_partial; a.cfl = cfl; a.ihZ = 1.0 / ctx->ph.dZ;
    a.spec_c1 = ctx->spectral ? ctx->spec_ctab : nullptr;
    a.k_first = ctx->k_first; a.k_last = ctx->k_last; a.kd_first = ctx->kd_first; a.kd_last = ctx->kd_last;
    alignas(64) CUtensorMap tmU;
    const bool tma = ctx->variant == 0 && !ctx->spectral && make_map(ctx, ctx->Un, 8, diag_tma_tile_z(), &tmU, 8);
    CK(launch_diag(a, need, d_out6, ctx->stream, tma ? &tmU : nullptr));
    ctx->launches += 2;
    return CLT_OK;
}

int clt_suggest_dt(clt_ctx *ctx, double cfl, double *dt_out)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !dt_out) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    if (!(cfl > 0.0)) cfl = ctx->par.cfl;
    if (!(cfl > 0.0) || !isfinite(cfl)) return CLT_EINVAL;
    double r6[6];
    int r = run_diag(ctx, cfl, r6);
    if (r) return r;
    *dt_out = r6[5];
    if (!(r6[5] > 0.0)) return CLT_ENONFINITE;      // a non-finite signal speed somewhere in the state
    return CLT_OK;
}

size_t clt_spectral_workspace_bytes(const clt_grid *grid)
{
    if (!grid_ok(grid) || grid->nphi > SPEC_MAX_NPHI) return 0;
    return (size_t)SPEC_COUNT * carve(grid).field_b + align_up(2 * SPEC_MAX_NPHI * sizeof(double));
}

int clt_set_phi_scheme(clt_ctx *ctx, int scheme, void *d_scratch, size_t bytes)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || scheme < 0 || scheme > 1) return CLT_EINVAL;
    CK(cudaStreamSynchronize(ctx->stream));
    destroy_graph(ctx);
    if (scheme == 0) { ctx->spectral = false; ctx->spec = nullptr; ctx->spec_ctab = nullptr; return CLT_OK; }
    const size_t need = clt_spectral_workspace_bytes(&ctx->grid);
    if (need == 0) return CLT_EINVAL;                      // nphi > SPEC_MAX_NPHI
    if (!d_scratch || bytes < need || ((uintptr_t)d_scratch % 256) != 0) return CLT_ENOMEM;
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, d_scratch);
    if (e != cudaSuccess) { cudaGetLastError(); return CLT_ECUDA; }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return CLT_ENOMEM;
    // closed-form weights of the Fourier differentiation matrices on N equispaced nodes of a period L
    // (kappa = 2 pi / L):  N even:  c1[m] = kappa/2 (-1)^(m+1) cot(pi m/N), c1[N/2] = 0;
    //                               c2[0] = -kappa^2 (N^2+2)/12, c2[m] = -kappa^2/2 (-1)^m / sin^2(pi m/N)
    //                      N odd:   c1[m] = kappa/2 (-1)^(m+1) / sin(pi m/N);
    //                               c2[0] = -kappa^2 (N^2-1)/12, c2[m] = -kappa^2/2 (-1)^m cos(pi m/N) / sin^2(pi m/N)
    const int N = ctx->grid.nphi;
    const long double PI = 3.141592653589793238462643383279502884L;
    const long double kap = 2.0L * PI / (long double)ctx->ph.Lphi;
    std::vector<double> tabv(2 * SPEC_MAX_NPHI, 0.0);
    for (int m = 0; m < N; ++m) {
        long double c1, c2;
        const long double th = PI * (long double)m / (long double)N, sg = (m % 2) ? -1.0L : 1.0L;
        if (m == 0) {
            c1 = 0.0L;
            c2 = -kap * kap * ((N % 2 == 0) ? ((long double)N * N + 2.0L) : ((long double)N * N - 1.0L)) / 12.0L;
        } else if (N % 2 == 0) {
            c1 = (2 * m == N) ? 0.0L : -0.5L * kap * sg * cosl(th) / sinl(th);
            c2 = -0.5L * kap * kap * sg / (sinl(th) * sinl(th));
        } else {
            c1 = -0.5L * kap * sg / sinl(th);
            c2 = -0.5L * kap * kap * sg * cosl(th) / (sinl(th) * sinl(th));
        }
        tabv[m] = (double)c1;
        tabv[SPEC_MAX_NPHI + m] = (double)c2;
    }
    const size_t fields_b = (size_t)SPEC_COUNT * carve(&ctx->grid).field_b;
    ctx->spec = (double *)d_scratch;
    ctx->spec_ctab = (double *)((char *)d_scratch + fields_b);
    CK(cudaMemsetAsync(d_scratch, 0, need, ctx->stream));
    CK(cudaMemcpyAsync(ctx->spec_ctab, tabv.data(), tabv.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->spectral = true;
    return CLT_OK;
}

int clt_step_stage(clt_ctx *ctx, int stage)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || stage < 1 || stage > 4) return CLT_EINVAL;
    if (!ctx->has_state || stage != ctx->next_stage) return CLT_ESTATE;
    if (!(ctx->dt > 0.0)) return CLT_EINVAL;
    int r = enqueue_stage(ctx, stage);
    if (r) return r;
    ctx->next_stage = stage == 4 ? 1 : stage + 1;
    if (stage == 4) { ctx->step += 1; if (!ctx->adaptive) ctx->time += ctx->dt; }     // adaptive: clt_cfl_close adds the time
    return CLT_OK;
}

// ---- adaptive stepping of a GROUP of contexts that share one time step (slabs of one grid; NEXT-1 + NEXT-4) ----------
int clt_cfl_open(clt_ctx *ctx, double cfl)
{
    DeviceGuard device_guard(ctx);
    if (!ctx) return CLT_EINVAL;
    if (!ctx->has_state || ctx->next_stage != 1 || ctx->adaptive) return CLT_ESTATE;
    if (!(cfl > 0.0)) cfl = ctx->par.cfl;
    if (!(cfl > 0.0) || !isfinite(cfl)) return CLT_EINVAL;
    int r;
    if ((r = resolve_v0(ctx))) return r;
    if ((r = enqueue_diag(ctx, cfl))) return r;       // result[5] = SETDT of the owned rows
    ctx->adaptive = true;
    ctx->adaptive_cfl = cfl;
    return CLT_OK;
}

int clt_cfl_commit(clt_ctx *const *ctxs, int n, int init)
{
    if (!ctxs || n < 1 || n > DT_GROUP_MAX) return CLT_EINVAL;
    DtGroup g;
    g.n = n;
    for (int c = 0; c < n; ++c) {
        if (!ctxs[c] || !ctxs[c]->adaptive || ctxs[c]->next_stage != 1) return ctxs[c] ? CLT_ESTATE : CLT_EINVAL;
        if (ctxs[c]->device != ctxs[0]->device) return CLT_EINVAL;       // one kernel reads every clock: one device
        g.clock[c] = ctxs[c]->result + 8;
        g.dtmin_bits[c] = (unsigned long long *)(ctxs[c]->result + 16);
        g.diag6[c] = ctxs[c]->result;
    }
    clt_ctx *ctx = ctxs[0];
    DeviceGuard device_guard(ctx);
    // the kernel runs on the first context's stream, after everything the others have enqueued; they wait for it
    cudaEvent_t ev = nullptr;
    bool others = false;
    for (int c = 1; c < n; ++c) others = others || ctxs[c]->stream != ctx->stream;
    if (others) {
        CK(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        for (int c = 1; c < n; ++c)
            if (ctxs[c]->stream != ctx->stream) {
                cudaError_t e = cudaEventRecord(ev, ctxs[c]->stream);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->stream, ev, 0);
                if (e != cudaSuccess) { cudaEventDestroy(ev); return cuda_fail(ctx, e, "clt_cfl_commit: stream order"); }
            }
    }
    cudaError_t e = launch_dt_commit_group(g, init, ctx->stream);
    if (e == cudaSuccess && others) {
        e = cudaEventRecord(ev, ctx->stream);
        for (int c = 1; c < n && e == cudaSuccess; ++c)
            if (ctxs[c]->stream != ctx->stream) e = cudaStreamWaitEvent(ctxs[c]->stream, ev, 0);
    }
    if (ev) cudaEventDestroy(ev);
    for (int c = 0; c < n; ++c) ctxs[c]->prof_chain = false;
    ctx->launches++;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "dt_commit_group_kernel");
    return CLT_OK;
}

int clt_cfl_close(clt_ctx *ctx, double *dt_next, double *time_advanced)
{
    DeviceGuard device_guard(ctx);
    if (!ctx) return CLT_EINVAL;
    if (!ctx->adaptive || ctx->next_stage != 1) return CLT_ESTATE;
    double h[6] = { 0, 0, 0, 0, 0, 0 };
    ctx->adaptive = false;
    CK(cudaMemcpyAsync(h, ctx->result + 8, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->time += h[4];
    if (dt_next) *dt_next = h[0];
    if (time_advanced) *time_advanced = h[4];
    if (h[5] != 0.0) return CLT_ENONFINITE;
    return CLT_OK;
}

static double *stage_buffer(clt_ctx *ctx, int buffer)
{
    return buffer == 0 ? ctx->Un : (buffer == 1 ? ctx->Ua : (buffer == 2 ? ctx->Ub : nullptr));
}

int clt_get_rows(clt_ctx *ctx, int buffer, int k0, int nrows, double *dst)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !dst || nrows < 1 || k0 < 0 || k0 + nrows > ctx->L.nZ || !stage_buffer(ctx, buffer)) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    return copy_rows(ctx, stage_buffer(ctx, buffer), k0, nrows, dst, true);
}

int clt_set_rows(clt_ctx *ctx, int buffer, int k0, int nrows, const double *src)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !src || nrows < 1 || k0 < 0 || k0 + nrows > ctx->L.nZ || !stage_buffer(ctx, buffer)) return CLT_EINVAL;
    if (!ctx->has_state) return CLT_ESTATE;
    return copy_rows(ctx, stage_buffer(ctx, buffer), k0, nrows, const_cast<double *>(src), false);
}

int clt_set_z_spacing(clt_ctx *ctx, double dZ)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !(dZ > 0.0) || !isfinite(dZ)) return CLT_EINVAL;
    Phys &ph = ctx->ph;
    ph.dZ = dZ;
    ph.cZ1 = 1.0 / (12.0 * dZ);
    ph.cZ2 = 1.0 / (12.0 * dZ * dZ);
    // everything derived from the old spacing goes: tables of the reference state, the state, a captured step
    ctx->has_state = false;
    ctx->has_v0 = false;
    ctx->v0_pending = false;
    destroy_graph(ctx);
    CK(cudaMemsetAsync(ctx->tab, 0, (size_t)T_COUNT * ctx->L.plane * sizeof(double), ctx->stream));
    CK(launch_tables(ctx->L, ctx->ph, ctx->tab, ctx->Rtab + LP, ctx->invRtab + LP, ctx->stream));
    ctx->launches++;
    return CLT_OK;
}

int clt_push_rows(clt_ctx *src, int buffer, int k0_src, int nrows, clt_ctx *dst, int k0_dst)
{
    if (!src || !dst || src == dst || nrows < 1 || !stage_buffer(src, buffer)) return CLT_EINVAL;
    if (k0_src < 0 || k0_src + nrows > src->L.nZ || k0_dst < 0 || k0_dst + nrows > dst->L.nZ) return CLT_EINVAL;
    if (src->L.nR != dst->L.nR || src->L.nphi != dst->L.nphi) return CLT_EINVAL;
    if (!src->has_state || !dst->has_state) return CLT_ESTATE;
    clt_ctx *ctx = dst;                                          // CK reports into the destination context
    DeviceGuard device_guard(dst);
    if (src->device != dst->device) {
        int can = 0;
        CK(cudaDeviceCanAccessPeer(&can, dst->device, src->device));
        if (!can) { snprintf(dst->cuda_err, sizeof(dst->cuda_err), "clt_push_rows: no peer access between devices %d and %d", dst->device, src->device); return CLT_ECUDA; }
        cudaError_t pe = cudaDeviceEnablePeerAccess(src->device, 0);
        if (pe != cudaSuccess && pe != cudaErrorPeerAccessAlreadyEnabled) return cuda_fail(dst, pe, "cudaDeviceEnablePeerAccess");
        cudaGetLastError();
    }
    const bool two_streams = src->stream != dst->stream || src->device != dst->device;
    cudaEvent_t ready = nullptr, done = nullptr;
    if (two_streams) {
        // order: src's stage kernel -> copy on dst's stream -> whatever src enqueues next (it will overwrite these rows)
        CK(cudaEventCreateWithFlags(&done, cudaEventDisableTiming));
        {
            DeviceGuard src_guard(src);
            cudaError_t e = cudaEventCreateWithFlags(&ready, cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventRecord(ready, src->stream);
            if (e != cudaSuccess) { cudaEventDestroy(done); if (ready) cudaEventDestroy(ready); return cuda_fail(dst, e, "clt_push_rows: event on the source stream"); }
        }
        CK(cudaStreamWaitEvent(dst->stream, ready, 0));
    }
    cudaError_t e = launch_push_rows(src->L, stage_buffer(src, buffer), k0_src, dst->L, stage_buffer(dst, buffer), k0_dst, nrows,
                                     dst->sm_count, dst->stream);
    dst->launches++;
    dst->prof_chain = false;
    if (two_streams) {
        if (e == cudaSuccess) e = cudaEventRecord(done, dst->stream);
        if (e == cudaSuccess) {
            DeviceGuard src_guard(src);
            e = cudaStreamWaitEvent(src->stream, done, 0);
        }
        cudaEventDestroy(ready);      // destruction is deferred until the events have completed
        cudaEventDestroy(done);
    }
    if (e != cudaSuccess) return cuda_fail(dst, e, "clt_push_rows");
    return CLT_OK;
}

int clt_set_owned_rows(clt_ctx *ctx, int k_first, int k_last, int deep_first, int deep_last)
{
    if (!ctx) return CLT_EINVAL;
    if (k_first < 2 || k_last > ctx->L.nZ - 3 || k_first > k_last) return CLT_EINVAL;
    if (deep_first < 2 || deep_last > ctx->L.nZ - 3) return CLT_EINVAL;      // an empty deep range is allowed
    ctx->k_first = k_first; ctx->k_last = k_last; ctx->kd_first = deep_first; ctx->kd_last = deep_last;
    destroy_graph(ctx);          // the row range is a kernel argument of the captured step
    return CLT_OK;
}

int clt_link_rows(clt_ctx *ctx, int side, clt_ctx *peer, int k0, int nrows, int k0_peer)
{
    if (!ctx || side < 0 || side > 1) return CLT_EINVAL;
    destroy_graph(ctx);
    if (!peer) { ctx->link[side].peer = nullptr; return CLT_OK; }
    if (peer == ctx || nrows < 1 || k0 < ctx->k_first || k0 + nrows - 1 > ctx->k_last) return CLT_EINVAL;   // owned rows only
    if (k0_peer < 0 || k0_peer + nrows > peer->L.nZ) return CLT_EINVAL;
    if (peer->L.nR != ctx->L.nR || peer->L.nphi != ctx->L.nphi) return CLT_EINVAL;
    if (peer->device != ctx->device) {
        DeviceGuard device_guard(ctx);
        int can = 0;
        CK(cudaDeviceCanAccessPeer(&can, ctx->device, peer->device));
        if (!can) { snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "clt_link_rows: no peer access between devices %d and %d", ctx->device, peer->device); return CLT_ECUDA; }
        cudaError_t pe = cudaDeviceEnablePeerAccess(peer->device, 0);
        if (pe != cudaSuccess && pe != cudaErrorPeerAccessAlreadyEnabled) return cuda_fail(ctx, pe, "cudaDeviceEnablePeerAccess");
        cudaGetLastError();
    }
    ctx->link[side].peer = peer;
    ctx->link[side].k0 = k0; ctx->link[side].k1 = k0 + nrows - 1; ctx->link[side].dk = k0_peer - k0;
    return CLT_OK;
}

int clt_sync_peers(clt_ctx *a, clt_ctx *b)
{
    if (!a || !b) return CLT_EINVAL;
    if (a->stream == b->stream && a->device == b->device) return CLT_OK;      // one stream: already ordered
    clt_ctx *ctx = a;
    cudaEvent_t ea = nullptr, eb = nullptr;
    cudaError_t e;
    {
        DeviceGuard ga(a);
        e = cudaEventCreateWithFlags(&ea, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventRecord(ea, a->stream);
    }
    if (e == cudaSuccess) {
        DeviceGuard gb(b);
        e = cudaEventCreateWithFlags(&eb, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventRecord(eb, b->stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(b->stream, ea, 0);
    }
    if (e == cudaSuccess) {
        DeviceGuard ga(a);
        e = cudaStreamWaitEvent(a->stream, eb, 0);
    }
    if (ea) cudaEventDestroy(ea);
    if (eb) cudaEventDestroy(eb);
    a->prof_chain = false; b->prof_chain = false;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "clt_sync_peers");
    return CLT_OK;
}

int clt_step_cfl(clt_ctx *ctx, int n, double cfl, double *dt_last, double *time_advanced)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || n < 0) return CLT_EINVAL;
    if (!ctx->has_state || ctx->next_stage != 1 || ctx->adaptive) return CLT_ESTATE;     // not between clt_cfl_open and clt_cfl_close
    if (!(cfl > 0.0)) cfl = ctx->par.cfl;
    if (!(cfl > 0.0) || !isfinite(cfl)) return CLT_EINVAL;
    double *clock = ctx->result + 8;
    unsigned long long *bits = (unsigned long long *)(ctx->result + 16);
    double h[6] = { 0, 0, 0, 0, 0, 0 };
    if (n > 0) {
        // dt of the first step: SETDT of the current state (the reduction kernel of clt_suggest_dt, no host round trip)
        int rd = enqueue_diag(ctx, cfl);
        if (rd) return rd;
        CK(launch_dt_commit(clock, bits, ctx->result, 1, ctx->stream));
        ctx->launches += 1;
        ctx->adaptive = true;
        ctx->adaptive_cfl = cfl;
        int r = CLT_OK;
        for (int s = 0; s < n && r == CLT_OK; ++s) {
            r = enqueue_step(ctx);                 // stage 4 collects the SETDT minimum of the new state
            if (r == CLT_OK) {
                cudaError_t e = launch_dt_commit(clock, bits, ctx->result, 0, ctx->stream);   // time += dt; dt = minimum
                ctx->prof_chain = false;
                if (e != cudaSuccess) r = cuda_fail(ctx, e, "dt_commit_kernel");
                ctx->launches++;
            }
        }
        ctx->adaptive = false;
        if (r) return r;
        CK(cudaMemcpyAsync(h, clock, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
    }
    ctx->step += n;
    ctx->time += h[4];
    if (dt_last) *dt_last = h[0];          // the SETDT value of the final state = the dt the next step would use
    if (time_advanced) *time_advanced = h[4];
    // a state whose signal speed is not finite (NaN / Inf anywhere in rho, p, B, or a NaN velocity) raised the clock's
    // mark and froze dt at 0: the call reports it instead of stepping on with a meaningless dt
    if (h[5] != 0.0) return CLT_ENONFINITE;
    return CLT_OK;
}

int clt_set_tuning(clt_ctx *ctx, int tile_z, int phi_chunks, int use_graph)
{
    if (!ctx) return CLT_EINVAL;
    if (tile_z != 0 && tile_z != rhs_tile_z()) return CLT_EINVAL;     // one tile shape is built (32 x 8); 0 = default
    if (phi_chunks < 0 || phi_chunks > 64 || use_graph < 0 || use_graph > 2) return CLT_EINVAL;
    ctx->phi_chunks = phi_chunks;
    ctx->use_graph = use_graph;
    return CLT_OK;
}

int clt_set_profiling(clt_ctx *ctx, int enable)
{
    DeviceGuard device_guard(ctx);
    if (!ctx) return CLT_EINVAL;
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->profiling = enable != 0;
    ctx->ev_used = 0;
    ctx->ev_dropped = 0;
    return CLT_OK;
}

int clt_get_profile(clt_ctx *ctx, clt_profile *out)
{
    DeviceGuard device_guard(ctx);
    if (!ctx || !out) return CLT_EINVAL;
    CK(cudaStreamSynchronize(ctx->stream));
    memset(out, 0, sizeof(*out));
    for (size_t n = 0; n < ctx->ev_used; ++n) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, (*ctx->ev)[(*ctx->ev_start)[n]], (*ctx->ev)[2 * n + 1]));
        const int kind = (*ctx->ev_kind)[n];
        if (kind == 5) { out->ms_curl += ms; out->n_curl++; }
        else if (kind == 6) { out->ms_phi += ms; out->n_phi++; }
        else { out->ms_rhs[kind] += ms; out->n_rhs[kind]++; }
    }
    out->dropped = ctx->ev_dropped;
    ctx->ev_used = 0;
    ctx->ev_dropped = 0;
    return CLT_OK;
}

int clt_set_kernel_variant(clt_ctx *ctx, int variant)
{
    if (!ctx || variant < 0 || variant > 1) return CLT_EINVAL;
    ctx->variant = variant;
    destroy_graph(ctx);
    return CLT_OK;
}

int64_t clt_launch_count(const clt_ctx *ctx) { return ctx ? ctx->launches : 0; }
void *clt_stream(const clt_ctx *ctx) { return ctx ? (void *)ctx->stream : nullptr; }

const char *clt_strerror(int code)
{
    switch (code) {
    case CLT_OK: return "ok";
    case CLT_EINVAL: return "invalid argument";
    case CLT_ENOMEM: return "workspace too small, misaligned or not device memory";
    case CLT_ESTATE: return "call out of order (set the state first)";
    case CLT_ECUDA: return "CUDA error";
    case CLT_ENONFINITE: return "non-finite diagnostic";
    default: return "unknown error";
    }
}
const char *clt_last_cuda_error(const clt_ctx *ctx) { return ctx ? ctx->cuda_err : ""; }
const char *clt_version(void) { return "clt-b200 0.1 (sm_100a, fp64)"; }

}  // extern "C"

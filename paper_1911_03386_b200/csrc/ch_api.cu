// ch_api.cu -- the C ABI of include/ch.h: argument checking, host precompute, workspace,
// kernel selection and launch.  No torch types, no exceptions across the boundary.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/ch.h"
#include "ch_factor.h"
#include "ch_kernels.cuh"
#include "ch_fused2d.cuh"
#include "ch_line2d.cuh"
#include "ch_rhs3d_stream.cuh"
#include "ch_cline2d.cuh"
#include "ch_local2d.cuh"
#include "ch_resident2d.cuh"

enum { KIND_RHS = 0, KIND_RHS_DIAG, KIND_FINISH, KIND_SWEEP_X, KIND_SWEEP_Y, KIND_SWEEP_Z,
       KIND_RHS_SWEEP_Y, KIND_RHS_SWEEP_Y_DIAG, KIND_SWEEP_X_UPDATE, KIND_SWEEP_XY, KIND_STEP_LOCAL, KIND_STEP_RESIDENT, KIND_COUNT };
static const char *const kKindNames[KIND_COUNT] = { "rhs", "rhs_diag", "finish", "sweep_x", "sweep_y", "sweep_z",
                                                    "rhs_sweep_y", "rhs_sweep_y_diag", "sweep_x_update", "sweep_xy", "step_local", "step_resident" };

struct ProfRec { int kind; cudaEvent_t e0, e1; };

struct ch_ctx {
    int M, N, D;
    double gamma, dt;
    size_t npts;            // N^D
    size_t total;           // M * N^D
    bool pow2;
    // factorisation
    ChFactor fac;
    bool chunked;           // chunked sweeps available for this N
    int LC;
    double *dW;             // device copy of fac.W
    double *dS2;            // device copy of fac.Mlane, fac.WG (two-level scan closure)
    double *dS2_16;         // device copy of fac16.Mlane, fac16.WG
    double *dS2c;           // cluster line SCAN kernels: fac16.Mlane then WG[8][4] of the cluster
    double *dW16;           // device copy of fac16.W (cluster line mode when c->LC is 32), else NULL
    double rscale;          // dt / c0^D: the 1/c0 of every sweep folded into the RHS
    // device arrays
    void *ws_base;          // cudaMalloc'ed or attached
    bool ws_owned;
    size_t ws_bytes;
    double *C, *w, *partials, *eout;
    int nparts;             // RHS tiles per member
    int rhs_tiles_x, rhs_tiles_y;
    // state
    bool has_state;
    long long n;            // steps since set_state
    double t0;
    double *series;
    int stride, capacity, cursor;
    long long last_sampled; // step index whose sample has been written (-1: none)
    cudaStream_t stream;
    // options
    int opt_sweep;          // 0 auto, 1 generic, 2 chunked
    // CUDA graph of CH_GRAPH_STEPS plain (non-sampling) steps for launch-bound (small) ensembles
    int opt_graph;          // 0 auto (graphs when the ensemble has <= 8 Mi points), 1 off, 2 always
    cudaGraphExec_t gexec;
    cudaStream_t cap_stream;
    long long gsig;         // option signature the graph was captured with
    long long glaunches;    // kernel nodes in the graph
    bool graph_broken;      // capture failed once: plain launches from then on
    int opt_scan;           // contiguous sweeps: 0 auto (shuffle-scan closure when K > 4), 1 off, 2 always
    int opt_linesync;       // line kernel: 0 auto (neighbour-warp sync when K <= 2), 1 CTA barriers
    int opt_fuse;           // 0 auto (fused 2D step when available), 1 off, 2 cluster kernel, 3 line kernel
    // fused 2D step (ch_fused2d.cuh)
    bool fused_ok;
    int f_CPB, f_CS, f_strips;   // chunks per CTA, CTAs per cluster, column strips per member
    // fused 2D step, line spread over a cluster of 512-row CTAs (ch_cline2d.cuh); needs K <= 2 at LC = 16
    bool cline_ok;
    int cl_CS, cl_strips, cl_resident;   // cluster size, column strips per member, clusters resident on the device
    ChFactor fac16;                      // factorisation tables at chunk length 16 (c->fac may use 32)
    // streaming 3D RHS (ch_rhs3d_stream.cuh)
    bool r3_ok;
    int r3_parts, r3_resident;   // partials per member, CTAs resident on the device
    int opt_rhs3;                // 0 auto (streaming kernel when available), 1 tile kernel
    bool xy_ok;                  // 3D, N in {64, 128}: x- and y-sweep of a z-plane in one pass (k_sweep_xy_plane)
    int dir3;                    // 3D: direction in which the next RHS launch walks the ensemble (alternates)
    int opt_sweep3;              // 0 auto (plane kernel when available), 1 separate x and y sweeps
    // fused 2D step, whole line in one CTA (ch_line2d.cuh)
    bool line_ok;
    int l_strips, l_resident;    // column strips per member, CTAs resident on the device
    // one-pass local 2D step for small gamma dt (ch_local2d.cuh)
    bool local_ok;
    int loc_H, loc_resident;     // decay reach (ch_factor_reach), CTAs resident on the device
    // member-resident stepping: one CTA holds a member in shared memory for a whole ch_step call (ch_resident2d.cuh)
    bool resident_ok;
    int res_clusters;            // clusters of that size resident on the device
    int sms;                     // multiprocessors of the device
    int opt_pdl;                 // 0: line kernel and x-sweep/update are launched as programmatic dependents, 1: plain launches
    int opt_resident;            // one-CTA kernel: 0 auto, 1 one line per thread, 2 two lines per thread
    int res_CS;                  // CTAs per member: 1 (N <= 96), else the cluster size (N = 128: 2, N = 256: 8)
    // ch_run_host: the kernels run on a member sub-range ("view"): M, total, C, w point at the view, these keep the whole
    int Mfull, view_m0;
    cudaStream_t rh_in, rh_comp, rh_out;     // its three internal streams (created on first use)
    long long launches;
    bool profiling;
    std::vector<ProfRec> prof;
    std::string err;
};

// which fused 2D step runs: 0 none (three-pass), 2 st.async cluster kernel, 3 line kernel, 4 cluster line kernel
// (mode 4 steps with the cluster line kernel and samples with the tile RHS kernel), 5 one-pass local step (small
// gamma dt only; samples with the line kernel's or the tile kernel's diagnostics-only launch)
static int fuse_mode(const ch_ctx *c)
{
    if (c->opt_fuse == 1 || c->opt_sweep == 1) return 0;
    if (c->opt_fuse == 5) return c->local_ok ? 5 : 0;
    if (c->opt_fuse == 6) return c->resident_ok ? 6 : 0;
    // auto: a member that fits one CTA's shared memory stays there for the whole ch_step call (measured on B200, 64^2: 3.3 vs 7.2 us
    // per step for one member, 2.7e11 vs 1.4e11 updates/s for 4096 members)
    // (128^2 over 2-CTA clusters: 1.59e11 vs 0.92e11 - 1.45e11; 256^2 over 8-CTA clusters is SLOWER than the line kernel, 1.13e11 vs
    // 1.40e11 -- 15 clusters fit the device and a CTA's phases do not overlap -- and stays an explicit option)
    if (c->opt_fuse == 0 && c->resident_ok && c->res_CS <= 2) return 6;
    // auto: the line kernels where the shape has one (measured faster: CFG3 0.218 vs 0.263 ms); everywhere else the
    // one-pass local step when gamma dt allows it (N = 768: 0.274 vs 0.324 ms; N % 16 != 0: 0.25 vs 2.5 - 6.3 ms)
    if (c->opt_fuse == 0 && c->local_ok && !c->line_ok && !c->cline_ok) return 5;
    if (c->opt_fuse == 2) return c->fused_ok ? 2 : 0;
    if (c->opt_fuse == 3) return c->line_ok ? 3 : 0;
    if (c->opt_fuse == 4) return c->cline_ok ? 4 : 0;
    return c->line_ok ? 3 : (c->cline_ok ? 4 : (c->fused_ok ? 2 : 0));
}

static bool use_rhs3_stream(const ch_ctx *c) { return c->r3_ok && c->opt_rhs3 != 1; }

// Launch that may overlap the tail of the kernel before it on the stream (programmatic dependent launch; the kernel calls pdl_wait()
// before it touches memory): option "pdl" 1 switches it off.
template <typename... KArgs, typename... Args>
static void pdl_launch(ch_ctx *c, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = c->opt_pdl == 1 ? 0 : 1;
    cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// member-resident stepping over clusters: (N, CTAs per member) instantiated
// (measured on B200, updates/s at 512 / 256 members: 128^2: 2 CTAs 1.59e11, 4 CTAs 1.41e11, 8 CTAs 1.44e11; 256^2: 8 CTAs 1.13e11, 16 CTAs 1.14e11)
#define RES_CL_CASES(X) X(128, 2) X(256, 8)
template <int NC, int CS>
static void res_cl_config(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *at, int members, cudaStream_t st)
{
    cfg.gridDim = dim3((unsigned)members * CS); cfg.blockDim = dim3(NC * (NC / CS) / RES_LC);
    cfg.dynamicSmemBytes = resident_cl_smem(NC, CS); cfg.stream = st;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
}
template <int NC, int CS>
static cudaError_t res_cl_setup(int *nclusters)
{
    cudaError_t e = cudaFuncSetAttribute(k_step2d_resident_cl<NC, CS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)resident_cl_smem(NC, CS));
    if (e == cudaSuccess && CS > 8) e = cudaFuncSetAttribute(k_step2d_resident_cl<NC, CS>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    res_cl_config<NC, CS>(cfg, at, 1, 0);
    return cudaOccupancyMaxActiveClusters(nclusters, k_step2d_resident_cl<NC, CS>, &cfg);
}
template <int NC, int CS>
static void res_cl_launch(ch_ctx *c, const SweepParams &prm, const ResidentParams &rp)
{
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    res_cl_config<NC, CS>(cfg, at, c->M, c->stream);
    cudaLaunchKernelEx(&cfg, k_step2d_resident_cl<NC, CS>, prm, rp, c->C);
}

// Brackets one kernel launch with CUDA events on the context's stream when profiling is on.
struct ProfScope {
    ch_ctx *c; int kind; cudaEvent_t e0;
    ProfScope(ch_ctx *ctx, int k) : c(ctx), kind(k), e0(nullptr)
    {
        if (c->profiling && cudaEventCreate(&e0) == cudaSuccess) cudaEventRecord(e0, c->stream);
    }
    ~ProfScope()
    {
        c->launches++;
        if (!e0) return;
        cudaEvent_t e1;
        if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return; }
        cudaEventRecord(e1, c->stream);
        c->prof.push_back({ kind, e0, e1 });
    }
};

static thread_local std::string g_create_err;

static int fail(ch_ctx *ctx, int code, const std::string &msg)
{
    if (ctx) ctx->err = msg; else g_create_err = msg;
    return code;
}

#define CUDA_TRY(ctx, call)                                                                         \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(ctx, CH_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
    } while (0)

static int chunk_len_for(int N);
static size_t ipow(size_t n, int d) { size_t p = 1; while (d-- > 0) p *= n; return p; }
static size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

static int rhs_parts(int N, int D)
{
    if (D == 2) return ((N + RHS2_TX - 1) / RHS2_TX) * ((N + RHS2_TY - 1) / RHS2_TY);
    return ((N + RHS3_TX - 1) / RHS3_TX) * ((N + RHS3_TY - 1) / RHS3_TY) * ((N + RHS3_TZ - 1) / RHS3_TZ);
}

// Fused 2D step geometry: chunks per CTA (CPB) and cluster size (CS) for P chunks per line.
// Returns false when no legal split exists (then the three-pass path is used).
static bool fused_geometry(int N, int D, int *CPB, int *CS, int *strips)
{
    const int LC = chunk_len_for(N);
    if (D != 2 || LC == 0) return false;
    const int P = N / LC;
    if (P > 64) return false;                      // exchange slots: 4 * P * 32 doubles of shared memory
    int best = 0;
    for (int cpb = 1; cpb <= 16 && cpb <= P; ++cpb)
        if (P % cpb == 0 && P / cpb <= 8) { best = cpb; if (cpb >= 8) break; }
    if (!best) return false;
    *CPB = best; *CS = P / best; *strips = (N + FUSED_VALID - 1) / FUSED_VALID;
    return true;
}

// Line kernel geometry: whole lines of P = N / 16 chunks in one CTA of N threads; N is a template
// parameter of the kernel, instantiated for the sizes below.
#define LINE_SIZES(X) X(32) X(64) X(96) X(128) X(160) X(192) X(224) X(256) X(320) X(384) X(448) X(512)
static bool line_geometry(int N, int D, int *strips)
{
    if (D != 2) return false;
    bool ok = false;
#define X(NC) ok = ok || N == NC;
    LINE_SIZES(X)
#undef X
    if (!ok) return false;
    *strips = (N + LINE_VALID - 1) / LINE_VALID;
    return true;
}

static bool rhs3_stream_geometry(int N, int D, int *parts)
{
    if (D != 3 || (N != 64 && N != 96 && N != 128)) return false;
    *parts = ((N + R3_VALID - 1) / R3_VALID) * (N / R3_ZR);
    return true;
}

static size_t line_smem(int N)
{
    const int P = N / LINE_LC;
    return (size_t)(LINE_LC + 4) * 16 * P * 16 + (size_t)4 * P * LINE_SS * 16;
}

static int max_parts(int N, int D)
{
    int n = rhs_parts(N, D), cpb, cs, st;
    if (fused_geometry(N, D, &cpb, &cs, &st) && st * cs > n) n = st * cs;
    if (line_geometry(N, D, &st) && st * (N / 32) > n) n = st * (N / 32);      // one partial per (strip, warp)
    if (rhs3_stream_geometry(N, D, &st) && st > n) n = st;
    return n;
}

static bool shape_ok(int ensemble, int N, int D) { return ensemble >= 1 && N >= 8 && (D == 2 || D == 3); }

extern "C" size_t ch_workspace_bytes(int ensemble, int N, int D)
{
    if (!shape_ok(ensemble, N, D)) return 0;
    const size_t total = (size_t)ensemble * ipow(N, D);
    return 2 * align256(total * 8) + align256((size_t)ensemble * max_parts(N, D) * 3 * 8) + align256((size_t)ensemble * 4 * 8);
}

static void carve(ch_ctx *c)
{
    char *p = (char *)c->ws_base;
    c->C = (double *)p; p += align256(c->total * 8);
    c->w = (double *)p; p += align256(c->total * 8);
    c->partials = (double *)p; p += align256((size_t)c->M * max_parts(c->N, c->D) * 3 * 8);
    c->eout = (double *)p;
}

static int chunk_len_for(int N)
{
    if (N % 16 != 0 || N < 16) return 0;
    if (N / 16 <= 64) return 16;
    if (N % 32 == 0 && N / 32 <= CH_MAX_P) return 32;
    return 0;
}

extern "C" int ch_create(ch_ctx **out, int ensemble, int N, int D, double gamma, double dt)
{
    if (!out) return fail(nullptr, CH_EINVAL, "ch_create: out is NULL");
    *out = nullptr;
    if (!shape_ok(ensemble, N, D)) return fail(nullptr, CH_EINVAL, "ch_create: need ensemble >= 1, N >= 8, D in {2,3}");
    if (!(gamma > 0) || !(dt > 0) || !std::isfinite(gamma) || !std::isfinite(dt))
        return fail(nullptr, CH_EINVAL, "ch_create: need finite gamma > 0 and dt > 0");
    if (ipow(N, D) * (size_t)ensemble > ((size_t)1 << 40)) return fail(nullptr, CH_EINVAL, "ch_create: problem too large");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, CH_ECUDA, "ch_create: no CUDA device (libch has no CPU fallback)");
    }
    ch_ctx *c = new (std::nothrow) ch_ctx();
    if (!c) return fail(nullptr, CH_ENOMEM, "ch_create: out of host memory");
    c->M = ensemble; c->N = N; c->D = D; c->gamma = gamma; c->dt = dt;
    c->npts = ipow(N, D); c->total = c->npts * ensemble;
    c->Mfull = ensemble; c->view_m0 = 0; c->rh_in = c->rh_comp = c->rh_out = nullptr;
    c->pow2 = (N & (N - 1)) == 0;
    c->LC = chunk_len_for(N);
    c->chunked = c->LC != 0;
    if (ch_factor_build(&c->fac, N, gamma * dt, c->LC) != 0) {
        delete c;
        return fail(nullptr, CH_EINVAL, "ch_create: factorisation of I + gamma dt (delta^2)^2 failed its self-check");
    }
    c->rscale = dt / std::pow(c->fac.c0, D);
    c->dW = nullptr; c->dW16 = nullptr; c->dS2 = nullptr; c->dS2c = nullptr; c->dS2_16 = nullptr;
    c->nparts = rhs_parts(N, D);
    if (D == 2) { c->rhs_tiles_x = (N + RHS2_TX - 1) / RHS2_TX; c->rhs_tiles_y = (N + RHS2_TY - 1) / RHS2_TY; }
    else { c->rhs_tiles_x = (N + RHS3_TX - 1) / RHS3_TX; c->rhs_tiles_y = (N + RHS3_TY - 1) / RHS3_TY; }
    c->ws_base = nullptr; c->ws_owned = false; c->ws_bytes = 0;
    c->C = c->w = c->partials = c->eout = nullptr;
    c->has_state = false; c->n = 0; c->t0 = 0.0;
    c->series = nullptr; c->stride = 0; c->capacity = 0; c->cursor = 0; c->last_sampled = -1;
    c->stream = 0; c->opt_sweep = 0; c->opt_fuse = 0; c->opt_linesync = 0; c->opt_scan = 0;
    c->opt_graph = 0; c->gexec = nullptr; c->cap_stream = nullptr; c->gsig = -1; c->glaunches = 0; c->graph_broken = false; c->launches = 0; c->profiling = false;
    c->f_CPB = c->f_CS = c->f_strips = 0;
    c->fused_ok = fused_geometry(N, D, &c->f_CPB, &c->f_CS, &c->f_strips);
    c->cline_ok = false; c->cl_CS = 0; c->cl_strips = 0; c->cl_resident = 0;
    // (the chunk tables of a truncated closure do not depend on N: build them at a line length ch_factor allows)
    if (D == 2 && (N == 1024 || N == 2048 || N == 4096) && ch_factor_build(&c->fac16, N < 2048 ? N : 2048, gamma * dt, LINE_LC) == 0) {
        c->cl_CS = N / CLINE_NC; c->cl_strips = (N + LINE_VALID - 1) / LINE_VALID;
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = c->cl_CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.gridDim = dim3(c->cl_CS * 64); cfg.blockDim = dim3(CLINE_NC); cfg.dynamicSmemBytes = cline_smem();
        cfg.attrs = at; cfg.numAttrs = 1;
        int ncl = 0;
        cudaError_t e = cudaSuccess;
#define X(CSV)                                                                                                               \
        if (c->cl_CS == CSV) {                                                                                                \
            e = cudaFuncSetAttribute(k_rhs_sweep_y_cline<CSV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cline_smem()); \
            if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs_sweep_y_cline<CSV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cline_smem()); \
            if (e == cudaSuccess) e = cudaOccupancyMaxActiveClusters(&ncl, k_rhs_sweep_y_cline<CSV, true>, &cfg);           \
        }
        X(2) X(4) X(8)
#undef X
        if (e == cudaSuccess && ncl >= 1) { c->cline_ok = true; c->cl_resident = ncl; }
        if (c->cline_ok && c->fac16.K > 2) {
            // long closure: tables of the scan kernels (M^lane of a 16-point chunk, group closure of the cluster)
            double tab[128 + 32];
            double WG[8][4];
            memcpy(tab, c->fac16.Mlane, sizeof(double) * 128);
            if (ch_factor_groups(&c->fac16, c->cl_CS, WG) != 0) c->cline_ok = false;
            memcpy(tab + 128, WG, sizeof(double) * 32);
            if (c->cline_ok) e = cudaMalloc((void **)&c->dS2c, sizeof(tab));
            if (c->cline_ok && e == cudaSuccess) e = cudaMemcpy(c->dS2c, tab, sizeof(tab), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) c->cline_ok = false;
        }
        if (c->cline_ok && c->LC != LINE_LC && N / LINE_LC <= CH_MAX_P) {
            // the x-sweep of the cluster line step also runs at chunk length 16 (69 registers instead of 123)
            e = cudaMalloc((void **)&c->dW16, sizeof(double) * 4 * CH_MAX_P);
            if (e == cudaSuccess) e = cudaMemcpy(c->dW16, c->fac16.W, sizeof(double) * 4 * CH_MAX_P, cudaMemcpyHostToDevice);
            if (e == cudaSuccess) e = cudaMalloc((void **)&c->dS2_16, sizeof(double) * 144);
            if (e == cudaSuccess) e = cudaMemcpy(c->dS2_16, c->fac16.Mlane, sizeof(double) * 128, cudaMemcpyHostToDevice);
            if (e == cudaSuccess) e = cudaMemcpy(c->dS2_16 + 128, c->fac16.WG, sizeof(double) * 16, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) {
                if (c->dW16) cudaFree(c->dW16);
                if (c->dS2_16) cudaFree(c->dS2_16);
                c->dW16 = nullptr; c->dS2_16 = nullptr;
            }
        }
        cudaGetLastError();
    }
    c->opt_sweep3 = 0; c->dir3 = 0;
    c->xy_ok = D == 3 && (N == 64 || N == 128) && c->chunked;
    if (c->xy_ok) {
        const int smem = N * N * 8 + 2 * (N / 16) * N * 8;
        cudaError_t e = N == 64 ? cudaFuncSetAttribute(k_sweep_xy_plane<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)
                                : cudaFuncSetAttribute(k_sweep_xy_plane<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess && N == 128)
            e = cudaFuncSetAttribute(k_sweep_xy_pair, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 128 * 8 + 2 * 2 * 8 * 128 * 8);
        if (e != cudaSuccess) c->xy_ok = false;
        cudaGetLastError();
    }
    c->r3_parts = 0; c->r3_resident = 0; c->opt_rhs3 = 0;
    c->r3_ok = rhs3_stream_geometry(N, D, &c->r3_parts);
    if (c->r3_ok) {
        const int smem = (int)rhs3_stream_smem(N);
        int per_sm = 0, dev = 0, sms = 0;
        cudaError_t e = cudaErrorInvalidValue;
#define X(NC)                                                                                                        \
        if (N == NC) {                                                                                               \
            e = cudaFuncSetAttribute(k_rhs3d_stream<NC, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);  \
            if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs3d_stream<NC, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
            if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_rhs3d_stream<NC, false>, 4 * NC, smem); \
        }
        X(64) X(96) X(128)
#undef X
        if (e == cudaSuccess) e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || per_sm < 1 || sms < 1) c->r3_ok = false;
        else c->r3_resident = per_sm * sms;
        cudaGetLastError();
    }
    c->l_strips = 0; c->l_resident = 0;
    c->line_ok = line_geometry(N, D, &c->l_strips);
    // one-pass local step: needs the decay reach of the recurrences within LOC_HMAX (gamma dt <~ 0.012)
    c->local_ok = false; c->loc_H = -1; c->loc_resident = 0;
    if (D == 2 && N % 4 == 0 && N >= 64) {
        c->loc_H = ch_factor_reach(&c->fac, ldexp(1.0, -56), LOC_HMAX);
        if (c->loc_H >= 0) {
            if (c->loc_H < 2) c->loc_H = 2;
            int per_sm = 0, dev = 0, sms = 0;
            cudaError_t e = cudaFuncSetAttribute(k_step2d_local, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)local_smem_bytes());
            if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_step2d_local, LOC_NT, local_smem_bytes());
            if (e == cudaSuccess) e = cudaGetDevice(&dev);
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e == cudaSuccess && per_sm >= 1 && sms >= 1) { c->local_ok = true; c->loc_resident = per_sm * sms; }
            cudaGetLastError();
        }
    }
    // member-resident stepping: the member and its work array in one CTA's shared memory
    c->resident_ok = false; c->res_CS = 1; c->sms = 1; c->opt_resident = 0; c->opt_pdl = 0;
    if (D == 2 && c->LC == RES_LC && (N == 128 || N == 256)) {
        c->res_CS = N == 128 ? 2 : 8;
        int nclusters = 0;
        cudaError_t e = cudaErrorInvalidValue;
#define X(NC, CS) if (N == NC && c->res_CS == CS) e = res_cl_setup<NC, CS>(&nclusters);
        RES_CL_CASES(X)
#undef X
        c->resident_ok = e == cudaSuccess && nclusters >= 1;
        c->res_clusters = nclusters;
        cudaGetLastError();
    }
    if (D == 2 && c->LC == RES_LC && (N == 32 || N == 64 || N == 96)) {
        cudaError_t e = cudaSuccess;
        const int smem = (int)resident_smem(N);
        if (N == 32) e = cudaFuncSetAttribute(k_step2d_resident<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        else if (N == 64) e = cudaFuncSetAttribute(k_step2d_resident<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        else e = cudaFuncSetAttribute(k_step2d_resident<96>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        const int smem2 = (int)resident2_smem(N);
        if (e == cudaSuccess && N == 32) e = cudaFuncSetAttribute(k_step2d_resident2<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2);
        if (e == cudaSuccess && N == 64) e = cudaFuncSetAttribute(k_step2d_resident2<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2);
        if (e == cudaSuccess && N == 96) e = cudaFuncSetAttribute(k_step2d_resident2<96>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2);
        int dev = 0;
        if (e == cudaSuccess) e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
        c->resident_ok = e == cudaSuccess;
        cudaGetLastError();
    }
    if (c->chunked) {
        cudaError_t e = cudaMalloc((void **)&c->dW, sizeof(double) * 4 * CH_MAX_P);
        if (e == cudaSuccess) e = cudaMemcpy(c->dW, c->fac.W, sizeof(double) * 4 * CH_MAX_P, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMalloc((void **)&c->dS2, sizeof(double) * 144);
        if (e == cudaSuccess) e = cudaMemcpy(c->dS2, c->fac.Mlane, sizeof(double) * 128, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(c->dS2 + 128, c->fac.WG, sizeof(double) * 16, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            std::string msg = std::string("ch_create: ") + cudaGetErrorString(e);
            cudaGetLastError();
            ch_destroy(c);            // frees every table allocated so far (dW, dS2, dS2c, dW16, dS2_16)
            return fail(nullptr, e == cudaErrorMemoryAllocation ? CH_ENOMEM : CH_ECUDA, msg);
        }
    }
    // opt in to the dynamic shared memory the kernels need
    cudaFuncSetAttribute(k_rhs3d<false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHS3_SMEM);
    cudaFuncSetAttribute(k_rhs3d<true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHS3_SMEM);
    cudaFuncSetAttribute(k_rhs3d<true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHS3_SMEM);
    cudaFuncSetAttribute(k_rhs3d<false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHS3_SMEM);
    cudaFuncSetAttribute(k_rhs3d<true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHS3_SMEM);
    cudaFuncSetAttribute(k_rhs3d<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHS3_SMEM);
    cudaFuncSetAttribute(k_sweep_pcr_x, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    cudaFuncSetAttribute(k_sweep_contig<16, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
    cudaFuncSetAttribute(k_sweep_contig<16, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
    cudaFuncSetAttribute(k_sweep_contig<32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
    cudaFuncSetAttribute(k_sweep_contig<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
    cudaFuncSetAttribute(k_rhs_sweep_y<16, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    cudaFuncSetAttribute(k_rhs_sweep_y<16, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    cudaFuncSetAttribute(k_rhs_sweep_y<32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    cudaFuncSetAttribute(k_rhs_sweep_y<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    cudaFuncSetAttribute(k_sweep_x_update<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_sweep_x_update<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (c->line_ok) {
        const int smem = (int)line_smem(N);
        int per_sm = 0, dev = 0, sms = 0;
        cudaError_t e = cudaErrorInvalidValue;
#define X(NC)                                                                                                             \
        if (N == NC) {                                                                                                    \
            e = cudaFuncSetAttribute(k_rhs_sweep_y_line<NC, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);   \
            if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs_sweep_y_line<NC, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
            if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs_sweep_y_line<NC, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
            if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs_sweep_y_line<NC, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
            if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_rhs_sweep_y_line<NC, false, false>, NC, smem); \
        }
        LINE_SIZES(X)
#undef X
        if (e == cudaSuccess) e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || per_sm < 1 || sms < 1) c->line_ok = false;
        else c->l_resident = per_sm * sms;
    }
    cudaGetLastError();
    *out = c;
    return CH_OK;
}

static void prof_clear(ch_ctx *ctx)
{
    for (auto &r : ctx->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    ctx->prof.clear();
}

extern "C" int ch_destroy(ch_ctx *ctx)
{
    if (!ctx) return CH_EINVAL;
    cudaStreamSynchronize(ctx->stream);
    prof_clear(ctx);
    if (ctx->ws_owned && ctx->ws_base) cudaFree(ctx->ws_base);
    if (ctx->dW) cudaFree(ctx->dW);
    if (ctx->dW16) cudaFree(ctx->dW16);
    if (ctx->dS2) cudaFree(ctx->dS2);
    if (ctx->dS2c) cudaFree(ctx->dS2c);
    if (ctx->gexec) cudaGraphExecDestroy(ctx->gexec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    if (ctx->rh_in) cudaStreamDestroy(ctx->rh_in);
    if (ctx->rh_comp) cudaStreamDestroy(ctx->rh_comp);
    if (ctx->rh_out) cudaStreamDestroy(ctx->rh_out);
    if (ctx->dS2_16) cudaFree(ctx->dS2_16);
    delete ctx;
    return CH_OK;
}

extern "C" const char *ch_last_error(const ch_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" int ch_set_stream(ch_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return CH_EINVAL;
    ctx->stream = (cudaStream_t)cuda_stream;
    return CH_OK;
}

extern "C" int ch_attach_workspace(ch_ctx *ctx, void *dev, size_t bytes)
{
    if (!ctx) return CH_EINVAL;
    if (!dev || ((uintptr_t)dev & 255)) return fail(ctx, CH_EINVAL, "ch_attach_workspace: need a 256-byte aligned device pointer");
    if (bytes < ch_workspace_bytes(ctx->M, ctx->N, ctx->D)) return fail(ctx, CH_EINVAL, "ch_attach_workspace: workspace too small");
    if (ctx->has_state) return fail(ctx, CH_ESTATE, "ch_attach_workspace: must precede ch_set_state");
    if (ctx->ws_owned && ctx->ws_base) cudaFree(ctx->ws_base);
    ctx->ws_base = dev; ctx->ws_owned = false; ctx->ws_bytes = bytes;
    carve(ctx);
    return CH_OK;
}

static int ensure_workspace(ch_ctx *ctx)
{
    if (ctx->ws_base) return CH_OK;
    const size_t bytes = ch_workspace_bytes(ctx->M, ctx->N, ctx->D);
    cudaError_t e = cudaMalloc(&ctx->ws_base, bytes);
    if (e != cudaSuccess) {
        ctx->ws_base = nullptr;
        cudaGetLastError();
        return fail(ctx, e == cudaErrorMemoryAllocation ? CH_ENOMEM : CH_ECUDA, std::string("cudaMalloc workspace: ") + cudaGetErrorString(e));
    }
    ctx->ws_owned = true; ctx->ws_bytes = bytes;
    carve(ctx);
    return CH_OK;
}

extern "C" int ch_set_state(ch_ctx *ctx, const double *C, int on_device)
{
    if (!ctx) return CH_EINVAL;
    if (!C) return fail(ctx, CH_EINVAL, "ch_set_state: C is NULL");
    int rc = ensure_workspace(ctx);
    if (rc) return rc;
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->C, C, ctx->total * 8, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    if (!on_device) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->has_state = true; ctx->n = 0; ctx->t0 = 0.0; ctx->cursor = 0; ctx->last_sampled = -1;
    return CH_OK;
}

extern "C" int ch_set_time(ch_ctx *ctx, double t0)
{
    if (!ctx) return CH_EINVAL;
    if (!std::isfinite(t0)) return fail(ctx, CH_EINVAL, "ch_set_time: t0 not finite");
    ctx->t0 = t0;
    return CH_OK;
}

extern "C" int ch_set_series(ch_ctx *ctx, double *series_dev, int stride, int capacity)
{
    if (!ctx) return CH_EINVAL;
    if (series_dev && (stride < 1 || capacity < 1)) return fail(ctx, CH_EINVAL, "ch_set_series: need stride >= 1 and capacity >= 1");
    ctx->series = series_dev; ctx->stride = series_dev ? stride : 0; ctx->capacity = series_dev ? capacity : 0;
    ctx->cursor = 0; ctx->last_sampled = -1;
    return CH_OK;
}

extern "C" int ch_series_count(const ch_ctx *ctx) { return ctx ? ctx->cursor : CH_EINVAL; }
extern "C" long long ch_step_count(const ch_ctx *ctx) { return ctx ? ctx->n : CH_EINVAL; }
extern "C" long long ch_launch_count(const ch_ctx *ctx) { return ctx ? ctx->launches : CH_EINVAL; }

extern "C" int ch_profile(ch_ctx *ctx, int enable)
{
    if (!ctx) return CH_EINVAL;
    prof_clear(ctx);
    ctx->profiling = enable != 0;
    return CH_OK;
}

extern "C" int ch_profile_read(ch_ctx *ctx, double *ms, long long *counts, int nkinds)
{
    if (!ctx || !ms || !counts || nkinds < 1) return CH_EINVAL;
    for (int k = 0; k < nkinds; ++k) { ms[k] = 0.0; counts[k] = 0; }
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    for (auto &r : ctx->prof) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, r.e0, r.e1) == cudaSuccess && r.kind < nkinds) { ms[r.kind] += t; counts[r.kind]++; }
    }
    prof_clear(ctx);
    return CH_OK;
}

extern "C" int ch_kernel_kinds(void) { return KIND_COUNT; }
extern "C" const char *ch_kernel_kind_name(int kind) { return kind >= 0 && kind < KIND_COUNT ? kKindNames[kind] : ""; }

extern "C" int ch_set_option(ch_ctx *ctx, const char *key, int value)
{
    if (!ctx || !key) return CH_EINVAL;
    if (!strcmp(key, "sweep")) {
        if (value < 0 || value > 3) return fail(ctx, CH_EINVAL, "ch_set_option: sweep must be 0 (auto), 1 (generic), 2 (chunked LU) or 3 (PCR x-sweep)");
        if (value == 3 && !(ctx->pow2 && ctx->N <= 4096)) return fail(ctx, CH_EINVAL, "ch_set_option: the PCR sweep needs N a power of two <= 4096");
        if (value == 2 && !ctx->chunked) return fail(ctx, CH_EINVAL, "ch_set_option: chunked sweeps need N % 16 == 0");
        ctx->opt_sweep = value;
        return CH_OK;
    }
    if (!strcmp(key, "graph")) {
        if (value < 0 || value > 2) return fail(ctx, CH_EINVAL, "ch_set_option: graph must be 0 (auto), 1 (off) or 2 (always)");
        ctx->opt_graph = value;
        return CH_OK;
    }
    if (!strcmp(key, "scan")) {
        if (value < 0 || value > 2) return fail(ctx, CH_EINVAL, "ch_set_option: scan must be 0 (auto), 1 (off) or 2 (always)");
        ctx->opt_scan = value;
        return CH_OK;
    }
    if (!strcmp(key, "sweep3")) {
        if (value < 0 || value > 2) return fail(ctx, CH_EINVAL, "ch_set_option: sweep3 must be 0 (auto), 1 (separate x and y sweeps) or 2 (one CTA per plane)");
        ctx->opt_sweep3 = value;
        return CH_OK;
    }
    if (!strcmp(key, "rhs3")) {
        if (value < 0 || value > 1) return fail(ctx, CH_EINVAL, "ch_set_option: rhs3 must be 0 (auto) or 1 (tile kernel)");
        ctx->opt_rhs3 = value;
        return CH_OK;
    }
    if (!strcmp(key, "linesync")) {
        if (value < 0 || value > 1) return fail(ctx, CH_EINVAL, "ch_set_option: linesync must be 0 (auto) or 1 (CTA barriers)");
        ctx->opt_linesync = value;
        return CH_OK;
    }
    if (!strcmp(key, "pdl")) {
        if (value < 0 || value > 1) return fail(ctx, CH_EINVAL, "ch_set_option: pdl must be 0 (programmatic dependent launches) or 1 (plain launches)");
        ctx->opt_pdl = value;
        return CH_OK;
    }
    if (!strcmp(key, "resident_lines")) {
        if (value < 0 || value > 2) return fail(ctx, CH_EINVAL, "ch_set_option: resident_lines must be 0 (auto), 1 (one line per thread) or 2 (two lines per thread)");
        ctx->opt_resident = value;
        return CH_OK;
    }
    if (!strcmp(key, "fuse")) {
        if (value < 0 || value > 6) return fail(ctx, CH_EINVAL, "ch_set_option: fuse must be 0 (auto), 1 (off), 2 (cluster), 3 (line), 4 (cluster line), 5 (one-pass local) or 6 (member-resident)");
        if (value == 6 && !ctx->resident_ok) return fail(ctx, CH_EINVAL, "ch_set_option: member-resident stepping needs D = 2 and N in {32, 64, 96, 128, 256}");
        if (value == 5 && !ctx->local_ok) return fail(ctx, CH_EINVAL, "ch_set_option: the one-pass local step needs D = 2, N % 4 == 0 and a decay reach <= 18 points (gamma dt <~ 0.012)");
        if (value == 4 && !ctx->cline_ok) return fail(ctx, CH_EINVAL, "ch_set_option: the cluster line step needs D = 2 and N in {1024, 2048, 4096}");
        if (value == 2 && !ctx->fused_ok) return fail(ctx, CH_EINVAL, "ch_set_option: the cluster-fused step needs D = 2 and N % 16 == 0");
        if (value == 3 && !ctx->line_ok) return fail(ctx, CH_EINVAL, "ch_set_option: the line-fused step needs D = 2 and N in {32, 64, 96, 128, 160, 192, 224, 256, 320, 384, 448, 512}");
        ctx->opt_fuse = value;
        return CH_OK;
    }
    return fail(ctx, CH_EINVAL, std::string("ch_set_option: unknown option ") + key);
}

extern "C" int ch_get_option(const ch_ctx *ctx, const char *key, int *value)
{
    if (!ctx || !key || !value) return CH_EINVAL;
    if (!strcmp(key, "sweep")) { *value = ctx->opt_sweep; return CH_OK; }
    if (!strcmp(key, "chunked")) { *value = ctx->chunked ? ctx->LC : 0; return CH_OK; }
    if (!strcmp(key, "K")) { *value = ctx->fac.K; return CH_OK; }
    if (!strcmp(key, "fuse")) { *value = ctx->opt_fuse; return CH_OK; }
    if (!strcmp(key, "linesync")) { *value = ctx->opt_linesync; return CH_OK; }
    if (!strcmp(key, "graph")) { *value = ctx->opt_graph; return CH_OK; }
    if (!strcmp(key, "scan")) { *value = ctx->opt_scan; return CH_OK; }
    if (!strcmp(key, "rhs3")) { *value = ctx->opt_rhs3; return CH_OK; }
    if (!strcmp(key, "sweep3")) { *value = ctx->opt_sweep3; return CH_OK; }
    if (!strcmp(key, "fused")) { *value = ctx->fused_ok ? ctx->f_CS : 0; return CH_OK; }
    if (!strcmp(key, "sweep_xy")) { *value = (ctx->xy_ok && ctx->opt_sweep3 != 1 && ctx->opt_sweep != 1) ? 1 : 0; return CH_OK; }
    if (!strcmp(key, "rhs3_stream")) { *value = use_rhs3_stream(ctx) ? ctx->r3_resident : 0; return CH_OK; }
    if (!strcmp(key, "cline")) { *value = ctx->cline_ok ? ctx->cl_resident : 0; return CH_OK; }
    if (!strcmp(key, "line")) { *value = ctx->line_ok ? ctx->l_resident : 0; return CH_OK; }
    if (!strcmp(key, "fuse_mode")) { *value = fuse_mode(ctx); return CH_OK; }
    if (!strcmp(key, "local")) { *value = ctx->local_ok ? ctx->loc_resident : 0; return CH_OK; }
    if (!strcmp(key, "local_reach")) { *value = ctx->loc_H; return CH_OK; }
    if (!strcmp(key, "resident")) { *value = ctx->resident_ok ? ctx->res_CS : 0; return CH_OK; }
    if (!strcmp(key, "resident_lines")) { *value = ctx->opt_resident; return CH_OK; }
    if (!strcmp(key, "pdl")) { *value = ctx->opt_pdl; return CH_OK; }
    if (!strcmp(key, "resident_clusters")) { *value = ctx->resident_ok ? ctx->res_clusters : 0; return CH_OK; }
    return CH_EINVAL;
}

// ---------------------------------------------------------------------------------------
// launches
// ---------------------------------------------------------------------------------------
// partials per member the RHS kernel in use writes on the three-/four-pass path
static int rhs_parts_in_use(const ch_ctx *c) { return use_rhs3_stream(c) ? c->r3_parts : c->nparts; }

template <bool DIAG, bool WRITE>
static void launch_rhs_t(ch_ctx *c, const double *C, double *r, double scale)
{
    ProfScope ps(c, DIAG ? KIND_RHS_DIAG : KIND_RHS);
    if (use_rhs3_stream(c)) {
        Rhs3Params p;
        p.gamma = c->gamma; p.mgam = -c->gamma; p.k1 = 6.0 * c->gamma - 1.0; p.scale = scale;
        p.nunits = c->r3_parts * c->M; p.write = WRITE ? 1 : 0; p.rev = c->dir3;
        const int grid = p.nunits < c->r3_resident ? p.nunits : c->r3_resident;
        const size_t smem = rhs3_stream_smem(c->N);
        if (c->N == 64) pdl_launch(c, k_rhs3d_stream<64, DIAG>, grid, 256, smem, p, C, r, c->partials);
        else if (c->N == 96) pdl_launch(c, k_rhs3d_stream<96, DIAG>, grid, 384, smem, p, C, r, c->partials);
        else pdl_launch(c, k_rhs3d_stream<128, DIAG>, grid, 512, smem, p, C, r, c->partials);
        return;
    }
    if (c->D == 2) {
        dim3 grid(c->nparts, c->M);
        if (c->pow2) k_rhs2d<DIAG, WRITE, true><<<grid, 256, 0, c->stream>>>(C, r, c->partials, c->N, c->gamma, scale, c->rhs_tiles_x);
        else k_rhs2d<DIAG, WRITE, false><<<grid, 256, 0, c->stream>>>(C, r, c->partials, c->N, c->gamma, scale, c->rhs_tiles_x);
    } else {
        dim3 grid(c->nparts, c->M);
        if (c->pow2) k_rhs3d<DIAG, WRITE, true><<<grid, 256, RHS3_SMEM, c->stream>>>(C, r, c->partials, c->N, c->gamma, scale, c->rhs_tiles_x, c->rhs_tiles_y);
        else k_rhs3d<DIAG, WRITE, false><<<grid, 256, RHS3_SMEM, c->stream>>>(C, r, c->partials, c->N, c->gamma, scale, c->rhs_tiles_x, c->rhs_tiles_y);
    }
}

static void launch_rhs(ch_ctx *c, const double *C, double *r, double scale, bool diag, bool write)
{
    if (diag && write) launch_rhs_t<true, true>(c, C, r, scale);
    else if (diag) launch_rhs_t<true, false>(c, C, r, scale);
    else launch_rhs_t<false, true>(c, C, r, scale);
}

// where the next sample of the members in view goes (ch_run_host steps member sub-ranges: view_m0, Mfull)
static double *series_slot(const ch_ctx *c) { return c->series + ((size_t)c->cursor * c->Mfull + c->view_m0) * 4; }

static void launch_finish(ch_ctx *c, double *out, double t, int nparts)
{
    ProfScope ps(c, KIND_FINISH);
    k_finish<<<c->M, 128, 0, c->stream>>>(c->partials, nparts, out, t);
}

static void fill_params(const ch_ctx *c, SweepParams &p, double oscale)
{
    p.np = c->fac.np; p.nq = c->fac.nq; p.oscale = oscale;
    memcpy(p.alpha, c->fac.alpha, sizeof(p.alpha));
    memcpy(p.beta, c->fac.beta, sizeof(p.beta));
    p.W = c->dW; p.K = c->fac.K; p.P = c->fac.P;
    // log-depth closure (contiguous-line kernels only): worth it once the K-term sum is long
    p.scan = 0; p.scan2 = 0; p.S2 = c->dS2; p.rev = 0;
    const int P = c->fac.P;
    if (c->opt_scan != 1 && (c->fac.K > 4 || c->opt_scan == 2) && P % 32 == 0 && P / 32 >= 2 && P / 32 <= 4) {
        p.scan2 = P / 32;
        memcpy(p.Mp, c->fac.Mpow2, sizeof(p.Mp));
    }
    if (c->opt_scan != 1 && (c->fac.K > 4 || c->opt_scan == 2) && P >= 2 && P <= 32 && (P & (P - 1)) == 0) {
        int lg = 0;
        while ((1 << lg) < P) ++lg;
        p.scan = lg;
        memcpy(p.Mp, c->fac.Mpow2, sizeof(p.Mp));
        memcpy(p.Wc, c->fac.Wclose, sizeof(p.Wc));
    }
}

// axis 0 = x, 1 = y, 2 = z.  update: C += result (last sweep of a step).  scale: multiply the output by oscale.
static void launch_sweep(ch_ctx *c, double *w, int axis, bool update, bool scale, double oscale, int rev = 0)
{
    const int N = c->N, D = c->D, M = c->M;
    const size_t n2 = (size_t)N * N, n3 = n2 * N;
    const bool chunked = c->chunked && c->opt_sweep != 1;
    ProfScope ps(c, KIND_SWEEP_X + axis);
    if (c->opt_sweep == 3 && axis == 0 && !update) {
        // parallel cyclic reduction (measured alternative); level tables in long double
        PcrParams p;
        long double a = c->fac.sigma / (1 + 6 * (long double)c->fac.sigma), b = -4 * a;
        const long double norm = 1 / (1 + 6 * (long double)c->fac.sigma);    // the initial division by the diagonal
        int L = 0;
        for (int st = 1; st < N && L < CH_PCR_MAX_LEVELS; st <<= 1, ++L) {
            if (fabsl(a) < 1e-22L && fabsl(b) < 1e-22L) break;
            const long double cp = 1 + 2 * a * a - 2 * b * b;
            p.A[L] = (double)(a / cp); p.B[L] = (double)(-b / cp); p.Cc[L] = (double)(1 / cp);
            const long double a2 = a * a / cp, b2 = (2 * a - b * b) / cp;
            a = a2; b = b2;
        }
        p.levels = L;
        p.final_scale = (double)(norm / (1 + 2 * a + 2 * b)) * c->fac.c0 * (scale ? oscale : 1.0);
        const long long total_lines = (long long)M * (D == 3 ? n2 : (size_t)N);
        k_sweep_pcr_x<<<(unsigned)total_lines, 256, (size_t)2 * N * 8, c->stream>>>(p, w, N);
        return;
    }
    if (!chunked) {
        long long n_lines = (long long)M * (D == 3 ? n2 : (size_t)N);
        int n_inner; size_t os, is, ls;
        if (axis == 0) { n_inner = 1; os = N; is = 0; ls = 1; }
        else if (axis == 1) { n_inner = N; os = n2; is = 1; ls = N; }
        else { n_inner = (int)n2; os = n3; is = 1; ls = n2; }
        const int blocks = (int)((n_lines + 127) / 128);
        const double *Wl = c->fac.Wline;
        if (update) k_sweep_generic<true><<<blocks, 128, 0, c->stream>>>(c->fac.np, c->fac.nq, Wl[0], Wl[1], Wl[2], Wl[3], scale ? oscale : 1.0, w, c->C, N, n_lines, n_inner, os, is, ls);
        else k_sweep_generic<false><<<blocks, 128, 0, c->stream>>>(c->fac.np, c->fac.nq, Wl[0], Wl[1], Wl[2], Wl[3], scale ? oscale : 1.0, w, c->C, N, n_lines, n_inner, os, is, ls);
        return;
    }
    SweepParams prm;
    fill_params(c, prm, oscale);
    prm.rev = rev;
    const int LC = c->LC, P = c->fac.P;
    if (axis == 0) {
        const long long total_lines = (long long)M * (D == 3 ? n2 : (size_t)N);
        int threads = 256;
        if (P > threads) threads = P;
        int LPB = threads / P;
        if (LPB > total_lines) LPB = (int)total_lines;
        threads = LPB * P;
        const int blocks = (int)((total_lines + LPB - 1) / LPB);
        const size_t smem = (size_t)LPB * N * 8 + (size_t)2 * LPB * P * 8;
        if (LC == 16) {
            if (scale) k_sweep_contig<16, true><<<blocks, threads, smem, c->stream>>>(prm, w, N, total_lines, LPB);
            else k_sweep_contig<16, false><<<blocks, threads, smem, c->stream>>>(prm, w, N, total_lines, LPB);
        } else {
            if (scale) k_sweep_contig<32, true><<<blocks, threads, smem, c->stream>>>(prm, w, N, total_lines, LPB);
            else k_sweep_contig<32, false><<<blocks, threads, smem, c->stream>>>(prm, w, N, total_lines, LPB);
        }
        return;
    }
    // strided
    size_t outer_stride, line_stride; int n_inner; long long n_outer;
    if (axis == 1) { n_inner = N; n_outer = (long long)M * (D == 3 ? N : 1); outer_stride = n2; line_stride = N; }
    else { n_inner = (int)n2; n_outer = M; outer_stride = n3; line_stride = n2; }
    int cols = 16;
    while (cols * P > 512 && cols > 4) cols >>= 1;
    const int inner_blocks = n_inner / cols;
    dim3 block(cols, P);
    const unsigned blocks = (unsigned)(inner_blocks * n_outer);
    const size_t smem = (size_t)2 * P * cols * 8;
#define LAUNCH_STRIDED(LCV)                                                                                                          \
    do {                                                                                                                             \
        if (update) pdl_launch(c, k_sweep_strided<LCV, true, false>, blocks, block, smem, prm, w, c->C, outer_stride, line_stride, inner_blocks); \
        else if (scale) pdl_launch(c, k_sweep_strided<LCV, false, true>, blocks, block, smem, prm, w, c->C, outer_stride, line_stride, inner_blocks); \
        else pdl_launch(c, k_sweep_strided<LCV, false, false>, blocks, block, smem, prm, w, c->C, outer_stride, line_stride, inner_blocks); \
    } while (0)
    if (LC == 16) LAUNCH_STRIDED(16); else LAUNCH_STRIDED(32);
#undef LAUNCH_STRIDED
}

static bool use_fused(const ch_ctx *c) { return fuse_mode(c) != 0; }

// 3D: x- and y-sweep of every z-plane in one pass
static void launch_sweep_xy(ch_ctx *c, double *w, int rev)
{
    ProfScope ps(c, KIND_SWEEP_XY);
    SweepParams prm;
    fill_params(c, prm, 1.0);
    const int P = c->fac.P;
    prm.scan = 0; prm.scan2 = 0; prm.rev = rev;
    while ((1 << prm.scan) < P) ++prm.scan;
    memcpy(prm.Mp, c->fac.Mpow2, sizeof(prm.Mp));
    memcpy(prm.Wc, c->fac.Wclose, sizeof(prm.Wc));
    const int N = c->N;
    const size_t smem = (size_t)N * N * 8 + (size_t)2 * P * N * 8;
    const unsigned planes = (unsigned)((size_t)c->M * N);
    if (N == 64) { pdl_launch(c, k_sweep_xy_plane<64>, planes, 256, smem, prm, w); return; }
    if (c->opt_sweep3 == 2) { pdl_launch(c, k_sweep_xy_plane<128>, planes, 1024, smem, prm, w); return; }
    // N = 128: half a plane per CTA, clusters of 2 (two CTAs of different planes per SM overlap load and compute)
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.gridDim = dim3(2 * planes); cfg.blockDim = dim3(512);
    cfg.dynamicSmemBytes = (size_t)64 * 128 * 8 + (size_t)2 * 2 * 8 * 128 * 8;
    cfg.stream = c->stream; cfg.attrs = at; cfg.numAttrs = c->opt_pdl == 1 ? 1 : 2;
    cudaLaunchKernelEx(&cfg, k_sweep_xy_pair, prm, w);
}

// ---- fused 2D step: (RHS + y-sweep) then (x-sweep + update) ------------------------------------
template <int LC, bool DIAG>
static void launch_rhs_sweep_y_t(ch_ctx *c, const SweepParams &prm, int write)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((size_t)c->f_CS * c->f_strips * c->M));
    cfg.blockDim = dim3(32, c->f_CPB);
    cfg.dynamicSmemBytes = (size_t)2 * c->fac.P * 32 * 16;
    cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c->f_CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, k_rhs_sweep_y<LC, DIAG>, prm, (const double *)c->C, c->w, c->partials, c->N, c->gamma,
                       c->rscale, c->f_strips, c->f_CS, write);
}

static void launch_rhs_sweep_y_line(ch_ctx *c, bool diag, bool write)
{
    LineParams p;
    p.np = c->fac.np; p.nq = c->fac.nq;
    p.gamma = c->gamma; p.mgam = -c->gamma; p.k1 = 4.0 * c->gamma - 1.0;
    memcpy(p.alpha, c->fac.alpha, sizeof(p.alpha));
    memcpy(p.beta, c->fac.beta, sizeof(p.beta));
    memcpy(p.W0, c->fac.W[0], sizeof(p.W0));
    memcpy(p.W1, c->fac.W[1], sizeof(p.W1));
    p.W = c->dW; p.K = c->fac.K;
    p.scan = 0;
    {
        const int P = c->fac.P;
        if (c->opt_scan != 1 && (p.K > 5 || c->opt_scan == 2) && (P & (P - 1)) == 0) {   // measured: K-term sum 0.123 ms (K = 3) .. 0.138 ms (K = 7), scan 0.131 ms
            while ((1 << p.scan) < P) ++p.scan;
            memcpy(p.Mp, c->fac.Mpow2, sizeof(p.Mp));
            memcpy(p.Wc, c->fac.Wclose, sizeof(p.Wc));
        }
    }
    p.ntiles = c->l_strips * c->M; p.write = write ? 1 : 0;
    p.M = c->M;
    {   // stepping kernels pack the ragged leftover strips of two members into one tile (ch_line2d.cuh, LineTiling)
        const int SF = c->N / LINE_VALID, REM = c->N - SF * LINE_VALID;
        if (!diag && REM > 0 && REM <= 12) p.ntiles = line_packed_tiles(c->N, c->M);
    }
    const int grid = p.ntiles < c->l_resident ? p.ntiles : c->l_resident;
    const size_t smem = line_smem(c->N);
    const bool nb = p.K <= 2 && c->opt_linesync != 1;     // neighbour-warp synchronisation instead of CTA barriers
#define X(NC)                                                                                                       \
    if (c->N == NC) {                                                                                               \
        if (diag && nb) k_rhs_sweep_y_line<NC, true, true><<<grid, NC, smem, c->stream>>>(p, c->C, c->w, c->partials); \
        else if (diag) k_rhs_sweep_y_line<NC, true, false><<<grid, NC, smem, c->stream>>>(p, c->C, c->w, c->partials); \
        else if (nb) pdl_launch(c, k_rhs_sweep_y_line<NC, false, true>, grid, NC, smem, p, (const double *)c->C, c->w, c->partials); \
        else pdl_launch(c, k_rhs_sweep_y_line<NC, false, false>, grid, NC, smem, p, (const double *)c->C, c->w, c->partials);       \
    }
    LINE_SIZES(X)
#undef X
}

static void launch_rhs_sweep_y_cline(ch_ctx *c)
{
    LineParams p;
    const ChFactor &f = c->fac16;
    p.np = f.np; p.nq = f.nq;
    p.gamma = c->gamma; p.mgam = -c->gamma; p.k1 = 4.0 * c->gamma - 1.0;
    memcpy(p.alpha, f.alpha, sizeof(p.alpha));
    memcpy(p.beta, f.beta, sizeof(p.beta));
    memcpy(p.W0, f.W[0], sizeof(p.W0));
    memcpy(p.W1, f.W[1], sizeof(p.W1));
    p.W = nullptr; p.K = f.K; p.scan = 0; p.S2 = c->dS2c;
    memcpy(p.Mp, f.Mpow2, sizeof(p.Mp));
    const bool scan = f.K > 2;
    p.ntiles = c->cl_strips * c->M; p.write = 1;
    const int ncl = p.ntiles < c->cl_resident ? p.ntiles : c->cl_resident;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c->cl_CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.gridDim = dim3(c->cl_CS * ncl); cfg.blockDim = dim3(CLINE_NC); cfg.dynamicSmemBytes = cline_smem();
    cfg.stream = c->stream; cfg.attrs = at; cfg.numAttrs = c->opt_pdl == 1 ? 1 : 2;
#define X(CSV)                                                                                                     \
    if (c->cl_CS == CSV) {                                                                                          \
        if (scan) cudaLaunchKernelEx(&cfg, k_rhs_sweep_y_cline<CSV, true>, p, (const double *)c->C, c->w);          \
        else cudaLaunchKernelEx(&cfg, k_rhs_sweep_y_cline<CSV, false>, p, (const double *)c->C, c->w);              \
    }
    X(2) X(4) X(8)
#undef X
}

// number of F/Fdot/mass partials per member the fused RHS kernel in use writes
static int fused_parts(const ch_ctx *c)
{
    const int mode = fuse_mode(c);
    if (mode == 5 || mode == 6) return c->line_ok ? c->l_strips * (c->N / 32) : c->nparts;
    return mode == 3 ? c->l_strips * (c->N / 32) : (mode == 4 ? c->nparts : c->f_strips * c->f_CS);
}

// diag: also reduce F, Fdot, mass of C^n into the partials; write == false (diag only): no sweep, w untouched.
// Returns true when w is left WITHOUT the RHS scale dt / c0^2 (k_sweep_x_update then applies it).
static bool launch_rhs_sweep_y(ch_ctx *c, bool diag, bool write)
{
    if (fuse_mode(c) == 5 || fuse_mode(c) == 6) {
        // one-pass local step, member-resident stepping: this entry only serves ch_energy / their sampling reduction (diagnostics-only launch)
        if (diag && c->line_ok) { ProfScope ps(c, KIND_RHS_SWEEP_Y_DIAG); launch_rhs_sweep_y_line(c, true, false); }
        else if (diag) launch_rhs(c, c->C, c->w, c->rscale, true, false);
        return true;
    }
    if (fuse_mode(c) == 4) {
        // cluster line step: the sampling reduction is a diagnostics-only launch of the tile RHS kernel
        // (reads C once more on the 1-in-stride sampling steps), the step itself never changes kernel
        if (diag) launch_rhs(c, c->C, c->w, c->rscale, true, false);
        if (write) {
            ProfScope ps(c, KIND_RHS_SWEEP_Y);
            launch_rhs_sweep_y_cline(c);
        }
        return true;
    }
    ProfScope ps(c, diag ? KIND_RHS_SWEEP_Y_DIAG : KIND_RHS_SWEEP_Y);
    if (fuse_mode(c) == 3) { launch_rhs_sweep_y_line(c, diag, write); return true; }
    SweepParams prm;
    fill_params(c, prm, 1.0);
    if (c->LC == 16) { if (diag) launch_rhs_sweep_y_t<16, true>(c, prm, write); else launch_rhs_sweep_y_t<16, false>(c, prm, 1); }
    else { if (diag) launch_rhs_sweep_y_t<32, true>(c, prm, write); else launch_rhs_sweep_y_t<32, false>(c, prm, 1); }
    return false;
}

// F, Fdot, mass partials of the current state with the same kernel (hence the same summation order)
// the stepping path samples with, so that splitting ch_step calls never changes a series value.
static int launch_diag_only(ch_ctx *c)
{
    if (use_fused(c)) { launch_rhs_sweep_y(c, true, false); return fused_parts(c); }
    launch_rhs(c, c->C, c->w, c->rscale, true, false);
    return rhs_parts_in_use(c);
}

static void launch_sweep_x_update(ch_ctx *c, bool unscaled)
{
    ProfScope ps(c, KIND_SWEEP_X_UPDATE);
    SweepParams prm;
    // the line kernels leave the RHS scale dt / c0^2 to this kernel's final fused multiply-add
    fill_params(c, prm, unscaled ? c->rscale : 1.0);
    int LC = c->LC;
    if (fuse_mode(c) == 4 && c->dW16) {
        memcpy(prm.alpha, c->fac16.alpha, sizeof(prm.alpha));
        memcpy(prm.beta, c->fac16.beta, sizeof(prm.beta));
        prm.W = c->dW16; prm.K = c->fac16.K; prm.P = c->fac16.P; prm.scan = 0; prm.scan2 = 0;
        if (c->opt_scan != 1 && (prm.K > 4 || c->opt_scan == 2) && prm.P % 32 == 0 && prm.P / 32 >= 2 && prm.P / 32 <= 4) {
            prm.scan2 = prm.P / 32; prm.S2 = c->dS2_16;
            memcpy(prm.Mp, c->fac16.Mpow2, sizeof(prm.Mp));
        }
        LC = LINE_LC;
    }
    const int N = c->N, P = prm.P;
    const long long total_lines = (long long)c->M * N;
    int threads = 128;          // measured on B200: 128-thread CTAs (4 lines at N = 512) beat 256 by 2 % (CFG3) to 11 % (CFG2)
    if (P > threads) threads = P;
    int LPB = threads / P;
    if (LPB > total_lines) LPB = (int)total_lines;
    threads = LPB * P;
    const int blocks = (int)((total_lines + LPB - 1) / LPB);
    const size_t smem = (size_t)2 * LPB * N * 8 + (size_t)2 * LPB * P * 8;
    if (LC == 16) pdl_launch(c, k_sweep_x_update<16>, blocks, threads, smem, prm, (const double *)c->w, c->C, N, total_lines, LPB);
    else pdl_launch(c, k_sweep_x_update<32>, blocks, threads, smem, prm, (const double *)c->w, c->C, N, total_lines, LPB);
}

// the whole 2D step in one pass (ch_local2d.cuh): reads c->C, writes c->w, then the two arrays swap roles
static void launch_step_local(ch_ctx *c)
{
    ProfScope ps(c, KIND_STEP_LOCAL);
    LocalParams p;
    p.np = c->fac.np; p.nq = c->fac.nq; p.mgam = -c->gamma; p.k1 = 4.0 * c->gamma - 1.0; p.oscale = c->rscale;
    p.N = c->N; p.M = c->M; p.H = c->loc_H;
    {   // homogeneous solutions of the recurrence (the same numbers as ChFactor::alpha / beta, to LOC_KC entries)
        long double a1 = 1, a2 = 0, b1 = 0, b2 = 1;
        for (int k = 0; k < LOC_KC; ++k) {
            const long double a = (long double)p.np * a1 + (long double)p.nq * a2, b = (long double)p.np * b1 + (long double)p.nq * b2;
            p.al[k] = (double)a; p.be[k] = (double)b;
            a2 = a1; a1 = a; b2 = b1; b1 = b;
        }
    }
    const int He = (p.H + 1) & ~1;
    const int swmax = (LOC_RW - 2 * He) & ~3;                  // produced columns a strip can hold, multiple of 4
    p.nstrips = (c->N + swmax - 1) / swmax;
    p.SW = (((c->N + p.nstrips - 1) / p.nstrips) + 3) & ~3;
    p.total_rows = (long long)c->M * p.nstrips * c->N;
    long long grid = c->loc_resident;
    const long long min_span = 128;                            // a segment costs 2 H + 4 extra rows: keep spans long
    if (grid * min_span > p.total_rows) grid = (p.total_rows + min_span - 1) / min_span;
    if (grid < 1) grid = 1;
    p.span = (p.total_rows + grid - 1) / grid;
    grid = (p.total_rows + p.span - 1) / p.span;
    pdl_launch(c, k_step2d_local, (unsigned)grid, LOC_NT, local_smem_bytes(), p, (const double *)c->C, c->w);
    double *t = c->C; c->C = c->w; c->w = t;
}

static long long samples_ahead(const ch_ctx *ctx, int nsteps);

// nsteps steps of the members in view, and the samples that fall inside them, in ONE launch (ch_resident2d.cuh)
// Which one-CTA kernel: the two-lines-per-thread version moves half the shared-memory bytes but runs half the warps; it wins as soon as
// several CTAs share an SM (64^2: 4096 members 3.39e11 vs 2.71e11 updates/s, 444 members 3.22e11 vs 2.59e11) and loses when a CTA has
// an SM to itself (148 members: 1.58e11 vs 1.82e11; one member 3.5 vs 3.3 us per step); 96^2 has one CTA per SM either way (2.26e11 vs 2.01e11)
static bool resident_two_lines(const ch_ctx *c)
{
    if (c->opt_resident == 1) return false;
    if (c->opt_resident == 2) return true;
    return c->N == 96 || c->M >= 2 * c->sms;
}

// energy_out != NULL: no steps, only {F, dF/dt, beta, mass} of the current state into energy_out[M][4] -- the same reduction,
// in the same order, as the samples written from inside a stepping launch (ch_energy equals the series entry bitwise)
static void launch_step_resident(ch_ctx *c, int nsteps, double *energy_out = nullptr)
{
    ProfScope ps(c, KIND_STEP_RESIDENT);
    SweepParams prm;
    fill_params(c, prm, 1.0);
    ResidentParams rp;
    rp.gamma = c->gamma; rp.mgam = -c->gamma; rp.k1 = 4.0 * c->gamma - 1.0; rp.scale = c->rscale;
    rp.t0 = c->t0; rp.dt = c->dt; rp.n0 = c->n; rp.last_sampled = c->last_sampled;
    rp.nsteps = nsteps; rp.stride = c->series ? c->stride : 0;
    rp.cursor0 = c->cursor; rp.Mfull = c->Mfull; rp.view_m0 = c->view_m0; rp.series = c->series;
    if (energy_out) {
        rp.nsteps = 0; rp.stride = 1; rp.last_sampled = -1; rp.cursor0 = 0; rp.Mfull = c->M; rp.view_m0 = 0; rp.series = energy_out;
    }
#define X(NC, CS) if (c->N == NC && c->res_CS == CS) res_cl_launch<NC, CS>(c, prm, rp);
    RES_CL_CASES(X)
#undef X
    const size_t smem = resident_smem(c->N);
    if (c->res_CS > 1) {}
    else if (resident_two_lines(c)) {
        const size_t smem2 = resident2_smem(c->N);
        if (c->N == 32) k_step2d_resident2<32><<<c->M, 16 * 2, smem2, c->stream>>>(prm, rp, c->C);
        else if (c->N == 64) k_step2d_resident2<64><<<c->M, 32 * 4, smem2, c->stream>>>(prm, rp, c->C);
        else k_step2d_resident2<96><<<c->M, 48 * 6, smem2, c->stream>>>(prm, rp, c->C);
    }
    else if (c->N == 32) k_step2d_resident<32><<<c->M, 32 * 32 / RES_LC, smem, c->stream>>>(prm, rp, c->C);
    else if (c->N == 64) k_step2d_resident<64><<<c->M, 64 * 64 / RES_LC, smem, c->stream>>>(prm, rp, c->C);
    else k_step2d_resident<96><<<c->M, 96 * 96 / RES_LC, smem, c->stream>>>(prm, rp, c->C);
    if (energy_out) return;
    const long long cnt = samples_ahead(c, nsteps);
    c->n += nsteps;
    if (cnt > 0) { c->cursor += (int)cnt; c->last_sampled = (c->n / c->stride) * c->stride; }
}

static int check_launch(ch_ctx *ctx, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(ctx, CH_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
    return CH_OK;
}

// one time step; sample: also reduce F, Fdot, mass of C^n and write the series entry
static void launch_one_step(ch_ctx *ctx, bool sample)
{
    const int D = ctx->D;
    const bool fused = use_fused(ctx);
    bool unscaled = false;
    if (fuse_mode(ctx) == 5) {
        if (sample) {
            const int np_ = launch_diag_only(ctx);
            launch_finish(ctx, series_slot(ctx), ctx->t0 + (double)ctx->n * ctx->dt, np_);
            ctx->cursor++; ctx->last_sampled = ctx->n;
        }
        launch_step_local(ctx);
        return;
    }
    if (fused) unscaled = launch_rhs_sweep_y(ctx, sample, true);
    else launch_rhs(ctx, ctx->C, ctx->w, ctx->rscale, sample, true);
    if (sample) {
        launch_finish(ctx, series_slot(ctx), ctx->t0 + (double)ctx->n * ctx->dt,
                      fused ? fused_parts(ctx) : rhs_parts_in_use(ctx));
        ctx->cursor++; ctx->last_sampled = ctx->n;
    }
    if (fused) launch_sweep_x_update(ctx, unscaled);
    else if (D == 3 && ctx->xy_ok && ctx->opt_sweep3 != 1 && ctx->opt_sweep != 1) {
        // RHS walks the ensemble in direction dir3, the plane kernel back, the z-sweep forth again, and the next
        // step starts from where this one ended: each kernel finds the tail of its predecessor's output in L2
        launch_sweep_xy(ctx, ctx->w, !ctx->dir3);
        launch_sweep(ctx, ctx->w, 2, true, false, 1.0, ctx->dir3);
        ctx->dir3 = !ctx->dir3;
    }
    else for (int axis = 0; axis < D; ++axis) launch_sweep(ctx, ctx->w, axis, axis == D - 1, false, 1.0);
}

// CUDA graph of CH_GRAPH_STEPS plain steps (their launches do not depend on the step index).  Captured on an
// internal stream (the caller's may be the legacy default stream, which cannot be captured) and replayed on
// the caller's.  Small ensembles are launch bound: CFG1's two 4096-point kernels per step.
#define CH_GRAPH_STEPS 8
static bool graph_wanted(const ch_ctx *c)
{
    if (c->opt_graph == 1 || c->graph_broken || c->profiling) return false;
    // every size: launch-bound ensembles gain most (CFG1-like: 2x), but the large configs still gain 0.3 - 1.3 % (CFG3 0.2265 -> 0.2236 ms median)
    return true;
}

static bool ensure_graph(ch_ctx *c)
{
    const long long sig = ((((((long long)(c->opt_sweep * 2 + c->opt_pdl) * 8 + c->opt_fuse) * 4 + c->opt_linesync) * 4 + c->opt_scan) * 4 + c->opt_rhs3) * 4
                           + c->opt_sweep3);
    if (c->gexec && c->gsig == sig) return true;
    if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); c->graph_broken = true; return false;
    }
    cudaStream_t user = c->stream;
    const long long l0 = c->launches;
    const int dir0 = c->dir3;
    double *const C0 = c->C, *const w0 = c->w;       // the local step ping-pongs them: an even number of steps restores them
    cudaGraph_t g = nullptr;
    c->stream = c->cap_stream;
    cudaError_t e = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        for (int i = 0; i < CH_GRAPH_STEPS; ++i) launch_one_step(c, false);
        e = cudaStreamEndCapture(c->cap_stream, &g);
    }
    c->stream = user; c->glaunches = c->launches - l0; c->launches = l0; c->dir3 = dir0;
    if (c->C != C0 || c->w != w0) { c->C = C0; c->w = w0; e = e == cudaSuccess ? cudaErrorUnknown : e; }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&c->gexec, g, 0);
    if (g) cudaGraphDestroy(g);
    if (e != cudaSuccess) { cudaGetLastError(); c->gexec = nullptr; c->graph_broken = true; return false; }
    c->gsig = sig;
    return true;
}

// samples a call of nsteps steps starting at step n0 will write: every n in [n0, n0 + nsteps] with n % stride == 0, not yet sampled
static long long samples_ahead(const ch_ctx *ctx, int nsteps)
{
    if (!ctx->series) return 0;
    long long n0 = ctx->n, n1 = ctx->n + nsteps, cnt = 0;
    long long first = ((n0 + ctx->stride - 1) / ctx->stride) * ctx->stride;
    if (first <= n1) cnt = (n1 - first) / ctx->stride + 1;
    if (first == ctx->last_sampled) cnt -= 1;
    return cnt;
}

// enqueue nsteps steps (and their samples) of the members in view on ctx->stream
static void step_body(ch_ctx *ctx, int nsteps, bool graphs)
{
    if (fuse_mode(ctx) == 6) { launch_step_resident(ctx, nsteps); return; }
    for (int s = 0; s < nsteps;) {
        const bool sample = ctx->series && (ctx->n % ctx->stride == 0) && ctx->last_sampled != ctx->n;
        if (!sample && graphs && ctx->dir3 == 0) {
            // plain steps ahead of the next sampling step (or of the end of this call)
            long long plain = nsteps - s;
            if (ctx->series) {
                const long long r = ctx->n % ctx->stride, until = r == 0 ? ctx->stride : ctx->stride - r;
                if (until < plain) plain = until;
            }
            if (plain >= CH_GRAPH_STEPS && ensure_graph(ctx)) {
                if (cudaGraphLaunch(ctx->gexec, ctx->stream) == cudaSuccess) {
                    ctx->launches += ctx->glaunches;
                    ctx->n += CH_GRAPH_STEPS; s += CH_GRAPH_STEPS;
                    continue;
                }
                cudaGetLastError(); ctx->graph_broken = true;
            }
        }
        launch_one_step(ctx, sample);
        ctx->n++; ++s;
    }
    if (ctx->series && (ctx->n % ctx->stride == 0) && ctx->last_sampled != ctx->n) {
        const int np_ = launch_diag_only(ctx);
        launch_finish(ctx, series_slot(ctx), ctx->t0 + (double)ctx->n * ctx->dt, np_);
        ctx->cursor++; ctx->last_sampled = ctx->n;
    }
}

extern "C" int ch_step(ch_ctx *ctx, int nsteps)
{
    if (!ctx) return CH_EINVAL;
    if (nsteps < 0) return fail(ctx, CH_EINVAL, "ch_step: nsteps < 0");
    if (!ctx->has_state) return fail(ctx, CH_ESTATE, "ch_step: no state (call ch_set_state first)");
    if (ctx->cursor + samples_ahead(ctx, nsteps) > ctx->capacity) return fail(ctx, CH_EINVAL, "ch_step: series full");
    step_body(ctx, nsteps, graph_wanted(ctx));
    return check_launch(ctx, "ch_step");
}

// The whole job from and to HOST memory, member chunk by member chunk, with the H2D copy of chunk k + 1, the steps of chunk k
// and the D2H copy of chunk k - 1 overlapping on three internal streams (members are independent: P:71).
extern "C" int ch_run_host(ch_ctx *ctx, const double *C_in, double *C_out, int nsteps, int chunk)
{
    if (!ctx) return CH_EINVAL;
    if (!C_in || !C_out) return fail(ctx, CH_EINVAL, "ch_run_host: C_in or C_out is NULL");
    if (nsteps < 0 || chunk < 0) return fail(ctx, CH_EINVAL, "ch_run_host: nsteps < 0 or chunk < 0");
    int rc = ensure_workspace(ctx);
    if (rc) return rc;
    if (!ctx->rh_in) {
        CUDA_TRY(ctx, cudaStreamCreateWithFlags(&ctx->rh_in, cudaStreamNonBlocking));
        CUDA_TRY(ctx, cudaStreamCreateWithFlags(&ctx->rh_comp, cudaStreamNonBlocking));
        CUDA_TRY(ctx, cudaStreamCreateWithFlags(&ctx->rh_out, cudaStreamNonBlocking));
    }
    // as after ch_set_state: n = 0, t0 = 0, series cursor reset
    ctx->has_state = true; ctx->n = 0; ctx->t0 = 0.0; ctx->cursor = 0; ctx->last_sampled = -1;
    if (samples_ahead(ctx, nsteps) > ctx->capacity) return fail(ctx, CH_EINVAL, "ch_run_host: series full");
    const int M = ctx->M;
    std::vector<int> sizes;                          // members per chunk, in order
    if (chunk == 0) {
        // default: about 4 Mi points per chunk -- 2 Mi for short jobs, whose time is the copies plus the first copy in and the last copy
        // out -- and at least 4 chunks.  Measured on CFG3, B200 (ms for 20 / 50 / 100 / 200 steps): 8 Mi-point chunks 7.7 / 13.6 / 24.7 /
        // 47.3, 4 Mi 6.8 / 12.5 / 23.7 / 46.1, 2 Mi 6.4 / 14.9 / 29.1 / 57.4 (small ensembles make the kernels less efficient); chunks
        // tapered towards both ends did not help (the very small end chunks cost more than they save)
        const size_t pts = (size_t)(nsteps <= 30 ? 2 : 4) << 20;
        const size_t want = pts / ctx->npts;
        chunk = (int)(want < 1 ? 1 : want);
        if (chunk > (M + 3) / 4) chunk = (M + 3) / 4;
        if (chunk < 1) chunk = 1;
    }
    if (chunk > M) chunk = M;
    if (sizes.empty()) for (int left = M; left > 0; left -= chunk) sizes.push_back(left < chunk ? left : chunk);
    double *const Cfull = ctx->C, *const wfull = ctx->w;
    const size_t total_full = ctx->total;
    cudaStream_t user = ctx->stream;
    cudaEvent_t ev_start = nullptr;
    CUDA_TRY(ctx, cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
    cudaEventRecord(ev_start, user);                 // everything enqueued before this call comes first
    cudaStreamWaitEvent(ctx->rh_in, ev_start, 0);
    cudaStreamWaitEvent(ctx->rh_comp, ev_start, 0);
    cudaStreamWaitEvent(ctx->rh_out, ev_start, 0);
    const int dir0 = ctx->dir3;
    long long n_end = 0; int cursor_end = 0; long long ls_end = -1;
    double *Cend = Cfull, *wend = wfull;
    cudaError_t err = cudaSuccess;
    int m0 = 0;
    for (size_t ci = 0; ci < sizes.size() && err == cudaSuccess; m0 += sizes[ci], ++ci) {
        const int mc = sizes[ci];
        const size_t off = (size_t)m0 * ctx->npts, cnt = (size_t)mc * ctx->npts;
        cudaEvent_t ev_in = nullptr, ev_comp = nullptr;
        err = cudaEventCreateWithFlags(&ev_in, cudaEventDisableTiming);
        if (err == cudaSuccess) err = cudaEventCreateWithFlags(&ev_comp, cudaEventDisableTiming);
        if (err != cudaSuccess) break;
        err = cudaMemcpyAsync(Cfull + off, C_in + off, cnt * 8, cudaMemcpyHostToDevice, ctx->rh_in);
        cudaEventRecord(ev_in, ctx->rh_in);
        cudaStreamWaitEvent(ctx->rh_comp, ev_in, 0);
        // the view: this chunk's members only
        ctx->C = Cfull + off; ctx->w = wfull + off; ctx->M = mc; ctx->total = cnt; ctx->view_m0 = m0;
        ctx->n = 0; ctx->cursor = 0; ctx->last_sampled = -1; ctx->dir3 = dir0; ctx->stream = ctx->rh_comp;
        step_body(ctx, nsteps, false);
        n_end = ctx->n; cursor_end = ctx->cursor; ls_end = ctx->last_sampled;
        // the one-pass local step ping-pongs the two arrays: the final state of the view is where ctx->C points now
        double *fin = ctx->C;
        if (m0 == 0) { Cend = fin - off; wend = ctx->w - off; }
        cudaEventRecord(ev_comp, ctx->rh_comp);
        cudaStreamWaitEvent(ctx->rh_out, ev_comp, 0);
        if (err == cudaSuccess) err = cudaMemcpyAsync(C_out + off, fin, cnt * 8, cudaMemcpyDeviceToHost, ctx->rh_out);
        cudaEventDestroy(ev_in); cudaEventDestroy(ev_comp);
    }
    // back to the whole ensemble
    ctx->C = Cend; ctx->w = wend; ctx->M = M; ctx->total = total_full; ctx->view_m0 = 0; ctx->stream = user;
    ctx->n = n_end; ctx->cursor = cursor_end; ctx->last_sampled = ls_end;
    cudaEventDestroy(ev_start);
    cudaError_t e1 = cudaStreamSynchronize(ctx->rh_in), e2 = cudaStreamSynchronize(ctx->rh_comp), e3 = cudaStreamSynchronize(ctx->rh_out);
    if (err == cudaSuccess) err = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
    if (err != cudaSuccess) return fail(ctx, CH_ECUDA, std::string("ch_run_host: ") + cudaGetErrorString(err));
    return check_launch(ctx, "ch_run_host");
}

extern "C" int ch_energy(ch_ctx *ctx, double *out, int on_device)
{
    if (!ctx) return CH_EINVAL;
    if (!out) return fail(ctx, CH_EINVAL, "ch_energy: out is NULL");
    if (!ctx->has_state) return fail(ctx, CH_ESTATE, "ch_energy: no state");
    const double t = ctx->t0 + (double)ctx->n * ctx->dt;
    if (fuse_mode(ctx) == 6) launch_step_resident(ctx, 0, on_device ? out : ctx->eout);
    else {
        const int np_ = launch_diag_only(ctx);
        launch_finish(ctx, on_device ? out : ctx->eout, t, np_);
    }
    int rc = check_launch(ctx, "ch_energy");
    if (rc) return rc;
    if (!on_device) {
        CUDA_TRY(ctx, cudaMemcpyAsync(out, ctx->eout, (size_t)ctx->M * 32, cudaMemcpyDeviceToHost, ctx->stream));
        CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
        for (int m = 0; m < ctx->M; ++m)
            if (!std::isfinite(out[4 * m])) return fail(ctx, CH_ENONFINITE, "ch_energy: non-finite free energy");
    }
    return CH_OK;
}

extern "C" int ch_get_state(ch_ctx *ctx, double *C, int on_device)
{
    if (!ctx) return CH_EINVAL;
    if (!C) return fail(ctx, CH_EINVAL, "ch_get_state: C is NULL");
    if (!ctx->has_state) return fail(ctx, CH_ESTATE, "ch_get_state: no state");
    CUDA_TRY(ctx, cudaMemcpyAsync(C, ctx->C, ctx->total * 8, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    if (!on_device) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return CH_OK;
}

extern "C" int ch_rhs(ch_ctx *ctx, double *r_out, int on_device)
{
    if (!ctx) return CH_EINVAL;
    if (!r_out) return fail(ctx, CH_EINVAL, "ch_rhs: r_out is NULL");
    if (!ctx->has_state) return fail(ctx, CH_ESTATE, "ch_rhs: no state");
    double *dst = on_device ? r_out : ctx->w;
    launch_rhs(ctx, ctx->C, dst, ctx->dt, false, true);
    int rc = check_launch(ctx, "ch_rhs");
    if (rc) return rc;
    if (!on_device) {
        CUDA_TRY(ctx, cudaMemcpyAsync(r_out, ctx->w, ctx->total * 8, cudaMemcpyDeviceToHost, ctx->stream));
        CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return CH_OK;
}

extern "C" int ch_sweep(ch_ctx *ctx, double *w, int axis, int on_device)
{
    if (!ctx) return CH_EINVAL;
    if (!w) return fail(ctx, CH_EINVAL, "ch_sweep: w is NULL");
    if (axis < 0 || axis >= ctx->D) return fail(ctx, CH_EINVAL, "ch_sweep: axis out of range");
    int rc = ensure_workspace(ctx);
    if (rc) return rc;
    double *buf = w;
    if (!on_device) {
        buf = ctx->w;
        CUDA_TRY(ctx, cudaMemcpyAsync(buf, w, ctx->total * 8, cudaMemcpyHostToDevice, ctx->stream));
    }
    launch_sweep(ctx, buf, axis, false, true, 1.0 / ctx->fac.c0);
    rc = check_launch(ctx, "ch_sweep");
    if (rc) return rc;
    if (!on_device) {
        CUDA_TRY(ctx, cudaMemcpyAsync(w, buf, ctx->total * 8, cudaMemcpyDeviceToHost, ctx->stream));
        CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return CH_OK;
}

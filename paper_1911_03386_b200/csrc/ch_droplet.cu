// ch_droplet.cu -- Model 1 of the paper on the GPU: ensembles of droplet populations.
//
//   dR_i/dt = H(R_i + eps) (-1/R_i^2 + ubar/R_i),  ubar = sum_i H(R_i) / sum_i H(R_i) R_i      eq. (39), eq. (14)
//   F = sum_i H(R_i) R_i^2 / 2,  dF/dt = -sum_i H(R_i) (1 - ubar R_i)^2 / R_i,  beta = -(t/F) dF/dt   eq. (31), (33), (36) P:319-342
//
// integrated with the Dormand-Prince 5(4) pair (the method behind the paper's ODE45) and the step controller of
// DESIGN.md reading G21.  One CTA per realisation (the paper: "one realisation of the ensemble per CPU core", P:435;
// M = 100, N = 128 ... 8192, Table 1); the whole time loop runs inside one launch.  A stage needs ubar of the
// STAGE state, i.e. a reduction over the population before the right-hand side: two passes per stage over arrays that
// stay in L1/L2 (N <= 65536 doubles per array), fixed-order block sums (warp shuffle, then warps in order), so results are
// bitwise reproducible.  Off the hot path of the Cahn-Hilliard stepper: kept small and simple on purpose.
#include <cmath>
#include <cstdio>
#include <new>
#include <string>

#include <cuda_runtime.h>

#include "../../include/ch.h"

namespace {

constexpr int DT = 256;     // threads per CTA

// Dormand-Prince 5(4) tableau (Dormand & Prince 1980); B5 is the last row of A (FSAL), E = B5 - B4
__constant__ double kA[7][6] = {
    { 0, 0, 0, 0, 0, 0 },
    { 1.0 / 5, 0, 0, 0, 0, 0 },
    { 3.0 / 40, 9.0 / 40, 0, 0, 0, 0 },
    { 44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0 },
    { 19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0 },
    { 9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0 },
    { 35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84 },
};
__constant__ double kE[7] = { 35.0 / 384 - 5179.0 / 57600, 0, 500.0 / 1113 - 7571.0 / 16695, 125.0 / 192 - 393.0 / 640,
                              -2187.0 / 6784 + 92097.0 / 339200, 11.0 / 84 - 187.0 / 2100, -1.0 / 40 };

struct Red2 { double a, b; };

// fixed-order block sums of two values; every thread gets the result
__device__ Red2 block_sum2(double a, double b, double *sh)
{
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) { sh[2 * w] = a; sh[2 * w + 1] = b; }
    __syncthreads();
    Red2 r = { 0.0, 0.0 };
    for (int q = 0; q < DT / 32; ++q) { r.a += sh[2 * q]; r.b += sh[2 * q + 1]; }
    return r;
}
__device__ double block_max(double a, double *sh)
{
    for (int o = 16; o > 0; o >>= 1) a = fmax(a, __shfl_down_sync(0xffffffffu, a, o));
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = a;
    __syncthreads();
    double r = 0.0;
    for (int q = 0; q < DT / 32; ++q) r = fmax(r, sh[q]);
    return r;
}

__device__ __forceinline__ double droplet_rhs(double r, double u, double eps)
{
    return (r + eps > 0.0 && r != 0.0) ? -1.0 / (r * r) + u / r : 0.0;
}

// k[s] = f(ys) for the stage state ys (held in ys[]): ubar of ys first (eq. (14)), then eq. (39)
__device__ void stage_rhs(const double *ys, double *ks, int N, double eps, double *sh)
{
    double cnt = 0.0, sum = 0.0;
    for (int i = threadIdx.x; i < N; i += DT) {
        const double r = ys[i];
        if (r > 0.0) { cnt += 1.0; sum += r; }
    }
    const Red2 t = block_sum2(cnt, sum, sh);
    const double u = t.b > 0.0 ? t.a / t.b : 0.0;
    for (int i = threadIdx.x; i < N; i += DT) ks[i] = droplet_rhs(ys[i], u, eps);
}

// one Dormand-Prince step of size h from R (k[0] = f(R) on entry): Rn = 5th-order solution, k[6] = f(Rn);
// returns the controller's error measure (reading G21)
__device__ double dopri_step(const double *R, double *Rn, double *ys, double *k, int N, double h, double eps,
                             double rtol, double atol, double *sh)
{
    for (int s = 1; s < 7; ++s) {
        double *dst = s == 6 ? Rn : ys;          // the 7th stage state IS the new solution (FSAL)
        for (int i = threadIdx.x; i < N; i += DT) {
            double y = R[i];
            for (int j = 0; j < s; ++j)
                if (kA[s][j] != 0.0) y += h * kA[s][j] * k[(size_t)j * N + i];
            dst[i] = y;
        }
        __syncthreads();
        stage_rhs(dst, k + (size_t)s * N, N, eps, sh);
        __syncthreads();
    }
    double err = 0.0;
    for (int i = threadIdx.x; i < N; i += DT) {
        double e = 0.0;
        for (int j = 0; j < 7; ++j)
            if (kE[j] != 0.0) e += h * kE[j] * k[(size_t)j * N + i];
        err = fmax(err, fabs(e) / (atol + rtol * fmax(fabs(R[i]), fabs(Rn[i]))));
    }
    return block_max(err, sh);
}

// scratch per realisation: R[N], Rn[N], ys[N], k[7][N]
struct DropletArrays { double *R, *Rn, *ys, *k; };
__device__ __forceinline__ DropletArrays droplet_arrays(double *base, int N, int m)
{
    double *p = base + (size_t)m * 10 * N;
    return { p, p + N, p + 2 * (size_t)N, p + 3 * (size_t)N };
}

// adaptive integration to t_end; steps_out (may be NULL): accepted step sizes, [M][max_record]
__global__ void __launch_bounds__(DT) k_droplet_integrate(double *base, double *tcur, int N, double eps, double t_end,
                                                           double rtol, double atol, double h0, long long max_steps,
                                                           double *steps_out, int max_record, int *nsteps_out)
{
    __shared__ double sh[2 * DT / 32];
    const int m = blockIdx.x;
    DropletArrays a = droplet_arrays(base, N, m);
    double t = tcur[m], h = h0;
    stage_rhs(a.R, a.k, N, eps, sh);
    __syncthreads();
    int accepted = 0;
    for (long long n = 0; n < max_steps && t < t_end; ++n) {
        h = fmin(h, t_end - t);
        const double err = dopri_step(a.R, a.Rn, a.ys, a.k, N, h, eps, rtol, atol, sh);
        if (err <= 1.0) {
            t += h;
            for (int i = threadIdx.x; i < N; i += DT) { a.R[i] = a.Rn[i]; a.k[i] = a.k[(size_t)6 * N + i]; }
            if (steps_out && accepted < max_record && threadIdx.x == 0) steps_out[(size_t)m * max_record + accepted] = h;
            ++accepted;
            __syncthreads();
        }
        h *= err > 0.0 ? fmin(5.0, fmax(0.2, 0.9 * pow(err, -0.2))) : 5.0;
    }
    if (threadIdx.x == 0) { tcur[m] = t; if (nsteps_out) nsteps_out[m] = accepted; }
}

// a given sequence of step sizes, no error control (what the fixed-sequence parity test compares with the oracle)
__global__ void __launch_bounds__(DT) k_droplet_replay(double *base, double *tcur, int N, double eps, const double *steps,
                                                        int nsteps, int stride)
{
    __shared__ double sh[2 * DT / 32];
    const int m = blockIdx.x;
    DropletArrays a = droplet_arrays(base, N, m);
    double t = tcur[m];
    stage_rhs(a.R, a.k, N, eps, sh);
    __syncthreads();
    for (int n = 0; n < nsteps; ++n) {
        const double h = steps[(size_t)m * stride + n];
        if (!(h > 0.0)) break;                      // sequences shorter than nsteps are padded with zeros
        dopri_step(a.R, a.Rn, a.ys, a.k, N, h, eps, 1.0, 1.0, sh);
        t += h;
        for (int i = threadIdx.x; i < N; i += DT) { a.R[i] = a.Rn[i]; a.k[i] = a.k[(size_t)6 * N + i]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) tcur[m] = t;
}

// out[m] = {F, dF/dt, beta, V}
__global__ void __launch_bounds__(DT) k_droplet_energy(const double *base, const double *tcur, int N, double *out)
{
    __shared__ double sh[2 * DT / 32];
    const int m = blockIdx.x;
    const double *R = base + (size_t)m * 10 * N;
    double cnt = 0.0, sum = 0.0;
    for (int i = threadIdx.x; i < N; i += DT) {
        const double r = R[i];
        if (r > 0.0) { cnt += 1.0; sum += r; }
    }
    const Red2 cs = block_sum2(cnt, sum, sh);
    const double u = cs.b > 0.0 ? cs.a / cs.b : 0.0;
    double F = 0.0, Fd = 0.0, V = 0.0;
    for (int i = threadIdx.x; i < N; i += DT) {
        const double r = R[i];
        if (r > 0.0) {
            const double q = 1.0 - u * r;
            F += 0.5 * r * r; Fd -= q * q / r; V += r * r * r;
        }
    }
    const Red2 fe = block_sum2(F, Fd, sh);
    const Red2 vv = block_sum2(V, 0.0, sh);
    if (threadIdx.x == 0) {
        const double t = tcur[m];
        out[4 * m] = fe.a; out[4 * m + 1] = fe.b;
        out[4 * m + 2] = fe.a > 0.0 ? -t * fe.b / fe.a : 0.0;
        out[4 * m + 3] = vv.a / 3.0;
    }
}

__global__ void k_droplet_scatter(double *base, const double *src, int N, int M, int to_ctx)
{
    const size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (idx >= (size_t)M * N) return;
    const size_t m = idx / N, i = idx - m * N;
    if (to_ctx) base[m * 10 * N + i] = src[idx];
    else const_cast<double *>(src)[idx] = base[m * 10 * N + i];
}

}  // namespace

struct ch_droplet_ctx {
    int M, N;
    double eps;
    double *base, *tcur, *tmp, *eout;
    bool has_state;
    cudaStream_t stream;
    std::string err;
};

static thread_local std::string g_dr_err;
static int dfail(ch_droplet_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_dr_err = msg;
    return code;
}
#define DR_TRY(ctx, call)                                                                              \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess) return dfail(ctx, CH_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

extern "C" int ch_droplet_create(ch_droplet_ctx **out, int realisations, int N, double eps)
{
    if (!out) return dfail(nullptr, CH_EINVAL, "ch_droplet_create: out is NULL");
    *out = nullptr;
    if (realisations < 1 || N < 1 || N > (1 << 20) || !(eps > 0) || !std::isfinite(eps))
        return dfail(nullptr, CH_EINVAL, "ch_droplet_create: need realisations >= 1, 1 <= N <= 2^20, finite eps > 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return dfail(nullptr, CH_ECUDA, "ch_droplet_create: no CUDA device (libch has no CPU fallback)");
    }
    ch_droplet_ctx *c = new (std::nothrow) ch_droplet_ctx();
    if (!c) return dfail(nullptr, CH_ENOMEM, "ch_droplet_create: out of host memory");
    c->M = realisations; c->N = N; c->eps = eps; c->has_state = false; c->stream = 0;
    c->base = c->tcur = c->tmp = c->eout = nullptr;
    const size_t MN = (size_t)realisations * N;
    cudaError_t e = cudaMalloc((void **)&c->base, MN * 10 * 8);
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->tmp, MN * 8);
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->tcur, (size_t)realisations * 8);
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->eout, (size_t)realisations * 32);
    if (e != cudaSuccess) {
        std::string msg = std::string("ch_droplet_create: ") + cudaGetErrorString(e);
        cudaGetLastError();
        ch_droplet_destroy(c);
        return dfail(nullptr, e == cudaErrorMemoryAllocation ? CH_ENOMEM : CH_ECUDA, msg);
    }
    *out = c;
    return CH_OK;
}

extern "C" int ch_droplet_destroy(ch_droplet_ctx *c)
{
    if (!c) return CH_EINVAL;
    cudaStreamSynchronize(c->stream);
    if (c->base) cudaFree(c->base);
    if (c->tmp) cudaFree(c->tmp);
    if (c->tcur) cudaFree(c->tcur);
    if (c->eout) cudaFree(c->eout);
    delete c;
    return CH_OK;
}

extern "C" const char *ch_droplet_last_error(const ch_droplet_ctx *c) { return c ? c->err.c_str() : g_dr_err.c_str(); }

extern "C" int ch_droplet_set_stream(ch_droplet_ctx *c, void *stream)
{
    if (!c) return CH_EINVAL;
    c->stream = (cudaStream_t)stream;
    return CH_OK;
}

extern "C" int ch_droplet_set_state(ch_droplet_ctx *c, const double *R, int on_device)
{
    if (!c) return CH_EINVAL;
    if (!R) return dfail(c, CH_EINVAL, "ch_droplet_set_state: R is NULL");
    const size_t MN = (size_t)c->M * c->N;
    const double *src = R;
    if (!on_device) {
        DR_TRY(c, cudaMemcpyAsync(c->tmp, R, MN * 8, cudaMemcpyHostToDevice, c->stream));
        src = c->tmp;
    }
    k_droplet_scatter<<<(unsigned)((MN + 255) / 256), 256, 0, c->stream>>>(c->base, src, c->N, c->M, 1);
    DR_TRY(c, cudaMemsetAsync(c->tcur, 0, (size_t)c->M * 8, c->stream));
    DR_TRY(c, cudaGetLastError());
    if (!on_device) DR_TRY(c, cudaStreamSynchronize(c->stream));
    c->has_state = true;
    return CH_OK;
}

extern "C" int ch_droplet_get_state(ch_droplet_ctx *c, double *R, int on_device)
{
    if (!c) return CH_EINVAL;
    if (!R) return dfail(c, CH_EINVAL, "ch_droplet_get_state: R is NULL");
    if (!c->has_state) return dfail(c, CH_ESTATE, "ch_droplet_get_state: no state");
    const size_t MN = (size_t)c->M * c->N;
    double *dst = on_device ? R : c->tmp;
    k_droplet_scatter<<<(unsigned)((MN + 255) / 256), 256, 0, c->stream>>>(c->base, dst, c->N, c->M, 0);
    DR_TRY(c, cudaGetLastError());
    if (!on_device) {
        DR_TRY(c, cudaMemcpyAsync(R, c->tmp, MN * 8, cudaMemcpyDeviceToHost, c->stream));
        DR_TRY(c, cudaStreamSynchronize(c->stream));
    }
    return CH_OK;
}

extern "C" int ch_droplet_integrate(ch_droplet_ctx *c, double t_end, double rtol, double atol, double h0, long long max_steps,
                                    double *steps_dev, int max_record, int *nsteps_dev)
{
    if (!c) return CH_EINVAL;
    if (!c->has_state) return dfail(c, CH_ESTATE, "ch_droplet_integrate: no state (call ch_droplet_set_state first)");
    if (!(rtol > 0) || !(atol > 0) || !(h0 > 0) || max_steps < 0 || !std::isfinite(t_end) || (steps_dev && max_record < 1))
        return dfail(c, CH_EINVAL, "ch_droplet_integrate: need rtol, atol, h0 > 0, max_steps >= 0, finite t_end");
    k_droplet_integrate<<<c->M, DT, 0, c->stream>>>(c->base, c->tcur, c->N, c->eps, t_end, rtol, atol, h0, max_steps,
                                                     steps_dev, max_record, nsteps_dev);
    DR_TRY(c, cudaGetLastError());
    return CH_OK;
}

extern "C" int ch_droplet_replay(ch_droplet_ctx *c, const double *steps_dev, int nsteps, int stride)
{
    if (!c) return CH_EINVAL;
    if (!c->has_state) return dfail(c, CH_ESTATE, "ch_droplet_replay: no state");
    if (!steps_dev || nsteps < 0 || stride < nsteps) return dfail(c, CH_EINVAL, "ch_droplet_replay: need steps, nsteps >= 0, stride >= nsteps");
    k_droplet_replay<<<c->M, DT, 0, c->stream>>>(c->base, c->tcur, c->N, c->eps, steps_dev, nsteps, stride);
    DR_TRY(c, cudaGetLastError());
    return CH_OK;
}

extern "C" int ch_droplet_energy(ch_droplet_ctx *c, double *out, int on_device)
{
    if (!c) return CH_EINVAL;
    if (!out) return dfail(c, CH_EINVAL, "ch_droplet_energy: out is NULL");
    if (!c->has_state) return dfail(c, CH_ESTATE, "ch_droplet_energy: no state");
    k_droplet_energy<<<c->M, DT, 0, c->stream>>>(c->base, c->tcur, c->N, on_device ? out : c->eout);
    DR_TRY(c, cudaGetLastError());
    if (!on_device) {
        DR_TRY(c, cudaMemcpyAsync(out, c->eout, (size_t)c->M * 32, cudaMemcpyDeviceToHost, c->stream));
        DR_TRY(c, cudaStreamSynchronize(c->stream));
    }
    return CH_OK;
}

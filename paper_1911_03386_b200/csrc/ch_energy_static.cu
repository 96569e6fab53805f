// ch_energy_static.cu -- the energy / beta reduction for callers that must not allocate: its reduction partials live in
// a file-scope __device__ array instead of a cudaMalloc'ed workspace.  include/ch.h "ch_energy_static".
//
//   k_energy_parts_static   per-part sums of F, Fdot, mass of every member     P:34 eq. (4), eq. (6)
//   k_energy_finish_static  fixed-order finish -> {F, Fdot, beta, mass}
//
// A variant of the diagnostics of k_rhs2d / k_rhs3d + k_finish (ch_kernels.cuh): same definitions (DESIGN.md section 1,
// readings G3-G6), no shared-memory tiles (neighbours come through L1/L2), and no context -- so no cudaMalloc, no
// cudaFree, no allocating library call anywhere on this path.  ch_energy (ch_api.cu) stays the fast path.
//
// The scratch array is held by every GPU that loads the library until the process exits (1.5 MiB).  Every call shares
// it, and it keeps the last call's contents: nothing in it has to start at zero (each call writes every slot it later
// reads, there are no atomics), but two calls that overlap on the GPU (different streams, or different host threads)
// RACE on it.
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/ch.h"

#define ES_PTS CH_ENERGY_STATIC_PART_POINTS
#define ES_MAX CH_ENERGY_STATIC_MAX_PARTS
#define ES_NT 256
#define ES_MAX_DEVICES 64

// [part][3] = F, Fdot, mass of ES_PTS consecutive grid points of one member; parts of a member are consecutive
static __device__ __align__(256) double g_energy_parts[(size_t)ES_MAX * 3];

// In host code `g_energy_parts` is only a stand-in for the symbol: the device address is looked up once per device,
// with that device current, and that pointer is what the kernels get.
static double *g_parts_ptr[ES_MAX_DEVICES];
static std::mutex g_parts_mutex;

static cudaError_t energy_parts_address(double **ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= ES_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_parts_mutex);
    if (!g_parts_ptr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_energy_parts);
        if (e != cudaSuccess) return e;
        g_parts_ptr[dev] = p;
    }
    *ptr = g_parts_ptr[dev];
    return cudaSuccess;
}

__device__ __forceinline__ int es_wrap(int i, int N) { return i < 0 ? i + N : (i >= N ? i - N : i); }

// mu = C^3 - C - gamma Lap_h C at (x, y, z) of one member (5- / 7-point Laplacian, periodic)     P:29-30 eq. (3)
template <int D>
__device__ __forceinline__ double es_mu(const double *__restrict__ Cm, int N, double gamma, int x, int y, int z)
{
    const size_t row = ((size_t)(D == 3 ? z : 0) * N + y) * N;
    const double c = Cm[row + x];
    double s = (Cm[row + es_wrap(x - 1, N)] + Cm[row + es_wrap(x + 1, N)])
             + (Cm[row - (size_t)y * N + (size_t)es_wrap(y - 1, N) * N + x] + Cm[row - (size_t)y * N + (size_t)es_wrap(y + 1, N) * N + x]);
    if (D == 3) {
        const size_t n2 = (size_t)N * N;
        s += Cm[(size_t)es_wrap(z - 1, N) * n2 + (size_t)y * N + x] + Cm[(size_t)es_wrap(z + 1, N) * n2 + (size_t)y * N + x];
    }
    return c * c * c - c - gamma * (s - 2.0 * D * c);
}

__device__ __forceinline__ double es_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// fixed-order sum of three values over a CTA of NW warps; the result is valid in thread 0
template <int NW>
__device__ __forceinline__ void es_block_sum3(double &a, double &b, double &c, double (*red)[3])
{
    a = es_warp_sum(a); b = es_warp_sum(b); c = es_warp_sum(c);
    if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5][0] = a; red[threadIdx.x >> 5][1] = b; red[threadIdx.x >> 5][2] = c; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = red[0][0]; b = red[0][1]; c = red[0][2];
        for (int w = 1; w < NW; ++w) { a += red[w][0]; b += red[w][1]; c += red[w][2]; }
    }
}

// grid = ensemble * ppm (ppm = parts per member), block = ES_NT.  CTA (m, part) sums over the ES_PTS consecutive points
// of member m that start at part * ES_PTS:
//   F    += (C^2 - 1)^2 / 4 + gamma / 2 sum_d (C_{i+e_d} - C_i)^2          P:34 eq. (4), forward differences (G3, G4)
//   Fdot -= sum_d (mu_{i+e_d} - mu_i)^2                                     analytic dissipation of the same state (G5)
//   mass += C
template <int D>
__global__ void __launch_bounds__(ES_NT) k_energy_parts_static(const double *__restrict__ C, double *__restrict__ parts,
                                                                int N, int ppm, double gamma)
{
    __shared__ double red[ES_NT / 32][3];
    const int m = blockIdx.x / ppm, part = blockIdx.x - m * ppm;
    const long long npts = D == 3 ? (long long)N * N * N : (long long)N * N;
    const double *Cm = C + (size_t)m * npts;
    double F = 0.0, Fd = 0.0, ms = 0.0;
    for (int k = 0; k < ES_PTS / ES_NT; ++k) {
        const long long idx = (long long)part * ES_PTS + k * ES_NT + threadIdx.x;
        if (idx < npts) {
            const int x = (int)(idx % N);
            const long long yz = idx / N;
            const int y = (int)(yz % N), z = (int)(yz / N);
            const int xp = es_wrap(x + 1, N), yp = es_wrap(y + 1, N), zp = D == 3 ? es_wrap(z + 1, N) : 0;
            const size_t n2 = (size_t)N * N;
            const double c = Cm[idx];
            const double dx = Cm[(size_t)z * n2 + (size_t)y * N + xp] - c, dy = Cm[(size_t)z * n2 + (size_t)yp * N + x] - c;
            double g2 = dx * dx + dy * dy;
            const double mu0 = es_mu<D>(Cm, N, gamma, x, y, z);
            const double mx = es_mu<D>(Cm, N, gamma, xp, y, z) - mu0, my = es_mu<D>(Cm, N, gamma, x, yp, z) - mu0;
            double d2 = mx * mx + my * my;
            if (D == 3) {
                const double dz = Cm[(size_t)zp * n2 + (size_t)y * N + x] - c;
                const double mz = es_mu<D>(Cm, N, gamma, x, y, zp) - mu0;
                g2 += dz * dz;
                d2 += mz * mz;
            }
            const double q = c * c - 1.0;
            F += 0.25 * q * q + 0.5 * gamma * g2;
            Fd -= d2;
            ms += c;
        }
    }
    es_block_sum3<ES_NT / 32>(F, Fd, ms, red);
    if (threadIdx.x == 0) {
        double *o = parts + (size_t)blockIdx.x * 3;
        o[0] = F; o[1] = Fd; o[2] = ms;
    }
}

// grid = ensemble, block = 128: out[m] = {F, Fdot, beta = -t Fdot / F (0 if F == 0), mass}     P:64 eq. (6), G6
__global__ void __launch_bounds__(128) k_energy_finish_static(const double *__restrict__ parts, int ppm, double t,
                                                              double *__restrict__ out)
{
    __shared__ double red[4][3];
    const double *p = parts + (size_t)blockIdx.x * ppm * 3;
    double F = 0.0, Fd = 0.0, ms = 0.0;
    for (int i = threadIdx.x; i < ppm; i += 128) { F += p[3 * i]; Fd += p[3 * i + 1]; ms += p[3 * i + 2]; }
    es_block_sum3<4>(F, Fd, ms, red);
    if (threadIdx.x == 0) {
        double *o = out + (size_t)blockIdx.x * 4;
        o[0] = F; o[1] = Fd; o[2] = (F == 0.0) ? 0.0 : -t * Fd / F; o[3] = ms;
    }
}

static int es_fail(char *errbuf, size_t errlen, int code, const char *msg)
{
    if (errbuf && errlen) snprintf(errbuf, errlen, "%s", msg);
    return code;
}

extern "C" int ch_energy_static(const double *C_dev, int ensemble, int N, int D, double gamma, double t, double *out_dev,
                                void *cuda_stream, char *errbuf, size_t errlen)
{
    if (errbuf && errlen) errbuf[0] = 0;
    if (!C_dev || !out_dev) return es_fail(errbuf, errlen, CH_EINVAL, "ch_energy_static: C_dev or out_dev is NULL");
    if (ensemble < 1 || N < 8 || (D != 2 && D != 3) || !(gamma > 0.0))
        return es_fail(errbuf, errlen, CH_EINVAL, "ch_energy_static: needs ensemble >= 1, N >= 8, D in {2, 3}, gamma > 0");
    const long long npts = D == 3 ? (long long)N * N * N : (long long)N * N;
    const long long ppm = (npts + ES_PTS - 1) / ES_PTS, total = ppm * ensemble;
    if (total > ES_MAX) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "ch_energy_static: ensemble * ceil(N^D / %d) = %lld partial sums exceed the static scratch of %d "
                 "(CH_ENERGY_STATIC_MAX_PARTS); use ch_energy, or split the ensemble over several calls",
                 ES_PTS, total, ES_MAX);
        return es_fail(errbuf, errlen, CH_EINVAL, msg);
    }
    double *parts = nullptr;
    cudaError_t e = energy_parts_address(&parts);
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof msg, "ch_energy_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        return es_fail(errbuf, errlen, CH_ECUDA, msg);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (D == 2) k_energy_parts_static<2><<<(unsigned)total, ES_NT, 0, st>>>(C_dev, parts, N, (int)ppm, gamma);
    else k_energy_parts_static<3><<<(unsigned)total, ES_NT, 0, st>>>(C_dev, parts, N, (int)ppm, gamma);
    k_energy_finish_static<<<ensemble, 128, 0, st>>>(parts, (int)ppm, t, out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof msg, "ch_energy_static: launch: %s", cudaGetErrorString(e));
        return es_fail(errbuf, errlen, CH_ECUDA, msg);
    }
    return CH_OK;
}

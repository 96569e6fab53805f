// ch_stats.cu -- ensemble statistics of the coarsening-rate series:
// the moments of beta over the ensemble, eq. (41a,b) P:452-456; the window average beta_0, eq. (42)
// P:460; the least-squares slope k of mu_2 = k t; and the histogram of beta per sample time
// (Figs 9, 14, 18).  Input is the series buffer ch_step writes: series[sample][member][4] =
// {F, dF/dt, beta, mass}.  Bytes are negligible (KBs); the kernels are written for determinism:
// fixed summation order, so the result does not depend on the launch.
#include <cmath>
#include <cuda_runtime.h>

#include "../../include/ch.h"

// one CTA per sample; threads stride over the members in a fixed order
__global__ void __launch_bounds__(256) k_stats_moments(const double *__restrict__ series, int M, double *__restrict__ mom)
{
    __shared__ double red[256];
    __shared__ double mean_s;
    const int s = blockIdx.x, t = threadIdx.x;
    const double *b = series + (size_t)s * M * 4 + 2;
    double acc = 0.0;
    for (int j = t; j < M; j += 256) acc += b[(size_t)j * 4];
    red[t] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) red[t] += red[t + o];
        __syncthreads();
    }
    if (t == 0) mean_s = red[0] / M;
    __syncthreads();
    const double mean = mean_s;
    double m2 = 0.0, m3 = 0.0, m4 = 0.0;
    for (int j = t; j < M; j += 256) {
        const double d = b[(size_t)j * 4] - mean, d2 = d * d;
        m2 += d2; m3 += d2 * d; m4 += d2 * d2;
    }
    double out[3] = { m2, m3, m4 };
    for (int q = 0; q < 3; ++q) {
        __syncthreads();
        red[t] = out[q];
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (t < o) red[t] += red[t + o];
            __syncthreads();
        }
        if (t == 0) mom[(size_t)s * 4 + 1 + q] = red[0] / M;
    }
    if (t == 0) mom[(size_t)s * 4] = mean;
}

// one CTA per sample; bin = floor((beta - lo) / width), values outside [lo, lo + nbins * width) are dropped
__global__ void __launch_bounds__(256) k_stats_hist(const double *__restrict__ series, int M, double lo, double width, int nbins,
                                                    int *__restrict__ hist)
{
    extern __shared__ int bins[];
    const int s = blockIdx.x, t = threadIdx.x;
    for (int i = t; i < nbins; i += 256) bins[i] = 0;
    __syncthreads();
    const double *b = series + (size_t)s * M * 4 + 2;
    for (int j = t; j < M; j += 256) {
        const double q = floor((b[(size_t)j * 4] - lo) / width);
        if (q >= 0.0 && q < (double)nbins) atomicAdd(&bins[(int)q], 1);     // integer counts: order does not matter
    }
    __syncthreads();
    for (int i = t; i < nbins; i += 256) hist[(size_t)s * nbins + i] = bins[i];
}

// single thread: trapezoid average of mu_1 and least-squares slope of mu_2 = k t over the samples in [t1, t2]
__global__ void k_stats_fit(const double *__restrict__ mom, int S, double t0, double dts, double t1, double t2, double *out)
{
    if (threadIdx.x || blockIdx.x) return;
    double integ = 0.0, stt = 0.0, stm = 0.0, tprev = 0.0, mprev = 0.0, tfirst = 0.0;
    int n = 0;
    for (int s = 0; s < S; ++s) {
        const double t = t0 + s * dts;
        if (t < t1 || t > t2) continue;
        const double m1 = mom[(size_t)s * 4], m2 = mom[(size_t)s * 4 + 1];
        if (n == 0) tfirst = t; else integ += 0.5 * (m1 + mprev) * (t - tprev);
        stt += t * t; stm += t * m2;
        tprev = t; mprev = m1; ++n;
    }
    out[0] = n >= 2 ? integ / (tprev - tfirst) : (n == 1 ? mprev : 0.0);
    out[1] = stt > 0.0 ? stm / stt : 0.0;
    out[2] = (double)n;
}

extern "C" int ch_stats_moments(const double *series_dev, int nsamples, int ensemble, double *moments_dev, void *stream)
{
    if (!series_dev || !moments_dev || nsamples < 1 || ensemble < 1) return CH_EINVAL;
    k_stats_moments<<<nsamples, 256, 0, (cudaStream_t)stream>>>(series_dev, ensemble, moments_dev);
    return cudaGetLastError() == cudaSuccess ? CH_OK : CH_ECUDA;
}

extern "C" int ch_stats_hist(const double *series_dev, int nsamples, int ensemble, double lo, double width, int nbins,
                             int *hist_dev, void *stream)
{
    if (!series_dev || !hist_dev || nsamples < 1 || ensemble < 1 || nbins < 1 || nbins > 8192 || !(width > 0) || !std::isfinite(lo))
        return CH_EINVAL;
    k_stats_hist<<<nsamples, 256, (size_t)nbins * sizeof(int), (cudaStream_t)stream>>>(series_dev, ensemble, lo, width, nbins, hist_dev);
    return cudaGetLastError() == cudaSuccess ? CH_OK : CH_ECUDA;
}

extern "C" int ch_stats_fit(const double *moments_dev, int nsamples, double t0, double dt_sample, double t1, double t2,
                            double *out_dev, void *stream)
{
    if (!moments_dev || !out_dev || nsamples < 1 || !(dt_sample > 0) || !(t2 >= t1)) return CH_EINVAL;
    k_stats_fit<<<1, 32, 0, (cudaStream_t)stream>>>(moments_dev, nsamples, t0, dt_sample, t1, t2, out_dev);
    return cudaGetLastError() == cudaSuccess ? CH_OK : CH_ECUDA;
}

// ---- grid-doubling self-convergence error, eq. (A.1) P:672-674 ----
// E[m] = (1 / nc^2) sum_{i,j < nc} | (1/4)(f[2i][2j] + f[2i][2j+1] + f[2i+1][2j] + f[2i+1][2j+1]) - c[i][j] |
// (|Omega| = nc^2 dx_c^2 cancels the cell area).  One CTA per member, fixed summation order.
__global__ void __launch_bounds__(1024) k_grid_doubling_error(const double *__restrict__ fine, const double *__restrict__ coarse,
                                                              int nc, double *__restrict__ out)
{
    __shared__ double red[1024];
    const int m = blockIdx.x, t = threadIdx.x, nf = 2 * nc;
    const double *f = fine + (size_t)m * nf * nf, *c = coarse + (size_t)m * nc * nc;
    double acc = 0.0;
    for (long long p = t; p < (long long)nc * nc; p += 1024) {
        const int i = (int)(p / nc), j = (int)(p - (long long)i * nc);
        const double *q = f + (size_t)(2 * i) * nf + 2 * j;
        acc += fabs(0.25 * ((q[0] + q[1]) + (q[nf] + q[nf + 1])) - c[p]);
    }
    red[t] = acc;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (t < o) red[t] += red[t + o];
        __syncthreads();
    }
    if (t == 0) out[m] = red[0] / ((double)nc * nc);
}

extern "C" int ch_grid_doubling_error(const double *fine_dev, const double *coarse_dev, int ensemble, int n_coarse,
                                      double *out_dev, void *stream)
{
    if (!fine_dev || !coarse_dev || !out_dev || ensemble < 1 || n_coarse < 1 || n_coarse > 16384) return CH_EINVAL;
    k_grid_doubling_error<<<ensemble, 1024, 0, (cudaStream_t)stream>>>(fine_dev, coarse_dev, n_coarse, out_dev);
    return cudaGetLastError() == cudaSuccess ? CH_OK : CH_ECUDA;
}

// ch_fused2d.cuh -- the fused 2D step kernels of libch (sm_100a, fp64).  DESIGN.md section 5.
//
//   k_rhs_sweep_y    r = scale * Lap_h mu(C) computed on the fly while marching down y, fed straight
//                    into the chunked periodic-LU y-sweep; writes w = A_y^-1 r   (16 B per point)
//                    (+ fused F, Fdot, mass partials on sampling steps)
//   k_sweep_x_update C += A_x^-1 w on contiguous lines                           (24 B per point)
//
// The ADI factors are commuting circulants (reading G10), so y-then-x equals the oracle's x-then-y
// to round-off.  The step moves 40 B per grid-point update instead of the 56 B of the three-pass
// structure: r never exists in memory.
#pragma once

#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "ch_kernels.cuh"

namespace cg = cooperative_groups;

#define FUSED_VALID 28        // columns a warp produces: 32 lanes minus a halo of 2 on either side

// ------------------------------------------------------------------------------------
// k_rhs_sweep_y.  One warp = 32 adjacent columns (28 produced + 2 halo lanes each side, x-neighbours
// by warp shuffle), thread (lane, cl) marches down the LC rows of chunk c = crank * CPB + cl.
// A thread-block cluster of CS = P / CPB CTAs covers the whole column strip; the 2-double chunk
// out-states are pushed into every CTA of the cluster through distributed shared memory, so the
// periodic closure (ch_factor.h) sees all P chunks of a line.
// grid.x = CS * strips * ensemble (cluster dim x = CS), block = (32, CPB).
// dynamic smem = 4 * P * 32 doubles: sa_f, sb_f, sa_b, sb_b indexed [chunk][lane].
// ------------------------------------------------------------------------------------
template <int LC, bool DIAG>
__global__ void __launch_bounds__(512) k_rhs_sweep_y(const __grid_constant__ SweepParams prm,
                                                     const double *__restrict__ C, double *__restrict__ w,
                                                     double *__restrict__ partials, int N, double gamma, double scale,
                                                     int strips, int CS, int write)
{
    extern __shared__ double sx[];
    __shared__ double red[16][3];
    cg::cluster_group cluster = cg::this_cluster();
    const int lane = threadIdx.x, cl = threadIdx.y, CPB = blockDim.y, P = prm.P;
    const int crank = blockIdx.x % CS, tile = blockIdx.x / CS;
    const int strip = tile % strips, m = tile / strips;
    const int c = crank * CPB + cl;
    const int X = strip * FUSED_VALID;
    int gx = X - 2 + lane;
    if (gx < 0) gx += N;
    while (gx >= N) gx -= N;
    const bool valid = lane >= 2 && lane < 30 && (X + lane - 2) < N;
    const int y0 = c * LC;
    const double *Cm = C + (size_t)m * N * N + gx;

    // C rows y0-2 .. y0+LC+1 of this thread's column (periodic in y)
    double cv[LC + 4];
#pragma unroll
    for (int j = 0; j < LC + 4; ++j) {
        int y = y0 - 2 + j;
        if (y < 0) y += N;
        if (y >= N) y -= N;
        cv[j] = __ldg(Cm + (size_t)y * N);
    }

    double v[LC];
    double F = 0.0, Fd = 0.0, ms = 0.0;
    const double np = prm.np, nq = prm.nq;
    {
        // mu of row index j (row y0-2+j), j = 1 .. LC+2
        double mu_a, mu_b, mu_c;        // rows j-1, j, j+1 of the rolling window
        double mub_l, mub_r;            // x-neighbours of mu_b
        auto mu_at = [&](int j) {
            const double cc = cv[j];
            const double cl_ = __shfl_up_sync(0xffffffffu, cc, 1), cr_ = __shfl_down_sync(0xffffffffu, cc, 1);
            const double lap = (cl_ + cr_) + (cv[j - 1] + cv[j + 1]) - 4.0 * cc;
            if (DIAG && j >= 2 && j < LC + 2 && valid) {
                const double dx = cr_ - cc, dy = cv[j + 1] - cc, q = cc * cc - 1.0;
                F += 0.25 * q * q + 0.5 * gamma * (dx * dx + dy * dy);
                ms += cc;
            }
            return cc * cc * cc - cc - gamma * lap;
        };
        mu_a = mu_at(1);
        mu_b = mu_at(2);
        mub_l = __shfl_up_sync(0xffffffffu, mu_b, 1);
        mub_r = __shfl_down_sync(0xffffffffu, mu_b, 1);
#pragma unroll
        for (int k = 0; k < LC; ++k) {
            mu_c = mu_at(k + 3);
            const double r = scale * ((mub_l + mub_r) + (mu_a + mu_c) - 4.0 * mu_b);
            if (DIAG && valid) {
                const double dmx = mub_r - mu_b, dmy = mu_c - mu_b;
                Fd -= dmx * dmx + dmy * dmy;
            }
            // forward recurrence from a zero state, inline
            if (k == 0) v[0] = r;
            else if (k == 1) v[1] = fma(np, v[0], r);
            else v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], r));
            mu_a = mu_b; mu_b = mu_c;
            if (k + 1 < LC) {
                mub_l = __shfl_up_sync(0xffffffffu, mu_b, 1);
                mub_r = __shfl_down_sync(0xffffffffu, mu_b, 1);
            }
        }
    }

    if (DIAG) {
        // deterministic block sum: warp shuffle, then warps in fixed order
        F = warp_sum(F); Fd = warp_sum(Fd); ms = warp_sum(ms);
        if (lane == 0) { red[cl][0] = F; red[cl][1] = Fd; red[cl][2] = ms; }
        __syncthreads();
        if (lane == 0 && cl == 0) {
            for (int q = 1; q < CPB; ++q) { F += red[q][0]; Fd += red[q][1]; ms += red[q][2]; }
            double *o = partials + ((size_t)m * (strips * CS) + strip * CS + crank) * 3;
            o[0] = F; o[1] = Fd; o[2] = ms;
        }
    }
    if (DIAG && !write) return;       // diagnostics only (grid-uniform): no sweep, no cluster traffic

    double *sa_f = sx, *sb_f = sx + P * 32, *sa_b = sx + 2 * P * 32, *sb_b = sx + 3 * P * 32;
    cluster.sync();                                     // every CTA of the cluster is resident
    for (int rk = 0; rk < CS; ++rk) {
        double *ra = cluster.map_shared_rank(sa_f, rk), *rb = cluster.map_shared_rank(sb_f, rk);
        ra[c * 32 + lane] = v[LC - 1];
        rb[c * 32 + lane] = v[LC - 2];
    }
    cluster.sync();
    double a, b;
    chunk_state_in<LC>(prm, sa_f + lane, sb_f + lane, c, 32, +1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
    // backward recurrence from a zero state
    v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
    for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
    for (int rk = 0; rk < CS; ++rk) {
        double *ra = cluster.map_shared_rank(sa_b, rk), *rb = cluster.map_shared_rank(sb_b, rk);
        ra[c * 32 + lane] = v[0];
        rb[c * 32 + lane] = v[1];
    }
    cluster.sync();                                     // after this nobody touches remote smem again
    chunk_state_in<LC>(prm, sa_b + lane, sb_b + lane, c, 32, -1, a, b);
    if (valid) {
        double *wm = w + (size_t)m * N * N + (size_t)y0 * N + gx;
#pragma unroll
        for (int k = 0; k < LC; ++k) wm[(size_t)k * N] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
    }
}

// ------------------------------------------------------------------------------------
// k_sweep_x_update: C += A_x^-1 w on contiguous lines.  CTA = LPB consecutive lines; both the w
// lines and the matching C lines are brought in with cp.async (16-byte, L2 only); w lands in the
// 16-byte-granule XOR swizzle of k_sweep_contig so the chunk phase (LDS.128 at a lane stride of
// LC*8 bytes) is bank-conflict free.  block = LPB * P threads,
// dynamic smem = 2 * LPB*N*8 (w, C) + 2*LPB*P*8 (exchange).
// ------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int NLEFT>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(NLEFT) : "memory"); }

template <int LC>
__global__ void k_sweep_x_update(const __grid_constant__ SweepParams prm, const double *__restrict__ w,
                                 double *__restrict__ C, int N, long long total_lines, int LPB)
{
    extern __shared__ double2 sl[];
    const int P = prm.P;
    const int nthreads = blockDim.x, t = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * LPB;
    const int nlines = (int)((total_lines - line0) < LPB ? (total_lines - line0) : LPB);
    const int G = nlines * (N / 2);                           // 16-byte granules held by this CTA
    const double2 *gw = reinterpret_cast<const double2 *>(w + (size_t)line0 * N);
    double2 *gC = reinterpret_cast<double2 *>(C + (size_t)line0 * N);
    double2 *sC = sl + (size_t)LPB * (N / 2);
    double *sa = reinterpret_cast<double *>(sC + (size_t)LPB * (N / 2));
    double *sb = sa + LPB * P;

    for (int g = t; g < G; g += nthreads) cp_async16(&sl[swz<LC>(g)], gw + g);
    cp_async_commit();
    for (int g = t; g < G; g += nthreads) cp_async16(&sC[g], gC + g);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();

    const int l = t / P, c = t - l * P;
    const int gbase = l * (N / 2) + c * (LC / 2);
    double v[LC];
    const bool live = l < nlines;
#pragma unroll
    for (int k = 0; k < LC / 2; ++k) {
        double2 x = live ? sl[swz<LC>(gbase + k)] : make_double2(0.0, 0.0);
        v[2 * k] = x.x; v[2 * k + 1] = x.y;
    }
    chunk_solve<LC>(prm, v, sa + l * P, sb + l * P, c, 1);
    if (live) {
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) sl[swz<LC>(gbase + k)] = make_double2(v[2 * k], v[2 * k + 1]);
    }
    cp_async_wait<0>();
    __syncthreads();
    for (int g = t; g < G; g += nthreads) {
        const double2 x = sl[swz<LC>(g)], cc = sC[g];
        gC[g] = make_double2(cc.x + x.x, cc.y + x.y);
    }
}

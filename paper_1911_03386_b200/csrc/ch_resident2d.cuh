// ch_resident2d.cuh -- member-resident 2D stepping for members that fit one CTA's shared memory (N <= 96).
// SURVEY.md section 8(f) NEXT-3 (ii), reduced to one CTA per member; DESIGN.md section 5c.
//
//   k_step2d_resident   nsteps whole steps  C^{n+1} = C^n + A_x^-1 A_y^-1 dt Lap_h mu(C^n)
//                       (+ the {F, dF/dt, beta, mass} samples that fall inside them)
//
// One CTA owns one member for the whole call: C^n and the work array w live in shared memory, global memory is read
// once at the start and written once at the end (plus 32 B per member and sample), so HBM traffic per update is
// 16 B / nsteps and the bound is the fp64 pipe, not the HBM roofline.  The arithmetic is the
// exact periodic solve of ch_factor.h (chunk_solve<16>: zero-state chunk recurrences + K-term closure), the same as
// the three-pass step's, for any gamma dt.
// Thread (j, c), j = tid % N, c = tid / N, owns 16 points twice:
//   phases 1-3 (column mapping)  column x = j, rows 16 c .. 16 c + 15: mu -> w; r = scale Lap_h mu; y-sweep -> w
//   phase 4    (row mapping)     row y = j, columns 16 c .. 16 c + 15: x-sweep, C += result
// The row pitch N + 1 (odd) makes both mappings bank-conflict free.
#pragma once

#include <cuda_runtime.h>

#include "ch_kernels.cuh"

#define RES_LC 16

struct ResidentParams {
    double gamma, mgam, k1, scale;      // mu = c (c^2 + k1) - gamma (sum of the 4 neighbours), k1 = 4 gamma - 1; scale = dt / c0^2
    double t0, dt;                      // sample time t = t0 + n dt
    long long n0, last_sampled;         // step count at entry; the step count whose sample is already in the series (-1: none)
    int nsteps, stride;                 // stride 0: no series
    int cursor0, Mfull, view_m0;        // series[(cursor * Mfull + view_m0 + m) * 4 + q]
    double *series;
};

static inline size_t resident_smem(int N)
{
    return ((size_t)2 * N * (N + 1) + (size_t)2 * (N / RES_LC) * N) * 8;
}

// grid = members, block = NC * NC / 16, dynamic smem = resident_smem(NC); C is updated in place
template <int NC>
__global__ void __launch_bounds__(NC * NC / RES_LC) k_step2d_resident(const __grid_constant__ SweepParams prm,
                                                                        const __grid_constant__ ResidentParams rp,
                                                                        double *__restrict__ C)
{
    constexpr int N = NC, LC = RES_LC, P = NC / LC, NT = NC * P, PITCH = NC + 1, NW = (NT + 31) / 32;
    extern __shared__ double rsm[];
    __shared__ double red[NW][3];
    double *sC = rsm, *sw = sC + N * PITCH, *sa = sw + N * PITCH, *sb = sa + P * N;
    const int tid = threadIdx.x, j = tid % N, c = tid / N, m = blockIdx.x;
    double *Cm = C + (size_t)m * N * N;
    for (int i = tid; i < N * N; i += NT) sC[(i / N) * PITCH + (i % N)] = Cm[i];
    __syncthreads();

    const double mgam = rp.mgam, k1 = rp.k1, scale = rp.scale;
    const int xm = j == 0 ? N - 1 : j - 1, xp = j == N - 1 ? 0 : j + 1;       // column mapping: x-neighbours of column j
    const int r0 = c * LC;                                                     // first row (column mapping) / column (row mapping)
    const int rm = r0 == 0 ? N - 1 : r0 - 1, rn = r0 + LC == N ? 0 : r0 + LC;  // the rows before / after the chunk
    int cursor = rp.cursor0;

    for (int i = 0;; ++i) {
        const long long n = rp.n0 + i;
        const bool sample = rp.stride > 0 && n % rp.stride == 0 && n != rp.last_sampled;
        const bool last = i == rp.nsteps;
        if (last && !sample) break;
        double F = 0.0, Fd = 0.0, ms = 0.0;
        // ---- phase 1: mu of the chunk's 16 points -> w (rolling window down the column)
        {
            double cu = sC[rm * PITCH + j], cc = sC[r0 * PITCH + j];
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const int row = r0 + k;
                const double cd = sC[(k == LC - 1 ? rn : row + 1) * PITCH + j];
                const double cl = sC[row * PITCH + xm], cr = sC[row * PITCH + xp];
                sw[row * PITCH + j] = fma(mgam, (cl + cr) + (cu + cd), cc * fma(cc, cc, k1));
                if (sample) {
                    const double dx = cr - cc, dy = cd - cc, q = cc * cc - 1.0;
                    F += 0.25 * q * q + 0.5 * rp.gamma * (dx * dx + dy * dy);
                    ms += cc;
                }
                cu = cc; cc = cd;
            }
        }
        __syncthreads();
        // ---- phase 2: r = scale Lap_h mu into registers (+ dF/dt on sampling steps)
        double v[LC];
        {
            double mu_u = sw[rm * PITCH + j], mu_c = sw[r0 * PITCH + j];
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const int row = r0 + k;
                const double mu_d = sw[(k == LC - 1 ? rn : row + 1) * PITCH + j];
                const double ml = sw[row * PITCH + xm], mr = sw[row * PITCH + xp];
                v[k] = scale * fma(-4.0, mu_c, (ml + mr) + (mu_u + mu_d));
                if (sample) {
                    const double dx = mr - mu_c, dy = mu_d - mu_c;
                    Fd -= dx * dx + dy * dy;
                }
                mu_u = mu_c; mu_c = mu_d;
            }
        }
        if (sample) {
            block_sum3<NW>(F, Fd, ms, red);
            if (tid == 0) {
                const double t = rp.t0 + (double)n * rp.dt;
                double *o = rp.series + ((size_t)cursor * rp.Mfull + rp.view_m0 + m) * 4;
                o[0] = F; o[1] = Fd; o[2] = (F == 0.0) ? 0.0 : -t * Fd / F; o[3] = ms;
            }
            ++cursor;
        }
        if (last) break;
        __syncthreads();                     // every mu has been read: w may be overwritten
        // ---- phase 3: y-sweep of the column (exact periodic solve, exchange slots [chunk][column])
        chunk_solve<LC>(prm, v, sa + j, sb + j, c, N);
#pragma unroll
        for (int k = 0; k < LC; ++k) sw[(r0 + k) * PITCH + j] = v[k];
        __syncthreads();
        // ---- phase 4: x-sweep of row j, columns r0 .. r0 + 15, and the update
#pragma unroll
        for (int k = 0; k < LC; ++k) v[k] = sw[j * PITCH + r0 + k];
        chunk_solve<LC>(prm, v, sa + j, sb + j, c, N);
#pragma unroll
        for (int k = 0; k < LC; ++k) sC[j * PITCH + r0 + k] += v[k];
        __syncthreads();
    }
    for (int i = tid; i < N * N; i += NT) Cm[i] = sC[(i / N) * PITCH + (i % N)];
}

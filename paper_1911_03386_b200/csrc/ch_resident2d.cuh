// ch_resident2d.cuh -- member-resident 2D stepping: a member and its work array stay in shared memory for a whole ch_step call.
// SURVEY.md section 8(f) NEXT-3 (ii); DESIGN.md section 5c.  One CTA per member for N <= 96 (first kernel), a thread-block
// cluster per member for N = 128 (2 CTAs) and N = 256 (8 CTAs) (second kernel, end of this file).
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

// Diagnostics terms of one point, with every rounding spelled out (no compiler contraction), so that the kernels of this file, which
// distribute the points over threads differently, add up the same numbers:
//   F term = (c^2 - 1)^2 / 4 + gamma / 2 ((c_right - c)^2 + (c_down - c)^2)     P:34 eq. (4), readings G3, G4
//   dissipation term = (mu_right - mu)^2 + (mu_down - mu)^2                      reading G5
__device__ __forceinline__ double res_F_term(double c, double c_right, double c_down, double gamma)
{
    const double dx = __dsub_rn(c_right, c), dy = __dsub_rn(c_down, c), q = __fma_rn(c, c, -1.0);
    return __fma_rn(__dmul_rn(0.25, q), q, __dmul_rn(__dmul_rn(0.5, gamma), __fma_rn(dx, dx, __dmul_rn(dy, dy))));
}
__device__ __forceinline__ double res_D_term(double mu, double mu_right, double mu_down)
{
    const double dx = __dsub_rn(mu_right, mu), dy = __dsub_rn(mu_down, mu);
    return __fma_rn(dx, dx, __dmul_rn(dy, dy));
}

// The exact periodic solve of chunk_solve (ch_kernels.cuh) with SEPARATE exchange slots for the forward (fa, fb) and the backward
// (ba, bb) pass: two CTA barriers per sweep instead of three.  Slots are [chunk * stride + line].  The first barrier also orders
// everything the CTA did before the sweep against everything after it.
template <int LC>
__device__ __forceinline__ void res_chunk_solve(const SweepParams &prm, double (&v)[LC], double *fa, double *fb, double *ba, double *bb,
                                                int c, int stride, int line)
{
    const double np = prm.np, nq = prm.nq;
    double a, b;
    v[1] = fma(np, v[0], v[1]);
#pragma unroll
    for (int k = 2; k < LC; ++k) v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], v[k]));
    fa[c * stride + line] = v[LC - 1];
    fb[c * stride + line] = v[LC - 2];
    __syncthreads();
    chunk_state_in<LC>(prm, fa + line, fb + line, c, stride, +1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
    v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
    for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
    ba[c * stride + line] = v[0];
    bb[c * stride + line] = v[1];
    __syncthreads();
    chunk_state_in<LC>(prm, ba + line, bb + line, c, stride, -1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
}

static inline size_t resident_smem(int N)
{
    return ((size_t)2 * N * (N + 1) + (size_t)4 * (N / RES_LC) * N) * 8;
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
    double *sC = rsm, *sw = sC + N * PITCH, *sa = sw + N * PITCH, *sb = sa + P * N, *ta = sb + P * N, *tb = ta + P * N;
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
                    F = __dadd_rn(F, res_F_term(cc, cr, cd, rp.gamma));
                    ms = __dadd_rn(ms, cc);
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
                if (sample) Fd = __dsub_rn(Fd, res_D_term(mu_c, mr, mu_d));
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
        // ---- phase 3: y-sweep of the column (exact periodic solve, exchange slots [chunk][column]); its first barrier comes after
        // every mu read above and before any write of w below
        res_chunk_solve<LC>(prm, v, sa, sb, ta, tb, c, N, j);
#pragma unroll
        for (int k = 0; k < LC; ++k) sw[(r0 + k) * PITCH + j] = v[k];
        __syncthreads();
        // ---- phase 4: x-sweep of row j, columns r0 .. r0 + 15, and the update
#pragma unroll
        for (int k = 0; k < LC; ++k) v[k] = sw[j * PITCH + r0 + k];
        res_chunk_solve<LC>(prm, v, sa, sb, ta, tb, c, N, j);
#pragma unroll
        for (int k = 0; k < LC; ++k) sC[j * PITCH + r0 + k] += v[k];
        __syncthreads();
    }
    for (int i = tid; i < N * N; i += NT) Cm[i] = sC[(i / N) * PITCH + (i % N)];
}

// ------------------------------------------------------------------------------------------------------------------
// The same for members that need the shared memory of a thread-block CLUSTER (N = 128: 2 CTAs, N = 256: 8 CTAs; the
// "256^2 member + work array = 1 MiB in an 8-CTA cluster" of SURVEY.md 8(f) NEXT-3 (ii)).  CTA `rank` owns rows
// rank * ROWS .. + ROWS - 1 (ROWS = N / CS) of C and w.  What crosses CTAs, all through distributed shared memory:
//   - the C and mu rows just above / below a slab: every CTA PUSHES its first and last row into its neighbours' halo
//     buffers (C after the update, mu in phase 1), so the stencils read local memory only;
//   - the y-sweep's chunk out-states: written locally, PULLED by the K following (forward) / preceding (backward)
//     chunks' owners after a cluster barrier (separate forward and backward slots: no barrier between the passes);
//   - the per-CTA F, dF/dt, mass partials on sampling steps (pushed to rank 0, summed there in rank order).
// x-lines lie inside a CTA (chunk_solve, CTA barriers).  Four cluster barriers per step (five on sampling steps).
// ------------------------------------------------------------------------------------------------------------------
#include <cooperative_groups.h>

static inline size_t resident_cl_smem(int N, int CS)
{
    const size_t rows = N / CS, nt = (size_t)N * rows / RES_LC;
    return ((size_t)2 * rows * (N + 1) + (size_t)4 * N + 8 * nt) * 8;
}

// grid = members * CS (cluster dimension CS), block = NC * (NC / CS) / 16, dynamic smem = resident_cl_smem(NC, CS)
template <int NC, int CS>
__global__ void __launch_bounds__(NC * (NC / CS) / RES_LC, 1) k_step2d_resident_cl(const __grid_constant__ SweepParams prm,
                                                                                     const __grid_constant__ ResidentParams rp,
                                                                                     double *__restrict__ C)
{
    namespace cg = cooperative_groups;
    constexpr int N = NC, LC = RES_LC, ROWS = NC / CS, PC = ROWS / LC, P = NC / LC, NT = NC * PC, PITCH = NC + 1, NW = NT / 32;
    static_assert(ROWS % LC == 0 && NT % 32 == 0 && NT <= 1024, "slab geometry");
    extern __shared__ double rsm[];
    __shared__ double red[NW][3];
    __shared__ double cpart[CS][3];
    double *sC = rsm, *sw = sC + ROWS * PITCH, *hC = sw + ROWS * PITCH, *hM = hC + 2 * N;      // halos: [0] row above, [1] row below
    double *yFa = hM + 2 * N, *yFb = yFa + NT, *yBa = yFb + NT, *yBb = yBa + NT, *xa = yBb + NT, *xb = xa + NT, *xc = xb + NT, *xd = xc + NT;
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), prevR = (rank + CS - 1) % CS, nextR = (rank + 1) % CS;
    const int tid = threadIdx.x, m = blockIdx.x / CS;
    double *Cm = C + (size_t)m * N * N + (size_t)rank * ROWS * N;
    // column mapping: column x, local chunk c (rows 16 c ..); row mapping: local row y, chunk cx (columns 16 cx ..)
    const int x = tid % N, c = tid / N, r0 = c * LC, g = rank * PC + c;
    const int y = tid % ROWS, cx = tid / ROWS, x0 = cx * LC;
    const int xm = x == 0 ? N - 1 : x - 1, xp = x == N - 1 ? 0 : x + 1;
    double *hC_prev = cluster.map_shared_rank(hC, prevR) + N, *hC_next = cluster.map_shared_rank(hC, nextR);   // my first row is prev's "below"
    double *hM_prev = cluster.map_shared_rank(hM, prevR) + N, *hM_next = cluster.map_shared_rank(hM, nextR);

    for (int i = tid; i < ROWS * N; i += NT) {
        const int yy = i / N, xx = i % N;
        const double v = Cm[i];
        sC[yy * PITCH + xx] = v;
        if (yy == 0) hC_prev[xx] = v;
        if (yy == ROWS - 1) hC_next[xx] = v;
    }
    cluster.sync();

    const double mgam = rp.mgam, k1 = rp.k1, scale = rp.scale, np = prm.np, nq = prm.nq;
    int cursor = rp.cursor0;
    for (int i = 0;; ++i) {
        const long long n = rp.n0 + i;
        const bool sample = rp.stride > 0 && n % rp.stride == 0 && n != rp.last_sampled;
        const bool last = i == rp.nsteps;
        if (last && !sample) break;
        double F = 0.0, Fd = 0.0, ms = 0.0;
        // ---- phase 1: mu -> w, edge rows also into the neighbours' halos
        {
            double cu = c == 0 ? hC[x] : sC[(r0 - 1) * PITCH + x], cc = sC[r0 * PITCH + x];
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const int row = r0 + k;
                const double cd = (k == LC - 1 && c == PC - 1) ? hC[N + x] : sC[(row + 1) * PITCH + x];
                const double cl = sC[row * PITCH + xm], cr = sC[row * PITCH + xp];
                const double mu = fma(mgam, (cl + cr) + (cu + cd), cc * fma(cc, cc, k1));
                sw[row * PITCH + x] = mu;
                if (k == 0 && c == 0) hM_prev[x] = mu;
                if (k == LC - 1 && c == PC - 1) hM_next[x] = mu;
                if (sample) {
                    F = __dadd_rn(F, res_F_term(cc, cr, cd, rp.gamma));
                    ms = __dadd_rn(ms, cc);
                }
                cu = cc; cc = cd;
            }
        }
        cluster.sync();
        // ---- phase 2: r = scale Lap_h mu
        double v[LC];
        {
            double mu_u = c == 0 ? hM[x] : sw[(r0 - 1) * PITCH + x], mu_c = sw[r0 * PITCH + x];
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const int row = r0 + k;
                const double mu_d = (k == LC - 1 && c == PC - 1) ? hM[N + x] : sw[(row + 1) * PITCH + x];
                const double ml = sw[row * PITCH + xm], mr = sw[row * PITCH + xp];
                v[k] = scale * fma(-4.0, mu_c, (ml + mr) + (mu_u + mu_d));
                if (sample) Fd = __dsub_rn(Fd, res_D_term(mu_c, mr, mu_d));
                mu_u = mu_c; mu_c = mu_d;
            }
        }
        if (sample) {
            block_sum3<NW>(F, Fd, ms, red);
            if (tid == 0) {
                double *o = cluster.map_shared_rank(&cpart[0][0], 0) + 3 * rank;
                o[0] = F; o[1] = Fd; o[2] = ms;
            }
            cluster.sync();
            if (rank == 0 && tid == 0) {
                double f = cpart[0][0], fd = cpart[0][1], s = cpart[0][2];
                for (int q = 1; q < CS; ++q) { f += cpart[q][0]; fd += cpart[q][1]; s += cpart[q][2]; }
                const double t = rp.t0 + (double)n * rp.dt;
                double *o = rp.series + ((size_t)cursor * rp.Mfull + rp.view_m0 + m) * 4;
                o[0] = f; o[1] = fd; o[2] = (f == 0.0) ? 0.0 : -t * fd / f; o[3] = s;
            }
            ++cursor;
        }
        if (last) break;
        // ---- phase 3: y-sweep, the line spread over the cluster (its first cluster barrier comes after every mu read above and
        // before any write of w below)
        {
            double a = 0.0, b = 0.0;
            v[1] = fma(np, v[0], v[1]);
#pragma unroll
            for (int k = 2; k < LC; ++k) v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], v[k]));
            yFa[c * N + x] = v[LC - 1];
            yFb[c * N + x] = v[LC - 2];
            cluster.sync();
            int s = g;
            for (int j = 0; j < prm.K; ++j) {
                s = s == 0 ? P - 1 : s - 1;
                const int owner = s / PC, ls = s - owner * PC;
                const double oa = cluster.map_shared_rank(yFa, owner)[ls * N + x], ob = cluster.map_shared_rank(yFb, owner)[ls * N + x];
                const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
                const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
                a = fma(W01.x, oa, fma(W01.y, ob, a));
                b = fma(W23.x, oa, fma(W23.y, ob, b));
            }
#pragma unroll
            for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
            v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
            for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
            yBa[c * N + x] = v[0];
            yBb[c * N + x] = v[1];
            cluster.sync();
            a = 0.0; b = 0.0; s = g;
            for (int j = 0; j < prm.K; ++j) {
                s = s == P - 1 ? 0 : s + 1;
                const int owner = s / PC, ls = s - owner * PC;
                const double oa = cluster.map_shared_rank(yBa, owner)[ls * N + x], ob = cluster.map_shared_rank(yBb, owner)[ls * N + x];
                const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
                const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
                a = fma(W01.x, oa, fma(W01.y, ob, a));
                b = fma(W23.x, oa, fma(W23.y, ob, b));
            }
#pragma unroll
            for (int k = 0; k < LC; ++k) sw[(r0 + k) * PITCH + x] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
        }
        __syncthreads();
        // ---- phase 4: x-sweep of local row y, columns x0 .. x0 + 15, the update, and the new edge rows into the neighbours' halos
#pragma unroll
        for (int k = 0; k < LC; ++k) v[k] = sw[y * PITCH + x0 + k];
        res_chunk_solve<LC>(prm, v, xa, xb, xc, xd, cx, ROWS, y);
#pragma unroll
        for (int k = 0; k < LC; ++k) {
            const double cn = sC[y * PITCH + x0 + k] + v[k];
            sC[y * PITCH + x0 + k] = cn;
            if (y == 0) hC_prev[x0 + k] = cn;
            if (y == ROWS - 1) hC_next[x0 + k] = cn;
        }
        cluster.sync();
    }
    cluster.sync();                          // nobody leaves while a neighbour may still push into its halos
    for (int i = tid; i < ROWS * N; i += NT) Cm[i] = sC[(i / N) * PITCH + (i % N)];
}

// ------------------------------------------------------------------------------------------------------------------
// Second version of the one-CTA kernel, built for the shared-memory data pipe that bounds the first (80 % busy, 106 B
// per update): a thread owns TWO lines in every phase, so that
//   - in the column mapping (columns 2 i, 2 i + 1) one of the two x-neighbours of every point is the thread's own
//     value: 4 LDS per row pair instead of 6, and mu stays in registers between phases 1 and 2 (2 LDS instead of 6);
//   - in the row mapping (rows y, y + N/2) the thread keeps its 2 x 16 values of C in REGISTERS for the whole launch:
//     the update needs no load of C.
// About 57 B per update through the data pipe.  Even and odd columns live in separate planes ([row][N/2 + 1], odd
// pitch), so that both mappings stay bank-conflict free with 8-byte accesses.
// ------------------------------------------------------------------------------------------------------------------
static inline size_t resident2_smem(int N)
{
    return ((size_t)4 * N * (N / 2 + 1) + (size_t)4 * (N / RES_LC) * N) * 8;
}

// res_chunk_solve for two lines at once (shared barriers)
template <int LC>
__device__ __forceinline__ void chunk_solve_pair(const SweepParams &prm, double (&u)[LC], double (&v)[LC], double *fa, double *fb,
                                                 double *ba, double *bb, int c, int stride, int i1, int i2)
{
    const double np = prm.np, nq = prm.nq;
    const int P = prm.P;
    auto state_in = [&](const double *sa, const double *sb, int dir, double &a1, double &b1, double &a2, double &b2) {
        a1 = b1 = a2 = b2 = 0.0;
        int s = c;
        for (int j = 0; j < prm.K; ++j) {
            s -= dir;
            if (s < 0) s += P;
            if (s >= P) s -= P;
            const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
            const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
            const double oa1 = sa[s * stride + i1], ob1 = sb[s * stride + i1], oa2 = sa[s * stride + i2], ob2 = sb[s * stride + i2];
            a1 = fma(W01.x, oa1, fma(W01.y, ob1, a1)); b1 = fma(W23.x, oa1, fma(W23.y, ob1, b1));
            a2 = fma(W01.x, oa2, fma(W01.y, ob2, a2)); b2 = fma(W23.x, oa2, fma(W23.y, ob2, b2));
        }
    };
    double a1, b1, a2, b2;
    u[1] = fma(np, u[0], u[1]); v[1] = fma(np, v[0], v[1]);
#pragma unroll
    for (int k = 2; k < LC; ++k) { u[k] = fma(np, u[k - 1], fma(nq, u[k - 2], u[k])); v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], v[k])); }
    fa[c * stride + i1] = u[LC - 1]; fb[c * stride + i1] = u[LC - 2];
    fa[c * stride + i2] = v[LC - 1]; fb[c * stride + i2] = v[LC - 2];
    __syncthreads();
    state_in(fa, fb, +1, a1, b1, a2, b2);
#pragma unroll
    for (int k = 0; k < LC; ++k) { u[k] = fma(prm.alpha[k], a1, fma(prm.beta[k], b1, u[k])); v[k] = fma(prm.alpha[k], a2, fma(prm.beta[k], b2, v[k])); }
    u[LC - 2] = fma(np, u[LC - 1], u[LC - 2]); v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
    for (int k = LC - 3; k >= 0; --k) { u[k] = fma(np, u[k + 1], fma(nq, u[k + 2], u[k])); v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k])); }
    ba[c * stride + i1] = u[0]; bb[c * stride + i1] = u[1];
    ba[c * stride + i2] = v[0]; bb[c * stride + i2] = v[1];
    __syncthreads();
    state_in(ba, bb, -1, a1, b1, a2, b2);
#pragma unroll
    for (int k = 0; k < LC; ++k) {
        u[k] = fma(prm.alpha[LC - 1 - k], a1, fma(prm.beta[LC - 1 - k], b1, u[k]));
        v[k] = fma(prm.alpha[LC - 1 - k], a2, fma(prm.beta[LC - 1 - k], b2, v[k]));
    }
}

// grid = members, block = (NC / 2) * (NC / 16), dynamic smem = resident2_smem(NC); C is updated in place
template <int NC>
__global__ void __launch_bounds__((NC / 2) * (NC / RES_LC), NC <= 64 ? 3 : 1) k_step2d_resident2(const __grid_constant__ SweepParams prm,
                                                                                                 const __grid_constant__ ResidentParams rp,
                                                                                                 double *__restrict__ C)
{
    constexpr int N = NC, LC = RES_LC, P = NC / LC, H = NC / 2, NT = H * P, PT = H + 1, NG = NT / 16;
    static_assert(NT % 32 == 0, "whole warps");
    extern __shared__ double rsm[];
    __shared__ double red[NG][3];
    double *sCE = rsm, *sCO = sCE + N * PT, *swE = sCO + N * PT, *swO = swE + N * PT, *sa = swO + N * PT, *sb = sa + P * N, *ta = sb + P * N, *tb = ta + P * N;
    const int tid = threadIdx.x, ih = tid % H, c = tid / H, m = blockIdx.x;
    double *Cm = C + (size_t)m * N * N;
    // row mapping: rows y1 = ih and y2 = ih + H, columns 16 c .. 16 c + 15; their C values stay in registers
    const int y1 = ih, y2 = ih + H, x0 = c * LC;
    double C1[LC], C2[LC];
    for (int i = tid; i < N * H; i += NT) {
        const int yy = i / H, ii = i - yy * H;
        const double2 v2 = *reinterpret_cast<const double2 *>(Cm + (size_t)yy * N + 2 * ii);
        sCE[yy * PT + ii] = v2.x; sCO[yy * PT + ii] = v2.y;
    }
#pragma unroll
    for (int k = 0; k < LC; ++k) { C1[k] = Cm[(size_t)y1 * N + x0 + k]; C2[k] = Cm[(size_t)y2 * N + x0 + k]; }
    __syncthreads();

    const double mgam = rp.mgam, k1 = rp.k1, scale = rp.scale;
    // column mapping: columns A = 2 ih (even plane, index ih) and B = 2 ih + 1 (odd plane, index ih), rows r0 .. r0 + 15
    const int im = ih == 0 ? H - 1 : ih - 1, ip = ih == H - 1 ? 0 : ih + 1;      // odd-plane index left of A, even-plane index right of B
    const int r0 = c * LC, rm = r0 == 0 ? N - 1 : r0 - 1, rn = r0 + LC == N ? 0 : r0 + LC;
    int cursor = rp.cursor0;

    for (int i = 0;; ++i) {
        const long long n = rp.n0 + i;
        const bool sample = rp.stride > 0 && n % rp.stride == 0 && n != rp.last_sampled;
        const bool last = i == rp.nsteps;
        if (last && !sample) break;
        // diagnostics are summed per COLUMN and combined in the order of the one-line kernel's shuffle tree (even columns, odd columns,
        // then 32-column groups in order), so a sample does not depend on which of the two kernels the ensemble size selects
        double FA = 0.0, FB = 0.0, FdA = 0.0, FdB = 0.0, msA = 0.0, msB = 0.0;
        double vA[LC], vB[LC];
        // ---- phase 1: mu of the 2 x 16 points -> registers and w
        {
            double cuA = sCE[rm * PT + ih], cuB = sCO[rm * PT + ih], ccA = sCE[r0 * PT + ih], ccB = sCO[r0 * PT + ih];
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const int row = r0 + k, rd = k == LC - 1 ? rn : row + 1;
                const double cdA = sCE[rd * PT + ih], cdB = sCO[rd * PT + ih];
                const double cl = sCO[row * PT + im], cr = sCE[row * PT + ip];
                vA[k] = fma(mgam, (cl + ccB) + (cuA + cdA), ccA * fma(ccA, ccA, k1));
                vB[k] = fma(mgam, (ccA + cr) + (cuB + cdB), ccB * fma(ccB, ccB, k1));
                swE[row * PT + ih] = vA[k]; swO[row * PT + ih] = vB[k];
                if (sample) {
                    FA = __dadd_rn(FA, res_F_term(ccA, ccB, cdA, rp.gamma)); msA = __dadd_rn(msA, ccA);
                    FB = __dadd_rn(FB, res_F_term(ccB, cr, cdB, rp.gamma)); msB = __dadd_rn(msB, ccB);
                }
                cuA = ccA; ccA = cdA; cuB = ccB; ccB = cdB;
            }
        }
        __syncthreads();
        // ---- phase 2: r = scale Lap_h mu, in place (own mu from registers, x-neighbours and the two edge rows from w)
        {
            double upA = swE[rm * PT + ih], upB = swO[rm * PT + ih];
            const double dnA = swE[rn * PT + ih], dnB = swO[rn * PT + ih];
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const int row = r0 + k;
                const double ml = swO[row * PT + im], mr = swE[row * PT + ip];
                const double mA = vA[k], mB = vB[k];
                const double mdA = k == LC - 1 ? dnA : vA[k + 1], mdB = k == LC - 1 ? dnB : vB[k + 1];
                vA[k] = scale * fma(-4.0, mA, (ml + mB) + (upA + mdA));
                vB[k] = scale * fma(-4.0, mB, (mA + mr) + (upB + mdB));
                if (sample) {
                    FdA = __dsub_rn(FdA, res_D_term(mA, mB, mdA));
                    FdB = __dsub_rn(FdB, res_D_term(mB, mr, mdB));
                }
                upA = mA; upB = mB;
            }
        }
        if (sample) {
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) {
                FA += __shfl_down_sync(0xffffffffu, FA, o, 16); FB += __shfl_down_sync(0xffffffffu, FB, o, 16);
                FdA += __shfl_down_sync(0xffffffffu, FdA, o, 16); FdB += __shfl_down_sync(0xffffffffu, FdB, o, 16);
                msA += __shfl_down_sync(0xffffffffu, msA, o, 16); msB += __shfl_down_sync(0xffffffffu, msB, o, 16);
            }
            if ((tid & 15) == 0) { red[tid >> 4][0] = FA + FB; red[tid >> 4][1] = FdA + FdB; red[tid >> 4][2] = msA + msB; }
            __syncthreads();
            if (tid == 0) {
                double F = red[0][0], Fd = red[0][1], ms = red[0][2];
                for (int q = 1; q < NG; ++q) { F += red[q][0]; Fd += red[q][1]; ms += red[q][2]; }
                const double t = rp.t0 + (double)n * rp.dt;
                double *o = rp.series + ((size_t)cursor * rp.Mfull + rp.view_m0 + m) * 4;
                o[0] = F; o[1] = Fd; o[2] = (F == 0.0) ? 0.0 : -t * Fd / F; o[3] = ms;
            }
            ++cursor;
        }
        if (last) break;
        // ---- phase 3: y-sweep of the two columns (first barrier: after every mu read above, before any write of w below)
        chunk_solve_pair<LC>(prm, vA, vB, sa, sb, ta, tb, c, N, 2 * ih, 2 * ih + 1);
#pragma unroll
        for (int k = 0; k < LC; ++k) { swE[(r0 + k) * PT + ih] = vA[k]; swO[(r0 + k) * PT + ih] = vB[k]; }
        __syncthreads();
        // ---- phase 4: x-sweep of rows y1, y2 (columns x0 .. x0 + 15) and the update of the register copy and of the planes
#pragma unroll
        for (int k = 0; k < LC; ++k) {
            const double *pl = (k & 1) ? swO : swE;
            vA[k] = pl[y1 * PT + (x0 + k) / 2]; vB[k] = pl[y2 * PT + (x0 + k) / 2];
        }
        chunk_solve_pair<LC>(prm, vA, vB, sa, sb, ta, tb, c, N, y1, y2);
#pragma unroll
        for (int k = 0; k < LC; ++k) {
            double *pl = (k & 1) ? sCO : sCE;
            C1[k] += vA[k]; C2[k] += vB[k];
            pl[y1 * PT + (x0 + k) / 2] = C1[k]; pl[y2 * PT + (x0 + k) / 2] = C2[k];
        }
        __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < LC; ++k) { Cm[(size_t)y1 * N + x0 + k] = C1[k]; Cm[(size_t)y2 * N + x0 + k] = C2[k]; }
}

// ch_kernels.cuh -- device kernels of libch (sm_100a, fp64).  See DESIGN.md for the
// data layout, the per-kernel byte model and the roofline each kernel is bound by.
//
//   k_rhs2d / k_rhs3d    r = scale * Lap_h mu(C)   (+ fused F, Fdot, mass partials)   include/ch.h
//   k_finish             deterministic finish of the partials -> {F, Fdot, beta, mass} P:64
//   k_sweep_contig       w := A_x^-1 w, lines contiguous (x), chunked periodic LU      ch_factor.h
//   k_sweep_strided      w := A_d^-1 w, lines at a stride (y, z), optional C += w
//   k_sweep_generic      any N >= 8: one thread per line, four passes through global memory
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "ch_factor.h"

struct SweepParams {
    double np, nq;              // recurrence  z_i = b_i + np z_{i-1} + nq z_{i-2}
    double oscale;              // output scale (1/c0 for the stand-alone ch_sweep, unused in the step)
    double alpha[CH_MAX_LC];
    double beta[CH_MAX_LC];
    const double *W;            // device [K][4]
    int K, P;
    // log-depth closure for contiguous lines (chunks of a line in consecutive lanes): used when scan != 0
    double Mp[5][4];            // M^(2^k)
    double Wc[4];               // (I - M^P)^-1
    int scan;                   // 0, or log2 P (P a power of two, 2 <= P <= 32)
    int rev;                    // 3D sweeps: walk the blocks from the last to the first (L2 reuse between consecutive kernels)
    int scan2;                  // 0, or W = P / 32 in 2..4: two-level scan (warp scan + W warp aggregates)
    const double *S2;           // device: Mlane[32][4] then WG[4][4] (ch_factor.h)
};

// 16-byte asynchronous global -> shared copy (L2 only), and its group fences
__device__ __forceinline__ void ck_cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void ck_cp_async_wait_all()
{
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
}

// Programmatic dependent launch: a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start while the
// kernel before it on the stream is still running; pdl_wait() blocks until that kernel has completed and its writes are visible
// (it must come before the first access to anything the predecessor touches), pdl_trigger() lets the NEXT kernel's CTAs be
// scheduled as soon as every CTA of this one has started.  Both are no-ops in a kernel launched the plain way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }

// ------------------------------------------------------------------------------------
// reductions
// ------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Sum three values over a block of NW warps in a fixed order; result valid in thread 0.
template <int NW>
__device__ __forceinline__ void block_sum3(double &a, double &b, double &c, double (*red)[3])
{
    a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { red[wid][0] = a; red[wid][1] = b; red[wid][2] = c; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = red[0][0]; b = red[0][1]; c = red[0][2];
#pragma unroll
        for (int w = 1; w < NW; ++w) { a += red[w][0]; b += red[w][1]; c += red[w][2]; }
    }
}

template <bool POW2>
__device__ __forceinline__ int wrapi(int i, int N)
{
    if (POW2) return i & (N - 1);
    i %= N;
    return i < 0 ? i + N : i;
}

// ------------------------------------------------------------------------------------
// RHS, 2D.  Tile TX x TY per CTA, C staged with halo 2, mu with halo 1 in shared memory.
// grid = (tiles_x * tiles_y, ensemble), block = 256.
// ------------------------------------------------------------------------------------
#define RHS2_TX 64
#define RHS2_TY 32

template <bool DIAG, bool WRITE, bool POW2>
__global__ void __launch_bounds__(256) k_rhs2d(const double *__restrict__ C, double *__restrict__ r,
                                               double *__restrict__ partials, int N, double gamma, double scale,
                                               int tiles_x)
{
    constexpr int TX = RHS2_TX, TY = RHS2_TY, CW = TX + 4, MW = TX + 2;
    __shared__ double sC[(TY + 4) * CW];
    __shared__ double sMu[(TY + 2) * MW];
    __shared__ double red[8][3];
    const int tid = threadIdx.x;
    const int tile = blockIdx.x, m = blockIdx.y;
    const int x0 = (tile % tiles_x) * TX, y0 = (tile / tiles_x) * TY;
    const double *Cm = C + (size_t)m * N * N;

    for (int i = tid; i < (TY + 4) * CW; i += 256) {
        const int ly = i / CW, lx = i - ly * CW;
        const int gy = wrapi<POW2>(y0 + ly - 2, N), gx = wrapi<POW2>(x0 + lx - 2, N);
        sC[i] = Cm[(size_t)gy * N + gx];
    }
    __syncthreads();
    for (int i = tid; i < (TY + 2) * MW; i += 256) {
        const int ly = i / MW, lx = i - ly * MW;
        const double *p = sC + (ly + 1) * CW + lx + 1;
        const double c = p[0];
        const double lap = (p[1] + p[-1]) + (p[CW] + p[-CW]) - 4.0 * c;
        sMu[i] = c * c * c - c - gamma * lap;
    }
    __syncthreads();
    double F = 0.0, Fd = 0.0, ms = 0.0;
    for (int i = tid; i < TY * TX; i += 256) {
        const int ly = i / TX, lx = i - ly * TX;
        const int gy = y0 + ly, gx = x0 + lx;
        if (gy < N && gx < N) {
            const double *q = sMu + (ly + 1) * MW + lx + 1;
            const double mu = q[0];
            if (WRITE) {
                const double lap = (q[1] + q[-1]) + (q[MW] + q[-MW]) - 4.0 * mu;
                r[(size_t)m * N * N + (size_t)gy * N + gx] = scale * lap;
            }
            if (DIAG) {
                const double *p = sC + (ly + 2) * CW + lx + 2;
                const double c = p[0], dcx = p[1] - c, dcy = p[CW] - c;
                const double dmx = q[1] - mu, dmy = q[MW] - mu;
                const double w = c * c - 1.0;
                F += 0.25 * w * w + 0.5 * gamma * (dcx * dcx + dcy * dcy);
                Fd -= dmx * dmx + dmy * dmy;
                ms += c;
            }
        }
    }
    if (DIAG) {
        block_sum3<8>(F, Fd, ms, red);
        if (tid == 0) {
            double *o = partials + ((size_t)m * gridDim.x + tile) * 3;
            o[0] = F; o[1] = Fd; o[2] = ms;
        }
    }
}

// ------------------------------------------------------------------------------------
// RHS, 3D.  Tile 32 x 8 x 8 per CTA, dynamic shared memory.
// grid = (tiles_x * tiles_y * tiles_z, ensemble), block = 256.
// ------------------------------------------------------------------------------------
#define RHS3_TX 32
#define RHS3_TY 8
#define RHS3_TZ 8
#define RHS3_SMEM (((RHS3_TZ + 4) * (RHS3_TY + 4) * (RHS3_TX + 4) + (RHS3_TZ + 2) * (RHS3_TY + 2) * (RHS3_TX + 2)) * 8)

template <bool DIAG, bool WRITE, bool POW2>
__global__ void __launch_bounds__(256) k_rhs3d(const double *__restrict__ C, double *__restrict__ r,
                                               double *__restrict__ partials, int N, double gamma, double scale,
                                               int tiles_x, int tiles_y)
{
    constexpr int TX = RHS3_TX, TY = RHS3_TY, TZ = RHS3_TZ;
    constexpr int CW = TX + 4, CH = TY + 4, CD = TZ + 4, MW = TX + 2, MH = TY + 2, MD = TZ + 2;
    extern __shared__ double smem3[];
    double *sC = smem3, *sMu = smem3 + CD * CH * CW;
    __shared__ double red[8][3];
    const int tid = threadIdx.x;
    const int tile = blockIdx.x, m = blockIdx.y;
    const int x0 = (tile % tiles_x) * TX, y0 = ((tile / tiles_x) % tiles_y) * TY, z0 = (tile / (tiles_x * tiles_y)) * TZ;
    const size_t n2 = (size_t)N * N;
    const double *Cm = C + (size_t)m * n2 * N;

    for (int i = tid; i < CD * CH * CW; i += 256) {
        const int lz = i / (CH * CW), rem = i - lz * (CH * CW), ly = rem / CW, lx = rem - ly * CW;
        const int gz = wrapi<POW2>(z0 + lz - 2, N), gy = wrapi<POW2>(y0 + ly - 2, N), gx = wrapi<POW2>(x0 + lx - 2, N);
        sC[i] = Cm[gz * n2 + (size_t)gy * N + gx];
    }
    __syncthreads();
    for (int i = tid; i < MD * MH * MW; i += 256) {
        const int lz = i / (MH * MW), rem = i - lz * (MH * MW), ly = rem / MW, lx = rem - ly * MW;
        const double *p = sC + ((lz + 1) * CH + ly + 1) * CW + lx + 1;
        const double c = p[0];
        const double lap = (p[1] + p[-1]) + (p[CW] + p[-CW]) + (p[CH * CW] + p[-CH * CW]) - 6.0 * c;
        sMu[i] = c * c * c - c - gamma * lap;
    }
    __syncthreads();
    double F = 0.0, Fd = 0.0, ms = 0.0;
    for (int i = tid; i < TZ * TY * TX; i += 256) {
        const int lz = i / (TY * TX), rem = i - lz * (TY * TX), ly = rem / TX, lx = rem - ly * TX;
        const int gz = z0 + lz, gy = y0 + ly, gx = x0 + lx;
        if (gz < N && gy < N && gx < N) {
            const double *q = sMu + ((lz + 1) * MH + ly + 1) * MW + lx + 1;
            const double mu = q[0];
            if (WRITE) {
                const double lap = (q[1] + q[-1]) + (q[MW] + q[-MW]) + (q[MH * MW] + q[-MH * MW]) - 6.0 * mu;
                r[(size_t)m * n2 * N + gz * n2 + (size_t)gy * N + gx] = scale * lap;
            }
            if (DIAG) {
                const double *p = sC + ((lz + 2) * CH + ly + 2) * CW + lx + 2;
                const double c = p[0], dcx = p[1] - c, dcy = p[CW] - c, dcz = p[CH * CW] - c;
                const double dmx = q[1] - mu, dmy = q[MW] - mu, dmz = q[MH * MW] - mu;
                const double w = c * c - 1.0;
                F += 0.25 * w * w + 0.5 * gamma * (dcx * dcx + dcy * dcy + dcz * dcz);
                Fd -= dmx * dmx + dmy * dmy + dmz * dmz;
                ms += c;
            }
        }
    }
    if (DIAG) {
        block_sum3<8>(F, Fd, ms, red);
        if (tid == 0) {
            double *o = partials + ((size_t)m * gridDim.x + tile) * 3;
            o[0] = F; o[1] = Fd; o[2] = ms;
        }
    }
}

// ------------------------------------------------------------------------------------
// Finish: out[m] = {F, Fdot, beta, mass}, beta = -t Fdot / F (0 if F == 0).
// grid = ensemble, block = 128; fixed summation order (bitwise reproducible).
// ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_finish(const double *__restrict__ partials, int nparts,
                                                double *__restrict__ out, double t)
{
    __shared__ double red[4][3];
    const int m = blockIdx.x;
    const double *p = partials + (size_t)m * nparts * 3;
    double F = 0.0, Fd = 0.0, ms = 0.0;
    for (int i = threadIdx.x; i < nparts; i += 128) { F += p[3 * i]; Fd += p[3 * i + 1]; ms += p[3 * i + 2]; }
    block_sum3<4>(F, Fd, ms, red);
    if (threadIdx.x == 0) {
        double *o = out + (size_t)m * 4;
        o[0] = F; o[1] = Fd; o[2] = (F == 0.0) ? 0.0 : -t * Fd / F; o[3] = ms;
    }
}

// ------------------------------------------------------------------------------------
// Chunked periodic-LU line solve on LC points held in registers (see ch_factor.h).
// Every thread owns chunk `c` of one line; sa/sb are the shared exchange slots of that
// line, indexed [chunk * cstride].  All threads of the CTA must call this together.
// ------------------------------------------------------------------------------------
template <int LC>
__device__ __forceinline__ void chunk_state_in(const SweepParams &prm, const double *sa, const double *sb,
                                               int c, int cstride, int dir, double &a, double &b)
{
    a = 0.0; b = 0.0;
    const int P = prm.P;
    int s = c;
    for (int j = 0; j < prm.K; ++j) {
        s -= dir;
        if (s < 0) s += P;
        if (s >= P) s -= P;
        const double oa = sa[s * cstride], ob = sb[s * cstride];
        const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
        const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
        a = fma(W01.x, oa, fma(W01.y, ob, a));
        b = fma(W23.x, oa, fma(W23.y, ob, b));
    }
}

// Log-depth closure: the P chunks of a line sit in P consecutive lanes (P a power of two <= 32).
// T_0(c) = out(c); T_{k+1}(c) = T_k(c) + M^(2^k) T_k(c -+ 2^k) with cyclic lane indices, so that
// T(c) = sum_{j<P} M^j out(c -+ j); state entering chunk c = (I - M^P)^-1 T(c -+ 1).  No shared memory.
__device__ __forceinline__ void chunk_state_scan(const SweepParams &prm, double oa, double ob, int c, int dir,
                                                 double &a, double &b)
{
    const int P = prm.P;
    // every thread of the CTA gets here together; the last warp may be partial: the mask comes from the launch
    // geometry, not from whichever threads happen to be converged (independent thread scheduling)
    const unsigned nthr = blockDim.x * blockDim.y * blockDim.z;
    const unsigned ltid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const unsigned left = nthr - (ltid & ~31u);
    const unsigned full = left >= 32u ? 0xffffffffu : ((1u << left) - 1u);
    double ta = oa, tb = ob;
    for (int k = 0; k < prm.scan; ++k) {
        const int src = (c - dir * (1 << k)) & (P - 1);
        const double ua = __shfl_sync(full, ta, src, P), ub = __shfl_sync(full, tb, src, P);
        ta = fma(prm.Mp[k][0], ua, fma(prm.Mp[k][1], ub, ta));
        tb = fma(prm.Mp[k][2], ua, fma(prm.Mp[k][3], ub, tb));
    }
    const int src = (c - dir) & (P - 1);
    const double ua = __shfl_sync(full, ta, src, P), ub = __shfl_sync(full, tb, src, P);
    a = fma(prm.Wc[0], ua, prm.Wc[1] * ub);
    b = fma(prm.Wc[2], ua, prm.Wc[3] * ub);
}

// Two-level form for P = 32 W chunks per line (W = 2..4 warps per line): a non-cyclic scan inside each warp,
// the W warp aggregates combined through shared memory (agg: 2 W doubles per line and direction), and the
// state entering the warp propagated to its lanes with the M^lane table.  One __syncthreads.
__device__ __forceinline__ void chunk_state_scan2(const SweepParams &prm, double oa, double ob, int c, int dir,
                                                  double *agg, double &a, double &b)
{
    const int W = prm.scan2, lane = c & 31, wl = c >> 5;
    const int pos = dir > 0 ? lane : 31 - lane;                   // chunks between this one and the warp's entry side
    double ta = oa, tb = ob;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int d = 1 << k;
        const int src = dir > 0 ? lane - d : lane + d;
        const double ua = __shfl_sync(0xffffffffu, ta, src & 31), ub = __shfl_sync(0xffffffffu, tb, src & 31);
        if (pos >= d) {
            ta = fma(prm.Mp[k][0], ua, fma(prm.Mp[k][1], ub, ta));
            tb = fma(prm.Mp[k][2], ua, fma(prm.Mp[k][3], ub, tb));
        }
    }
    if (pos == 31) { agg[2 * wl] = ta; agg[2 * wl + 1] = tb; }     // the warp's aggregate out-state
    // exclusive part: what the chunks before this one (inside the warp) contribute
    const int prev = dir > 0 ? lane - 1 : lane + 1;
    double ea = __shfl_sync(0xffffffffu, ta, prev & 31), eb = __shfl_sync(0xffffffffu, tb, prev & 31);
    if (pos == 0) { ea = 0.0; eb = 0.0; }
    __syncthreads();
    double sa_ = 0.0, sb_ = 0.0;
    int w = wl;
    for (int q = 0; q < W; ++q) {
        w -= dir;
        if (w < 0) w += W;
        if (w >= W) w -= W;
        const double ga = agg[2 * w], gb = agg[2 * w + 1];
        const double *G = prm.S2 + 128 + 4 * q;
        sa_ = fma(__ldg(G), ga, fma(__ldg(G + 1), gb, sa_));
        sb_ = fma(__ldg(G + 2), ga, fma(__ldg(G + 3), gb, sb_));
    }
    const double2 m01 = __ldg(reinterpret_cast<const double2 *>(prm.S2) + 2 * pos);
    const double2 m23 = __ldg(reinterpret_cast<const double2 *>(prm.S2) + 2 * pos + 1);
    a = fma(m01.x, sa_, fma(m01.y, sb_, ea));
    b = fma(m23.x, sa_, fma(m23.y, sb_, eb));
}

// Same solve as chunk_solve for kernels whose thread index is line * P + chunk (contiguous lines):
// closure by warp-shuffle scan, no shared memory and no barrier.
template <int LC>
__device__ __forceinline__ void chunk_solve_scan(const SweepParams &prm, double (&v)[LC], int c, double *agg)
{
    const double np = prm.np, nq = prm.nq;
    double a, b;
    v[1] = fma(np, v[0], v[1]);
#pragma unroll
    for (int k = 2; k < LC; ++k) v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], v[k]));
    if (prm.scan2) chunk_state_scan2(prm, v[LC - 1], v[LC - 2], c, +1, agg, a, b);
    else chunk_state_scan(prm, v[LC - 1], v[LC - 2], c, +1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
    v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
    for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
    if (prm.scan2) chunk_state_scan2(prm, v[0], v[1], c, -1, agg + 8, a, b);
    else chunk_state_scan(prm, v[0], v[1], c, -1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
}

template <int LC>
__device__ __forceinline__ void chunk_solve(const SweepParams &prm, double (&v)[LC], double *sa, double *sb,
                                            int c, int cstride)
{
    const double np = prm.np, nq = prm.nq;
    double a, b;
    // forward: z_k = b_k + np z_{k-1} + nq z_{k-2}, zero state
    v[1] = fma(np, v[0], v[1]);
#pragma unroll
    for (int k = 2; k < LC; ++k) v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], v[k]));
    sa[c * cstride] = v[LC - 1];
    sb[c * cstride] = v[LC - 2];
    __syncthreads();
    chunk_state_in<LC>(prm, sa, sb, c, cstride, +1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
    __syncthreads();
    // backward: x_k = z_k + np x_{k+1} + nq x_{k+2}, zero state
    v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
    for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
    sa[c * cstride] = v[0];
    sb[c * cstride] = v[1];
    __syncthreads();
    chunk_state_in<LC>(prm, sa, sb, c, cstride, -1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
}

// ------------------------------------------------------------------------------------
// Strided sweep (y, z): thread (tx, c) owns chunk c of the line through inner position tx.
// block = (COLS, P); grid.x = inner_blocks * n_outer.  A warp reads COLS*8 contiguous bytes
// per line point.  UPDATE: C += w instead of writing w (last sweep of the step).
// ------------------------------------------------------------------------------------
template <int LC, bool UPDATE, bool SCALE>
__global__ void __launch_bounds__(512) k_sweep_strided(const __grid_constant__ SweepParams prm, double *__restrict__ w,
                                double *__restrict__ C, size_t outer_stride, size_t line_stride, int inner_blocks)
{
    extern __shared__ double sx[];
    pdl_trigger();
    pdl_wait();
    const int COLS = blockDim.x, P = blockDim.y;
    const int tx = threadIdx.x, c = threadIdx.y;
    const unsigned bid = prm.rev ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    const int ib = bid % inner_blocks, o = bid / inner_blocks;
    const size_t base = (size_t)o * outer_stride + (size_t)c * LC * line_stride + (size_t)ib * COLS + tx;
    double *sa = sx + tx, *sb = sx + P * COLS + tx;

    double v[LC];
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = w[base + k * line_stride];
    chunk_solve<LC>(prm, v, sa, sb, c, COLS);
    if (UPDATE) {
#pragma unroll
        for (int k0 = 0; k0 < LC; k0 += 8) {
            double cc[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) cc[k] = C[base + (k0 + k) * line_stride];
#pragma unroll
            for (int k = 0; k < 8; ++k) C[base + (k0 + k) * line_stride] = cc[k] + v[k0 + k];
        }
    } else {
#pragma unroll
        for (int k = 0; k < LC; ++k) w[base + k * line_stride] = SCALE ? v[k] * prm.oscale : v[k];
    }
}

// ------------------------------------------------------------------------------------
// Contiguous sweep (x): CTA = LPB consecutive lines, thread (l, c) = chunk c of line l.
// Lines are staged through shared memory with a 16-byte-granule XOR swizzle so that both
// the coalesced global phase and the chunk phase (LDS.128, lane stride LC*8 bytes) are
// bank-conflict free.  block = LPB * P threads, dynamic smem = LPB*N*8 + 2*LPB*P*8.
// ------------------------------------------------------------------------------------
template <int LC>
__device__ __forceinline__ int swz(int g)
{
    constexpr int SH = LC == 8 ? 2 : (LC == 16 ? 3 : 4);
    return g ^ ((g >> SH) & 7);
}

template <int LC, bool SCALE>
__global__ void k_sweep_contig(const __grid_constant__ SweepParams prm, double *__restrict__ w, int N,
                               long long total_lines, int LPB)
{
    extern __shared__ double2 sl[];
    const int P = prm.P;
    const int nthreads = blockDim.x, t = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * LPB;
    const int nlines = (int)((total_lines - line0) < LPB ? (total_lines - line0) : LPB);
    const int G = nlines * (N / 2);                           // granules held by this CTA
    double2 *g2 = reinterpret_cast<double2 *>(w + (size_t)line0 * N);
    double *sa = reinterpret_cast<double *>(sl + (size_t)LPB * (N / 2));
    double *sb = sa + LPB * P;

    for (int g = t; g < G; g += nthreads) ck_cp_async16(&sl[swz<LC>(g)], g2 + g);
    ck_cp_async_wait_all();
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
    if (prm.scan || prm.scan2) chunk_solve_scan<LC>(prm, v, c, sa + l * P);      // (sa, sb are contiguous: 2 P doubles per line pair)
    else chunk_solve<LC>(prm, v, sa + l * P, sb + l * P, c, 1);
    if (live) {
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) {
            double2 x;
            x.x = SCALE ? v[2 * k] * prm.oscale : v[2 * k];
            x.y = SCALE ? v[2 * k + 1] * prm.oscale : v[2 * k + 1];
            sl[swz<LC>(gbase + k)] = x;
        }
    }
    __syncthreads();
    for (int g = t; g < G; g += nthreads) g2[g] = sl[swz<LC>(g)];
}

// ------------------------------------------------------------------------------------
// Generic sweep, any N >= 8: one thread per line, the cyclic recurrences run through
// global memory (four passes).  Correct for every N; slow.  lines are enumerated as
// (outer, inner): address = outer * outer_stride + inner * inner_stride + i * line_stride.
// ------------------------------------------------------------------------------------
template <bool UPDATE>
__global__ void __launch_bounds__(128) k_sweep_generic(double np, double nq, double W0, double W1, double W2, double W3,
                                                       double oscale, double *__restrict__ w, double *__restrict__ C,
                                                       int N, long long n_lines, int n_inner, size_t outer_stride,
                                                       size_t inner_stride, size_t line_stride)
{
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= n_lines) return;
    const size_t base = (size_t)(id / n_inner) * outer_stride + (size_t)(id % n_inner) * inner_stride;
    double *x = w + base;
    double z1 = 0.0, z2 = 0.0;
    for (int i = 0; i < N; ++i) {
        const double z = fma(np, z1, fma(nq, z2, x[i * line_stride]));
        x[i * line_stride] = z; z2 = z1; z1 = z;
    }
    double u1 = W0 * z1 + W1 * z2, u2 = W2 * z1 + W3 * z2;
    for (int i = 0; i < N; ++i) {
        const double u = np * u1 + nq * u2;
        x[i * line_stride] += u; u2 = u1; u1 = u;
    }
    z1 = 0.0; z2 = 0.0;
    for (int i = N - 1; i >= 0; --i) {
        const double z = fma(np, z1, fma(nq, z2, x[i * line_stride]));
        x[i * line_stride] = z; z2 = z1; z1 = z;
    }
    u1 = W0 * z1 + W1 * z2; u2 = W2 * z1 + W3 * z2;
    for (int i = N - 1; i >= 0; --i) {
        const double u = np * u1 + nq * u2;
        const double val = (x[i * line_stride] + u) * oscale;
        if (UPDATE) C[base + i * line_stride] += val; else x[i * line_stride] = val;
        u2 = u1; u1 = u;
    }
}

// ------------------------------------------------------------------------------------
// Parallel cyclic reduction (PCR) x-sweep, N a power of two: the alternative BASELINE.json's north
// star asks to be measured against the periodic-LU sweep for N >= 1024.
// Level l (stride s = 2^l): multiplying A_s = a S^2s + b S^s + 1 + b S^-s + a S^-2s by
// a S^2s - b S^s + 1 - b S^-s + a S^-2s gives a system of the same shape at stride 2s with
// a' = a^2, b' = 2a - b^2, c' = 1 + 2a^2 - 2b^2 (divided through by c'); indices are taken mod N,
// so after log2 N levels the matrix is (1 + 2a + 2b) I.  The host stops early once |a|, |b| < 1e-22.
// One CTA per line, the line double buffered in shared memory: block = 256, smem = 2 * N * 8.
// ------------------------------------------------------------------------------------
#define CH_PCR_MAX_LEVELS 13
struct PcrParams {
    double A[CH_PCR_MAX_LEVELS], B[CH_PCR_MAX_LEVELS], Cc[CH_PCR_MAX_LEVELS];   // a / c', -b / c', 1 / c' per level
    double final_scale;                                                      // 1 / (1 + 2a + 2b) of the last level, times oscale
    int levels;
};

__global__ void __launch_bounds__(256) k_sweep_pcr_x(const __grid_constant__ PcrParams prm, double *__restrict__ w, int N)
{
    extern __shared__ double sp[];
    double *cur = sp, *nxt = sp + N;
    double *g = w + (size_t)blockIdx.x * N;
    const int mask = N - 1;
    for (int i = threadIdx.x; i < N; i += 256) cur[i] = g[i];
    __syncthreads();
    int s = 1;
    for (int l = 0; l < prm.levels; ++l, s <<= 1) {
        const double a = prm.A[l], b = prm.B[l], c = prm.Cc[l];
        for (int i = threadIdx.x; i < N; i += 256) {
            const double f2 = cur[(i + 2 * s) & mask] + cur[(i - 2 * s) & mask];
            const double f1 = cur[(i + s) & mask] + cur[(i - s) & mask];
            nxt[i] = fma(a, f2, fma(b, f1, c * cur[i]));
        }
        __syncthreads();
        double *t = cur; cur = nxt; nxt = t;
    }
    for (int i = threadIdx.x; i < N; i += 256) g[i] = cur[i] * prm.final_scale;
}

// ------------------------------------------------------------------------------------
// 3D: x- and y-sweep of one z-plane in one pass (N = 64, 128: the plane, N^2 * 8 B <= 128 KB, lives in
// shared memory), w := A_y^-1 A_x^-1 w.  Saves one full read + write of the field: 16 B per update
// instead of 32 B.  CTA = one plane of one member, NC * NC / 16 threads.
//   x phase: thread (row, chunk of 16 contiguous points), plane in the swizzled granule layout of
//            k_sweep_contig, closure by width-P shuffle scan (the P = NC / 16 chunks of a row sit in
//            consecutive lanes): no barrier;
//   y phase: thread (column, chunk of 16 rows) reads its column from shared memory (a warp reads 32
//            consecutive doubles of a row), chunk_solve with the exchange through shared memory,
//            results written straight to global memory (coalesced rows).
// dynamic smem = NC * NC * 8 + 2 * (NC / 16) * NC * 8.  prm.scan must be log2(NC / 16) with Mp, Wc filled.
// ------------------------------------------------------------------------------------
template <int NC>
__global__ void __launch_bounds__(NC * NC / 16, NC == 64 ? 3 : 1) k_sweep_xy_plane(const __grid_constant__ SweepParams prm, double *__restrict__ w)
{
    pdl_trigger();
    pdl_wait();
    constexpr int LC = 16, P = NC / LC, NT = NC * NC / LC, G = NC * NC / 2;
    extern __shared__ double2 sl[];
    double *sx = reinterpret_cast<double *>(sl + G);
    const int t = threadIdx.x;
    const unsigned bid = prm.rev ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    double2 *g2 = reinterpret_cast<double2 *>(w + (size_t)bid * NC * NC);
#pragma unroll
    for (int k = 0; k < G / NT; ++k) ck_cp_async16(&sl[swz<LC>(k * NT + t)], g2 + k * NT + t);
    ck_cp_async_wait_all();
    __syncthreads();
    double v[LC];
    {   // x phase
        const int l = t / P, c = t - l * P, gbase = l * (NC / 2) + c * (LC / 2);
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) { const double2 x = sl[swz<LC>(gbase + k)]; v[2 * k] = x.x; v[2 * k + 1] = x.y; }
        chunk_solve_scan<LC>(prm, v, c, nullptr);
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) sl[swz<LC>(gbase + k)] = make_double2(v[2 * k], v[2 * k + 1]);
    }
    __syncthreads();
    {   // y phase
        const int x = t % NC, c = t / NC;
        const double *sd = reinterpret_cast<const double *>(sl);
#pragma unroll
        for (int k = 0; k < LC; ++k) {
            const int g = (c * LC + k) * (NC / 2) + (x >> 1);
            v[k] = sd[2 * swz<LC>(g) + (x & 1)];
        }
        chunk_solve<LC>(prm, v, sx + x, sx + P * NC + x, c, NC);      // the strided closure sums K terms through shared memory
        double *o = w + (size_t)bid * NC * NC + (size_t)c * LC * NC + x;
#pragma unroll
        for (int k = 0; k < LC; ++k) o[k * NC] = v[k];
    }
}

// ------------------------------------------------------------------------------------
// k_sweep_xy_pair: the plane kernel for N = 128 on a thread-block cluster of 2 CTAs, each holding half
// the plane (64 rows x 128 columns, 64 KB), so that two CTAs of different planes share an SM and one
// loads while the other computes.  x phase as in k_sweep_xy_plane (rows are complete in a CTA).
// y phase: thread (column, local chunk of 16 rows); every chunk state is written to the local exchange
// arrays AND to the peer CTA's (distributed shared memory), one cluster barrier per direction, then the
// usual K-term closure over all 8 chunks.  grid = 2 * planes, cluster (2,1,1), block 512,
// dynamic smem = 64 KB + 2 directions * 2 * 8 * 128 * 8 B.
// ------------------------------------------------------------------------------------
__device__ __forceinline__ void pair_store_remote(double *local, unsigned peer, double v)
{
    unsigned ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(ra) : "r"((unsigned)__cvta_generic_to_shared(local)), "r"(peer));
    asm volatile("st.shared::cluster.f64 [%0], %1;\n" ::"r"(ra), "d"(v) : "memory");
}
__device__ __forceinline__ void pair_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

__global__ void __launch_bounds__(512, 2) k_sweep_xy_pair(const __grid_constant__ SweepParams prm, double *__restrict__ w)
{
    constexpr int NC = 128, LC = 16, P = NC / LC, HR = NC / 2, NT = 512, G = HR * NC / 2;     // G granules per half plane
    extern __shared__ double2 sl[];
    double *sxf = reinterpret_cast<double *>(sl + G), *sxb = sxf + 2 * P * NC;                // [a|b][chunk][column] per direction
    const int t = threadIdx.x;
    unsigned rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(rank));
    const unsigned peer = rank ^ 1u;
    pdl_trigger();
    pdl_wait();
    const size_t plane = prm.rev ? (gridDim.x >> 1) - 1 - (blockIdx.x >> 1) : (blockIdx.x >> 1);
    double *wp = w + plane * NC * NC + (size_t)rank * HR * NC;
    double2 *g2 = reinterpret_cast<double2 *>(wp);
#pragma unroll
    for (int k = 0; k < G / NT; ++k) ck_cp_async16(&sl[swz<LC>(k * NT + t)], g2 + k * NT + t);
    ck_cp_async_wait_all();
    __syncthreads();
    double v[LC];
    {   // x phase: rows of this half
        const int l = t / P, c = t - l * P, gbase = l * (NC / 2) + c * (LC / 2);
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) { const double2 x = sl[swz<LC>(gbase + k)]; v[2 * k] = x.x; v[2 * k + 1] = x.y; }
        chunk_solve_scan<LC>(prm, v, c, nullptr);
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) sl[swz<LC>(gbase + k)] = make_double2(v[2 * k], v[2 * k + 1]);
    }
    __syncthreads();
    {   // y phase: column x, local chunk cl (global chunk c = rank * 4 + cl)
        const int x = t % NC, cl = t / NC, c = (int)rank * (P / 2) + cl;
        const double *sd = reinterpret_cast<const double *>(sl);
#pragma unroll
        for (int k = 0; k < LC; ++k) {
            const int g = (cl * LC + k) * (NC / 2) + (x >> 1);
            v[k] = sd[2 * swz<LC>(g) + (x & 1)];
        }
        const double np = prm.np, nq = prm.nq;
        double a, b;
        v[1] = fma(np, v[0], v[1]);
#pragma unroll
        for (int k = 2; k < LC; ++k) v[k] = fma(np, v[k - 1], fma(nq, v[k - 2], v[k]));
        double *fa = sxf + c * NC + x, *fb = sxf + (P + c) * NC + x;
        *fa = v[LC - 1]; *fb = v[LC - 2];
        pair_store_remote(fa, peer, v[LC - 1]); pair_store_remote(fb, peer, v[LC - 2]);
        pair_sync();
        chunk_state_in<LC>(prm, sxf + x, sxf + P * NC + x, c, NC, +1, a, b);
#pragma unroll
        for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
        v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
        for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
        double *ba = sxb + c * NC + x, *bb = sxb + (P + c) * NC + x;
        *ba = v[0]; *bb = v[1];
        pair_store_remote(ba, peer, v[0]); pair_store_remote(bb, peer, v[1]);
        pair_sync();
        chunk_state_in<LC>(prm, sxb + x, sxb + P * NC + x, c, NC, -1, a, b);
        double *o = wp + (size_t)cl * LC * NC + x;
#pragma unroll
        for (int k = 0; k < LC; ++k) o[k * NC] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
    }
    pair_sync();      // the peer may still be storing into this CTA's exchange arrays until both have passed the last read
}

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
#include "ch_line2d.cuh"

namespace cg = cooperative_groups;

#define FUSED_VALID 28        // columns a warp produces: 32 lanes minus a halo of 2 on either side

// ------------------------------------------------------------------------------------
// Distributed-shared-memory plumbing (sm_90+ PTX): cluster barrier split into arrive / wait,
// mbarrier with a transaction count, and st.async -- a remote shared-memory store that signals
// the receiving CTA's mbarrier when it lands, so the chunk-state exchange needs no fences.
// ------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_init(unsigned mbar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned mbar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(mbar), "r"(parity) : "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ unsigned map_rank(unsigned local, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_async_2f64(unsigned remote_addr, double a, double b, unsigned remote_mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];\n" ::"r"(remote_addr),
                 "l"(__double_as_longlong(a)), "l"(__double_as_longlong(b)), "r"(remote_mbar)
                 : "memory");
}

// read-only global load as volatile asm: keeps the compiler from sinking it below later code, so a
// thread's loads are all in flight together
__device__ __forceinline__ double ldg_nc_f64(const double *p)
{
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];\n" : "=d"(v) : "l"(p));
    return v;
}

// state entering chunk c from the K chunks before it (dir = +1) or after it (dir = -1); slots hold
// (a, b) pairs indexed [chunk][lane]
__device__ __forceinline__ void chunk_state_in2(const SweepParams &prm, const double2 *slots, int c, int lane, int dir,
                                                double &a, double &b)
{
    a = 0.0; b = 0.0;
    const int P = prm.P;
    int s = c;
    for (int j = 0; j < prm.K; ++j) {
        s -= dir;
        if (s < 0) s += P;
        if (s >= P) s -= P;
        const double2 o = slots[s * 32 + lane];
        const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
        const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
        a = fma(W01.x, o.x, fma(W01.y, o.y, a));
        b = fma(W23.x, o.x, fma(W23.y, o.y, b));
    }
}

// ------------------------------------------------------------------------------------
// k_rhs_sweep_y.  One warp = 32 adjacent columns (28 produced + 2 halo lanes each side, x-neighbours
// by warp shuffle), thread (lane, cl) marches down the LC rows of chunk c = crank * CPB + cl.
// A thread-block cluster of CS = P / CPB CTAs covers the whole column strip; the 2-double chunk
// out-states are pushed into every CTA of the cluster with st.async (distributed shared memory +
// mbarrier transaction counts), so the periodic closure (ch_factor.h) sees all P chunks of a line.
// grid.x = CS * strips * ensemble (cluster dim x = CS), block = (32, CPB).
// dynamic smem = 2 * P * 32 double2: forward and backward exchange slots, indexed [chunk][lane].
// ------------------------------------------------------------------------------------
template <int LC, bool DIAG>
__global__ void __launch_bounds__(512) k_rhs_sweep_y(const __grid_constant__ SweepParams prm,
                                                     const double *__restrict__ C, double *__restrict__ w,
                                                     double *__restrict__ partials, int N, double gamma, double scale,
                                                     int strips, int CS, int write)
{
    extern __shared__ double2 sx2[];
    __shared__ double red[16][3];
    __shared__ __align__(8) unsigned long long mbar[2];
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
    const size_t n2 = (size_t)N * N;

    const unsigned mb_f = smem_u32(&mbar[0]), mb_b = smem_u32(&mbar[1]);
    if (lane == 0 && cl == 0) {
        mbar_init(mb_f, 1);
        mbar_init(mb_b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        mbar_expect_tx(mb_f, (unsigned)P * 32 * 16);
        mbar_expect_tx(mb_b, (unsigned)P * 32 * 16);
    }
    cluster_arrive();        // waited on just before the first remote store, long after every CTA has started

    // C rows y0-2 .. y0+LC+1 of this thread's column; only the two halo rows on either end can wrap
    double cv[LC + 4];
    {
        const double *p = C + (size_t)m * n2 + gx + (ptrdiff_t)(y0 - 2) * N;
        const double *plo = (c == 0) ? p + n2 : p;
        const double *phi = (c == P - 1) ? p - n2 : p;
#pragma unroll
        for (int j = 0; j < LC + 4; ++j) {
            const double *q = (j < 2) ? plo : ((j >= LC + 2) ? phi : p);
            cv[j] = ldg_nc_f64(q + (ptrdiff_t)j * N);
        }
    }
    asm volatile("" ::: "memory");    // all LC+4 loads are issued before any arithmetic (keeps them in flight together)

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
    cluster_wait();                   // every CTA of the cluster has initialised its mbarriers
    if (DIAG && !write) return;       // diagnostics only (grid-uniform): no sweep, no cluster traffic

    double2 *sf = sx2, *sb = sx2 + P * 32;
    const unsigned slot_f = smem_u32(sf + c * 32 + lane), slot_b = smem_u32(sb + c * 32 + lane);
    for (int rk = 0; rk < CS; ++rk) st_async_2f64(map_rank(slot_f, rk), v[LC - 1], v[LC - 2], map_rank(mb_f, rk));
    mbar_wait(mb_f, 0);
    double a, b;
    chunk_state_in2(prm, sf, c, lane, +1, a, b);
#pragma unroll
    for (int k = 0; k < LC; ++k) v[k] = fma(prm.alpha[k], a, fma(prm.beta[k], b, v[k]));
    // backward recurrence from a zero state
    v[LC - 2] = fma(np, v[LC - 1], v[LC - 2]);
#pragma unroll
    for (int k = LC - 3; k >= 0; --k) v[k] = fma(np, v[k + 1], fma(nq, v[k + 2], v[k]));
    for (int rk = 0; rk < CS; ++rk) st_async_2f64(map_rank(slot_b, rk), v[0], v[1], map_rank(mb_b, rk));
    mbar_wait(mb_b, 0);               // all P chunk states have landed here: nobody writes this CTA again
    chunk_state_in2(prm, sb, c, lane, -1, a, b);
    if (valid) {
        double *wm = w + (size_t)m * n2 + (size_t)y0 * N + gx;
#pragma unroll
        for (int k = 0; k < LC; ++k) wm[(ptrdiff_t)k * N] = fma(prm.alpha[LC - 1 - k], a, fma(prm.beta[LC - 1 - k], b, v[k]));
    }
}

// ------------------------------------------------------------------------------------
// k_sweep_x_update: C += oscale * A_x^-1 w on contiguous lines.  CTA = LPB consecutive lines; both the w
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
    // lines are taken from the END of the ensemble backwards: the fused RHS + y-sweep kernel before this one walks the
    // members upwards, so its last ~100 MB of w and C are still in L2 -- and the C this kernel writes last (the first
    // members) is what the next step's first tiles read
    const long long line0 = (long long)(gridDim.x - 1 - blockIdx.x) * LPB;
    const int nlines = (int)((total_lines - line0) < LPB ? (total_lines - line0) : LPB);
    const int G = nlines * (N / 2);                           // 16-byte granules held by this CTA
    const double2 *gw = reinterpret_cast<const double2 *>(w + (size_t)line0 * N);
    double2 *gC = reinterpret_cast<double2 *>(C + (size_t)line0 * N);
    double2 *sC = sl + (size_t)LPB * (N / 2);
    double *sa = reinterpret_cast<double *>(sC + (size_t)LPB * (N / 2));
    double *sb = sa + LPB * P;

    const unsigned long long pol = l2_evict_first_policy();     // w is dead after this read; C is overwritten below
    pdl_trigger();
    pdl_wait();
    for (int g = t; g < G; g += nthreads) line_cp_async16_hint(&sl[swz<LC>(g)], gw + g, pol);
    cp_async_commit();
    for (int g = t; g < G; g += nthreads) line_cp_async16_hint(&sC[g], gC + g, pol);
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
    if (prm.scan || prm.scan2) chunk_solve_scan<LC>(prm, v, c, sa + l * P);
    else chunk_solve<LC>(prm, v, sa + l * P, sb + l * P, c, 1);
    if (live) {
#pragma unroll
        for (int k = 0; k < LC / 2; ++k) sl[swz<LC>(gbase + k)] = make_double2(v[2 * k], v[2 * k + 1]);
    }
    cp_async_wait<0>();
    __syncthreads();
    for (int g = t; g < G; g += nthreads) {
        const double2 x = sl[swz<LC>(g)], cc = sC[g];
        gC[g] = make_double2(fma(prm.oscale, x.x, cc.x), fma(prm.oscale, x.y, cc.y));
    }
}

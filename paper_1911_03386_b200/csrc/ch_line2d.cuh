// ch_line2d.cuh -- fused RHS + y-sweep of the 2D step for lines that fit one CTA (N <= 512).
// DESIGN.md section 5.
//
//   k_rhs_sweep_y_line   w = A_y^-1 (scale * Lap_h mu(C))                     P:29-30, include/ch.h
//                        (+ fused F, Fdot, mass partials on sampling steps)
//
// A persistent CTA owns whole columns: tile = one column strip (28 produced columns + a halo of 2 on
// either side) x all N rows of one member.  Thread (li, c) -- half-warp lane li, chunk c of 16 rows --
// carries two adjacent columns.  It stages its own 20 C rows (16 + halo 2 + 2) with cp.async, forms mu
// and r = Lap_h mu in a rolling register window (x-neighbours in the lane or by half-warp shuffle) and
// feeds r straight into the chunked periodic-LU recurrence of ch_factor.h, whose 2-double chunk states
// are exchanged through shared memory (the whole line is in this CTA: no cluster, no global traffic).
// r and the forward/backward intermediates never exist in memory: 16 B per grid-point update.
// A thread reads back only the rows it staged itself, so its staging slots are free as soon as its
// forward pass is done: the loads of the CTA's NEXT tile are issued there and fly during the closure,
// the backward pass and the write-out of the current tile.
#pragma once

#include <cuda_runtime.h>

#include "ch_kernels.cuh"

#define LINE_LC 16
#define LINE_VALID 28         // columns a half-warp produces: 16 lanes x 2 columns minus a halo of 2 on either side
#define LINE_MAX_P 32         // chunks per line: 16 * P threads per CTA

struct LineParams {
    double np, nq;                  // recurrence  z_i = b_i + np z_{i-1} + nq z_{i-2}
    double gamma, mgam, k1, scale;  // mu = c (c^2 + k1) - gamma * (sum of the 4 neighbours), k1 = 4 gamma - 1
    double alpha[LINE_LC], beta[LINE_LC];
    const double *W;                // device [K][4] (ch_factor.h)
    int K, P, N, strips, ntiles, write;
};

__device__ __forceinline__ void line_cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void line_cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void line_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

__device__ __forceinline__ double hshfl_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1, 16); }
__device__ __forceinline__ double hshfl_down(double v) { return __shfl_down_sync(0xffffffffu, v, 1, 16); }

// states entering chunk c (both columns of the lane) from the K chunks before it (dir = +1) or after
// it (dir = -1); slots are [column A|B][chunk][16 lanes] pairs (value next to the boundary, one further in)
__device__ __forceinline__ void line_state_in(const LineParams &prm, const double2 *slots, int c, int li, int dir,
                                              double &aA, double &bA, double &aB, double &bB)
{
    aA = bA = aB = bB = 0.0;
    const int P = prm.P;
    int s = c;
    for (int j = 0; j < prm.K; ++j) {
        s -= dir;
        if (s < 0) s += P;
        if (s >= P) s -= P;
        const double2 oA = slots[s * 16 + li], oB = slots[(P + s) * 16 + li];
        const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
        const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
        aA = fma(W01.x, oA.x, fma(W01.y, oA.y, aA));
        bA = fma(W23.x, oA.x, fma(W23.y, oA.y, bA));
        aB = fma(W01.x, oB.x, fma(W01.y, oB.y, aB));
        bB = fma(W23.x, oB.x, fma(W23.y, oB.y, bB));
    }
}

// grid = min(ntiles, resident CTAs), block = 16 * P threads (P even),
// dynamic smem = 20 * blockDim.x * 16 (staging) + 2 * 2 * P * 16 * 16 (forward, backward exchange slots).
template <bool DIAG>
__global__ void __launch_bounds__(16 * LINE_MAX_P, 1) k_rhs_sweep_y_line(const __grid_constant__ LineParams prm,
                                                                        const double *__restrict__ C, double *__restrict__ w,
                                                                        double *__restrict__ partials)
{
    constexpr int LC = LINE_LC, NR = LC + 4;
    extern __shared__ double2 sm2[];
    __shared__ double red[16][3];
    const int tid = threadIdx.x, NT = blockDim.x, li = tid & 15, c = tid >> 4;
    const int N = prm.N, P = prm.P, strips = prm.strips, ntiles = prm.ntiles;
    const int y0 = c * LC;
    const size_t n2 = (size_t)N * N;
    const bool lane_ok = li >= 1 && li < 15;

    double2 *stage = sm2 + tid;                                   // row j of this thread: stage[j * NT]
    double2 *slotF = sm2 + (size_t)NR * NT, *slotB = slotF + 2 * P * 16;

    // C rows y0-2 .. y0+LC+1 of this thread's column pair; only the two halo rows on either end can wrap
    auto issue = [&](int tile) {
        const int strip = tile % strips, m = tile / strips;
        int gx = strip * LINE_VALID - 2 + 2 * li;
        if (gx < 0) gx += N;
        while (gx >= N) gx -= N;
        const double *p = C + (size_t)m * n2 + gx + (ptrdiff_t)(y0 - 2) * N;
        const double *plo = (c == 0) ? p + n2 : p;
        const double *phi = (c == P - 1) ? p - n2 : p;
#pragma unroll
        for (int j = 0; j < NR; ++j) {
            const double *q = (j < 2) ? plo : ((j >= LC + 2) ? phi : p);
            line_cp_async16(stage + j * NT, q + (ptrdiff_t)j * N);
        }
        line_cp_async_commit();
    };

    int tile = blockIdx.x;
    if (tile < ntiles) issue(tile);
    const double np = prm.np, nq = prm.nq, mgam = prm.mgam, k1 = prm.k1;

    for (; tile < ntiles; tile += gridDim.x) {
        const int strip = tile % strips, m = tile / strips;
        const int X = strip * LINE_VALID;
        const bool valid = lane_ok && (X + 2 * (li - 1)) < N;
        line_cp_async_wait_all();          // a thread reads back only what it staged itself: no barrier needed

        double vA[LC], vB[LC];
        double F = 0.0, Fd = 0.0, ms = 0.0;
        {
            // mu of the row whose C is `cc`, with the rows above (cu) and below (cd)
            auto mu_row = [&](const double2 cu, const double2 cc, const double2 cd, bool own) {
                const double lft = hshfl_up(cc.y), rgt = hshfl_down(cc.x);
                const double sA = (lft + cc.y) + (cu.x + cd.x), sB = (cc.x + rgt) + (cu.y + cd.y);
                if (DIAG && own && valid) {
                    const double dxA = cc.y - cc.x, dyA = cd.x - cc.x, qA = cc.x * cc.x - 1.0;
                    const double dxB = rgt - cc.y, dyB = cd.y - cc.y, qB = cc.y * cc.y - 1.0;
                    F += (0.25 * qA * qA + 0.5 * prm.gamma * (dxA * dxA + dyA * dyA))
                       + (0.25 * qB * qB + 0.5 * prm.gamma * (dxB * dxB + dyB * dyB));
                    ms += cc.x + cc.y;
                }
                double2 mu;
                mu.x = fma(mgam, sA, cc.x * fma(cc.x, cc.x, k1));
                mu.y = fma(mgam, sB, cc.y * fma(cc.y, cc.y, k1));
                return mu;
            };
            double2 c0 = stage[0], c1 = stage[NT], c2 = stage[2 * NT], c3 = stage[3 * NT];
            double2 mu_a = mu_row(c0, c1, c2, false);
            double2 mu_b = mu_row(c1, c2, c3, true);
            double ml = hshfl_up(mu_b.y), mr = hshfl_down(mu_b.x);
            c0 = c2; c1 = c3;                                        // rows j-1, j of the next mu row
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const double2 cn = stage[(k + 4) * NT];
                const double2 mu_c = mu_row(c0, c1, cn, k + 1 < LC);   // staged row k + 3
                const double rA = fma(-4.0, mu_b.x, (ml + mu_b.y) + (mu_a.x + mu_c.x));
                const double rB = fma(-4.0, mu_b.y, (mu_b.x + mr) + (mu_a.y + mu_c.y));
                if (DIAG && valid) {
                    const double dxA = mu_b.y - mu_b.x, dyA = mu_c.x - mu_b.x, dxB = mr - mu_b.y, dyB = mu_c.y - mu_b.y;
                    Fd -= (dxA * dxA + dyA * dyA) + (dxB * dxB + dyB * dyB);
                }
                // forward recurrence from a zero state, inline
                if (k == 0) { vA[0] = rA; vB[0] = rB; }
                else if (k == 1) { vA[1] = fma(np, vA[0], rA); vB[1] = fma(np, vB[0], rB); }
                else { vA[k] = fma(np, vA[k - 1], fma(nq, vA[k - 2], rA)); vB[k] = fma(np, vB[k - 1], fma(nq, vB[k - 2], rB)); }
                mu_a = mu_b; mu_b = mu_c; c0 = c1; c1 = cn;
                if (k + 1 < LC) { ml = hshfl_up(mu_b.y); mr = hshfl_down(mu_b.x); }
            }
        }
        // this thread's staging slots are consumed: put the next tile's loads in flight
        if (tile + (int)gridDim.x < ntiles) issue(tile + gridDim.x);

        if (DIAG) {
            // deterministic block sum: warp shuffle, then warps in fixed order
            F = warp_sum(F); Fd = warp_sum(Fd); ms = warp_sum(ms);
            if ((tid & 31) == 0) { red[tid >> 5][0] = F; red[tid >> 5][1] = Fd; red[tid >> 5][2] = ms; }
            __syncthreads();
            if (tid == 0) {
                for (int q = 1; q < (NT >> 5); ++q) { F += red[q][0]; Fd += red[q][1]; ms += red[q][2]; }
                double *o = partials + ((size_t)m * strips + strip) * 3;
                o[0] = F; o[1] = Fd; o[2] = ms;
            }
            __syncthreads();
            if (!prm.write) continue;         // diagnostics only (grid-uniform): no sweep
        }

        // ---- forward closure
        slotF[c * 16 + li] = make_double2(vA[LC - 1], vA[LC - 2]);
        slotF[(P + c) * 16 + li] = make_double2(vB[LC - 1], vB[LC - 2]);
        __syncthreads();
        {
            double aA, bA, aB, bB;
            line_state_in(prm, slotF, c, li, +1, aA, bA, aB, bB);
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                vA[k] = fma(prm.alpha[k], aA, fma(prm.beta[k], bA, vA[k]));
                vB[k] = fma(prm.alpha[k], aB, fma(prm.beta[k], bB, vB[k]));
            }
        }
        // ---- backward recurrence from a zero state
        vA[LC - 2] = fma(np, vA[LC - 1], vA[LC - 2]);
        vB[LC - 2] = fma(np, vB[LC - 1], vB[LC - 2]);
#pragma unroll
        for (int k = LC - 3; k >= 0; --k) {
            vA[k] = fma(np, vA[k + 1], fma(nq, vA[k + 2], vA[k]));
            vB[k] = fma(np, vB[k + 1], fma(nq, vB[k + 2], vB[k]));
        }
        slotB[c * 16 + li] = make_double2(vA[0], vA[1]);
        slotB[(P + c) * 16 + li] = make_double2(vB[0], vB[1]);
        __syncthreads();      // also orders this tile's slotF reads before the next tile's slotF writes
        {
            double aA, bA, aB, bB;
            line_state_in(prm, slotB, c, li, -1, aA, bA, aB, bB);
            if (valid) {
                const double sc = prm.scale;
                int gx = X - 2 + 2 * li;                            // valid lanes: 0 <= gx < N
                double2 *wm = reinterpret_cast<double2 *>(w + (size_t)m * n2 + (size_t)y0 * N + gx);
#pragma unroll
                for (int k = 0; k < LC; ++k) {
                    double2 o;
                    o.x = sc * fma(prm.alpha[LC - 1 - k], aA, fma(prm.beta[LC - 1 - k], bA, vA[k]));
                    o.y = sc * fma(prm.alpha[LC - 1 - k], aB, fma(prm.beta[LC - 1 - k], bB, vB[k]));
                    wm[(size_t)k * (N / 2)] = o;
                }
            }
        }
        // slotB reads of this tile are ordered before the next tile's slotB writes by the next
        // tile's first __syncthreads
    }
}

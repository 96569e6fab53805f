// ch_rhs3d_stream.cuh -- explicit RHS of the 3D step as a z-marching ("2.5-D") kernel, N in {64, 96, 128}.
// DESIGN.md section 5.
//
//   k_rhs3d_stream   r = scale * Lap_h mu(C),  mu = C^3 - C - gamma Lap_h C  (7-point Laplacians)    P:29-30, include/ch.h
//                    (+ fused F, Fdot, mass partials on sampling steps)
//
// A CTA owns an x-strip of 28 produced columns (+2 halo columns either side) x ALL N rows of y (so y
// wraps inside the CTA: no y halo) and marches over a range of R3_ZR z-planes.  Thread = half-warp lane
// li (two adjacent columns) x 4 consecutive rows.  Per plane step it keeps C(z), C(z+1) and mu(z-1),
// mu(z) of its 8 points in registers, takes C(z+2) from a thread-private cp.async ring (3 planes deep,
// so loads fly for two plane periods and need no barrier), forms mu(z+1) and then r(z):
//   x-neighbours  : inside the lane or one half-warp shuffle away
//   y-neighbours  : inside the thread, or -- for its first and last row -- the edge rows that the
//                   half-warps above and below published to shared memory one step earlier
//   z-neighbours  : registers (rolling window)
// One __syncthreads per plane step (the published rows are double buffered by step parity).
// HBM traffic: C read once (+ halo columns and the 4 warm-up planes of a range, served by L2),
// r written once: 16 B per grid-point update.
#pragma once

#include <cuda_runtime.h>

#include "ch_kernels.cuh"
#include "ch_line2d.cuh"      // cp.async and half-warp shuffle helpers

#define R3_VALID 28           // columns a half-warp produces
#define R3_RY 4               // rows per thread
#define R3_ZR 16              // planes per work unit (+4 warm-up planes read, +2 mu planes recomputed)

struct Rhs3Params {
    double gamma, mgam, k1, scale;      // mu = c (c^2 + k1) - gamma * (sum of the 6 neighbours), k1 = 6 gamma - 1
    int nunits, write, rev;             // rev: take the units from the last to the first
};

static inline size_t rhs3_stream_smem(int N)
{
    const size_t NT = (size_t)N * 4, NHW = (size_t)N / R3_RY;
    return 3 * R3_RY * NT * 16 + 2 * (2 * 2 * NHW * 16 * 16);
}

// grid = min(nunits, resident CTAs), block = 4 * NC threads, dynamic smem = rhs3_stream_smem(NC).
// unit = (member, strip, z-range); partials[(m * strips + strip) * (NC / R3_ZR) + zr][3].
template <int NC, bool DIAG>
__global__ void __launch_bounds__(4 * NC, 1) k_rhs3d_stream(const __grid_constant__ Rhs3Params prm,
                                                            const double *__restrict__ C, double *__restrict__ r,
                                                            double *__restrict__ partials)
{
    constexpr int N = NC, NT = 4 * NC, RY = R3_RY, NHW = NC / RY, ZR = R3_ZR, NZ = NC / ZR;
    constexpr int strips = (NC + R3_VALID - 1) / R3_VALID;
    constexpr size_t n2 = (size_t)N * N, n3 = n2 * N;
    static_assert((ZR + 2) % 6 == 0, "the plane loop is unrolled by 6 (ring of 3 slots x 2 parities)");
    extern __shared__ double2 sm2[];
    __shared__ double red[16][3];
    const int tid = threadIdx.x, li = tid & 15, hw = tid >> 4;
    const int hwm = (hw + NHW - 1) % NHW, hwp = (hw + 1) % NHW;
    pdl_trigger();
    pdl_wait();
    double2 *stage = sm2 + tid;                                   // plane slot p, row j: stage[(p * RY + j) * NT]
    // published edge rows: [parity][top|bottom][half-warp][lane]
    double2 *exC = sm2 + (size_t)3 * RY * NT, *exM = exC + 2 * 2 * NHW * 16;
    const double mgam = prm.mgam, k1 = prm.k1, scale = prm.scale;

    for (int u = blockIdx.x; u < prm.nunits; u += gridDim.x) {
        const int unit = prm.rev ? prm.nunits - 1 - u : u;
        const int zr = unit % NZ, t = unit / NZ, strip = t % strips, m = t / strips;
        const int X = strip * R3_VALID, z0 = zr * ZR;
        int gx = X - 2 + 2 * li;
        if (gx < 0) gx += N;
        if (gx >= N) gx -= N;
        const bool valid = li >= 1 && li < 15 && (X + 2 * (li - 1)) < N;
        const double *pC = C + (size_t)m * n3 + (size_t)(hw * RY) * N + gx;
        auto load_plane = [&](int zz, int slot) {
            const double *p = pC + (size_t)((zz + N) % N) * n2;          // N is a compile-time constant
#pragma unroll
            for (int j = 0; j < RY; ++j) line_cp_async16(stage + (slot * RY + j) * NT, p + j * N);
            line_cp_async_commit();
        };
        load_plane(z0 - 2, 0);
        load_plane(z0 - 1, 1);
        load_plane(z0, 2);
        asm volatile("cp.async.wait_group 1;\n" ::: "memory");
        double2 Cm[RY], C0[RY], mum[RY], mu0[RY];
#pragma unroll
        for (int j = 0; j < RY; ++j) {
            Cm[j] = stage[j * NT];
            C0[j] = stage[(RY + j) * NT];
            mum[j] = make_double2(0.0, 0.0);
            mu0[j] = make_double2(0.0, 0.0);
        }
        // plane z0-1 is "C(z+1)" of step 0: its edge rows go where step 0 looks for them (parity 1)
        exC[((1 * 2 + 0) * NHW + hw) * 16 + li] = C0[0];
        exC[((1 * 2 + 1) * NHW + hw) * 16 + li] = C0[RY - 1];
        exM[((1 * 2 + 0) * NHW + hw) * 16 + li] = make_double2(0.0, 0.0);
        exM[((1 * 2 + 1) * NHW + hw) * 16 + li] = make_double2(0.0, 0.0);
        __syncthreads();
        double F = 0.0, Fd = 0.0, ms = 0.0;
        double *pr = r + (size_t)m * n3 + (size_t)(hw * RY) * N + (X - 2 + 2 * li);

        for (int s0 = 0; s0 < ZR + 2; s0 += 6) {
#pragma unroll
            for (int ss = 0; ss < 6; ++ss) {
                const int s = s0 + ss;                 // step s: z = z0 - 2 + s; mu(z+1) and r(z)
                const int par = ss & 1, slot = (ss + 2) % 3;
                // next plane into the slot that was consumed two steps ago; plane z+2 has then landed
                if (s + 1 < ZR + 2) load_plane(z0 + s + 1, ss % 3);
                else line_cp_async_commit();
                asm volatile("cp.async.wait_group 1;\n" ::: "memory");
                double2 Cp[RY], mup[RY];
#pragma unroll
                for (int j = 0; j < RY; ++j) Cp[j] = stage[(slot * RY + j) * NT];
                const double2 Cup = exC[(((par ^ 1) * 2 + 1) * NHW + hwm) * 16 + li];
                const double2 Cdn = exC[(((par ^ 1) * 2 + 0) * NHW + hwp) * 16 + li];
                const double2 Mup = exM[(((par ^ 1) * 2 + 1) * NHW + hwm) * 16 + li];
                const double2 Mdn = exM[(((par ^ 1) * 2 + 0) * NHW + hwp) * 16 + li];
                // ---- mu(z+1) from C(z+1) = C0, its in-plane neighbours, C(z) = Cm and C(z+2) = Cp
#pragma unroll
                for (int j = 0; j < RY; ++j) {
                    const double2 up = j == 0 ? Cup : C0[j - 1], dn = j == RY - 1 ? Cdn : C0[j + 1], cc = C0[j];
                    const double lft = hshfl_up(cc.y), rgt = hshfl_down(cc.x);
                    const double sA = ((lft + cc.y) + (up.x + dn.x)) + (Cm[j].x + Cp[j].x);
                    const double sB = ((cc.x + rgt) + (up.y + dn.y)) + (Cm[j].y + Cp[j].y);
                    mup[j].x = fma(mgam, sA, cc.x * fma(cc.x, cc.x, k1));
                    mup[j].y = fma(mgam, sB, cc.y * fma(cc.y, cc.y, k1));
                    if (DIAG && valid && s >= 1 && s <= ZR) {       // F and mass of plane z+1 = z0 + s - 1
                        const double dxA = cc.y - cc.x, dyA = dn.x - cc.x, dzA = Cp[j].x - cc.x, qA = cc.x * cc.x - 1.0;
                        const double dxB = rgt - cc.y, dyB = dn.y - cc.y, dzB = Cp[j].y - cc.y, qB = cc.y * cc.y - 1.0;
                        F += (0.25 * qA * qA + 0.5 * prm.gamma * (dxA * dxA + dyA * dyA + dzA * dzA))
                           + (0.25 * qB * qB + 0.5 * prm.gamma * (dxB * dxB + dyB * dyB + dzB * dzB));
                        ms += cc.x + cc.y;
                    }
                }
                // ---- r(z) from mu(z) = mu0, its in-plane neighbours, mu(z-1) = mum and mu(z+1) = mup
                const bool out = s >= 2;
#pragma unroll
                for (int j = 0; j < RY; ++j) {
                    const double2 up = j == 0 ? Mup : mu0[j - 1], dn = j == RY - 1 ? Mdn : mu0[j + 1], mc = mu0[j];
                    const double ml = hshfl_up(mc.y), mr = hshfl_down(mc.x);
                    const double sA = ((ml + mc.y) + (up.x + dn.x)) + (mum[j].x + mup[j].x);
                    const double sB = ((mc.x + mr) + (up.y + dn.y)) + (mum[j].y + mup[j].y);
                    if (DIAG && valid && out) {                     // Fdot of plane z = z0 + s - 2
                        const double dxA = mc.y - mc.x, dyA = dn.x - mc.x, dzA = mup[j].x - mc.x;
                        const double dxB = mr - mc.y, dyB = dn.y - mc.y, dzB = mup[j].y - mc.y;
                        Fd -= (dxA * dxA + dyA * dyA + dzA * dzA) + (dxB * dxB + dyB * dyB + dzB * dzB);
                    }
                    if (out && valid && (!DIAG || prm.write)) {
                        double2 o;
                        o.x = scale * fma(-6.0, mc.x, sA);
                        o.y = scale * fma(-6.0, mc.y, sB);
                        *reinterpret_cast<double2 *>(pr + (size_t)(z0 + s - 2) * n2 + j * N) = o;
                    }
                }
                // ---- publish the edge rows of C(z+2) and mu(z+1) for the next step, rotate the window
                exC[((par * 2 + 0) * NHW + hw) * 16 + li] = Cp[0];
                exC[((par * 2 + 1) * NHW + hw) * 16 + li] = Cp[RY - 1];
                exM[((par * 2 + 0) * NHW + hw) * 16 + li] = mup[0];
                exM[((par * 2 + 1) * NHW + hw) * 16 + li] = mup[RY - 1];
#pragma unroll
                for (int j = 0; j < RY; ++j) { Cm[j] = C0[j]; C0[j] = Cp[j]; mum[j] = mu0[j]; mu0[j] = mup[j]; }
                __syncthreads();
            }
        }
        if (DIAG) {
            F = warp_sum(F); Fd = warp_sum(Fd); ms = warp_sum(ms);
            if ((tid & 31) == 0) { red[tid >> 5][0] = F; red[tid >> 5][1] = Fd; red[tid >> 5][2] = ms; }
            __syncthreads();
            if (tid == 0) {
                for (int q = 1; q < (NT >> 5); ++q) { F += red[q][0]; Fd += red[q][1]; ms += red[q][2]; }
                double *o = partials + (((size_t)m * strips + strip) * NZ + zr) * 3;
                o[0] = F; o[1] = Fd; o[2] = ms;
            }
            __syncthreads();
        }
    }
}

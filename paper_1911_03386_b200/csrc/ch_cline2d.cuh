// ch_cline2d.cuh -- the line kernel of ch_line2d.cuh for lines longer than one CTA can hold
// (N = 512 * CS, CS = 2, 4, 8: CFG5's 2048-point lines).  DESIGN.md section 5.
//
//   k_rhs_sweep_y_cline   w = A_y^-1 Lap_h mu(C)  (scale applied by k_sweep_x_update)
//
// Same tile, thread mapping, private cp.async staging and register-resident chunk solve as
// k_rhs_sweep_y_line.  The line is spread over a thread-block cluster of CS CTAs (512 rows each).
// Only the truncated closure (K <= 2 chunks, small gamma dt) is handled here: a chunk needs the two
// chunks next to it, so the only traffic between CTAs is the last warp of CTA r pushing its two chunk
// states into "ghost" slots of CTA r+1 (forward) and the first warp of CTA r+1 pushing its states into
// CTA r (backward) -- remote shared-memory stores followed by a release store of a sequence number at
// cluster scope, polled locally with acquire loads.  No cluster barrier inside the tile loop.
// Larger K (paper-regime gamma dt) and sampling steps use the st.async cluster kernel of ch_fused2d.cuh.
#pragma once

#include <cuda_runtime.h>

#include "ch_line2d.cuh"

__device__ __forceinline__ unsigned cl_rank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cl_map(const void *local, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"((unsigned)__cvta_generic_to_shared(local)), "r"(rank));
    return r;
}
__device__ __forceinline__ void cl_store2(unsigned remote, double2 v)
{
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};\n" ::"r"(remote), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void cl_flag_release(unsigned remote_flag, unsigned seq)
{
    asm volatile("st.release.cluster.shared::cluster.u32 [%0], %1;\n" ::"r"(remote_flag), "r"(seq) : "memory");
}
__device__ __forceinline__ void cl_flag_wait(const unsigned *flag, unsigned seq)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(flag);
    unsigned v;
    do {
        asm volatile("ld.acquire.cluster.shared::cta.u32 %0, [%1];\n" : "=r"(v) : "r"(a) : "memory");
    } while (v < seq);
#ifdef CH_DEBUG_SYNC
    if (v != seq) __trap();           // the neighbouring CTA is never a whole tile ahead (ch_line2d.cuh, flag_wait)
#endif
}
__device__ __forceinline__ void cl_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

// slots of one direction: [column A|B][P + 2 chunks][16 lanes]; forward slots hold chunks -2 .. P-1
// (index s + 2, the first two are ghosts written by the previous CTA), backward slots chunks 0 .. P+1
// (the last two are ghosts written by the next CTA).
#define CLINE_NC 512
#define CLINE_P (CLINE_NC / LINE_LC)
#define CLINE_SS 17                              /* lane stride of a chunk's slots in the SCAN kernels (conflict-free transposed access) */
#define CLINE_SLOT ((CLINE_P + 2) * CLINE_SS)

#define CH_MAX_CS 8
static inline size_t cline_smem() { return (size_t)(LINE_LC + 4) * CLINE_NC * 16 + (size_t)4 * CLINE_SLOT * 16 + (size_t)2 * CH_MAX_CS * 32 * 16; }

// first: index of the nearer of the two chunks (c - 1 + 2 forward, c + 1 backward); step: -1 / +1
__device__ __forceinline__ void cline_state_in(const LineParams &prm, const double2 *slots, int first, int step, int li,
                                               double &aA, double &bA, double &aB, double &bB)
{
    const double2 oA = slots[first * 16 + li], oB = slots[CLINE_SLOT + first * 16 + li];
    aA = fma(prm.W0[0], oA.x, prm.W0[1] * oA.y);
    bA = fma(prm.W0[2], oA.x, prm.W0[3] * oA.y);
    aB = fma(prm.W0[0], oB.x, prm.W0[1] * oB.y);
    bB = fma(prm.W0[2], oB.x, prm.W0[3] * oB.y);
    if (prm.K == 2) {
        const int s = first + step;
        const double2 pA = slots[s * 16 + li], pB = slots[CLINE_SLOT + s * 16 + li];
        aA = fma(prm.W1[0], pA.x, fma(prm.W1[1], pA.y, aA));
        bA = fma(prm.W1[2], pA.x, fma(prm.W1[3], pA.y, bA));
        aB = fma(prm.W1[0], pB.x, fma(prm.W1[1], pB.y, aB));
        bB = fma(prm.W1[2], pB.x, fma(prm.W1[3], pB.y, bB));
    }
}

// Closure for long K (SCAN kernels; paper-regime gamma dt): called by every thread after its chunk states
// are in `slots` ([column A|B][P + 2 chunks][16 lanes], this direction's local chunks at index base + c).
//  1. CTA barrier; the slots are re-read transposed (lane = chunk, one column per warp pass, two passes) and
//     scanned NON-cyclically with shuffles: T(c) = sum_{j <= pos} M^j out(c -+ j), pos = chunks since the CTA's
//     entry side; the exclusive part goes back into the slot, the CTA aggregate T(pos = 31) is pushed into
//     agg[rank][column] of EVERY CTA of the cluster (remote shared-memory stores);
//  2. cluster barrier (release/acquire: the pushes are visible, and it is a CTA barrier too);
//  3. state entering chunk c = exclusive(c) + M^pos S,  S = sum_{q=1..CS} WG[q-1] A_{rank -+ q}
//     (ch_factor.h, two-level form; tables prm.S2 = Mlane[32][4] then WG[8][4] in device memory).
template <int CS>
__device__ __forceinline__ void cline_scan_closure(const LineParams &prm, double2 *slots, int base, double2 *agg, int tid,
                                                   unsigned rank, int dir, double &aA, double &bA, double &aB, double &bB)
{
    constexpr int P = CLINE_P;
    const int lane = tid & 31, wid = tid >> 5, li = tid & 15, c = tid >> 4;
    __syncthreads();
    const int pos_l = dir > 0 ? lane : 31 - lane;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int col = q * 16 + wid;                                 // 0..31: [column A|B][16 lanes]
        double2 *slot = slots + (col >> 4) * CLINE_SLOT + (base + lane) * CLINE_SS + (col & 15);
        const double2 o = *slot;
        double ta = o.x, tb = o.y;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const int d = 1 << k, src = dir > 0 ? lane - d : lane + d;
            const double ua = __shfl_sync(0xffffffffu, ta, src & 31), ub = __shfl_sync(0xffffffffu, tb, src & 31);
            if (pos_l >= d) {
                ta = fma(prm.Mp[k][0], ua, fma(prm.Mp[k][1], ub, ta));
                tb = fma(prm.Mp[k][2], ua, fma(prm.Mp[k][3], ub, tb));
            }
        }
        const int prev = dir > 0 ? lane - 1 : lane + 1;
        double ea = __shfl_sync(0xffffffffu, ta, prev & 31), eb = __shfl_sync(0xffffffffu, tb, prev & 31);
        if (pos_l == 0) { ea = 0.0; eb = 0.0; }
        *slot = make_double2(ea, eb);
        if (pos_l == 31) {
            const double2 A = make_double2(ta, tb);
#pragma unroll 1
            for (unsigned rk = 0; rk < CS; ++rk) cl_store2(cl_map(agg + rank * 32 + col, rk), A);
        }
    }
    cl_sync_all();
    double SaA = 0.0, SbA = 0.0, SaB = 0.0, SbB = 0.0;
    int r = (int)rank;
#pragma unroll 1
    for (int q = 0; q < CS; ++q) {
        r -= dir;
        if (r < 0) r += CS;
        if (r >= CS) r -= CS;
        const double2 gA = agg[r * 32 + li], gB = agg[r * 32 + 16 + li];
        const double2 w01 = __ldg(reinterpret_cast<const double2 *>(prm.S2) + 64 + 2 * q);
        const double2 w23 = __ldg(reinterpret_cast<const double2 *>(prm.S2) + 64 + 2 * q + 1);
        SaA = fma(w01.x, gA.x, fma(w01.y, gA.y, SaA)); SbA = fma(w23.x, gA.x, fma(w23.y, gA.y, SbA));
        SaB = fma(w01.x, gB.x, fma(w01.y, gB.y, SaB)); SbB = fma(w23.x, gB.x, fma(w23.y, gB.y, SbB));
    }
    const int pos = dir > 0 ? c : P - 1 - c;
    const double2 m01 = __ldg(reinterpret_cast<const double2 *>(prm.S2) + 2 * pos);
    const double2 m23 = __ldg(reinterpret_cast<const double2 *>(prm.S2) + 2 * pos + 1);
    const double2 eA = slots[(base + c) * CLINE_SS + li], eB = slots[CLINE_SLOT + (base + c) * CLINE_SS + li];
    aA = fma(m01.x, SaA, fma(m01.y, SbA, eA.x)); bA = fma(m23.x, SaA, fma(m23.y, SbA, eA.y));
    aB = fma(m01.x, SaB, fma(m01.y, SbB, eB.x)); bB = fma(m23.x, SaB, fma(m23.y, SbB, eB.y));
}

// grid = CS * min(ntiles, resident clusters) with cluster dimension CS, block = 512,
// dynamic smem = cline_smem().  SCAN == false requires prm.K <= 2 (neighbour flags); SCAN == true handles any K.
template <int CS, bool SCAN>
__global__ void __launch_bounds__(CLINE_NC, 1) k_rhs_sweep_y_cline(const __grid_constant__ LineParams prm,
                                                                  const double *__restrict__ C, double *__restrict__ w)
{
    constexpr int LC = LINE_LC, NR = LC + 4, NT = CLINE_NC, P = CLINE_P, N = CLINE_NC * CS, NW = NT / 32;
    constexpr int strips = (N + LINE_VALID - 1) / LINE_VALID;
    constexpr int SS = SCAN ? CLINE_SS : 16;
    constexpr size_t n2 = (size_t)N * N;
    extern __shared__ double2 sm2[];
    __shared__ unsigned flagF[NW], flagB[NW], gflagF, gflagB;
    const int tid = threadIdx.x, li = tid & 15, c = tid >> 4, wid = tid >> 5;
    const unsigned rank = cl_rank();
    const int cid = blockIdx.x / CS, ncl = gridDim.x / CS, ntiles = prm.ntiles;
    const int cg = (int)rank * P + c;                              // chunk index along the whole line
    double2 *stage = sm2 + tid;
    double2 *slotF = sm2 + (size_t)NR * NT, *slotB = slotF + 2 * CLINE_SLOT;
    double2 *aggF = slotB + 2 * CLINE_SLOT, *aggB = aggF + CH_MAX_CS * 32;      // SCAN: CTA aggregates [rank][32 columns]
    if (tid < NW) { flagF[tid] = 0; flagB[tid] = 0; }
    if (tid == 0) { gflagF = 0; gflagB = 0; }
    __syncthreads();
    pdl_trigger();
    cl_sync_all();                 // every CTA of the cluster has initialised its flags before anyone pushes
    pdl_wait();
    // where the boundary warps push their chunk states: ghost slots and ghost flag of the neighbouring CTA
    unsigned remSlot = 0, remFlag = 0;
    if (wid == NW - 1) {
        const unsigned nxt = (rank + 1) % CS;
        remSlot = cl_map(&slotF[(c - (P - 2)) * 16 + li], nxt);
        remFlag = cl_map(&gflagF, nxt);
    } else if (wid == 0) {
        const unsigned prv = (rank + CS - 1) % CS;
        remSlot = cl_map(&slotB[(P + c) * 16 + li], prv);
        remFlag = cl_map(&gflagB, prv);
    }
    unsigned seq = 0;

    auto tile_base = [&](int tile) {
        const int strip = tile % strips, m = tile / strips;
        int gx = strip * LINE_VALID - 2 + 2 * li;
        if (gx < 0) gx += N;
        if (gx >= N) gx -= N;
        return C + (size_t)m * n2 + gx + (ptrdiff_t)(cg * LC - 2) * N;
    };
    auto load_row = [&](const double *p, int j) {
        const double *q = p + (ptrdiff_t)j * N;
        if (j < 2 && cg == 0) q += n2;
        if (j >= LC + 2 && cg == CS * P - 1) q -= n2;
        line_cp_async16(stage + j * NT, q);
    };

    int tile = cid;
    if (tile < ntiles) {
        const double *p = tile_base(tile);
#pragma unroll
        for (int j = 0; j < NR; ++j) load_row(p, j);
        line_cp_async_commit();
    }
    const double np = prm.np, nq = prm.nq, mgam = prm.mgam, k1 = prm.k1;

    for (; tile < ntiles; tile += ncl) {
        const bool more = tile + ncl < ntiles;
        const double *pn = tile_base(more ? tile + ncl : tile);
        line_cp_async_wait_all();
        double vA[LC], vB[LC];
        {
            auto mu_row = [&](const double2 cu, const double2 cc, const double2 cd) {
                const double lft = hshfl_up(cc.y), rgt = hshfl_down(cc.x);
                const double sA = (lft + cc.y) + (cu.x + cd.x), sB = (cc.x + rgt) + (cu.y + cd.y);
                double2 mu;
                mu.x = fma(mgam, sA, cc.x * fma(cc.x, cc.x, k1));
                mu.y = fma(mgam, sB, cc.y * fma(cc.y, cc.y, k1));
                return mu;
            };
            double2 c0 = stage[0], c1 = stage[NT], c2 = stage[2 * NT], c3 = stage[3 * NT];
            double2 mu_a = mu_row(c0, c1, c2);
            double2 mu_b = mu_row(c1, c2, c3);
            double ml = hshfl_up(mu_b.y), mr = hshfl_down(mu_b.x);
            c0 = c2; c1 = c3;
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                const double2 cn = stage[(k + 4) * NT];
                if (more) load_row(pn, k);              // refill the consumed staging row with the next tile's row k
                const double2 mu_c = mu_row(c0, c1, cn);
                const double rA = fma(-4.0, mu_b.x, (ml + mu_b.y) + (mu_a.x + mu_c.x));
                const double rB = fma(-4.0, mu_b.y, (mu_b.x + mr) + (mu_a.y + mu_c.y));
                if (k == 0) { vA[0] = rA; vB[0] = rB; }
                else if (k == 1) { vA[1] = fma(np, vA[0], rA); vB[1] = fma(np, vB[0], rB); }
                else { vA[k] = fma(np, vA[k - 1], fma(nq, vA[k - 2], rA)); vB[k] = fma(np, vB[k - 1], fma(nq, vB[k - 2], rB)); }
                mu_a = mu_b; mu_b = mu_c; c0 = c1; c1 = cn;
                if (k + 1 < LC) { ml = hshfl_up(mu_b.y); mr = hshfl_down(mu_b.x); }
            }
        }
        if (more) {
#pragma unroll
            for (int j = LC; j < NR; ++j) load_row(pn, j);
        }
        line_cp_async_commit();

        // ---- forward closure: publish, push across the CTA boundary, wait for the warp before
        ++seq;
        {
            const double2 sA = make_double2(vA[LC - 1], vA[LC - 2]), sB = make_double2(vB[LC - 1], vB[LC - 2]);
            slotF[(c + 2) * SS + li] = sA;
            slotF[CLINE_SLOT + (c + 2) * SS + li] = sB;
            double aA, bA, aB, bB;
            if (SCAN) {
                cline_scan_closure<CS>(prm, slotF, 2, aggF, tid, rank, +1, aA, bA, aB, bB);
            } else {
                if (wid == NW - 1) { cl_store2(remSlot, sA); cl_store2(remSlot + CLINE_SLOT * 16, sB); }
                __syncwarp();
                if ((tid & 31) == 0) {
                    flag_release(&flagF[wid], seq);
                    if (wid == NW - 1) cl_flag_release(remFlag, seq);
                }
                if (wid == 0) cl_flag_wait(&gflagF, seq); else flag_wait(&flagF[wid - 1], seq);
                __syncwarp();
                cline_state_in(prm, slotF, c + 1, -1, li, aA, bA, aB, bB);
            }
#pragma unroll
            for (int k = 0; k < LC; ++k) {
                vA[k] = fma(prm.alpha[k], aA, fma(prm.beta[k], bA, vA[k]));
                vB[k] = fma(prm.alpha[k], aB, fma(prm.beta[k], bB, vB[k]));
            }
        }
        // ---- backward recurrence from a zero state, then the same exchange in the other direction
        vA[LC - 2] = fma(np, vA[LC - 1], vA[LC - 2]);
        vB[LC - 2] = fma(np, vB[LC - 1], vB[LC - 2]);
#pragma unroll
        for (int k = LC - 3; k >= 0; --k) {
            vA[k] = fma(np, vA[k + 1], fma(nq, vA[k + 2], vA[k]));
            vB[k] = fma(np, vB[k + 1], fma(nq, vB[k + 2], vB[k]));
        }
        {
            const double2 sA = make_double2(vA[0], vA[1]), sB = make_double2(vB[0], vB[1]);
            slotB[c * SS + li] = sA;
            slotB[CLINE_SLOT + c * SS + li] = sB;
            double aA, bA, aB, bB;
            if (SCAN) {
                cline_scan_closure<CS>(prm, slotB, 0, aggB, tid, rank, -1, aA, bA, aB, bB);
            } else {
                if (wid == 0) { cl_store2(remSlot, sA); cl_store2(remSlot + CLINE_SLOT * 16, sB); }
                __syncwarp();
                if ((tid & 31) == 0) {
                    flag_release(&flagB[wid], seq);
                    if (wid == 0) cl_flag_release(remFlag, seq);
                }
                if (wid == NW - 1) cl_flag_wait(&gflagB, seq); else flag_wait(&flagB[wid + 1], seq);
                __syncwarp();
                cline_state_in(prm, slotB, c + 1, +1, li, aA, bA, aB, bB);
            }
            const int t2 = opaque(tile), tid2 = opaque(tid);
            const int strip2 = t2 % strips, m2 = t2 / strips, li2 = tid2 & 15;
            const int gx = strip2 * LINE_VALID - 2 + 2 * li2;
            if (li2 >= 1 && li2 < 15 && gx < N) {
                double2 *wm = reinterpret_cast<double2 *>(w + (size_t)m2 * n2 + (size_t)((int)rank * P + (tid2 >> 4)) * (LC * N) + gx);
#pragma unroll
                for (int k = 0; k < LC; ++k) {
                    double2 o;
                    o.x = fma(prm.alpha[LC - 1 - k], aA, fma(prm.beta[LC - 1 - k], bA, vA[k]));
                    o.y = fma(prm.alpha[LC - 1 - k], aB, fma(prm.beta[LC - 1 - k], bB, vB[k]));
                    wm[(size_t)k * (N / 2)] = o;
                }
            }
        }
    }
    cl_sync_all();                 // nobody leaves while a neighbour may still push into its shared memory
}

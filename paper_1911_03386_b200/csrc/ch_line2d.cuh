// ch_line2d.cuh -- fused RHS + y-sweep of the 2D step for lines that fit one CTA (N <= 512).
// DESIGN.md section 5.
//
//   k_rhs_sweep_y_line   w = A_y^-1 Lap_h mu(C)   (scale applied by k_sweep_x_update)                   P:29-30, include/ch.h
//                        (+ fused F, Fdot, mass partials on sampling steps)
//
// A persistent CTA owns whole columns: tile = one column strip (28 produced columns + a halo of 2 on
// either side) x all N rows of one member.  Thread (li, c) -- half-warp lane li, chunk c of 16 rows --
// carries two adjacent columns.  It stages its own 20 C rows (16 + halo 2 + 2) with cp.async, forms mu
// and r = Lap_h mu in a rolling register window (x-neighbours in the lane or by half-warp shuffle) and
// feeds r straight into the chunked periodic-LU recurrence of ch_factor.h, whose 2-double chunk states
// are exchanged through shared memory (the whole line is in this CTA: no cluster, no global traffic).
// r and the forward/backward intermediates never exist in memory: 16 B per grid-point update.
// A thread reads back only the rows it staged itself, so there is no barrier between load and compute and a
// staging row is free a few rows after it was read: row k of the CTA's NEXT tile is issued from inside the
// forward loop at row k, so the next tile's loads are in flight for a whole tile period without a second buffer.
// Synchronisation of the chunk exchange: neighbour-warp release/acquire flags when the closure is truncated to
// K <= 2 chunks (NB kernels), CTA barriers + K-term sum or log-depth shuffle scan otherwise.
#pragma once

#include <cuda_runtime.h>

#include "ch_kernels.cuh"

#define LINE_LC 16
#define LINE_VALID 28         // columns a half-warp produces: 16 lanes x 2 columns minus a halo of 2 on either side
#define LINE_SS 17            // lane stride of the slots in the barrier kernels (conflict-free transposed re-read)
#define LINE_MAX_P 32         // chunks per line: 16 * P threads per CTA

struct LineParams {
    double np, nq;                  // recurrence  z_i = b_i + np z_{i-1} + nq z_{i-2}
    double gamma, mgam, k1;         // mu = c (c^2 + k1) - gamma * (sum of the 4 neighbours), k1 = 4 gamma - 1
    double alpha[LINE_LC], beta[LINE_LC];
    double W0[4], W1[4];            // first two closure matrices (all of them when K <= 2)
    const double *W;                // device [K][4] (ch_factor.h)
    int K, ntiles, write;
    int M;                          // ensemble members in this launch
    // log-depth closure of the barrier kernels when the K-term sum is long (ch_factor.h, Mpow2 / Wclose)
    double Mp[5][4], Wc[4];
    int scan;                       // 0, or log2 P (P a power of two)
    const double *S2;               // cluster line SCAN kernels: device Mlane[32][4] then WG[8][4] (ch_factor.h)
};

__device__ __forceinline__ void line_cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
// same copy with an L2 evict-first hint: for streams that are read once (they should not displace what the NEXT
// kernel will find in L2: the w this kernel writes, the C the previous kernel wrote)
__device__ __forceinline__ unsigned long long l2_evict_first_policy()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ void line_cp_async16_hint(void *smem_dst, const void *gsrc, unsigned long long policy)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "l"(policy) : "memory");
}
__device__ __forceinline__ void line_cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void line_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

__device__ __forceinline__ double hshfl_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1, 16); }
__device__ __forceinline__ double hshfl_down(double v) { return __shfl_down_sync(0xffffffffu, v, 1, 16); }

// Neighbour synchronisation (NB kernels, K <= 2): a warp holds chunks 2w and 2w+1, and with K <= 2 the
// state entering a chunk depends on the two chunks before (forward) or after (backward) it only, i.e. on
// the warp itself and ONE neighbouring warp.  Instead of a CTA-wide barrier each warp publishes a
// sequence number (release) after writing its exchange slots and polls its neighbour's (acquire), so
// the warps of a CTA drift apart and their load / fp64 / store phases overlap.
// CH_DEBUG_SYNC (python -m paper_1911_03386_b200.build --debug-sync -> libch_debugsync.so; tests/test_parity_gpu.py runs the
// stress shapes against it): the protocol's invariants are checked in the kernel and a violation traps.  A warp publishes
// tile numbers in steps of exactly one, and when a waiter's condition becomes true the flag it polls equals the tile it
// waits for -- a neighbour can never be a whole tile ahead, because it rewrites a slot only after the reader of that slot
// has published the NEXT flag of the tile in between.
__device__ __forceinline__ void flag_release(unsigned *flag, unsigned seq)
{
#ifdef CH_DEBUG_SYNC
    {
        unsigned old;
        asm volatile("ld.relaxed.cta.shared.u32 %0, [%1];\n" : "=r"(old) : "r"((unsigned)__cvta_generic_to_shared(flag)) : "memory");
        if (old + 1u != seq) __trap();
    }
#endif
    asm volatile("st.release.cta.shared.u32 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(flag)), "r"(seq) : "memory");
}
__device__ __forceinline__ void flag_wait(const unsigned *flag, unsigned seq)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(flag);
    unsigned v;
    do {
        asm volatile("ld.acquire.cta.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(a) : "memory");
    } while (v < seq);
#ifdef CH_DEBUG_SYNC
    if (v != seq) __trap();
#endif
}

// keeps the compiler from carrying values derived from x across the long tile body in registers:
// what is needed again at the end of a tile is recomputed there from an opaque copy
__device__ __forceinline__ int opaque(int x) { asm volatile("" : "+r"(x)); return x; }

// states entering chunk c (both columns of the lane) from the K chunks before it (dir = +1) or after
// it (dir = -1); slots are [column A|B][chunk][16 lanes] pairs (value next to the boundary, one further in)
template <int P, int SS>
__device__ __forceinline__ void line_state_in(const LineParams &prm, const double2 *slots, int tid, int dir,
                                              double &aA, double &bA, double &aB, double &bB)
{
    const int c = tid >> 4, li = tid & 15;
    aA = bA = aB = bB = 0.0;
    auto acc = [&](int s, double w0, double w1, double w2, double w3) {
        const double2 oA = slots[s * SS + li], oB = slots[(P + s) * SS + li];
        aA = fma(w0, oA.x, fma(w1, oA.y, aA));
        bA = fma(w2, oA.x, fma(w3, oA.y, bA));
        aB = fma(w0, oB.x, fma(w1, oB.y, aB));
        bB = fma(w2, oB.x, fma(w3, oB.y, bB));
    };
    int s = c;
    auto next = [&]() { s -= dir; if (s < 0) s += P; if (s >= P) s -= P; };
    if (prm.K <= 2) {                       // small gamma dt: the tables sit in the constant bank
        next(); acc(s, prm.W0[0], prm.W0[1], prm.W0[2], prm.W0[3]);
        if (prm.K == 2) { next(); acc(s, prm.W1[0], prm.W1[1], prm.W1[2], prm.W1[3]); }
        return;
    }
    for (int j = 0; j < prm.K; ++j) {
        next();
        const double2 W01 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j);
        const double2 W23 = __ldg(reinterpret_cast<const double2 *>(prm.W) + 2 * j + 1);
        acc(s, W01.x, W01.y, W23.x, W23.y);
    }
}

// Log-depth closure for the barrier kernels (after the CTA barrier that follows the slot writes): the
// slots are re-read TRANSPOSED -- lane = chunk, 32 / P columns per warp pass, two passes cover the 32
// columns -- scanned with width-P shuffles exactly as chunk_state_scan (ch_kernels.cuh), written back in
// place as the states ENTERING each chunk, and after one more barrier every thread picks up its own.
template <int P, int SS>
__device__ __forceinline__ void line_scan_closure(const LineParams &prm, double2 *slots, int tid, int dir,
                                                  double &aA, double &bA, double &aB, double &bB)
{
    constexpr int CPW = 32 / P;
    const int lane = tid & 31, wid = tid >> 5, ch = lane % P;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int col = q * 16 + wid * CPW + lane / P;
        double2 *slot = slots + ((col >> 4) * P + ch) * SS + (col & 15);
        const double2 o = *slot;
        double ta = o.x, tb = o.y;
        for (int k = 0; k < prm.scan; ++k) {
            const int src = (ch - dir * (1 << k)) & (P - 1);
            const double ua = __shfl_sync(0xffffffffu, ta, src, P), ub = __shfl_sync(0xffffffffu, tb, src, P);
            ta = fma(prm.Mp[k][0], ua, fma(prm.Mp[k][1], ub, ta));
            tb = fma(prm.Mp[k][2], ua, fma(prm.Mp[k][3], ub, tb));
        }
        const int src = (ch - dir) & (P - 1);
        const double ua = __shfl_sync(0xffffffffu, ta, src, P), ub = __shfl_sync(0xffffffffu, tb, src, P);
        *slot = make_double2(fma(prm.Wc[0], ua, prm.Wc[1] * ub), fma(prm.Wc[2], ua, prm.Wc[3] * ub));
    }
    __syncthreads();
    const double2 sA = slots[(tid >> 4) * SS + (tid & 15)], sB = slots[(P + (tid >> 4)) * SS + (tid & 15)];
    aA = sA.x; bA = sA.y; aB = sB.x; bB = sB.y;
}

// Tiling of the columns.  Plain: ceil(NC / 28) strips per member, the last one ragged.  Packed (stepping kernels,
// when the NC % 28 leftover columns fit a fraction of a half-warp): the leftover strips of G consecutive members share
// ONE tile -- G = 2: lanes 0..7 work on member 2j, lanes 8..15 on member 2j+1 (leftover <= 12 columns); G = 4: four
// lanes per member (leftover <= 4 columns) -- so a ragged strip costs 1/G of a tile
// (N = 512, 128 members: 2432 -> 2368 tiles = exactly 16 rounds of 148 CTAs; N = 256, 64 members: 640 -> 592 tiles =
// exactly 2 rounds of 2 x 148 CTAs).
template <int NC>
struct LineTiling {
    static constexpr int SF = NC / LINE_VALID, REM = NC - SF * LINE_VALID;
    static constexpr bool PACKABLE = REM > 0 && REM <= 12;
    static constexpr int G = REM <= 4 ? 4 : 2;          // members per shared leftover tile
};
static inline int line_packed_tiles(int N, int M)
{
    const int SF = N / LINE_VALID, REM = N - SF * LINE_VALID, G = REM <= 4 ? 4 : 2;
    return (M / G) * (G * SF + 1) + ((M % G) ? (M % G) * SF + 1 : 0);
}

// member, first column (wrapped, even) and "produces output" of half-warp lane li in `tile`.
// Packed order: members come in groups of G; group p owns the PT = G SF + 1 consecutive tiles p PT .. (p + 1) PT - 1:
// SF full strips of each of its members in turn, then the tile their leftover strips share.  An ensemble that is not
// a multiple of G ends with a short group: SF full strips per member and a partly idle leftover tile.
template <int NC, bool PACK>
__device__ __forceinline__ void line_tile_decode(int tile, int M, int li, int &m, int &gx, bool &ok)
{
    constexpr int strips = (NC + LINE_VALID - 1) / LINE_VALID, SF = LineTiling<NC>::SF, REM = LineTiling<NC>::REM;
    constexpr int G = LineTiling<NC>::G, S = 16 / G, PT = G * SF + 1;
    if (!PACK) {
        const int strip = tile % strips;
        m = tile / strips;
        gx = strip * LINE_VALID - 2 + 2 * li;
        ok = li >= 1 && li < 15 && gx < NC;
    } else {
        const int grp = tile / PT, k = tile - grp * PT;
        const int nm = (M - G * grp) < G ? (M - G * grp) : G;      // members of this group
        if (k < nm * SF) {
            const int q = k / SF;
            m = G * grp + q;
            gx = (k - q * SF) * LINE_VALID - 2 + 2 * li;
            ok = li >= 1 && li < 15;
        } else {
            const int ls = li & (S - 1);
            m = G * grp + li / S;
            gx = SF * LINE_VALID - 2 + 2 * ls;
            ok = ls >= 1 && ls <= REM / 2 && m < M;
            if (m >= M) m = M - 1;              // the idle lanes work on valid memory and store nothing
        }
    }
    if (gx < 0) gx += NC;
    if (gx >= NC) gx -= NC;
}

// NC = N at compile time (row offsets become immediates).
// grid = min(ntiles, resident CTAs), block = NC threads (= 16 threads per chunk, P = NC / 16 even),
// dynamic smem = 20 * NC * 16 (staging) + 2 * 2 * P * 16 * 16 (forward, backward exchange slots).
// NB: neighbour-warp synchronisation (needs K <= 2) instead of CTA barriers.  DIAG: also F, Fdot, mass partials, one per
// (member, strip, warp): partials[((m * strips + strip) * (NC / 32) + warp) * 3].
template <int NC, bool DIAG, bool NB>
__global__ void __launch_bounds__(NC, (NC <= 256 && !DIAG) ? 2 : 1) k_rhs_sweep_y_line(const __grid_constant__ LineParams prm,
                                                                                   const double *__restrict__ C,
                                                                                   double *__restrict__ w,
                                                                                   double *__restrict__ partials)
{
    constexpr int LC = LINE_LC, NR = LC + 4, N = NC, NT = NC, P = NC / LC;
    constexpr size_t n2 = (size_t)N * N;
    extern __shared__ double2 sm2[];
    __shared__ unsigned flagF[16], flagB[16];
    constexpr int NW = NC / 32;
    const int tid = threadIdx.x, li = tid & 15, c = tid >> 4, wid = tid >> 5;
    constexpr int strips = (NC + LINE_VALID - 1) / LINE_VALID;
    const int ntiles = prm.ntiles;
    pdl_trigger();
    if (NB) {
        if (tid < 16) { flagF[tid] = 0; flagB[tid] = 0; }
        __syncthreads();
    }
    pdl_wait();
    unsigned seq = 0;
    const int y0 = c * LC;
    const bool lane_ok = li >= 1 && li < 15;

    double2 *stage = sm2 + tid;                                   // row j of this thread: stage[j * NT]
    constexpr int SS = NB ? 16 : LINE_SS;                       // lane stride of a chunk's slots
    double2 *slotF = sm2 + (size_t)NR * NT, *slotB = slotF + 2 * P * LINE_SS;

    // C rows y0-2 .. y0+LC+1 of this thread's column pair; only the two halo rows on either end wrap
    constexpr bool PACK = !DIAG && LineTiling<NC>::PACKABLE;
    auto tile_base = [&](int tile) {
        int m, gx; bool ok;
        line_tile_decode<NC, PACK>(tile, prm.M, li, m, gx, ok);
        return C + (size_t)m * n2 + gx + (ptrdiff_t)(y0 - 2) * N;
    };
    auto load_row = [&](const double *p, int j) {     // j is a compile-time constant after unrolling
        const double *q = p + (ptrdiff_t)j * N;
        if (j < 2 && c == 0) q += n2;
        if (j >= LC + 2 && c == P - 1) q -= n2;
        line_cp_async16(stage + j * NT, q);
    };

    int tile = blockIdx.x;
    if (tile < ntiles) {
        const double *p = tile_base(tile);
#pragma unroll
        for (int j = 0; j < NR; ++j) load_row(p, j);
        line_cp_async_commit();
    }
    const double np = prm.np, nq = prm.nq, mgam = prm.mgam, k1 = prm.k1;

    for (; tile < ntiles; tile += gridDim.x) {
        const int strip = tile % strips, m = tile / strips;
        const bool valid = lane_ok && (strip * LINE_VALID + 2 * (li - 1)) < N;     // used by the DIAG sums only
        const bool more = tile + (int)gridDim.x < ntiles;
        const double *pn = tile_base(more ? tile + gridDim.x : tile);
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
                // staging row k was consumed at least four rows ago: refill it with the NEXT tile's row k,
                // so the next tile's loads are in flight for a whole tile period
                if (more) load_row(pn, k);
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
        if (more) {
#pragma unroll
            for (int j = LC; j < NR; ++j) load_row(pn, j);
        }
        line_cp_async_commit();

        if (DIAG) {
            // deterministic sums without a CTA barrier (round 2): one partial per warp (fixed shuffle tree), k_finish adds
            // the strips x warps partials of a member in index order; the sampling kernel can then use the same
            // neighbour-warp synchronisation as the stepping kernel
            F = warp_sum(F); Fd = warp_sum(Fd); ms = warp_sum(ms);
            if ((tid & 31) == 0) {
                double *o = partials + (((size_t)m * strips + strip) * NW + wid) * 3;
                o[0] = F; o[1] = Fd; o[2] = ms;
            }
            if (!prm.write) continue;         // diagnostics only (grid-uniform): no sweep
        }

        // ---- forward closure
        if (NB) {                                                       // [column A|B][chunk][lane]: c * 16 + li == tid
            slotF[tid] = make_double2(vA[LC - 1], vA[LC - 2]);
            slotF[NT + tid] = make_double2(vB[LC - 1], vB[LC - 2]);
        } else {
            slotF[c * SS + li] = make_double2(vA[LC - 1], vA[LC - 2]);
            slotF[(P + c) * SS + li] = make_double2(vB[LC - 1], vB[LC - 2]);
        }
        ++seq;
        if (NB) {
            __syncwarp();
            if ((tid & 31) == 0) flag_release(&flagF[wid], seq);
            flag_wait(&flagF[(wid + NW - 1) % NW], seq);
            __syncwarp();
        } else {
            __syncthreads();
        }
        {
            double aA, bA, aB, bB;
            if (!NB && (P & (P - 1)) == 0 && prm.scan) line_scan_closure<P, SS>(prm, slotF, tid, +1, aA, bA, aB, bB);
            else line_state_in<P, SS>(prm, slotF, tid, +1, aA, bA, aB, bB);
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
        if (NB) {
            slotB[tid] = make_double2(vA[0], vA[1]);
            slotB[NT + tid] = make_double2(vB[0], vB[1]);
        } else {
            slotB[c * SS + li] = make_double2(vA[0], vA[1]);
            slotB[(P + c) * SS + li] = make_double2(vB[0], vB[1]);
        }
        if (NB) {
            __syncwarp();
            if ((tid & 31) == 0) flag_release(&flagB[wid], seq);
            flag_wait(&flagB[(wid + 1) % NW], seq);
            __syncwarp();
        } else {
            __syncthreads();  // also orders this tile's slotF reads before the next tile's slotF writes
        }
        {
            double aA, bA, aB, bB;
            if (!NB && (P & (P - 1)) == 0 && prm.scan) line_scan_closure<P, SS>(prm, slotB, tid, -1, aA, bA, aB, bB);
            else line_state_in<P, SS>(prm, slotB, tid, -1, aA, bA, aB, bB);
            // where this thread's results go, recomputed from the tile and thread index
            const int t2 = opaque(tile), tid2 = opaque(tid);
            int m2, gx; bool ok2;
            line_tile_decode<NC, PACK>(t2, prm.M, tid2 & 15, m2, gx, ok2);
            if (ok2) {                                              // producing lanes: 0 <= gx < N
                double2 *wm = reinterpret_cast<double2 *>(w + (size_t)m2 * n2 + (size_t)(tid2 >> 4) * (LC * N) + gx);
#pragma unroll
                for (int k = 0; k < LC; ++k) {
                    double2 o;
                    o.x = fma(prm.alpha[LC - 1 - k], aA, fma(prm.beta[LC - 1 - k], bA, vA[k]));
                    o.y = fma(prm.alpha[LC - 1 - k], aB, fma(prm.beta[LC - 1 - k], bB, vB[k]));
                    wm[(size_t)k * (N / 2)] = o;
                }
            }
        }
        // barrier kernels: slotB reads of this tile are ordered before the next tile's slotB writes by
        // the next tile's first __syncthreads.  NB kernels: a warp rewrites a slot only after the
        // neighbour that reads it has published a later sequence number.
    }
}

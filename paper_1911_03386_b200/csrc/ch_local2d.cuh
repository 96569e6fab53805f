// ch_local2d.cuh -- the whole 2D step in ONE pass over HBM when gamma dt is small (SURVEY.md section 8(f) NEXT-3 (i),
// DESIGN.md section 5b): read C^n once, write C^{n+1} once (16 B per grid-point update instead of 40).
//
//   k_step2d_local   C^{n+1} = C^n + (dt / c0^2) Lx^-T Lx^-1 Ly^-T Ly^-1 Lap_h mu(C^n)          P:29-30, include/ch.h
//
// Why it is legal.  A_d = c0 L^T L with L = I + p S^-1 + q S^-2 (ch_factor.h); the impulse response h_k of L^-1 decays
// like rho^k, rho = |root| (0.0972 at gamma dt = 0.01).  A recurrence started from a ZERO state H points before the
// first point that is used differs from the cyclic one by at most T(H) = sum_{k >= H} |h_k| times the data, and the
// host picks the smallest H with 2 G T(H) / c0 <= 2^-56 (ch_factor_reach; G = sum |h_k|): the truncation is below an
// eighth of an ulp of the local max |w| per sweep.  If that needs H > LOC_HMAX the exact two-kernel step runs instead.
//
// Structure.  The columns of a member are cut into strips of SW produced columns; a strip is computed on
// SW + 2 He columns (r-region, He = H rounded up to even) from SW + 2 He + 4 columns of C.  All strips of all members,
// stacked row after row, form a "tape"; every CTA (2 per SM, 7 warps) marches down an equal span of it, segment by
// segment (a segment = consecutive rows of one strip; it starts H + 2 rows early and ends H + 2 rows late, rows wrap).
// Per block of 32 rows:
//   P1 (warp w, lane l = r-region column 30 w + l - 1; lanes 1..30 produce, warps overlap by two columns)
//        the warp stages the 34 C columns it needs itself: one cp.async.bulk per row issued by an elected lane, completion on
//        the warp's own three mbarriers, 12-row ring (an extra L2 prefetch ahead of it measured SLOWER: 0.2585 vs
//        0.2521 ms on CFG3, and read 9 % more DRAM bytes).  Rolling register window: mu of the
//        next row (x-neighbours of C from the ring, of mu by shuffle), r = Lap_h mu, forward y-recurrence z (exact
//        streaming, state in registers), z -> z-ring.  No CTA barrier: warps drift apart, load / fp64 phases overlap.
//   P2 (same thread, its own column)   backward y-recurrence from a zero state at the newest row, H throw-away rows, in
//        place: the 32 rows that are H behind the front are final
//   P3 (lane = row, warp = chunk of 30 columns)   forward then backward x-recurrence of the chunk from a zero state, in
//        place; the state entering a chunk is its neighbour's zero-state out-state (exact to rho^28), applied as
//        alpha_k a + beta_k b to the first / last LOC_KC points: the forward correction inside the backward pass, the
//        backward correction inside P4.  Two CTA barriers.
//   P4 (warp = its own 30 columns, half-warp = row parity, lane = column pair)   C^{n+1} = C^n + scale (w + correction),
//        C^n re-read through L2, 16-byte stores.  P4 and the next P1 of a warp touch the same columns: no barrier needed.
// The result goes to a second array (the halo of a strip is another strip's interior): ch_step ping-pongs C and w.
// Measured and bounded in profiles/r02_ncu_full_local.md (shared-memory data pipe 69 %, issue 48 %, 2 x 7 warps per SM).
#pragma once

#include <cuda_runtime.h>

#include <type_traits>

#include "ch_kernels.cuh"     // pdl_wait / pdl_trigger

#define LOC_NW 7                          // warps per CTA
#define LOC_NT (32 * LOC_NW)
#define LOC_LB 32                         // rows per block
#define LOC_HMAX 18                       // largest reach the geometry below allows
#define LOC_XC 30                         // columns a warp produces in P1 / one x-chunk in P3
#define LOC_RW (LOC_XC * LOC_NW)          // widest r-region: 210 columns
#define LOC_ZP LOC_RW                     // pitch of the z-ring; ZP / 2 odd: LDS.128 with lane = row is conflict free
#define LOC_ZR (LOC_LB + LOC_HMAX)        // rows of the z-ring
#define LOC_WC 34                         // C columns a warp stages: its 32 + one on either side
#define LOC_SR 12                         // rows of a warp's C staging ring: 3 groups of 4
#define LOC_KC LOC_HMAX                   // points of a chunk the state of its neighbour still reaches

struct LocalParams {
    double np, nq;                  // recurrence  z_i = b_i + np z_{i-1} + nq z_{i-2}
    double mgam, k1;                // mu = c (c^2 + k1) - gamma * (sum of the 4 neighbours), k1 = 4 gamma - 1
    double oscale;                  // dt / c0^2
    double al[LOC_KC], be[LOC_KC];  // homogeneous solutions u_k of the recurrence for (u_-1, u_-2) = (1, 0) and (0, 1)
    int N, M, H;                    // H = reach (rows / columns of zero-state warm-up), <= LOC_HMAX
    int nstrips, SW;                // strips per member, produced columns of a full strip (multiple of 4)
    long long total_rows, span;     // tape rows = M * nstrips * N, rows per CTA
};

#define LOC_ZRING (LOC_ZR * LOC_ZP)
#define LOC_STAGE (LOC_NW * LOC_SR * LOC_WC)
#define LOC_SIDE (2 * (LOC_NW + 1) * LOC_LB * 2)     // [dir][chunk boundary][row] pairs of doubles
static inline size_t local_smem_bytes() { return (size_t)(LOC_ZRING + LOC_STAGE + LOC_SIDE) * 8; }

// ---- shared-memory access by 32-bit shared address (keeps ptxas from re-deriving the shared window base per access)
__device__ __forceinline__ double loc_lds(unsigned a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void loc_sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;\n" ::"r"(a), "d"(v) : "memory"); }
// ---- mbarrier + bulk global->shared copy (SASS: SYNCS / UBLKCP)
__device__ __forceinline__ void loc_mbar_init(unsigned mbar, unsigned count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(mbar), "r"(count) : "memory"); }
__device__ __forceinline__ void loc_mbar_expect_tx(unsigned mbar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void loc_bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}
__device__ __forceinline__ bool loc_elect_one()       // one lane of the (converged) warp, chosen by the hardware
{
    unsigned pred;
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "elect.sync _|p, 0xffffffff;\n"
                 "selp.u32 %0, 1, 0, p;\n"
                 "}\n" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void loc_mbar_wait(unsigned mbar, unsigned parity)
{
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "LOC_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@p bra LOC_DONE;\n"
                 "bra LOC_WAIT;\n"
                 "LOC_DONE:\n"
                 "}\n" ::"r"(mbar), "r"(parity) : "memory");
}

__global__ void __launch_bounds__(LOC_NT, 2) k_step2d_local(const __grid_constant__ LocalParams prm,
                                                             const double *__restrict__ Cin, double *__restrict__ Cout)
{
    extern __shared__ double2 loc_sm[];
    __shared__ unsigned long long loc_mbar[LOC_NW * 3];
    double *const zring = reinterpret_cast<double *>(loc_sm);           // [LOC_ZR][LOC_ZP]
    double *const stage = zring + LOC_ZRING;                              // [LOC_NW][LOC_SR][LOC_WC]
    double2 *const side = reinterpret_cast<double2 *>(stage + LOC_STAGE); // [2][LOC_NW + 1][LOC_LB]
    const int tid = threadIdx.x, lane = tid & 31;
    pdl_trigger();
    pdl_wait();
    const int wid = __shfl_sync(0xffffffffu, tid >> 5, 0);     // warp-uniform for the compiler: loader addresses stay in uniform registers
    const int N = prm.N, H = prm.H, He = (H + 1) & ~1;
    const double np = prm.np, nq = prm.nq, mgam = prm.mgam, k1 = prm.k1;
    const size_t n2 = (size_t)N * N;
    double *const cw = stage + wid * (LOC_SR * LOC_WC);                   // this warp's staging ring
    double2 *const sideF = side, *const sideB = side + (LOC_NW + 1) * LOC_LB;
    const unsigned zs = (unsigned)__cvta_generic_to_shared(zring);
    const unsigned cws = (unsigned)__cvta_generic_to_shared(cw);
    const unsigned mb = (unsigned)__cvta_generic_to_shared(loc_mbar + 3 * wid);
    constexpr unsigned ZPB = LOC_ZP * 8, ROWB = LOC_WC * 8;               // pitches in bytes

    if (lane == 0) {
        loc_mbar_init(mb, 1); loc_mbar_init(mb + 8, 1); loc_mbar_init(mb + 16, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncwarp();
    unsigned par = 0;                                // bit g: parity the next wait on staging group g expects

    long long tape = (long long)blockIdx.x * prm.span;
    const long long tape_end = tape + prm.span < prm.total_rows ? tape + prm.span : prm.total_rows;

    while (tape < tape_end) {
        // ---- this segment: rows ya .. ya + len - 1 of strip s of member m
        const long long line = tape / N;
        const int ya = (int)(tape - line * N);
        const int len = (int)((long long)(N - ya) < tape_end - tape ? (long long)(N - ya) : tape_end - tape);
        const int m = (int)(line / prm.nstrips), s = (int)(line - (long long)m * prm.nstrips);
        const int x0 = s * prm.SW, wd = prm.SW < N - x0 ? prm.SW : N - x0;
        tape += len;
        const int RWs = wd + 2 * He;                 // r-region: columns x0 - He .. x0 + wd + He - 1
        // r rows: row t is global row ya - H + t; produced rows are t in [H, H + len); rounded up to a multiple of 4
        // (the extra rows are real rows: they only lengthen the backward warm-up)
        const int T = (len + 2 * H + 3) & ~3;
        const int NU = T + 4;                        // C rows: row u is global row ya - H - 2 + u
        const double *const Cm = Cin + (size_t)m * n2;
        double *const Om = Cout + (size_t)m * n2;

        // P1 / P2 mapping: warp w, lane l <-> r-region column rc = 30 w + l - 1; lanes 1..30 produce.  The warp stages the
        // 34 C columns it needs itself (one bulk copy per row, issued by lane 0, completion on the warp's own mbarriers),
        // so P1 and P2 need no CTA barrier: warps drift apart and their load / fp64 phases overlap.
        const int rc = LOC_XC * wid + lane - 1;
        const bool p1_valid = lane >= 1 && lane <= LOC_XC && rc < RWs;
        const bool warp_on = LOC_XC * wid < RWs;     // warps beyond the strip stay idle in P1 / P2
        int gxw = (x0 - He - 2 + LOC_XC * wid) % N;  // first global column of the warp's 34-column window (even)
        if (gxw < 0) gxw += N;
        const int wa = gxw + LOC_WC <= N ? LOC_WC : N - gxw;   // columns before the periodic wrap
        // loader state (warp-uniform): global row and source pointer of the next C row to fetch, ring address, mbarrier
        int lgy = (ya - H - 2) % N;
        if (lgy < 0) lgy += N;
        const double *lsrc = Cm + (size_t)lgy * N + gxw;
        unsigned ldst = cws, lbar = mb;
        int lu = 0;                                  // next C row to fetch
        auto issue_group = [&]() {                   // the next 4 C rows into ring rows lu % 12 ..
            if (lu < NU) {                           // NU is a multiple of 4: a group is fetched whole or not at all
                if (loc_elect_one()) {
                    loc_mbar_expect_tx(lbar, 4 * ROWB);
                    if (lgy + 4 <= N && wa == LOC_WC) {          // the common case: no periodic wrap inside the group
                        loc_bulk_g2s(ldst, lsrc, ROWB, lbar);
                        loc_bulk_g2s(ldst + ROWB, lsrc + N, ROWB, lbar);
                        loc_bulk_g2s(ldst + 2 * ROWB, lsrc + 2 * (size_t)N, ROWB, lbar);
                        loc_bulk_g2s(ldst + 3 * ROWB, lsrc + 3 * (size_t)N, ROWB, lbar);
                    } else {
                        int gy = lgy;
                        const double *src = lsrc;
                        for (int h = 0; h < 4; ++h) {
                            loc_bulk_g2s(ldst + h * ROWB, src, wa * 8, lbar);
                            if (wa < LOC_WC) loc_bulk_g2s(ldst + h * ROWB + wa * 8, src - gxw, (LOC_WC - wa) * 8, lbar);
                            src += N;
                            if (++gy >= N) { gy -= N; src -= n2; }
                        }
                    }
                }
                lsrc += (size_t)4 * N; lgy += 4;
                if (lgy >= N) { lgy -= N; lsrc -= n2; }
                ldst += 4 * ROWB; lbar += 8;
                if (lbar == mb + 24) { lbar = mb; ldst -= 12 * ROWB; }
            }
            lu += 4;
        };
        auto wait_group = [&](int g) {               // staging group g (rows 4 g .. 4 g + 3 of the ring) has landed
            loc_mbar_wait(mb + 8 * g, (par >> g) & 1u);
            par ^= 1u << g;
        };
        double z1 = 0.0, z2 = 0.0, c_lo = 0.0, c_mid = 0.0, mu_a = 0.0, mu_b = 0.0, hs = 0.0;
        unsigned zw = zs + (unsigned)(rc < 0 ? 0 : rc) * 8;     // shared address of (row t of the z-ring, this thread's column); t = 0 now
        int zrow = 0;                                           // its ring row
        const double *const cown = cw + lane + 1;

        if (warp_on) { issue_group(); issue_group(); issue_group(); }
        const int nblocks = (T + LOC_LB - 1) / LOC_LB;
        for (int b = 0; b < nblocks; ++b) {
            const int top = LOC_LB * b + LOC_LB < T ? LOC_LB * b + LOC_LB : T;
            // rows [lo, hi) become final in this block
            const int lo = LOC_LB * b - H > H ? LOC_LB * b - H : H;
            const int hi = top - H < H + len ? top - H : H + len;
            if (warp_on) {
                // ---------------- P1: RHS + forward y-recurrence of rows 32 b .. top - 1
                // step t reads C row t + 4 only (own column and its two neighbours); one staging group = 4 rows
                int sg = ((LOC_LB * b + 4) >> 2) % 3;            // staging group of C rows t + 4 ..
                for (int t0 = LOC_LB * b; t0 < top; t0 += 4) {
                    if (t0 == 0) {
                        wait_group(0);
                        const double *q = cown;      // rows 0..3
                        const double C0 = q[0], C1 = q[LOC_WC], C2 = q[2 * LOC_WC], C3 = q[3 * LOC_WC];
                        mu_a = fma(mgam, (q[LOC_WC - 1] + q[LOC_WC + 1]) + (C0 + C2), C1 * fma(C1, C1, k1));
                        mu_b = fma(mgam, (q[2 * LOC_WC - 1] + q[2 * LOC_WC + 1]) + (C1 + C3), C2 * fma(C2, C2, k1));
                        c_lo = C2; c_mid = C3;
                        hs = q[3 * LOC_WC - 1] + q[3 * LOC_WC + 1];
                    }
                    wait_group(sg);                  // C rows t0 + 4 .. t0 + 7
                    __syncwarp();                    // every lane is done with rows t0 .. t0 + 3: their slots can be refilled
                    issue_group();                   // rows t0 + 12 .. t0 + 15
                    const double *rowp = cown + sg * (4 * LOC_WC);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double c_hi = rowp[i * LOC_WC];
                        const double hn = rowp[i * LOC_WC - 1] + rowp[i * LOC_WC + 1];
                        const double mu_c = fma(mgam, hs + (c_lo + c_hi), c_mid * fma(c_mid, c_mid, k1));
                        const double ml = __shfl_up_sync(0xffffffffu, mu_b, 1), mr = __shfl_down_sync(0xffffffffu, mu_b, 1);
                        const double r = fma(-4.0, mu_b, (ml + mr) + (mu_a + mu_c));
                        const double z = fma(np, z1, fma(nq, z2, r));
                        z2 = z1; z1 = z;
                        if (p1_valid) loc_sts(zw, z);
                        zw += ZPB;
                        if (++zrow == LOC_ZR) { zrow = 0; zw -= LOC_ZR * ZPB; }
                        mu_a = mu_b; mu_b = mu_c; c_lo = c_mid; c_mid = c_hi; hs = hn;
                    }
                    if (++sg == 3) sg = 0;
                }
                // ---------------- P2: backward y-recurrence of this thread's own column, zero state at row top
                // (>= H throw-away rows); rows [lo, hi) are final afterwards.  Runs between ring wraps: no per-row wrap test.
                if (hi > lo && p1_valid) {
                    double v1 = 0.0, v2 = 0.0;
                    int prow = zrow - 1;             // ring row of r row top - 1
                    unsigned pa = zw - ZPB;
                    if (prow < 0) { prow += LOC_ZR; pa += LOC_ZR * ZPB; }
                    auto sweep = [&](int cnt, auto store) {
                        while (cnt > 0) {
                            int run = cnt < prow + 1 ? cnt : prow + 1;
                            cnt -= run; prow -= run;
                            for (; run >= 4; run -= 4) {
#pragma unroll
                                for (int i = 0; i < 4; ++i) {
                                    const double v = fma(np, v1, fma(nq, v2, loc_lds(pa - i * ZPB)));
                                    v2 = v1; v1 = v;
                                    if (decltype(store)::value) loc_sts(pa - i * ZPB, v);
                                }
                                pa -= 4 * ZPB;
                            }
                            for (; run > 0; --run) {
                                const double v = fma(np, v1, fma(nq, v2, loc_lds(pa)));
                                v2 = v1; v1 = v;
                                if (decltype(store)::value) loc_sts(pa, v);
                                pa -= ZPB;
                            }
                            if (prow < 0) { prow += LOC_ZR; pa += LOC_ZR * ZPB; }
                        }
                    };
                    sweep(top - hi, std::false_type());
                    sweep(hi - lo, std::true_type());
                }
            }
            if (hi <= lo) continue;                  // CTA-uniform
            const int nf = hi - lo;
            __syncthreads();
            // ---------------- P3: x-sweep of rows lo .. hi - 1 (lane = row, warp = chunk of 30 columns).  Every chunk runs
            // from a zero state; the state entering it is its neighbour's zero-state out-state (exact to rho^28), applied
            // as alpha_k a + beta_k b to the first / last LOC_KC points: forward correction inside the backward pass,
            // backward correction inside P4.
            const int c0 = LOC_XC * wid, c1 = c0 + LOC_XC < RWs ? c0 + LOC_XC : RWs;
            const bool act = lane < nf && c0 < RWs;
            double *const rowp = zring + ((lo + lane) % LOC_ZR) * LOC_ZP;
            if (act) {
                double a1 = 0.0, a2 = 0.0;
#pragma unroll 5
                for (int c = c0; c < c1; c += 2) {
                    const double2 v = *reinterpret_cast<const double2 *>(rowp + c);
                    const double x = fma(np, a1, fma(nq, a2, v.x)), y = fma(np, x, fma(nq, a1, v.y));
                    a2 = x; a1 = y;
                    *reinterpret_cast<double2 *>(rowp + c) = make_double2(x, y);
                }
                sideF[(wid + 1) * LOC_LB + lane] = make_double2(a1, a2);      // state entering chunk wid + 1
            }
            __syncthreads();
            if (act) {
                double2 fin = wid > 0 ? sideF[wid * LOC_LB + lane] : make_double2(0.0, 0.0);
                double a1 = 0.0, a2 = 0.0;
                int c = c1 - 2;
                for (; c >= c0 + LOC_KC; c -= 2) {
                    const double2 v = *reinterpret_cast<const double2 *>(rowp + c);
                    const double y = fma(np, a1, fma(nq, a2, v.y)), x = fma(np, y, fma(nq, a1, v.x));
                    a2 = y; a1 = x;
                    *reinterpret_cast<double2 *>(rowp + c) = make_double2(x, y);
                }
#pragma unroll
                for (int k = LOC_KC - 2; k >= 0; k -= 2) {
                    if (c0 + k < c1) {
                        double2 v = *reinterpret_cast<const double2 *>(rowp + c0 + k);
                        v.x = fma(prm.al[k], fin.x, fma(prm.be[k], fin.y, v.x));
                        v.y = fma(prm.al[k + 1], fin.x, fma(prm.be[k + 1], fin.y, v.y));
                        const double y = fma(np, a1, fma(nq, a2, v.y)), x = fma(np, y, fma(nq, a1, v.x));
                        a2 = y; a1 = x;
                        *reinterpret_cast<double2 *>(rowp + c0 + k) = make_double2(x, y);
                    }
                }
                sideB[wid * LOC_LB + lane] = make_double2(a1, a2);            // state entering chunk wid - 1 from the right
            }
            // ---------------- P4: C^{n+1} = C^n + scale * (w + backward correction); warp = its own 30 columns,
            // half-warp = row parity, lane & 15 = column pair.  The first eight C^n rows are requested BEFORE the barrier that
            // ends P3 (C^n is read-only here), so their L2 latency hides behind it.
            const int half = lane >> 4, c = c0 + 2 * (lane & 15);                // r-region column of the pair
            const bool p4_on = (lane & 15) < LOC_XC / 2 && c >= He && c < He + wd;
            const size_t off = (size_t)(ya + lo - H + half) * N + (size_t)(x0 + c - He);
            const double2 *ci = reinterpret_cast<const double2 *>(Cm + (p4_on ? off : 0));
            const size_t N1 = (size_t)N;                                         // two rows = N double2
            const int nr = p4_on ? (nf - half + 1) >> 1 : 0;                     // rows of this parity
            double2 cv[8];
#pragma unroll
            for (int i = 0; i < 8; ++i)
                if (i < nr) cv[i] = __ldg(ci + (size_t)i * N1);
            __syncthreads();
            if (p4_on) {
                const int kb = c1 - 2 - c;                                       // distance of the pair's right column from the chunk end
                const bool corr = kb < LOC_KC && c1 < RWs;
                const double ax = corr ? prm.al[kb + 1] : 0.0, bx = corr ? prm.be[kb + 1] : 0.0;
                const double ay = corr ? prm.al[kb] : 0.0, by = corr ? prm.be[kb] : 0.0;
                double2 *co = reinterpret_cast<double2 *>(Om + off);
                const double2 *sb = sideB + (wid + 1) * LOC_LB + half;
                int zrow4 = (lo + half) % LOC_ZR;
                const double *zp = zring + zrow4 * LOC_ZP + c;
                const double osc = prm.oscale;
                for (int r0 = 0; r0 < nr; r0 += 8) {
                    if (r0 > 0) {
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            if (r0 + i < nr) cv[i] = __ldg(ci + (size_t)i * N1);
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        if (r0 + i < nr) {
                            double2 wv = *reinterpret_cast<const double2 *>(zp);
                            if (corr) {              // (never multiply an unwritten slot by zero: it may hold a NaN pattern)
                                const double2 bin = sb[2 * (r0 + i)];
                                wv.x = fma(ax, bin.x, fma(bx, bin.y, wv.x));
                                wv.y = fma(ay, bin.x, fma(by, bin.y, wv.y));
                            }
                            co[(size_t)i * N1] = make_double2(fma(osc, wv.x, cv[i].x), fma(osc, wv.y, cv[i].y));
                            zp += 2 * LOC_ZP; zrow4 += 2;
                            if (zrow4 >= LOC_ZR) { zrow4 -= LOC_ZR; zp -= LOC_ZRING; }
                        }
                    ci += 8 * N1; co += 8 * N1;
                }
            }
        }
        __syncthreads();
    }
}

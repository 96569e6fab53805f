// ch_local2d.cuh -- the whole 2D step in ONE pass over HBM when gamma dt is small (SURVEY.md section 8(f) NEXT-3 (i),
// DESIGN.md section 5b): read C^n once, write C^{n+1} once (16 B per grid-point update instead of 40).
//
//   k_step2d_local   C^{n+1} = C^n + (dt / c0^2) Lx^-T Lx^-1 Ly^-T Ly^-1 Lap_h mu(C^n)          P:29-30, include/ch.h
//
// Why it is legal.  A_d = c0 L^T L with L = I + p S^-1 + q S^-2 (ch_factor.h); the impulse response h_k of L^-1 decays
// like rho^k, rho = |root| (0.0976 at gamma dt = 0.01).  A recurrence started from a ZERO state H points before the
// first point that is used differs from the cyclic one by at most T(H) = sum_{k >= H} |h_k| times the data, and the
// host picks the smallest H with 2 G T(H) / c0 <= 2^-56 (ch_factor_reach; G = sum |h_k|): the truncation is below an
// eighth of an ulp of the local max |w| per sweep.  If that needs H > LOC_HMAX the exact two-kernel step runs instead.
//
// Structure.  The columns of a member are cut into strips of SW produced columns; a strip is computed on
// SW + 2 H columns (r-region) from SW + 2 H + 4 columns of C.  All strips of all members, stacked row after row, form a
// "tape"; every CTA (2 per SM, 7 warps) marches down an equal span of it, segment by segment (a segment = consecutive
// rows of one strip; it starts H + 2 rows early and ends H + 2 rows late, rows wrap).  Per block of 32 rows:
//   P1 (thread = column)   rows arrive by 16-byte cp.async in a 16-row ring; rolling register window: mu of the next row
//                          (x-neighbours of C from the ring, of mu by shuffle -- the 7 warps overlap by two columns),
//                          r = Lap_h mu, forward y-recurrence z (exact streaming, state in registers), z -> z-ring
//   P2 (thread = column)   backward y-recurrence over the block from a zero state H rows below it (H throw-away
//                          rows), in place: the 32 rows that are H rows behind the front are final
//   P3 (lane = row, warp = 30-column chunk)   x-sweep of those rows in place: forward / backward recurrence over the
//                          chunk after an H-column zero-state warm-up read from the neighbouring chunk
//   P4 (thread = column)   C^{n+1} = C^n + scale * w, C^n re-read through L2 (it was read ~50 rows ago), coalesced
// The result goes to a second array (the halo of a strip is another strip's interior): ch_step ping-pongs C and w.
#pragma once

#include <cuda_runtime.h>

#define LOC_NW 7                          // warps per CTA
#define LOC_NT (32 * LOC_NW)
#define LOC_LB 32                         // rows per block
#define LOC_HMAX 18                       // largest reach the geometry below allows
#define LOC_XC 30                         // columns a warp produces in P1 / one x-chunk in P3
#define LOC_RW (LOC_XC * LOC_NW)          // widest r-region: 210 columns
#define LOC_ZP LOC_RW                     // pitch of the z-ring; ZP / 2 odd: LDS.128 with lane = row is conflict free
#define LOC_ZR (LOC_LB + LOC_HMAX + 2)    // rows of the z-ring (a multiple of 4)
#define LOC_CP 216                        // pitch of the C staging ring (>= LOC_RW + 4 + 2, even)
#define LOC_SR 16                         // rows of the C staging ring: 4 groups of 4
#define LOC_SW_MAX (LOC_RW - 2 * LOC_HMAX)   // 174 produced columns at H = 18

struct LocalParams {
    double np, nq;                  // recurrence  z_i = b_i + np z_{i-1} + nq z_{i-2}
    double mgam, k1;                // mu = c (c^2 + k1) - gamma * (sum of the 4 neighbours), k1 = 4 gamma - 1
    double oscale;                  // dt / c0^2
    int N, M, H;                    // H = reach (rows / columns of zero-state warm-up), <= LOC_HMAX
    int nstrips, SW;                // strips per member, produced columns of a full strip (multiple of 4)
    long long total_rows, span;     // tape rows = M * nstrips * N, rows per CTA
};

static inline size_t local_smem_bytes() { return (size_t)(LOC_ZR * LOC_ZP + LOC_SR * LOC_CP) * 8; }

__device__ __forceinline__ void loc_cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void loc_cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int NPEND>
__device__ __forceinline__ void loc_cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(NPEND) : "memory"); }

__global__ void __launch_bounds__(LOC_NT, 2) k_step2d_local(const __grid_constant__ LocalParams prm,
                                                             const double *__restrict__ Cin, double *__restrict__ Cout)
{
    extern __shared__ double2 loc_sm[];
    double *const zring = reinterpret_cast<double *>(loc_sm);           // [LOC_ZR][LOC_ZP]
    double *const cst = zring + LOC_ZR * LOC_ZP;                          // [LOC_SR][LOC_CP]
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int N = prm.N, H = prm.H, He = (H + 1) & ~1;
    const double np = prm.np, nq = prm.nq, mgam = prm.mgam, k1 = prm.k1;
    const size_t n2 = (size_t)N * N;
    constexpr int ZRING = LOC_ZR * LOC_ZP;

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
        const int CWs = RWs + 4;                     // C-region: two more on either side
        // r rows: row t is global row ya - H + t; produced rows are t in [H, H + len); rounded up to a multiple of 4
        // (the extra rows are real rows: they only lengthen the backward warm-up)
        const int T = (len + 2 * H + 3) & ~3;
        const int NU = T + 4;                        // C rows: row u is global row ya - H - 2 + u
        const double *const Cm = Cin + (size_t)m * n2;
        double *const Om = Cout + (size_t)m * n2;

        // loader: thread = (row of a pair, column pair); lp walks down its column pair, wrapping at row N
        const int lrow = tid >= 112 ? 1 : 0, lpair = tid - 112 * lrow;
        const bool ldr = 2 * lpair < CWs;
        int lgx = (x0 - He - 2 + 2 * lpair) % N;
        if (lgx < 0) lgx += N;
        int lgy = (ya - H - 2 + lrow) % N;           // global row of the loader's next C row
        if (lgy < 0) lgy += N;
        int lu = lrow;                               // its index u
        double *ldst = cst + lrow * LOC_CP + 2 * lpair;
        auto issue_group = [&]() {                   // the next 4 C rows (two per loader row) into the ring
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (ldr && lu < NU) loc_cp_async16(ldst + (lu & (LOC_SR - 1)) * LOC_CP - lrow * LOC_CP, Cm + (size_t)lgy * N + lgx);
                lu += 2; lgy += 2;
                if (lgy >= N) lgy -= N;
            }
            loc_cp_async_commit();
        };

        // P1 mapping: warp w, lane l <-> r-region column rc = 30 w + l - 1 (C-region column cc = rc + 2); lanes 1..30 produce
        const int rc = LOC_XC * wid + lane - 1, cc = rc + 2;
        int p1_valid = lane >= 1 && lane <= LOC_XC && rc < RWs;
        asm volatile("" : "+r"(p1_valid));           // one predicate, not three re-derived branches
        double z1 = 0.0, z2 = 0.0, c_lo = 0.0, c_mid = 0.0, mu_a = 0.0, mu_b = 0.0;
        int zw = rc;                                 // row t of the z-ring, this thread's column (t = 0 now), as an offset
        const double *const cown = cst + cc;

        issue_group(); issue_group(); issue_group();
        const int nblocks = (T + LOC_LB - 1) / LOC_LB;
        for (int b = 0; b < nblocks; ++b) {
            const int top = LOC_LB * b + LOC_LB < T ? LOC_LB * b + LOC_LB : T;
            // ---------------- P1: RHS + forward y-recurrence of rows 32 b .. top - 1 (16 rows per trip: ring rows are immediates)
            for (int t16 = LOC_LB * b; t16 < top; t16 += 16) {
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    if (t16 + 4 * g < top) {         // CTA-uniform
                        loc_cp_async_wait<1>();      // all groups but the newest: C rows <= t + 7 have landed
                        __syncthreads();
                        issue_group();
                        if (g == 0 && t16 == 0) {
                            const double *q = cown;
                            const double C0 = q[0], C1 = q[LOC_CP], C2 = q[2 * LOC_CP], C3 = q[3 * LOC_CP];
                            mu_a = fma(mgam, (q[LOC_CP - 1] + q[LOC_CP + 1]) + (C0 + C2), C1 * fma(C1, C1, k1));
                            mu_b = fma(mgam, (q[2 * LOC_CP - 1] + q[2 * LOC_CP + 1]) + (C1 + C3), C2 * fma(C2, C2, k1));
                            c_lo = C2; c_mid = C3;
                        }
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int k = 4 * g + i;                                       // t = t16 + k, t16 % 16 == 0
                            const double *rowm = cown + ((k + 3) & (LOC_SR - 1)) * LOC_CP;
                            const double c_hi = cown[((k + 4) & (LOC_SR - 1)) * LOC_CP];
                            const double s4 = (rowm[-1] + rowm[1]) + (c_lo + c_hi);
                            const double mu_c = fma(mgam, s4, c_mid * fma(c_mid, c_mid, k1));
                            const double ml = __shfl_up_sync(0xffffffffu, mu_b, 1), mr = __shfl_down_sync(0xffffffffu, mu_b, 1);
                            const double r = fma(-4.0, mu_b, (ml + mr) + (mu_a + mu_c));
                            const double z = fma(np, z1, fma(nq, z2, r));
                            z2 = z1; z1 = z;
                            if (p1_valid) zring[zw + i * LOC_ZP] = z;
                            mu_a = mu_b; mu_b = mu_c; c_lo = c_mid; c_mid = c_hi;
                        }
                        zw += 4 * LOC_ZP;
                        if (zw >= ZRING) zw -= ZRING;
                    }
                }
            }
            // rows [lo, hi) become final in this block
            const int lo = LOC_LB * b - H > H ? LOC_LB * b - H : H;
            const int hi = top - H < H + len ? top - H : H + len;
            if (hi <= lo) continue;                  // CTA-uniform
            const int nf = hi - lo;
            __syncthreads();
            // ---------------- P2: backward y-recurrence, zero state at row top (>= H throw-away rows); thread = column pair
            if (2 * tid < RWs) {
                double vx1 = 0.0, vx2 = 0.0, vy1 = 0.0, vy2 = 0.0;
                // (ring position kept as an int: a shared-memory pointer that steps below the ring base wraps around
                // in the 32-bit shared window, so pointer comparisons cannot detect it)
                int po = ((top - 1) % LOC_ZR) * LOC_ZP + 2 * tid;
                for (int t = top - 1; t >= hi; --t) {
                    const double2 zz = *reinterpret_cast<const double2 *>(zring + po);
                    const double vx = fma(np, vx1, fma(nq, vx2, zz.x)), vy = fma(np, vy1, fma(nq, vy2, zz.y));
                    vx2 = vx1; vx1 = vx; vy2 = vy1; vy1 = vy;
                    po -= LOC_ZP;
                    if (po < 0) po += ZRING;
                }
                for (int t = hi - 1; t >= lo; --t) {
                    const double2 zz = *reinterpret_cast<const double2 *>(zring + po);
                    const double vx = fma(np, vx1, fma(nq, vx2, zz.x)), vy = fma(np, vy1, fma(nq, vy2, zz.y));
                    vx2 = vx1; vx1 = vx; vy2 = vy1; vy1 = vy;
                    *reinterpret_cast<double2 *>(zring + po) = make_double2(vx, vy);
                    po -= LOC_ZP;
                    if (po < 0) po += ZRING;
                }
            }
            __syncthreads();
            // ---------------- P3: x-sweep of rows lo .. hi - 1 (lane = row, warp = chunk of 30 columns)
            {
                const int c0 = LOC_XC * wid, c1 = c0 + LOC_XC < RWs ? c0 + LOC_XC : RWs;
                const bool act = lane < nf && c0 < RWs;
                double *rowp = zring + ((lo + lane) % LOC_ZR) * LOC_ZP;
                double a1 = 0.0, a2 = 0.0;
                if (act) {
#pragma unroll 3
                    for (int c = c0 - He > 0 ? c0 - He : 0; c < c0; c += 2) {
                        const double2 v = *reinterpret_cast<const double2 *>(rowp + c);
                        const double x = fma(np, a1, fma(nq, a2, v.x)), y = fma(np, x, fma(nq, a1, v.y));
                        a2 = x; a1 = y;
                    }
                }
                __syncthreads();
                if (act) {
#pragma unroll 5
                    for (int c = c0; c < c1; c += 2) {
                        const double2 v = *reinterpret_cast<const double2 *>(rowp + c);
                        const double x = fma(np, a1, fma(nq, a2, v.x)), y = fma(np, x, fma(nq, a1, v.y));
                        a2 = x; a1 = y;
                        *reinterpret_cast<double2 *>(rowp + c) = make_double2(x, y);
                    }
                }
                __syncthreads();
                a1 = 0.0; a2 = 0.0;
                if (act) {
#pragma unroll 3
                    for (int c = (c1 + He < RWs ? c1 + He : RWs) - 2; c >= c1; c -= 2) {
                        const double2 v = *reinterpret_cast<const double2 *>(rowp + c);
                        const double y = fma(np, a1, fma(nq, a2, v.y)), x = fma(np, y, fma(nq, a1, v.x));
                        a2 = y; a1 = x;
                    }
                }
                __syncthreads();
                if (act) {
#pragma unroll 5
                    for (int c = c1 - 2; c >= c0; c -= 2) {
                        const double2 v = *reinterpret_cast<const double2 *>(rowp + c);
                        const double y = fma(np, a1, fma(nq, a2, v.y)), x = fma(np, y, fma(nq, a1, v.x));
                        a2 = y; a1 = x;
                        *reinterpret_cast<double2 *>(rowp + c) = make_double2(x, y);
                    }
                }
                __syncthreads();
            }
            // ---------------- P4: C^{n+1} = C^n + scale * w on the produced columns; thread = column pair
            if (2 * tid < wd) {
                const size_t off = (size_t)(ya + lo - H) * N + (size_t)(x0 + 2 * tid);
                const double2 *ci = reinterpret_cast<const double2 *>(Cm + off);
                double2 *co = reinterpret_cast<double2 *>(Om + off);
                int zp = (lo % LOC_ZR) * LOC_ZP + He + 2 * tid;
                const double osc = prm.oscale;
                const int N2 = N >> 1;
                for (int r0 = 0; r0 < nf; r0 += 8) {
                    double2 cv[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        if (r0 + i < nf) cv[i] = __ldg(ci + (size_t)i * N2);
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        if (r0 + i < nf) {
                            const double2 wv = *reinterpret_cast<const double2 *>(zring + zp);
                            co[(size_t)i * N2] = make_double2(fma(osc, wv.x, cv[i].x), fma(osc, wv.y, cv[i].y));
                            zp += LOC_ZP;
                            if (zp >= ZRING) zp -= ZRING;
                        }
                    ci += (size_t)8 * N2; co += (size_t)8 * N2;
                }
            }
        }
        loc_cp_async_wait<0>();
        __syncthreads();
    }
}

// ch_factor.h -- host-side periodic (circulant) LU factorisation of
//   A = I + s (delta^2)^2 = circulant(s, -4s, 1+6s, -4s, s),   s = gamma dt      (include/ch.h)
//
// A is a circulant, so its symbol factors exactly (spectral factorisation):
//   s z^2 - 4 s z + (1+6s) - 4 s z^-1 + s z^-2 = c0 (1 + p z^-1 + q z^-2)(1 + p z + q z^2)
// with the two roots of 1 + p z^-1 + q z^-2 inside the unit circle.  Replacing z by the
// cyclic shift gives A = c0 * U * L with L = I + p S^-1 + q S^-2 (cyclic lower band) and
// U = L^T: the periodic LU factorisation with constant bands.  A v = b is then two cyclic
// two-term recurrences
//   forward : z_i = b_i - p z_{i-1} - q z_{i-2}            (indices mod N)
//   backward: v_i = z_i - p v_{i+1} - q v_{i+2},   result v / c0
// and each cyclic recurrence is solved chunk-parallel: every chunk of LC points runs from a
// zero state, the true state entering chunk c is
//   s_in(c) = sum_{j>=1} M^{j-1} out(c-j)       M = transfer matrix of one chunk,
// closed over the period by (I - M^P)^-1 (this is the Sherman-Morrison/Woodbury closure of
// the periodic factorisation), and the chunk is corrected by alpha_k a + beta_k b.
// Everything below is O(LC + P) doubles per (N, s), shared by all lines, axes and members.
#pragma once

#define CH_MAX_LC 32      // longest chunk a thread holds in registers
#define CH_MAX_P 128      // most chunks per line on the chunked path

struct ChFactor {
    double sigma;
    double np, nq;             // -p, -q of the recurrence
    double c0;                 // A = c0 U L
    double rho;                // modulus of the roots inside the unit circle
    // chunked path
    int LC, P, K;              // chunk length, chunks per line, neighbours summed (K == P: closed exactly)
    double alpha[CH_MAX_LC];   // homogeneous solutions: u_k for (u_-1,u_-2) = (1,0)
    double beta[CH_MAX_LC];    //                                   ... = (0,1)
    double W[CH_MAX_P][4];     // W_j = M^{j-1} (I - M^P)^-1 (K == P) or M^{j-1} (K < P), row-major 2x2
    // log-depth closure (warp-shuffle scan over the chunks of a line, used when K is large):
    // T_{k+1}(c) = T_k(c) + M^(2^k) T_k(c - 2^k) (cyclic), s_in(c) = (I - M^P)^-1 T_log2P(c - 1)
    double Mpow2[7][4];        // M^(2^k), k = 0..6, row-major 2x2
    double Wclose[4];          // (I - M^P)^-1
    // two-level form for lines of P = 32 W chunks, W = 2..4 (one warp scans 32 chunks, W warp aggregates are combined):
    // state entering chunk c = [sum_{j=1..lane} M^(j-1) out(c-j)] + M^lane S_w,  S_w = sum_{q=1..W} WG[q-1] A_{w-q},
    // A_w = sum_{j<32} M^j out(32 w + 31 - j),  WG[q-1] = (M^32)^(q-1) (I - M^P)^-1
    double Mlane[32][4];       // M^j, j = 0..31
    double WG[4][4];
    // generic path (one thread per line): closure of the whole line, (I - T^N)^-1
    double Wline[4];
};

// Fill f for line length N and chunk length LC (LC == 0: generic path only).
// Returns 0, or -1 if the factorisation failed its self-check.
int ch_factor_build(ChFactor *f, int N, double sigma, int LC);

// WG[q] = (M^32)^q (I - (M^32)^groups)^-1, q = 0..7, for a line of `groups` groups of 32 chunks of f->LC points
// (the two-level closure across the CTAs of a cluster, ch_cline2d.cuh).  Returns 0, or -1 on bad arguments.
int ch_factor_groups(const ChFactor *f, int groups, double WG[8][4]);

// Decay reach of the factor recurrences (one-pass local step, ch_local2d.cuh): the smallest H such that a forward and a
// backward recurrence each started from a ZERO state H points before the first point that is used reproduce
// w = A^-1 b to within  eps * max|b|:   2 G T(H) / c0 <= eps,   h_0 = 1, h_1 = np, h_k = np h_{k-1} + nq h_{k-2}
// (impulse response of L^-1), G = sum_k |h_k|, T(H) = sum_{k >= H} |h_k|.  Returns H, or -1 if it exceeds hmax.
int ch_factor_reach(const ChFactor *f, double eps, int hmax);

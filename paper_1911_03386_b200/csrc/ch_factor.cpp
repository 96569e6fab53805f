// ch_factor.cpp -- see ch_factor.h.  Host only; long double throughout, rounded once.
#include "ch_factor.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <vector>

namespace {

typedef long double ld;

struct M2 { ld a, b, c, d; };   // [[a b],[c d]]

M2 mul(const M2 &x, const M2 &y)
{
    return { x.a * y.a + x.b * y.c, x.a * y.b + x.b * y.d, x.c * y.a + x.d * y.c, x.c * y.b + x.d * y.d };
}

ld maxabs(const M2 &x) { return fmaxl(fmaxl(fabsl(x.a), fabsl(x.b)), fmaxl(fabsl(x.c), fabsl(x.d))); }

// (I - X)^-1
M2 inv_i_minus(const M2 &x)
{
    ld a = 1 - x.a, b = -x.b, c = -x.c, d = 1 - x.d, det = a * d - b * c;
    return { d / det, -b / det, -c / det, a / det };
}

// transfer matrix over n points: [[alpha_{n-1}, beta_{n-1}],[alpha_{n-2}, beta_{n-2}]]
M2 transfer(ld np, ld nq, int n, ld *alpha, ld *beta)
{
    ld a1 = 1, a2 = 0, b1 = 0, b2 = 1;     // u_{-1}, u_{-2}
    for (int k = 0; k < n; ++k) {
        ld a = np * a1 + nq * a2, b = np * b1 + nq * b2;
        if (alpha) { alpha[k] = a; beta[k] = b; }
        a2 = a1; a1 = a; b2 = b1; b1 = b;
    }
    return { a1, b1, a2, b2 };
}

}  // namespace

int ch_factor_build(ChFactor *f, int N, double sigma, int LC)
{
    std::memset(f, 0, sizeof(*f));
    if (!(sigma > 0) || N < 5 || LC < 0 || LC > CH_MAX_LC) return -1;
    f->sigma = sigma;
    // roots of z + 1/z = 2 + i / sqrt(s): the inside pair is z, conj(z)
    std::complex<ld> w(2.0L, 1.0L / sqrtl((ld)sigma));
    std::complex<ld> sq = std::sqrt(w * w - (ld)4);
    std::complex<ld> z = (ld)2 / (w + sq);
    if (std::abs(z) >= 1) z = (ld)2 / (w - sq);
    if (!(std::abs(z) < 1)) return -1;
    ld p = -2 * z.real(), q = std::norm(z), c0 = (ld)sigma / q;
    // polish (p, q) by Newton on  c0 (1+p^2+q^2) = 1+6s,  c0 p (1+q) = -4s  with c0 = s/q
    for (int it = 0; it < 3; ++it) {
        ld s = sigma;
        ld f1 = s * (1 + p * p + q * q) - (1 + 6 * s) * q;      // multiplied through by q
        ld f2 = p * (1 + q) + 4 * q;                            // divided by s, multiplied by q
        ld j11 = 2 * s * p, j12 = 2 * s * q - (1 + 6 * s), j21 = 1 + q, j22 = p + 4;
        ld det = j11 * j22 - j12 * j21;
        if (det == 0) break;
        p -= (f1 * j22 - f2 * j12) / det;
        q -= (j11 * f2 - j21 * f1) / det;
    }
    c0 = (ld)sigma / q;
    // self-check of the three symbol coefficients
    ld e0 = fabsl(c0 * (1 + p * p + q * q) - (1 + 6 * (ld)sigma)) / (1 + 6 * (ld)sigma);
    ld e1 = fabsl(c0 * p * (1 + q) + 4 * (ld)sigma) / (4 * (ld)sigma);
    if (!(e0 < 1e-15L && e1 < 1e-15L) || !(q < 1)) return -1;
    f->np = (double)-p; f->nq = (double)-q; f->c0 = (double)c0; f->rho = (double)sqrtl(q);
    // the tables are built from the ROUNDED coefficients, so that they are the exact
    // homogeneous solutions of the recurrence the kernels run
    ld np = f->np, nq = f->nq;

    M2 TN = transfer(np, nq, N, nullptr, nullptr);
    M2 WL = inv_i_minus(TN);
    f->Wline[0] = (double)WL.a; f->Wline[1] = (double)WL.b; f->Wline[2] = (double)WL.c; f->Wline[3] = (double)WL.d;

    if (LC == 0) return 0;
    if (N % LC != 0 || N / LC > CH_MAX_P || LC < 2) return -1;
    f->LC = LC; f->P = N / LC;
    ld alpha[CH_MAX_LC], beta[CH_MAX_LC];
    M2 M = transfer(np, nq, LC, alpha, beta);
    for (int k = 0; k < LC; ++k) { f->alpha[k] = (double)alpha[k]; f->beta[k] = (double)beta[k]; }
    // K: neighbours to sum.  Truncate when M^K is far below one ulp of the data, else close exactly.
    int K = f->P;
    {
        M2 pw = { 1, 0, 0, 1 };
        for (int j = 1; j < f->P; ++j) {
            pw = mul(pw, M);
            if (maxabs(pw) < 1e-22L) { K = j; break; }
        }
    }
    f->K = K;
    {
        M2 pw = M;
        for (int k = 0; k < 7; ++k) {
            f->Mpow2[k][0] = (double)pw.a; f->Mpow2[k][1] = (double)pw.b; f->Mpow2[k][2] = (double)pw.c; f->Mpow2[k][3] = (double)pw.d;
            pw = mul(pw, pw);
        }
        M2 MP = { 1, 0, 0, 1 };
        for (int j = 0; j < f->P; ++j) MP = mul(MP, M);
        const M2 wc = inv_i_minus(MP);
        f->Wclose[0] = (double)wc.a; f->Wclose[1] = (double)wc.b; f->Wclose[2] = (double)wc.c; f->Wclose[3] = (double)wc.d;
        M2 pj = { 1, 0, 0, 1 };
        for (int j = 0; j < 32; ++j) {
            f->Mlane[j][0] = (double)pj.a; f->Mlane[j][1] = (double)pj.b; f->Mlane[j][2] = (double)pj.c; f->Mlane[j][3] = (double)pj.d;
            pj = mul(pj, M);
        }
        M2 g = wc;                       // pj is now M^32
        for (int q = 0; q < 4; ++q) {
            f->WG[q][0] = (double)g.a; f->WG[q][1] = (double)g.b; f->WG[q][2] = (double)g.c; f->WG[q][3] = (double)g.d;
            g = mul(pj, g);
        }
    }
    M2 close = { 1, 0, 0, 1 };
    if (K == f->P) {
        M2 MP = { 1, 0, 0, 1 };
        for (int j = 0; j < f->P; ++j) MP = mul(MP, M);
        close = inv_i_minus(MP);
    }
    M2 pw = close;
    for (int j = 0; j < K; ++j) {
        f->W[j][0] = (double)pw.a; f->W[j][1] = (double)pw.b; f->W[j][2] = (double)pw.c; f->W[j][3] = (double)pw.d;
        pw = mul(M, pw);
    }
    return 0;
}

int ch_factor_groups(const ChFactor *f, int groups, double WG[8][4])
{
    if (f->LC < 2 || groups < 1 || groups > 8) return -1;
    const M2 M = transfer((ld)f->np, (ld)f->nq, f->LC, nullptr, nullptr);
    M2 M32 = { 1, 0, 0, 1 };
    for (int j = 0; j < 32; ++j) M32 = mul(M32, M);
    M2 MP = { 1, 0, 0, 1 };
    for (int j = 0; j < groups; ++j) MP = mul(MP, M32);
    M2 g = inv_i_minus(MP);
    for (int q = 0; q < 8; ++q) {
        WG[q][0] = (double)g.a; WG[q][1] = (double)g.b; WG[q][2] = (double)g.c; WG[q][3] = (double)g.d;
        g = mul(M32, g);
    }
    return 0;
}

int ch_factor_reach(const ChFactor *f, double eps, int hmax)
{
    // |h_k| summed far enough that the remainder is below 1e-40 of the total (rho < 1)
    const int KMAX = 4096;
    std::vector<ld> habs(KMAX);
    ld h1 = 1, h2 = 0, G = 0;
    int n = 0;
    for (; n < KMAX; ++n) {
        habs[n] = fabsl(h1);
        G += habs[n];
        const ld h = (ld)f->np * h1 + (ld)f->nq * h2;
        h2 = h1; h1 = h;
        if (n > 8 && habs[n] < 1e-40L * G && fabsl(h1) < 1e-40L * G) { ++n; break; }
    }
    if (n == KMAX) return -1;                     // no decay to speak of (large gamma dt)
    ld T = 0;
    int H = -1;
    for (int k = n - 1; k >= 0; --k) {            // T(k) = sum_{j >= k} |h_j|
        T += habs[k];
        if (2 * G * T / (ld)f->c0 > (ld)eps) { H = k + 1; break; }
    }
    if (H < 0) H = 0;
    return H <= hmax ? H : -1;
}

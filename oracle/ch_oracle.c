/*
 * oracle/ch_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 restatement of the ensemble Cahn-Hilliard ADI step and of
 * its diagnostics, written from the paper (citations P:nnn = line nnn of
 * /root/reference/PAPER.md) and from the readings listed in DESIGN.md.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant generator with paper_1911_03386_b200/csrc/.
 *
 * What it computes (h = 1, periodic grid of N^D points per member, x fastest;
 * all index arithmetic mod N):
 *
 *   mu   = C^3 - C - gamma * Lap_h C                  chemical potential of eq.(3)
 *   r    = dt * Lap_h mu                              explicit right-hand side
 *   w    = A_z^-1 A_y^-1 A_x^-1 r                     one cyclic pentadiagonal solve per
 *                                                     line and axis (ADI)
 *   C'   = C + w
 *
 * with A_d = I + gamma*dt*(delta_d^2)^2 the N x N circulant matrix whose rows are
 * (s, -4s, 1+6s, -4s, s), s = gamma*dt.  This "delta form" is algebraically the
 * north_star scheme  (I + a dxx^2)(I + a dyy^2) C' = C + dt Lap[(C)^3 - C]
 * - 2a dxx dyy C + a^2 dxx^2 dyy^2 C  (reading G1/G2); the literal form
 * is kept below as cho_step_literal() for the cross-check pin.
 *
 * Diagnostics of a state (eq.(4) P:34 with the 1/4 prefactor, reading G3; forward
 * differences, reading G4; analytic dissipation, reading G5; eq.(6); eq.(43)):
 *
 *   F    = sum_i [ (C_i^2-1)^2/4 + gamma/2 * sum_d (C_{i+e_d}-C_i)^2 ]
 *   Fdot = - sum_i sum_d (mu_{i+e_d} - mu_i)^2
 *   mass = sum_i C_i
 *   beta = - t * Fdot / F        (0 if F == 0)
 *
 * The line solve is the plain definition "solve A v = b": Schur bordering of a
 * banded Gaussian elimination (cho_plan_*), or for N <= 64 a dense Gaussian
 * elimination with partial pivoting (cho_solve_dense).  No blocking, fusion or
 * reordering.  OpenMP only over ensemble members.
 *
 * Pins (tests/test_oracle_pins.py): dense numpy solves of the circulant on 8/16-point
 * lines, DFT closed form, closed-form growth factor of a Fourier mode (2D, 3D),
 * closed-form finite-amplitude single-mode step, dense Kronecker solve of the whole
 * step, literal-vs-delta form, mass conservation, monotone F, centred difference of F
 * against Fdot (pins the 1/4), E[F(0)] closed form, tanh-kink energy and
 * near-stationarity, discrete steady state, equivariances.
 * Unpinned: the time origin of beta (convention G6) -- nothing in the paper fixes it.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

static long pmod(long i, long n) { i %= n; return i < 0 ? i + n : i; }

static long ipow(long n, int d) { long p = 1; while (d-- > 0) p *= n; return p; }

int cho_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void cho_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------ */
/* Cyclic pentadiagonal solve  A v = b,  A = circulant(s,-4s,1+6s,-4s,s) */
/* ------------------------------------------------------------------ */

/* Entry (i,j) of the N x N cyclic matrix, accumulating coincident wraps. */
static double cyc_entry(long N, double s, long i, long j)
{
    const double row[5] = { s, -4.0 * s, 1.0 + 6.0 * s, -4.0 * s, s };
    double v = 0.0;
    for (int o = -2; o <= 2; ++o)
        if (pmod(i + o, N) == j) v += row[o + 2];
    return v;
}

/* Dense Gaussian elimination with partial pivoting; a is n x n row-major and is
 * destroyed, b is overwritten by the solution.  Returns 0, or -1 if singular. */
int cho_dense_gauss(int n, double *a, double *b)
{
    for (int k = 0; k < n; ++k) {
        int piv = k;
        for (int i = k + 1; i < n; ++i)
            if (fabs(a[(long)i * n + k]) > fabs(a[(long)piv * n + k])) piv = i;
        if (a[(long)piv * n + k] == 0.0) return -1;
        if (piv != k) {
            for (int j = 0; j < n; ++j) {
                double t = a[(long)k * n + j]; a[(long)k * n + j] = a[(long)piv * n + j]; a[(long)piv * n + j] = t;
            }
            double t = b[k]; b[k] = b[piv]; b[piv] = t;
        }
        for (int i = k + 1; i < n; ++i) {
            double m = a[(long)i * n + k] / a[(long)k * n + k];
            if (m == 0.0) continue;
            for (int j = k; j < n; ++j) a[(long)i * n + j] -= m * a[(long)k * n + j];
            b[i] -= m * b[k];
        }
    }
    for (int i = n - 1; i >= 0; --i) {
        double t = b[i];
        for (int j = i + 1; j < n; ++j) t -= a[(long)i * n + j] * b[j];
        b[i] = t / a[(long)i * n + i];
    }
    return 0;
}

/* Dense path (N <= 64 intended): build the cyclic matrix and eliminate. */
int cho_solve_dense(int N, double sigma, double *b)
{
    double *a = (double *)malloc(sizeof(double) * (size_t)N * N);
    if (!a) return -2;
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) a[(long)i * N + j] = cyc_entry(N, sigma, i, j);
    int rc = cho_dense_gauss(N, a, b);
    free(a);
    return rc;
}

/* Banded (bandwidth 2) Gaussian elimination without pivoting of the open
 * n x n block A11 (it is symmetric positive definite), kept as multipliers. */
typedef struct {
    int N, n;              /* full size, n = N-2                         */
    double sigma;
    double *m1, *m2;       /* multipliers of row k applied to rows k+1,k+2 */
    double *d, *u1, *u2;   /* eliminated diagonal and two super-diagonals */
    double *G;             /* n x 2 : A11^-1 A12                          */
    double *A21full;       /* 2 x n dense rows of A21                     */
    double Sinv[2][2];     /* inverse of the Schur complement             */
} cho_plan;

static void band_solve(const cho_plan *p, double *x)   /* x := A11^-1 x */
{
    const int n = p->n;
    for (int k = 0; k < n; ++k) {
        if (k + 1 < n) x[k + 1] -= p->m1[k] * x[k];
        if (k + 2 < n) x[k + 2] -= p->m2[k] * x[k];
    }
    for (int i = n - 1; i >= 0; --i) {
        double t = x[i];
        if (i + 1 < n) t -= p->u1[i] * x[i + 1];
        if (i + 2 < n) t -= p->u2[i] * x[i + 2];
        x[i] = t / p->d[i];
    }
}

void cho_plan_free(cho_plan *p)
{
    if (!p) return;
    free(p->m1); free(p->m2); free(p->d); free(p->u1); free(p->u2); free(p->G); free(p->A21full);
    free(p);
}

cho_plan *cho_plan_create(int N, double sigma)
{
    if (N < 5) return NULL;
    cho_plan *p = (cho_plan *)calloc(1, sizeof(cho_plan));
    const int n = N - 2;
    p->N = N; p->n = n; p->sigma = sigma;
    p->m1 = (double *)calloc(n, sizeof(double)); p->m2 = (double *)calloc(n, sizeof(double));
    p->d = (double *)calloc(n, sizeof(double)); p->u1 = (double *)calloc(n, sizeof(double));
    p->u2 = (double *)calloc(n, sizeof(double)); p->G = (double *)calloc((size_t)2 * n, sizeof(double));
    p->A21full = (double *)calloc((size_t)2 * n, sizeof(double));
    /* band storage of A11: l2,l1 (sub), d, u1,u2 (super) per row */
    double *l1 = (double *)calloc(n, sizeof(double)), *l2 = (double *)calloc(n, sizeof(double));
    for (int i = 0; i < n; ++i) {
        p->d[i] = cyc_entry(N, sigma, i, i);
        if (i + 1 < n) { p->u1[i] = cyc_entry(N, sigma, i, i + 1); l1[i + 1] = cyc_entry(N, sigma, i + 1, i); }
        if (i + 2 < n) { p->u2[i] = cyc_entry(N, sigma, i, i + 2); l2[i + 2] = cyc_entry(N, sigma, i + 2, i); }
    }
    for (int k = 0; k < n; ++k) {
        if (k + 1 < n) {
            double m = l1[k + 1] / p->d[k];
            p->m1[k] = m;
            p->d[k + 1] -= m * p->u1[k];
            p->u1[k + 1] -= m * p->u2[k];
        }
        if (k + 2 < n) {
            double m = l2[k + 2] / p->d[k];
            p->m2[k] = m;
            l1[k + 2] -= m * p->u1[k];
            p->d[k + 2] -= m * p->u2[k];
        }
    }
    free(l1); free(l2);
    /* borders: unknowns N-2, N-1 */
    double S[2][2];
    for (int c = 0; c < 2; ++c) {
        double *g = p->G + (size_t)c * n;
        for (int i = 0; i < n; ++i) g[i] = cyc_entry(N, sigma, i, N - 2 + c);     /* column c of A12 */
        band_solve(p, g);
    }
    for (int r = 0; r < 2; ++r)
        for (int j = 0; j < n; ++j) p->A21full[(size_t)r * n + j] = cyc_entry(N, sigma, N - 2 + r, j);
    for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 2; ++c) {
            double t = cyc_entry(N, sigma, N - 2 + r, N - 2 + c);
            for (int j = 0; j < n; ++j) t -= p->A21full[(size_t)r * n + j] * p->G[(size_t)c * n + j];
            S[r][c] = t;
        }
    double det = S[0][0] * S[1][1] - S[0][1] * S[1][0];
    p->Sinv[0][0] = S[1][1] / det; p->Sinv[0][1] = -S[0][1] / det;
    p->Sinv[1][0] = -S[1][0] / det; p->Sinv[1][1] = S[0][0] / det;
    return p;
}

/* Solve A v = b for one contiguous line b[0..N) in place (banded + bordering). */
void cho_plan_solve(const cho_plan *p, double *b)
{
    const int n = p->n;
    band_solve(p, b);                                   /* y1 = A11^-1 b1 */
    double t0 = b[n], t1 = b[n + 1];
    for (int j = 0; j < n; ++j) {
        t0 -= p->A21full[j] * b[j];
        t1 -= p->A21full[(size_t)n + j] * b[j];
    }
    double x0 = p->Sinv[0][0] * t0 + p->Sinv[0][1] * t1;
    double x1 = p->Sinv[1][0] * t0 + p->Sinv[1][1] * t1;
    for (int j = 0; j < n; ++j) b[j] -= p->G[j] * x0 + p->G[(size_t)n + j] * x1;
    b[n] = x0; b[n + 1] = x1;
}

/* Solve `count` contiguous lines of length N in place (banded path). use_dense != 0
 * switches to the dense pivoted elimination (for the small-N cross-check). */
int cho_solve_lines(int N, double sigma, double *b, long count, int use_dense)
{
    if (use_dense) {
        for (long l = 0; l < count; ++l) { int rc = cho_solve_dense(N, sigma, b + l * N); if (rc) return rc; }
        return 0;
    }
    cho_plan *p = cho_plan_create(N, sigma);
    if (!p) return -1;
    for (long l = 0; l < count; ++l) cho_plan_solve(p, b + l * N);
    cho_plan_free(p);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Stencils                                                             */
/* ------------------------------------------------------------------ */

/* out_i = sum_d (f_{i+e_d} + f_{i-e_d}) - 2 D f_i  on one member */
static void laplacian(const double *f, double *out, int N, int D)
{
    const long n1 = N, n2 = (long)N * N;
    const int NZ = D == 3 ? N : 1;
    for (int z = 0; z < NZ; ++z)
        for (int y = 0; y < N; ++y)
            for (int x = 0; x < N; ++x) {
                long i = z * n2 + y * n1 + x;
                double s = f[z * n2 + y * n1 + pmod(x + 1, N)] + f[z * n2 + y * n1 + pmod(x - 1, N)];
                s += f[z * n2 + pmod(y + 1, N) * n1 + x] + f[z * n2 + pmod(y - 1, N) * n1 + x];
                if (D == 3) s += f[pmod(z + 1, N) * n2 + y * n1 + x] + f[pmod(z - 1, N) * n2 + y * n1 + x];
                out[i] = s - 2.0 * D * f[i];
            }
}

/* mu = C^3 - C - gamma Lap C  (eq.(3)) */
static void chem_potential(const double *C, double *mu, double *tmp, int N, int D, double gamma)
{
    const long npts = ipow(N, D);
    laplacian(C, tmp, N, D);
    for (long i = 0; i < npts; ++i) mu[i] = C[i] * C[i] * C[i] - C[i] - gamma * tmp[i];
}

/* second difference along one axis: out = delta_d^2 f */
static void d2_axis(const double *f, double *out, int N, int D, int axis)
{
    const long n1 = N, n2 = (long)N * N;
    const int NZ = D == 3 ? N : 1;
    for (int z = 0; z < NZ; ++z)
        for (int y = 0; y < N; ++y)
            for (int x = 0; x < N; ++x) {
                long i = z * n2 + y * n1 + x, ip, im;
                if (axis == 0) { ip = z * n2 + y * n1 + pmod(x + 1, N); im = z * n2 + y * n1 + pmod(x - 1, N); }
                else if (axis == 1) { ip = z * n2 + pmod(y + 1, N) * n1 + x; im = z * n2 + pmod(y - 1, N) * n1 + x; }
                else { ip = pmod(z + 1, N) * n2 + y * n1 + x; im = pmod(z - 1, N) * n2 + y * n1 + x; }
                out[i] = f[ip] - 2.0 * f[i] + f[im];
            }
}

/* solve A_axis v = w for every line of one member, in place */
static void sweep_axis(const cho_plan *p, double *w, double *line, int N, int D, int axis, int use_dense)
{
    const long n1 = N, n2 = (long)N * N;
    const long stride = axis == 0 ? 1 : (axis == 1 ? n1 : n2);
    const int NZ = D == 3 ? N : 1;
    /* enumerate the lines by their two (or one) fixed coordinates */
    for (int a = 0; a < NZ; ++a)
        for (int b = 0; b < N; ++b) {
            long base;
            if (axis == 0) base = a * n2 + b * n1;            /* fixed z=a, y=b */
            else if (axis == 1) base = a * n2 + b;            /* fixed z=a, x=b */
            else base = (long)a * n1 + b;                     /* axis z: fixed y=a, x=b (NZ == N) */
            for (int i = 0; i < N; ++i) line[i] = w[base + i * stride];
            if (use_dense) cho_solve_dense(N, p->sigma, line); else cho_plan_solve(p, line);
            for (int i = 0; i < N; ++i) w[base + i * stride] = line[i];
        }
}

/* r = dt * Lap mu(C) for the whole ensemble (exported for per-kernel parity). */
int cho_rhs(const double *C, double *r, int ensemble, int N, int D, double gamma, double dt)
{
    if (!C || !r || ensemble < 1 || N < 5 || (D != 2 && D != 3)) return -1;
    const long npts = ipow(N, D);
#pragma omp parallel for schedule(static)
    for (int m = 0; m < ensemble; ++m) {
        double *mu = (double *)malloc(sizeof(double) * npts), *tmp = (double *)malloc(sizeof(double) * npts);
        chem_potential(C + m * npts, mu, tmp, N, D, gamma);
        laplacian(mu, tmp, N, D);
        for (long i = 0; i < npts; ++i) r[m * npts + i] = dt * tmp[i];
        free(mu); free(tmp);
    }
    return 0;
}

/* w := A_axis^-1 w for every line of every member (exported for per-kernel parity). */
int cho_sweep(double *w, int ensemble, int N, int D, double sigma, int axis)
{
    if (!w || ensemble < 1 || N < 5 || (D != 2 && D != 3) || axis < 0 || axis >= D) return -1;
    const long npts = ipow(N, D);
    cho_plan *p = cho_plan_create(N, sigma);
    if (!p) return -1;
#pragma omp parallel for schedule(static)
    for (int m = 0; m < ensemble; ++m) {
        double *line = (double *)malloc(sizeof(double) * N);
        sweep_axis(p, w + m * npts, line, N, D, axis, 0);
        free(line);
    }
    cho_plan_free(p);
    return 0;
}

/* ------------------------------------------------------------------ */
/* The step (delta form) and the literal north_star form                */
/* ------------------------------------------------------------------ */

static void step_member(const cho_plan *p, double *C, double *mu, double *w, double *line,
                        int N, int D, double gamma, double dt, int use_dense)
{
    const long npts = ipow(N, D);
    chem_potential(C, mu, w, N, D, gamma);          /* mu^n                    */
    laplacian(mu, w, N, D);                         /* w = Lap mu              */
    for (long i = 0; i < npts; ++i) w[i] *= dt;     /* r = dt Lap mu           */
    for (int axis = 0; axis < D; ++axis)            /* x, then y, then z (G10) */
        sweep_axis(p, w, line, N, D, axis, use_dense);
    for (long i = 0; i < npts; ++i) C[i] += w[i];   /* C^{n+1} = C^n + w       */
}

/* Advance every member by nsteps steps in place.  use_dense: dense pivoted line solves. */
int cho_step(double *C, int ensemble, int N, int D, double gamma, double dt, long nsteps, int use_dense)
{
    if (!C || ensemble < 1 || N < 5 || (D != 2 && D != 3) || gamma <= 0 || dt <= 0 || nsteps < 0) return -1;
    const long npts = ipow(N, D);
    cho_plan *p = cho_plan_create(N, gamma * dt);
    if (!p) return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int m = 0; m < ensemble; ++m) {
        double *mu = (double *)malloc(sizeof(double) * npts), *w = (double *)malloc(sizeof(double) * npts);
        double *line = (double *)malloc(sizeof(double) * N);
        for (long s = 0; s < nsteps; ++s) step_member(p, C + m * npts, mu, w, line, N, D, gamma, dt, use_dense);
        free(mu); free(w); free(line);
    }
    cho_plan_free(p);
    return 0;
}

/* Literal north_star form (readings G1, G2), one member, one step:
 *   P C' = C + dt Lap(C^3-C) - 2a sum_{d<e} d2_d d2_e C + a^2 sum_{d<e} L_d L_e C (+ a^3 Lx Ly Lz C in 3D),
 *   a = gamma dt, L_d = d2_d d2_d, P = prod_d (I + a L_d). */
static void step_member_literal(const cho_plan *p, double *C, int N, int D, double gamma, double dt)
{
    const long npts = ipow(N, D);
    const double a = gamma * dt;
    double *rhs = (double *)malloc(sizeof(double) * npts), *phi = (double *)malloc(sizeof(double) * npts);
    double *t1 = (double *)malloc(sizeof(double) * npts), *t2 = (double *)malloc(sizeof(double) * npts);
    double *t3 = (double *)malloc(sizeof(double) * npts), *line = (double *)malloc(sizeof(double) * N);
    for (long i = 0; i < npts; ++i) phi[i] = C[i] * C[i] * C[i] - C[i];
    laplacian(phi, t1, N, D);
    for (long i = 0; i < npts; ++i) rhs[i] = C[i] + dt * t1[i];
    for (int d = 0; d < D; ++d)
        for (int e = d + 1; e < D; ++e) {
            d2_axis(C, t1, N, D, d); d2_axis(t1, t2, N, D, e);              /* d2_d d2_e C   */
            for (long i = 0; i < npts; ++i) rhs[i] -= 2.0 * a * t2[i];
            d2_axis(t2, t1, N, D, d); d2_axis(t1, t3, N, D, e);              /* L_d L_e C     */
            for (long i = 0; i < npts; ++i) rhs[i] += a * a * t3[i];
        }
    if (D == 3) {
        memcpy(t1, C, sizeof(double) * npts);
        for (int d = 0; d < 3; ++d) { d2_axis(t1, t2, N, D, d); d2_axis(t2, t1, N, D, d); }   /* Lx Ly Lz C */
        for (long i = 0; i < npts; ++i) rhs[i] += a * a * a * t1[i];
    }
    for (int axis = 0; axis < D; ++axis) sweep_axis(p, rhs, line, N, D, axis, 0);
    memcpy(C, rhs, sizeof(double) * npts);
    free(rhs); free(phi); free(t1); free(t2); free(t3); free(line);
}

int cho_step_literal(double *C, int ensemble, int N, int D, double gamma, double dt, long nsteps)
{
    if (!C || ensemble < 1 || N < 5 || (D != 2 && D != 3) || gamma <= 0 || dt <= 0 || nsteps < 0) return -1;
    const long npts = ipow(N, D);
    cho_plan *p = cho_plan_create(N, gamma * dt);
    if (!p) return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int m = 0; m < ensemble; ++m)
        for (long s = 0; s < nsteps; ++s) step_member_literal(p, C + m * npts, N, D, gamma, dt);
    cho_plan_free(p);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Diagnostics                                                          */
/* ------------------------------------------------------------------ */

/* out[m][4] = {F, Fdot, beta, mass} of the state at time t (eq.(4), (6), (43)). */
int cho_energy(const double *C, int ensemble, int N, int D, double gamma, double t, double *out)
{
    if (!C || !out || ensemble < 1 || N < 5 || (D != 2 && D != 3)) return -1;
    const long npts = ipow(N, D);
    const long n1 = N, n2 = (long)N * N;
    const int NZ = D == 3 ? N : 1;
#pragma omp parallel for schedule(static)
    for (int m = 0; m < ensemble; ++m) {
        const double *c = C + m * npts;
        double *mu = (double *)malloc(sizeof(double) * npts), *tmp = (double *)malloc(sizeof(double) * npts);
        chem_potential(c, mu, tmp, N, D, gamma);
        long double F = 0.0L, Fd = 0.0L, mass = 0.0L;
        for (int z = 0; z < NZ; ++z)
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    long i = z * n2 + y * n1 + x;
                    long nb[3];
                    nb[0] = z * n2 + y * n1 + pmod(x + 1, N);
                    nb[1] = z * n2 + pmod(y + 1, N) * n1 + x;
                    nb[2] = pmod(z + 1, N) * n2 + y * n1 + x;
                    long double ci = c[i], g2 = 0.0L, m2 = 0.0L;
                    for (int d = 0; d < D; ++d) {
                        long double dc = (long double)c[nb[d]] - ci, dm = (long double)mu[nb[d]] - (long double)mu[i];
                        g2 += dc * dc; m2 += dm * dm;
                    }
                    long double q = ci * ci - 1.0L;
                    F += 0.25L * q * q + 0.5L * (long double)gamma * g2;
                    Fd -= m2;
                    mass += ci;
                }
        out[4 * m + 0] = (double)F;
        out[4 * m + 1] = (double)Fd;
        out[4 * m + 2] = F == 0.0L ? 0.0 : (double)(-(long double)t * Fd / F);
        out[4 * m + 3] = (double)mass;
        free(mu); free(tmp);
    }
    return 0;
}

/* Run nsteps steps from time t0, sampling {F,Fdot,beta,mass} of the state after
 * n = 0, stride, 2 stride, ... steps (sample k at t = t0 + k stride dt, reading G6)
 * into series[k][m][4]; returns the number of samples written (<= capacity) or < 0. */
long cho_run(double *C, int ensemble, int N, int D, double gamma, double dt, long nsteps,
             long stride, double t0, double *series, long capacity)
{
    if (stride < 1 || !series) return -1;
    long k = 0, n = 0;
    for (;;) {
        if (n % stride == 0 && k < capacity) {
            int rc = cho_energy(C, ensemble, N, D, gamma, t0 + (double)n * dt, series + k * ensemble * 4);
            if (rc) return rc;
            ++k;
        }
        if (n >= nsteps) break;
        long adv = nsteps - n < stride ? nsteps - n : stride;
        int rc = cho_step(C, ensemble, N, D, gamma, dt, adv, 0);
        if (rc) return rc;
        n += adv;
    }
    return k;
}
